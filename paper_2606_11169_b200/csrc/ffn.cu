// ffn.cu — the FFN tasks of the chunk (F4, B2-B4 of SURVEY.md §8a) as seen by the chunk scheduler:
// problem descriptions for the routed experts and the shared expert, and the choice between the
// tcgen05 kernels (bf16) and the FP32-ALU kernels (fp32 storage, or PIPER_GEMM_SIMT).
#include "piper_internal.cuh"

namespace piper {

FfnProblem routed_problem(const piper_ctx* c, const piper_chunk_args* a) {
    const piper_moe_desc& D = c->D;
    FfnProblem p{};
    p.G = D.E_loc, p.d = D.d, p.I = D.I;
    p.max_rows = (int)piper_a_cap(&D);
    p.max_group_rows = D.T + D.row_align - 1;
    p.exp_rows = (int)((long long)D.T * D.k * D.E_loc / D.E);
    p.accumulate = c->wgrad_accumulate;
    p.offsets = a->offsets, p.counts = a->counts;
    p.xp = a->xp, p.w_gate = a->w_gate, p.w_up = a->w_up, p.w_down = a->w_down;
    p.g = a->g_save, p.u = a->u_save, p.h = a->h_save, p.o = a->o;
    p.d_o = a->d_o, p.dg = a->dg, p.du = a->du, p.dxp = a->dxp;
    p.dw_gate = a->dw_gate, p.dw_up = a->dw_up, p.dw_down = a->dw_down;
    return p;
}

FfnProblem shared_problem(const piper_ctx* c, const piper_chunk_args* a) {
    const piper_moe_desc& D = c->D;
    FfnProblem p{};
    p.G = 1, p.d = D.d, p.I = D.I_shared;
    p.max_rows = D.T, p.max_group_rows = D.T, p.exp_rows = D.T;
    p.accumulate = c->wgrad_accumulate;
    p.offsets = c->shared_offsets, p.counts = c->shared_offsets + 1;
    p.xp = a->x, p.w_gate = a->ws_gate, p.w_up = a->ws_up, p.w_down = a->ws_down;
    p.g = a->gs_save, p.u = a->us_save, p.h = a->hs_save, p.o = a->s;
    p.d_o = a->dy, p.dg = a->dgs, p.du = a->dus, p.dxp = a->dxs;
    p.dw_gate = a->dws_gate, p.dw_up = a->dws_up, p.dw_down = a->dws_down;
    return p;
}

static bool use_tc(const piper_ctx* c, const FfnProblem& p) {
    return c->D.dtype == PIPER_DTYPE_BF16 && c->D.gemm_impl == PIPER_GEMM_AUTO && tc_supported(c, p);
}

// N2 fusion: only the rows-on-N kernels (fwd1, dgrad1) and the CTA-pair wgrad can gather
bool fused_gather(const piper_ctx* c) {
    if (!c->fused_gather) return false;
    piper_chunk_args a{};
    const FfnProblem p = routed_problem(c, &a);
    return use_tc(c, p) && tc_gather_ok(c, p);
}

int ffn_gemm1(piper_ctx* c, Lane ln, const FfnProblem& p) { return use_tc(c, p) ? tc_ffn_fwd1(c, ln, p) : simt_ffn_fwd(c, ln, p, 1); }
int ffn_gemm2(piper_ctx* c, Lane ln, const FfnProblem& p) { return use_tc(c, p) ? tc_ffn_fwd2(c, ln, p) : simt_ffn_fwd(c, ln, p, 2); }
int ffn_dgrad1(piper_ctx* c, Lane ln, const FfnProblem& p) { return use_tc(c, p) ? tc_ffn_dgrad1(c, ln, p) : simt_ffn_dgrad(c, ln, p, 1); }
int ffn_dgrad2(piper_ctx* c, Lane ln, const FfnProblem& p) { return use_tc(c, p) ? tc_ffn_dgrad2(c, ln, p) : simt_ffn_dgrad(c, ln, p, 2); }
int ffn_wgrad(piper_ctx* c, Lane ln, const FfnProblem& p) {
    if (use_tc(c, p)) return tc_ffn_wgrad(c, ln, p);
    if (p.accumulate || c->D.dw_dtype != c->D.dtype) return PIPER_ERR_UNSUPPORTED;  // fp32 dW of bf16 layers: tcgen05 only
    return simt_ffn_wgrad(c, ln, p);
}

}  // namespace piper
