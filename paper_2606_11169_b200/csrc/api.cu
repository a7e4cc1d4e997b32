// api.cu — context management and the per-step C-ABI entry points of include/piper.h.
// Argument checks happen here on the host; the kernels live in route.cu / permute.cu / gemm_*.cu.
#include "piper_internal.cuh"

using namespace piper;

namespace {

bool desc_ok(const piper_moe_desc* D) {
    if (!D) return false;
    if (D->T < 1 || D->d < 8 || D->E < 1 || D->k < 1 || D->E_loc < 1 || D->I < 8 || D->I_shared < 0) return false;
    if (D->k > D->E || D->k > kMaxK || D->E > kMaxE) return false;
    if (D->e_lo < 0 || D->e_lo + D->E_loc > D->E) return false;
    if (D->d % 8 || D->I % 8 || D->I_shared % 8) return false;
    if (D->dtype != PIPER_DTYPE_F32 && D->dtype != PIPER_DTYPE_BF16) return false;
    if (D->gate_mode < 0 || D->gate_mode > 2) return false;
    if (D->row_align < 1 || D->row_align > 1024) return false;
    if (D->dw_dtype != D->dtype && !(D->dtype == PIPER_DTYPE_BF16 && D->dw_dtype == PIPER_DTYPE_F32)) return false;
    if (D->gemm_impl != PIPER_GEMM_AUTO && D->gemm_impl != PIPER_GEMM_SIMT) return false;
    if ((int64_t)D->T * D->k > (1ll << 30)) return false;
    return true;
}

inline int n_chunks_of(const piper_moe_desc* D) { return cdiv(D->T * D->k, kScanChunk); }
inline size_t round256(size_t v) { return (v + 255) & ~(size_t)255; }

struct WsLayout {
    size_t chunk_counts, chunk_counts_per, ep_scratch, shared_offsets, tc_scratch, total;
};
WsLayout ws_layout(const piper_moe_desc* D) {
    WsLayout L{};
    const size_t per = round256(sizeof(int32_t) * (size_t)n_chunks_of(D) * D->E_loc);
    size_t at = 0;
    L.chunk_counts = at, L.chunk_counts_per = per, at += per * kSchedSlots;
    L.ep_scratch = at, at += round256(sizeof(int32_t) * (size_t)n_chunks_of(D) * D->E);
    L.shared_offsets = at, at += 256;
    L.tc_scratch = at, at += tc_scratch_bytes(D);
    L.total = at;
    return L;
}

template <typename... P>
bool all_aligned(P... ptrs) {
    return (aligned16(ptrs) && ...);
}

inline Lane full_lane(piper_ctx* c, void* stream) { return Lane{static_cast<cudaStream_t>(stream), c->num_sms}; }

// Can this context's kernel variants serve its layer?  A bf16 layer under PIPER_GEMM_AUTO must run on the tcgen05
// kernels (no silent ~100x slower path), and fp32 dW of a bf16 layer exists only in the CTA-pair wgrad.
int variant_ok(const piper_ctx* c) {
    if (c->D.dtype != PIPER_DTYPE_BF16) return PIPER_OK;
    piper_chunk_args a{};
    const FfnProblem p = routed_problem(c, &a);
    const bool tc = c->D.gemm_impl == PIPER_GEMM_AUTO && tc_supported(c, p);
    if (c->D.gemm_impl == PIPER_GEMM_AUTO && !tc) return PIPER_ERR_UNSUPPORTED;
    if (c->D.dw_dtype == PIPER_DTYPE_F32 && !(tc && tc_wgrad_f32_ok(c, p))) return PIPER_ERR_UNSUPPORTED;
    return PIPER_OK;
}

}  // namespace

namespace piper {

int stream_slot(piper_ctx* c, cudaStream_t stream) {
    unsigned long long cap_id = 0;
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamGetCaptureInfo(stream, &st, &cap_id) != cudaSuccess) cudaGetLastError(), st = cudaStreamCaptureStatusNone;
    if (st != cudaStreamCaptureStatusActive) cap_id = 0;
    int match = -1, free_slot = -1, lru = 0;
    for (int i = 0; i < kSchedSlots; ++i) {
        const SchedSlot& e = c->sched_slots[i];
        if (!e.used) {
            if (free_slot < 0) free_slot = i;
        } else if (e.stream == stream && e.capture_id == cap_id) {
            match = i;
            break;
        } else if (e.last_use < c->sched_slots[lru].last_use || !c->sched_slots[lru].used) {
            lru = i;
        }
    }
    // no entry yet: a free one, else the least recently used stream / graph gives up its slot
    const int pick = match >= 0 ? match : (free_slot >= 0 ? free_slot : lru);
    SchedSlot& e = c->sched_slots[pick];
    e.used = true, e.stream = stream, e.capture_id = cap_id, e.last_use = ++c->sched_clock;
    return pick;
}

int32_t* scan_scratch(piper_ctx* c, cudaStream_t stream) {
    return c->chunk_counts + (size_t)stream_slot(c, stream) * c->chunk_counts_stride;
}

}  // namespace piper

extern "C" {

int64_t piper_a_cap(const piper_moe_desc* D) {
    if (!D) return 0;
    const int64_t kk = D->k < D->E_loc ? D->k : D->E_loc;
    return (int64_t)D->T * kk + (int64_t)D->E_loc * (D->row_align - 1);
}

int piper_workspace_bytes(const piper_moe_desc* D, size_t* bytes) {
    if (!desc_ok(D) || !bytes) return PIPER_ERR_INVALID;
    *bytes = ws_layout(D).total;
    return PIPER_OK;
}

int piper_create(const piper_moe_desc* D, int device, void* workspace, size_t workspace_bytes, piper_ctx** out) {
    if (!desc_ok(D) || !out || !workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return PIPER_ERR_INVALID;
    const WsLayout L = ws_layout(D);
    if (workspace_bytes < L.total) return PIPER_ERR_WORKSPACE;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) return PIPER_ERR_CUDA;
    piper_ctx* c = new (std::nothrow) piper_ctx();
    if (!c) return PIPER_ERR_INVALID;
    memset(c, 0, sizeof(*c));
    c->D = *D;
    c->device = device;
    c->ws = static_cast<char*>(workspace);
    c->ws_bytes = workspace_bytes;
    c->n_chunks = n_chunks_of(D);
    c->chunk_counts = reinterpret_cast<int32_t*>(c->ws + L.chunk_counts);
    c->chunk_counts_stride = L.chunk_counts_per / sizeof(int32_t);
    c->ep_scratch = reinterpret_cast<int32_t*>(c->ws + L.ep_scratch);
    c->shared_offsets = reinterpret_cast<int32_t*>(c->ws + L.shared_offsets);
    c->tc_scratch = c->ws + L.tc_scratch;
    bool ok = cudaSetDevice(device) == cudaSuccess &&
              cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device) == cudaSuccess;
    const int32_t so[2] = {0, D->T};
    ok = ok && cudaMemcpy(c->shared_offsets, so, sizeof(so), cudaMemcpyHostToDevice) == cudaSuccess;
    for (int i = 0; ok && i < kMaxEvents; ++i)
        ok = cudaEventCreateWithFlags(&c->events[i], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && tc_init(c) == PIPER_OK;
    if (!ok) {
        piper_destroy(c);
        return PIPER_ERR_CUDA;
    }
    c->move_items = 8, c->move_cap = 16;  // measured on C3
    c->fused_gather = 0;  // N2 fusion is built and parity-tested but measured slower than pack + TMA (DESIGN.md finding 19)
    c->pair_order = PIPER_ORDER_PROFILE, c->pair_part = PIPER_PART_SHARED;  // the policy that does not lose to serial
    const int rc = variant_ok(c);
    if (rc != PIPER_OK) {
        piper_destroy(c);
        return rc;
    }
    *out = c;
    return PIPER_OK;
}

int piper_destroy(piper_ctx* c) {
    if (!c) return PIPER_ERR_INVALID;
    pair_release(c);
    tc_release(c);
    if (c->side_stream) cudaStreamDestroy(c->side_stream);
    for (int i = 0; i < kMaxEvents; ++i)
        if (c->events[i]) cudaEventDestroy(c->events[i]);
    delete c;
    return PIPER_OK;
}

const char* piper_last_cuda_error(const piper_ctx* c) { return c ? c->err : "null context"; }
int64_t piper_kernel_launches(const piper_ctx* c) { return c ? c->launches : 0; }
int piper_gemm_path(const piper_ctx* c) {
    if (!c || c->D.dtype != PIPER_DTYPE_BF16 || c->D.gemm_impl != PIPER_GEMM_AUTO) return 0;
    piper_chunk_args a{};
    return tc_supported(c, routed_problem(c, &a)) ? 1 : 0;
}
const void* piper_debug_tc_counters(const piper_ctx* c) { return c && c->tc_prof ? c->tc_scratch : nullptr; }

int piper_chunk_gathers(const piper_ctx* c) { return c && fused_gather(c) ? 1 : 0; }

int piper_get_option(const piper_ctx* c, int option, int* value) {
    if (!c || !value) return PIPER_ERR_INVALID;
    switch (option) {
        case PIPER_OPT_TC_ROWS_ON_N: *value = c->tc_rows_on_n; return PIPER_OK;
        case PIPER_OPT_TC_2CTA: *value = c->tc_two_cta; return PIPER_OK;
        case PIPER_OPT_T_SMALL_ROWS: *value = c->tc_small_rows; return PIPER_OK;
        case PIPER_OPT_T_GREEDY: *value = c->tc_greedy; return PIPER_OK;
        case PIPER_OPT_TC_PROFILE: *value = c->tc_prof; return PIPER_OK;
        case PIPER_OPT_FUSED_GATHER: *value = c->fused_gather; return PIPER_OK;
        case PIPER_OPT_T_DUAL: *value = c->tc_dual; return PIPER_OK;
        case PIPER_OPT_WGRAD_STORE_WARP: *value = c->tc_store_warp; return PIPER_OK;
        case PIPER_OPT_MOVE_ITEMS: *value = c->move_items; return PIPER_OK;
        case PIPER_OPT_MOVE_CAP: *value = c->move_cap; return PIPER_OK;
    }
    return PIPER_ERR_INVALID;
}

int piper_set_option(piper_ctx* c, int option, int value) {
    int old = 0;
    if (piper_get_option(c, option, &old) != PIPER_OK) return PIPER_ERR_INVALID;
    int* field = nullptr;
    switch (option) {
        case PIPER_OPT_TC_ROWS_ON_N: field = &c->tc_rows_on_n; if (value != 0 && value != 1) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_TC_2CTA: field = &c->tc_two_cta; if (value < 0 || value > 2) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_T_SMALL_ROWS: field = &c->tc_small_rows; if (value < 0 || value > 128) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_T_GREEDY: field = &c->tc_greedy; if (value != 0 && value != 1) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_TC_PROFILE: field = &c->tc_prof; if (value != 0 && value != 1) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_FUSED_GATHER: field = &c->fused_gather; if (value < 0 || value > 2) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_T_DUAL: field = &c->tc_dual; if (value != 0 && value != 1) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_WGRAD_STORE_WARP: field = &c->tc_store_warp; if (value < 0 || value > 2) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_MOVE_ITEMS: field = &c->move_items; if (value < 1 || value > 64) return PIPER_ERR_INVALID; break;
        case PIPER_OPT_MOVE_CAP: field = &c->move_cap; if (value < 1 || value > 64) return PIPER_ERR_INVALID; break;
    }
    *field = value;
    const int rc = variant_ok(c);  // e.g. row_align 16 needs the rows-on-N + CTA-pair kernels, fp32 dW the CTA-pair wgrad
    if (rc != PIPER_OK) *field = old;
    return rc;
}
int piper_pair_partition_mode(const piper_ctx* c) { return c ? c->pair_mode : 0; }
int piper_set_wgrad_accumulate(piper_ctx* c, int accumulate) {
    if (!c || (accumulate != 0 && accumulate != 1)) return PIPER_ERR_INVALID;
    if (accumulate && (c->D.dw_dtype != PIPER_DTYPE_F32 || c->D.dtype != PIPER_DTYPE_BF16)) return PIPER_ERR_UNSUPPORTED;
    c->wgrad_accumulate = accumulate;
    return PIPER_OK;
}

int piper_route_topk(piper_ctx* c, const float* logits, int32_t* topk_idx, float* gates, int32_t* counts_global,
                     void* stream) {
    if (!c || !all_aligned(logits, topk_idx, gates, counts_global)) return PIPER_ERR_INVALID;
    return launch_route_topk(c, full_lane(c, stream), logits, topk_idx, gates, counts_global);
}

int piper_dispatch_pack(piper_ctx* c, const void* x, const int32_t* topk_idx, const float* gates, int32_t* counts,
                        int32_t* offsets, int32_t* row_of, int32_t* src_of, float* gate_rows, void* xp, void* stream) {
    if (!c || !all_aligned(x, topk_idx, gates, counts, offsets, row_of, src_of, gate_rows, xp)) return PIPER_ERR_INVALID;
    const Lane ln = full_lane(c, stream);
    const int rc = launch_scan_rank(c, ln, topk_idx, gates, counts, offsets, row_of, src_of, gate_rows);
    if (rc != PIPER_OK) return rc;
    return launch_pack(c, ln, x, offsets, row_of, src_of, xp);
}

int piper_expert_ffn_fwd(piper_ctx* c, const void* xp, const int32_t* offsets, const void* w_gate, const void* w_up,
                         const void* w_down, void* g_save, void* u_save, void* h_save, void* o, void* stream) {
    if (!c || !all_aligned(xp, offsets, w_gate, w_up, w_down, g_save, u_save, h_save, o)) return PIPER_ERR_INVALID;
    piper_chunk_args a{};
    a.xp = const_cast<void*>(xp), a.offsets = const_cast<int32_t*>(offsets);
    a.w_gate = w_gate, a.w_up = w_up, a.w_down = w_down;
    a.g_save = g_save, a.u_save = u_save, a.h_save = h_save, a.o = o;
    const FfnProblem p = routed_problem(c, &a);
    const Lane ln = full_lane(c, stream);
    const int rc = ffn_gemm1(c, ln, p);
    return rc != PIPER_OK ? rc : ffn_gemm2(c, ln, p);
}

int piper_shared_ffn_fwd(piper_ctx* c, const void* x, const void* ws_gate, const void* ws_up, const void* ws_down,
                         void* g_save, void* u_save, void* h_save, void* s, void* stream) {
    if (!c || c->D.I_shared == 0 || !all_aligned(x, ws_gate, ws_up, ws_down, g_save, u_save, h_save, s))
        return PIPER_ERR_INVALID;
    piper_chunk_args a{};
    a.x = x, a.ws_gate = ws_gate, a.ws_up = ws_up, a.ws_down = ws_down;
    a.gs_save = g_save, a.us_save = u_save, a.hs_save = h_save, a.s = s;
    const FfnProblem p = shared_problem(c, &a);
    const Lane ln = full_lane(c, stream);
    const int rc = ffn_gemm1(c, ln, p);
    return rc != PIPER_OK ? rc : ffn_gemm2(c, ln, p);
}

int piper_combine(piper_ctx* c, const void* o, const int32_t* row_of, const float* gates, const void* s, void* y,
                  void* stream) {
    if (!c || !all_aligned(o, row_of, gates, y) || (s && !aligned16(s))) return PIPER_ERR_INVALID;
    return launch_combine(c, full_lane(c, stream), o, row_of, gates, s, nullptr, y, true);
}

int piper_combine_bwd(piper_ctx* c, const void* dy, const void* o, const int32_t* src_of, const int32_t* row_of,
                      const float* gates, const int32_t* offsets, void* d_o, float* dgates, void* stream) {
    if (!c || !all_aligned(dy, o, src_of, row_of, gates, offsets, d_o, dgates)) return PIPER_ERR_INVALID;
    return launch_combine_bwd(c, full_lane(c, stream), dy, o, src_of, row_of, gates, offsets, d_o, dgates);
}

int piper_expert_ffn_bwd(piper_ctx* c, const void* d_o, const void* xp, const void* g_save, const void* u_save,
                         const void* h_save, const int32_t* offsets, const void* w_gate, const void* w_up,
                         const void* w_down, void* dg, void* du, void* dxp, void* dw_gate, void* dw_up, void* dw_down,
                         int accumulate, void* stream) {
    if (!c || !all_aligned(d_o, xp, g_save, u_save, h_save, offsets, w_gate, w_up, w_down, dg, du, dxp, dw_gate, dw_up,
                           dw_down))
        return PIPER_ERR_INVALID;
    if (accumulate != 0 && accumulate != 1) return PIPER_ERR_INVALID;
    piper_chunk_args a{};
    a.d_o = const_cast<void*>(d_o), a.xp = const_cast<void*>(xp), a.offsets = const_cast<int32_t*>(offsets);
    a.g_save = const_cast<void*>(g_save), a.u_save = const_cast<void*>(u_save), a.h_save = const_cast<void*>(h_save);
    a.w_gate = w_gate, a.w_up = w_up, a.w_down = w_down;
    a.dg = dg, a.du = du, a.dxp = dxp, a.dw_gate = dw_gate, a.dw_up = dw_up, a.dw_down = dw_down;
    FfnProblem p = routed_problem(c, &a);
    p.accumulate = accumulate;
    const Lane ln = full_lane(c, stream);
    int rc = ffn_dgrad1(c, ln, p);
    if (rc == PIPER_OK) rc = ffn_dgrad2(c, ln, p);
    if (rc == PIPER_OK) rc = ffn_wgrad(c, ln, p);
    return rc;
}

int piper_shared_ffn_bwd(piper_ctx* c, const void* dy, const void* x, const void* g_save, const void* u_save,
                         const void* h_save, const void* ws_gate, const void* ws_up, const void* ws_down, void* dgs,
                         void* dus, void* dxs, void* dws_gate, void* dws_up, void* dws_down, int accumulate,
                         void* stream) {
    if (!c || c->D.I_shared == 0 ||
        !all_aligned(dy, x, g_save, u_save, h_save, ws_gate, ws_up, ws_down, dgs, dus, dxs, dws_gate, dws_up, dws_down))
        return PIPER_ERR_INVALID;
    if (accumulate != 0 && accumulate != 1) return PIPER_ERR_INVALID;
    piper_chunk_args a{};
    a.dy = dy, a.x = x;
    a.gs_save = const_cast<void*>(g_save), a.us_save = const_cast<void*>(u_save), a.hs_save = const_cast<void*>(h_save);
    a.ws_gate = ws_gate, a.ws_up = ws_up, a.ws_down = ws_down;
    a.dgs = dgs, a.dus = dus, a.dxs = dxs, a.dws_gate = dws_gate, a.dws_up = dws_up, a.dws_down = dws_down;
    FfnProblem p = shared_problem(c, &a);
    p.accumulate = accumulate;
    const Lane ln = full_lane(c, stream);
    int rc = ffn_dgrad1(c, ln, p);
    if (rc == PIPER_OK) rc = ffn_dgrad2(c, ln, p);
    if (rc == PIPER_OK) rc = ffn_wgrad(c, ln, p);
    return rc;
}

int piper_dispatch_unpack(piper_ctx* c, const void* dxp, const int32_t* row_of, const void* dx_shared, void* dx,
                          void* stream) {
    if (!c || !all_aligned(dxp, row_of, dx) || (dx_shared && !aligned16(dx_shared))) return PIPER_ERR_INVALID;
    return launch_combine(c, full_lane(c, stream), dxp, row_of, nullptr, dx_shared, nullptr, dx, false);
}

int piper_dispatch_unpack_router(piper_ctx* c, const void* dxp, const int32_t* row_of, const void* dx_shared,
                                 const void* dx_router, void* dx, void* stream) {
    if (!c || !all_aligned(dxp, row_of, dx) || (dx_shared && !aligned16(dx_shared)) || (dx_router && !aligned16(dx_router)))
        return PIPER_ERR_INVALID;
    return launch_combine(c, full_lane(c, stream), dxp, row_of, nullptr, dx_shared, dx_router, dx, false);
}

int piper_router_fwd(piper_ctx* c, const void* x, const void* w_r, const float* bias, float* logits, void* stream) {
    if (!c || !all_aligned(x, w_r, logits) || (bias && !aligned16(bias))) return PIPER_ERR_INVALID;
    return launch_router_fwd(c, full_lane(c, stream), x, w_r, bias, logits);
}

int piper_router_bwd(piper_ctx* c, const void* x, const void* w_r, const int32_t* topk_idx, const float* dz_sel,
                     void* dz_scratch, float* dw_r, void* dx_router, void* stream) {
    if (!c || !all_aligned(x, w_r, topk_idx, dz_sel, dz_scratch, dw_r, dx_router)) return PIPER_ERR_INVALID;
    return launch_router_bwd(c, full_lane(c, stream), x, w_r, topk_idx, dz_sel, dz_scratch, dw_r, dx_router);
}

int piper_route_bwd(piper_ctx* c, const float* logits, const int32_t* topk_idx, const float* gates, const float* dgates,
                    float* dz_sel, void* stream) {
    if (!c || !all_aligned(logits, topk_idx, gates, dgates, dz_sel)) return PIPER_ERR_INVALID;
    return launch_route_bwd(c, full_lane(c, stream), logits, topk_idx, gates, dgates, dz_sel);
}

}  // extern "C"
