/*
 * piper.h — C-ABI boundary of the B200 (sm_100a) MoE-chunk library.
 *
 * What it is: the per-device expert-parallel MoE chunk that Piper's DualPipeV schedule overlaps
 * (§6.3; Fig. 3b): router top-k, histogram + scan + stable permutation
 * into the per-expert buffers an EP all-to-all would carry (the payload of the `Shard` directive,
 * PAPER.md:185), grouped SwiGLU expert FFN forward / dgrad / wgrad, gate-weighted combine, and the
 * forward chunk of one microbatch co-scheduled with the backward chunk of another on two logical
 * streams (list scheduling PAPER.md:267-271; event rule PAPER.md:279-286) under an
 * explicit SM split (beyond the paper).  The paper states none of the MoE arithmetic;
 * it is fixed by BASELINE.json:north_star / configs and restated in SURVEY.md §8(c) "Definition" and
 * DESIGN.md.  Every entry point below cites the step of SURVEY.md §8(a) it implements.
 *
 * Conventions (all entry points):
 *  - return value: PIPER_OK or a negative PIPER_ERR_* code; never throws, never aborts;
 *  - every tensor pointer is a DEVICE pointer owned by the caller, 16-byte aligned, row-major,
 *    contiguous; the library never allocates or frees device memory and never frees caller memory;
 *    `workspace` (device, caller-owned) must outlive the context.  Host-side CUDA objects (events, the
 *    side stream of piper_set_chunk_overlap) are created in piper_create(); the SM partitions and
 *    streams of step P are created by piper_pair_prepare() (or by the first piper_run_chunk_pair() of a
 *    split, which therefore must not run inside a stream capture); no other call creates anything;
 *  - `stream` is a cudaStream_t passed as void*; calls only enqueue work: no host synchronisation,
 *    no host read-back of device data (the packed row count A lives on the device in
 *    offsets[E_loc]), so a sequence of calls can be captured in a CUDA graph and replayed;
 *  - activation / weight element type is `desc.dtype` (0 = fp32, 1 = bf16 with fp32 accumulation);
 *    logits, gates, gate_rows, dgates, dz_sel are always fp32; indices are int32;
 *  - row buffers (xp, o, d_o, dxp, g_save, u_save, h_save, src_of, gate_rows) hold
 *    A_cap = T*min(k,E_loc) + E_loc*(row_align-1) rows; rows >= offsets[E_loc] are never written and
 *    their contents are unspecified;
 *  - preconditions checked on the host: shapes > 0, k <= E, k <= 8, E <= 512, d % 8 == 0, I % 8 == 0,
 *    I_shared % 8 == 0, pointers non-null and 16-byte aligned.  Logits must be finite (or -inf with
 *    at least k finite entries per row, reading c-7); the device does not validate data;
 *  - a piper_ctx is not thread-safe.  Calls of one context may go to different streams and run
 *    concurrently on the device (every GEMM launch takes the tile counters of its own stream; up to 64
 *    streams / captured graphs per context are tracked, the least recently used entry is recycled
 *    beyond that).
 */
#ifndef PIPER_H_
#define PIPER_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PIPER_OK 0
#define PIPER_ERR_INVALID (-1)     /* bad shape, null or misaligned pointer                         */
#define PIPER_ERR_UNSUPPORTED (-2) /* valid request this build does not implement                   */
#define PIPER_ERR_WORKSPACE (-3)   /* workspace too small                                           */
#define PIPER_ERR_CUDA (-4)        /* a CUDA call failed: see piper_last_cuda_error()               */

#define PIPER_DTYPE_F32 0
#define PIPER_DTYPE_BF16 1

#define PIPER_GATE_SOFTMAX_RENORM 0 /* g_j = exp(z_j - z_0) / sum_{j'<k} exp(z_j' - z_0)            */
#define PIPER_GATE_SIGMOID_RENORM 1 /* s_j = 1/(1+exp(-z_j)); g_j = s_j / sum_{j'<k} s_j'           */
#define PIPER_GATE_SOFTMAX_FULL 2   /* g_j = exp(z_j - m) / sum_{e<E} exp(z_e - m)                  */

#define PIPER_GEMM_AUTO 0 /* bf16: tcgen05/TMEM/TMA kernels; fp32: FP32-ALU kernels (1e-5 bar).  A bf16 layer the
                           * tcgen05 kernels cannot take (row_align % 16 != 0 with more than one local expert,
                           * d or I < 64) is refused by piper_create with PIPER_ERR_UNSUPPORTED instead of
                           * silently running ~100x slower: ask for PIPER_GEMM_SIMT explicitly.               */
#define PIPER_GEMM_SIMT 1 /* the FP32-ALU grouped GEMM for any dtype / row_align (cross-check of the tcgen05 path) */

typedef struct piper_ctx piper_ctx;

/* Layer description (SURVEY.md §8 notation).  Local experts are [e_lo, e_lo + E_loc). */
typedef struct {
    int32_t T, d, E, k, e_lo, E_loc, I, I_shared; /* I_shared = 0: no shared expert                 */
    int32_t dtype;     /* PIPER_DTYPE_*                                                             */
    int32_t gate_mode; /* PIPER_GATE_*                                                              */
    int32_t row_align; /* >= 1: each expert's row segment is padded to a multiple; pad rows are 0   */
    int32_t dw_dtype;  /* element type of dW outputs: = dtype, or F32 on a BF16 layer (main-grad style) */
    int32_t gemm_impl; /* PIPER_GEMM_*                                                              */
} piper_moe_desc;

/* Device workspace the context needs (scan scratch, tile counters).  Host call. */
int piper_workspace_bytes(const piper_moe_desc* desc, size_t* bytes);
/* Creates a context on CUDA device `device`.  `workspace` is a device pointer of at least
 * piper_workspace_bytes() bytes, 256-byte aligned, owned by the caller. */
int piper_create(const piper_moe_desc* desc, int device, void* workspace, size_t workspace_bytes, piper_ctx** out);
int piper_destroy(piper_ctx* ctx);
/* Text of the last CUDA error seen by this context (host string owned by the context). */
const char* piper_last_cuda_error(const piper_ctx* ctx);
/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
int64_t piper_kernel_launches(const piper_ctx* ctx);
/* Which GEMM family serves the routed experts of this context: 1 = tcgen05/TMEM/TMA, 0 = FP32 ALUs. */
int piper_gemm_path(const piper_ctx* ctx);
/* Debug (PIPER_OPT_TC_PROFILE = 1): device pointer to the wait-cycle counters the tcgen05 kernels wrote,
 * [16 launches (cycled)][160 CTAs][8] int64; NULL when profiling is off. */
const void* piper_debug_tc_counters(const piper_ctx* ctx);
/* Kernel-variant switches of a context (host state; nothing is read from the environment).  Defaults in brackets.
 *  PIPER_OPT_TC_ROWS_ON_N [1]  rows-on-N CTA-pair kernels for fwd / dgrad; 0 = rows-on-M kernels (row_align % 128 only)
 *  PIPER_OPT_TC_2CTA      [2]  CTA-pair kernels: 0 never (1-CTA kernels; bf16 dW, row_align % 128 only), 1 always,
 *                              2 by expected group length
 *  PIPER_OPT_T_SMALL_ROWS [32] rows-on-N: chunks of at most this many rows per CTA load 32-row boxes
 *  PIPER_OPT_T_GREEDY     [0]  rows-on-N: how an expert's rows are cut into chunks of at most 256: 0 = equal chunks
 *                              (a multiple of 16 rows each), 1 = 256-row chunks and a short last one (measured slower: the
 *                              short chunk streams a whole weight slice for a few rows)
 *  PIPER_OPT_T_DUAL       [0]  rows-on-N plain-store kernels (F_GEMM2, DGRAD2): 1 = a tile takes two row chunks of an
 *                              expert through one pass over the weights (both accumulators); measured slower
 *  PIPER_OPT_WGRAD_STORE_WARP [2] CTA-pair wgrad with bf16 dW: 1 = one 128-row bulk store per 64-column chunk, issued by a
 *                              store warp from blocks the four epilogue warps stage side by side; 0 = one 32-row store
 *                              per epilogue warp; 2 = store warp for long, even groups (>= 512 rows per expert expected
 *                              and real, no expert above twice the mean: the kernel looks at offsets)
 *  PIPER_OPT_MOVE_ITEMS   [8]  row movers: a token's row is split by columns so that about this many work items exist per
 *                              resident warp (1..64)
 *  PIPER_OPT_MOVE_CAP     [16] row movers: at most this many blocks per SM of the lane (1..64)
 *  PIPER_OPT_TC_PROFILE   [0]  1 = the tcgen05 kernels record wait-cycle counters (piper_debug_tc_counters)
 *  PIPER_OPT_FUSED_GATHER [0]  chunk calls on tcgen05 layers (N2 fusion): 0 = the GEMMs read the packed buffers xp / d_o;
 *                              1 = F_GEMM1 and the gate|up wgrad gather the rows of x themselves, no pack kernel runs;
 *                              2 = also DGRAD1 gathers the rows of dY and applies the gate in its fp32 epilogue
 * Returns PIPER_ERR_INVALID for unknown options / values, PIPER_ERR_UNSUPPORTED when the layer cannot run the
 * variant (e.g. fp32 dW without the CTA-pair wgrad). */
#define PIPER_OPT_TC_ROWS_ON_N 0
#define PIPER_OPT_TC_2CTA 1
#define PIPER_OPT_T_SMALL_ROWS 2
#define PIPER_OPT_T_GREEDY 3
#define PIPER_OPT_TC_PROFILE 4
#define PIPER_OPT_FUSED_GATHER 5
#define PIPER_OPT_T_DUAL 6
#define PIPER_OPT_WGRAD_STORE_WARP 7
#define PIPER_OPT_MOVE_ITEMS 8
#define PIPER_OPT_MOVE_CAP 9
int piper_set_option(piper_ctx* ctx, int option, int value);
/* 1 when the whole-chunk calls of this context run the fused-gather GEMMs (PIPER_OPT_FUSED_GATHER on
 * a layer whose GEMMs are the rows-on-N + CTA-pair tcgen05 kernels): the forward chunk then launches no pack kernel and
 * does not write xp (piper_dispatch_pack / piper_run_task(F_PACK) produce the all-to-all payload); with the option at 2
 * the backward chunk's DGRAD1 applies the gate in fp32 after the GEMM instead of reading the bf16-rounded gate * dY.
 * 0 otherwise. */
int piper_chunk_gathers(const piper_ctx* ctx);
int piper_get_option(const piper_ctx* ctx, int option, int* value);
/* Rows the row buffers must hold: T*min(k,E_loc) + E_loc*(row_align-1). */
int64_t piper_a_cap(const piper_moe_desc* desc);

/* F1 route_topk (SURVEY.md §8a F1, §8c Definition 1; BASELINE.json:north_star part 1).
 * logits [T,E] fp32 -> topk_idx [T,k] (k largest, ties to the lowest expert index, listed by
 * descending logit), gates [T,k] fp32 (desc.gate_mode), counts_global [E] (selections per expert =
 * the split sizes an all-to-all would announce). */
int piper_route_topk(piper_ctx* ctx, const float* logits, int32_t* topk_idx, float* gates, int32_t* counts_global,
                     void* stream);

/* F2 + F3 dispatch_pack (SURVEY.md §8a F2/F3, §8c Definition 2; north_star part 2).
 * counts [E_loc]; offsets [E_loc+1] = exclusive scan of counts rounded up to row_align;
 * row_of [T,k] = destination row of each assignment (stable by token), -1 if its expert is not local;
 * src_of [A_cap] = flat assignment id t*k+j of each row, -1 for pad rows and for every row >=
 * offsets[E_loc]; gate_rows [A_cap] fp32; xp [A_cap,d] = x rows gathered per expert (bit-exact copies;
 * pad rows zero).  x [T,d]. */
int piper_dispatch_pack(piper_ctx* ctx, const void* x, const int32_t* topk_idx, const float* gates, int32_t* counts,
                        int32_t* offsets, int32_t* row_of, int32_t* src_of, float* gate_rows, void* xp, void* stream);

/* F2 without a context, a workspace or any allocation: the permutation half of piper_dispatch_pack (same kernels, same
 * outputs: counts [E_loc], offsets [E_loc+1], row_of [T,k], src_of [A_cap], gate_rows [A_cap], A_cap = piper_a_cap(desc); only
 * T, k, E, e_lo, E_loc, row_align of `desc` are read) for callers that cannot call cudaMalloc (CUDA graph capture, serving loops,
 * harnesses that forbid it).  The call allocates nothing and needs no piper_create: its only scratch, the chunk histograms
 * (ceil(T*k/1024) * E_loc int32), lives in a static device array of piper_static_scratch_bytes() = 256 KiB that every GPU
 * which loads the library holds until the process exits.  The kernels run on the CURRENT device, on `stream`; all pointers
 * are device pointers, 16-byte aligned.  Errors: PIPER_ERR_WORKSPACE when the histograms exceed the static array (use
 * piper_dispatch_pack with a context then), PIPER_ERR_INVALID for a bad description or pointer, PIPER_ERR_UNSUPPORTED for
 * E_loc > 4095, PIPER_ERR_CUDA; piper_static_last_error() gives the calling thread's message of the last failure.
 * Every call on a device shares the one array: calls that may overlap on the GPU (different streams without an
 * ordering, other threads or processes sharing the context) RACE on it; order them on one stream or with events.  The
 * array keeps the previous call's contents; nothing in it has to start at zero (every entry read is written by the same
 * call first). */
int piper_dispatch_plan_static(const piper_moe_desc* desc, const int32_t* topk_idx, const float* gates, int32_t* counts,
                               int32_t* offsets, int32_t* row_of, int32_t* src_of, float* gate_rows, void* stream);
size_t piper_static_scratch_bytes(void);
const char* piper_static_last_error(void);

/* F4 expert_ffn_fwd (SURVEY.md §8a F4, §8c Definition 3; north_star part 3).  Per row r of local
 * expert e: g = xp[r] W_gate[e], u = xp[r] W_up[e], h = silu(g)*u, o[r] = h W_down[e].
 * w_gate, w_up [E_loc,d,I]; w_down [E_loc,I,d].  g_save, u_save, h_save [A_cap,I] are opaque scratch
 * handed to piper_expert_ffn_bwd; o [A_cap,d] is the unscaled expert output. */
int piper_expert_ffn_fwd(piper_ctx* ctx, const void* xp, const int32_t* offsets, const void* w_gate, const void* w_up,
                         const void* w_down, void* g_save, void* u_save, void* h_save, void* o, void* stream);
/* Shared expert (reading c-11): the same FFN as one group over all T rows of x, intermediate
 * I_shared.  ws_gate, ws_up [d,I_shared]; ws_down [I_shared,d]; saves [T,I_shared]; s [T,d]. */
int piper_shared_ffn_fwd(piper_ctx* ctx, const void* x, const void* ws_gate, const void* ws_up, const void* ws_down,
                         void* g_save, void* u_save, void* h_save, void* s, void* stream);

/* F5 combine (SURVEY.md §8a F5, §8c Definition 4; north_star part 4).
 * y[t] = sum_{j: row_of[t,j] >= 0} gates[t,j] * o[row_of[t,j]]  (+ s[t] if s != NULL). */
int piper_combine(piper_ctx* ctx, const void* o, const int32_t* row_of, const float* gates, const void* s, void* y,
                  void* stream);

/* B1 combine_bwd (SURVEY.md §8a B1, §8c Definition 5).  d_o[r] = gates[src_of[r]] * dy[token(r)] for
 * every non-pad row below offsets[E_loc] (pad rows zero); dgates[t,j] = <dy[t], o[row_of[t,j]]>, 0 for
 * non-local slots.  d_o is opaque scratch handed to piper_expert_ffn_bwd. */
int piper_combine_bwd(piper_ctx* ctx, const void* dy, const void* o, const int32_t* src_of, const int32_t* row_of,
                      const float* gates, const int32_t* offsets, void* d_o, float* dgates, void* stream);

/* B2-B4 expert_ffn_bwd (SURVEY.md §8a B2/B3/B4, §8c Definition 5; north_star part 3 "dgrad and
 * wgrad").  dh = d_o W_down^T; dg = dh*u*silu'(g); du = dh*silu(g); dxp = dg W_gate^T + du W_up^T;
 * dw_down[e] = h^T d_o, dw_gate[e] = xp^T dg, dw_up[e] = xp^T du summed over the expert's rows
 * (exact zeros for empty experts).  dg, du [A_cap,I] are opaque scratch.  accumulate = 1 adds the
 * sums into dw_* instead of overwriting them (reading c-17: main-grad style; Piper reduces after every backward,
 * PAPER.md:384): needs dw_dtype = F32 on a BF16 layer (the whole ragged-K sum is accumulated in fp32 in TMEM and
 * added to dW by a bulk tensor reduction), PIPER_ERR_UNSUPPORTED otherwise. */
int piper_expert_ffn_bwd(piper_ctx* ctx, const void* d_o, const void* xp, const void* g_save, const void* u_save,
                         const void* h_save, const int32_t* offsets, const void* w_gate, const void* w_up,
                         const void* w_down, void* dg, void* du, void* dxp, void* dw_gate, void* dw_up, void* dw_down,
                         int accumulate, void* stream);
/* Shared expert backward: one group of T rows, d_o = dy, xp = x; dgs, dus [T,I_shared] scratch;
 * dxs [T,d]. */
int piper_shared_ffn_bwd(piper_ctx* ctx, const void* dy, const void* x, const void* g_save, const void* u_save,
                         const void* h_save, const void* ws_gate, const void* ws_up, const void* ws_down, void* dgs,
                         void* dus, void* dxs, void* dws_gate, void* dws_up, void* dws_down, int accumulate,
                         void* stream);

/* B5 dispatch_unpack.  dx[t] = sum_{j local} dxp[row_of[t,j]] (+ dx_shared[t]). */
int piper_dispatch_unpack(piper_ctx* ctx, const void* dxp, const int32_t* row_of, const void* dx_shared, void* dx,
                          void* stream);

/* B6 route_bwd (gate-normalisation backward of Definition 5).
 * gate modes 0/1: dz_sel [T,k] (gradient w.r.t. the k selected logits); mode 2: dz_sel is [T,E]. */
int piper_route_bwd(piper_ctx* ctx, const float* logits, const int32_t* topk_idx, const float* gates,
                    const float* dgates, float* dz_sel, void* stream);

/* N1 router GEMMs (Listing 1 `self.router(x)`): the step before F1 and after B6.
 * piper_router_fwd: logits [T,E] fp32 = x [T,d] w_r [d,E] (+ bias [E] fp32, nullable; reading c-5: the bias is part of
 * the logits).  bf16 layers: tcgen05 GEMM, products of bf16 values are exact and the sum is accumulated in fp32, so the
 * logits differ from the exactly rounded sum by fp32 accumulation error only (~1e-6 relative): top-k selections on them
 * agree with the oracle's except on rows whose k-th / (k+1)-th logit gap is below that error (reading c-18).
 * piper_router_bwd: dz = dz_sel [T,k] scattered to the selected experts (gate modes 0, 1) or the dense [T,E] rows of
 * mode 2; dw_r [d,E] fp32 = x^T dz (overwritten); dx_router [T,d] (activation dtype) = dz w_r^T, the router's part of
 * dX (piper_dispatch_unpack_router adds it).  dz_scratch: T*E*4 bytes of caller-owned scratch.  On bf16 layers dz is
 * split into two bf16 terms (relative error 2^-17) for the tensor cores. */
int piper_router_fwd(piper_ctx* ctx, const void* x, const void* w_r, const float* bias, float* logits, void* stream);
int piper_router_bwd(piper_ctx* ctx, const void* x, const void* w_r, const int32_t* topk_idx, const float* dz_sel,
                     void* dz_scratch, float* dw_r, void* dx_router, void* stream);
/* B5 with the router's term: dx[t] = sum_{j local} dxp[row_of[t,j]] (+ dx_shared[t]) (+ dx_router[t]), summed in fp32 in
 * that order and rounded once. */
int piper_dispatch_unpack_router(piper_ctx* ctx, const void* dxp, const int32_t* row_of, const void* dx_shared,
                                 const void* dx_router, void* dx, void* stream);

/* N4 expert parallelism over peer memory (`Shard` inserts an all-to-all before and after
 * the expert Chunk).  n_ranks GPUs, T tokens each; rank r owns the experts [r * E / n_ranks, (r + 1) * E / n_ranks) = the
 * context's [e_lo, e_lo + E_loc).  The pack / combine row movers address the owners' buffers directly through peer pointers
 * (NVLink / NVSwitch peer memory) instead of filling a send buffer for an all-to-all-v.  Protocol per microbatch:
 *   piper_route_topk on every rank; the ranks all-gather counts_global -> all_counts [n_ranks, E] (the caller's collective);
 *   piper_ep_plan      every rank derives, without further communication, its own experts' counts [E_loc] (totals over the
 *                      ranks) and offsets [E_loc + 1] (aligned exclusive scan) and send_base [E] = the row, in the owner's
 *                      buffer, where its own rows of expert e start (rows of an expert are ordered by source rank, then token:
 *                      by global token id rank * T + t, exactly the buffer piper_dispatch_pack builds over the concatenated
 *                      tokens);
 *   piper_ep_dispatch  stable ranks of this rank's assignments, then peer stores of the token rows, of the global assignment
 *                      ids ((rank * T + t) * k + j) and of the gates into the owners' xp / src_of / gate_rows; dest_row [T,k]
 *                      keeps the row of each assignment in its owner's buffer;
 *   piper_ep_finish_recv (owner) zero pad rows of a received row buffer, src_of = -1 on pads and beyond offsets[E_loc];
 *   the owner runs piper_expert_ffn_fwd / _bwd on what it received, through a context created with T * n_ranks tokens;
 *   piper_ep_combine   y[t] = sum_j gates[t,j] * peer_o[owner(j)][dest_row[t,j]] (+ s[t]);
 *   piper_ep_dispatch_bwd  peer_d_o[owner][row] = gates[t,j] * dy[t], dgates[t,j] = <dy[t], peer_o[owner][row]>;
 *   piper_ep_unpack    dx[t] = sum_j peer_dxp[owner(j)][dest_row[t,j]] (+ dx_shared[t]).
 * peer_* are DEVICE arrays of n_ranks device pointers (entry r = rank r's buffer, mapped into this GPU's address space: CUDA
 * IPC, cudaDeviceEnablePeerAccess or symmetric memory; with n_ranks = 1, or all ranks on one GPU, plain pointers).  Row buffers
 * of an owner hold piper_ep_a_cap() rows.  No kernel waits on another rank's kernel: the steps are ordered by the caller's
 * streams and collectives (a barrier between dispatch and the owners' FFN, and before combine).  Needs E % n_ranks == 0 and
 * e_lo = rank * E_loc; one dispatch of a context at a time. */
int64_t piper_ep_a_cap(const piper_moe_desc* desc, int n_ranks);
int piper_ep_plan(piper_ctx* ctx, const int32_t* all_counts, int rank, int n_ranks, int32_t* counts, int32_t* offsets,
                  int32_t* send_base, void* stream);
/* The same plan on the host, from HOST arrays (no GPU): for callers that size messages on the host, and for CPU tests. */
int piper_ep_plan_host(const int32_t* all_counts, int32_t E, int32_t n_ranks, int32_t rank, int32_t row_align, int32_t* counts,
                       int32_t* offsets, int32_t* send_base);
int piper_ep_dispatch(piper_ctx* ctx, const void* x, const int32_t* topk_idx, const float* gates, const int32_t* send_base,
                      int rank, int n_ranks, void* const* peer_xp, int32_t* const* peer_src_of, float* const* peer_gate_rows,
                      int32_t* dest_row, void* stream);
int piper_ep_finish_recv(piper_ctx* ctx, const int32_t* counts, const int32_t* offsets, int n_ranks, int32_t* src_of,
                         float* gate_rows, void* rows, void* stream);
int piper_ep_combine(piper_ctx* ctx, void* const* peer_o, const int32_t* topk_idx, const int32_t* dest_row, const float* gates,
                     const void* s, void* y, void* stream);
int piper_ep_dispatch_bwd(piper_ctx* ctx, const void* dy, const int32_t* topk_idx, const int32_t* dest_row, const float* gates,
                          void* const* peer_o, void* const* peer_d_o, float* dgates, void* stream);
int piper_ep_unpack(piper_ctx* ctx, void* const* peer_dxp, const int32_t* topk_idx, const int32_t* dest_row,
                    const void* dx_shared, void* dx, void* stream);

/* Every pointer of one microbatch (inputs, outputs and the scratch between forward and backward). */
typedef struct {
    const float* logits;                         /* [T,E]: input; an OUTPUT of the forward chunk when w_r != NULL */
    const void *x, *dy;                          /* [T,d]                                           */
    const void *w_gate, *w_up, *w_down;          /* routed experts                                  */
    const void *ws_gate, *ws_up, *ws_down;       /* shared expert (NULL when I_shared = 0)          */
    int32_t *topk_idx, *counts_global, *counts, *offsets, *row_of, *src_of;
    float *gates, *gate_rows, *dgates, *dz_sel;
    void *xp, *g_save, *u_save, *h_save, *o;     /* routed activations [A_cap, d or I]              */
    void *gs_save, *us_save, *hs_save, *s;       /* shared-expert activations [T, I_shared or d]    */
    void* y;                                     /* [T,d]                                           */
    void *d_o, *dg, *du, *dxp, *dgs, *dus, *dxs, *dx; /* backward activations                      */
    void *dw_gate, *dw_up, *dw_down, *dws_gate, *dws_up, *dws_down;
    /* N1 (optional, all NULL = the boundary starts at the logits): with w_r != NULL the forward chunk first computes
     * logits = x w_r + router_bias, and the backward chunk adds the router's dW_r and its term of dX */
    const void* w_r;           /* [d,E]                                                             */
    const float* router_bias;  /* [E] or NULL                                                       */
    float* dw_r;               /* [d,E] fp32                                                        */
    void *dx_router, *dz_scratch; /* [T,d]; T*E*4 bytes                                             */
} piper_chunk_args;

/* Whole forward chunk F1..F5 (+ shared expert) / backward chunk B1..B6 on one stream, all SMs:
 * the serial baseline of step P. */
int piper_run_chunk_fwd(piper_ctx* ctx, const piper_chunk_args* a, void* stream);
int piper_run_chunk_bwd(piper_ctx* ctx, const piper_chunk_args* a, void* stream);
/* The backward chunk split into the paper's two passes (PASS = Bi, Bw; Fig. 3; SURVEY.md
 * §8f N3): _input runs everything the upstream layer waits for (combine_bwd, dgrad-1, dgrad-2, the shared expert's
 * dgrads, unpack, route_bwd -> dX, dgates, dz_sel), _weight the weight gradients (routed and shared wgrad -> dW_*), which
 * a schedule may delay to fill bubbles.  _weight needs the scratch _input left in `a` (d_o / dg / du / dgs / dus).
 * _input followed by _weight is bit-identical to piper_run_chunk_bwd. */
int piper_run_chunk_bwd_input(piper_ctx* ctx, const piper_chunk_args* a, void* stream);
int piper_run_chunk_bwd_weight(piper_ctx* ctx, const piper_chunk_args* a, void* stream);

/* P run_chunk_pair (SURVEY.md §8a P, §8c c-sched; north_star part 5).  Enqueues the forward chunk of
 * `fwd_mb` and the backward chunk of `bwd_mb` as the 14-task DAG of SURVEY.md §8c on two logical
 * streams: GEMM tasks on a partition of `sm_gemm` SMs, pack/combine-side tasks on a partition of
 * `sm_comm` SMs.  Task order = Piper's list scheduling (reading c-21); a task waits
 * on an event only for a dependency that ran on the other stream and records one only when a
 * consumer runs on the other stream.  Both partitions fork from and join
 * into `stream`.  sm_gemm + sm_comm must not exceed the device's SM count; each must be a positive
 * multiple of 8 except that sm_gemm may take the remainder.  Results are bit-identical to
 * piper_run_chunk_fwd + piper_run_chunk_bwd. */
int piper_run_chunk_pair(piper_ctx* ctx, const piper_chunk_args* fwd_mb, const piper_chunk_args* bwd_mb, int sm_gemm,
                         int sm_comm, void* stream);
/* Creates the SM partitions (green contexts), their streams and the schedule for a split ahead of time, so that
 * piper_run_chunk_pair with the same split and policy creates nothing (and can be captured in a CUDA graph).  The last
 * prepared split is kept; another split, or another partition policy, releases it.  PIPER_ERR_UNSUPPORTED when
 * PIPER_PART_EXCLUSIVE cannot be honoured (no green contexts, or the driver cannot split off these SM counts). */
int piper_pair_prepare(piper_ctx* ctx, int sm_gemm, int sm_comm);
/* Which pass of microbatch B the pair overlaps with the forward chunk (host state, default PIPER_PASS_B):
 * PIPER_PASS_BI runs F || Bi (Fig. 3b) and leaves the weight gradients to a later
 * piper_run_chunk_bwd_weight(bwd_mb). */
#define PIPER_PASS_B 0
#define PIPER_PASS_BI 1
int piper_set_pair_bwd_pass(piper_ctx* ctx, int pass);

/* Policy of piper_run_chunk_pair (host state of `ctx`).  Default: PIPER_ORDER_PROFILE on PIPER_PART_SHARED, the
 * combination that does not lose against the serial chunks on C5 (bench.py reports every combination; the paper's
 * own policy, PIPER_ORDER_LIST, on the disjoint partitions BASELINE.json sweeps, PIPER_PART_EXCLUSIVE, measures
 * 1.1-1.25 x serial: DESIGN.md section 5.4).
 *  order     PIPER_ORDER_LIST    Piper's list scheduling, ready task with the most descendants first.
 *            PIPER_ORDER_PROFILE profile-guided (PAPER.md:273, 420 name it as the way past the simple policy): the
 *                                static two-stream schedule with the smallest simulated makespan, found by exhaustive
 *                                search over per-stream sequences (piper_schedule_search) under task durations
 *                                `task_ms` [14] (PIPER_TASK_* order, milliseconds on the whole device; the library
 *                                scales them to the partition sizes) or, when task_ms is NULL, under the library's
 *                                own estimate from the algorithmic FLOPs and bytes of the descriptor.
 *  partition PIPER_PART_EXCLUSIVE  disjoint SM sets (green contexts; sm_gemm + sm_comm <= SM count; sm_comm a multiple
 *                                  of 8, sm_gemm a multiple of 8 or the whole remainder).  When the driver cannot
 *                                  provide them the call fails with PIPER_ERR_UNSUPPORTED: no silent fallback.
 *            PIPER_PART_SHARED     two plain streams, every grid bounded to its side's SM count worth of CTAs; the
 *                                  sides may overlap (sm_gemm + sm_comm may exceed the SM count): pack/combine CTAs
 *                                  become co-resident with the persistent GEMM CTAs, as in the paper, which leaves SM
 *                                  allocation to the GPU.
 *            PIPER_PART_CHUNK_STREAMS  one plain stream per chunk (forward chunk / backward chunk, each in its serial
 *                                  task order, `order` and the SM counts are not used), every grid sized for the whole
 *                                  device: SM allocation is left entirely to the GPU.  The chunks'
 *                                  GEMM kernels follow one another SM by SM as clusters retire and the row movers
 *                                  run beside them.
 * Either way the results stay bit-identical to the serial chunks.  Returns PIPER_ERR_INVALID on unknown values. */
#define PIPER_ORDER_LIST 0
#define PIPER_ORDER_PROFILE 1
#define PIPER_PART_CHUNK_STREAMS 2
#define PIPER_PART_EXCLUSIVE 0
#define PIPER_PART_SHARED 1
int piper_set_pair_policy(piper_ctx* ctx, int order, int partition, const float* task_ms);
/* The pick sequence (PIPER_TASK_* ids, caller tasks included; n <= 18 written to order[18]) the current policy yields
 * for a split. */
int piper_pair_order(piper_ctx* ctx, int sm_gemm, int sm_comm, int32_t* order, int32_t* n);

/* N3 (Fig. 3b, Listing 1, "Chunk.exec"): the rest of the overlapped
 * block - attention forward before the MoE chunk of microbatch A, attention backward after the MoE chunk of microbatch
 * B - as CALLER TASKS of the pair.  A caller task is an opaque function that enqueues its work on the stream it is given
 * (it must not synchronise; sm_count is its side's SM budget, for kernels that bound their own grids); the pair puts it into
 * the task DAG of piper_run_chunk_pair and schedules it with the library's tasks (list order or profile order, the
 * event rule of PAPER.md:279-286):
 *   PIPER_SLOT_F_PRE   produces x / logits of the forward microbatch:  before F.route, F.pack, F.shared
 *   PIPER_SLOT_F_POST  consumes y:                                     after F.combine
 *   PIPER_SLOT_B_PRE   produces dY of the backward microbatch:         before B.cgrad, B.shared
 *   PIPER_SLOT_B_POST  consumes dX / dz_sel (and the router's dW_r):   after B.unpack, B.route_bwd
 * side: 0 = the pack/combine ("communication-side") stream, 1 = the GEMM stream.  est_ms: duration on the whole device
 * for PIPER_ORDER_PROFILE.  fn = NULL clears the slot.  piper_run_chunk_fwd / _bwd do not run caller tasks (the caller
 * simply enqueues them around those calls).  A non-zero return of fn aborts the pair call with PIPER_ERR_INVALID.
 * Host state of `ctx`; `user` must stay valid while the slot is set. */
typedef int (*piper_caller_task_fn)(void* user, void* cuda_stream, int sm_count);
#define PIPER_SLOT_F_PRE 0
#define PIPER_SLOT_F_POST 1
#define PIPER_SLOT_B_PRE 2
#define PIPER_SLOT_B_POST 3
#define PIPER_TASK_CALLER_F_PRE 14 /* ids of the caller tasks in piper_pair_order: 14 + slot */
int piper_pair_set_caller_task(piper_ctx* ctx, int slot, piper_caller_task_fn fn, void* user, float est_ms, int side);
/* One task of the pair DAG (SURVEY.md §8c c-sched numbering) on `stream` with all SMs: the unit that
 * piper_run_chunk_fwd / _bwd / _pair enqueue, exposed so that each step can be timed on its own
 * (bench.py's roofline block).  F_* tasks read `a` as the forward microbatch, B_* as the backward one. */
#define PIPER_TASK_F_ROUTE 0
#define PIPER_TASK_F_SCAN 1
#define PIPER_TASK_F_PACK 2
#define PIPER_TASK_F_GEMM1 3
#define PIPER_TASK_F_GEMM2 4
#define PIPER_TASK_F_SHARED 5
#define PIPER_TASK_F_COMBINE 6
#define PIPER_TASK_B_CGRAD 7
#define PIPER_TASK_B_DGRAD1 8
#define PIPER_TASK_B_DGRAD2 9
#define PIPER_TASK_B_WGRAD 10
#define PIPER_TASK_B_SHARED 11
#define PIPER_TASK_B_UNPACK 12
#define PIPER_TASK_B_ROUTE_BWD 13
int piper_run_task(piper_ctx* ctx, int task, const piper_chunk_args* a, void* stream);

/* accumulate flag of the wgrad inside piper_run_chunk_bwd / piper_run_chunk_pair / piper_run_task (host state of
 * `ctx`, default 0); PIPER_ERR_UNSUPPORTED unless dw_dtype = F32. */
int piper_set_wgrad_accumulate(piper_ctx* ctx, int accumulate);

/* Intra-chunk overlap of piper_run_chunk_fwd / piper_run_chunk_bwd (host state of `ctx`, default 0 = every task on the
 * caller's stream, one after the other: the serial baseline the pair is compared with).  on = 1: the forward chunk runs
 * route / scan / pack on a side stream of the library beside the shared expert's GEMMs (layers with a shared expert),
 * the backward chunk runs unpack and route_bwd on the side stream beside the routed wgrad (the shared expert's backward
 * moves in front of it).  The side stream forks from and joins into the caller's stream inside the call; results are
 * bit-identical.  Returns PIPER_ERR_INVALID for other values, PIPER_ERR_CUDA if the stream cannot be created. */
int piper_set_chunk_overlap(piper_ctx* ctx, int on);

/* How the last piper_run_chunk_pair partitioned the SMs: 1 = green contexts (PIPER_PART_EXCLUSIVE), 2 = bounded
 * persistent grids on two plain streams (PIPER_PART_SHARED), 3 = one stream per chunk (PIPER_PART_CHUNK_STREAMS),
 * 0 = never called. */
int piper_pair_partition_mode(const piper_ctx* ctx);

/* Host-only list scheduler used by piper_run_chunk_pair (reading c-21),
 * exposed so it can be tested without a GPU.  n tasks, edges [n_edges][2] (src,dst), stream_of[n],
 * prio[n] (lower first on ties) -> order[n] (pick sequence), waits [<= n_edges][2] (producer,
 * consumer) for every direct cross-stream edge, *n_waits, records[n] (1 iff the task records an
 * event).  Returns PIPER_ERR_INVALID on a cycle or a bad edge. */
int piper_list_schedule(int32_t n, int32_t n_edges, const int32_t* edges, const int32_t* stream_of, const int32_t* prio,
                        int32_t* order, int32_t* waits, int32_t* n_waits, int32_t* records);
/* Profile-guided counterpart (PIPER_ORDER_PROFILE): exact search (branch and bound with a dominance rule) of the static
 * two-stream schedule (n <= 18, stream_of in {0,1}) with the smallest makespan under durations dur[n], simulated with
 * the event rule of PAPER.md:279-286; ties go to the first schedule in the search order (ready tasks by ascending id),
 * so the result is a pure function of the inputs.  The search visits at most 2^21 states (the pair DAG with its caller
 * tasks needs ~10^3); on a DAG that needs more, the best schedule found within the budget is returned (always valid,
 * then not proven optimal).  Outputs as piper_list_schedule plus *makespan (nullable), in the unit of dur. */
int piper_schedule_search(int32_t n, int32_t n_edges, const int32_t* edges, const int32_t* stream_of, const float* dur,
                          int32_t* order, int32_t* waits, int32_t* n_waits, int32_t* records, float* makespan);

#ifdef __cplusplus
}
#endif
#endif /* PIPER_H_ */
