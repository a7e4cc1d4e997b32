// piper_internal.cuh — shared declarations of the CUDA library (not part of the C-ABI).
// The oracle (oracle/) includes nothing from this directory and this directory nothing from it.
#pragma once
#include <cuda.h>  // CUtensorMap type and enums only; the driver is reached through cudaGetDriverEntryPoint
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "piper.h"

namespace piper {

constexpr int kMaxK = 8;          // top-k bound (register arrays in route / combine kernels)
constexpr int kMaxE = 512;        // expert bound of the router kernel (16 values per lane)
constexpr int kScanChunk = 1024;  // assignments per block of the histogram / rank kernels
constexpr int kMaxEvents = 24;    // one per pair task (14 + 4 caller tasks) + fork/join

// Where a task's kernels run: stream + the number of SMs its persistent grids may occupy.
struct Lane {
    cudaStream_t stream;
    int sms;
};

struct GreenPartition;  // chunk.cu

// Tile counters of the dynamically scheduled tcgen05 kernels: one {next tile, clusters done} pair per stream (kernels
// of one stream are ordered, and the last cluster of a launch re-arms the pair), so launches that run concurrently on
// different streams never share one.  A stream under capture is keyed by (capture id, stream): a captured graph
// keeps its own pair wherever it is replayed.
constexpr int kSchedSlots = 64;
struct SchedSlot {
    cudaStream_t stream;
    unsigned long long capture_id;  // 0 = eager
    unsigned long long last_use;
    bool used;
};
// occupancy of a cluster kernel on a lane, queried once per (kernel, stream, SM count)
constexpr int kClusterCache = 64;
struct ClusterCacheEntry {
    const void* fn;
    cudaStream_t stream;
    int sms, n;
};
// encoded tensor maps, keyed by what cuTensorMapEncodeTiled was given (the same ~40 maps are needed every step)
constexpr int kMapCache = 512;
struct MapCacheEntry {
    const void* base;
    long long inner, rows, groups;
    int box_inner, box_rows, kind;  // kind: 0 unused, 1 bf16, 2 fp32, 3 bf16 gather rows
    CUtensorMap map;
};

}  // namespace piper

struct piper_ctx {
    piper_moe_desc D;
    int device;
    int num_sms;
    char* ws;
    size_t ws_bytes;
    int n_chunks;            // ceil(T*k / kScanChunk)
    int32_t* chunk_counts;   // [kSchedSlots][n_chunks][E_loc]  per-chunk local-expert histograms, one set per stream slot
    size_t chunk_counts_stride;  // int32 elements between two slots' histograms
    int32_t* ep_scratch;     // [n_chunks][E] chunk histograms over all experts (N4 dispatch)
    int32_t* shared_offsets; // [2] = {0, T}: the shared expert as one group
    int64_t launches;
    int pair_mode;
    int wgrad_accumulate;        // piper_set_wgrad_accumulate: the chunk calls' wgrad adds into dW
    int chunk_overlap;           // piper_set_chunk_overlap: the chunk calls run their row movers on a side stream
    cudaStream_t side_stream;    // created on first use
    int pair_order, pair_part;   // piper_set_pair_policy
    int pair_have_ms;
    void* pair_plan;             // cached schedule of the pair for (plan_sm_gemm, plan_sm_comm)
    int plan_sm_gemm, plan_sm_comm;
    float pair_task_ms[14];      // caller's task durations on the whole device (PIPER_ORDER_PROFILE)
    piper_caller_task_fn caller_fn[4];  // N3: caller tasks of the pair (piper_pair_set_caller_task), by slot
    void* caller_user[4];
    float caller_ms[4];
    int caller_side[4];
    char err[256];
    void* encode_tiled;      // cuTensorMapEncodeTiled, resolved at create time
    piper::GreenPartition* green;
    char* tc_scratch;        // debug counters + tile counters of the persistent tcgen05 kernels (gemm_tc.cu)
    int tc_next_slot;        // round-robin debug-counter slot in tc_scratch
    int tc_two_cta;          // CTA-pair (cta_group::2) kernels: 0 never, 1 always, 2 by expected group length
    int tc_rows_on_n;        // rows-on-N kernels for fwd / dgrad (PIPER_OPT_TC_ROWS_ON_N, default on)
    int tc_small_rows, tc_greedy;  // PIPER_OPT_T_SMALL_ROWS / PIPER_OPT_T_GREEDY: row chunking of the rows-on-N kernels
    int tc_dual;             // PIPER_OPT_T_DUAL: two-chunk tiles in the plain-store rows-on-N kernels
    int tc_store_warp;       // PIPER_OPT_WGRAD_STORE_WARP: 0 / 1 / 2 = by expected group length
    int tc_prof;             // PIPER_OPT_TC_PROFILE: the tcgen05 kernels record wait-cycle counters in tc_scratch
    int fused_gather;        // PIPER_OPT_FUSED_GATHER: chunk calls let the GEMMs gather x / dY rows (N2)
    int pair_bwd_pass;       // piper_set_pair_bwd_pass
    int move_items, move_cap;  // PIPER_OPT_MOVE_ITEMS / PIPER_OPT_MOVE_CAP: work items per resident warp / blocks per SM of the row movers
    unsigned long long sched_clock;
    piper::SchedSlot sched_slots[piper::kSchedSlots];
    piper::ClusterCacheEntry cluster_cache[piper::kClusterCache];
    int cluster_cache_used;
    piper::MapCacheEntry* map_cache;  // [kMapCache], host
    cudaEvent_t events[piper::kMaxEvents];
};

namespace piper {

inline int cuda_fail(piper_ctx* c, cudaError_t e, const char* what) {
    snprintf(c->err, sizeof(c->err), "%s: %s", what, cudaGetErrorString(e));
    return PIPER_ERR_CUDA;
}
#define PIPER_CUDA(ctx, call)                                            \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return piper::cuda_fail(ctx, e__, #call); \
    } while (0)
// after a kernel launch
#define PIPER_LAUNCHED(ctx, name)                                          \
    do {                                                                   \
        (ctx)->launches += 1;                                              \
        cudaError_t e__ = cudaGetLastError();                              \
        if (e__ != cudaSuccess) return piper::cuda_fail(ctx, e__, name);   \
    } while (0)

inline bool aligned16(const void* p) { return p != nullptr && (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline size_t esize(int dtype) { return dtype == PIPER_DTYPE_BF16 ? 2 : 4; }
inline int cdiv(int a, int b) { return (a + b - 1) / b; }

// ---- launchers implemented per translation unit -------------------------------------------------
// route.cu
int launch_route_topk(piper_ctx*, Lane, const float* logits, int32_t* topk_idx, float* gates, int32_t* counts_global);
int launch_route_bwd(piper_ctx*, Lane, const float* logits, const int32_t* topk_idx, const float* gates,
                     const float* dgates, float* dz);
// permute.cu
int launch_scan_rank(piper_ctx*, Lane, const int32_t* topk_idx, const float* gates, int32_t* counts, int32_t* offsets,
                     int32_t* row_of, int32_t* src_of, float* gate_rows);
int launch_pack(piper_ctx*, Lane, const void* x, const int32_t* offsets, const int32_t* row_of, const int32_t* src_of,
                void* xp);
int launch_combine(piper_ctx*, Lane, const void* o, const int32_t* row_of, const float* gates, const void* s,
                   const void* s2, void* y, bool weighted);
int launch_combine_bwd(piper_ctx*, Lane, const void* dy, const void* o, const int32_t* src_of, const int32_t* row_of,
                       const float* gates, const int32_t* offsets, void* d_o, float* dgates);

// One grouped SwiGLU FFN problem: `G` groups; group g owns rows [offsets[g], offsets[g+1]) of the row
// buffers and weight slice g.  The shared expert is the same problem with G = 1, offsets = {0, T}.
struct FfnProblem {
    int G, d, I;
    int max_rows;            // host-side bound on offsets[G] (sizes the tensor maps and SIMT grids)
    int max_group_rows;      // host-side bound on the rows of one group
    int exp_rows;            // rows expected under uniform routing (kernel-variant choice only)
    int accumulate;          // wgrad adds into dW (fp32 dW only)
    const int32_t* offsets;  // device, [G+1]
    const int32_t* counts;   // device, [G]: real rows per group (offsets are padded to row_align)
    const void *xp, *w_gate, *w_up, *w_down;
    void *g, *u, *h, *o;                                 // forward outputs
    const void* d_o;                                     // backward inputs / outputs
    void *dg, *du, *dxp, *dw_gate, *dw_up, *dw_down;
    // N2 fusion (routed problem of the chunk calls, tcgen05 rows-on-N + CTA-pair kernels only): when set, the GEMMs
    // gather the rows of x / dY through src_of themselves instead of reading xp / d_o
    const void *gather_x, *gather_dy;
    const int32_t* src_of;    // [max_rows] flat assignment id of each packed row, -1 = pad
    const float* gate_rows;   // [max_rows]
};
// gemm_simt.cu (FP32 ALUs; fp32 or bf16 storage)
// `which`: bit 0 = first GEMM of the pass (fwd1 / dgrad1), bit 1 = second (fwd2 / dgrad2)
int simt_ffn_fwd(piper_ctx*, Lane, const FfnProblem&, int which);
int simt_ffn_dgrad(piper_ctx*, Lane, const FfnProblem&, int which);
int simt_ffn_wgrad(piper_ctx*, Lane, const FfnProblem&);
// gemm_tc.cu (tcgen05 / TMEM / TMA; bf16 storage)
size_t tc_scratch_bytes(const piper_moe_desc*);
int tc_init(piper_ctx*);  // resolves cuTensorMapEncodeTiled, sets kernel attributes
void tc_release(piper_ctx*);
bool tc_supported(const piper_ctx*, const FfnProblem&);
bool tc_wgrad_f32_ok(const piper_ctx*, const FfnProblem&);
bool tc_gather_ok(const piper_ctx*, const FfnProblem&);     // the kernel families that can gather x / dY rows (N2)  // fp32 dW (and accumulate) exist in the CTA-pair wgrad only
int tc_ffn_fwd1(piper_ctx*, Lane, const FfnProblem&);    // G,U,H = swiglu(xp W_gate, xp W_up)
int tc_ffn_fwd2(piper_ctx*, Lane, const FfnProblem&);    // O = H W_down
int tc_ffn_dgrad1(piper_ctx*, Lane, const FfnProblem&);  // dG,dU from dO W_down^T and G,U
int tc_ffn_dgrad2(piper_ctx*, Lane, const FfnProblem&);  // dXp = dG W_gate^T + dU W_up^T
int tc_ffn_wgrad(piper_ctx*, Lane, const FfnProblem&);   // dW_gate, dW_up, dW_down

// dense GEMMs of the router (N1) on the 1-CTA tcgen05 kernel
bool tc_router_supported(const piper_ctx*);
int tc_router_fwd(piper_ctx*, Lane, const void* x, const void* w_r, const float* bias, float* logits);
int tc_router_wgrad(piper_ctx*, Lane, const void* x, const void* dz_hi, const void* dz_lo, float* dw_r);
int tc_router_dgrad(piper_ctx*, Lane, const void* dz_hi, const void* dz_lo, const void* w_r, void* dx_r);
// router.cu
int launch_router_fwd(piper_ctx*, Lane, const void* x, const void* w_r, const float* bias, float* logits);
int launch_router_bwd(piper_ctx*, Lane, const void* x, const void* w_r, const int32_t* topk_idx, const float* dz_sel,
                      void* dz_scratch, float* dw_r, void* dx_router);

// ffn.cu: dispatch between the two GEMM families, task granularity used by the chunk scheduler
int ffn_gemm1(piper_ctx*, Lane, const FfnProblem&);
int ffn_gemm2(piper_ctx*, Lane, const FfnProblem&);
int ffn_dgrad1(piper_ctx*, Lane, const FfnProblem&);
int ffn_dgrad2(piper_ctx*, Lane, const FfnProblem&);
int ffn_wgrad(piper_ctx*, Lane, const FfnProblem&);
FfnProblem routed_problem(const piper_ctx*, const piper_chunk_args*);
FfnProblem shared_problem(const piper_ctx*, const piper_chunk_args*);
// ffn.cu: do the chunk calls of this context let the routed GEMMs gather x / dY rows themselves (N2 fusion)?
bool fused_gather(const piper_ctx*);
// chunk.cu
void pair_release(piper_ctx*);
void pair_plan_release(piper_ctx*);
// api.cu: per-stream scratch of a context (see SchedSlot): the slot of a stream, its scan histograms, its tile counters
int stream_slot(piper_ctx*, cudaStream_t);
int32_t* scan_scratch(piper_ctx*, cudaStream_t);
// gemm_tc.cu: forget what the context cached about a stream that is being destroyed
void tc_forget_stream(piper_ctx*, cudaStream_t);

// ---- small device helpers -----------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ int4 ld_nc16(const void* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
__device__ __forceinline__ void st16(void* p, const int4& v) {
    asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w)
                 : "memory");
}
// bf16x2 <-> float2 (exact widening; RNE narrowing)
__device__ __forceinline__ float2 bf2_to_f2(uint32_t v) {
    return make_float2(__uint_as_float(v << 16), __uint_as_float(v & 0xFFFF0000u));
}
__device__ __forceinline__ uint32_t f2_to_bf2(float lo, float hi) {
    __nv_bfloat162 b = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&b);
}
#endif

}  // namespace piper
