// router.cu — N1 of SURVEY.md §8(f): the router's own GEMMs on the path (Listing 1 `self.router(x)`).
//   forward   z[T,E]   = x[T,d] W_r[d,E] (+ bias[E])          fp32 logits, feeding F1 route_topk
//   backward  dW_r[d,E] = x^T dz ,  dX_r[T,d] = dz W_r^T       dz = dz_sel scattered to the selected experts (modes 0, 1)
//                                                             or the dense rows of mode 2
// bf16 layers: tcgen05 dense GEMMs (gemm_tc.cu, 1-CTA kernel).  x and W_r are bf16, so every product is exact in fp32 and
// the sum is accumulated in fp32 (TMEM).  dz is fp32: it is split into two bf16 tensors hi = bf16(dz), lo = bf16(dz - hi)
// (relative error 2^-17) and both products run into one accumulator.  fp32 layers (C1) and shapes the tensor path does
// not take: FP32-FMA kernels below (no fast-math needed: plain fmaf).
#include "piper_internal.cuh"

namespace piper {
namespace {

template <typename TS> __device__ __forceinline__ float ldv(const TS* p);
template <> __device__ __forceinline__ float ldv<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ldv<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }
template <typename TS> __device__ __forceinline__ void stv(TS* p, float v);
template <> __device__ __forceinline__ void stv<float>(float* p, float v) { *p = v; }
template <> __device__ __forceinline__ void stv<__nv_bfloat16>(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }

// ---- FP32-FMA fallbacks: one warp per output row segment, lanes over the contraction --------------------------------
// z[t,e] = sum_i x[t,i] W[i,e] + bias[e]: block = 4 tokens x 64 experts, x rows staged in shared memory.
template <typename TS>
__global__ void __launch_bounds__(256) router_fwd_simt(const TS* __restrict__ x, const TS* __restrict__ w,
                                                       const float* __restrict__ bias, int T, int d, int E,
                                                       float* __restrict__ z) {
    extern __shared__ float xs[];  // [4][d]
    const int t0 = blockIdx.x * 4;
    for (int i = threadIdx.x; i < 4 * d; i += 256) {
        const int r = i / d, cidx = i - r * d;
        xs[i] = t0 + r < T ? ldv<TS>(x + (size_t)(t0 + r) * d + cidx) : 0.f;
    }
    __syncthreads();
    const int r = threadIdx.x >> 6, e0 = threadIdx.x & 63;
    if (t0 + r >= T) return;
    for (int e = e0; e < E; e += 64) {
        float acc = 0.f;
        for (int i = 0; i < d; ++i) acc = fmaf(xs[r * d + i], ldv<TS>(w + (size_t)i * E + e), acc);
        z[(size_t)(t0 + r) * E + e] = acc + (bias ? bias[e] : 0.f);
    }
}
// dW_r[i,e] = sum_t x[t,i] dz[t,e]: thread per (i, e), loop over tokens (dense dz in fp32)
template <typename TS>
__global__ void __launch_bounds__(256) router_wgrad_simt(const TS* __restrict__ x, const float* __restrict__ dz, int T,
                                                         int d, int E, float* __restrict__ dw) {
    const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (idx >= (size_t)d * E) return;
    const int i = (int)(idx / E), e = (int)(idx - (size_t)i * E);
    float acc = 0.f;
    for (int t = 0; t < T; ++t) acc = fmaf(ldv<TS>(x + (size_t)t * d + i), dz[(size_t)t * E + e], acc);
    dw[idx] = acc;
}
// dX_r[t,i] = sum_e dz[t,e] W[i,e]: thread per (t, i)
template <typename TS>
__global__ void __launch_bounds__(256) router_dgrad_simt(const float* __restrict__ dz, const TS* __restrict__ w, int T,
                                                         int d, int E, TS* __restrict__ dx) {
    const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (idx >= (size_t)T * d) return;
    const int t = (int)(idx / d), i = (int)(idx - (size_t)t * d);
    float acc = 0.f;
    for (int e = 0; e < E; ++e) acc = fmaf(dz[(size_t)t * E + e], ldv<TS>(w + (size_t)i * E + e), acc);
    stv<TS>(dx + idx, acc);
}

// ---- dz_sel [T,k] (modes 0, 1) or dense dz [T,E] (mode 2) -> dense operands ---------------------------------------------
// SPLIT: two bf16 tensors hi, lo [T,E] (tensor path); else one dense fp32 tensor.  A warp per token row: zero fill, then
// lanes < k scatter the selected entries (the k experts of a token are distinct).
template <bool SPLIT>
__global__ void __launch_bounds__(256) dz_dense_kernel(const float* __restrict__ dz_sel, const int32_t* __restrict__ topk_idx,
                                                       int T, int E, int k, int dense_in, __nv_bfloat16* __restrict__ hi,
                                                       __nv_bfloat16* __restrict__ lo, float* __restrict__ dense) {
    const int lane = threadIdx.x & 31;
    const int t = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (t >= T) return;
    const size_t row = (size_t)t * E;
    if (dense_in) {
        for (int e = lane; e < E; e += 32) {
            const float v = dz_sel[row + e];
            if (SPLIT) {
                const __nv_bfloat16 h = __float2bfloat16_rn(v);
                hi[row + e] = h, lo[row + e] = __float2bfloat16_rn(v - __bfloat162float(h));
            } else {
                dense[row + e] = v;
            }
        }
        return;
    }
    for (int e = lane; e < E; e += 32) {
        if (SPLIT) hi[row + e] = __float2bfloat16_rn(0.f), lo[row + e] = __float2bfloat16_rn(0.f);
        else dense[row + e] = 0.f;
    }
    __syncwarp();
    if (lane < k) {
        const int e = topk_idx[(size_t)t * k + lane];
        const float v = dz_sel[(size_t)t * k + lane];
        if (SPLIT) {
            const __nv_bfloat16 h = __float2bfloat16_rn(v);
            hi[row + e] = h, lo[row + e] = __float2bfloat16_rn(v - __bfloat162float(h));
        } else {
            dense[row + e] = v;
        }
    }
}

}  // namespace

int launch_router_fwd(piper_ctx* c, Lane ln, const void* x, const void* w_r, const float* bias, float* logits) {
    const piper_moe_desc& D = c->D;
    if (tc_router_supported(c) && D.gemm_impl == PIPER_GEMM_AUTO) return tc_router_fwd(c, ln, x, w_r, bias, logits);
    const size_t smem = sizeof(float) * 4 * (size_t)D.d;
    if (smem > 48 * 1024) return PIPER_ERR_UNSUPPORTED;
    if (D.dtype == PIPER_DTYPE_BF16)
        router_fwd_simt<__nv_bfloat16><<<cdiv(D.T, 4), 256, smem, ln.stream>>>(
            static_cast<const __nv_bfloat16*>(x), static_cast<const __nv_bfloat16*>(w_r), bias, D.T, D.d, D.E, logits);
    else
        router_fwd_simt<float><<<cdiv(D.T, 4), 256, smem, ln.stream>>>(static_cast<const float*>(x),
                                                                         static_cast<const float*>(w_r), bias, D.T, D.d, D.E, logits);
    PIPER_LAUNCHED(c, "router_fwd_simt");
    return PIPER_OK;
}

// dz_scratch: [T,E] fp32-sized caller-owned scratch (hi | lo bf16 halves on the tensor path, dense fp32 otherwise)
int launch_router_bwd(piper_ctx* c, Lane ln, const void* x, const void* w_r, const int32_t* topk_idx, const float* dz_sel,
                      void* dz_scratch, float* dw_r, void* dx_router) {
    const piper_moe_desc& D = c->D;
    const int dense_in = D.gate_mode == PIPER_GATE_SOFTMAX_FULL ? 1 : 0;
    char* scratch = static_cast<char*>(dz_scratch);
    const size_t n = (size_t)D.T * D.E;
    if (tc_router_supported(c) && D.gemm_impl == PIPER_GEMM_AUTO) {
        __nv_bfloat16* hi = reinterpret_cast<__nv_bfloat16*>(scratch);
        __nv_bfloat16* lo = hi + n;
        dz_dense_kernel<true><<<cdiv(D.T, 8), 256, 0, ln.stream>>>(dz_sel, topk_idx, D.T, D.E, D.k, dense_in, hi, lo, nullptr);
        PIPER_LAUNCHED(c, "dz_dense_kernel");
        int rc = tc_router_wgrad(c, ln, x, hi, lo, dw_r);
        if (rc == PIPER_OK) rc = tc_router_dgrad(c, ln, hi, lo, w_r, dx_router);
        return rc;
    }
    float* dense = reinterpret_cast<float*>(scratch);
    dz_dense_kernel<false><<<cdiv(D.T, 8), 256, 0, ln.stream>>>(dz_sel, topk_idx, D.T, D.E, D.k, dense_in, nullptr, nullptr, dense);
    PIPER_LAUNCHED(c, "dz_dense_kernel");
    const unsigned gw = (unsigned)(((size_t)D.d * D.E + 255) / 256), gd = (unsigned)(((size_t)D.T * D.d + 255) / 256);
    if (D.dtype == PIPER_DTYPE_BF16) {
        router_wgrad_simt<__nv_bfloat16><<<gw, 256, 0, ln.stream>>>(static_cast<const __nv_bfloat16*>(x), dense, D.T, D.d, D.E, dw_r);
        PIPER_LAUNCHED(c, "router_wgrad_simt");
        router_dgrad_simt<__nv_bfloat16><<<gd, 256, 0, ln.stream>>>(dense, static_cast<const __nv_bfloat16*>(w_r), D.T, D.d, D.E,
                                                                   static_cast<__nv_bfloat16*>(dx_router));
    } else {
        router_wgrad_simt<float><<<gw, 256, 0, ln.stream>>>(static_cast<const float*>(x), dense, D.T, D.d, D.E, dw_r);
        PIPER_LAUNCHED(c, "router_wgrad_simt");
        router_dgrad_simt<float><<<gd, 256, 0, ln.stream>>>(dense, static_cast<const float*>(w_r), D.T, D.d, D.E,
                                                           static_cast<float*>(dx_router));
    }
    PIPER_LAUNCHED(c, "router_dgrad_simt");
    return PIPER_OK;
}

}  // namespace piper
