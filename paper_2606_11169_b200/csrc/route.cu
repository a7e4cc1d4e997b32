// route.cu — F1 route_topk and B6 route_bwd (SURVEY.md §8a F1/B6, §8c Definition 1 and 5).
// One warp per token.  Selection is k rounds of a warp arg-max under the total order
// (value descending, expert index ascending) — pure fp32 compares, so indices are bit-exact
// (reading c-6).  The per-expert histogram is an integer smem histogram flushed with integer atomics
// (order-independent result).  HBM-side: logits are read once, 128-bit per lane when E % 128 == 0.
#include "piper_internal.cuh"

namespace piper {
namespace {

constexpr int kRouteWarps = 8;

// Element owned by (lane, slot i).  VEC = 4: float4 loads, lane owns 4 consecutive experts of each
// 128-wide segment; VEC = 1: strided scalars.  In both, slots ascend with the expert index.
template <int VEC>
__device__ __forceinline__ int elem_of(int lane, int i) {
    return VEC == 4 ? (i >> 2) * 128 + lane * 4 + (i & 3) : i * 32 + lane;
}
template <int VEC>
__device__ __forceinline__ int lane_of(int e) {
    return VEC == 4 ? (e & 127) >> 2 : e & 31;
}
template <int VEC>
__device__ __forceinline__ int slot_of(int e) {
    return VEC == 4 ? ((e >> 7) << 2) + (e & 3) : e >> 5;
}

template <int NPL, int VEC>
__global__ void __launch_bounds__(kRouteWarps * 32)
route_topk_kernel(const float* __restrict__ z, int T, int E, int k, int mode, int32_t* __restrict__ topk_idx,
                  float* __restrict__ gates, int32_t* __restrict__ counts_global) {
    extern __shared__ int32_t hist[];
    for (int e = threadIdx.x; e < E; e += blockDim.x) hist[e] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int warp = blockIdx.x * kRouteWarps + (threadIdx.x >> 5);
    const int nwarps = gridDim.x * kRouteWarps;
    const float NEG_INF = __int_as_float(0xff800000);

    for (int t = warp; t < T; t += nwarps) {
        const float* zt = z + (size_t)t * E;
        float v[NPL];
        uint32_t used = 0;  // bit i: slot i already selected or out of range
        if (VEC == 4) {
#pragma unroll
            for (int q = 0; q < NPL / 4; ++q) {
                const int e0 = q * 128 + lane * 4;
                if (e0 < E) {
                    const float4 f = __ldg(reinterpret_cast<const float4*>(zt + e0));
                    v[4 * q] = f.x, v[4 * q + 1] = f.y, v[4 * q + 2] = f.z, v[4 * q + 3] = f.w;
                } else {
                    v[4 * q] = v[4 * q + 1] = v[4 * q + 2] = v[4 * q + 3] = NEG_INF;
                    used |= 0xFu << (4 * q);
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i < NPL; ++i) {
                const int e = i * 32 + lane;
                if (e < E) {
                    v[i] = __ldg(zt + e);
                } else {
                    v[i] = NEG_INF;
                    used |= 1u << i;
                }
            }
        }
        float selv[kMaxK];
        int sele[kMaxK];
#pragma unroll
        for (int j = 0; j < kMaxK; ++j) {
            selv[j] = 0.f, sele[j] = 0;
            if (j < k) {
                // lane-local best: ascending slots = ascending expert index, strict '>' keeps the lowest index
                float bv = NEG_INF;
                int bi = 0x7fffffff;
#pragma unroll
                for (int i = 0; i < NPL; ++i)
                    if (!((used >> i) & 1u) && (bi == 0x7fffffff || v[i] > bv)) bv = v[i], bi = elem_of<VEC>(lane, i);
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) {
                    const float ov = __shfl_xor_sync(0xffffffffu, bv, off);
                    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
                    if (ov > bv || (ov == bv && oi < bi)) bv = ov, bi = oi;
                }
                if (lane_of<VEC>(bi) == lane) used |= 1u << slot_of<VEC>(bi);
                selv[j] = bv, sele[j] = bi;
            }
        }
        // gates (fp32; every lane computes the same k values)
        float g[kMaxK];
        if (mode == PIPER_GATE_SOFTMAX_RENORM) {
            float s = 0.f;
#pragma unroll
            for (int j = 0; j < kMaxK; ++j) {
                g[j] = j < k ? expf(selv[j] - selv[0]) : 0.f;
                s += g[j];
            }
#pragma unroll
            for (int j = 0; j < kMaxK; ++j) g[j] = g[j] / s;
        } else if (mode == PIPER_GATE_SIGMOID_RENORM) {
            float s = 0.f;
#pragma unroll
            for (int j = 0; j < kMaxK; ++j) {
                g[j] = j < k ? 1.f / (1.f + expf(-selv[j])) : 0.f;
                s += g[j];
            }
#pragma unroll
            for (int j = 0; j < kMaxK; ++j) g[j] = g[j] / s;
        } else {  // softmax over all E, not renormalised
            const float m = selv[0];
            float s = 0.f;
#pragma unroll
            for (int i = 0; i < NPL; ++i)
                if (elem_of<VEC>(lane, i) < E) s += expf(v[i] - m);
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
#pragma unroll
            for (int j = 0; j < kMaxK; ++j) g[j] = j < k ? expf(selv[j] - m) / s : 0.f;
        }
        int my_e = 0;
        float my_g = 0.f;
#pragma unroll
        for (int j = 0; j < kMaxK; ++j)
            if (lane == j) my_e = sele[j], my_g = g[j];
        if (lane < k) {
            topk_idx[(size_t)t * k + lane] = my_e;
            gates[(size_t)t * k + lane] = my_g;
            atomicAdd(&hist[my_e], 1);
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < E; e += blockDim.x)
        if (hist[e]) atomicAdd(&counts_global[e], hist[e]);
}

// Gate-normalisation backward on the selected logits (modes 0, 1): one thread per token.
__global__ void route_bwd_sel_kernel(const float* __restrict__ z, const int32_t* __restrict__ topk_idx,
                                     const float* __restrict__ gates, const float* __restrict__ dgates, int T, int E,
                                     int k, int mode, float* __restrict__ dz) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    float dot = 0.f;
    for (int j = 0; j < k; ++j) dot += gates[(size_t)t * k + j] * dgates[(size_t)t * k + j];
    if (mode == PIPER_GATE_SOFTMAX_RENORM) {
        // dz_j = g_j (dgates_j - sum_j' g_j' dgates_j')
        for (int j = 0; j < k; ++j) dz[(size_t)t * k + j] = gates[(size_t)t * k + j] * (dgates[(size_t)t * k + j] - dot);
    } else {
        // ds_j = (dgates_j - dot) / sum s ; dz_j = ds_j s_j (1 - s_j)
        float sg[kMaxK], s = 0.f;
        for (int j = 0; j < k; ++j) {
            sg[j] = 1.f / (1.f + expf(-z[(size_t)t * E + topk_idx[(size_t)t * k + j]]));
            s += sg[j];
        }
        for (int j = 0; j < k; ++j) dz[(size_t)t * k + j] = (dgates[(size_t)t * k + j] - dot) / s * sg[j] * (1.f - sg[j]);
    }
}

// Mode 2 (full softmax, not renormalised): dz[t,e] = sum_j dgates_j p_{e_j} ([e = e_j] - p_e); warp per token.
__global__ void route_bwd_full_kernel(const float* __restrict__ z, const int32_t* __restrict__ topk_idx,
                                      const float* __restrict__ gates, const float* __restrict__ dgates, int T, int E,
                                      int k, float* __restrict__ dz) {
    const int lane = threadIdx.x & 31;
    const int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (t >= T) return;
    const float* zt = z + (size_t)t * E;
    const float m = zt[topk_idx[(size_t)t * k]];
    float s = 0.f;
    for (int e = lane; e < E; e += 32) s += expf(zt[e] - m);
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    float dot = 0.f;  // sum_j dgates_j p_{e_j}; gates[t,j] = p_{e_j} in this mode
    for (int j = 0; j < k; ++j) dot += gates[(size_t)t * k + j] * dgates[(size_t)t * k + j];
    for (int e = lane; e < E; e += 32) {
        const float p = expf(zt[e] - m) / s;
        float val = -p * dot;
        for (int j = 0; j < k; ++j)
            if (topk_idx[(size_t)t * k + j] == e) val += dgates[(size_t)t * k + j] * gates[(size_t)t * k + j];
        dz[(size_t)t * E + e] = val;
    }
}

template <int NPL, int VEC>
int launch_topk(piper_ctx* c, Lane ln, const float* z, int32_t* idx, float* gates, int32_t* cg) {
    const piper_moe_desc& D = c->D;
    int blocks = cdiv(D.T, kRouteWarps);
    const int cap = ln.sms * 8;  // (2 blocks per SM, to flush fewer block histograms, measured slower: C3 33 -> 38 us)
    if (blocks > cap) blocks = cap;
    route_topk_kernel<NPL, VEC><<<blocks, kRouteWarps * 32, D.E * sizeof(int32_t), ln.stream>>>(
        z, D.T, D.E, D.k, D.gate_mode, idx, gates, cg);
    PIPER_LAUNCHED(c, "route_topk_kernel");
    return PIPER_OK;
}

}  // namespace

int launch_route_topk(piper_ctx* c, Lane ln, const float* z, int32_t* idx, float* gates, int32_t* cg) {
    const int E = c->D.E;
    PIPER_CUDA(c, cudaMemsetAsync(cg, 0, sizeof(int32_t) * E, ln.stream));
    if (E % 128 == 0) {
        if (E == 128) return launch_topk<4, 4>(c, ln, z, idx, gates, cg);
        if (E == 256) return launch_topk<8, 4>(c, ln, z, idx, gates, cg);
        return launch_topk<16, 4>(c, ln, z, idx, gates, cg);
    }
    if (E <= 32) return launch_topk<1, 1>(c, ln, z, idx, gates, cg);
    if (E <= 64) return launch_topk<2, 1>(c, ln, z, idx, gates, cg);
    if (E <= 128) return launch_topk<4, 1>(c, ln, z, idx, gates, cg);
    if (E <= 256) return launch_topk<8, 1>(c, ln, z, idx, gates, cg);
    return launch_topk<16, 1>(c, ln, z, idx, gates, cg);
}

int launch_route_bwd(piper_ctx* c, Lane ln, const float* z, const int32_t* idx, const float* gates,
                     const float* dgates, float* dz) {
    const piper_moe_desc& D = c->D;
    if (D.gate_mode == PIPER_GATE_SOFTMAX_FULL) {
        route_bwd_full_kernel<<<cdiv(D.T, 8), 256, 0, ln.stream>>>(z, idx, gates, dgates, D.T, D.E, D.k, dz);
        PIPER_LAUNCHED(c, "route_bwd_full_kernel");
    } else {
        route_bwd_sel_kernel<<<cdiv(D.T, 128), 128, 0, ln.stream>>>(z, idx, gates, dgates, D.T, D.E, D.k, D.gate_mode,
                                                                    dz);
        PIPER_LAUNCHED(c, "route_bwd_sel_kernel");
    }
    return PIPER_OK;
}

}  // namespace piper
