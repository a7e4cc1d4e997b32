// gemm_simt.cu — grouped SwiGLU FFN GEMMs on the FP32 ALUs (§8c Definition 3, 5).
// This is the product path of the fp32 config C1 (the 1e-5 bar rules out tf32 tensor cores, SURVEY.md
// §7 hard part 6) and a debug cross-check of the tcgen05 path on bf16 storage (PIPER_GEMM_SIMT).
// One generic 64x64x16 tile loop serves every contraction of the FFN through element strides:
//   C[m,n] = sum_k A[m*a_sm + k*a_sk] * B[k*b_sk + n*b_sn]      (fp32 FMA accumulation)
// No fast-math in this translation unit.
#include "piper_internal.cuh"

namespace piper {
namespace {

constexpr int TM = 64, TN = 64, TK = 16, LDS = 65;

template <typename TS> __device__ __forceinline__ float ldf(const TS* p);
template <> __device__ __forceinline__ float ldf<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ldf<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }
template <typename TS> __device__ __forceinline__ void stf(TS* p, float v);
template <> __device__ __forceinline__ void stf<float>(float* p, float v) { *p = v; }
template <> __device__ __forceinline__ void stf<__nv_bfloat16>(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }

// acc += A_tile * B_tile over K.  A points at (m0, k=0), B at (k=0, n0); rows >= m_valid and columns
// >= n_valid read as zero.  256 threads; thread (ty,tx) owns the 4x4 block at (4ty, 4tx).
template <typename TS>
__device__ __forceinline__ void tile_mac(float (&acc)[4][4], const TS* __restrict__ A, long a_sm, long a_sk, int m_valid,
                                         const TS* __restrict__ B, long b_sk, long b_sn, int n_valid, int K, float* As,
                                         float* Bs) {
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    for (int k0 = 0; k0 < K; k0 += TK) {
#pragma unroll
        for (int i = tid; i < TM * TK; i += 256) {
            int m, kk;
            if (a_sk == 1) m = i >> 4, kk = i & 15; else kk = i >> 6, m = i & 63;
            float v = 0.f;
            if (m < m_valid && k0 + kk < K) v = ldf<TS>(A + m * a_sm + (long)(k0 + kk) * a_sk);
            As[kk * LDS + m] = v;
        }
#pragma unroll
        for (int i = tid; i < TN * TK; i += 256) {
            int n, kk;
            if (b_sk == 1) n = i >> 4, kk = i & 15; else kk = i >> 6, n = i & 63;
            float v = 0.f;
            if (n < n_valid && k0 + kk < K) v = ldf<TS>(B + (long)(k0 + kk) * b_sk + n * b_sn);
            Bs[kk * LDS + n] = v;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < TK; ++kk) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = As[kk * LDS + ty * 4 + i], b[i] = Bs[kk * LDS + tx * 4 + i];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
}

// Which (group, first row, valid rows) does M-tile `tile` belong to?  Linear walk of offsets by one
// thread; tiles past the last group return false.
__device__ __forceinline__ bool find_m_tile(const int32_t* __restrict__ offsets, int G, int tile, int& g, int& r0,
                                            int& m_valid) {
    __shared__ int sh[3];
    if (threadIdx.x == 0) {
        int found = -1, lo = 0, rows = 0;
        for (int q = 0; q < G; ++q) {
            lo = offsets[q];
            rows = offsets[q + 1] - lo;
            const int nt = (rows + TM - 1) / TM;
            if (tile < nt) { found = q; break; }
            tile -= nt;
        }
        sh[0] = found;
        sh[1] = lo + tile * TM;
        sh[2] = found < 0 ? 0 : min(TM, rows - tile * TM);
    }
    __syncthreads();
    g = sh[0], r0 = sh[1], m_valid = sh[2];
    return g >= 0;
}

__device__ __forceinline__ void zero_acc(float (&acc)[4][4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
}

// ---- forward 1: G = Xp Wg, U = Xp Wu, H = silu(G) * U ----------------------------------------------
template <typename TS>
__global__ void __launch_bounds__(256)
simt_fwd1_kernel(const int32_t* __restrict__ offsets, int G_, int d, int I, const TS* __restrict__ xp,
                 const TS* __restrict__ wg, const TS* __restrict__ wu, TS* __restrict__ g_out, TS* __restrict__ u_out,
                 TS* __restrict__ h_out) {
    __shared__ float As[TK * LDS], Bs[TK * LDS];
    int g, r0, mv;
    if (!find_m_tile(offsets, G_, blockIdx.y, g, r0, mv)) return;
    const int n0 = blockIdx.x * TN, nv = min(TN, I - n0);
    float ag[4][4], au[4][4];
    zero_acc(ag), zero_acc(au);
    const TS* A = xp + (size_t)r0 * d;
    tile_mac<TS>(ag, A, d, 1, mv, wg + (size_t)g * d * I + n0, I, 1, nv, d, As, Bs);
    tile_mac<TS>(au, A, d, 1, mv, wu + (size_t)g * d * I + n0, I, 1, nv, d, As, Bs);
    const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int m = ty * 4 + i, n = tx * 4 + j;
            if (m < mv && n < nv) {
                const size_t at = (size_t)(r0 + m) * I + n0 + n;
                const float gv = ag[i][j], uv = au[i][j];
                stf<TS>(g_out + at, gv);
                stf<TS>(u_out + at, uv);
                stf<TS>(h_out + at, gv / (1.f + expf(-gv)) * uv);
            }
        }
}

// ---- forward 2: O = H Wd ------------------------------------------------------------------------------
template <typename TS>
__global__ void __launch_bounds__(256)
simt_fwd2_kernel(const int32_t* __restrict__ offsets, int G_, int d, int I, const TS* __restrict__ h,
                 const TS* __restrict__ wd, TS* __restrict__ o) {
    __shared__ float As[TK * LDS], Bs[TK * LDS];
    int g, r0, mv;
    if (!find_m_tile(offsets, G_, blockIdx.y, g, r0, mv)) return;
    const int n0 = blockIdx.x * TN, nv = min(TN, d - n0);
    float acc[4][4];
    zero_acc(acc);
    tile_mac<TS>(acc, h + (size_t)r0 * I, I, 1, mv, wd + (size_t)g * I * d + n0, d, 1, nv, I, As, Bs);
    const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int m = ty * 4 + i, n = tx * 4 + j;
            if (m < mv && n < nv) stf<TS>(o + (size_t)(r0 + m) * d + n0 + n, acc[i][j]);
        }
}

// ---- dgrad 1: dH = dO Wd^T; dG = dH * U * silu'(G); dU = dH * silu(G) ---------------------------------
template <typename TS>
__global__ void __launch_bounds__(256)
simt_dgrad1_kernel(const int32_t* __restrict__ offsets, int G_, int d, int I, const TS* __restrict__ d_o,
                   const TS* __restrict__ wd, const TS* __restrict__ g_in, const TS* __restrict__ u_in,
                   TS* __restrict__ dg, TS* __restrict__ du) {
    __shared__ float As[TK * LDS], Bs[TK * LDS];
    int g, r0, mv;
    if (!find_m_tile(offsets, G_, blockIdx.y, g, r0, mv)) return;
    const int n0 = blockIdx.x * TN, nv = min(TN, I - n0);
    float acc[4][4];
    zero_acc(acc);
    // B[k = dd, n = i] = Wd[i, dd]
    tile_mac<TS>(acc, d_o + (size_t)r0 * d, d, 1, mv, wd + (size_t)g * I * d + (size_t)n0 * d, 1, d, nv, d, As, Bs);
    const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int m = ty * 4 + i, n = tx * 4 + j;
            if (m < mv && n < nv) {
                const size_t at = (size_t)(r0 + m) * I + n0 + n;
                const float gv = ldf<TS>(g_in + at), uv = ldf<TS>(u_in + at), dh = acc[i][j];
                const float s = 1.f / (1.f + expf(-gv));
                stf<TS>(dg + at, dh * uv * (s * (1.f + gv * (1.f - s))));
                stf<TS>(du + at, dh * (gv * s));
            }
        }
}

// ---- dgrad 2: dXp = dG Wg^T + dU Wu^T -------------------------------------------------------------------
template <typename TS>
__global__ void __launch_bounds__(256)
simt_dgrad2_kernel(const int32_t* __restrict__ offsets, int G_, int d, int I, const TS* __restrict__ dg,
                   const TS* __restrict__ du, const TS* __restrict__ wg, const TS* __restrict__ wu,
                   TS* __restrict__ dxp) {
    __shared__ float As[TK * LDS], Bs[TK * LDS];
    int g, r0, mv;
    if (!find_m_tile(offsets, G_, blockIdx.y, g, r0, mv)) return;
    const int n0 = blockIdx.x * TN, nv = min(TN, d - n0);
    float acc[4][4];
    zero_acc(acc);
    // B[k = i, n = dd] = W[dd, i]
    tile_mac<TS>(acc, dg + (size_t)r0 * I, I, 1, mv, wg + (size_t)g * d * I + (size_t)n0 * I, 1, I, nv, I, As, Bs);
    tile_mac<TS>(acc, du + (size_t)r0 * I, I, 1, mv, wu + (size_t)g * d * I + (size_t)n0 * I, 1, I, nv, I, As, Bs);
    const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int m = ty * 4 + i, n = tx * 4 + j;
            if (m < mv && n < nv) stf<TS>(dxp + (size_t)(r0 + m) * d + n0 + n, acc[i][j]);
        }
}

// ---- wgrad: C[g][m, n] = sum_{r in group g} A[r, m] * B[r, n]  (exact zeros for empty groups) ---------
template <typename TS>
__global__ void __launch_bounds__(256)
simt_wgrad_kernel(const int32_t* __restrict__ offsets, int M, int N, const TS* __restrict__ a, const TS* __restrict__ b,
                  TS* __restrict__ c) {
    __shared__ float As[TK * LDS], Bs[TK * LDS];
    const int g = blockIdx.z, lo = offsets[g], rows = offsets[g + 1] - lo;
    const int m0 = blockIdx.y * TM, n0 = blockIdx.x * TN, mv = min(TM, M - m0), nv = min(TN, N - n0);
    float acc[4][4];
    zero_acc(acc);
    tile_mac<TS>(acc, a + (size_t)lo * M + m0, 1, M, mv, b + (size_t)lo * N + n0, N, 1, nv, rows, As, Bs);
    const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int m = ty * 4 + i, n = tx * 4 + j;
            if (m < mv && n < nv) stf<TS>(c + (size_t)g * M * N + (size_t)(m0 + m) * N + n0 + n, acc[i][j]);
        }
}

inline int m_tiles_bound(const FfnProblem& p) { return cdiv(p.max_rows, TM) + p.G; }

template <typename TS>
int fwd_t(piper_ctx* c, Lane ln, const FfnProblem& p, int which) {
    const dim3 g1(cdiv(p.I, TN), m_tiles_bound(p)), g2(cdiv(p.d, TN), m_tiles_bound(p));
    if (which & 1) {
        simt_fwd1_kernel<TS><<<g1, 256, 0, ln.stream>>>(p.offsets, p.G, p.d, p.I, (const TS*)p.xp,
                                                        (const TS*)p.w_gate, (const TS*)p.w_up, (TS*)p.g, (TS*)p.u,
                                                        (TS*)p.h);
        PIPER_LAUNCHED(c, "simt_fwd1_kernel");
    }
    if (which & 2) {
        simt_fwd2_kernel<TS><<<g2, 256, 0, ln.stream>>>(p.offsets, p.G, p.d, p.I, (const TS*)p.h, (const TS*)p.w_down,
                                                        (TS*)p.o);
        PIPER_LAUNCHED(c, "simt_fwd2_kernel");
    }
    return PIPER_OK;
}
template <typename TS>
int dgrad_t(piper_ctx* c, Lane ln, const FfnProblem& p, int which) {
    const dim3 g1(cdiv(p.I, TN), m_tiles_bound(p)), g2(cdiv(p.d, TN), m_tiles_bound(p));
    if (which & 1) {
        simt_dgrad1_kernel<TS><<<g1, 256, 0, ln.stream>>>(p.offsets, p.G, p.d, p.I, (const TS*)p.d_o,
                                                          (const TS*)p.w_down, (const TS*)p.g, (const TS*)p.u,
                                                          (TS*)p.dg, (TS*)p.du);
        PIPER_LAUNCHED(c, "simt_dgrad1_kernel");
    }
    if (which & 2) {
        simt_dgrad2_kernel<TS><<<g2, 256, 0, ln.stream>>>(p.offsets, p.G, p.d, p.I, (const TS*)p.dg, (const TS*)p.du,
                                                          (const TS*)p.w_gate, (const TS*)p.w_up, (TS*)p.dxp);
        PIPER_LAUNCHED(c, "simt_dgrad2_kernel");
    }
    return PIPER_OK;
}
template <typename TS>
int wgrad_t(piper_ctx* c, Lane ln, const FfnProblem& p) {
    const dim3 gw(cdiv(p.I, TN), cdiv(p.d, TM), p.G), gd(cdiv(p.d, TN), cdiv(p.I, TM), p.G);
    simt_wgrad_kernel<TS><<<gw, 256, 0, ln.stream>>>(p.offsets, p.d, p.I, (const TS*)p.xp, (const TS*)p.dg,
                                                     (TS*)p.dw_gate);
    PIPER_LAUNCHED(c, "simt_wgrad_kernel");
    simt_wgrad_kernel<TS><<<gw, 256, 0, ln.stream>>>(p.offsets, p.d, p.I, (const TS*)p.xp, (const TS*)p.du,
                                                     (TS*)p.dw_up);
    PIPER_LAUNCHED(c, "simt_wgrad_kernel");
    simt_wgrad_kernel<TS><<<gd, 256, 0, ln.stream>>>(p.offsets, p.I, p.d, (const TS*)p.h, (const TS*)p.d_o,
                                                     (TS*)p.dw_down);
    PIPER_LAUNCHED(c, "simt_wgrad_kernel");
    return PIPER_OK;
}

}  // namespace

int simt_ffn_fwd(piper_ctx* c, Lane ln, const FfnProblem& p, int which) {
    return c->D.dtype == PIPER_DTYPE_BF16 ? fwd_t<__nv_bfloat16>(c, ln, p, which) : fwd_t<float>(c, ln, p, which);
}
int simt_ffn_dgrad(piper_ctx* c, Lane ln, const FfnProblem& p, int which) {
    return c->D.dtype == PIPER_DTYPE_BF16 ? dgrad_t<__nv_bfloat16>(c, ln, p, which) : dgrad_t<float>(c, ln, p, which);
}
int simt_ffn_wgrad(piper_ctx* c, Lane ln, const FfnProblem& p) {
    return c->D.dtype == PIPER_DTYPE_BF16 ? wgrad_t<__nv_bfloat16>(c, ln, p) : wgrad_t<float>(c, ln, p);
}

}  // namespace piper
