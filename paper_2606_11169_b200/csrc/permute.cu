// permute.cu — F2 histogram + scan + rank, F3 dispatch_pack, F5 combine, B1 combine_bwd, B5 unpack
// (SURVEY.md §8a, §8c Definition 2, 4, 5).  All HBM-bound row movers are TOKEN-major: a warp owns a
// token, reads its source row once with 128-bit loads and touches each packed row exactly once, so the
// traffic equals the algorithmic bytes of SURVEY.md §8d.  Ranks are deterministic (no atomics decide an
// index): per-chunk histograms, a prefix over chunks, then __match_any_sync ranks inside a chunk.
#include "piper_internal.cuh"

#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace piper {
namespace {

#ifndef PIPER_MOVE_WARPS
#define PIPER_MOVE_WARPS 8
#endif
#ifndef PIPER_MOVE_U
#define PIPER_MOVE_U 4
#endif
constexpr int kMoveWarps = PIPER_MOVE_WARPS;  // warps per block of the row movers

// ---- F2 phase 1: per-chunk histogram of local experts ------------------------------------------
__global__ void __launch_bounds__(kScanChunk)
chunk_hist_kernel(const int32_t* __restrict__ topk_idx, int n_assign, int e_lo, int E_loc,
                  int32_t* __restrict__ chunk_counts) {
    extern __shared__ int32_t hist[];
    for (int e = threadIdx.x; e < E_loc; e += blockDim.x) hist[e] = 0;
    __syncthreads();
    const int a = blockIdx.x * kScanChunk + threadIdx.x;
    if (a < n_assign) {
        const int i = topk_idx[a] - e_lo;
        if (i >= 0 && i < E_loc) atomicAdd(&hist[i], 1);  // integer count: order-independent
    }
    __syncthreads();
    for (int e = threadIdx.x; e < E_loc; e += blockDim.x) chunk_counts[(size_t)blockIdx.x * E_loc + e] = hist[e];
}

// ---- F2 phase 2: prefix over chunks, aligned exclusive scan -> offsets, stable ranks, row_of and src_of ----------
// Block = one chunk of kScanChunk assignments in flat order a = t*k + j.  Every block derives what it needs from the
// chunk histograms itself (n_chunks * E_loc integers, L2-resident): the experts' totals, its own base = the counts of
// the chunks before it, and the aligned exclusive scan of the totals (block 0 also writes counts / offsets), so no
// single-block scan kernel sits between the histogram and the ranks.  Ranks: warps take turns (ascending a); inside a
// warp __match_any_sync groups equal experts and the rank is the number of lower lanes of the group; a shared running
// count per expert carries the rank across warps.  No atomic decides an index.  src_of entries that hold no
// assignment (pad rows of a segment and every row from offsets[E_loc] to a_cap) are written as -1 by the same launch:
// the blocks share those ranges.  gate_rows[row] = gates[a] (0 on a segment's pad rows) is written here too, so that the
// gate of a packed row exists whether or not the rows themselves are materialised (N2 fusion).
__global__ void __launch_bounds__(kScanChunk)
scan_rank_kernel(const int32_t* __restrict__ topk_idx, const float* __restrict__ gates, int n_assign, int e_lo, int E_loc,
                 int row_align, int a_cap, const int32_t* __restrict__ chunk_counts, int32_t* __restrict__ counts,
                 int32_t* __restrict__ offsets, int32_t* __restrict__ row_of, int32_t* __restrict__ src_of,
                 float* __restrict__ gate_rows) {
    extern __shared__ int32_t sm[];
    int32_t* run = sm;                  // [E_loc] next free row of each expert for this chunk
    int32_t* s_cnt = sm + E_loc;        // [E_loc] real rows
    int32_t* s_off = sm + 2 * E_loc;    // [E_loc + 1] aligned exclusive scan
    __shared__ int32_t warp_tot[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int n_chunks = gridDim.x;
    // totals and this chunk's base, experts strided over the block (E_loc <= 512 < blockDim)
    int total = 0, base = 0;
    const int e = threadIdx.x;
    if (e < E_loc) {
        for (int c = 0; c < n_chunks; ++c) {
            const int v = chunk_counts[(size_t)c * E_loc + e];
            if (c < (int)blockIdx.x) base += v;
            total += v;
        }
        s_cnt[e] = total;
    }
    const int padded = e < E_loc ? (total + row_align - 1) / row_align * row_align : 0;
    int inc = padded;  // inclusive warp scan by shuffles, then over the warps' totals
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += o;
    }
    if (lane == 31) warp_tot[w] = inc;
    __syncthreads();
    if (w == 0) {
        const int t = warp_tot[lane];
        int ti = t;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, ti, off);
            if (lane >= off) ti += o;
        }
        warp_tot[lane] = ti - t;  // exclusive
    }
    __syncthreads();
    const int excl = warp_tot[w] + inc - padded;
    if (e < E_loc) {
        s_off[e] = excl, run[e] = excl + base;
        if (e == E_loc - 1) s_off[E_loc] = excl + padded;
        if (blockIdx.x == 0) {
            counts[e] = total, offsets[e] = excl;
            if (e == E_loc - 1) offsets[E_loc] = excl + padded;
        }
    }
    __syncthreads();
    // rows without an assignment: segment pads (experts dealt round-robin over the blocks) and the unused tail
    for (int g = blockIdx.x; g < E_loc; g += n_chunks)
        for (int r = s_off[g] + s_cnt[g] + threadIdx.x; r < s_off[g + 1]; r += blockDim.x) src_of[r] = -1, gate_rows[r] = 0.f;
    {
        const int used = s_off[E_loc], tail = a_cap - used;
        const int per = (tail + n_chunks - 1) / n_chunks;
        const int lo = used + (int)blockIdx.x * per, hi = min(a_cap, lo + per);
        for (int r = lo + threadIdx.x; r < hi; r += blockDim.x) src_of[r] = -1;
    }
    const int a = blockIdx.x * kScanChunk + threadIdx.x;
    int i = -1;
    if (a < n_assign) {
        i = topk_idx[a] - e_lo;
        if (i < 0 || i >= E_loc) i = -1;
    }
    const unsigned peers = __match_any_sync(0xffffffffu, i);
    const int below = __popc(peers & ((1u << lane) - 1u));
    const int leader = __ffs(peers) - 1;
    int row = -1;
    for (int turn = 0; turn < kScanChunk / 32; ++turn) {
        if (turn == w && i >= 0) {
            int b0 = 0;
            if (lane == leader) {
                b0 = run[i];
                run[i] = b0 + __popc(peers);
            }
            b0 = __shfl_sync(peers, b0, leader);
            row = b0 + below;
        }
        __syncthreads();
    }
    if (a < n_assign) {
        row_of[a] = row;
        if (row >= 0) src_of[row] = a, gate_rows[row] = gates[a];  // the row's gate travels with the permutation
    }
}

// ---- element helpers for the row movers -----------------------------------------------------------
// A 16-byte packet holds 8 bf16 or 4 fp32 values; acc[] always has 8 slots.
template <bool BF16>
__device__ __forceinline__ void unpack_add(const int4& v, float (&acc)[8], float scale) {
    if (BF16) {
        const uint32_t w[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float2 f = bf2_to_f2(w[q]);
            acc[2 * q] = fmaf(scale, f.x, acc[2 * q]);
            acc[2 * q + 1] = fmaf(scale, f.y, acc[2 * q + 1]);
        }
    } else {
        acc[0] = fmaf(scale, __int_as_float(v.x), acc[0]);
        acc[1] = fmaf(scale, __int_as_float(v.y), acc[1]);
        acc[2] = fmaf(scale, __int_as_float(v.z), acc[2]);
        acc[3] = fmaf(scale, __int_as_float(v.w), acc[3]);
    }
}
template <bool BF16>
__device__ __forceinline__ int4 pack_out(const float (&acc)[8]) {
    int4 r;
    if (BF16) {
        r.x = (int)f2_to_bf2(acc[0], acc[1]);
        r.y = (int)f2_to_bf2(acc[2], acc[3]);
        r.z = (int)f2_to_bf2(acc[4], acc[5]);
        r.w = (int)f2_to_bf2(acc[6], acc[7]);
    } else {
        r.x = __float_as_int(acc[0]), r.y = __float_as_int(acc[1]);
        r.z = __float_as_int(acc[2]), r.w = __float_as_int(acc[3]);
    }
    return r;
}
template <bool BF16>
__device__ __forceinline__ float dot_packets(const int4& a, const int4& b) {
    float za[8] = {0, 0, 0, 0, 0, 0, 0, 0}, zb[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    unpack_add<BF16>(a, za, 1.f);
    unpack_add<BF16>(b, zb, 1.f);
    float s = 0.f;
#pragma unroll
    for (int q = 0; q < (BF16 ? 8 : 4); ++q) s = fmaf(za[q], zb[q], s);
    return s;
}

// ---- row movers: common shape ----------------------------------------------------------------------
// Work item = (token, column split): a warp moves `U` 16-byte packets per lane per step (2 KB per warp and
// source row), with the next source row's packets already in flight while the current ones are consumed.
// Splitting a row over several items keeps every resident warp busy when T is small (no cross-split
// reduction exists in pack / combine / unpack; combine_bwd's dot products need the whole row and do not
// split).  No per-thread arrays indexed at run time: row indices are re-read from row_of (L1 hits).
constexpr int U = PIPER_MOVE_U;       // packets per lane per step
constexpr int kStep = 32 * U;        // packets per warp per step

__device__ __forceinline__ void load_step(int4 (&v)[U], const int4* __restrict__ src, int p0, int lane, int hi) {
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int p = p0 + u * 32 + lane;
        v[u] = p < hi ? ld_nc16(src + p) : make_int4(0, 0, 0, 0);
    }
}

// ---- F3 dispatch_pack ----------------------------------------------------------------------------
// Token items [0, T*S): copy the split's columns of x[t] into each local row of the token (the rows' gates are
// written with the permutation, scan_rank_kernel).  Row items [T*S, T*S + a_cap): zero the pad rows inside [0, offsets[E_loc]).
__global__ void __launch_bounds__(kMoveWarps * 32)
pack_kernel(const int4* __restrict__ x, const int32_t* __restrict__ offsets, const int32_t* __restrict__ row_of,
            const int32_t* __restrict__ src_of, int T, int k, int E_loc, int a_cap, int row_packets, int S,
            int split_packets, int4* __restrict__ xp) {
    const int lane = threadIdx.x & 31;
    const int warp = blockIdx.x * kMoveWarps + (threadIdx.x >> 5);
    const int nwarps = gridDim.x * kMoveWarps;
    const int used = offsets[E_loc];
    const int n_tok_items = T * S;
    for (int item = warp; item < n_tok_items + a_cap; item += nwarps) {
        if (item < n_tok_items) {
            const int t = item / S, sp = item - t * S;
            const int32_t* ro = row_of + (size_t)t * k;
            const int my_row = lane < k ? ro[lane] : -1;
            if (__ballot_sync(0xffffffffu, my_row >= 0) == 0) continue;
            const int lo = sp * split_packets, hi = min(row_packets, lo + split_packets);
            const int4* src = x + (size_t)t * row_packets;
            for (int p0 = lo; p0 < hi; p0 += kStep) {
                int4 v[U];
                load_step(v, src, p0, lane, hi);
                for (int j = 0; j < k; ++j) {
                    const int r = __shfl_sync(0xffffffffu, my_row, j);
                    if (r < 0) continue;
                    int4* dst = xp + (size_t)r * row_packets;
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int p = p0 + u * 32 + lane;
                        if (p < hi) st16(dst + p, v[u]);
                    }
                }
            }
        } else {
            const int r = item - n_tok_items;
            if (r >= used || src_of[r] >= 0) continue;
            int4* dst = xp + (size_t)r * row_packets;
            for (int p = lane; p < row_packets; p += 32) st16(dst + p, make_int4(0, 0, 0, 0));
        }
    }
}

// ---- F5 combine / B5 unpack ------------------------------------------------------------------------
// y[t] = sum_{j local} w_j * o[row_of[t,j]] (+ s[t]);  WEIGHTED: w_j = gates[t,j], else 1 (unpack).
// fp32 accumulation in slot order j = 0..k-1 then s, one rounding on store.
// TWO: a second token-row addend s2 after s (the router's term of dX, N1); the common kernels are compiled without it.
template <bool BF16, bool WEIGHTED, bool TWO>
__global__ void __launch_bounds__(kMoveWarps * 32)
combine_kernel(const int4* __restrict__ o, const int32_t* __restrict__ row_of, const float* __restrict__ gates,
               const int4* __restrict__ s, const int4* __restrict__ s2, int T, int k, int row_packets, int S,
               int split_packets, int4* __restrict__ y) {
    const int lane = threadIdx.x & 31;
    const int warp = blockIdx.x * kMoveWarps + (threadIdx.x >> 5);
    const int nwarps = gridDim.x * kMoveWarps;
    const int n_src = k + (s != nullptr ? 1 : 0) + (TWO ? 1 : 0);
    for (int item = warp; item < T * S; item += nwarps) {
        const int t = item / S, sp = item - t * S;
        const int my_row = lane < k ? row_of[(size_t)t * k + lane] : -1;
        const float my_w = (WEIGHTED && lane < k) ? gates[(size_t)t * k + lane] : 1.f;
        const int lo = sp * split_packets, hi = min(row_packets, lo + split_packets);
        for (int p0 = lo; p0 < hi; p0 += kStep) {
            float acc[U][8];
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[u][q] = 0.f;
            int4 cur[U];
            float wc = 0.f;
            bool have = false;
            for (int j = 0; j < n_src; ++j) {
                const int4* src;
                float w = 1.f;
                if (j < k) {
                    const int r = __shfl_sync(0xffffffffu, my_row, j);
                    w = __shfl_sync(0xffffffffu, my_w, j);
                    if (r < 0) continue;
                    src = o + (size_t)r * row_packets;
                } else {
                    src = ((TWO && (j > k || s == nullptr)) ? s2 : s) + (size_t)t * row_packets;
                }
                int4 nxt[U];
                load_step(nxt, src, p0, lane, hi);  // in flight while the previous source is accumulated
                if (have) {
#pragma unroll
                    for (int u = 0; u < U; ++u) unpack_add<BF16>(cur[u], acc[u], wc);
                }
#pragma unroll
                for (int u = 0; u < U; ++u) cur[u] = nxt[u];
                wc = w, have = true;
            }
            if (have) {
#pragma unroll
                for (int u = 0; u < U; ++u) unpack_add<BF16>(cur[u], acc[u], wc);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int p = p0 + u * 32 + lane;
                if (p < hi) st16(y + (size_t)t * row_packets + p, pack_out<BF16>(acc[u]));
            }
        }
    }
}

// ---- B1 combine_bwd ---------------------------------------------------------------------------------
// Token items: for every local slot j: d_o[row] = gates[t,j] * dy[t]; dgates[t,j] = <dy[t], o[row]> (0 for
// non-local slots).  Slot-outer loop: dy[t] is re-read per local slot (L1/L2 hits), the dot product stays a
// scalar.  Row items: zero the pad rows of d_o inside [0, offsets[E_loc]).
// WRITE_DO = false (N2 fusion: the GEMMs gather dY rows themselves): only the dgates dot products, d_o is not touched.
template <bool BF16, bool WRITE_DO>
__global__ void __launch_bounds__(kMoveWarps * 32)
combine_bwd_kernel(const int4* __restrict__ dy, const int4* __restrict__ o, const int32_t* __restrict__ src_of,
                   const int32_t* __restrict__ row_of, const float* __restrict__ gates,
                   const int32_t* __restrict__ offsets, int T, int k, int E_loc, int a_cap, int row_packets,
                   int4* __restrict__ d_o, float* __restrict__ dgates) {
    const int lane = threadIdx.x & 31;
    const int warp = blockIdx.x * kMoveWarps + (threadIdx.x >> 5);
    const int nwarps = gridDim.x * kMoveWarps;
    const int used = offsets[E_loc];
    for (int item = warp; item < T + a_cap; item += nwarps) {
        if (item < T) {
            const int t = item;
            const int my_row = lane < k ? row_of[(size_t)t * k + lane] : -1;
            const float my_w = lane < k ? gates[(size_t)t * k + lane] : 0.f;
            if (lane < k && my_row < 0) dgates[(size_t)t * k + lane] = 0.f;
            const int4* src = dy + (size_t)t * row_packets;
            for (int j = 0; j < k; ++j) {
                const int r = __shfl_sync(0xffffffffu, my_row, j);
                const float w = __shfl_sync(0xffffffffu, my_w, j);
                if (r < 0) continue;
                const int4* orow = o + (size_t)r * row_packets;
                int4* drow = d_o + (size_t)r * row_packets;
                float dot = 0.f;
                for (int p0 = 0; p0 < row_packets; p0 += kStep) {
                    int4 v[U], ov[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int p = p0 + u * 32 + lane;
                        v[u] = p < row_packets ? __ldg(src + p) : make_int4(0, 0, 0, 0);
                    }
                    load_step(ov, orow, p0, lane, row_packets);
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int p = p0 + u * 32 + lane;
                        if (p < row_packets) {
                            dot += dot_packets<BF16>(v[u], ov[u]);
                            if (WRITE_DO) {
                                float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
                                unpack_add<BF16>(v[u], acc, w);
                                st16(drow + p, pack_out<BF16>(acc));
                            }
                        }
                    }
                }
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
                if (lane == 0) dgates[(size_t)t * k + j] = dot;
            }
        } else if (WRITE_DO) {
            const int r = item - T;
            if (r >= used || src_of[r] >= 0) continue;
            int4* dst = d_o + (size_t)r * row_packets;
            for (int p = lane; p < row_packets; p += 32) st16(dst + p, make_int4(0, 0, 0, 0));
        }
    }
}

// Column splits per token so that about move_items (PIPER_OPT_MOVE_ITEMS) items exist per resident warp of the lane: with sparse local
// slots (C3: a third of the tokens has none, the others 1-4) the work per item varies, and finer items even it out
// (C3 combine 82.8 -> 75.8 us, unpack 81.9 -> 73.7 us against 2 items per warp; C2 unchanged).
inline void choose_split(const piper_ctx* c, Lane ln, int T, int row_packets, int& S, int& split_packets) {
    const int warps = ln.sms * 48;
    int want = (c->move_items * warps + T - 1) / T;
    const int max_s = (row_packets + kStep - 1) / kStep;
    if (want > max_s) want = max_s;
    if (want < 1) want = 1;
    split_packets = ((row_packets + want - 1) / want + kStep - 1) / kStep * kStep;
    S = (row_packets + split_packets - 1) / split_packets;
}

// Grid: one warp per item up to a few waves of resident blocks (more, shorter-lived blocks than fit at once
// measured faster than an exactly-resident persistent grid: finishing blocks are replaced at once).
template <typename K>
inline int mover_blocks(const piper_ctx* c, Lane ln, int items, K) {
    int blocks = cdiv(items, kMoveWarps);
    const int cap = ln.sms * c->move_cap;
    return blocks < cap ? (blocks < 1 ? 1 : blocks) : cap;
}

}  // namespace

int launch_scan_rank(piper_ctx* c, Lane ln, const int32_t* topk_idx, const float* gates, int32_t* counts, int32_t* offsets,
                     int32_t* row_of, int32_t* src_of, float* gate_rows) {
    const piper_moe_desc& D = c->D;
    const int n_assign = D.T * D.k;
    int32_t* chunk_counts = scan_scratch(c, ln.stream);  // per stream: forward chunks of two streams may overlap
    chunk_hist_kernel<<<c->n_chunks, kScanChunk, sizeof(int32_t) * D.E_loc, ln.stream>>>(topk_idx, n_assign, D.e_lo,
                                                                                        D.E_loc, chunk_counts);
    PIPER_LAUNCHED(c, "chunk_hist_kernel");
    scan_rank_kernel<<<c->n_chunks, kScanChunk, sizeof(int32_t) * (3 * D.E_loc + 1), ln.stream>>>(
        topk_idx, gates, n_assign, D.e_lo, D.E_loc, D.row_align, (int)piper_a_cap(&D), chunk_counts, counts, offsets, row_of,
        src_of, gate_rows);
    PIPER_LAUNCHED(c, "scan_rank_kernel");
    return PIPER_OK;
}

int launch_pack(piper_ctx* c, Lane ln, const void* x, const int32_t* offsets, const int32_t* row_of,
                const int32_t* src_of, void* xp) {
    const piper_moe_desc& D = c->D;
    const int a_cap = (int)piper_a_cap(&D);
    const int row_packets = (int)((size_t)D.d * esize(D.dtype) / 16);
    int S, split_packets;
    choose_split(c, ln, D.T, row_packets, S, split_packets);
    pack_kernel<<<mover_blocks(c, ln, D.T * S + a_cap, pack_kernel), kMoveWarps * 32, 0, ln.stream>>>(
        static_cast<const int4*>(x), offsets, row_of, src_of, D.T, D.k, D.E_loc, a_cap, row_packets, S, split_packets,
        static_cast<int4*>(xp));
    PIPER_LAUNCHED(c, "pack_kernel");
    return PIPER_OK;
}

int launch_combine(piper_ctx* c, Lane ln, const void* o, const int32_t* row_of, const float* gates, const void* s,
                   const void* s2, void* y, bool weighted) {
    const piper_moe_desc& D = c->D;
    const int row_packets = (int)((size_t)D.d * esize(D.dtype) / 16);
    int S, split_packets;
    choose_split(c, ln, D.T, row_packets, S, split_packets);
    const int items = D.T * S;
    const int4 *o4 = static_cast<const int4*>(o), *s4 = static_cast<const int4*>(s), *s24 = static_cast<const int4*>(s2);
    int4* y4 = static_cast<int4*>(y);
#define PIPER_COMBINE(BF, W, TW)                                                                          \
    combine_kernel<BF, W, TW><<<mover_blocks(c, ln, items, combine_kernel<BF, W, TW>), kMoveWarps * 32, 0, ln.stream>>>(o4, row_of, gates, s4, s24, D.T, D.k, row_packets, S, split_packets, y4)
    if (s2 != nullptr) {  // only B5 with the router's term carries a second addend
        if (weighted) return PIPER_ERR_INVALID;
        if (D.dtype == PIPER_DTYPE_BF16) PIPER_COMBINE(true, false, true); else PIPER_COMBINE(false, false, true);
    } else if (D.dtype == PIPER_DTYPE_BF16) {
        if (weighted) PIPER_COMBINE(true, true, false); else PIPER_COMBINE(true, false, false);
    } else {
        if (weighted) PIPER_COMBINE(false, true, false); else PIPER_COMBINE(false, false, false);
    }
#undef PIPER_COMBINE
    PIPER_LAUNCHED(c, "combine_kernel");
    return PIPER_OK;
}

int launch_combine_bwd(piper_ctx* c, Lane ln, const void* dy, const void* o, const int32_t* src_of,
                       const int32_t* row_of, const float* gates, const int32_t* offsets, void* d_o, float* dgates) {
    const piper_moe_desc& D = c->D;
    const int a_cap = (int)piper_a_cap(&D);
    const int row_packets = (int)((size_t)D.d * esize(D.dtype) / 16);
    const bool write_do = d_o != nullptr;  // NULL: dgates only (the fused chunk calls)
    const int items = D.T + (write_do ? a_cap : 0);
#define PIPER_CGRAD(BF, W)                                                                                             \
    combine_bwd_kernel<BF, W><<<mover_blocks(c, ln, items, combine_bwd_kernel<BF, W>), kMoveWarps * 32, 0, ln.stream>>>(      \
        static_cast<const int4*>(dy), static_cast<const int4*>(o), src_of, row_of, gates, offsets, D.T, D.k, D.E_loc,   \
        write_do ? a_cap : 0, row_packets, static_cast<int4*>(d_o), dgates)
    if (D.dtype == PIPER_DTYPE_BF16) {
        if (write_do) PIPER_CGRAD(true, true); else PIPER_CGRAD(true, false);
    } else {
        if (write_do) PIPER_CGRAD(false, true); else PIPER_CGRAD(false, false);
    }
#undef PIPER_CGRAD
    PIPER_LAUNCHED(c, "combine_bwd_kernel");
    return PIPER_OK;
}

}  // namespace piper

// ---- piper_dispatch_plan_static: F2 without a context, a workspace or any allocation -----------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
// the same two kernels as launch_scan_rank, with the chunk histograms - the one piece of scratch memory F2 needs - in a
// file-scope device array instead of the context's workspace.  Every GPU that loads the library holds the array
// (kStaticScratchBytes) until the process exits.  In host code `g_static_scratch` is only the host-side stand-in of the
// array, not a device address: its address on each device is looked up once, with that device current, through
// cudaGetSymbolAddress and kept.
namespace piper {
namespace {

constexpr size_t kStaticScratchBytes = 256 * 1024;  // 65536 chunk-histogram entries: n_chunks * E_loc of one call
constexpr int kStaticMaxDevices = 64;
static __device__ __align__(256) int32_t g_static_scratch[kStaticScratchBytes / sizeof(int32_t)];

std::mutex g_static_mutex;
int32_t* g_static_ptr[kStaticMaxDevices];  // device address of g_static_scratch on each device, nullptr = not looked up
thread_local char g_static_err[256] = "";

int static_fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_static_err, sizeof(g_static_err), fmt, ap);
    va_end(ap);
    return code;
}

}  // namespace
}  // namespace piper

extern "C" {

size_t piper_static_scratch_bytes(void) { return piper::kStaticScratchBytes; }
const char* piper_static_last_error(void) { return piper::g_static_err; }

int piper_dispatch_plan_static(const piper_moe_desc* D, const int32_t* topk_idx, const float* gates, int32_t* counts,
                               int32_t* offsets, int32_t* row_of, int32_t* src_of, float* gate_rows, void* stream) {
    using namespace piper;
    if (!D || D->T < 1 || D->k < 1 || D->E < 1 || D->E_loc < 1 || D->k > D->E || D->e_lo < 0 || D->e_lo + D->E_loc > D->E ||
        D->row_align < 1 || D->row_align > 1024 || (int64_t)D->T * D->k > (1ll << 30))
        return static_fail(PIPER_ERR_INVALID, "piper_dispatch_plan_static: invalid layer description");
    for (const void* p : {(const void*)topk_idx, (const void*)gates, (const void*)counts, (const void*)offsets,
                          (const void*)row_of, (const void*)src_of, (const void*)gate_rows})
        if (!p || (reinterpret_cast<uintptr_t>(p) & 15u))
            return static_fail(PIPER_ERR_INVALID, "piper_dispatch_plan_static: null or misaligned pointer");
    const int n_assign = D->T * D->k, n_chunks = cdiv(n_assign, kScanChunk);
    const size_t need = sizeof(int32_t) * (size_t)n_chunks * (size_t)D->E_loc;
    if (need > kStaticScratchBytes)
        return static_fail(PIPER_ERR_WORKSPACE,
                           "piper_dispatch_plan_static: ceil(T*k/%d) * E_loc = %d * %d histogram entries (%zu bytes) exceed the "
                           "static scratch of %zu bytes; use piper_dispatch_pack with a context",
                           kScanChunk, n_chunks, D->E_loc, need, kStaticScratchBytes);
    const size_t smem = sizeof(int32_t) * (3 * (size_t)D->E_loc + 1);
    if (smem > 48 * 1024)
        return static_fail(PIPER_ERR_UNSUPPORTED, "piper_dispatch_plan_static: E_loc = %d needs %zu bytes of shared memory", D->E_loc, smem);
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kStaticMaxDevices)
        return static_fail(PIPER_ERR_CUDA, "piper_dispatch_plan_static: no current CUDA device (or device id >= %d)", kStaticMaxDevices);
    int32_t* scratch;
    {
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_static_ptr[dev]) {  // once per device, with that device current
            void* p = nullptr;
            const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
            if (e != cudaSuccess || !p)
                return static_fail(PIPER_ERR_CUDA, "piper_dispatch_plan_static: cudaGetSymbolAddress failed on device %d: %s", dev,
                                   cudaGetErrorString(e));
            g_static_ptr[dev] = static_cast<int32_t*>(p);
        }
        scratch = g_static_ptr[dev];
    }
    // Nothing has to start at zero: chunk_hist_kernel writes every one of the n_chunks * E_loc entries that scan_rank_kernel
    // reads, so the contents the previous call left behind are never seen.
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int64_t kk = D->k < D->E_loc ? D->k : D->E_loc;
    const int a_cap = (int)((int64_t)D->T * kk + (int64_t)D->E_loc * (D->row_align - 1));
    chunk_hist_kernel<<<n_chunks, kScanChunk, sizeof(int32_t) * D->E_loc, s>>>(topk_idx, n_assign, D->e_lo, D->E_loc, scratch);
    scan_rank_kernel<<<n_chunks, kScanChunk, smem, s>>>(topk_idx, gates, n_assign, D->e_lo, D->E_loc, D->row_align, a_cap, scratch,
                                                        counts, offsets, row_of, src_of, gate_rows);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(PIPER_ERR_CUDA, "piper_dispatch_plan_static: launch failed: %s", cudaGetErrorString(e));
    g_static_err[0] = 0;
    return PIPER_OK;
}

}  // extern "C"
