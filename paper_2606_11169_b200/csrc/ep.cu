// ep.cu — N4 of SURVEY.md §8(f): expert parallelism over several GPUs with the pack / combine row movers fused with their
// all-to-all (`Shard` inserts an all-to-all before and after the expert Chunk).
//
// n_ranks GPUs; every rank holds T tokens and owns the E_loc = E / n_ranks experts [rank * E_loc, (rank + 1) * E_loc)
// (the context's e_lo / E_loc).  Instead of packing into a local send buffer and calling an all-to-all-v, the row movers
// address the owners' buffers directly through peer pointers (NVLink / NVSwitch peer memory: plain stores and loads):
//   1. F1 on every rank gives counts_global[E], the split sizes an all-to-all would announce; the ranks exchange them
//      (an all-gather of E integers per rank, by the caller: NCCL / torch.distributed) -> all_counts[n_ranks][E].
//   2. piper_ep_plan: from all_counts every rank derives, without further communication, the layout of every owner's
//      receive buffer (the rows of an expert ordered by (source rank, token), i.e. by global token id rank * T + t,
//      segments padded to row_align: exactly the buffer piper_dispatch_pack builds over the concatenated tokens), its own
//      experts' counts / offsets, and send_base[e] = the row where its own rows of expert e start in the owner's buffer.
//   3. piper_ep_dispatch: ranks its assignments (deterministic, stable by token, as F2) and stores the token rows, the
//      global assignment ids and the gates straight into the owners' buffers; dest_row[T,k] remembers where each went.
//      piper_ep_finish_recv (owner side) fills the pad rows.
//   4. the owners run the grouped expert FFN on what they received (the existing entry points);
//   5. piper_ep_combine gathers the expert outputs from the owners' buffers, gate-weighted (F5); backward mirrors it:
//      piper_ep_dispatch_bwd scatters gate * dY and gathers the dgates dot products, piper_ep_unpack gathers dXp.
// No kernel waits on another rank's kernel: the steps are ordered by the caller's stream / collective as usual, so the
// whole protocol also runs with all ranks on one GPU (tests) or with peer pointers obtained from CUDA IPC / symmetric memory.
#include "piper_internal.cuh"

namespace piper {
namespace {

constexpr int kEpWarps = 8;

// ---- plan: one block, thread e < E ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512)
ep_plan_kernel(const int32_t* __restrict__ all_counts, int E, int E_loc, int rank, int n_ranks, int row_align,
               int32_t* __restrict__ counts, int32_t* __restrict__ offsets, int32_t* __restrict__ send_base) {
    __shared__ int32_t padded[kMaxE], excl[kMaxE];
    const int e = threadIdx.x;
    int total = 0, before = 0;
    if (e < E) {
        for (int r = 0; r < n_ranks; ++r) {
            const int v = all_counts[(size_t)r * E + e];
            if (r < rank) before += v;
            total += v;
        }
        padded[e] = (total + row_align - 1) / row_align * row_align;
    }
    __syncthreads();
    if (e < E) {  // exclusive scan inside the owner's expert range (E_loc <= 512 terms: a short serial walk per thread)
        const int o_lo = e / E_loc * E_loc;
        int x = 0;
        for (int i = o_lo; i < e; ++i) x += padded[i];
        excl[e] = x;
        send_base[e] = x + before;
        if (e / E_loc == rank) {
            counts[e - o_lo] = total, offsets[e - o_lo] = x;
            if (e - o_lo == E_loc - 1) offsets[E_loc] = x + padded[e];
        }
    }
}

// ---- dispatch phase 1: chunk histograms over all E experts (permute.cu's scheme with e_lo = 0, E_loc = E) -----------------
__global__ void __launch_bounds__(kScanChunk)
ep_hist_kernel(const int32_t* __restrict__ topk_idx, int n_assign, int E, int32_t* __restrict__ chunk_counts) {
    extern __shared__ int32_t hist[];
    for (int e = threadIdx.x; e < E; e += blockDim.x) hist[e] = 0;
    __syncthreads();
    const int a = blockIdx.x * kScanChunk + threadIdx.x;
    if (a < n_assign) atomicAdd(&hist[topk_idx[a]], 1);  // integer count: order-independent
    __syncthreads();
    for (int e = threadIdx.x; e < E; e += blockDim.x) chunk_counts[(size_t)blockIdx.x * E + e] = hist[e];
}

// ---- dispatch phase 2: stable rank of every assignment inside its expert, destination row in the owner's buffer; the
// assignment's global id and gate are stored there (peer stores) ---------------------------------------------------------------
__global__ void __launch_bounds__(kScanChunk)
ep_rank_kernel(const int32_t* __restrict__ topk_idx, const float* __restrict__ gates, int n_assign, int E, int E_loc, int k,
               long long first_assignment, const int32_t* __restrict__ chunk_counts, const int32_t* __restrict__ send_base,
               int32_t* const* __restrict__ peer_src_of, float* const* __restrict__ peer_gate_rows,
               int32_t* __restrict__ dest_row) {
    extern __shared__ int32_t run[];
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        int base = send_base[e];
        for (int c = 0; c < (int)blockIdx.x; ++c) base += chunk_counts[(size_t)c * E + e];
        run[e] = base;
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int a = blockIdx.x * kScanChunk + threadIdx.x;
    const int e = a < n_assign ? topk_idx[a] : -1;
    const unsigned peers = __match_any_sync(0xffffffffu, e);
    const int below = __popc(peers & ((1u << lane) - 1u));
    const int leader = __ffs(peers) - 1;
    int row = -1;
    for (int turn = 0; turn < kScanChunk / 32; ++turn) {
        if (turn == w && e >= 0) {
            int b0 = 0;
            if (lane == leader) {
                b0 = run[e];
                run[e] = b0 + __popc(peers);
            }
            b0 = __shfl_sync(peers, b0, leader);
            row = b0 + below;
        }
        __syncthreads();
    }
    if (a < n_assign) {
        dest_row[a] = row;
        const int o = e / E_loc;
        peer_src_of[o][row] = (int32_t)(first_assignment + a);  // global assignment id (rank * T + t) * k + j
        peer_gate_rows[o][row] = gates[a];
    }
}

// ---- owner side: pad rows of the received buffers ------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
ep_finish_kernel(const int32_t* __restrict__ counts, const int32_t* __restrict__ offsets, int E_loc, int a_cap, int row_packets,
                 int32_t* __restrict__ src_of, float* __restrict__ gate_rows, int4* __restrict__ xp) {
    const int lane = threadIdx.x & 31;
    const int warp = blockIdx.x * 8 + (threadIdx.x >> 5), nwarps = gridDim.x * 8;
    const int used = offsets[E_loc];
    for (int g = 0; g < E_loc; ++g)
        for (int r = offsets[g] + counts[g] + warp; r < offsets[g + 1]; r += nwarps) {
            if (lane == 0) src_of[r] = -1, gate_rows[r] = 0.f;
            int4* dst = xp + (size_t)r * row_packets;
            for (int p = lane; p < row_packets; p += 32) st16(dst + p, make_int4(0, 0, 0, 0));
        }
    for (int r = used + blockIdx.x * blockDim.x + threadIdx.x; r < a_cap; r += gridDim.x * blockDim.x) src_of[r] = -1;
}

template <bool BF16>
__device__ __forceinline__ void scale_packet(int4& v, float w) {
    if (BF16) {
        uint32_t u[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float2 f = bf2_to_f2(u[q]);
            u[q] = f2_to_bf2(w * f.x, w * f.y);
        }
        v = make_int4((int)u[0], (int)u[1], (int)u[2], (int)u[3]);
    } else {
        v.x = __float_as_int(w * __int_as_float(v.x)), v.y = __float_as_int(w * __int_as_float(v.y));
        v.z = __float_as_int(w * __int_as_float(v.z)), v.w = __float_as_int(w * __int_as_float(v.w));
    }
}
template <bool BF16>
__device__ __forceinline__ float dot_packet(const int4& a, const int4& b) {
    float s = 0.f;
    if (BF16) {
        const uint32_t ua[4] = {(uint32_t)a.x, (uint32_t)a.y, (uint32_t)a.z, (uint32_t)a.w};
        const uint32_t ub[4] = {(uint32_t)b.x, (uint32_t)b.y, (uint32_t)b.z, (uint32_t)b.w};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float2 fa = bf2_to_f2(ua[q]), fb = bf2_to_f2(ub[q]);
            s = fmaf(fa.x, fb.x, s), s = fmaf(fa.y, fb.y, s);
        }
    } else {
        s = fmaf(__int_as_float(a.x), __int_as_float(b.x), s), s = fmaf(__int_as_float(a.y), __int_as_float(b.y), s);
        s = fmaf(__int_as_float(a.z), __int_as_float(b.z), s), s = fmaf(__int_as_float(a.w), __int_as_float(b.w), s);
    }
    return s;
}

// ---- scatter: a warp per token; row t of `src` goes to peer_dst[owner(slot)][dest_row[t, slot]] for each of the k slots,
// SCALED by the slot's gate when BWD (d_o = gate * dY), and BWD also gathers dgates[t, slot] = <src[t], peer_o[owner][row]> ------
template <bool BF16, bool BWD>
__global__ void __launch_bounds__(kEpWarps * 32)
ep_scatter_kernel(const int4* __restrict__ src, const int32_t* __restrict__ topk_idx, const int32_t* __restrict__ dest_row,
                  const float* __restrict__ gates, int T, int k, int E_loc, int row_packets, int4* const* __restrict__ peer_dst,
                  const int4* const* __restrict__ peer_o, float* __restrict__ dgates) {
    const int lane = threadIdx.x & 31;
    const int warp = blockIdx.x * kEpWarps + (threadIdx.x >> 5), nwarps = gridDim.x * kEpWarps;
    for (int t = warp; t < T; t += nwarps) {
        const int4* s = src + (size_t)t * row_packets;
        for (int j = 0; j < k; ++j) {
            const int o = topk_idx[(size_t)t * k + j] / E_loc, row = dest_row[(size_t)t * k + j];
            const float w = BWD ? gates[(size_t)t * k + j] : 1.f;
            int4* dst = peer_dst[o] + (size_t)row * row_packets;
            const int4* orow = BWD ? peer_o[o] + (size_t)row * row_packets : nullptr;
            float dot = 0.f;
            for (int p = lane; p < row_packets; p += 32) {
                int4 v = __ldg(s + p);
                if (BWD) {
                    dot += dot_packet<BF16>(v, ld_nc16(orow + p));
                    scale_packet<BF16>(v, w);
                }
                st16(dst + p, v);
            }
            if (BWD) {
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, off);
                if (lane == 0) dgates[(size_t)t * k + j] = dot;
            }
        }
    }
}

// ---- gather: y[t] = sum_j w_j * peer_src[owner(slot j)][dest_row[t, j]] (+ s[t]); w_j = gates (combine) or 1 (unpack);
// fp32 accumulation in slot order then s, one rounding (the arithmetic of combine_kernel) ----------------------------------------
template <bool BF16, bool WEIGHTED>
__global__ void __launch_bounds__(kEpWarps * 32)
ep_gather_kernel(const int4* const* __restrict__ peer_src, const int32_t* __restrict__ topk_idx,
                 const int32_t* __restrict__ dest_row, const float* __restrict__ gates, const int4* __restrict__ s, int T, int k,
                 int E_loc, int row_packets, int4* __restrict__ y) {
    const int lane = threadIdx.x & 31;
    const int warp = blockIdx.x * kEpWarps + (threadIdx.x >> 5), nwarps = gridDim.x * kEpWarps;
    for (int t = warp; t < T; t += nwarps) {
        for (int p = lane; p < row_packets; p += 32) {
            float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            for (int j = 0; j < k; ++j) {
                const int o = topk_idx[(size_t)t * k + j] / E_loc, row = dest_row[(size_t)t * k + j];
                const float w = WEIGHTED ? gates[(size_t)t * k + j] : 1.f;
                const int4 v = ld_nc16(peer_src[o] + (size_t)row * row_packets + p);
                if (BF16) {
                    const uint32_t u[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const float2 f = bf2_to_f2(u[q]);
                        acc[2 * q] = fmaf(w, f.x, acc[2 * q]), acc[2 * q + 1] = fmaf(w, f.y, acc[2 * q + 1]);
                    }
                } else {
                    acc[0] = fmaf(w, __int_as_float(v.x), acc[0]), acc[1] = fmaf(w, __int_as_float(v.y), acc[1]);
                    acc[2] = fmaf(w, __int_as_float(v.z), acc[2]), acc[3] = fmaf(w, __int_as_float(v.w), acc[3]);
                }
            }
            if (s) {
                const int4 v = ld_nc16(s + (size_t)t * row_packets + p);
                if (BF16) {
                    const uint32_t u[4] = {(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const float2 f = bf2_to_f2(u[q]);
                        acc[2 * q] += f.x, acc[2 * q + 1] += f.y;
                    }
                } else {
                    acc[0] += __int_as_float(v.x), acc[1] += __int_as_float(v.y);
                    acc[2] += __int_as_float(v.z), acc[3] += __int_as_float(v.w);
                }
            }
            int4 r;
            if (BF16) {
                r.x = (int)f2_to_bf2(acc[0], acc[1]), r.y = (int)f2_to_bf2(acc[2], acc[3]);
                r.z = (int)f2_to_bf2(acc[4], acc[5]), r.w = (int)f2_to_bf2(acc[6], acc[7]);
            } else {
                r.x = __float_as_int(acc[0]), r.y = __float_as_int(acc[1]), r.z = __float_as_int(acc[2]), r.w = __float_as_int(acc[3]);
            }
            st16(y + (size_t)t * row_packets + p, r);
        }
    }
}

bool ep_ok(const piper_ctx* c, int rank, int n_ranks) {
    const piper_moe_desc& D = c->D;
    return n_ranks >= 1 && n_ranks <= 64 && rank >= 0 && rank < n_ranks && D.E % n_ranks == 0 && D.E_loc == D.E / n_ranks &&
           D.e_lo == rank * D.E_loc && (long long)D.T * n_ranks * D.k < (1ll << 31);
}
inline int ep_blocks(Lane ln, int T) {
    const int b = cdiv(T, kEpWarps), cap = ln.sms * 8;
    return b < cap ? (b < 1 ? 1 : b) : cap;
}

}  // namespace
}  // namespace piper

using namespace piper;

extern "C" {

int64_t piper_ep_a_cap(const piper_moe_desc* D, int n_ranks) {
    if (!D || n_ranks < 1) return 0;
    const int64_t kk = D->k < D->E_loc ? D->k : D->E_loc;
    return (int64_t)D->T * n_ranks * kk + (int64_t)D->E_loc * (D->row_align - 1);
}

// Host restatement of ep_plan_kernel (no GPU): for callers that size messages on the host and for the CPU tests.
int piper_ep_plan_host(const int32_t* all_counts, int32_t E, int32_t n_ranks, int32_t rank, int32_t row_align, int32_t* counts,
                       int32_t* offsets, int32_t* send_base) {
    if (!all_counts || !counts || !offsets || !send_base || n_ranks < 1 || rank < 0 || rank >= n_ranks || E < 1 || E % n_ranks ||
        row_align < 1)
        return PIPER_ERR_INVALID;
    const int E_loc = E / n_ranks;
    for (int o = 0; o < n_ranks; ++o) {
        int at = 0;
        for (int i = 0; i < E_loc; ++i) {
            const int e = o * E_loc + i;
            int total = 0, before = 0;
            for (int r = 0; r < n_ranks; ++r) {
                if (r < rank) before += all_counts[(size_t)r * E + e];
                total += all_counts[(size_t)r * E + e];
            }
            send_base[e] = at + before;
            if (o == rank) counts[i] = total, offsets[i] = at;
            at += (total + row_align - 1) / row_align * row_align;
        }
        if (o == rank) offsets[E_loc] = at;
    }
    return PIPER_OK;
}

int piper_ep_plan(piper_ctx* c, const int32_t* all_counts, int rank, int n_ranks, int32_t* counts, int32_t* offsets,
                  int32_t* send_base, void* stream) {
    if (!c || !ep_ok(c, rank, n_ranks) || !aligned16(all_counts) || !aligned16(counts) || !aligned16(offsets) || !aligned16(send_base))
        return PIPER_ERR_INVALID;
    ep_plan_kernel<<<1, 512, 0, static_cast<cudaStream_t>(stream)>>>(all_counts, c->D.E, c->D.E_loc, rank, n_ranks, c->D.row_align,
                                                                     counts, offsets, send_base);
    PIPER_LAUNCHED(c, "ep_plan_kernel");
    return PIPER_OK;
}

int piper_ep_dispatch(piper_ctx* c, const void* x, const int32_t* topk_idx, const float* gates, const int32_t* send_base, int rank,
                      int n_ranks, void* const* peer_xp, int32_t* const* peer_src_of, float* const* peer_gate_rows,
                      int32_t* dest_row, void* stream) {
    if (!c || !ep_ok(c, rank, n_ranks) || !aligned16(x) || !aligned16(topk_idx) || !aligned16(gates) || !aligned16(send_base) ||
        !peer_xp || !peer_src_of || !peer_gate_rows || !aligned16(dest_row))
        return PIPER_ERR_INVALID;
    const piper_moe_desc& D = c->D;
    const Lane ln{static_cast<cudaStream_t>(stream), c->num_sms};
    const int n_assign = D.T * D.k;
    int32_t* hist = c->ep_scratch;  // [n_chunks][E]; one dispatch of a context at a time (stream-ordered)
    ep_hist_kernel<<<c->n_chunks, kScanChunk, sizeof(int32_t) * D.E, ln.stream>>>(topk_idx, n_assign, D.E, hist);
    PIPER_LAUNCHED(c, "ep_hist_kernel");
    ep_rank_kernel<<<c->n_chunks, kScanChunk, sizeof(int32_t) * D.E, ln.stream>>>(
        topk_idx, gates, n_assign, D.E, D.E_loc, D.k, (long long)rank * n_assign, hist, send_base, peer_src_of, peer_gate_rows,
        dest_row);
    PIPER_LAUNCHED(c, "ep_rank_kernel");
    const int row_packets = (int)((size_t)D.d * esize(D.dtype) / 16);
    int4* const* dst = reinterpret_cast<int4* const*>(peer_xp);
    if (D.dtype == PIPER_DTYPE_BF16)
        ep_scatter_kernel<true, false><<<ep_blocks(ln, D.T), kEpWarps * 32, 0, ln.stream>>>(
            static_cast<const int4*>(x), topk_idx, dest_row, gates, D.T, D.k, D.E_loc, row_packets, dst, nullptr, nullptr);
    else
        ep_scatter_kernel<false, false><<<ep_blocks(ln, D.T), kEpWarps * 32, 0, ln.stream>>>(
            static_cast<const int4*>(x), topk_idx, dest_row, gates, D.T, D.k, D.E_loc, row_packets, dst, nullptr, nullptr);
    PIPER_LAUNCHED(c, "ep_scatter_kernel");
    return PIPER_OK;
}

int piper_ep_finish_recv(piper_ctx* c, const int32_t* counts, const int32_t* offsets, int n_ranks, int32_t* src_of, float* gate_rows,
                         void* xp, void* stream) {
    if (!c || n_ranks < 1 || !aligned16(counts) || !aligned16(offsets) || !aligned16(src_of) || !aligned16(gate_rows) || !aligned16(xp))
        return PIPER_ERR_INVALID;
    const piper_moe_desc& D = c->D;
    const int row_packets = (int)((size_t)D.d * esize(D.dtype) / 16);
    ep_finish_kernel<<<c->num_sms, 256, 0, static_cast<cudaStream_t>(stream)>>>(
        counts, offsets, D.E_loc, (int)piper_ep_a_cap(&D, n_ranks), row_packets, src_of, gate_rows, static_cast<int4*>(xp));
    PIPER_LAUNCHED(c, "ep_finish_kernel");
    return PIPER_OK;
}

static int ep_gather(piper_ctx* c, void* const* peer_src, const int32_t* topk_idx, const int32_t* dest_row, const float* gates,
                     const void* s, void* y, bool weighted, void* stream) {
    if (!c || !peer_src || !aligned16(topk_idx) || !aligned16(dest_row) || !aligned16(y) || (weighted && !aligned16(gates)) ||
        (s && !aligned16(s)))
        return PIPER_ERR_INVALID;
    const piper_moe_desc& D = c->D;
    const Lane ln{static_cast<cudaStream_t>(stream), c->num_sms};
    const int row_packets = (int)((size_t)D.d * esize(D.dtype) / 16);
    const int4* const* src = reinterpret_cast<const int4* const*>(peer_src);
#define PIPER_EP_GATHER(BF, W)                                                                                             \
    ep_gather_kernel<BF, W><<<ep_blocks(ln, D.T), kEpWarps * 32, 0, ln.stream>>>(src, topk_idx, dest_row, gates,          \
                                                                                static_cast<const int4*>(s), D.T, D.k, \
                                                                                D.E_loc, row_packets, static_cast<int4*>(y))
    if (D.dtype == PIPER_DTYPE_BF16) {
        if (weighted) PIPER_EP_GATHER(true, true); else PIPER_EP_GATHER(true, false);
    } else {
        if (weighted) PIPER_EP_GATHER(false, true); else PIPER_EP_GATHER(false, false);
    }
#undef PIPER_EP_GATHER
    PIPER_LAUNCHED(c, "ep_gather_kernel");
    return PIPER_OK;
}

int piper_ep_combine(piper_ctx* c, void* const* peer_o, const int32_t* topk_idx, const int32_t* dest_row, const float* gates,
                     const void* s, void* y, void* stream) {
    return ep_gather(c, peer_o, topk_idx, dest_row, gates, s, y, true, stream);
}

int piper_ep_unpack(piper_ctx* c, void* const* peer_dxp, const int32_t* topk_idx, const int32_t* dest_row, const void* dx_shared,
                    void* dx, void* stream) {
    return ep_gather(c, peer_dxp, topk_idx, dest_row, nullptr, dx_shared, dx, false, stream);
}

int piper_ep_dispatch_bwd(piper_ctx* c, const void* dy, const int32_t* topk_idx, const int32_t* dest_row, const float* gates,
                          void* const* peer_o, void* const* peer_d_o, float* dgates, void* stream) {
    if (!c || !aligned16(dy) || !aligned16(topk_idx) || !aligned16(dest_row) || !aligned16(gates) || !peer_o || !peer_d_o ||
        !aligned16(dgates))
        return PIPER_ERR_INVALID;
    const piper_moe_desc& D = c->D;
    const Lane ln{static_cast<cudaStream_t>(stream), c->num_sms};
    const int row_packets = (int)((size_t)D.d * esize(D.dtype) / 16);
    int4* const* dst = reinterpret_cast<int4* const*>(peer_d_o);
    const int4* const* o = reinterpret_cast<const int4* const*>(peer_o);
    if (D.dtype == PIPER_DTYPE_BF16)
        ep_scatter_kernel<true, true><<<ep_blocks(ln, D.T), kEpWarps * 32, 0, ln.stream>>>(
            static_cast<const int4*>(dy), topk_idx, dest_row, gates, D.T, D.k, D.E_loc, row_packets, dst, o, dgates);
    else
        ep_scatter_kernel<false, true><<<ep_blocks(ln, D.T), kEpWarps * 32, 0, ln.stream>>>(
            static_cast<const int4*>(dy), topk_idx, dest_row, gates, D.T, D.k, D.E_loc, row_packets, dst, o, dgates);
    PIPER_LAUNCHED(c, "ep_scatter_kernel");
    return PIPER_OK;
}

}  // extern "C"
