// gemm_tc.cu — grouped SwiGLU expert-FFN GEMMs on the 5th-generation tensor cores (F4, B2-B4 of SURVEY.md
// §8a; BASELINE.json:north_star part 3).  bf16 x bf16 -> fp32 accumulation in TMEM, one rounding to bf16
// per stored tensor (SURVEY.md §8c "Error budget").
//
// Three persistent, warp-specialised kernel templates, all with
//   warp 0  : TMA producer (cp.async.bulk.tensor, 128-byte swizzle) into a shared-memory ring
//   warp 1  : single-thread tcgen05.mma issuer, tcgen05.commit hand-off to the ring and to the epilogue
//   warp 2  : TMEM allocator (512 columns = two fp32 accumulators: the epilogue of tile i overlaps the main
//             loop of tile i+1)
//   warps 4-7: epilogue, tcgen05.ld TMEM -> registers -> fused math -> global
//  tc_gemmT_kernel  rows-on-N CTA pair (cta_group::2): fwd1, fwd2, dgrad1, dgrad2.  Weights on M (256 features per
//                   pair), the expert's rows on N in multiples of 16; transposing TMA-store epilogues.
//  tc_gemm2_kernel  CTA pair, 256 x 256 tiles: wgrad (K = the expert's rows, both operands MN-major, K blocks of
//                   128); TMEM -> swizzled shared memory -> TMA-store epilogue.  Also the rows-on-M form of the
//                   four contractions above (PIPER_OPT_TC_ROWS_ON_N = 0).
//  tc_gemm_kernel   1-CTA 128 x 256 tiles, direct-store epilogue: fallback (> 192 groups, PIPER_OPT_TC_2CTA = 0).
// Operand layouts are taken as they lie in memory (no transposed copies): the descriptors select K-major
// or MN-major per operand.  In the rows-on-M form:
//   fwd1   G|U = Xp Wg | Xp Wu      A K-major  (Xp [rows,d]),   B MN-major (W [d,I], two 128-col halves)
//   fwd2   O   = H Wd               A K-major  (H  [rows,I]),   B MN-major (Wd [I,d])
//   dgrad1 dH  = dO Wd^T            A K-major  (dO [rows,d]),   B K-major  (Wd [I,d])
//   dgrad2 dXp = dG Wg^T + dU Wu^T  A K-major  (dG,dU [rows,I]),B K-major  (Wg,Wu [d,I]); K runs over both
//   wgrad  dWg|dWu = Xp^T dG|dU ; dWd = H^T dO    A, B MN-major (row buffers), K = the expert's rows
// (rows-on-N: the same products transposed, the weight operand first.)
// Ragged groups: segments are padded to row_align = 128 rows (pad rows are zero in every row buffer), so
// an M tile never straddles two experts and the ragged K of wgrad is a whole number of tiles; the tile ->
// expert map is computed on the device from `offsets` / `counts` (no host read-back).  Tails in d / I / T are
// handled by TMA zero fill on loads and TMA clipping / bounds checks on stores.
#include "piper_internal.cuh"

namespace piper {
namespace {

constexpr int BM = 128, BN = 256, BK = 64, UK = 16, STAGES = 4;
constexpr int A_BYTES = BM * BK * 2, B_BYTES = BN * BK * 2, STAGE_BYTES = A_BYTES + B_BYTES;
constexpr int MN_BLOCK_BYTES = 64 * BK * 2;  // one 64(MN) x 64(K) box of an MN-major operand
constexpr int kThreads = 256;
constexpr int kMaxGroups = kMaxE;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 256 /*barriers*/ +
                           (kMaxGroups + 1) * 4 /*tile prefix*/;
constexpr int kProfSlots = 16, kProfSlotWords = 160 * 8;  // debug counters: 16 launches x 160 CTAs x 8 words
constexpr int PANEL_M = 8;  // M tiles per panel of the tile order (L2 reuse of the weight tile)

enum : int { K_MAJOR = 0, MN_MAJOR = 1 };
enum : int { EPI_SWIGLU_FWD = 0, EPI_STORE = 1, EPI_SWIGLU_BWD = 2, EPI_WGRAD_SPLIT = 3, EPI_WGRAD = 4, EPI_STORE_F32 = 5 };

struct alignas(64) TcParams {
    CUtensorMap a[2], b[2];
    CUtensorMap bs[2];         // rows-on-N kernel: the activation operand again with 32-row boxes (short chunks)
    CUtensorMap o[3], ein[2];  // CTA-pair kernel: outputs / epilogue inputs as 64-column x 32-row store / load boxes
    CUtensorMap ow[2];         // CTA-pair wgrad with the store warp: the dW outputs as 64-column x 128-row boxes
    const int32_t* offsets;  // [G+1] device
    int G;
    int ragged_m;    // 1: tiles run over the packed rows (fwd / dgrad); 0: over groups (wgrad)
    int n_tiles;     // tiles along N
    int m_tiles;     // wgrad: tiles along M per group
    int kb_per_src;  // ragged_m: K blocks per source
    int n_src;       // 1, or 2 when K runs over two (A, B) pairs (dgrad2)
    int b_split;     // B tile = [b[0]: 128 columns | b[1]: 128 columns] (fwd1, wgrad gate|up)
    int tile_n;      // output columns per tile (128 when split, else 256)
    int m_limit;     // wgrad: rows of one dW matrix
    int n_limit;     // columns of the outputs
    long long ld;            // leading dimension of outputs / epilogue inputs (elements)
    long long group_stride;  // wgrad: elements between two experts' dW
    __nv_bfloat16 *out0, *out1, *out2;
    const __nv_bfloat16 *in0, *in1;
    int store_warp;   // CTA-pair wgrad, bf16 dW: one 128-row bulk store per chunk from warp 2 (long K ranges), see Cfg2::STORE_WARP
    long long* prof;  // debug (PIPER_OPT_TC_PROFILE): [gridDim.x][8] wait-cycle counters, else NULL
    // rows-on-N kernel (tc_gemmT_kernel)
    const int32_t* counts;  // [G] device: real rows per group
    int f_tiles;            // tiles along the feature (output column) dimension
    int f_limit;            // output columns
    int* sched;             // rows-on-N kernel: {next tile, clusters done} counters of this launch (both 0 between launches)
    int out_f32;            // wgrad: dW is fp32 (o[] are fp32 maps, 32-column boxes); accum: add into dW (TMA reduce)
    int accum;
    int greedy;             // chunking: 1 = 256-row chunks and a short last one, 0 = equal chunks
    const float* bias;      // EPI_STORE_F32: added per output column (router logits), or NULL
    // N2 fusion (GATHER kernels): the packed row r of an operand is row src_of[r] / k of a token-major tensor (x or dY),
    // gathered by cp.async straight into the operand tile; pad rows (src_of < 0) are zero-filled
    const int32_t* src_of;      // [rows] flat assignment id of each packed row, -1 = pad
    const void* gsrc;           // token-major source [T, g_cols] bf16
    unsigned long long g_magic; // ceil(2^35 / k): a / k = (a * g_magic) >> 35 for a < 2^30, k <= 8
    int g_cols;                 // columns of the source (= the contraction / feature length d)
    const float* row_scale;     // DGRAD1 with gathered dY: the epilogue multiplies row r of dH by row_scale[r] (the gate)
    int small_rows;         // chunks of at most this many rows per CTA load 32-row activation boxes
};

// ---- PTX wrappers ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
// the same wait with cluster-scope acquire: pairs with a peer CTA's st.shared::cluster + mbarrier.arrive.release.cluster
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
// 16-byte asynchronous copy global -> shared (LDGSTS); src_bytes = 0 writes zeros (the source is not read)
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint32_t src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
// the same with a predicate: ignore != 0 writes zeros and does not read the source
__device__ __forceinline__ void cp_async16_z(uint32_t dst, const void* src, uint32_t ignore) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\tcp.async.cg.shared.global [%0], [%1], 16, p;\n\t}" ::"r"(dst), "l"(src), "r"(ignore) : "memory");
}
// the mbarrier receives one arrival from this thread once all its cp.async issued so far have landed
__device__ __forceinline__ void cp_async_arrive(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// One lane of a converged warp (elect.sync).  Code that issues tcgen05.mma / bulk tensor copies runs warp-uniformly up to
// this predicate: the operands of those instructions live in uniform registers, and inside an `if (lane == 0)` region the
// compiler cannot prove uniformity and wraps every such instruction in a loop of R2UR broadcasts (~25 instructions per
// MMA, ~130 cycles of issue time per MMA whatever its shape: profiles/r2_tc_wait_cycles.md).
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
// a value every lane holds, made provably warp-uniform for the compiler
__device__ __forceinline__ int uni(int v) { return __shfl_sync(0xffffffffu, v, 0); }
__device__ __forceinline__ uint32_t uni(uint32_t v) { return __shfl_sync(0xffffffffu, v, 0); }
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t* dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst_smem)), "r"(cols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem], 128 x 256 x 16, bf16 inputs, fp32 accumulate
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
        : "memory");
}
// mbarrier arrives once every tcgen05 operation issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
// 16 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}
// wait for the loads above; the registers are in/out operands so that no use is scheduled before the wait
__device__ __forceinline__ void tmem_ld_wait(uint32_t (&r)[16]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
                   "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15])
                 :
                 : "memory");
}

// Shared-memory matrix descriptor (tcgen05 "matrix descriptor", version 1, 128-byte swizzle).
//  K-major : rows of 64 elements (128 B), 8-row swizzle atoms 1024 B apart (SBO); LBO unused.
//  MN-major: 64(MN) x 8(K) atoms of 1024 B; SBO = 1024 B between 8-K groups, LBO = bytes between 64-wide MN blocks.
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
    d |= (uint64_t)1 << 46;  // descriptor version (Blackwell)
    d |= (uint64_t)2 << 61;  // SWIZZLE_128B
    return d;
}
// Instruction descriptor: D fp32, A/B bf16, M = 128, N = 256, majors per operand.
__host__ __device__ constexpr uint32_t make_idesc(int a_major, int b_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_major << 15) | ((uint32_t)b_major << 16) |
           ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}

// ---- tile schedule (identical in every role) ----------------------------------------------------------
struct Tile {
    int g;    // group (expert)
    int m0;   // ragged_m: first packed row of the tile; wgrad: first row of dW
    int n0;   // first output column
    int k0;   // wgrad: first packed row of the group's K range
    int nkb;  // K blocks of this tile
};

// tp[g] = first M tile of group g (ragged_m), tp[G] = number of M tiles.
__device__ __forceinline__ int total_tiles(const TcParams& P, const int* tp) {
    return P.ragged_m ? tp[P.G] * P.n_tiles : P.G * P.m_tiles * P.n_tiles;
}

__device__ __forceinline__ Tile decode_tile(const TcParams& P, const int* tp, const int32_t* __restrict__ offsets, int t) {
    Tile r;
    if (P.ragged_m) {
        // group-major; inside a group panels of PANEL_M M tiles; inside a panel N-major with M fastest, so
        // the CTAs of one wave share a few weight tiles (L2) and the panel's rows stay L2-resident.
        int g = 0;
        while (g + 1 < P.G && tp[g + 1] * P.n_tiles <= t) ++g;
        const int local = t - tp[g] * P.n_tiles, mg = tp[g + 1] - tp[g];
        const int per_panel = PANEL_M * P.n_tiles;
        const int panel = local / per_panel, rem = local - panel * per_panel;
        const int pm = min(PANEL_M, mg - panel * PANEL_M);
        const int nt = rem / pm, mt = tp[g] + panel * PANEL_M + (rem - nt * pm);
        r.g = g, r.m0 = mt * BM, r.n0 = nt * P.tile_n, r.k0 = 0, r.nkb = P.kb_per_src * P.n_src;
    } else {
        const int per_group = P.m_tiles * P.n_tiles;
        const int g = t / per_group, local = t - g * per_group;
        const int nt = local / P.m_tiles, mt = local - nt * P.m_tiles;
        const int lo = offsets[g], hi = offsets[g + 1];
        // n_src = 2 (dense dW_r = x^T dz_hi + x^T dz_lo): the K range is walked once per (A, B) pair, kb_per_src blocks each
        r.g = g, r.m0 = mt * BM, r.n0 = nt * P.tile_n, r.k0 = lo, r.nkb = (hi - lo + BK - 1) / BK * P.n_src;
    }
    return r;
}

// ---- epilogue helpers ---------------------------------------------------------------------------------
__device__ __forceinline__ uint4 pack8(const float* v) {
    uint4 r;
    r.x = f2_to_bf2(v[0], v[1]), r.y = f2_to_bf2(v[2], v[3]), r.z = f2_to_bf2(v[4], v[5]), r.w = f2_to_bf2(v[6], v[7]);
    return r;
}
__device__ __forceinline__ void unpack8(const uint4& q, float* v) {
    float2 f;
    f = bf2_to_f2(q.x), v[0] = f.x, v[1] = f.y;
    f = bf2_to_f2(q.y), v[2] = f.x, v[3] = f.y;
    f = bf2_to_f2(q.z), v[4] = f.x, v[5] = f.y;
    f = bf2_to_f2(q.w), v[6] = f.x, v[7] = f.y;
}
__device__ __forceinline__ float sigmoidf_fast(float x) { return __fdividef(1.f, 1.f + __expf(-x)); }

// 16 output columns [col, col+16) of one row: store the halves that lie below n_limit (n_limit % 8 == 0).
__device__ __forceinline__ void store16(__nv_bfloat16* row_ptr, int col, int n_limit, const float* v) {
    if (col < n_limit) *reinterpret_cast<uint4*>(row_ptr + col) = pack8(v);
    if (col + 8 < n_limit) *reinterpret_cast<uint4*>(row_ptr + col + 8) = pack8(v + 8);
}
__device__ __forceinline__ void load16(const __nv_bfloat16* row_ptr, int col, int n_limit, float* v) {
    uint4 q0 = make_uint4(0, 0, 0, 0), q1 = q0;
    if (col < n_limit) q0 = *reinterpret_cast<const uint4*>(row_ptr + col);
    if (col + 8 < n_limit) q1 = *reinterpret_cast<const uint4*>(row_ptr + col + 8);
    unpack8(q0, v), unpack8(q1, v + 8);
}

// One accumulator tile (this thread's TMEM lane = one output row) -> fused math -> global.
template <int EPI>
__device__ __forceinline__ void epilogue_tile(const TcParams& P, uint32_t taddr, bool row_ok, bool zero, long long base,
                                              int n0) {
                if (EPI == EPI_SWIGLU_FWD || EPI == EPI_WGRAD_SPLIT) {
    #pragma unroll 1
                    for (int c = 0; c < 128; c += 16) {
                        uint32_t r0[16], r1[16];
                        tmem_ld16(taddr + c, r0);
                        tmem_ld16(taddr + 128 + c, r1);
                        tmem_ld_wait(r0);
                        tmem_ld_wait(r1);
                        float v0[16], v1[16], h[16];
    #pragma unroll
                        for (int i = 0; i < 16; ++i) {
                            v0[i] = zero ? 0.f : __uint_as_float(r0[i]);
                            v1[i] = zero ? 0.f : __uint_as_float(r1[i]);
                        }
                        if (row_ok) {
                            store16(P.out0 + base, n0 + c, P.n_limit, v0);
                            store16(P.out1 + base, n0 + c, P.n_limit, v1);
                            if (EPI == EPI_SWIGLU_FWD) {
    #pragma unroll
                                for (int i = 0; i < 16; ++i) h[i] = v0[i] * sigmoidf_fast(v0[i]) * v1[i];
                                store16(P.out2 + base, n0 + c, P.n_limit, h);
                            }
                        }
                    }
                } else {
    #pragma unroll 1
                    for (int c = 0; c < BN; c += 16) {
                        uint32_t r0[16];
                        tmem_ld16(taddr + c, r0);
                        tmem_ld_wait(r0);
                        float v[16];
    #pragma unroll
                        for (int i = 0; i < 16; ++i) v[i] = zero ? 0.f : __uint_as_float(r0[i]);
                        if (row_ok && EPI == EPI_STORE_F32) {
                            // fp32 output (router logits / dW_r): acc (+ bias[column]), columns below n_limit (% 4 == 0)
                            float* orow = reinterpret_cast<float*>(P.out0) + base;
#pragma unroll
                            for (int i = 0; i < 16; i += 4) {
                                const int col = n0 + c + i;
                                if (col < P.n_limit) {
                                    float4 o = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
                                    if (P.bias) {
                                        const float4 bb = *reinterpret_cast<const float4*>(P.bias + col);
                                        o.x += bb.x, o.y += bb.y, o.z += bb.z, o.w += bb.w;
                                    }
                                    *reinterpret_cast<float4*>(orow + col) = o;
                                }
                            }
                        } else if (row_ok) {
                            if (EPI == EPI_SWIGLU_BWD) {
                                // v = dH; dG = dH * U * silu'(G), dU = dH * silu(G)
                                float gv[16], uv[16], dg[16], du[16];
                                load16(P.in0 + base, n0 + c, P.n_limit, gv);
                                load16(P.in1 + base, n0 + c, P.n_limit, uv);
    #pragma unroll
                                for (int i = 0; i < 16; ++i) {
                                    const float s = sigmoidf_fast(gv[i]);
                                    dg[i] = v[i] * uv[i] * (s * (1.f + gv[i] * (1.f - s)));
                                    du[i] = v[i] * (gv[i] * s);
                                }
                                store16(P.out0 + base, n0 + c, P.n_limit, dg);
                                store16(P.out1 + base, n0 + c, P.n_limit, du);
                            } else {
                                store16(P.out0 + base, n0 + c, P.n_limit, v);
                            }
                        }
                    }
                }
}

// ---- the kernel ---------------------------------------------------------------------------------------
template <int A_MAJOR, int B_MAJOR, int EPI>
__global__ void __launch_bounds__(kThreads, 1) tc_gemm_kernel(const __grid_constant__ TcParams P) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + STAGES * STAGE_BYTES);
    uint64_t* empty_bar = full_bar + STAGES;
    uint64_t* tfull_bar = empty_bar + STAGES;  // [2] accumulator ready
    uint64_t* tempty_bar = tfull_bar + 2;      // [2] accumulator drained
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tempty_bar + 2);
    int* tp = reinterpret_cast<int*>(smem + STAGES * STAGE_BYTES + 256);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int32_t* __restrict__ offsets = P.offsets;

    if (P.ragged_m)
        for (int g = threadIdx.x; g <= P.G; g += kThreads) tp[g] = (offsets[g] + BM - 1) / BM;
    if (warp == 0 && lane == 0) {
        prefetch_tmap(&P.a[0]), prefetch_tmap(&P.b[0]);
        if (P.n_src == 2) prefetch_tmap(&P.a[1]);
        if (P.n_src == 2 || P.b_split) prefetch_tmap(&P.b[1]);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(&full_bar[s], 1), mbar_init(&empty_bar[s], 1);
        for (int s = 0; s < 2; ++s) mbar_init(&tfull_bar[s], 1), mbar_init(&tempty_bar[s], 128);
        fence_barrier_init();
    }
    if (warp == 2) tmem_alloc(tmem_ptr, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;
    const int n_total = total_tiles(P, tp);

    if (warp == 0) {
        // ===== TMA producer (the warp runs converged, one elected lane issues: see elect_one) =====
        int stage = 0, phase = 0;
        long long w_empty = 0;
        for (int t = blockIdx.x; t < n_total; t += gridDim.x) {
            Tile T = decode_tile(P, tp, offsets, t);
            T.g = uni(T.g), T.m0 = uni(T.m0), T.n0 = uni(T.n0), T.k0 = uni(T.k0), T.nkb = uni(T.nkb);
            for (int kb = 0; kb < T.nkb; ++kb) {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&empty_bar[stage], phase ^ 1);
                if (P.prof) w_empty += clock64() - c0;
                if (elect_one()) {
                    uint8_t* sa = smem + stage * STAGE_BYTES;
                    uint8_t* sb = sa + A_BYTES;
                    uint64_t* bar = &full_bar[stage];
                    mbar_expect_tx(bar, STAGE_BYTES);
                    int src = 0, kk = kb;
                    if (P.n_src == 2 && kb >= P.kb_per_src) src = 1, kk = kb - P.kb_per_src;
                    const int k = T.k0 + kk * BK;
                    // A: ragged_m -> rows m0.. of a row buffer (z = 0); wgrad -> columns m0.. of a row buffer
                    if (A_MAJOR == K_MAJOR) {
                        tma_load_3d(sa, &P.a[src], bar, k, T.m0, 0);
                    } else {
#pragma unroll
                        for (int j = 0; j < BM / 64; ++j)
                            tma_load_3d(sa + j * MN_BLOCK_BYTES, &P.a[src], bar, T.m0 + 64 * j, k, 0);
                    }
                    // B: ragged_m -> weights of group g (z = g); wgrad -> columns n0.. of a row buffer (z = 0)
                    const int bz = P.ragged_m ? T.g : 0;
                    if (B_MAJOR == K_MAJOR) {
                        tma_load_3d(sb, &P.b[src], bar, k, T.n0, bz);
                    } else {
#pragma unroll
                        for (int j = 0; j < BN / 64; ++j) {
                            const int half = P.b_split ? (j >> 1) : src;
                            const int col = P.b_split ? T.n0 + 64 * (j & 1) : T.n0 + 64 * j;
                            tma_load_3d(sb + j * MN_BLOCK_BYTES, &P.b[half], bar, col, k, bz);
                        }
                    }
                }
                __syncwarp();
                if (++stage == STAGES) stage = 0, phase ^= 1;
            }
        }
        if (P.prof && lane == 0) P.prof[blockIdx.x * 8 + 3] = w_empty;
    } else if (warp == 1) {
        // ===== MMA issuer (warp 1, converged; one elected lane issues) =====
        constexpr uint32_t idesc = make_idesc(A_MAJOR, B_MAJOR);
        constexpr uint32_t a_lbo = A_MAJOR == K_MAJOR ? 16 : MN_BLOCK_BYTES, b_lbo = B_MAJOR == K_MAJOR ? 16 : MN_BLOCK_BYTES;
        constexpr uint32_t a_kstep = A_MAJOR == K_MAJOR ? UK * 2 : UK * 128, b_kstep = B_MAJOR == K_MAJOR ? UK * 2 : UK * 128;
        const uint32_t smem_base = uni(smem_u32(smem)), tmem_u = uni(tmem_base);
        const uint64_t a_desc0 = make_desc(smem_base, a_lbo, 1024), b_desc0 = make_desc(smem_base + A_BYTES, b_lbo, 1024);
        int stage = 0, phase = 0, as = 0, aphase = 0;
        long long w_full = 0, w_tempty = 0, n_tiles_done = 0;
        const long long t_begin = P.prof ? clock64() : 0;
        for (int t = blockIdx.x; t < n_total; t += gridDim.x) {
            const int t_nkb = uni(decode_tile(P, tp, offsets, t).nkb);
            {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&tempty_bar[as], aphase ^ 1);
                if (P.prof) w_tempty += clock64() - c0, ++n_tiles_done;
                tc_fence_after();
            }
            const uint32_t d_tmem = tmem_u + as * BN;
            for (int kb = 0; kb < t_nkb; ++kb) {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&full_bar[stage], phase);
                if (P.prof) w_full += clock64() - c0;
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t soff = (uint32_t)(stage * STAGE_BYTES) >> 4;
#pragma unroll
                    for (int kk = 0; kk < BK / UK; ++kk) {
                        const uint64_t ad = a_desc0 + (soff + ((kk * a_kstep) >> 4));
                        const uint64_t bd = b_desc0 + (soff + ((kk * b_kstep) >> 4));
                        umma_bf16(d_tmem, ad, bd, idesc, (kb | kk) != 0);
                    }
                    umma_commit(&empty_bar[stage]);  // frees the smem slot when these MMAs have read it
                }
                __syncwarp();
                if (++stage == STAGES) stage = 0, phase ^= 1;
            }
            if (elect_one()) umma_commit(&tfull_bar[as]);  // accumulator complete (immediately if nkb == 0)
            __syncwarp();
            if (++as == 2) as = 0, aphase ^= 1;
        }
        if (P.prof && lane == 0) {
            long long* q = P.prof + blockIdx.x * 8;
            q[0] = w_full, q[1] = w_tempty, q[2] = clock64() - t_begin, q[6] = n_tiles_done;
        }
    } else if (warp >= 4) {
        // ===== epilogue: warp w owns TMEM lanes 32 (w % 4) .. +31 = tile rows =====
        const int wq = warp & 3, row = wq * 32 + lane;
        int as = 0, aphase = 0;
        long long w_tfull = 0;
        const long long t_begin = P.prof ? clock64() : 0;
        const int rows_total = P.ragged_m ? offsets[P.G] : P.m_limit;
        for (int t = blockIdx.x; t < n_total; t += gridDim.x) {
            const Tile T = decode_tile(P, tp, offsets, t);
            const long long c0 = P.prof ? clock64() : 0;
            mbar_wait(&tfull_bar[as], aphase);
            if (P.prof) w_tfull += clock64() - c0;
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(wq * 32) << 16) + as * BN;
            const int grow = T.m0 + row;
            const bool row_ok = grow < rows_total;
            const bool zero = T.nkb == 0;  // empty expert in wgrad: exact zeros, the accumulator is stale
            const long long base = (P.ragged_m ? 0 : (long long)T.g * P.group_stride) + (long long)grow * P.ld;
            epilogue_tile<EPI>(P, taddr, row_ok, zero, base, T.n0);
            tc_fence_before();
            mbar_arrive(&tempty_bar[as]);
            if (++as == 2) as = 0, aphase ^= 1;
        }
        if (P.prof && threadIdx.x == 128) P.prof[blockIdx.x * 8 + 4] = w_tfull, P.prof[blockIdx.x * 8 + 5] = clock64() - t_begin;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc(tmem_base, 512);
    }
}


// ---- staged epilogue of the CTA-pair kernel: TMEM -> registers -> swizzled shared memory -> TMA store ----------
// A thread owns one row of the tile; direct row stores cost one L1 wavefront per thread and instruction (32 rows =
// 32 lines), which made the epilogue the limiter of the short-K tiles.  Each epilogue warp stages 32 rows x 64
// columns (4 KB, 128-byte rows in the TMA 128-byte swizzle: conflict-free 16-byte st.shared) and one lane issues
// a bulk tensor store, which also clips rows and columns at the tensor bounds.
constexpr int STG_BYTES = 32 * 128;  // one staging buffer: 32 rows x 64 bf16
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
                 : "=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]),"=r"(r[4]),"=r"(r[5]),"=r"(r[6]),"=r"(r[7]),"=r"(r[8]),"=r"(r[9]),"=r"(r[10]),"=r"(r[11]),"=r"(r[12]),"=r"(r[13]),"=r"(r[14]),"=r"(r[15]),"=r"(r[16]),"=r"(r[17]),"=r"(r[18]),"=r"(r[19]),"=r"(r[20]),"=r"(r[21]),"=r"(r[22]),"=r"(r[23]),"=r"(r[24]),"=r"(r[25]),"=r"(r[26]),"=r"(r[27]),"=r"(r[28]),"=r"(r[29]),"=r"(r[30]),"=r"(r[31])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void tmem_ld_wait32(uint32_t (&r)[32]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r[0]),"+r"(r[1]),"+r"(r[2]),"+r"(r[3]),"+r"(r[4]),"+r"(r[5]),"+r"(r[6]),"+r"(r[7]),"+r"(r[8]),"+r"(r[9]),"+r"(r[10]),"+r"(r[11]),"+r"(r[12]),"+r"(r[13]),"+r"(r[14]),"+r"(r[15]),"+r"(r[16]),"+r"(r[17]),"+r"(r[18]),"+r"(r[19]),"+r"(r[20]),"+r"(r[21]),"+r"(r[22]),"+r"(r[23]),"+r"(r[24]),"+r"(r[25]),"+r"(r[26]),"+r"(r[27]),"+r"(r[28]),"+r"(r[29]),"+r"(r[30]),"+r"(r[31]) : : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, const void* src, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(map),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void tma_reduce_add_3d(const CUtensorMap* map, const void* src, int c0, int c1, int c2) {
    asm volatile("cp.reduce.async.bulk.tensor.3d.global.shared::cta.add.tile.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(map),
                 "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void st_shared16(uint8_t* p, const uint4& v) {
    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(smem_u32(p)), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint4 ld_shared16(const uint8_t* p) {
    uint4 v;
    asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u16(uint32_t a, uint32_t v) {
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((unsigned short)v) : "memory");
}
__device__ __forceinline__ float lds_bf16(uint32_t a) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a) : "memory");
    return __uint_as_float((uint32_t)v << 16);
}
__device__ __forceinline__ void sts_f32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ float lds_f32(uint32_t a) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory");
    return v;
}
// address of 16-byte chunk `ch` (0..7) of row `r` (0..31) in a staging buffer (128-byte swizzle)
__device__ __forceinline__ uint8_t* stg_at(uint8_t* buf, int r, int ch) { return buf + r * 128 + ((ch ^ (r & 7)) << 4); }
// 32 fp32 columns -> bf16 -> chunks [4 half, 4 half + 4) of this thread's staging row
__device__ __forceinline__ void stage32(uint8_t* buf, int r, int half, const float* v) {
#pragma unroll
    for (int j = 0; j < 4; ++j) st_shared16(stg_at(buf, r, 4 * half + j), pack8(v + 8 * j));
}

// =====================================================================================================
// 2-CTA variant: a cluster of two CTAs (one TPC) works on two M tiles that share one B tile.  The leader CTA
// issues tcgen05.mma.cta_group::2 (M = 256: rows 0-127 accumulate in the leader's TMEM, 128-255 in the
// peer's); each CTA stages its own 128 x 64 A tile and one 128-column half of the 256 x 64 B tile, so a
// stage costs 32 KB per CTA instead of 48 KB: one third less L2 -> SM traffic (the measured limiter of the
// 1-CTA kernel) and a 6-stage ring.  The two M tiles need not be adjacent: in the ragged problems they are
// two tiles of the same expert (an odd last tile is paired with a duplicate whose stores are skipped); in
// wgrad they are two 128-row slices of dW.
// =====================================================================================================
#ifndef PIPER_WGRAD_BK
#define PIPER_WGRAD_BK 128
#endif
#ifndef PIPER_WGRAD_EPI_WARPS
#define PIPER_WGRAD_EPI_WARPS 4
#endif
// Ring depth and staging buffers per epilogue warp: the SwiGLU backward epilogue also stages its G, U inputs.
constexpr int kMaxGroups2 = 192;  // groups the CTA-pair kernel can index (its tile-prefix arrays share the 227 KB)
template <int EPI>
struct Cfg2 {
    // wgrad (both operands MN-major: TMA boxes of 64 columns x BK rows) takes K blocks of 128 rows, so that a box is
    // 16 KB like the K-major ones (8 KB boxes measured slower), in a 3-stage ring
    static constexpr bool WG = EPI == EPI_WGRAD || EPI == EPI_WGRAD_SPLIT;
    static constexpr int BKc = WG ? PIPER_WGRAD_BK : BK;
    static constexpr int NST = BKc == 128 ? 3 : 5;
    // wgrad: PIPER_WGRAD_EPI_WARPS = 8 gives two epilogue warps per TMEM lane quarter (each half of the tile's columns,
    // one staging buffer each).  Measured: C3 wgrad (2-3 K blocks per tile) 0.840 -> 0.824 ms, C2 2.10 -> 2.13 ms, so
    // the epilogue's dependent chain is not what bounds the short-K tiles; default 4.
    static constexpr int EPI_WARPS = WG ? PIPER_WGRAD_EPI_WARPS : 4;
    static constexpr int THREADS = 128 + 32 * EPI_WARPS;
    static constexpr int NBUF = EPI == EPI_SWIGLU_BWD ? 4 : (BKc == 128 ? (EPI_WARPS == 8 ? 1 : 2) : 3);
    static constexpr int A_B = BM * BKc * 2, B_B = (BN / 2) * BKc * 2, STAGE_B = A_B + B_B, MNB = 64 * BKc * 2;
    static constexpr int RING_BYTES = NST * STAGE_B, STG_TOTAL = EPI_WARPS * NBUF * STG_BYTES;
    // wgrad (bf16 output, no gathered operand): warp 2, idle after the TMEM allocation, issues the bulk
    // stores of the blocks the epilogue warps stage, so that the drain of an accumulator does not wait for the store issue
    static constexpr bool STORE_WARP = WG && EPI_WARPS == 4;  // NBUF = 2
    static constexpr int BAR_BYTES = 320;  // barriers (256) + the store warp's "staging buffer free" barriers (8 x 8)
    static constexpr int SMEM = RING_BYTES + STG_TOTAL + 1024 + BAR_BYTES + 2 * (kMaxGroups2 + 1) * 4;
    static_assert(SMEM <= 232448, "shared memory per CTA");
};
constexpr int PANEL_PAIRS = 8;

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_alloc2(uint32_t* dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst_smem)), "r"(cols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
// D[tmem of both CTAs] (+)= A * B, 256 x 256 x 16 across the CTA pair
__device__ __forceinline__ void umma2_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
        : "memory");
}
// arrives on the barrier at this offset in BOTH CTAs once the MMAs issued so far have completed
__device__ __forceinline__ void umma2_commit(uint64_t* bar) {
    asm volatile(
        "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
            smem_u32(bar)),
        "h"((uint16_t)3)
        : "memory");
}
__host__ __device__ constexpr uint32_t make_idesc2(int a_major, int b_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_major << 15) | ((uint32_t)b_major << 16) |
           ((uint32_t)(BN >> 3) << 17) | ((uint32_t)((2 * BM) >> 4) << 24);
}

struct Tile2 {
    int g, m0, n0, k0, nkb;
    bool store;  // false: this CTA's M tile duplicates the leader's (odd tile count), nothing is stored
};

// tp[g] = first M tile of group g; tpp[g] = first tile PAIR of group g (ragged_m).
__device__ __forceinline__ int total_pairs(const TcParams& P, const int* tpp) {
    return P.ragged_m ? tpp[P.G] * P.n_tiles : P.G * ((P.m_tiles + 1) / 2) * P.n_tiles;
}
// t / d for 0 <= t < 2^22, 0 < d < 2^22 with the reciprocal of d hoisted out of the tile loop (one correction step makes
// the float estimate exact); an integer division costs the issuing thread ~100 cycles between two short wgrad tiles
__device__ __forceinline__ int div_rcp(int t, int d, float rcp, int& rem) {
    int q = __float2int_rz(__int2float_rz(t) * rcp);
    int r = t - q * d;
    if (r < 0) --q, r += d;
    else if (r >= d) ++q, r -= d;
    rem = r;
    return q;
}
__device__ __forceinline__ Tile2 decode_pair(const TcParams& P, const int* tp, const int* tpp,
                                             const int32_t* __restrict__ offsets, int t, int rank, int bk = BK,
                                             float rcp_group = 0.f, float rcp_pairs = 0.f) {
    Tile2 r;
    if (P.ragged_m) {
        int g = 0;
        while (g + 1 < P.G && tpp[g + 1] * P.n_tiles <= t) ++g;
        const int local = t - tpp[g] * P.n_tiles, mg = tp[g + 1] - tp[g], pg = tpp[g + 1] - tpp[g];
        const int per_panel = PANEL_PAIRS * P.n_tiles;
        const int panel = local / per_panel, rem = local - panel * per_panel;
        const int pp = min(PANEL_PAIRS, pg - panel * PANEL_PAIRS);
        const int nt = rem / pp, pair = panel * PANEL_PAIRS + (rem - nt * pp);
        int mt = 2 * pair + rank;
        r.store = mt < mg;
        if (!r.store) mt = 2 * pair;
        r.g = g, r.m0 = (tp[g] + mt) * BM, r.n0 = nt * P.tile_n, r.k0 = 0, r.nkb = P.kb_per_src * P.n_src;
    } else {
        // wgrad: tp[] holds the groups' offsets (copied to shared memory in the prologue: a tile of 2-8 K blocks is too
        // short to hide two dependent global loads of the issuing thread between tiles)
        const int pairs = (P.m_tiles + 1) / 2, per_group = pairs * P.n_tiles;
        int g, local, nt, pair;
        if (rcp_group != 0.f) {
            g = div_rcp(t, per_group, rcp_group, local);
            nt = div_rcp(local, pairs, rcp_pairs, pair);
        } else {
            g = t / per_group, local = t - g * per_group;
            nt = local / pairs, pair = local - nt * pairs;
        }
        const int lo = tp[g], hi = tp[g + 1];
        r.store = true;  // rows beyond m_limit are clipped by the bounds checks
        r.g = g, r.m0 = (2 * pair + rank) * BM, r.n0 = nt * P.tile_n, r.k0 = lo, r.nkb = (hi - lo + bk - 1) / bk;
    }
    return r;
}

__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// TMA load into this CTA's shared memory, bytes counted on the mbarrier at cluster address `bar_cluster`
__device__ __forceinline__ void tma_load_3d_pair(void* dst, const CUtensorMap* map, uint32_t bar_cluster, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(bar_cluster), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t bar_cluster) {
    // default semantics (.release.cta): the .release.cluster form costs a MEMBAR.ALL.GPU per tile; the TMEM reads it must
    // follow are ordered by tcgen05.fence::before_thread_sync
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(bar_cluster) : "memory");
}

// Tile feed of the CTA-pair kernels: tiles are handed out dynamically (a static stride leaves whole tiles of imbalance
// when a cluster draws the long chunks, and stalls when a co-scheduled kernel slows one SM).  One thread of the leader
// CTA draws tile numbers from a global counter and publishes them, in order, in a ring of kFeed slots in both CTAs'
// shared memory; every consumer warp (producer, MMA issuer, 4 epilogue warps per CTA) reads slot it % kFeed for its
// it-th tile and releases it to the feeder.  A number >= the tile count ends every loop.  The ring is two deep and the
// first tile of a cluster is its own index, so the clusters start on neighbouring tiles (shared weight tiles in L2)
// and every later tile is drawn only when the cluster is about to need it.
constexpr int kFeed = 2, kFeedConsumers = 2 * 5 + 1;
constexpr int kFeedWords = 8;  // rows-on-N kernels: a slot holds the decoded tile {t, g, f, r0, n, zend}
struct TileFeed {
    int* ids;             // [kFeed][stride] this CTA
    uint64_t* full;       // [kFeed] this CTA
    uint32_t empty_addr;  // cluster address of the leader's empty barriers [kFeed]
    int stride = 1;       // ints per slot
    __device__ __forceinline__ int peek(int it) const {
        mbar_wait_cluster(&full[it & (kFeed - 1)], (it / kFeed) & 1);
        return *reinterpret_cast<volatile int*>(&ids[(it & (kFeed - 1)) * stride]);
    }
    // words 1.. of the slot of tile `it` (valid between peek(it) and this warp's release in take(it))
    __device__ __forceinline__ const volatile int* slot(int it) const { return ids + (it & (kFeed - 1)) * stride; }
    // all lanes of a consumer warp: done with slot `it` (after every lane has read what it needs from it)
    __device__ __forceinline__ void release(int it, int lane) const {
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(empty_addr + (it & (kFeed - 1)) * 8);
    }
    // all lanes of a consumer warp call this
    __device__ __forceinline__ int take(int it, int lane) const {
        const int t = peek(it);
        __syncwarp();
        if (lane == 0 && t >= 0) mbar_arrive_cluster(empty_addr + (it & (kFeed - 1)) * 8);
        return t;
    }
};

// GATHER_A (wgrad gate|up, N2 fusion): the A operand Xp^T is not read from the packed buffer; warp 2 gathers K row r of the
// tile (= packed row k0 + r) from the token-major x through src_of with 16-byte cp.async copies, in the layout of the two
// 64-column TMA boxes (see the GATHER note at tc_gemmT_kernel for the barrier protocol).
constexpr int kGatherWarpsA = 4;  // GATHER_A: warp 2 and three extra warps (behind the epilogue warps) share the K rows of a block
template <int A_MAJOR, int B_MAJOR, int EPI, bool GATHER_A = false>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(Cfg2<EPI>::THREADS + (GATHER_A ? 32 * (kGatherWarpsA - 1) : 0), 1)
tc_gemm2_kernel(const __grid_constant__ TcParams P) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    constexpr int STAGES2 = Cfg2<EPI>::NST, NBUF = Cfg2<EPI>::NBUF, BKc = Cfg2<EPI>::BKc, MNB = Cfg2<EPI>::MNB;
    constexpr int A2_BYTES = Cfg2<EPI>::A_B, STAGE2_BYTES = Cfg2<EPI>::STAGE_B;
    uint8_t* stg_base = smem + Cfg2<EPI>::RING_BYTES;
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(stg_base + Cfg2<EPI>::STG_TOTAL);  // used in the leader CTA
    uint64_t* empty_bar = full_bar + STAGES2;                                            // one set per CTA
    uint64_t* tfull_bar = empty_bar + STAGES2;                                           // [2] one set per CTA
    uint64_t* tempty_bar = tfull_bar + 2;                                                // [2] used in the leader CTA
    uint64_t* ld_bar = tempty_bar + 2;                                                   // [4 warps][2 sets] epilogue inputs
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(ld_bar + 8);
    uint64_t* feed_full = ld_bar + 9;         // [kFeed] one set per CTA
    uint64_t* feed_empty = feed_full + kFeed;  // [kFeed] used in the leader CTA
    int* feed_ids = reinterpret_cast<int*>(feed_empty + kFeed);
    uint64_t* gfull_bar = reinterpret_cast<uint64_t*>(feed_ids + 2);  // [STAGES2] GATHER_A: peer CTA's local "A rows landed"
    static_assert(!GATHER_A || (2 * STAGES2 + 4 + 9 + 2 * kFeed + 1 + STAGES2) * 8 <= 256, "barrier area");
    uint64_t* sfull_bar = ld_bar;  // store warp: [2] block staged by the four epilogue warps (the SwiGLU input barriers are unused then)
    uint64_t* sempty_bar = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(full_bar) + 256);  // [2] block read by its store
    int* tp = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(full_bar) + Cfg2<EPI>::BAR_BYTES);
    int* tpp = tp + (kMaxGroups2 + 1);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rank = (int)cluster_ctarank();
    const int pair_id = blockIdx.x >> 1, n_pairs_grid = gridDim.x >> 1;
    // the store warp serves bf16 outputs of long K ranges (the host decides); fp32 dW blocks and short tiles keep one
    // 32-row store per epilogue warp
    bool store_warp = Cfg2<EPI>::STORE_WARP && !GATHER_A && P.store_warp != 0;
    const int32_t* __restrict__ offsets = P.offsets;

    if (!P.ragged_m) {  // wgrad: offsets and real row counts of the groups (read by decode_pair / the MMA issuer)
        for (int g = threadIdx.x; g <= P.G; g += Cfg2<EPI>::THREADS) {
            tp[g] = offsets[g];
            if (g < P.G) tpp[g] = P.counts ? P.counts[g] : offsets[g + 1] - offsets[g];
        }
    }
    if (P.ragged_m) {
        for (int g = threadIdx.x; g <= P.G; g += Cfg2<EPI>::THREADS) tp[g] = (offsets[g] + BM - 1) / BM;
        __syncthreads();
        if (warp == 3) {  // exclusive scan of the tile pairs per group
            int carry = 0;
            for (int g0 = 0; g0 < P.G; g0 += 32) {
                const int g = g0 + lane;
                const int v = g < P.G ? (tp[g + 1] - tp[g] + 1) >> 1 : 0;
                int x = v;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int y = __shfl_up_sync(0xffffffffu, x, o);
                    if (lane >= o) x += y;
                }
                if (g < P.G) tpp[g] = carry + x - v;
                carry += __shfl_sync(0xffffffffu, x, 31);
            }
            if (lane == 0) tpp[P.G] = carry;
        }
    }
    // wgrad: draw tiles from the counter only when the experts' K ranges are long and uneven (C4: one expert holds 16% of
    // the rows, so a static stride leaves some clusters two of its tiles); equal or short tiles keep the static stride
    // (the draw costs an atomic and a cluster-scope release per tile: -2% on C2, -7% on C3's 2-3 K-block tiles).
    bool dynamic = true;  // computed by every warp (same data, same answer): static tiles bypass the feed altogether
    if (!P.ragged_m) {
        int mx = 0;
        for (int g = lane; g < P.G; g += 32) mx = max(mx, offsets[g + 1] - offsets[g]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        const int total = offsets[P.G];
        dynamic = total >= 512 * P.G && (long long)mx * P.G > 2ll * total;
        if (P.store_warp == 2 && (dynamic || total < 512 * P.G)) store_warp = false;  // by the real group lengths
    }
    if (warp == 0 && lane == 0) {
        prefetch_tmap(&P.a[0]), prefetch_tmap(&P.b[0]);
        if (P.n_src == 2) prefetch_tmap(&P.a[1]);
        if (P.n_src == 2 || P.b_split) prefetch_tmap(&P.b[1]);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < STAGES2; ++s) {  // GATHER_A: + the leader's 32 gather lanes + the peer's forwarder
            mbar_init(&full_bar[s], GATHER_A ? 2 + 32 * kGatherWarpsA : 1), mbar_init(&empty_bar[s], 1);
            if (GATHER_A) mbar_init(&gfull_bar[s], 32 * kGatherWarpsA);
        }
        for (int s = 0; s < 2; ++s) mbar_init(&tfull_bar[s], 1), mbar_init(&tempty_bar[s], 2 * Cfg2<EPI>::EPI_WARPS);  // both CTAs
        for (int s = 0; s < 8; ++s) mbar_init(&ld_bar[s], store_warp && s < 2 ? 4 : 1), mbar_init(&sempty_bar[s], 1);
        for (int s = 0; s < kFeed; ++s)  // consumers: (producer + epilogue warps) x 2 CTAs + the MMA issuer (+ gather warps, forwarder / store warps)
            mbar_init(&feed_full[s], 1), mbar_init(&feed_empty[s], 2 * (1 + Cfg2<EPI>::EPI_WARPS) + 1 + (GATHER_A ? 2 * kGatherWarpsA + 1 : 0) + (store_warp ? 2 : 0));
        fence_barrier_init();
    }
    if (warp == 2) tmem_alloc2(tmem_ptr, 512);
    tc_fence_before();
    cluster_sync_all();  // barriers of both CTAs initialised before any remote arrive / multicast commit
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;
    const int n_total = total_pairs(P, tpp);
    // wgrad tile decode: reciprocals of the two divisors (0: plain integer division, ragged problems / huge tile counts)
    const int wg_pairs = (P.m_tiles + 1) / 2, wg_group = wg_pairs * P.n_tiles;
    const bool wg_fast = !P.ragged_m && n_total < (1 << 22);
    const float rcp_group = wg_fast ? 1.f / (float)wg_group : 0.f, rcp_pairs = wg_fast ? 1.f / (float)wg_pairs : 0.f;
    TileFeed feed;
    feed.ids = feed_ids, feed.full = feed_full, feed.empty_addr = mapa_u32(smem_u32(feed_empty), 0);

    if (dynamic && warp == 3 && rank == 0 && lane == 0) {
        // ===== tile feeder (one thread of the leader CTA), see TileFeed =====
        const uint32_t peer_ids = mapa_u32(smem_u32(feed_ids), 1), peer_full = mapa_u32(smem_u32(feed_full), 1);
        for (int it = 0;; ++it) {
            const int slot = it & (kFeed - 1);
            mbar_wait(&feed_empty[slot], ((it / kFeed) & 1) ^ 1);
            const int t = it == 0 ? pair_id : n_pairs_grid + atomicAdd(P.sched, 1);
            *reinterpret_cast<volatile int*>(&feed_ids[slot]) = t;
            asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(peer_ids + slot * 4), "r"(t) : "memory");
            mbar_arrive(&feed_full[slot]);
            asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(peer_full + slot * 8) : "memory");
            if (t >= n_total) break;
        }
        __threadfence();
        if (atomicAdd(P.sched + 1, 1) == n_pairs_grid - 1) {
            __threadfence();
            P.sched[0] = 0, P.sched[1] = 0;
        }
    }

    if (warp == 0) {
        // ===== TMA producer (both CTAs; the warp runs converged, one elected lane issues): own A tile + own 128-column
        // half of B, counted on the leader's barrier =====
        const uint32_t leader_full = uni(mapa_u32(smem_u32(full_bar), 0));
        const int urank = uni(rank);
        int stage = 0, phase = 0;
        long long w_empty = 0;
        for (int it = 0;; ++it) {
            const int t = uni(dynamic ? feed.take(it, lane) : pair_id + it * n_pairs_grid);
            if (t >= n_total) break;
            Tile2 T = decode_pair(P, tp, tpp, offsets, t, urank, BKc, rcp_group, rcp_pairs);
            T.g = uni(T.g), T.m0 = uni(T.m0), T.n0 = uni(T.n0), T.k0 = uni(T.k0), T.nkb = uni(T.nkb);
            for (int kb = 0; kb < T.nkb; ++kb) {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&empty_bar[stage], phase ^ 1);
                if (P.prof) w_empty += clock64() - c0;
                if (elect_one()) {
                    uint8_t* sa = smem + stage * STAGE2_BYTES;
                    uint8_t* sb = sa + A2_BYTES;
                    if (urank == 0) mbar_expect_tx(&full_bar[stage], GATHER_A ? 2 * Cfg2<EPI>::B_B : 2 * STAGE2_BYTES);
                    const uint32_t bar = leader_full + stage * 8;
                    int src = 0, kk = kb;
                    if (P.ragged_m && kb >= P.kb_per_src) src = 1, kk = kb - P.kb_per_src;
                    const int k = T.k0 + kk * BKc;
                    if (GATHER_A) {
                        // the A tile is gathered by warp 2
                    } else if (A_MAJOR == K_MAJOR) {
                        tma_load_3d_pair(sa, &P.a[src], bar, k, T.m0, 0);
                    } else {
#pragma unroll
                        for (int j = 0; j < BM / 64; ++j)
                            tma_load_3d_pair(sa + j * MNB, &P.a[src], bar, T.m0 + 64 * j, k, 0);
                    }
                    const int bz = P.ragged_m ? T.g : 0;
                    if (B_MAJOR == K_MAJOR) {
                        tma_load_3d_pair(sb, &P.b[src], bar, k, T.n0 + urank * (BN / 2), bz);
                    } else {
                        const int half = P.b_split ? urank : src;
                        const int col = P.b_split ? T.n0 : T.n0 + urank * (BN / 2);
#pragma unroll
                        for (int j = 0; j < BN / 128; ++j)
                            tma_load_3d_pair(sb + j * MNB, &P.b[half], bar, col + 64 * j, k, bz);
                    }
                }
                __syncwarp();
                if (++stage == STAGES2) stage = 0, phase ^= 1;
            }
        }
        if (P.prof && lane == 0) P.prof[blockIdx.x * 8 + 3] = w_empty;
    } else if (GATHER_A && (warp == 2 || warp >= 4 + Cfg2<EPI>::EPI_WARPS)) {
        // ===== A producers, gathered (both CTAs; kGatherWarpsA warps, all 32 lanes): a lane owns one 16-byte chunk (ch) of
        // the two 64-column boxes of the K rows r = 16 q + 4 gw + rs; their swizzle term r & 7 = 4 (gw & 1) + rs is a constant
        // of the lane, so the destination of copy (q, box j) is a fixed address + q * 2048 + j * MNB =====
        const int gw = warp == 2 ? 0 : warp - (3 + Cfg2<EPI>::EPI_WARPS);
        const int ch = lane & 7, rs = lane >> 3, r_lane = 4 * gw + rs;
        const char* gbase = static_cast<const char*>(P.gsrc);
        const uint32_t pitch16 = (uint32_t)P.g_cols >> 3;
        const uint32_t dst_lane = smem_u32(smem) + r_lane * 128 + ((ch ^ (r_lane & 7)) << 4);
        constexpr int NQ = BKc / (4 * kGatherWarpsA);
        int stage = 0, phase = 0;
        for (int it = 0;; ++it) {
            const int t = dynamic ? feed.take(it, lane) : pair_id + it * n_pairs_grid;
            if (t >= n_total) break;
            const Tile2 T = decode_pair(P, tp, tpp, offsets, t, rank, BKc, rcp_group, rcp_pairs);
            const int seg_end = tp[T.g + 1];  // rows of the next expert are never issued to the tensor core: not loaded
            const int col0 = T.m0 + ch * 8;
            const uint32_t c_bad0 = col0 < P.g_cols ? 0u : 1u, c_bad1 = col0 + 64 < P.g_cols ? 0u : 1u;
            const char* src0 = gbase + (c_bad0 ? 0 : (size_t)col0 * 2);
            const char* src1 = gbase + (c_bad1 ? 0 : (size_t)(col0 + 64) * 2);
            for (int kb = 0; kb < T.nkb; ++kb) {
                const int k = T.k0 + kb * BKc;
                uint32_t off[NQ], zmask = 0;
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    const int row = k + 4 * kGatherWarpsA * q + r_lane;
                    const int a = row < seg_end ? P.src_of[row] : -1;
                    off[q] = a >= 0 ? (uint32_t)(((unsigned long long)a * P.g_magic) >> 35) * pitch16 : 0u;
                    zmask |= a >= 0 ? 0u : 1u << q;
                }
                if (lane == 0) mbar_wait(&empty_bar[stage], phase ^ 1);
                __syncwarp();
                const uint32_t dst = dst_lane + stage * STAGE2_BYTES;
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    const uint32_t z = zmask & (1u << q);
                    const size_t ob = (size_t)off[q] * 16;
                    cp_async16_z(dst + q * (4 * kGatherWarpsA * 128), src0 + ob, z | c_bad0);
                    cp_async16_z(dst + q * (4 * kGatherWarpsA * 128) + MNB, src1 + ob, z | c_bad1);
                }
                cp_async_arrive(rank == 0 ? &full_bar[stage] : &gfull_bar[stage]);
                if (++stage == STAGES2) stage = 0, phase ^= 1;
            }
        }
    } else if (GATHER_A && warp == 1 && rank == 1) {
        // ===== peer CTA: forward "my A rows of this stage have landed" to the leader's full barrier =====
        const uint32_t leader_full = mapa_u32(smem_u32(full_bar), 0);
        int stage = 0, phase = 0;
        for (int it = 0;; ++it) {
            const int t = dynamic ? feed.take(it, lane) : pair_id + it * n_pairs_grid;
            if (t >= n_total) break;
            const Tile2 T = decode_pair(P, tp, tpp, offsets, t, rank, BKc, rcp_group, rcp_pairs);
            for (int kb = 0; kb < T.nkb; ++kb) {
                if (lane == 0) {
                    mbar_wait(&gfull_bar[stage], phase);
                    fence_proxy_async();
                    // plain remote arrive: the cluster-scope release form is a GPU-scope membar per K block (1-2 us in this
                    // thread: the whole kernel ran at its pace).  The rows are read by this CTA's own tensor core, after the
                    // proxy fence above; the arrival only tells the leader that it may issue.
                    mbar_arrive_cluster(leader_full + stage * 8);
                }
                __syncwarp();
                if (++stage == STAGES2) stage = 0, phase ^= 1;
            }
        }
    } else if (warp == 1 && rank == 0) {
        // ===== MMA issuer (warp 1 of the leader CTA, converged; one elected lane issues) =====
        constexpr uint32_t idesc = make_idesc2(A_MAJOR, B_MAJOR);
        constexpr uint32_t a_lbo = A_MAJOR == K_MAJOR ? 16 : MNB, b_lbo = B_MAJOR == K_MAJOR ? 16 : MNB;
        constexpr uint32_t a_kstep = A_MAJOR == K_MAJOR ? UK * 2 : UK * 128, b_kstep = B_MAJOR == K_MAJOR ? UK * 2 : UK * 128;
        const uint32_t smem_base = uni(smem_u32(smem)), tmem_u = uni(tmem_base);
        const uint64_t a_desc0 = make_desc(smem_base, a_lbo, 1024), b_desc0 = make_desc(smem_base + A2_BYTES, b_lbo, 1024);
        int stage = 0, phase = 0, as = 0, aphase = 0;
        long long w_full = 0, w_tempty = 0, n_tiles_done = 0;
        const long long t_begin = P.prof ? clock64() : 0;
        for (int it = 0;; ++it) {
            const int t = uni(dynamic ? feed.take(it, lane) : pair_id + it * n_pairs_grid);
            if (t >= n_total) break;
            const Tile2 T = decode_pair(P, tp, tpp, offsets, t, 0, BKc, rcp_group, rcp_pairs);
            const int t_nkb = uni(T.nkb);
            // wgrad: the K range ends with the expert's zero pad rows; K slices (16 rows) that hold only pad rows are
            // not issued (C2: 640 of 8832 rows, 7% of the tensor work)
            const int k_valid = uni(!P.ragged_m ? tpp[T.g] : 0x3fffffff);
            {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&tempty_bar[as], aphase ^ 1);
                if (P.prof) w_tempty += clock64() - c0, ++n_tiles_done;
                tc_fence_after();
            }
            const uint32_t d_tmem = tmem_u + as * BN;
            for (int kb = 0; kb < t_nkb; ++kb) {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&full_bar[stage], phase);
                if (GATHER_A) fence_proxy_async();  // gathered rows were written through the generic proxy
                if (P.prof) w_full += clock64() - c0;
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t soff = (uint32_t)(stage * STAGE2_BYTES) >> 4;
                    const int kk_end = (k_valid - kb * BKc + UK - 1) / UK;  // >= 1 in block 0 of a non-empty expert
#pragma unroll
                    for (int kk = 0; kk < BKc / UK; ++kk) {
                        if (kk >= kk_end) break;
                        const uint64_t ad = a_desc0 + (soff + ((kk * a_kstep) >> 4));
                        const uint64_t bd = b_desc0 + (soff + ((kk * b_kstep) >> 4));
                        umma2_bf16(d_tmem, ad, bd, idesc, (kb | kk) != 0);
                    }
                    umma2_commit(&empty_bar[stage]);  // frees this stage in both CTAs
                }
                __syncwarp();
                if (++stage == STAGES2) stage = 0, phase ^= 1;
            }
            if (elect_one()) umma2_commit(&tfull_bar[as]);  // both CTAs' epilogues
            __syncwarp();
            if (++as == 2) as = 0, aphase ^= 1;
        }
        if (P.prof && lane == 0) {
            long long* pq = P.prof + blockIdx.x * 8;
            pq[0] = w_full, pq[1] = w_tempty, pq[2] = clock64() - t_begin, pq[6] = n_tiles_done;
        }
    } else if (Cfg2<EPI>::STORE_WARP && !GATHER_A && warp == 2) {
        // ===== store warp (both CTAs, wgrad with bf16 output): one bulk store of 128 rows x 64 columns per chunk instead
        // of one per epilogue warp (a bulk tensor store costs its issuing warp ~130 cycles whatever its size: 16 of them per
        // tile were 12 % of the epilogue warps' time on the short K ranges of C3).  The four epilogue warps stage their 32
        // rows side by side in block n & 1; this warp stores the block and hands it back once the copy has read it.
        if (store_warp) {
            const int urank = uni(rank);
            const bool leader = elect_one();  // one lane issues every store: the bulk groups are per thread
            uint32_t n = 0;                   // chunks so far: block n & 1, barrier phase (n >> 1) & 1
            for (int it = 0;; ++it) {
                const int t = uni(dynamic ? feed.take(it, lane) : pair_id + it * n_pairs_grid);
                if (t >= n_total) break;
                Tile2 T = decode_pair(P, tp, tpp, offsets, t, urank, BKc, rcp_group, rcp_pairs);
                T.g = uni(T.g), T.m0 = uni(T.m0), T.n0 = uni(T.n0), T.store = uni((int)T.store) != 0;
                const int z = P.ragged_m ? 0 : T.g;
#pragma unroll 1
                for (int c = 0; c < 4; ++c) {
                    const bool split = EPI == EPI_WGRAD_SPLIT;
                    const CUtensorMap* om = split ? &P.ow[c >> 1] : &P.ow[0];
                    const int col = split ? T.n0 + 64 * (c & 1) : T.n0 + 64 * c;
                    if (col >= P.n_limit) continue;
                    const int b = n & 1, ph = (n >> 1) & 1;
                    ++n;
                    mbar_wait(&sfull_bar[b], ph);
                    if (leader) {
                        if (T.store) {
                            tma_store_3d(om, stg_base + b * (4 * STG_BYTES), col, T.m0, z);
                            bulk_commit();
                            bulk_wait_read<0>();
                        }
                        mbar_arrive(&sempty_bar[b]);
                    }
                    __syncwarp();
                }
            }
            if (leader) bulk_wait_all();
        }
    } else if (warp >= 4) {
        // ===== epilogue (both CTAs): this CTA's 128 rows of the 256-row accumulator =====
        // (warp-uniform values are made provably so, and one elected lane issues the bulk tensor copies: see elect_one)
        const int uwarp = uni(warp), urank = uni(rank);
        const bool leader = elect_one();
        const int wq = uwarp & 3;            // TMEM lane quarter of this warp
        const int chalf = (uwarp - 4) >> 2;  // 8 epilogue warps: the second warp of a quarter takes the tile's upper columns
        constexpr int C_PER_WARP = 4 / (Cfg2<EPI>::EPI_WARPS / 4);
        const uint32_t leader_tempty = uni(mapa_u32(smem_u32(tempty_bar), 0));
        uint8_t* stg = stg_base + (uwarp - 4) * NBUF * STG_BYTES;
        int as = 0, aphase = 0, ring = 0;
        long long w_tfull = 0, w_stg = 0;
        const long long t_begin = P.prof ? clock64() : 0;
        uint32_t q = 0;  // SwiGLU backward: running chunk number -> input set q & 1, barrier phase (q >> 1) & 1
        // G, U of 32 rows x 64 columns -> set `set` of this warp's staging buffers (bytes counted on ld_bar)
        auto load_inputs = [&](const Tile2& Tn, int c, int set) {
            if (leader) {
                bulk_wait_read<0>();  // the stores that last read this set are done with it
                uint64_t* bar = &ld_bar[wq * 2 + set];
                mbar_expect_tx(bar, 2 * STG_BYTES);
                tma_load_3d(stg + (2 * set) * STG_BYTES, &P.ein[0], bar, Tn.n0 + 64 * c, Tn.m0 + wq * 32, 0);
                tma_load_3d(stg + (2 * set + 1) * STG_BYTES, &P.ein[1], bar, Tn.n0 + 64 * c, Tn.m0 + wq * 32, 0);
            }
        };
        if (EPI == EPI_SWIGLU_BWD) {
            const int t0 = dynamic ? feed.peek(0) : pair_id;
            if (t0 < n_total) load_inputs(decode_pair(P, tp, tpp, offsets, t0, rank, BKc, rcp_group, rcp_pairs), 0, 0);
        }
        for (int it = 0;; ++it) {
            const int t = uni(dynamic ? feed.take(it, lane) : pair_id + it * n_pairs_grid);
            if (t >= n_total) break;
            Tile2 T = decode_pair(P, tp, tpp, offsets, t, urank, BKc, rcp_group, rcp_pairs);
            T.g = uni(T.g), T.m0 = uni(T.m0), T.n0 = uni(T.n0), T.nkb = uni(T.nkb), T.store = uni((int)T.store) != 0;
            const long long c0 = P.prof ? clock64() : 0;
            mbar_wait(&tfull_bar[as], aphase);
            if (P.prof) w_tfull += clock64() - c0;
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(wq * 32) << 16) + as * BN;
            const int row0 = T.m0 + wq * 32, z = P.ragged_m ? 0 : T.g;
            const bool zero = T.nkb == 0;  // empty expert in wgrad: exact zeros, the accumulator is stale
            if (EPI == EPI_SWIGLU_FWD) {
                // accumulator columns [0,128) = G, [128,256) = U of output columns n0 .. n0+127
#pragma unroll 1
                for (int c = 0; c < 2; ++c) {
                    const int col = T.n0 + 64 * c;
                    if (col >= P.n_limit) break;
                    const long long c1 = P.prof ? clock64() : 0;
                    if (leader) bulk_wait_read<0>();
                    __syncwarp();
                    if (P.prof) w_stg += clock64() - c1;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        uint32_t rg[32], ru[32];
                        tmem_ld32(taddr + 64 * c + 32 * h, rg);
                        tmem_ld32(taddr + 128 + 64 * c + 32 * h, ru);
                        tmem_ld_wait32(rg);
                        tmem_ld_wait32(ru);
                        float g[32], u[32];
#pragma unroll
                        for (int i = 0; i < 32; ++i) g[i] = __uint_as_float(rg[i]), u[i] = __uint_as_float(ru[i]);
                        stage32(stg, lane, h, g);
                        stage32(stg + STG_BYTES, lane, h, u);
#pragma unroll
                        for (int i = 0; i < 32; ++i) g[i] = g[i] * sigmoidf_fast(g[i]) * u[i];
                        stage32(stg + 2 * STG_BYTES, lane, h, g);
                    }
                    fence_proxy_async();
                    __syncwarp();
                    if (leader && T.store) {
                        tma_store_3d(&P.o[0], stg, col, row0, z);
                        tma_store_3d(&P.o[1], stg + STG_BYTES, col, row0, z);
                        tma_store_3d(&P.o[2], stg + 2 * STG_BYTES, col, row0, z);
                        bulk_commit();
                    }
                }
            } else if (EPI == EPI_SWIGLU_BWD) {
                // accumulator = dH; dG = dH * U * silu'(G), dU = dH * silu(G), computed in place over the staged G, U
#pragma unroll 1
                for (int c = 0; c < 4; ++c, ++q) {
                    const int set = q & 1;
                    uint8_t* bg = stg + (2 * set) * STG_BYTES;
                    uint8_t* bu = bg + STG_BYTES;
                    const long long c1 = P.prof ? clock64() : 0;
                    mbar_wait(&ld_bar[wq * 2 + set], (q >> 1) & 1);
                    if (P.prof) w_stg += clock64() - c1;
                    if (c < 3) {
                        load_inputs(T, c + 1, set ^ 1);
                    } else {
                        const int tn = dynamic ? feed.peek(it + 1) : t + n_pairs_grid;
                        if (tn < n_total) load_inputs(decode_pair(P, tp, tpp, offsets, tn, rank, BKc, rcp_group, rcp_pairs), 0, set ^ 1);
                    }
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        uint32_t r[32];
                        tmem_ld32(taddr + 64 * c + 32 * h, r);
                        tmem_ld_wait32(r);
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            uint8_t* pg = stg_at(bg, lane, 4 * h + j);
                            uint8_t* pu = stg_at(bu, lane, 4 * h + j);
                            float gv[8], uv[8], dg[8], du[8];
                            unpack8(ld_shared16(pg), gv);
                            unpack8(ld_shared16(pu), uv);
#pragma unroll
                            for (int i = 0; i < 8; ++i) {
                                const float v = __uint_as_float(r[8 * j + i]);
                                const float sg = sigmoidf_fast(gv[i]);
                                dg[i] = v * uv[i] * (sg * (1.f + gv[i] * (1.f - sg)));
                                du[i] = v * (gv[i] * sg);
                            }
                            st_shared16(pg, pack8(dg));
                            st_shared16(pu, pack8(du));
                        }
                    }
                    fence_proxy_async();
                    __syncwarp();
                    if (leader && T.store) {
                        tma_store_3d(&P.o[0], bg, T.n0 + 64 * c, row0, z);
                        tma_store_3d(&P.o[1], bu, T.n0 + 64 * c, row0, z);
                        bulk_commit();
                    }
                }
            } else {
                // one output of 256 columns, or (wgrad gate|up) two outputs of 128 columns each
#pragma unroll 1
                for (int c = chalf * C_PER_WARP; c < (chalf + 1) * C_PER_WARP; ++c) {
                    const bool split = EPI == EPI_WGRAD_SPLIT;
                    const CUtensorMap* om = split ? &P.o[c >> 1] : &P.o[0];
                    const int col = split ? T.n0 + 64 * (c & 1) : T.n0 + 64 * c;
                    if (col >= P.n_limit) continue;
                    if (P.out_f32) {
                        // fp32 dW (main-grad style): two blocks of 32 columns x 32 rows fp32, stored or added into
                        // dW by the TMA (cp.reduce.async.bulk.tensor .add: no read-modify-write on the SM)
#pragma unroll 1
                        for (int h = 0; h < 2; ++h) {
                            if (col + 32 * h >= P.n_limit) break;
                            uint8_t* fbuf = stg + ring * STG_BYTES;
                            if (++ring == NBUF) ring = 0;
                            if (leader) bulk_wait_read<NBUF - 1>();
                            __syncwarp();
                            uint32_t r[32];
                            tmem_ld32(taddr + 64 * c + 32 * h, r);
                            tmem_ld_wait32(r);
#pragma unroll
                            for (int j = 0; j < 8; ++j) {
                                uint4 q4;
                                q4.x = zero ? 0u : r[4 * j], q4.y = zero ? 0u : r[4 * j + 1];
                                q4.z = zero ? 0u : r[4 * j + 2], q4.w = zero ? 0u : r[4 * j + 3];
                                st_shared16(stg_at(fbuf, lane, j), q4);
                            }
                            fence_proxy_async();
                            __syncwarp();
                            if (leader && T.store) {
                                if (P.accum) tma_reduce_add_3d(om, fbuf, col + 32 * h, row0, z);
                                else tma_store_3d(om, fbuf, col + 32 * h, row0, z);
                                bulk_commit();
                            }
                        }
                        continue;
                    }
                    // store warp: the four warps' blocks of chunk q lie side by side in block q & 1 (one 128-row store)
                    uint8_t* buf = store_warp ? stg_base + (ring * 4 + (uwarp - 4)) * STG_BYTES : stg + ring * STG_BYTES;
                    const int sb = ring;
                    if (++ring == NBUF) ring = 0;
                    const long long c1 = P.prof ? clock64() : 0;
                    if (store_warp) {
                        mbar_wait(&sempty_bar[sb], ((q >> 1) & 1) ^ 1);
                    } else {
                        if (leader) bulk_wait_read<NBUF - 1>();
                        __syncwarp();
                    }
                    if (P.prof) w_stg += clock64() - c1;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        uint32_t r[32];
                        tmem_ld32(taddr + 64 * c + 32 * h, r);
                        tmem_ld_wait32(r);
                        float v[32];
#pragma unroll
                        for (int i = 0; i < 32; ++i) v[i] = zero ? 0.f : __uint_as_float(r[i]);
                        stage32(buf, lane, h, v);
                    }
                    fence_proxy_async();
                    __syncwarp();
                    if (store_warp) {
                        if (leader) mbar_arrive(&sfull_bar[sb]);
                        ++q;
                    } else if (leader && T.store) {
                        tma_store_3d(om, buf, col, row0, z);
                        bulk_commit();
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (leader) mbar_arrive_cluster(leader_tempty + as * 8);
            if (++as == 2) as = 0, aphase ^= 1;
        }
        if (leader) bulk_wait_all();
        if (P.prof && threadIdx.x == 128) {
            long long* pq = P.prof + blockIdx.x * 8;
            pq[4] = w_tfull, pq[5] = clock64() - t_begin, pq[7] = w_stg;
        }
    }
    tc_fence_before();
    cluster_sync_all();  // the peer's barriers and TMEM stay alive until the leader's last commit has landed
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc2(tmem_base, 512);
    }
}


// =====================================================================================================
// Rows-on-N variant of the CTA-pair kernel for the four ragged-M contractions (fwd1, fwd2, dgrad1, dgrad2).
// The tensor core works on 128 M rows per SM whatever the tile holds, so with the packed rows on M every expert
// pays for its segment rounded up to 128 rows and, in the CTA pair, to 256.  Here the operands swap roles: the
// weights are the M operand (256 output features per CTA pair, always full) and the expert's rows are the N
// operand, which tcgen05.mma takes in multiples of 16 (N <= 256).  An expert's rows are cut into equal chunks of
// at most 256 rows rounded up to 16, so the tensor work follows the real row counts.  The accumulator holds the
// transposed tile (TMEM lane = feature, column = row); the epilogue transposes through shared memory and
// writes the row-major outputs with bulk tensor stores.
// =====================================================================================================
enum : int { TEPI_STORE = 0, TEPI_SWIGLU_FWD = 1, TEPI_SWIGLU_BWD = 2 };
constexpr int TB_BOX_ROWS = 128, TB_SMALL_ROWS = 32;  // rows per activation TMA box (long / short chunks)
constexpr int T_PANEL = 8;  // chunks per panel of the tile order (the panel's rows stay in L2 across feature tiles)
//                           // rows per activation TMA box
constexpr int TA_BYTES = 128 * BK * 2;                     // 128 features x 64 K
constexpr int TB_BYTES = 128 * BK * 2;                     // up to 128 rows x 64 K per CTA
constexpr int TSTG_BYTES = 32 * 32 * 2;                    // staging block: 32 rows x 32 features bf16
// DUAL: a tile may carry two row chunks of one expert (up to 2 x 256 rows) through one pass over the weights: a stage holds
// the weight slice once and both chunks' row slices, and both TMEM accumulators belong to the tile (see tc_gemmT_kernel).
template <int EPI, bool DUAL = false>
struct CfgT {
    static constexpr int NST = DUAL ? 4 : 5;
    static constexpr int NBUF = DUAL ? 3 : 4;              // staging blocks per epilogue warp
    static constexpr int STAGE_BYTES = TA_BYTES + (DUAL ? 2 : 1) * TB_BYTES;
    static constexpr int RING_BYTES = NST * STAGE_BYTES, STG_TOTAL = 4 * NBUF * TSTG_BYTES;
    static constexpr int XCH_BYTES = EPI == TEPI_SWIGLU_FWD ? 2 * 2 * 32 * 32 * 4 : 0;  // fp32 U exchange, 2 pairs x 2
    static constexpr int ZERO_BYTES = 16 * 32 * 2;         // a zero block for the pad rows
    static constexpr int SCHED_BYTES = 256;                // tile feed: 8 ids + 2 x 8 mbarriers
    static constexpr int SMEM = RING_BYTES + STG_TOTAL + XCH_BYTES + ZERO_BYTES + SCHED_BYTES + 1024 + 256 + 3 * (kMaxGroups2 + 1) * 4;
    static_assert(SMEM <= 232448, "shared memory per CTA");
};

struct TileT {
    int g, f, r0, n;  // group, feature tile, first packed row, rows (multiple of 16, <= 256)
    int zend;         // last chunk of a group: end of the group's padded segment (rows [r0 + n + n1, zend) are zeroed)
    int n1;           // DUAL: rows of the tile's second chunk (it starts at r0 + n), 0 = none
};
// An expert's rows are cut into nch chunks of cs rows: about equal, cs a multiple of 16 and <= 256.
__device__ __forceinline__ void t_plan(int rows, int& nch, int& cs, int greedy) {
    const int n0 = (rows + 255) >> 8;
    cs = greedy ? 256 : (n0 ? ((rows + n0 - 1) / n0 + 15) & ~15 : 16);
    nch = (rows + cs - 1) / cs;
}
// tq / so / sc: first tile, first packed row and real row count of each group, in shared memory.  dual: a tile takes two
// consecutive chunks (the last tile of a group with an odd chunk count takes one).
__device__ __forceinline__ TileT decode_t(const TcParams& P, const int* tq, const int* so, const int* sc, int t, bool dual) {
    int g = 0;
    while (g + 1 < P.G && tq[g + 1] <= t) ++g;
    const int local = t - tq[g], rows = sc[g];
    const int* offsets = so;
    int nch, cs;
    t_plan(rows, nch, cs, P.greedy);
    const int nun = dual ? (nch + 1) >> 1 : nch;  // tiles along the rows
    // panels of T_PANEL row tiles; inside a panel feature-major with the row tile fastest
    const int per_panel = T_PANEL * P.f_tiles;
    const int panel = local / per_panel, rem = local - panel * per_panel;
    const int pc = min(T_PANEL, nun - panel * T_PANEL);
    const int f = rem / pc, u = panel * T_PANEL + (rem - f * pc);
    const int c = dual ? 2 * u : u;
    const int left = rows - c * cs;
    TileT r;
    r.g = g, r.f = f, r.r0 = offsets[g] + c * cs, r.n = min(cs, (left + 15) & ~15);
    r.n1 = (dual && c + 1 < nch) ? min(cs, (left - cs + 15) & ~15) : 0;
    const bool last = (r.n1 ? c + 1 : c) == nch - 1;
    r.zend = last ? offsets[g + 1] : r.r0 + r.n + r.n1;
    return r;
}
__host__ __device__ constexpr uint32_t make_idesc_t(int a_major, int n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_major << 15) | ((uint32_t)K_MAJOR << 16) |
           ((uint32_t)(n >> 3) << 17) | ((uint32_t)((2 * BM) >> 4) << 24);
}


// GATHER (N2 fusion): the rows operand is not read from a packed buffer; warp 2 gathers row r of the tile from the
// token-major tensor P.gsrc (row src_of[r] / k) with 16-byte cp.async copies written in the same 128-byte-swizzled
// K-major layout a TMA box would have.  The leader's lanes arrive on the stage's full barrier themselves
// (cp.async.mbarrier.arrive); the peer CTA's lanes arrive on a local barrier that the peer's otherwise idle warp 1
// forwards to the leader (proxy fence + cluster-scope release).
constexpr int kGatherWarps = 2;  // GATHER: warp 2 and one extra warp (8) share the rows of a tile
template <int A_MAJOR, int EPI, bool GATHER = false, bool DUAL = false>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(GATHER ? kThreads + 32 * (kGatherWarps - 1) : kThreads, 1)
tc_gemmT_kernel(const __grid_constant__ TcParams P) {
    static_assert(!DUAL || (EPI == TEPI_STORE && !GATHER), "two-chunk tiles: plain-store kernels only");
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    using Cfg = CfgT<EPI, DUAL>;
    constexpr int NST = Cfg::NST, NBUF = Cfg::NBUF, TSTAGE = Cfg::STAGE_BYTES;
    uint8_t* stg_base = smem + Cfg::RING_BYTES;
    uint8_t* xch_base = stg_base + Cfg::STG_TOTAL;
    uint8_t* zero_blk = xch_base + Cfg::XCH_BYTES;
    uint64_t* feed_full = reinterpret_cast<uint64_t*>(zero_blk + Cfg::ZERO_BYTES);  // [kFeed] one set per CTA
    uint64_t* feed_empty = feed_full + kFeed;                                              // [kFeed] used in the leader CTA
    int* feed_ids = reinterpret_cast<int*>(feed_empty + kFeed);                            // [kFeed] one set per CTA
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(feed_full) + Cfg::SCHED_BYTES);
    uint64_t* empty_bar = full_bar + NST;                                                // one set per CTA
    uint64_t* tfull_bar = empty_bar + NST;                                               // [2] one set per CTA
    uint64_t* tempty_bar = tfull_bar + 2;                                                // [2] used in the leader CTA
    uint64_t* ld_bar = tempty_bar + 2;                                                   // [4 warps][2 sets]
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(ld_bar + 8);
    uint64_t* gfull_bar = ld_bar + 9;                                                    // [NST] GATHER: peer CTA's local "rows landed"
    static_assert((2 * NST + 4 + 9 + NST) * 8 <= 256, "barrier area");
    int* tq = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(full_bar) + 256);       // first tile of each group
    int* so = tq + (kMaxGroups2 + 1);                                                    // offsets of the groups
    int* sc = so + (kMaxGroups2 + 1);                                                    // real rows of the groups

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rank = (int)cluster_ctarank();
    const int pair_id = blockIdx.x >> 1, n_pairs_grid = gridDim.x >> 1;
    const int32_t* __restrict__ offsets = P.offsets;
    const int32_t* __restrict__ counts = P.counts;

    if (warp == 3) {  // zero block; exclusive scan of the tiles per group
        for (int i = lane; i < Cfg::ZERO_BYTES / 16; i += 32) st_shared16(zero_blk + 16 * i, make_uint4(0, 0, 0, 0));
        fence_proxy_async();
        int carry = 0;
        if (lane == 0) so[P.G] = offsets[P.G];
        for (int g0 = 0; g0 < P.G; g0 += 32) {
            const int g = g0 + lane;
            int nch = 0, cs;
            if (g < P.G) {
                const int lo = offsets[g], rows = counts ? counts[g] : offsets[g + 1] - lo;
                so[g] = lo, sc[g] = rows;
                t_plan(rows, nch, cs, P.greedy);
            }
            const int v = (DUAL ? (nch + 1) >> 1 : nch) * P.f_tiles;
            int x = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, x, o);
                if (lane >= o) x += y;
            }
            if (g < P.G) tq[g] = carry + x - v;
            carry += __shfl_sync(0xffffffffu, x, 31);
        }
        if (lane == 0) tq[P.G] = carry;
    }
    if (warp == 0 && lane == 0) {
        prefetch_tmap(&P.a[0]), prefetch_tmap(&P.b[0]);
        if (P.n_src == 2 || EPI == TEPI_SWIGLU_FWD) prefetch_tmap(&P.a[1]);
        if (P.n_src == 2) prefetch_tmap(&P.b[1]), prefetch_tmap(&P.bs[1]);
        prefetch_tmap(&P.bs[0]);
    }
    if (warp == 1 && lane == 0) {
        // full: the weight producer's expect_tx arrival + the rows producer's (TMA: one expect_tx arrival; GATHER: the
        // leader's 32 lanes + the peer's forwarder)
        for (int s = 0; s < NST; ++s)
            mbar_init(&full_bar[s], GATHER ? 2 + 32 * kGatherWarps : 2), mbar_init(&empty_bar[s], 1), mbar_init(&gfull_bar[s], 32 * kGatherWarps);
        for (int s = 0; s < 2; ++s) mbar_init(&tfull_bar[s], 1), mbar_init(&tempty_bar[s], 8);  // 4 warps x 2 CTAs
        for (int s = 0; s < 8; ++s) mbar_init(&ld_bar[s], 1);
        for (int s = 0; s < kFeed; ++s)  // + the second producer warp of each CTA (+ the peer's forwarder)
            mbar_init(&feed_full[s], 1), mbar_init(&feed_empty[s], kFeedConsumers + 2 + (GATHER ? 1 + 2 * (kGatherWarps - 1) : 0));
        fence_barrier_init();
    }
    if (warp == 2) tmem_alloc2(tmem_ptr, 512);
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr;
    const int n_total = tq[P.G];
    const int nkb = P.kb_per_src * P.n_src;
    TileFeed feed;
    feed.ids = feed_ids, feed.full = feed_full, feed.empty_addr = mapa_u32(smem_u32(feed_empty), 0);
    feed.stride = kFeedWords;
    // the tile of iteration `it` as the feeder decoded it (all lanes of a consumer warp; after feed.peek / before the release)
    auto tile_of = [&](int it) {
        const volatile int* w = feed.slot(it);
        TileT T;
        T.g = w[1], T.f = w[2], T.r0 = w[3], T.n = w[4], T.zend = w[5], T.n1 = DUAL ? w[6] : 0;
        return T;
    };

    if (warp == 3 && rank == 0 && lane == 0) {
        // ===== tile feeder (one thread of the leader CTA): draws the tile and decodes it once for every consumer warp
        // of both CTAs (the issuing thread's own decode cost 1500-2000 cycles between two tiles) =====
        const uint32_t peer_ids = mapa_u32(smem_u32(feed_ids), 1), peer_full = mapa_u32(smem_u32(feed_full), 1);
        for (int it = 0;; ++it) {
            const int slot = it & (kFeed - 1);
            mbar_wait(&feed_empty[slot], ((it / kFeed) & 1) ^ 1);
            const int t = it == 0 ? pair_id : n_pairs_grid + atomicAdd(P.sched, 1);
            int w[7] = {t, 0, 0, 0, 0, 0, 0};
            if (t < n_total) {
                const TileT T = decode_t(P, tq, so, sc, t, DUAL);
                w[1] = T.g, w[2] = T.f, w[3] = T.r0, w[4] = T.n, w[5] = T.zend, w[6] = T.n1;
            }
#pragma unroll
            for (int i = 0; i < 7; ++i) {
                *reinterpret_cast<volatile int*>(&feed_ids[slot * kFeedWords + i]) = w[i];
                asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(peer_ids + (slot * kFeedWords + i) * 4), "r"(w[i]) : "memory");
            }
            mbar_arrive(&feed_full[slot]);
            // the peer must see the id before the arrival: cluster-scope release (a membar on this otherwise idle thread)
            asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(peer_full + slot * 8) : "memory");
            if (t >= n_total) break;
        }
        // the last cluster to finish re-arms the counters for the next launch that uses this slot
        __threadfence();
        if (atomicAdd(P.sched + 1, 1) == n_pairs_grid - 1) {
            __threadfence();
            P.sched[0] = 0, P.sched[1] = 0;
        }
    }

    if (GATHER && (warp == 2 || warp >= 8)) {
        // ===== rows producers, gathered (both CTAs; kGatherWarps warps, all 32 lanes): a lane owns one 16-byte chunk
        // (ch) of the 128-byte K slice of the rows r = 8 q + 4 gw + rs; their swizzle term r & 7 = 4 gw + rs is a constant of
        // the lane, so the destination of copy q is a fixed address + q * 1024 =====
        const int gw = warp == 2 ? 0 : warp - 7;
        const int ch = lane & 7, rs = lane >> 3, r_lane = 4 * gw + rs;
        const char* gbase = static_cast<const char*>(P.gsrc);
        const uint32_t pitch16 = (uint32_t)P.g_cols >> 3;  // 16-byte units per source row
        const uint32_t dst_lane = smem_u32(smem) + TA_BYTES + r_lane * 128 + ((ch ^ r_lane) << 4);
        constexpr int NQ = 128 / (4 * kGatherWarps);  // copies per lane and K block at most
        int stage = 0, phase = 0;
        for (int it = 0;; ++it) {
            const int t = feed.peek(it);
            const TileT T = tile_of(it);
            feed.release(it, lane);
            if (t >= n_total) break;
            const int nb = T.n >> 1, rb = T.r0 + rank * nb;
            uint32_t off[NQ];   // source row of tile row 8 q + r_lane in 16-byte units
            uint32_t zmask = 0; // bit q: pad row (zero fill)
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const int r = 4 * kGatherWarps * q + r_lane;
                const int a = r < nb ? P.src_of[rb + r] : -1;
                off[q] = a >= 0 ? (uint32_t)(((unsigned long long)a * P.g_magic) >> 35) * pitch16 : 0u;
                zmask |= a >= 0 ? 0u : 1u << q;
            }
            const int nq = (nb - r_lane + 4 * kGatherWarps - 1) / (4 * kGatherWarps);  // rows r < nb
            for (int kb = 0; kb < nkb; ++kb) {
                if (lane == 0) mbar_wait(&empty_bar[stage], phase ^ 1);
                __syncwarp();
                const uint32_t dst = dst_lane + stage * TSTAGE;
                const int kcol = kb * BK + ch * 8;
                const uint32_t k_bad = kcol < P.g_cols ? 0u : 0xFFFFFFFFu;  // K tail: zero fill, as a TMA box does
                const char* src_k = gbase + (k_bad ? 0 : (size_t)kcol * 2);
#pragma unroll
                for (int q = 0; q < NQ; ++q)
                    if (q < nq) cp_async16_z(dst + q * (4 * kGatherWarps * 128), src_k + (size_t)off[q] * 16, (zmask & (1u << q)) | k_bad);
                cp_async_arrive(rank == 0 ? &full_bar[stage] : &gfull_bar[stage]);
                if (++stage == NST) stage = 0, phase ^= 1;
            }
        }
    } else if (GATHER && warp == 1 && rank == 1) {
        // ===== peer CTA: forward "my rows of this stage have landed" to the leader's full barrier =====
        const uint32_t leader_full = mapa_u32(smem_u32(full_bar), 0);
        int stage = 0, phase = 0;
        for (int it = 0;; ++it) {
            const int t = feed.peek(it);
            feed.release(it, lane);
            if (t >= n_total) break;
            for (int kb = 0; kb < nkb; ++kb) {
                if (lane == 0) {
                    mbar_wait(&gfull_bar[stage], phase);
                    fence_proxy_async();  // the copies are generic-proxy writes; the tensor core reads through the async proxy
                    // plain remote arrive: the cluster-scope release form is a GPU-scope membar per K block (1-2 us in this
                    // thread: the whole kernel ran at its pace).  The rows are read by this CTA's own tensor core, after the
                    // proxy fence above; the arrival only tells the leader that it may issue.
                    mbar_arrive_cluster(leader_full + stage * 8);
                }
                __syncwarp();
                if (++stage == NST) stage = 0, phase ^= 1;
            }
        }
    } else if (warp == 0 || warp == 2) {
        // ===== TMA producers (both CTAs): warp 0 loads the CTA's 128 features of the weights, warp 2 (idle after the
        // TMEM allocation) its half of the rows.  The warps run converged; one elected lane issues the copies. =====
        const bool load_a = uni(warp) == 0;
        const uint32_t leader_full = uni(mapa_u32(smem_u32(full_bar), 0));
        const int urank = uni(rank);
        int stage = 0, phase = 0;
        long long w_empty = 0;
        for (int it = 0;; ++it) {
            const int t = uni(feed.peek(it));
            TileT T = tile_of(it);
            T.g = uni(T.g), T.f = uni(T.f), T.r0 = uni(T.r0), T.n = uni(T.n), T.n1 = uni(T.n1);
            feed.release(it, lane);
            if (t >= n_total) break;
            const int nb = T.n >> 1, rb = T.r0 + urank * nb;
            const bool small = nb <= P.small_rows;
            const int nbox = small ? (nb + TB_SMALL_ROWS - 1) / TB_SMALL_ROWS : 1;
            const int box_bytes = (small ? TB_SMALL_ROWS : TB_BOX_ROWS) * BK * 2;
            // DUAL: the second chunk's half of this CTA, behind the first one's slot
            const int nb1 = T.n1 >> 1, rb1 = T.r0 + T.n + urank * nb1;
            const bool small1 = nb1 <= P.small_rows;
            const int nbox1 = nb1 == 0 ? 0 : (small1 ? (nb1 + TB_SMALL_ROWS - 1) / TB_SMALL_ROWS : 1);
            const int box_bytes1 = (small1 ? TB_SMALL_ROWS : TB_BOX_ROWS) * BK * 2;
            for (int kb = 0; kb < nkb; ++kb) {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&empty_bar[stage], phase ^ 1);
                if (P.prof) w_empty += clock64() - c0;
                if (elect_one()) {
                    uint8_t* sa = smem + stage * TSTAGE;
                    uint8_t* sb = sa + TA_BYTES;
                    if (urank == 0)
                        mbar_expect_tx(&full_bar[stage], load_a ? 2 * TA_BYTES : 2 * (nbox * box_bytes + (DUAL ? nbox1 * box_bytes1 : 0)));
                    const uint32_t bar = leader_full + stage * 8;
                    int src = 0, kk = kb;
                    if (kb >= P.kb_per_src) src = 1, kk = kb - P.kb_per_src;
                    const int k = kk * BK;
                    if (!load_a) {
                        if (small) {
                            for (int i = 0; i < nbox; ++i)
                                tma_load_3d_pair(sb + i * box_bytes, &P.bs[src], bar, k, rb + i * TB_SMALL_ROWS, 0);
                        } else {
                            tma_load_3d_pair(sb, &P.b[src], bar, k, rb, 0);
                        }
                        if (DUAL && nb1) {
                            uint8_t* sb1 = sb + TB_BYTES;
                            if (small1) {
                                for (int i = 0; i < nbox1; ++i)
                                    tma_load_3d_pair(sb1 + i * box_bytes1, &P.bs[src], bar, k, rb1 + i * TB_SMALL_ROWS, 0);
                            } else {
                                tma_load_3d_pair(sb1, &P.b[src], bar, k, rb1, 0);
                            }
                        }
                    } else if (EPI == TEPI_SWIGLU_FWD) {  // 64 gate features | the same 64 up features
                        const int fc = T.f * 128 + urank * 64;
                        tma_load_3d_pair(sa, &P.a[0], bar, fc, k, T.g);
                        tma_load_3d_pair(sa + MN_BLOCK_BYTES, &P.a[1], bar, fc, k, T.g);
                    } else if (A_MAJOR == MN_MAJOR) {
                        const int fc = T.f * 256 + urank * 128;
                        tma_load_3d_pair(sa, &P.a[src], bar, fc, k, T.g);
                        tma_load_3d_pair(sa + MN_BLOCK_BYTES, &P.a[src], bar, fc + 64, k, T.g);
                    } else {
                        tma_load_3d_pair(sa, &P.a[src], bar, k, T.f * 256 + urank * 128, T.g);
                    }
                }
                __syncwarp();
                if (++stage == NST) stage = 0, phase ^= 1;
            }
        }
        if (P.prof && lane == 0 && load_a) P.prof[blockIdx.x * 8 + 3] = w_empty;
    } else if (warp == 1 && rank == 0) {
        // ===== MMA issuer (warp 1 of the leader CTA, converged; one elected lane issues): D^T[256 features, n rows] += W-tile * rows^T
        constexpr uint32_t a_lbo = A_MAJOR == K_MAJOR ? 16 : MN_BLOCK_BYTES;
        constexpr uint32_t a_kstep = A_MAJOR == K_MAJOR ? UK * 2 : UK * 128;
        const uint32_t smem_base = uni(smem_u32(smem)), tmem_u = uni(tmem_base);
        // descriptors of stage 0, K step 0: the address field (bits 0-13, 16-byte units) advances by plain additions
        const uint64_t a_desc0 = make_desc(smem_base, a_lbo, 1024), b_desc0 = make_desc(smem_base + TA_BYTES, 16, 1024);
        int stage = 0, phase = 0, as = 0, aphase = 0;
        long long w_full = 0, w_tempty = 0, n_tiles_done = 0;
        const long long t_begin = P.prof ? clock64() : 0;
        for (int it = 0;; ++it) {
            const int t = uni(feed.peek(it));
            const int tn = uni(tile_of(it).n), tn1 = DUAL ? uni(tile_of(it).n1) : 0;
            feed.release(it, lane);
            if (t >= n_total) break;
            const uint32_t idesc = make_idesc_t(A_MAJOR, tn);
            {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&tempty_bar[as], aphase ^ 1);
                if (P.prof) w_tempty += clock64() - c0, ++n_tiles_done;
                tc_fence_after();
            }
            const uint32_t d_tmem = tmem_u + as * BN;
            // DUAL: the tile's second chunk accumulates in the other buffer (the next one in the epilogue's order), from
            // the same weight slice of every stage
            const int as1 = as ^ 1, aphase1 = as == 1 ? aphase ^ 1 : aphase;
            const uint32_t idesc1 = make_idesc_t(A_MAJOR, tn1 ? tn1 : 16), d_tmem1 = tmem_u + as1 * BN;
            if (DUAL && tn1) {
                mbar_wait(&tempty_bar[as1], aphase1 ^ 1);
                tc_fence_after();
            }
            for (int kb = 0; kb < nkb; ++kb) {
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&full_bar[stage], phase);
                if (GATHER) fence_proxy_async();  // gathered rows were written through the generic proxy
                if (P.prof) w_full += clock64() - c0;
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t soff = (uint32_t)(stage * TSTAGE) >> 4;
#pragma unroll
                    for (int kk = 0; kk < BK / UK; ++kk) {
                        const uint64_t ad = a_desc0 + (soff + ((kk * a_kstep) >> 4));
                        const uint64_t bd = b_desc0 + (soff + ((kk * UK * 2) >> 4));
                        umma2_bf16(d_tmem, ad, bd, idesc, (kb | kk) != 0);
                    }
                    if (DUAL && tn1) {
#pragma unroll
                        for (int kk = 0; kk < BK / UK; ++kk) {
                            const uint64_t ad = a_desc0 + (soff + ((kk * a_kstep) >> 4));
                            const uint64_t bd = b_desc0 + (soff + ((TB_BYTES + kk * UK * 2) >> 4));
                            umma2_bf16(d_tmem1, ad, bd, idesc1, (kb | kk) != 0);
                        }
                    }
                    umma2_commit(&empty_bar[stage]);
                }
                __syncwarp();
                if (++stage == NST) stage = 0, phase ^= 1;
            }
            if (elect_one()) {
                umma2_commit(&tfull_bar[as]);
                if (DUAL && tn1) umma2_commit(&tfull_bar[as1]);
            }
            __syncwarp();
            if (++as == 2) as = 0, aphase ^= 1;
            if (DUAL && tn1 && ++as == 2) as = 0, aphase ^= 1;
        }
        if (P.prof && lane == 0) {
            long long* pq = P.prof + blockIdx.x * 8;
            pq[0] = w_full, pq[1] = w_tempty, pq[2] = clock64() - t_begin, pq[6] = n_tiles_done;
        }
    } else if (warp >= 4) {
        // ===== epilogue (both CTAs): TMEM lane = feature, column = row; transposed through shared memory =====
        // (warp-uniform values are made provably so, and one elected lane issues the bulk tensor copies: see elect_one)
        const int wq = uni(warp) & 3, urank = uni(rank);
        const bool leader = elect_one();
        const uint32_t leader_tempty = uni(mapa_u32(smem_u32(tempty_bar), 0));
        uint8_t* stg = stg_base + wq * NBUF * TSTG_BYTES;
        int as = 0, aphase = 0, ring = 0;
        long long w_tfull = 0, w_stg = 0;
        const long long t_begin = P.prof ? clock64() : 0;
        uint32_t q = 0;  // running 32-row block number (SwiGLU epilogues: exchange slot / input set q & 1)
        // one staged block [32 rows][32 features] -> out rows row.. (the second 16-row half only if `both`)
        auto store_block = [&](const CUtensorMap* om, const uint8_t* buf, int fcol, int row, bool both) {
            tma_store_3d(om, buf, fcol, row, 0);
            if (both) tma_store_3d(om, buf + TSTG_BYTES / 2, fcol, row + 16, 0);
        };
        auto stage_col = [&](uint8_t* buf, const float* v) {  // this thread's feature: 32 rows of one column
            const uint32_t a = smem_u32(buf) + lane * 2;
#pragma unroll
            for (int i = 0; i < 32; i += 2) {
                const uint32_t pk = f2_to_bf2(v[i], v[i + 1]);
                sts_u16(a + i * 64, pk & 0xffffu);
                sts_u16(a + (i + 1) * 64, pk >> 16);
            }
        };
        auto next_buf = [&]() {
            uint8_t* buf = stg + ring * TSTG_BYTES;
            if (++ring == NBUF) ring = 0;
            return buf;
        };
        // SwiGLU backward: G, U of 32 rows x 32 features -> input set `set` (two staging blocks)
        auto load_inputs = [&](int fcol, int row, int set) {
            if (leader) {
                bulk_wait_read<0>();
                uint64_t* bar = &ld_bar[wq * 2 + set];
                mbar_expect_tx(bar, 2 * TSTG_BYTES);
                tma_load_3d(stg + (2 * set) * TSTG_BYTES, &P.ein[0], bar, fcol, row, 0);
                tma_load_3d(stg + (2 * set + 1) * TSTG_BYTES, &P.ein[1], bar, fcol, row, 0);
            }
        };
        const int pr = wq & 1;  // SwiGLU forward: warps pr (G lanes) and pr + 2 (U lanes) hold the same 32 features
        auto feat_col = [&](const TileT& T) {
            return EPI == TEPI_SWIGLU_FWD ? T.f * 128 + urank * 64 + 32 * pr : T.f * 256 + urank * 128 + 32 * wq;
        };
        if (EPI == TEPI_SWIGLU_BWD) {
            const int t0 = uni(feed.peek(0));
            if (t0 < n_total) {
                TileT T0 = tile_of(0);
                T0.f = uni(T0.f), T0.r0 = uni(T0.r0);
                load_inputs(feat_col(T0), T0.r0, 0);
            }
        }
        for (int it = 0;; ++it) {
            const int t = uni(feed.peek(it));
            TileT T = tile_of(it);
            T.g = uni(T.g), T.f = uni(T.f), T.r0 = uni(T.r0), T.n = uni(T.n), T.zend = uni(T.zend), T.n1 = uni(T.n1);
            feed.release(it, lane);
            if (t >= n_total) break;
            // DUAL: a tile's two chunks are drained one after the other, the second from the other accumulator
            const int n_half = (DUAL && T.n1) ? 2 : 1;
#pragma unroll 1
            for (int half = 0; half < n_half; ++half) {
                TileT H = T;
                if (half) H.r0 = T.r0 + T.n, H.n = T.n1;
                if (half + 1 < n_half) H.zend = T.r0 + T.n;
                const long long c0 = P.prof ? clock64() : 0;
                mbar_wait(&tfull_bar[as], aphase);
                if (P.prof) w_tfull += clock64() - c0;
                tc_fence_after();
                const uint32_t taddr = tmem_base + ((uint32_t)(wq * 32) << 16) + as * BN;
                const int fcol = feat_col(H);
                const bool f_ok = fcol < P.f_limit;
    #pragma unroll 1
                for (int j = 0; j < H.n; j += 32, ++q) {
                    const bool both = j + 16 < H.n;
                    uint32_t r[32];
                    float v[32];
                    if (EPI == TEPI_STORE) {
                        if (!f_ok) break;
                        uint8_t* buf = next_buf();
                        if (leader) bulk_wait_read<NBUF - 1>();
                        __syncwarp();
                        tmem_ld32(taddr + j, r);
                        tmem_ld_wait32(r);
    #pragma unroll
                        for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
                        stage_col(buf, v);
                        fence_proxy_async();
                        __syncwarp();
                        if (leader) {
                            store_block(&P.o[0], buf, fcol, H.r0 + j, both);
                            bulk_commit();
                        }
                    } else if (EPI == TEPI_SWIGLU_FWD) {
                        const uint32_t xch = smem_u32(xch_base) + (pr * 2 + (q & 1)) * 4096 + lane * 4;
                        tmem_ld32(taddr + j, r);
                        tmem_ld_wait32(r);
    #pragma unroll
                        for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
                        if (wq >= 2) {  // U lanes: hand the fp32 values to the G warp, store U
    #pragma unroll
                            for (int i = 0; i < 32; ++i) sts_f32(xch + i * 128, v[i]);
                            asm volatile("bar.sync %0, 64;" ::"r"(1 + pr) : "memory");
                            uint8_t* buf = next_buf();
                            if (leader) bulk_wait_read<NBUF - 1>();
                            __syncwarp();
                            stage_col(buf, v);
                            fence_proxy_async();
                            __syncwarp();
                            if (leader && f_ok) {
                                store_block(&P.o[1], buf, fcol, H.r0 + j, both);
                                bulk_commit();
                            }
                        } else {  // G lanes: store G, H = silu(G) * U
                            uint8_t* bg = next_buf();
                            uint8_t* bh = next_buf();
                            if (leader) bulk_wait_read<1>();  // two blocks per commit group, ring of four
                            __syncwarp();
                            stage_col(bg, v);
                            asm volatile("bar.sync %0, 64;" ::"r"(1 + pr) : "memory");
    #pragma unroll
                            for (int i = 0; i < 32; ++i) v[i] = v[i] * sigmoidf_fast(v[i]) * lds_f32(xch + i * 128);
                            stage_col(bh, v);
                            fence_proxy_async();
                            __syncwarp();
                            if (leader && f_ok) {
                                store_block(&P.o[0], bg, fcol, H.r0 + j, both);
                                store_block(&P.o[2], bh, fcol, H.r0 + j, both);
                                bulk_commit();
                            }
                        }
                    } else {
                        // accumulator = dH; dG = dH * U * silu'(G), dU = dH * silu(G), in place over the staged G, U
                        const int set = q & 1;
                        const uint32_t bg = smem_u32(stg + (2 * set) * TSTG_BYTES) + lane * 2, bu = bg + TSTG_BYTES;
                        const long long c1 = P.prof ? clock64() : 0;
                        mbar_wait(&ld_bar[wq * 2 + set], (q >> 1) & 1);
                        if (P.prof) w_stg += clock64() - c1;
                        if (j + 32 < H.n) {
                            load_inputs(fcol, H.r0 + j + 32, set ^ 1);
                        } else {
                            const int tn = uni(feed.peek(it + 1));
                            if (tn < n_total) {
                                TileT Tn = tile_of(it + 1);
                                Tn.f = uni(Tn.f), Tn.r0 = uni(Tn.r0);
                                load_inputs(feat_col(Tn), Tn.r0, set ^ 1);
                            }
                        }
                        tmem_ld32(taddr + j, r);
                        tmem_ld_wait32(r);
                        // gathered dY rows are unscaled: dH[r] = gate_rows[r] * (dY[token(r)] Wd^T), the gate applied in fp32
                        const float* rsc = P.row_scale ? P.row_scale + H.r0 + j : nullptr;
    #pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            float dg[2], du[2];
    #pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const float dh = __uint_as_float(r[i + e]) * ((rsc && i + e < H.n - j) ? __ldg(rsc + i + e) : 1.f);
                                const float gv = lds_bf16(bg + (i + e) * 64), uv = lds_bf16(bu + (i + e) * 64);
                                const float sg = sigmoidf_fast(gv);
                                dg[e] = dh * uv * (sg * (1.f + gv * (1.f - sg)));
                                du[e] = dh * (gv * sg);
                            }
                            const uint32_t pg = f2_to_bf2(dg[0], dg[1]), pu = f2_to_bf2(du[0], du[1]);
                            sts_u16(bg + i * 64, pg & 0xffffu), sts_u16(bg + (i + 1) * 64, pg >> 16);
                            sts_u16(bu + i * 64, pu & 0xffffu), sts_u16(bu + (i + 1) * 64, pu >> 16);
                        }
                        fence_proxy_async();
                        __syncwarp();
                        if (leader && f_ok) {
                            store_block(&P.o[0], stg + (2 * set) * TSTG_BYTES, fcol, H.r0 + j, both);
                            store_block(&P.o[1], stg + (2 * set + 1) * TSTG_BYTES, fcol, H.r0 + j, both);
                            bulk_commit();
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (leader) mbar_arrive_cluster(leader_tempty + as * 8);
                if (++as == 2) as = 0, aphase ^= 1;
                // pad rows behind the group's last chunk: exact zeros (wgrad reads them as part of its K range)
                if (leader && f_ok && H.r0 + H.n < H.zend) {
                    for (int row = H.r0 + H.n; row < H.zend; row += 16) {
                        if (EPI == TEPI_STORE) {
                            tma_store_3d(&P.o[0], zero_blk, fcol, row, 0);
                        } else if (EPI == TEPI_SWIGLU_FWD) {
                            if (wq >= 2) {
                                tma_store_3d(&P.o[1], zero_blk, fcol, row, 0);
                            } else {
                                tma_store_3d(&P.o[0], zero_blk, fcol, row, 0);
                                tma_store_3d(&P.o[2], zero_blk, fcol, row, 0);
                            }
                        } else {
                            tma_store_3d(&P.o[0], zero_blk, fcol, row, 0);
                            tma_store_3d(&P.o[1], zero_blk, fcol, row, 0);
                        }
                    }
                    bulk_commit();
                }
        
            }
        }
        if (leader) bulk_wait_all();
        if (P.prof && threadIdx.x == 128) {
            long long* pq = P.prof + blockIdx.x * 8;
            pq[4] = w_tfull, pq[5] = clock64() - t_begin, pq[7] = w_stg;
        }
    }
    tc_fence_before();
    cluster_sync_all();
    if (warp == 2) {
        tc_fence_after();
        tmem_dealloc2(tmem_base, 512);
    }
}

// ---- host side ------------------------------------------------------------------------------------------
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// bf16 tensor [groups][rows][inner] (row-major), box = box_inner elements x box_rows rows; 128-byte swizzle when the
// box is 64 elements (128 B) wide, else none.
// The same maps are needed every step (the caller's pointers do not change): keep the encoded descriptors, keyed by
// everything cuTensorMapEncodeTiled was given (open addressing, overwritten on collision of a full probe window).
MapCacheEntry* map_cache_find(piper_ctx* c, const void* base, long long inner, long long rows, long long groups,
                              int box_inner, int box_rows, int kind, bool* hit) {
    *hit = false;
    if (!c->map_cache) return nullptr;
    uint64_t h = reinterpret_cast<uintptr_t>(base) * 0x9E3779B97F4A7C15ull;
    h ^= (uint64_t)inner * 0xC2B2AE3D27D4EB4Full + (uint64_t)rows * 0x165667B19E3779F9ull + (uint64_t)groups * 31 +
         (uint64_t)box_inner * 131 + (uint64_t)box_rows * 8191 + (uint64_t)kind;
    h ^= h >> 29;
    const int start = (int)(h % kMapCache);
    for (int i = 0; i < 8; ++i) {
        MapCacheEntry* e = &c->map_cache[(start + i) % kMapCache];
        if (e->kind == 0) return e;
        if (e->kind == kind && e->base == base && e->inner == inner && e->rows == rows && e->groups == groups &&
            e->box_inner == box_inner && e->box_rows == box_rows) {
            *hit = true;
            return e;
        }
    }
    return &c->map_cache[start];  // probe window full: recycle its first entry
}
void map_cache_fill(MapCacheEntry* e, const CUtensorMap* m, const void* base, long long inner, long long rows,
                    long long groups, int box_inner, int box_rows, int kind) {
    if (!e) return;
    e->base = base, e->inner = inner, e->rows = rows, e->groups = groups;
    e->box_inner = box_inner, e->box_rows = box_rows, e->kind = kind, e->map = *m;
}

int make_map2(piper_ctx* c, CUtensorMap* m, const void* base, long long inner, long long rows, long long groups,
              int box_inner, int box_rows) {
    bool hit;
    MapCacheEntry* ce = map_cache_find(c, base, inner, rows, groups, box_inner, box_rows, 1, &hit);
    if (hit) {
        *m = ce->map;
        return PIPER_OK;
    }
    const cuuint64_t dims[3] = {(cuuint64_t)inner, (cuuint64_t)rows, (cuuint64_t)groups};
    const cuuint64_t strides[2] = {(cuuint64_t)inner * 2, (cuuint64_t)inner * 2 * (cuuint64_t)rows};
    const cuuint32_t box[3] = {(cuuint32_t)box_inner, (cuuint32_t)box_rows, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = reinterpret_cast<EncodeTiledFn>(c->encode_tiled)(
        m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
        CU_TENSOR_MAP_INTERLEAVE_NONE, box_inner == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(c->err, sizeof(c->err), "cuTensorMapEncodeTiled failed (%d): inner %lld rows %lld groups %lld box %dx%d",
                 (int)r, inner, rows, groups, box_inner, box_rows);
        return PIPER_ERR_CUDA;
    }
    map_cache_fill(ce, m, base, inner, rows, groups, box_inner, box_rows, 1);
    return PIPER_OK;
}
int make_map(piper_ctx* c, CUtensorMap* m, const void* base, long long inner, long long rows, long long groups,
             int box_rows) {
    return make_map2(c, m, base, inner, rows, groups, 64, box_rows);
}
// fp32 tensor [groups][rows][inner], box = 32 columns (128 B, swizzled) x 32 rows: the fp32 dW outputs of wgrad
int make_map_f32(piper_ctx* c, CUtensorMap* m, const void* base, long long inner, long long rows, long long groups) {
    bool hit;
    MapCacheEntry* ce = map_cache_find(c, base, inner, rows, groups, 32, 32, 2, &hit);
    if (hit) {
        *m = ce->map;
        return PIPER_OK;
    }
    const cuuint64_t dims[3] = {(cuuint64_t)inner, (cuuint64_t)rows, (cuuint64_t)groups};
    const cuuint64_t strides[2] = {(cuuint64_t)inner * 4, (cuuint64_t)inner * 4 * (cuuint64_t)rows};
    const cuuint32_t box[3] = {32, 32, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = reinterpret_cast<EncodeTiledFn>(c->encode_tiled)(
        m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(base), dims, strides, box, estr,
        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(c->err, sizeof(c->err), "cuTensorMapEncodeTiled (fp32) failed (%d): inner %lld rows %lld groups %lld", (int)r,
                 inner, rows, groups);
        return PIPER_ERR_CUDA;
    }
    map_cache_fill(ce, m, base, inner, rows, groups, 32, 32, 2);
    return PIPER_OK;
}
#define PIPER_MAP2(...)                                \
    do {                                               \
        const int rc__ = make_map2(c, __VA_ARGS__);    \
        if (rc__ != PIPER_OK) return rc__;             \
    } while (0)
#define PIPER_MAP(...)                                 \
    do {                                               \
        const int rc__ = make_map(c, __VA_ARGS__);     \
        if (rc__ != PIPER_OK) return rc__;             \
    } while (0)

// Co-resident CTA pairs of a cluster kernel on the lane's stream (a green-context partition may hold fewer whole
// pairs than sms / 2): the persistent grids stride over this many pairs, so it must not exceed what fits at once.
// Queried once per (kernel, SM count of the lane) and kept.
template <typename K>
int resident_clusters(piper_ctx* c, Lane ln, K kernel, int smem_bytes, int threads = kThreads) {
    const void* key = reinterpret_cast<const void*>(kernel);
    const int used = c->cluster_cache_used < kClusterCache ? c->cluster_cache_used : kClusterCache;
    for (int i = 0; i < used; ++i) {
        const ClusterCacheEntry& e = c->cluster_cache[i];
        if (e.fn == key && e.sms == ln.sms && e.stream == ln.stream) return e.n;
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = 2, attr.val.clusterDim.y = 1, attr.val.clusterDim.z = 1;
    cfg.gridDim = dim3(2 * (ln.sms / 2)), cfg.blockDim = dim3(threads), cfg.dynamicSmemBytes = smem_bytes;
    cfg.stream = ln.stream, cfg.attrs = &attr, cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, kernel, &cfg) != cudaSuccess || n < 1) {
        cudaGetLastError();
        n = ln.sms / 2;
    }
    if (n > ln.sms / 2) n = ln.sms / 2;
    ClusterCacheEntry& e = c->cluster_cache[c->cluster_cache_used++ % kClusterCache];
    e.fn = key, e.stream = ln.stream, e.sms = ln.sms, e.n = n;
    return n;
}

// The {next tile, clusters done} counters of a launch on `stream`: see SchedSlot (piper_internal.cuh).
int* sched_counters(piper_ctx* c, cudaStream_t stream) {
    return reinterpret_cast<int*>(c->tc_scratch + (size_t)kProfSlots * kProfSlotWords * 8) + 2 * stream_slot(c, stream);
}

template <int A_MAJOR, int B_MAJOR, int EPI, bool GATHER_A = false>
int launch(piper_ctx* c, Lane ln, const TcParams& P, long long tile_bound, bool two_cta, const char* name) {
    TcParams Q = P;
    if (c->tc_prof) {  // debug: slot per launch, cycled
        Q.prof = reinterpret_cast<long long*>(c->tc_scratch) + (size_t)(c->tc_next_slot % kProfSlots) * kProfSlotWords;
        c->tc_next_slot += 1;
    }
    if (two_cta) {
        // tile_bound counts tile pairs; one cluster of two CTAs per pair, one CTA per SM
        constexpr int threads = Cfg2<EPI>::THREADS + (GATHER_A ? 32 * (kGatherWarpsA - 1) : 0);
        long long clusters = resident_clusters(c, ln, tc_gemm2_kernel<A_MAJOR, B_MAJOR, EPI, GATHER_A>, Cfg2<EPI>::SMEM, threads);
        if (tile_bound < clusters) clusters = tile_bound;
        if (clusters < 1) clusters = 1;
        Q.sched = sched_counters(c, ln.stream);
        tc_gemm2_kernel<A_MAJOR, B_MAJOR, EPI, GATHER_A><<<(unsigned)(2 * clusters), threads, Cfg2<EPI>::SMEM, ln.stream>>>(Q);
        PIPER_LAUNCHED(c, name);
        return PIPER_OK;
    }
    if (GATHER_A) return PIPER_ERR_UNSUPPORTED;  // the gather exists in the CTA-pair kernel only
    long long grid = tile_bound < ln.sms ? tile_bound : ln.sms;
    if (grid < 1) grid = 1;
    tc_gemm_kernel<A_MAJOR, B_MAJOR, EPI><<<(unsigned)grid, kThreads, SMEM_BYTES, ln.stream>>>(Q);
    PIPER_LAUNCHED(c, name);
    return PIPER_OK;
}

template <int A_MAJOR, int B_MAJOR, int EPI>
bool set_smem_attr() {
    return cudaFuncSetAttribute(tc_gemm_kernel<A_MAJOR, B_MAJOR, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                SMEM_BYTES) == cudaSuccess &&
           cudaFuncSetAttribute(tc_gemm2_kernel<A_MAJOR, B_MAJOR, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                Cfg2<EPI>::SMEM) == cudaSuccess;
}

template <int A_MAJOR, int B_MAJOR, int EPI>
bool set_smem_attr1() {  // 1-CTA kernel only (the router's dense GEMMs)
    return cudaFuncSetAttribute(tc_gemm_kernel<A_MAJOR, B_MAJOR, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                SMEM_BYTES) == cudaSuccess;
}

template <int A_MAJOR, int EPI, bool GATHER = false, bool DUAL = false>
int launch_t(piper_ctx* c, Lane ln, const TcParams& P, long long tile_bound, const char* name) {
    constexpr int threads = GATHER ? kThreads + 32 * (kGatherWarps - 1) : kThreads;
    long long clusters = resident_clusters(c, ln, tc_gemmT_kernel<A_MAJOR, EPI, GATHER, DUAL>, CfgT<EPI, DUAL>::SMEM, threads);
    if (tile_bound < clusters) clusters = tile_bound;
    if (clusters < 1) clusters = 1;
    TcParams Q = P;
    if (c->tc_prof) {  // debug: slot per launch, cycled
        Q.prof = reinterpret_cast<long long*>(c->tc_scratch) + (size_t)(c->tc_next_slot % kProfSlots) * kProfSlotWords;
        c->tc_next_slot += 1;
    }
    Q.sched = sched_counters(c, ln.stream);
    tc_gemmT_kernel<A_MAJOR, EPI, GATHER, DUAL><<<(unsigned)(2 * clusters), threads, CfgT<EPI, DUAL>::SMEM, ln.stream>>>(Q);
    PIPER_LAUNCHED(c, name);
    return PIPER_OK;
}
template <int A_MAJOR, int EPI, bool GATHER = false, bool DUAL = false>
bool set_smem_attr_t() {
    return cudaFuncSetAttribute(tc_gemmT_kernel<A_MAJOR, EPI, GATHER, DUAL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                CfgT<EPI, DUAL>::SMEM) == cudaSuccess;
}
// gather fields of a launch whose rows operand comes from the token-major tensor `src` [T, cols]
void set_gather(TcParams& P, const piper_ctx* c, const FfnProblem& p, const void* src, int cols) {
    P.src_of = p.src_of, P.gsrc = src, P.g_cols = cols;
    P.g_magic = ((1ull << 35) + (unsigned long long)c->D.k - 1) / (unsigned long long)c->D.k;
}
// rows-on-N kernel for the ragged-M contractions (PIPER_OPT_TC_ROWS_ON_N = 0 switches it off)
bool rows_on_n(const piper_ctx* c, const FfnProblem& p) { return c->tc_rows_on_n && p.G <= kMaxGroups2; }
TcParams t_params(const piper_ctx* c, const FfnProblem& p, int F, int K, int f_tile) {
    TcParams P;
    memset(&P, 0, sizeof(P));
    P.offsets = p.offsets, P.counts = p.counts, P.G = p.G, P.n_src = 1;
    P.f_tiles = cdiv(F, f_tile), P.f_limit = F, P.kb_per_src = cdiv(K, BK);
    P.small_rows = c->tc_small_rows, P.greedy = c->tc_greedy;
    return P;
}
// two-chunk tiles (DUAL) for the plain-store rows-on-N kernels: when a group can hold more than one chunk
bool dual_tiles(const piper_ctx* c, const FfnProblem& p) { return c->tc_dual && p.max_group_rows > 256; }
inline long long t_tile_bound(const FfnProblem& p, int f_tiles) { return (long long)(cdiv(p.max_rows, 256) + p.G) * f_tiles; }

// Pairing M tiles of one expert costs a duplicate tile per odd group: use the CTA-pair kernel when the groups are
// long enough for that to be small (host-side expectation; the sizes themselves stay on the device).
bool pair_ragged(const piper_ctx* c, const FfnProblem& p) {
    if (c->tc_two_cta == 0 || p.G > kMaxGroups2) return false;
    if (c->tc_two_cta == 1) return true;
    return (long long)p.exp_rows >= (long long)p.G * 4 * BM || p.G == 1;
}
bool pair_wgrad(const piper_ctx* c, const FfnProblem& p) { return c->tc_two_cta != 0 && p.G <= kMaxGroups2; }

TcParams base_params(const FfnProblem& p, bool ragged_m) {
    TcParams P;
    memset(&P, 0, sizeof(P));
    P.offsets = p.offsets, P.G = p.G, P.ragged_m = ragged_m ? 1 : 0, P.n_src = 1, P.tile_n = BN;
    return P;
}
inline long long m_tile_bound(const FfnProblem& p, bool two) {
    // pairs: sum_g ceil(tiles_g / 2) <= (tiles + G) / 2
    return two ? (cdiv(p.max_rows, BM) + p.G + 1) / 2 : cdiv(p.max_rows, BM);
}

}  // namespace

size_t tc_scratch_bytes(const piper_moe_desc*) { return (size_t)kProfSlots * kProfSlotWords * 8 + kSchedSlots * 8; }

void tc_release(piper_ctx* c) {
    delete[] c->map_cache;
    c->map_cache = nullptr;
}

void tc_forget_stream(piper_ctx* c, cudaStream_t stream) {
    for (int i = 0; i < kSchedSlots; ++i)
        if (c->sched_slots[i].used && c->sched_slots[i].stream == stream) c->sched_slots[i].used = false;
    int n = 0;
    const int used = c->cluster_cache_used < kClusterCache ? c->cluster_cache_used : kClusterCache;
    for (int i = 0; i < used; ++i)
        if (c->cluster_cache[i].stream != stream) c->cluster_cache[n++] = c->cluster_cache[i];
    c->cluster_cache_used = n;
}

int tc_init(piper_ctx* c) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
        fn = nullptr;
    cudaGetLastError();
    c->encode_tiled = fn;
    if (cudaMemset(c->tc_scratch + (size_t)kProfSlots * kProfSlotWords * 8, 0, kSchedSlots * 8) != cudaSuccess) return PIPER_ERR_CUDA;
    c->tc_prof = 0, c->tc_rows_on_n = 1, c->tc_small_rows = TB_SMALL_ROWS, c->tc_two_cta = 2;
    c->tc_greedy = 0;  // equal chunks: C2 -6 %, C3 -0.9 %, C4 -0.2 % per step against 256-row chunks + a short tail (finding 31)
    c->tc_dual = 0;  // measured slower (DESIGN.md finding 22)
    c->tc_store_warp = 2;
    c->map_cache = new (std::nothrow) MapCacheEntry[kMapCache]();
    bool ok = set_smem_attr<K_MAJOR, MN_MAJOR, EPI_SWIGLU_FWD>() && set_smem_attr<K_MAJOR, MN_MAJOR, EPI_STORE>() &&
              set_smem_attr<K_MAJOR, K_MAJOR, EPI_SWIGLU_BWD>() && set_smem_attr<K_MAJOR, K_MAJOR, EPI_STORE>() &&
              set_smem_attr<MN_MAJOR, MN_MAJOR, EPI_WGRAD_SPLIT>() && set_smem_attr<MN_MAJOR, MN_MAJOR, EPI_WGRAD>() &&
              set_smem_attr_t<MN_MAJOR, TEPI_SWIGLU_FWD>() && set_smem_attr_t<MN_MAJOR, TEPI_STORE>() &&
              set_smem_attr_t<K_MAJOR, TEPI_SWIGLU_BWD>() && set_smem_attr_t<K_MAJOR, TEPI_STORE>() &&
              cudaFuncSetAttribute(tc_gemm2_kernel<MN_MAJOR, MN_MAJOR, EPI_WGRAD_SPLIT, true>,
                                   cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg2<EPI_WGRAD_SPLIT>::SMEM) == cudaSuccess &&
              set_smem_attr_t<MN_MAJOR, TEPI_STORE, false, true>() && set_smem_attr_t<K_MAJOR, TEPI_STORE, false, true>() &&
              set_smem_attr_t<MN_MAJOR, TEPI_SWIGLU_FWD, true>() && set_smem_attr_t<K_MAJOR, TEPI_SWIGLU_BWD, true>() &&
              set_smem_attr1<K_MAJOR, MN_MAJOR, EPI_STORE_F32>() && set_smem_attr1<MN_MAJOR, MN_MAJOR, EPI_STORE_F32>();
    if (!ok) {
        cudaGetLastError();
        c->encode_tiled = nullptr;  // not an sm_100a device: the FP32-ALU kernels serve every request
    }
    return PIPER_OK;
}

bool tc_supported(const piper_ctx* c, const FfnProblem& p) {
    if (!c->encode_tiled) return false;
    if (p.G > kMaxGroups || p.d < 64 || p.I < 64 || p.d % 8 || p.I % 8) return false;
    if (p.G > 1) {
        // the rows-on-N kernels and the CTA-pair wgrad work in 16-row units (chunks rounded up to 16 rows, K slices of
        // 16 rows issued up to the expert's real count); the rows-on-M and 1-CTA families need whole 128-row tiles
        if (c->D.row_align % 16) return false;
        if (c->D.row_align % BM && !(rows_on_n(c, p) && pair_wgrad(c, p))) return false;
    }
    return true;
}

bool tc_wgrad_f32_ok(const piper_ctx* c, const FfnProblem& p) { return pair_wgrad(c, p); }
bool tc_gather_ok(const piper_ctx* c, const FfnProblem& p) { return rows_on_n(c, p) && pair_wgrad(c, p) && c->D.k <= 8; }

// G|U = Xp Wg | Xp Wu, H = silu(G) * U
int tc_ffn_fwd1(piper_ctx* c, Lane ln, const FfnProblem& p) {
    if (rows_on_n(c, p)) {
        TcParams P = t_params(c, p, p.I, p.d, 128);
        PIPER_MAP(&P.a[0], p.w_gate, p.I, p.d, p.G, 64);
        PIPER_MAP(&P.a[1], p.w_up, p.I, p.d, p.G, 64);
        PIPER_MAP(&P.b[0], p.xp, p.d, p.max_rows, 1, TB_BOX_ROWS);
        PIPER_MAP(&P.bs[0], p.xp, p.d, p.max_rows, 1, TB_SMALL_ROWS);
        PIPER_MAP2(&P.o[0], p.g, p.I, p.max_rows, 1, 32, 16);
        PIPER_MAP2(&P.o[1], p.u, p.I, p.max_rows, 1, 32, 16);
        PIPER_MAP2(&P.o[2], p.h, p.I, p.max_rows, 1, 32, 16);
        if (p.gather_x) {  // N2: the expert's rows are gathered from x, the packed buffer xp is not read
            set_gather(P, c, p, p.gather_x, p.d);
            return launch_t<MN_MAJOR, TEPI_SWIGLU_FWD, true>(c, ln, P, t_tile_bound(p, P.f_tiles), "tc_ffn_fwd1_t_gather");
        }
        return launch_t<MN_MAJOR, TEPI_SWIGLU_FWD>(c, ln, P, t_tile_bound(p, P.f_tiles), "tc_ffn_fwd1_t");
    }
    const bool two = pair_ragged(c, p);
    TcParams P = base_params(p, true);
    PIPER_MAP(&P.a[0], p.xp, p.d, p.max_rows, 1, BM);
    PIPER_MAP(&P.b[0], p.w_gate, p.I, p.d, p.G, 64);
    PIPER_MAP(&P.b[1], p.w_up, p.I, p.d, p.G, 64);
    P.b_split = 1, P.tile_n = 128, P.n_tiles = cdiv(p.I, 128), P.kb_per_src = cdiv(p.d, BK);
    P.n_limit = p.I, P.ld = p.I;
    P.out0 = (__nv_bfloat16*)p.g, P.out1 = (__nv_bfloat16*)p.u, P.out2 = (__nv_bfloat16*)p.h;
    if (two) {
        PIPER_MAP(&P.o[0], p.g, p.I, p.max_rows, 1, 32);
        PIPER_MAP(&P.o[1], p.u, p.I, p.max_rows, 1, 32);
        PIPER_MAP(&P.o[2], p.h, p.I, p.max_rows, 1, 32);
    }
    return launch<K_MAJOR, MN_MAJOR, EPI_SWIGLU_FWD>(c, ln, P, m_tile_bound(p, two) * P.n_tiles, two, "tc_ffn_fwd1");
}

// O = H Wd
int tc_ffn_fwd2(piper_ctx* c, Lane ln, const FfnProblem& p) {
    if (rows_on_n(c, p)) {
        TcParams P = t_params(c, p, p.d, p.I, 256);
        PIPER_MAP(&P.a[0], p.w_down, p.d, p.I, p.G, 64);
        PIPER_MAP(&P.b[0], p.h, p.I, p.max_rows, 1, TB_BOX_ROWS);
        PIPER_MAP(&P.bs[0], p.h, p.I, p.max_rows, 1, TB_SMALL_ROWS);
        PIPER_MAP2(&P.o[0], p.o, p.d, p.max_rows, 1, 32, 16);
        if (dual_tiles(c, p)) return launch_t<MN_MAJOR, TEPI_STORE, false, true>(c, ln, P, t_tile_bound(p, P.f_tiles), "tc_ffn_fwd2_t2");
        return launch_t<MN_MAJOR, TEPI_STORE>(c, ln, P, t_tile_bound(p, P.f_tiles), "tc_ffn_fwd2_t");
    }
    const bool two = pair_ragged(c, p);
    TcParams P = base_params(p, true);
    PIPER_MAP(&P.a[0], p.h, p.I, p.max_rows, 1, BM);
    PIPER_MAP(&P.b[0], p.w_down, p.d, p.I, p.G, 64);
    P.n_tiles = cdiv(p.d, BN), P.kb_per_src = cdiv(p.I, BK), P.n_limit = p.d, P.ld = p.d;
    P.out0 = (__nv_bfloat16*)p.o;
    if (two) PIPER_MAP(&P.o[0], p.o, p.d, p.max_rows, 1, 32);
    return launch<K_MAJOR, MN_MAJOR, EPI_STORE>(c, ln, P, m_tile_bound(p, two) * P.n_tiles, two, "tc_ffn_fwd2");
}

// dH = dO Wd^T; dG = dH * U * silu'(G); dU = dH * silu(G)
int tc_ffn_dgrad1(piper_ctx* c, Lane ln, const FfnProblem& p) {
    if (rows_on_n(c, p)) {
        TcParams P = t_params(c, p, p.I, p.d, 256);
        PIPER_MAP(&P.a[0], p.w_down, p.d, p.I, p.G, 128);
        PIPER_MAP(&P.b[0], p.d_o, p.d, p.max_rows, 1, TB_BOX_ROWS);
        PIPER_MAP(&P.bs[0], p.d_o, p.d, p.max_rows, 1, TB_SMALL_ROWS);
        PIPER_MAP2(&P.o[0], p.dg, p.I, p.max_rows, 1, 32, 16);
        PIPER_MAP2(&P.o[1], p.du, p.I, p.max_rows, 1, 32, 16);
        PIPER_MAP2(&P.ein[0], p.g, p.I, p.max_rows, 1, 32, 32);
        PIPER_MAP2(&P.ein[1], p.u, p.I, p.max_rows, 1, 32, 32);
        if (p.gather_dy) {  // N2: rows of dY gathered, the gate applied to dH in the fp32 epilogue; d_o is not read
            set_gather(P, c, p, p.gather_dy, p.d);
            P.row_scale = p.gate_rows;
            return launch_t<K_MAJOR, TEPI_SWIGLU_BWD, true>(c, ln, P, t_tile_bound(p, P.f_tiles), "tc_ffn_dgrad1_t_gather");
        }
        return launch_t<K_MAJOR, TEPI_SWIGLU_BWD>(c, ln, P, t_tile_bound(p, P.f_tiles), "tc_ffn_dgrad1_t");
    }
    const bool two = pair_ragged(c, p);
    TcParams P = base_params(p, true);
    PIPER_MAP(&P.a[0], p.d_o, p.d, p.max_rows, 1, BM);
    PIPER_MAP(&P.b[0], p.w_down, p.d, p.I, p.G, two ? BN / 2 : BN);
    P.n_tiles = cdiv(p.I, BN), P.kb_per_src = cdiv(p.d, BK), P.n_limit = p.I, P.ld = p.I;
    P.in0 = (const __nv_bfloat16*)p.g, P.in1 = (const __nv_bfloat16*)p.u;
    P.out0 = (__nv_bfloat16*)p.dg, P.out1 = (__nv_bfloat16*)p.du;
    if (two) {
        PIPER_MAP(&P.o[0], p.dg, p.I, p.max_rows, 1, 32);
        PIPER_MAP(&P.o[1], p.du, p.I, p.max_rows, 1, 32);
        PIPER_MAP(&P.ein[0], p.g, p.I, p.max_rows, 1, 32);
        PIPER_MAP(&P.ein[1], p.u, p.I, p.max_rows, 1, 32);
    }
    return launch<K_MAJOR, K_MAJOR, EPI_SWIGLU_BWD>(c, ln, P, m_tile_bound(p, two) * P.n_tiles, two, "tc_ffn_dgrad1");
}

// dXp = dG Wg^T + dU Wu^T  (one accumulator, K runs over both products)
int tc_ffn_dgrad2(piper_ctx* c, Lane ln, const FfnProblem& p) {
    if (rows_on_n(c, p)) {
        TcParams P = t_params(c, p, p.d, p.I, 256);
        PIPER_MAP(&P.a[0], p.w_gate, p.I, p.d, p.G, 128);
        PIPER_MAP(&P.a[1], p.w_up, p.I, p.d, p.G, 128);
        PIPER_MAP(&P.b[0], p.dg, p.I, p.max_rows, 1, TB_BOX_ROWS);
        PIPER_MAP(&P.b[1], p.du, p.I, p.max_rows, 1, TB_BOX_ROWS);
        PIPER_MAP(&P.bs[0], p.dg, p.I, p.max_rows, 1, TB_SMALL_ROWS);
        PIPER_MAP(&P.bs[1], p.du, p.I, p.max_rows, 1, TB_SMALL_ROWS);
        P.n_src = 2;
        PIPER_MAP2(&P.o[0], p.dxp, p.d, p.max_rows, 1, 32, 16);
        if (dual_tiles(c, p)) return launch_t<K_MAJOR, TEPI_STORE, false, true>(c, ln, P, t_tile_bound(p, P.f_tiles), "tc_ffn_dgrad2_t2");
        return launch_t<K_MAJOR, TEPI_STORE>(c, ln, P, t_tile_bound(p, P.f_tiles), "tc_ffn_dgrad2_t");
    }
    const bool two = pair_ragged(c, p);
    TcParams P = base_params(p, true);
    PIPER_MAP(&P.a[0], p.dg, p.I, p.max_rows, 1, BM);
    PIPER_MAP(&P.a[1], p.du, p.I, p.max_rows, 1, BM);
    PIPER_MAP(&P.b[0], p.w_gate, p.I, p.d, p.G, two ? BN / 2 : BN);
    PIPER_MAP(&P.b[1], p.w_up, p.I, p.d, p.G, two ? BN / 2 : BN);
    P.n_src = 2, P.n_tiles = cdiv(p.d, BN), P.kb_per_src = cdiv(p.I, BK), P.n_limit = p.d, P.ld = p.d;
    P.out0 = (__nv_bfloat16*)p.dxp;
    if (two) PIPER_MAP(&P.o[0], p.dxp, p.d, p.max_rows, 1, 32);
    return launch<K_MAJOR, K_MAJOR, EPI_STORE>(c, ln, P, m_tile_bound(p, two) * P.n_tiles, two, "tc_ffn_dgrad2");
}

// dWg|dWu[e] = Xp^T dG | Xp^T dU ; dWd[e] = H^T dO over the expert's rows (K ragged; zeros for empty experts)
int tc_ffn_wgrad(piper_ctx* c, Lane ln, const FfnProblem& p) {
    const bool two = pair_wgrad(c, p);
    const bool f32 = c->D.dw_dtype == PIPER_DTYPE_F32;  // fp32 dW from bf16 operands: the CTA-pair kernel only
    if ((f32 || p.accumulate) && !(two && f32)) return PIPER_ERR_UNSUPPORTED;
    // One 128-row store per chunk from the store warp when the K ranges are long and even (>= 512 rows per expert expected
    // under uniform routing, and the kernel finds no expert with more than twice the mean: C2 wgrad 2.31 -> 2.21 ms).  On
    // short ranges the epilogue warps are the critical path and the hand-over costs more than the store issue it saves
    // (C3, 252 rows per expert: 0.83 -> 0.96 ms; C4, skewed: 1.46 -> 1.55 ms), so they keep their own 32-row stores.
    const bool sw = two && !f32 && Cfg2<EPI_WGRAD>::STORE_WARP &&
                    (c->tc_store_warp == 2 ? (long long)p.exp_rows >= 512ll * p.G : c->tc_store_warp == 1);
    {
        TcParams P = base_params(p, false);
        P.counts = p.counts;
        const int kbox = two ? Cfg2<EPI_WGRAD_SPLIT>::BKc : BK;
        PIPER_MAP(&P.a[0], p.xp, p.d, p.max_rows, 1, kbox);
        PIPER_MAP(&P.b[0], p.dg, p.I, p.max_rows, 1, kbox);
        PIPER_MAP(&P.b[1], p.du, p.I, p.max_rows, 1, kbox);
        P.b_split = 1, P.tile_n = 128, P.n_tiles = cdiv(p.I, 128), P.m_tiles = cdiv(p.d, BM);
        P.m_limit = p.d, P.n_limit = p.I, P.ld = p.I, P.group_stride = (long long)p.d * p.I;
        P.out0 = (__nv_bfloat16*)p.dw_gate, P.out1 = (__nv_bfloat16*)p.dw_up;
        if (f32) {
            int rc = make_map_f32(c, &P.o[0], p.dw_gate, p.I, p.d, p.G);
            if (rc == PIPER_OK) rc = make_map_f32(c, &P.o[1], p.dw_up, p.I, p.d, p.G);
            if (rc != PIPER_OK) return rc;
            P.out_f32 = 1, P.accum = p.accumulate;
        } else if (two) {
            P.store_warp = (sw && !p.gather_x) ? c->tc_store_warp : 0;
            PIPER_MAP(&P.o[0], p.dw_gate, p.I, p.d, p.G, 32);
            PIPER_MAP(&P.o[1], p.dw_up, p.I, p.d, p.G, 32);
            if (P.store_warp) {
                PIPER_MAP(&P.ow[0], p.dw_gate, p.I, p.d, p.G, 128);
                PIPER_MAP(&P.ow[1], p.dw_up, p.I, p.d, p.G, 128);
            }
        }
        const long long mt = two ? (P.m_tiles + 1) / 2 : P.m_tiles;
        int rc;
        if (p.gather_x && two) {  // N2: the A operand Xp^T is gathered from x, the packed buffer is not read
            set_gather(P, c, p, p.gather_x, p.d);
            rc = launch<MN_MAJOR, MN_MAJOR, EPI_WGRAD_SPLIT, true>(c, ln, P, (long long)p.G * mt * P.n_tiles, two,
                                                                  "tc_ffn_wgrad_gate_up_gather");
        } else {
            rc = launch<MN_MAJOR, MN_MAJOR, EPI_WGRAD_SPLIT>(c, ln, P, (long long)p.G * mt * P.n_tiles, two,
                                                            "tc_ffn_wgrad_gate_up");
        }
        if (rc != PIPER_OK) return rc;
    }
    TcParams P = base_params(p, false);
    P.counts = p.counts;
    const int kbox = two ? Cfg2<EPI_WGRAD>::BKc : BK;
    PIPER_MAP(&P.a[0], p.h, p.I, p.max_rows, 1, kbox);
    PIPER_MAP(&P.b[0], p.d_o, p.d, p.max_rows, 1, kbox);
    P.n_tiles = cdiv(p.d, BN), P.m_tiles = cdiv(p.I, BM);
    P.m_limit = p.I, P.n_limit = p.d, P.ld = p.d, P.group_stride = (long long)p.I * p.d;
    P.out0 = (__nv_bfloat16*)p.dw_down;
    if (f32) {
        const int rc = make_map_f32(c, &P.o[0], p.dw_down, p.d, p.I, p.G);
        if (rc != PIPER_OK) return rc;
        P.out_f32 = 1, P.accum = p.accumulate;
    } else if (two) {
        P.store_warp = sw ? c->tc_store_warp : 0;
        PIPER_MAP(&P.o[0], p.dw_down, p.d, p.I, p.G, 32);
        if (sw) PIPER_MAP(&P.ow[0], p.dw_down, p.d, p.I, p.G, 128);
    }
    const long long mt = two ? (P.m_tiles + 1) / 2 : P.m_tiles;
    return launch<MN_MAJOR, MN_MAJOR, EPI_WGRAD>(c, ln, P, (long long)p.G * mt * P.n_tiles, two, "tc_ffn_wgrad_down");
}

// ---- dense GEMMs of the router (N1: z = x W_r, dW_r = x^T dz, dX_r = dz W_r^T) on the 1-CTA kernel ----------------------
// One group over all T rows (offsets = {0, T}); 128 x 256 tiles; N <= 256 experts is a single N tile whose columns beyond
// E the TMA fills with zeros.  bf16 x bf16 products are exact in fp32 and the accumulation is fp32 (TMEM).
bool tc_router_supported(const piper_ctx* c) {
    const piper_moe_desc& D = c->D;
    return c->encode_tiled && D.dtype == PIPER_DTYPE_BF16 && D.E % 8 == 0 && D.d >= 64 && D.d % 8 == 0 && D.T >= 1;
}

// logits [T,E] fp32 = x [T,d] W_r [d,E] (+ bias[E])
int tc_router_fwd(piper_ctx* c, Lane ln, const void* x, const void* w_r, const float* bias, float* logits) {
    const piper_moe_desc& D = c->D;
    TcParams P;
    memset(&P, 0, sizeof(P));
    P.offsets = c->shared_offsets, P.G = 1, P.ragged_m = 1, P.n_src = 1, P.tile_n = BN;
    PIPER_MAP(&P.a[0], x, D.d, D.T, 1, BM);
    PIPER_MAP(&P.b[0], w_r, D.E, D.d, 1, 64);
    P.n_tiles = cdiv(D.E, BN), P.kb_per_src = cdiv(D.d, BK), P.n_limit = D.E, P.ld = D.E;
    P.out0 = reinterpret_cast<__nv_bfloat16*>(logits), P.bias = bias;
    return launch<K_MAJOR, MN_MAJOR, EPI_STORE_F32>(c, ln, P, (long long)cdiv(D.T, BM) * P.n_tiles, false, "tc_router_fwd");
}

// dW_r [d,E] fp32 = x^T dz with dz = hi + lo (two bf16 [T,E] tensors): one accumulator over both products
int tc_router_wgrad(piper_ctx* c, Lane ln, const void* x, const void* dz_hi, const void* dz_lo, float* dw_r) {
    const piper_moe_desc& D = c->D;
    TcParams P;
    memset(&P, 0, sizeof(P));
    P.offsets = c->shared_offsets, P.G = 1, P.ragged_m = 0, P.n_src = 2, P.tile_n = BN;
    PIPER_MAP(&P.a[0], x, D.d, D.T, 1, BK);
    P.a[1] = P.a[0];
    PIPER_MAP(&P.b[0], dz_hi, D.E, D.T, 1, BK);
    PIPER_MAP(&P.b[1], dz_lo, D.E, D.T, 1, BK);
    P.n_tiles = cdiv(D.E, BN), P.m_tiles = cdiv(D.d, BM), P.kb_per_src = cdiv(D.T, BK);
    P.m_limit = D.d, P.n_limit = D.E, P.ld = D.E, P.group_stride = 0;
    P.out0 = reinterpret_cast<__nv_bfloat16*>(dw_r);
    return launch<MN_MAJOR, MN_MAJOR, EPI_STORE_F32>(c, ln, P, (long long)P.m_tiles * P.n_tiles, false, "tc_router_wgrad");
}

// dX_r [T,d] bf16 = dz W_r^T with dz = hi + lo
int tc_router_dgrad(piper_ctx* c, Lane ln, const void* dz_hi, const void* dz_lo, const void* w_r, void* dx_r) {
    const piper_moe_desc& D = c->D;
    TcParams P;
    memset(&P, 0, sizeof(P));
    P.offsets = c->shared_offsets, P.G = 1, P.ragged_m = 1, P.n_src = 2, P.tile_n = BN;
    PIPER_MAP(&P.a[0], dz_hi, D.E, D.T, 1, BM);
    PIPER_MAP(&P.a[1], dz_lo, D.E, D.T, 1, BM);
    PIPER_MAP(&P.b[0], w_r, D.E, D.d, 1, BN);
    P.b[1] = P.b[0];
    P.n_tiles = cdiv(D.d, BN), P.kb_per_src = cdiv(D.E, BK), P.n_limit = D.d, P.ld = D.d;
    P.out0 = static_cast<__nv_bfloat16*>(dx_r);
    return launch<K_MAJOR, K_MAJOR, EPI_STORE>(c, ln, P, (long long)cdiv(D.T, BM) * P.n_tiles, false, "tc_router_dgrad");
}

}  // namespace piper
