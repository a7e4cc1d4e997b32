// chunk.cu — whole-chunk entry points: piper_run_chunk_fwd / _bwd (serial baseline, one stream, all SMs)
// and P piper_run_chunk_pair (SURVEY.md §8a P, §8c c-sched; BASELINE.json:north_star part 5).
//
// The pair is the task DAG of SURVEY.md §8c on two logical streams:
//   "comm"  (pack/combine side): F.route, F.scan, F.pack, F.combine, B.cgrad, B.unpack, B.route_bwd
//   "gemm"  (compute side)     : F.gemm1, F.gemm2, F.shared, B.dgrad1, B.dgrad2, B.wgrad, B.shared_bwd
// ordered by piper_list_schedule and synchronised by the event rule of PAPER.md:279-286:
// a task waits only on dependencies that ran on the other stream, and records an event only if a
// consumer runs on the other stream.  The SM split is enforced with green contexts (driver API reached
// through cudaGetDriverEntryPoint, so the library has no link-time dependency on libcuda); if they are
// unavailable the two streams are plain streams and every kernel bounds its own grid to its lane's SM
// count.  The paper itself leaves SM allocation to the GPU.
#include "piper_internal.cuh"

using namespace piper;

namespace piper {

struct GreenPartition {
    int sm_gemm = 0, sm_comm = 0;
    CUgreenCtx gctx[2] = {nullptr, nullptr};  // 0 = comm, 1 = gemm
    cudaStream_t stream[2] = {nullptr, nullptr};
    bool green = false;
};

namespace {

struct DriverApi {
    CUresult (*DeviceGet)(CUdevice*, int) = nullptr;
    CUresult (*DeviceGetDevResource)(CUdevice, CUdevResource*, CUdevResourceType) = nullptr;
    CUresult (*DevSmResourceSplitByCount)(CUdevResource*, unsigned int*, const CUdevResource*, CUdevResource*,
                                          unsigned int, unsigned int) = nullptr;
    CUresult (*DevResourceGenerateDesc)(CUdevResourceDesc*, CUdevResource*, unsigned int) = nullptr;
    CUresult (*GreenCtxCreate)(CUgreenCtx*, CUdevResourceDesc, CUdevice, unsigned int) = nullptr;
    CUresult (*GreenCtxDestroy)(CUgreenCtx) = nullptr;
    CUresult (*GreenCtxStreamCreate)(CUstream*, CUgreenCtx, unsigned int, int) = nullptr;
    bool ok = false;
};

template <typename F>
bool resolve(const char* name, F& fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint(name, &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !p)
        return false;
    fn = reinterpret_cast<F>(p);
    return true;
}

DriverApi& driver() {
    static DriverApi d = [] {
        DriverApi a;
        a.ok = resolve("cuDeviceGet", a.DeviceGet) && resolve("cuDeviceGetDevResource", a.DeviceGetDevResource) &&
               resolve("cuDevSmResourceSplitByCount", a.DevSmResourceSplitByCount) &&
               resolve("cuDevResourceGenerateDesc", a.DevResourceGenerateDesc) &&
               resolve("cuGreenCtxCreate", a.GreenCtxCreate) && resolve("cuGreenCtxDestroy", a.GreenCtxDestroy) &&
               resolve("cuGreenCtxStreamCreate", a.GreenCtxStreamCreate);
        return a;
    }();
    return d;
}

void destroy_partition(piper_ctx* c, GreenPartition* g) {
    if (!g) return;
    for (int i = 0; i < 2; ++i) {
        if (g->stream[i]) tc_forget_stream(c, g->stream[i]), cudaStreamDestroy(g->stream[i]);
        if (g->gctx[i] && driver().ok) driver().GreenCtxDestroy(g->gctx[i]);
    }
    delete g;
}

// Split the device's SMs into {sm_comm, rest}; the gemm side keeps the first sm_gemm of the rest.
GreenPartition* make_partition(piper_ctx* c, int sm_gemm, int sm_comm, bool want_green) {
    GreenPartition* g = new GreenPartition();
    g->sm_gemm = sm_gemm, g->sm_comm = sm_comm;
    DriverApi& api = driver();
    bool ok = api.ok && want_green;
    CUdevice dev = 0;
    CUdevResource all{}, part{}, rest{};
    unsigned int n_groups = 1;
    ok = ok && api.DeviceGet(&dev, c->device) == CUDA_SUCCESS;
    ok = ok && api.DeviceGetDevResource(dev, &all, CU_DEV_RESOURCE_TYPE_SM) == CUDA_SUCCESS;
    ok = ok && api.DevSmResourceSplitByCount(&part, &n_groups, &all, &rest, 0, (unsigned)sm_comm) == CUDA_SUCCESS &&
         n_groups == 1 && (int)part.sm.smCount == sm_comm && (int)rest.sm.smCount >= sm_gemm;
    if (ok && (int)rest.sm.smCount > sm_gemm) {  // trim the compute side to sm_gemm (multiples of the granularity)
        CUdevResource keep{}, drop{};
        unsigned int one = 1;
        ok = api.DevSmResourceSplitByCount(&keep, &one, &rest, &drop, 0, (unsigned)sm_gemm) == CUDA_SUCCESS &&
             one == 1 && (int)keep.sm.smCount == sm_gemm;
        rest = keep;
    }
    CUdevResource res[2] = {part, rest};
    for (int i = 0; ok && i < 2; ++i) {
        CUdevResourceDesc desc{};
        ok = api.DevResourceGenerateDesc(&desc, &res[i], 1) == CUDA_SUCCESS &&
             api.GreenCtxCreate(&g->gctx[i], desc, dev, CU_GREEN_CTX_DEFAULT_STREAM) == CUDA_SUCCESS;
        CUstream s = nullptr;
        ok = ok && api.GreenCtxStreamCreate(&s, g->gctx[i], CU_STREAM_NON_BLOCKING, 0) == CUDA_SUCCESS;
        g->stream[i] = reinterpret_cast<cudaStream_t>(s);
    }
    if (ok) {
        g->green = true;
        return g;
    }
    for (int i = 0; i < 2; ++i) {
        if (g->stream[i]) cudaStreamDestroy(g->stream[i]), g->stream[i] = nullptr;
        if (g->gctx[i] && api.ok) api.GreenCtxDestroy(g->gctx[i]), g->gctx[i] = nullptr;
    }
    cudaGetLastError();
    if (want_green) {  // disjoint SM sets were asked for and cannot be had: no silent fallback
        delete g;
        return nullptr;
    }
    // PIPER_PART_SHARED / _CHUNK_STREAMS: plain streams, grids bounded by Lane::sms
    for (int i = 0; i < 2; ++i)
        if (cudaStreamCreateWithFlags(&g->stream[i], cudaStreamNonBlocking) != cudaSuccess) {
            destroy_partition(c, g);
            return nullptr;
        }
    g->green = false;
    return g;
}

// ---- the tasks ------------------------------------------------------------------------------------
enum Task {
    F_ROUTE, F_SCAN, F_PACK, F_GEMM1, F_GEMM2, F_SHARED, F_COMBINE,
    B_CGRAD, B_DGRAD1, B_DGRAD2, B_WGRAD, B_SHARED, B_UNPACK, B_ROUTE_BWD, N_TASKS,
    // N3: caller tasks of the pair (piper_pair_set_caller_task), id = N_TASKS + slot
    X_F_PRE = N_TASKS, X_F_POST, X_B_PRE, X_B_POST, N_ALL
};
constexpr int COMM = 0, GEMM = 1;
const int kStreamOf[N_TASKS] = {COMM, COMM, COMM, GEMM, GEMM, GEMM, COMM, COMM, GEMM, GEMM, GEMM, GEMM, COMM, COMM};
const int kEdges[][2] = {{F_ROUTE, F_SCAN},   {F_SCAN, F_PACK},    {F_PACK, F_GEMM1},     {F_GEMM1, F_GEMM2},
                         {F_GEMM2, F_COMBINE}, {F_SCAN, F_GEMM1},   {F_SCAN, F_COMBINE},   {F_SHARED, F_COMBINE},
                         {B_CGRAD, B_DGRAD1},  {B_DGRAD1, B_DGRAD2}, {B_DGRAD2, B_UNPACK},  {B_CGRAD, B_WGRAD},
                         {B_DGRAD1, B_WGRAD},  {B_SHARED, B_UNPACK}, {B_CGRAD, B_ROUTE_BWD}};
// caller tasks: x / logits of the forward microbatch come from F_PRE, y goes to F_POST; dY of the backward microbatch
// comes from B_PRE, dX / dz_sel go to B_POST (include/piper.h, piper_pair_set_caller_task)
const int kCallerEdges[][2] = {{X_F_PRE, F_ROUTE},  {X_F_PRE, F_PACK},  {X_F_PRE, F_SHARED},    {F_COMBINE, X_F_POST},
                               {X_B_PRE, B_CGRAD},  {X_B_PRE, B_SHARED}, {B_UNPACK, X_B_POST}, {B_ROUTE_BWD, X_B_POST}};

// `parts` of the backward tasks that hold both passes (B_SHARED): bit 0 = input gradients (Bi), bit 1 = weight gradients (Bw)
constexpr int PART_BI = 1, PART_BW = 2, PART_ALL = 3;

// N2 fusion (PIPER_OPT_FUSED_GATHER on a tcgen05 layer): the routed GEMMs of the chunk tasks gather the rows of x / dY
// through src_of themselves (F_GEMM1, the gate|up wgrad: x; DGRAD1: dY with the gate applied in its fp32 epilogue), so
// the forward chunk does not materialise xp at all; piper_dispatch_pack / piper_run_task(F_PACK) still produce it as
// the all-to-all payload.
FfnProblem routed_fwd_problem(const piper_ctx* c, const piper_chunk_args* f) {
    FfnProblem p = routed_problem(c, f);
    if (fused_gather(c)) p.gather_x = f->x, p.src_of = f->src_of;
    return p;
}
FfnProblem routed_bwd_problem(const piper_ctx* c, const piper_chunk_args* b) {
    FfnProblem p = routed_problem(c, b);
    if (fused_gather(c)) {
        p.gather_x = b->x, p.src_of = b->src_of;
        if (c->fused_gather >= 2) p.gather_dy = b->dy, p.gate_rows = b->gate_rows;  // DGRAD1 from dY, gate in its epilogue
    }
    return p;
}

// in_chunk: called from a whole-chunk entry point (fused layers skip F_PACK there), not from piper_run_task
int run_task(piper_ctx* c, int task, Lane ln, const piper_chunk_args* f, const piper_chunk_args* b, int parts = PART_ALL,
             bool in_chunk = true) {
    if (task >= X_F_PRE && task < N_ALL) {  // the caller's function enqueues its own work on the lane's stream
        const int slot = task - X_F_PRE;
        if (!c->caller_fn[slot]) return PIPER_ERR_INVALID;
        if (c->caller_fn[slot](c->caller_user[slot], ln.stream, ln.sms) != 0) {
            snprintf(c->err, sizeof(c->err), "caller task of slot %d failed", slot);
            return PIPER_ERR_INVALID;
        }
        return PIPER_OK;
    }
    switch (task) {
        case F_ROUTE: {
            if (f->w_r) {  // N1: the router GEMM writes the logits F1 reads
                const int rc = launch_router_fwd(c, ln, f->x, f->w_r, f->router_bias, const_cast<float*>(f->logits));
                if (rc != PIPER_OK) return rc;
            }
            return launch_route_topk(c, ln, f->logits, f->topk_idx, f->gates, f->counts_global);
        }
        case F_SCAN:
            return launch_scan_rank(c, ln, f->topk_idx, f->gates, f->counts, f->offsets, f->row_of, f->src_of, f->gate_rows);
        case F_PACK:
            if (in_chunk && fused_gather(c)) return PIPER_OK;  // N2: no GEMM of the chunk reads xp
            return launch_pack(c, ln, f->x, f->offsets, f->row_of, f->src_of, f->xp);
        case F_GEMM1: return ffn_gemm1(c, ln, routed_fwd_problem(c, f));
        case F_GEMM2: return ffn_gemm2(c, ln, routed_problem(c, f));
        case F_SHARED: {
            const FfnProblem p = shared_problem(c, f);
            const int rc = ffn_gemm1(c, ln, p);
            return rc != PIPER_OK ? rc : ffn_gemm2(c, ln, p);
        }
        case F_COMBINE:
            return launch_combine(c, ln, f->o, f->row_of, f->gates, c->D.I_shared ? f->s : nullptr, nullptr, f->y, true);
        case B_CGRAD:
            return launch_combine_bwd(c, ln, b->dy, b->o, b->src_of, b->row_of, b->gates, b->offsets, b->d_o, b->dgates);
        case B_DGRAD1: return ffn_dgrad1(c, ln, routed_bwd_problem(c, b));
        case B_DGRAD2: return ffn_dgrad2(c, ln, routed_problem(c, b));
        case B_WGRAD: return ffn_wgrad(c, ln, routed_bwd_problem(c, b));
        case B_SHARED: {
            const FfnProblem p = shared_problem(c, b);
            int rc = PIPER_OK;
            if (parts & PART_BI) {
                rc = ffn_dgrad1(c, ln, p);
                if (rc == PIPER_OK) rc = ffn_dgrad2(c, ln, p);
            }
            if (rc == PIPER_OK && (parts & PART_BW)) rc = ffn_wgrad(c, ln, p);
            return rc;
        }
        case B_UNPACK:
            return launch_combine(c, ln, b->dxp, b->row_of, nullptr, c->D.I_shared ? b->dxs : nullptr,
                                  b->w_r ? b->dx_router : nullptr, b->dx, false);
        case B_ROUTE_BWD: {
            const int rc = launch_route_bwd(c, ln, b->logits, b->topk_idx, b->gates, b->dgates, b->dz_sel);
            if (rc != PIPER_OK || !b->w_r) return rc;
            // N1: dW_r = x^T dz and the router's term of dX (added by B_UNPACK, which therefore follows this task)
            return launch_router_bwd(c, ln, b->x, b->w_r, b->topk_idx, b->dz_sel, b->dz_scratch, b->dw_r, b->dx_router);
        }
    }
    return PIPER_ERR_INVALID;
}

bool fwd_args_ok(const piper_ctx* c, const piper_chunk_args* a) {
    bool ok = a && aligned16(a->logits) && aligned16(a->x) && aligned16(a->w_gate) && aligned16(a->w_up) &&
              aligned16(a->w_down) && aligned16(a->topk_idx) && aligned16(a->counts_global) && aligned16(a->counts) &&
              aligned16(a->offsets) && aligned16(a->row_of) && aligned16(a->src_of) && aligned16(a->gates) &&
              aligned16(a->gate_rows) && aligned16(a->xp) && aligned16(a->g_save) && aligned16(a->u_save) &&
              aligned16(a->h_save) && aligned16(a->o) && aligned16(a->y);
    if (ok && c->D.I_shared)
        ok = aligned16(a->ws_gate) && aligned16(a->ws_up) && aligned16(a->ws_down) && aligned16(a->gs_save) &&
             aligned16(a->us_save) && aligned16(a->hs_save) && aligned16(a->s);
    if (ok && a->w_r) ok = aligned16(a->w_r) && (!a->router_bias || aligned16(a->router_bias));
    return ok;
}
bool bwd_args_ok(const piper_ctx* c, const piper_chunk_args* a) {
    bool ok = fwd_args_ok(c, a) && aligned16(a->dy) && aligned16(a->dgates) && aligned16(a->dz_sel) &&
              aligned16(a->d_o) && aligned16(a->dg) && aligned16(a->du) && aligned16(a->dxp) && aligned16(a->dx) &&
              aligned16(a->dw_gate) && aligned16(a->dw_up) && aligned16(a->dw_down);
    if (ok && c->D.I_shared)
        ok = aligned16(a->dgs) && aligned16(a->dus) && aligned16(a->dxs) && aligned16(a->dws_gate) &&
             aligned16(a->dws_up) && aligned16(a->dws_down);
    if (ok && a->w_r) ok = aligned16(a->dw_r) && aligned16(a->dx_router) && aligned16(a->dz_scratch);
    return ok;
}

}  // namespace

struct PairPlan {
    bool router;  // the DAG has the N1 edge B.route_bwd -> B.unpack
    int32_t n, n_waits;
    int32_t task_of[N_ALL], stream_of[N_ALL], order[N_ALL], waits[32][2], records[N_ALL];
};

void pair_plan_release(piper_ctx* c) {
    delete static_cast<PairPlan*>(c->pair_plan);
    c->pair_plan = nullptr;
}

void pair_release(piper_ctx* c) {
    destroy_partition(c, c->green);
    c->green = nullptr;
    pair_plan_release(c);
}

}  // namespace piper

extern "C" {

int piper_set_chunk_overlap(piper_ctx* c, int on) {
    if (!c || (on != 0 && on != 1)) return PIPER_ERR_INVALID;
    c->chunk_overlap = on;  // the side stream exists since piper_create
    return PIPER_OK;
}

int piper_run_chunk_fwd(piper_ctx* c, const piper_chunk_args* a, void* stream) {
    if (!c || !fwd_args_ok(c, a)) return PIPER_ERR_INVALID;
    const Lane ln{static_cast<cudaStream_t>(stream), c->num_sms};
    if (c->chunk_overlap && c->D.I_shared) {
        // The shared expert does not depend on the routing: route / scan / pack run on the side stream beside its
        // (compute-bound) GEMMs, the same two-stream rule as the pair inside one chunk.
        const Lane side{c->side_stream, c->num_sms};
        cudaEvent_t fork = c->events[14], packed = c->events[15];
        PIPER_CUDA(c, cudaEventRecord(fork, ln.stream));
        PIPER_CUDA(c, cudaStreamWaitEvent(side.stream, fork, 0));
        for (int t : {F_ROUTE, F_SCAN, F_PACK}) {
            const int rc = run_task(c, t, side, a, nullptr);
            if (rc != PIPER_OK) return rc;
        }
        PIPER_CUDA(c, cudaEventRecord(packed, side.stream));
        int rc = run_task(c, F_SHARED, ln, a, nullptr);
        if (rc != PIPER_OK) return rc;
        PIPER_CUDA(c, cudaStreamWaitEvent(ln.stream, packed, 0));
        for (int t : {F_GEMM1, F_GEMM2, F_COMBINE}) {
            rc = run_task(c, t, ln, a, nullptr);
            if (rc != PIPER_OK) return rc;
        }
        return PIPER_OK;
    }
    const int seq[] = {F_ROUTE, F_SCAN, F_PACK, F_SHARED, F_GEMM1, F_GEMM2, F_COMBINE};
    for (int t : seq) {
        if (t == F_SHARED && !c->D.I_shared) continue;
        const int rc = run_task(c, t, ln, a, nullptr);
        if (rc != PIPER_OK) return rc;
    }
    return PIPER_OK;
}

int piper_run_task(piper_ctx* c, int task, const piper_chunk_args* a, void* stream) {
    if (!c || task < 0 || task >= N_TASKS) return PIPER_ERR_INVALID;
    if (!(task < B_CGRAD ? fwd_args_ok(c, a) : bwd_args_ok(c, a))) return PIPER_ERR_INVALID;
    if ((task == F_SHARED || task == B_SHARED) && !c->D.I_shared) return PIPER_ERR_INVALID;
    const Lane ln{static_cast<cudaStream_t>(stream), c->num_sms};
    return run_task(c, task, ln, a, a, PART_ALL, false);
}

int piper_run_chunk_bwd(piper_ctx* c, const piper_chunk_args* a, void* stream) {
    if (!c || !bwd_args_ok(c, a)) return PIPER_ERR_INVALID;
    const Lane ln{static_cast<cudaStream_t>(stream), c->num_sms};
    if (c->chunk_overlap) {
        // unpack and route_bwd need no wgrad output: they run on the side stream beside the routed wgrad
        const Lane side{c->side_stream, c->num_sms};
        cudaEvent_t fork = c->events[14], joined = c->events[16];
        for (int t : {B_CGRAD, B_DGRAD1, B_DGRAD2, B_SHARED}) {
            if (t == B_SHARED && !c->D.I_shared) continue;
            const int rc = run_task(c, t, ln, nullptr, a);
            if (rc != PIPER_OK) return rc;
        }
        PIPER_CUDA(c, cudaEventRecord(fork, ln.stream));
        PIPER_CUDA(c, cudaStreamWaitEvent(side.stream, fork, 0));
        int rc = run_task(c, B_WGRAD, ln, nullptr, a);
        if (rc != PIPER_OK) return rc;
        for (int t : {B_ROUTE_BWD, B_UNPACK}) {
            rc = run_task(c, t, side, nullptr, a);
            if (rc != PIPER_OK) return rc;
        }
        PIPER_CUDA(c, cudaEventRecord(joined, side.stream));
        PIPER_CUDA(c, cudaStreamWaitEvent(ln.stream, joined, 0));
        return PIPER_OK;
    }
    const int seq[] = {B_CGRAD, B_DGRAD1, B_DGRAD2, B_WGRAD, B_SHARED, B_ROUTE_BWD, B_UNPACK};
    for (int t : seq) {
        if (t == B_SHARED && !c->D.I_shared) continue;
        const int rc = run_task(c, t, ln, nullptr, a);
        if (rc != PIPER_OK) return rc;
    }
    return PIPER_OK;
}

int piper_run_chunk_bwd_input(piper_ctx* c, const piper_chunk_args* a, void* stream) {
    if (!c || !bwd_args_ok(c, a)) return PIPER_ERR_INVALID;
    const Lane ln{static_cast<cudaStream_t>(stream), c->num_sms};
    const int seq[] = {B_CGRAD, B_DGRAD1, B_DGRAD2, B_SHARED, B_ROUTE_BWD, B_UNPACK};
    for (int t : seq) {
        if (t == B_SHARED && !c->D.I_shared) continue;
        const int rc = run_task(c, t, ln, nullptr, a, PART_BI);
        if (rc != PIPER_OK) return rc;
    }
    return PIPER_OK;
}

int piper_run_chunk_bwd_weight(piper_ctx* c, const piper_chunk_args* a, void* stream) {
    if (!c || !bwd_args_ok(c, a)) return PIPER_ERR_INVALID;
    const Lane ln{static_cast<cudaStream_t>(stream), c->num_sms};
    int rc = run_task(c, B_WGRAD, ln, nullptr, a);
    if (rc == PIPER_OK && c->D.I_shared) rc = run_task(c, B_SHARED, ln, nullptr, a, PART_BW);
    return rc;
}

int piper_set_pair_bwd_pass(piper_ctx* c, int pass) {
    if (!c || (pass != PIPER_PASS_B && pass != PIPER_PASS_BI)) return PIPER_ERR_INVALID;
    if (pass != c->pair_bwd_pass) pair_plan_release(c);
    c->pair_bwd_pass = pass;
    return PIPER_OK;
}

namespace {

// Task durations in ms on the whole device: the caller's profile, else an estimate from the algorithmic work
// (GEMM tasks at 1.2 PFLOP/s, row movers at 4.5 TB/s, the small routing kernels at a launch-sized 10 us).
void task_durations(const piper_ctx* c, float* ms) {
    if (c->pair_have_ms) {
        for (int t = 0; t < N_TASKS; ++t) ms[t] = c->pair_task_ms[t];
        return;
    }
    const piper_moe_desc& D = c->D;
    const double A = (double)D.T * D.k * D.E_loc / D.E, b = (double)esize(D.dtype), sh = D.I_shared ? 1.0 : 0.0;
    const double di = (double)D.d * D.I, dis = (double)D.d * D.I_shared, tf = 1.2e12, bw = 4.5e9;
    const double rows = (A + D.T + sh * D.T) * D.d * b;
    ms[F_ROUTE] = ms[F_SCAN] = ms[B_ROUTE_BWD] = 0.01f;
    ms[F_PACK] = (float)(2 * A * D.d * b / bw), ms[F_COMBINE] = ms[B_UNPACK] = (float)(rows / bw);
    ms[B_CGRAD] = (float)(3 * A * D.d * b / bw);
    ms[F_GEMM1] = ms[B_DGRAD2] = (float)(4 * di * A / tf), ms[F_GEMM2] = ms[B_DGRAD1] = (float)(2 * di * A / tf);
    ms[B_WGRAD] = (float)(6 * di * A / tf);
    ms[F_SHARED] = (float)(6 * dis * D.T / tf), ms[B_SHARED] = (float)(12 * dis * D.T / tf);
}

int make_plan_uncached(piper_ctx* c, int sm_gemm, int sm_comm, bool router, PairPlan* pl);

// The plan is a pure function of (descriptor, policy, split): computed once and kept (the profile-guided search
// costs milliseconds of host time, which would otherwise sit between two launches).
int make_plan(piper_ctx* c, int sm_gemm, int sm_comm, bool router, PairPlan* pl) {
    PairPlan* cached = static_cast<PairPlan*>(c->pair_plan);
    if (cached && c->plan_sm_gemm == sm_gemm && c->plan_sm_comm == sm_comm && cached->router == router) {
        *pl = *cached;
        return PIPER_OK;
    }
    const int rc = make_plan_uncached(c, sm_gemm, sm_comm, router, pl);
    if (rc != PIPER_OK) return rc;
    if (!cached) cached = new (std::nothrow) PairPlan(), c->pair_plan = cached;
    if (cached) *cached = *pl, c->plan_sm_gemm = sm_gemm, c->plan_sm_comm = sm_comm;
    return PIPER_OK;
}

int make_plan_uncached(piper_ctx* c, int sm_gemm, int sm_comm, bool router, PairPlan* pl) {
    pl->router = router;
    // task list of this layer (no shared expert -> its two tasks and their edges drop out)
    const bool shared = c->D.I_shared != 0;
    int32_t id_of[N_ALL], n = 0;
    for (int t = 0; t < N_ALL; ++t) {
        id_of[t] = -1;
        if (!shared && (t == F_SHARED || t == B_SHARED)) continue;
        if (t == B_WGRAD && c->pair_bwd_pass == PIPER_PASS_BI) continue;  // F || Bi: the weight gradients run later
        if (t >= X_F_PRE && !c->caller_fn[t - X_F_PRE]) continue;          // N3: caller tasks that are set
        id_of[t] = n, pl->task_of[n] = t, ++n;
    }
    pl->n = n;
    int32_t edges[32][2], n_edges = 0, prio[N_ALL];
    for (const auto& e : kEdges)
        if (id_of[e[0]] >= 0 && id_of[e[1]] >= 0) edges[n_edges][0] = id_of[e[0]], edges[n_edges][1] = id_of[e[1]], ++n_edges;
    for (const auto& e : kCallerEdges)
        if (id_of[e[0]] >= 0 && id_of[e[1]] >= 0) edges[n_edges][0] = id_of[e[0]], edges[n_edges][1] = id_of[e[1]], ++n_edges;
    if (router)  // N1: B.route_bwd also produces the router's term of dX, which B.unpack adds
        edges[n_edges][0] = id_of[B_ROUTE_BWD], edges[n_edges][1] = id_of[B_UNPACK], ++n_edges;
    for (int i = 0; i < n; ++i) {
        const int t = pl->task_of[i];
        pl->stream_of[i] = t >= X_F_PRE ? c->caller_side[t - X_F_PRE] : kStreamOf[t];
        prio[i] = (t >= B_CGRAD && t < N_TASKS) || t == X_B_PRE || t == X_B_POST ? 1 : 0;
    }
    pl->n_waits = 0;
    if (c->pair_order == PIPER_ORDER_LIST)
        return piper_list_schedule(n, n_edges, &edges[0][0], pl->stream_of, prio, pl->order, &pl->waits[0][0], &pl->n_waits,
                                   pl->records);
    // durations on the partitions: GEMM tasks scale with the SM count; the row movers saturate HBM with about a
    // third of the SMs, below that they scale with the SM count
    float full[N_ALL], dur[N_ALL];
    task_durations(c, full);
    for (int sl = 0; sl < 4; ++sl) full[X_F_PRE + sl] = c->caller_ms[sl];
    const float fg = (float)c->num_sms / (float)(sm_gemm < c->num_sms ? sm_gemm : c->num_sms);
    const float fc = sm_comm * 3 >= c->num_sms ? 1.f : (float)c->num_sms / (3.f * (float)sm_comm);
    for (int i = 0; i < n; ++i) dur[i] = full[pl->task_of[i]] * (pl->stream_of[i] == GEMM ? fg : fc);
    if (c->pair_bwd_pass == PIPER_PASS_BI && id_of[B_SHARED] >= 0) dur[id_of[B_SHARED]] *= 2.f / 3.f;  // dgrads only
    return piper_schedule_search(n, n_edges, &edges[0][0], pl->stream_of, dur, pl->order, &pl->waits[0][0], &pl->n_waits,
                                 pl->records, nullptr);
}

bool split_ok(const piper_ctx* c, int sm_gemm, int sm_comm) {
    if (sm_gemm < 1 || sm_comm < 8 || sm_comm % 8 || sm_gemm > c->num_sms || sm_comm > c->num_sms) return false;
    if (c->pair_part != PIPER_PART_EXCLUSIVE) return true;
    // disjoint green-context partitions come in multiples of 8 SMs; the GEMM side may instead take the whole remainder
    return sm_gemm + sm_comm <= c->num_sms && (sm_gemm % 8 == 0 || sm_gemm + sm_comm == c->num_sms);
}

// Partition + streams + schedule of a split (created once, kept until the split or the partition policy changes).
int pair_prepare(piper_ctx* c, int sm_gemm, int sm_comm, bool router, PairPlan* pl) {
    if (!split_ok(c, sm_gemm, sm_comm)) return PIPER_ERR_INVALID;
    if (!c->green || c->green->sm_gemm != sm_gemm || c->green->sm_comm != sm_comm) {
        pair_release(c);
        c->green = make_partition(c, sm_gemm, sm_comm, c->pair_part == PIPER_PART_EXCLUSIVE);
        if (!c->green) {
            snprintf(c->err, sizeof(c->err), "SM partition %d:%d unavailable (%s)", sm_gemm, sm_comm,
                     c->pair_part == PIPER_PART_EXCLUSIVE ? "green contexts" : "stream creation");
            return c->pair_part == PIPER_PART_EXCLUSIVE ? PIPER_ERR_UNSUPPORTED : PIPER_ERR_CUDA;
        }
    }
    return make_plan(c, sm_gemm, sm_comm, router, pl);
}

}  // namespace

int piper_set_pair_policy(piper_ctx* c, int order, int partition, const float* task_ms) {
    if (!c || (order != PIPER_ORDER_LIST && order != PIPER_ORDER_PROFILE) ||
        (partition != PIPER_PART_EXCLUSIVE && partition != PIPER_PART_SHARED && partition != PIPER_PART_CHUNK_STREAMS))
        return PIPER_ERR_INVALID;
    if (task_ms)
        for (int t = 0; t < N_TASKS; ++t)
            if (!(task_ms[t] >= 0.f)) return PIPER_ERR_INVALID;
    if (partition != c->pair_part) pair_release(c);
    pair_plan_release(c);
    c->pair_order = order, c->pair_part = partition, c->pair_have_ms = task_ms != nullptr;
    if (task_ms)
        for (int t = 0; t < N_TASKS; ++t) c->pair_task_ms[t] = task_ms[t];
    return PIPER_OK;
}

int piper_pair_set_caller_task(piper_ctx* c, int slot, piper_caller_task_fn fn, void* user, float est_ms, int side) {
    if (!c || slot < 0 || slot > 3 || (side != COMM && side != GEMM) || !(est_ms >= 0.f)) return PIPER_ERR_INVALID;
    c->caller_fn[slot] = fn, c->caller_user[slot] = fn ? user : nullptr;
    c->caller_ms[slot] = fn ? est_ms : 0.f, c->caller_side[slot] = side;
    pair_plan_release(c);  // the DAG changes
    return PIPER_OK;
}

int piper_pair_order(piper_ctx* c, int sm_gemm, int sm_comm, int32_t* order, int32_t* n) {
    if (!c || !order || !n || !split_ok(c, sm_gemm, sm_comm)) return PIPER_ERR_INVALID;
    PairPlan pl;
    const int rc = make_plan(c, sm_gemm, sm_comm, false, &pl);
    if (rc != PIPER_OK) return rc;
    for (int i = 0; i < pl.n; ++i) order[i] = pl.task_of[pl.order[i]];
    *n = pl.n;
    return PIPER_OK;
}

int piper_pair_prepare(piper_ctx* c, int sm_gemm, int sm_comm) {
    if (!c) return PIPER_ERR_INVALID;
    PairPlan pl;
    return pair_prepare(c, sm_gemm, sm_comm, false, &pl);
}

int piper_run_chunk_pair(piper_ctx* c, const piper_chunk_args* f, const piper_chunk_args* b, int sm_gemm, int sm_comm,
                         void* stream) {
    if (!c || !fwd_args_ok(c, f) || !bwd_args_ok(c, b)) return PIPER_ERR_INVALID;
    PairPlan pl;
    int rc = pair_prepare(c, sm_gemm, sm_comm, b->w_r != nullptr, &pl);
    if (rc != PIPER_OK) return rc;
    GreenPartition* g = c->green;
    c->pair_mode = c->pair_part == PIPER_PART_CHUNK_STREAMS ? 3 : (g->green ? 1 : 2);
    const int parts = c->pair_bwd_pass == PIPER_PASS_BI ? PART_BI : PART_ALL;

    cudaStream_t user = static_cast<cudaStream_t>(stream);
    if (c->pair_part == PIPER_PART_CHUNK_STREAMS) {
        // One stream per chunk, every grid sized for the whole device, no cross-stream edge (the two microbatches are
        // independent): which SM runs what is left to the GPU's block scheduler, as in the paper.  The
        // persistent GEMM grids of the two chunks cannot be co-resident (one CTA fills an SM's shared memory), so a
        // chunk's next GEMM moves in SM by SM as the other's clusters retire (the tile feeds are dynamic or strided:
        // no kernel waits on a CTA that is not resident), and the row movers run beside whichever GEMM is resident.
        const Lane lf{g->stream[0], c->num_sms}, lb{g->stream[1], c->num_sms};
        cudaEvent_t fork = c->events[kMaxEvents - 1], join0 = c->events[kMaxEvents - 2], join1 = c->events[kMaxEvents - 3];
        PIPER_CUDA(c, cudaEventRecord(fork, user));
        PIPER_CUDA(c, cudaStreamWaitEvent(lf.stream, fork, 0));
        PIPER_CUDA(c, cudaStreamWaitEvent(lb.stream, fork, 0));
        const int fseq[] = {X_F_PRE, F_ROUTE, F_SCAN, F_PACK, F_SHARED, F_GEMM1, F_GEMM2, F_COMBINE, X_F_POST};
        const int bseq[] = {X_B_PRE, B_CGRAD, B_DGRAD1, B_DGRAD2, B_WGRAD, B_SHARED, B_ROUTE_BWD, B_UNPACK, X_B_POST};
        auto in_plan = [&](int t) {
            if (t >= X_F_PRE) return c->caller_fn[t - X_F_PRE] != nullptr;
            if ((t == F_SHARED || t == B_SHARED) && !c->D.I_shared) return false;
            return !(t == B_WGRAD && parts == PART_BI);
        };
        for (int i = 0; i < 9; ++i) {  // enqueued alternately, each chunk in its serial order
            if (in_plan(fseq[i])) {
                rc = run_task(c, fseq[i], lf, f, b);
                if (rc != PIPER_OK) return rc;
            }
            if (in_plan(bseq[i])) {
                rc = run_task(c, bseq[i], lb, f, b, parts);
                if (rc != PIPER_OK) return rc;
            }
        }
        PIPER_CUDA(c, cudaEventRecord(join0, lf.stream));
        PIPER_CUDA(c, cudaEventRecord(join1, lb.stream));
        PIPER_CUDA(c, cudaStreamWaitEvent(user, join0, 0));
        PIPER_CUDA(c, cudaStreamWaitEvent(user, join1, 0));
        return PIPER_OK;
    }
    const Lane lanes[2] = {{g->stream[COMM], sm_comm}, {g->stream[GEMM], sm_gemm}};
    // fork: both partitions start after the work already queued on the caller's stream
    cudaEvent_t fork = c->events[kMaxEvents - 1], join0 = c->events[kMaxEvents - 2], join1 = c->events[kMaxEvents - 3];
    PIPER_CUDA(c, cudaEventRecord(fork, user));
    PIPER_CUDA(c, cudaStreamWaitEvent(lanes[0].stream, fork, 0));
    PIPER_CUDA(c, cudaStreamWaitEvent(lanes[1].stream, fork, 0));
    for (int step = 0; step < pl.n; ++step) {
        const int v = pl.order[step];
        const Lane ln = lanes[pl.stream_of[v]];
        for (int w = 0; w < pl.n_waits; ++w)  // wait for dependencies that ran on another stream
            if (pl.waits[w][1] == v) PIPER_CUDA(c, cudaStreamWaitEvent(ln.stream, c->events[pl.waits[w][0]], 0));
        rc = run_task(c, pl.task_of[v], ln, f, b, parts);
        if (rc != PIPER_OK) return rc;
        if (pl.records[v]) PIPER_CUDA(c, cudaEventRecord(c->events[v], ln.stream));
    }
    PIPER_CUDA(c, cudaEventRecord(join0, lanes[0].stream));
    PIPER_CUDA(c, cudaEventRecord(join1, lanes[1].stream));
    PIPER_CUDA(c, cudaStreamWaitEvent(user, join0, 0));
    PIPER_CUDA(c, cudaStreamWaitEvent(user, join1, 0));
    return PIPER_OK;
}

}  // extern "C"
