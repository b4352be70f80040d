// fmm_api.cu -- the C-ABI entry points of include/fmm.h and the host orchestration of
// Alg 5.12: fmm_plan_create = subdivide + dualtraversefillitl (a0-a3),
// fmm_eval = upward pass, M2L + P2P over the lists, downward pass (a4-a10).
#include "fmm_internal.cuh"

#include <math.h>
#include <algorithm>
#include <new>

std::atomic<int64_t> g_fmm_launches{0};
static thread_local char g_last_error[256] = "";

// ---------------------------------------------------------------------------------------
// context: allocator, stream, error text
// ---------------------------------------------------------------------------------------
static void ctx_init(fmm_ctx *c, fmm_alloc_fn alloc, fmm_free_fn free_, void *user, void *stream)
{
    c->alloc = alloc;
    c->free_ = free_;
    c->user = user;
    c->stream = (cudaStream_t)stream;
    c->err[0] = 0;
    c->bytes = 0;
    c->arena = NULL;
    c->arena_cap = c->arena_top = c->arena_need = 0;
    c->arena_on = 0;
}

static void ctx_set_error(fmm_ctx *c, const char *msg)
{
    snprintf(c->err, sizeof(c->err), "%s", msg);
    snprintf(g_last_error, sizeof(g_last_error), "%s", msg);
}

int ctx_cuda_fail(fmm_ctx *c, cudaError_t e, const char *what)
{
    char buf[256];
    snprintf(buf, sizeof(buf), "%s: %s", what, cudaGetErrorString(e));
    ctx_set_error(c, buf);
    return FMM_ECUDA;
}

void *ctx_alloc(fmm_ctx *c, size_t bytes)
{
    if (c->arena_on) {
        const size_t need = ((bytes ? bytes : 8) + 255) & ~(size_t)255;
        c->arena_need += need;
        if (c->arena_top + need <= c->arena_cap) {
            void *p = c->arena + c->arena_top;
            c->arena_marks.push_back(c->arena_top);
            c->arena_live.push_back(1);
            c->arena_top += need;
            return p;
        }
    }
    return ctx_alloc_keep(c, bytes);
}

int ctx_arena_begin(fmm_ctx *c, size_t estimate)
{
    size_t want = estimate > c->arena_need + c->arena_need / 8 ? estimate : c->arena_need + c->arena_need / 8;  // what the last build asked for
    if (want > c->arena_cap) {
        if (c->arena) ctx_free_keep(c, c->arena);
        c->arena = NULL;
        c->arena_cap = 0;
        c->arena = (char *)ctx_alloc_keep(c, want);
        if (!c->arena) return FMM_ENOMEM;
        c->arena_cap = want;
    }
    c->arena_top = c->arena_need = 0;
    c->arena_marks.clear();
    c->arena_live.clear();
    c->arena_on = 1;
    return FMM_OK;
}

void ctx_arena_end(fmm_ctx *c) { c->arena_on = 0; }

void *ctx_alloc_keep(fmm_ctx *c, size_t bytes)
{
    if (bytes == 0) bytes = 8;
    void *p = NULL;
    if (c->alloc) {
        p = c->alloc(bytes, c->user);
    } else {
        if (cudaMallocAsync(&p, bytes, c->stream) != cudaSuccess) p = NULL;
    }
    if (!p) {
        char buf[128];
        snprintf(buf, sizeof(buf), "allocator returned NULL for %zu bytes", bytes);
        ctx_set_error(c, buf);
        return NULL;
    }
    c->owned.push_back(p);
    c->owned_bytes.push_back(bytes);
    c->bytes += (int64_t)bytes;
    return p;
}

void ctx_free(fmm_ctx *c, void *p)
{
    if (!p) return;
    if (c->arena && (char *)p >= c->arena && (char *)p < c->arena + c->arena_cap) {
        // arena block: its space comes back once it is the newest live block (together with everything freed below it)
        const size_t at = (size_t)((char *)p - c->arena);
        for (size_t k = c->arena_marks.size(); k-- > 0;)
            if (c->arena_marks[k] == at) { c->arena_live[k] = 0; break; }
        while (!c->arena_marks.empty() && !c->arena_live.back()) {
            c->arena_top = c->arena_marks.back();
            c->arena_marks.pop_back();
            c->arena_live.pop_back();
        }
        return;
    }
    ctx_free_keep(c, p);
}

void ctx_free_keep(fmm_ctx *c, void *p)
{
    if (!p) return;
    for (size_t k = c->owned.size(); k-- > 0;) {
        if (c->owned[k] == p) {
            c->bytes -= (int64_t)c->owned_bytes[k];
            c->owned.erase(c->owned.begin() + k);
            c->owned_bytes.erase(c->owned_bytes.begin() + k);
            break;
        }
    }
    if (c->free_) c->free_(p, c->user);
    else cudaFreeAsync(p, c->stream);
}

void ctx_free_all(fmm_ctx *c)
{
    while (!c->owned.empty()) ctx_free_keep(c, c->owned.back());
    c->arena = NULL;
    c->arena_cap = 0;
}

// One side stream per device for the near / far overlap, created on first use and kept for the life of the process
// (creating a stream costs about a millisecond, too much for fmm_field_host, which builds a plan per call).  Plans that
// share it are still ordered correctly: every fmm_eval forks from and joins into its own stream with events.
#include <mutex>
static cudaError_t side_stream_for_current_device(cudaStream_t *out)
{
    static std::mutex mu;
    static cudaStream_t streams[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!streams[dev]) {
        e = cudaStreamCreateWithFlags(&streams[dev], cudaStreamNonBlocking);
        if (e != cudaSuccess) return e;
    }
    *out = streams[dev];
    return cudaSuccess;
}

static int check_particles(const fmm_particles_t *in)
{
    if (!in || in->N < 1 || in->N >= ((int64_t)1 << 31)) return FMM_EINVAL;
    if (!in->x || !in->y || !in->z || !in->px || !in->py || !in->pz) return FMM_EINVAL;
    return FMM_OK;
}

extern "C" const char *fmm_strerror(int code)
{
    switch (code) {
        case FMM_OK: return "ok";
        case FMM_EINVAL: return "invalid argument";
        case FMM_ENOMEM: return "device allocator returned NULL";
        case FMM_ECUDA: return "CUDA error";
        case FMM_ENONFINITE: return "NaN or Inf among the positions, momenta or charges";
        case FMM_EOVERFLOW: return "interaction list exceeds 2^31-1 entries";
    }
    return "unknown error code";
}

extern "C" const char *fmm_last_error(const fmm_plan_t *plan) { return plan ? plan->ctx.err : g_last_error; }
extern "C" const char *fmm_version(void) { return "fmm_b200 0.1 (sm_100a, FP64)"; }
extern "C" int64_t fmm_launch_count(void) { return g_fmm_launches.load(); }

// ---------------------------------------------------------------------------------------
// plan: a0-a3
// ---------------------------------------------------------------------------------------
static int plan_alloc_fixed(fmm_plan *p)
{
    fmm_ctx *c = &p->ctx;
    const size_t N = (size_t)p->N, nodes1 = (size_t)p->nodes + 2;
#define ALLOC(field, type, count)                                         \
    do {                                                                  \
        p->field = (type *)ctx_alloc(c, sizeof(type) * (size_t)(count));  \
        if (!p->field) return FMM_ENOMEM;                                 \
    } while (0)
    ALLOC(tx, double, N); ALLOC(ty, double, N); ALLOC(tz, double, N);
    ALLOC(w0, double, N); ALLOC(w1, double, N); ALLOC(w2, double, N); ALLOC(w3, double, N);
    if (p->flags & FMM_KERNEL_SOURCE_MOMENTUM) {
        ALLOC(pmx, double, N); ALLOC(pmy, double, N); ALLOC(pmz, double, N);
    }
    ALLOC(perm, int32_t, N);
    ALLOC(hdr, fmm_hdr, 1);
    ALLOC(node_lo, int32_t, nodes1); ALLOC(node_hi, int32_t, nodes1);
    ALLOC(bbox, double, 6 * nodes1); ALLOC(node_geo, double, 4 * nodes1);
    ALLOC(node_xi, double, 48 * nodes1);
    ALLOC(xfer_sync, int, 2 * nodes1);
    if (cudaMemsetAsync(p->xfer_sync, 0, sizeof(int) * 2 * nodes1, c->stream) != cudaSuccess) return FMM_ECUDA;
    ALLOC(node_T, double, (size_t)((3 * p->n1 * p->n1 + 1) & ~1) * nodes1);
    ALLOC(p2p_off, int32_t, nodes1 + 1); ALLOC(m2l_off, int32_t, nodes1 + 1);
    ALLOC(p2p_order, int32_t, nodes1); ALLOC(m2l_order, int32_t, nodes1);
    ALLOC(M, double, 4 * (size_t)p->P * nodes1);
    ALLOC(L, double, 6 * (size_t)p->P * nodes1);
#undef ALLOC
    return FMM_OK;
}

// a4 + a5 (P2M, M2M): the moments depend on the tree and the particles only, so a build enqueues them itself, right behind
// the copies its one host wait is for (kernels_dtt.cu): the GPU works on them while the host reads the list lengths, returns
// to the caller and comes back with fmm_eval, instead of idling for that time.  fmm_eval finds them done.
int plan_upward(fmm_plan *p)
{
    if (p->upward_done) return FMM_OK;
    if (p->timing) FMM_CUDA(&p->ctx, cudaEventRecord(p->ev[EV_P2M], p->ctx.stream));
    FMM_TRY(interp_p2m(p));          // Alg 5.3 at the leaves
    if (p->timing) FMM_CUDA(&p->ctx, cudaEventRecord(p->ev[EV_M2M], p->ctx.stream));
    FMM_TRY(interp_m2m(p));          // Alg 5.4, levels kappa-1 .. 0 (Alg 5.5)
    if (p->timing) FMM_CUDA(&p->ctx, cudaEventRecord(p->ev[EV_UPEND], p->ctx.stream));
    p->upward_done = 1;
    return FMM_OK;
}

static int plan_build(fmm_plan *p, const fmm_particles_t *in, bool refit = false, bool keep_lists = false, double *eta_eff = NULL)
{
    fmm_ctx *c = &p->ctx;
    if (keep_lists && !p->valid) {
        snprintf(c->err, sizeof(c->err), "fmm_plan_refit_keep_lists: the plan has no valid lists to keep");
        return FMM_EINVAL;
    }
    p->valid = 0;  // a build that fails part-way leaves lists that must not be used (fmm_eval then returns FMM_EINVAL)
    // scratch of the whole build from one arena block: sort keys and index lists of the tree (about 100 N bytes), frontier
    // and pair buffers of the traversal; sized from the last build once there was one
    const size_t estimate = (size_t)(p->N >= ((int64_t)1 << 21) ? 184 : 120) * (size_t)p->N + (size_t)64 * (size_t)(p->list_cap > 0 ? p->list_cap : p->leaves * 128) +
                            (size_t)64 * (size_t)p->nodes + ((size_t)4 << 20);
    FMM_TRY(ctx_arena_begin(c, estimate));
    struct arena_guard { fmm_ctx *c; ~arena_guard() { ctx_arena_end(c); } } guard{c};
    for (int round = 0; round < 2; ++round) {
        if (round == 1) {  // the quantised sort keys of the KD build were not enough (kernels_kd.cu): once more with exact keys
            p->kd_exact = 1;
            ctx_arena_end(c);
            FMM_TRY(ctx_arena_begin(c, estimate + (size_t)48 * (size_t)p->N));
        }
        p->upward_done = 0;
        FMM_CUDA(c, cudaEventRecord(p->ev_plan[0], c->stream));
        FMM_TRY(tree_scan_inputs(p, in));  // a0: gamma_bar, coordinate ranges, input check -> p->hdr (device)
        FMM_TRY(refit ? tree_refit(p, in) : tree_build(p, in));
        FMM_CUDA(c, cudaEventRecord(p->ev_plan[1], c->stream));
        if (keep_lists) {
            FMM_TRY(dtt_keep_lists(p, eta_eff));
            break;
        }
        FMM_TRY(dtt_build_lists(p));       // (reads gamma_bar and the input check back together with the list lengths; records
                                           //  ev_plan[2] behind its last kernel and enqueues the upward pass before it waits)
        if (!p->kd_retry) break;
    }
    FMM_TRY(pairs_p2p_prepare(p));
    FMM_TRY(pairs_m2l_prepare(p));
    p->plan_ms_pending = 1;  // (read in fmm_plan_stats: the tail of the build is enqueue-only)
    p->ev_valid = 0;
    p->valid = 1;
    return FMM_OK;
}

extern "C" void fmm_plan_destroy(fmm_plan_t *p)
{
    if (!p) return;
    cudaStreamSynchronize(p->ctx.stream);
    ctx_free_all(&p->ctx);
    for (int k = 0; k < EV_COUNT; ++k)
        if (p->ev[k]) cudaEventDestroy(p->ev[k]);
    for (int k = 0; k < 3; ++k)
        if (p->ev_plan[k]) cudaEventDestroy(p->ev_plan[k]);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    delete p;
}

extern "C" int fmm_plan_create(fmm_plan_t **out, const fmm_particles_t *in, const fmm_params_t *prm,
                               fmm_alloc_fn alloc, fmm_free_fn free_, void *user, void *cuda_stream)
{
    if (!out) return FMM_EINVAL;
    *out = NULL;
    if (check_particles(in) != FMM_OK || !prm) return FMM_EINVAL;
    if (prm->order_n < 1 || prm->order_n > FMM_MAX_ORDER || prm->leaf_size < 1) return FMM_EINVAL;
    if (!(prm->theta > 0.0) || !isfinite(prm->theta)) return FMM_EINVAL;
    if ((alloc == NULL) != (free_ == NULL)) return FMM_EINVAL;
    if (isnan(prm->gamma_bar) || isinf(prm->gamma_bar)) return FMM_EINVAL;
    fmm_plan *p = new (std::nothrow) fmm_plan();
    if (!p) return FMM_ENOMEM;
    ctx_init(&p->ctx, alloc, free_, user, cuda_stream);
    p->N = in->N;
    p->n = prm->order_n;
    p->n1 = p->n + 1;
    p->P = p->n1 * p->n1 * p->n1;
    p->N0 = prm->leaf_size;
    p->theta = prm->theta;
    p->gamma_bar_param = prm->gamma_bar;
    p->flags = prm->flags;
    int kappa = 0;  // T-1: smallest kappa with N0 2^kappa >= N
    while (((int64_t)p->N0 << kappa) < p->N) ++kappa;
    p->kappa = kappa;
    p->leaves = (int64_t)1 << kappa;
    p->nodes = ((int64_t)2 << kappa) - 1;
    p->stop_level = -1;
    p->early_leaves = 0;
    p->maxleaf = (int)((p->N + p->leaves - 1) / p->leaves);
    if ((p->flags & FMM_TREE_STOP_AT_N0) && kappa >= 1) {
        // sizes on level kappa-1 are floor or ceil of N / 2^(kappa-1) > N0: clusters of exactly N0 exist iff the floor is N0
        const int64_t m = (int64_t)1 << (kappa - 1);
        if (p->N / m == p->N0) {
            p->stop_level = kappa - 1;
            p->early_leaves = (int)(m - p->N % m);
            p->maxleaf = p->N0;
        }
    }
    int rc = FMM_OK;
    for (int k = 0; k < EV_COUNT && rc == FMM_OK; ++k)
        if (cudaEventCreate(&p->ev[k]) != cudaSuccess) rc = FMM_ECUDA;
    for (int k = 0; k < 3 && rc == FMM_OK; ++k)
        if (cudaEventCreate(&p->ev_plan[k]) != cudaSuccess) rc = FMM_ECUDA;
    if (rc == FMM_OK && (side_stream_for_current_device(&p->side) != cudaSuccess ||
                         cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                         cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming) != cudaSuccess))
        rc = FMM_ECUDA;
    p->overlap = 0;  // opt-in (fmm_plan_set_overlap): +2 % at the headline workload, but up to -45 % when P2P dominates
    if (rc == FMM_OK) rc = plan_alloc_fixed(p);
    if (rc == FMM_OK) rc = plan_build(p, in);
    if (rc != FMM_OK) {
        snprintf(g_last_error, sizeof(g_last_error), "%s", p->ctx.err);
        fmm_plan_destroy(p);
        return rc;
    }
    *out = p;
    return FMM_OK;
}

extern "C" int fmm_plan_update(fmm_plan_t *p, const fmm_particles_t *in)
{
    if (!p || check_particles(in) != FMM_OK || in->N != p->N) return FMM_EINVAL;
    return plan_build(p, in);
}

extern "C" int fmm_plan_refit(fmm_plan_t *p, const fmm_particles_t *in)
{
    if (!p || check_particles(in) != FMM_OK || in->N != p->N) return FMM_EINVAL;
    return plan_build(p, in, true);
}

extern "C" int fmm_plan_refit_keep_lists(fmm_plan_t *p, const fmm_particles_t *in, double *eta_eff)
{
    if (!p || check_particles(in) != FMM_OK || in->N != p->N) return FMM_EINVAL;
    if (p->flags & FMM_METHOD_TREECODE) return FMM_EINVAL;
    return plan_build(p, in, true, true, eta_eff);
}

extern "C" int fmm_plan_set_overlap(fmm_plan_t *p, int on)
{
    if (!p) return FMM_EINVAL;
    p->overlap = on ? 1 : 0;
    return FMM_OK;
}

extern "C" int fmm_plan_set_timing(fmm_plan_t *p, int on)
{
    if (!p) return FMM_EINVAL;
    p->timing = on ? 1 : 0;
    p->ev_valid = 0;
    p->upward_done = 0;  // (the next fmm_eval runs the upward pass again, between its own events)
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// evaluation: a4-a10
// ---------------------------------------------------------------------------------------
#define MARK(p, id)                                                                   \
    do {                                                                              \
        if ((p)->timing) FMM_CUDA(&(p)->ctx, cudaEventRecord((p)->ev[id], (p)->ctx.stream)); \
    } while (0)

extern "C" int fmm_eval(fmm_plan_t *p, double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz)
{
    if (!p || !Ex || !Ey || !Ez || !Bx || !By || !Bz) return FMM_EINVAL;
    if (!p->valid) {
        snprintf(p->ctx.err, sizeof(p->ctx.err), "the last fmm_plan_update / fmm_plan_refit of this plan failed: its lists are not usable");
        return FMM_EINVAL;
    }
    if (p->flags & FMM_METHOD_TREECODE) {  // P2M, M2M, particle-cluster + P2P, finalise (no M2L / L2L / far L2P)
        FMM_TRY(plan_upward(p));
        MARK(p, EV_M2L);
        FMM_TRY(pairs_pc(p));
        MARK(p, EV_L2L);
        MARK(p, EV_P2P);
        FMM_TRY(pairs_p2p(p));
        MARK(p, EV_L2P);
        FMM_TRY(interp_l2p_finalize(p, Ex, Ey, Ez, Bx, By, Bz));
        MARK(p, EV_END);
        if (p->timing) p->ev_valid = 1;
        return FMM_OK;
    }
    if (p->overlap && !p->timing) {
        // a7 does not depend on a4-a6/a8: it runs on the side stream, forked after everything already enqueued on the
        // caller's stream and joined before L2P adds near + far.  Results are identical (each kernel is deterministic).
        fmm_ctx *c = &p->ctx;
        cudaStream_t main_stream = c->stream;
        FMM_CUDA(c, cudaEventRecord(p->ev_fork, main_stream));
        FMM_CUDA(c, cudaStreamWaitEvent(p->side, p->ev_fork, 0));
        FMM_TRY(plan_upward(p));
        FMM_TRY(pairs_m2l(p));
        c->stream = p->side;
        int rc = pairs_p2p(p);
        c->stream = main_stream;
        FMM_TRY(rc);
        FMM_CUDA(c, cudaEventRecord(p->ev_join, p->side));
        FMM_TRY(interp_l2l(p));
        FMM_CUDA(c, cudaStreamWaitEvent(main_stream, p->ev_join, 0));
        FMM_TRY(interp_l2p_finalize(p, Ex, Ey, Ez, Bx, By, Bz));
        return FMM_OK;
    }
    FMM_TRY(plan_upward(p));         // Alg 5.3-5.5 (already enqueued by the build unless timing was switched on since)
    MARK(p, EV_M2L);
    FMM_TRY(pairs_m2l(p));           // Alg 5.9 over m2l_itl
    MARK(p, EV_L2L);
    FMM_TRY(interp_l2l(p));          // Alg 5.13, levels 1 .. kappa (Alg 5.15)
    MARK(p, EV_P2P);
    FMM_TRY(pairs_p2p(p));           // Alg 5.10 over p2p_itl
    MARK(p, EV_L2P);
    FMM_TRY(interp_l2p_finalize(p, Ex, Ey, Ez, Bx, By, Bz));  // Alg 5.14 + eq. (3.1) prefactors
    MARK(p, EV_END);
    if (p->timing) p->ev_valid = 1;
    return FMM_OK;
}

extern "C" int fmm_plan_stats(fmm_plan_t *p, fmm_stats_t *s)
{
    if (!p || !s) return FMM_EINVAL;
    memset(s, 0, sizeof(*s));
    s->N = p->N;
    s->order_n = p->n;
    s->P = p->P;
    s->leaf_size = p->N0;
    s->kappa = p->kappa;
    s->nodes = p->nodes;
    s->leaves = p->leaves;
    s->n_p2p = p->n_p2p;
    s->n_m2l = p->n_m2l;
    s->p2p_pairs = p->p2p_pairs;
    s->m2l_pairs = p->m2l_pairs;
    s->gamma_bar = p->gamma_bar;
    s->theta = p->theta;
    s->flags = p->flags;
    if (p->plan_ms_pending) {
        fmm_ctx *c = &p->ctx;
        FMM_CUDA(c, cudaEventSynchronize(p->ev_plan[2]));
        FMM_CUDA(c, cudaEventElapsedTime(&p->ms_tree, p->ev_plan[0], p->ev_plan[1]));
        FMM_CUDA(c, cudaEventElapsedTime(&p->ms_lists, p->ev_plan[1], p->ev_plan[2]));
        p->plan_ms_pending = 0;
    }
    s->ms_tree = p->ms_tree;
    s->ms_lists = p->ms_lists;
    s->workspace_bytes = p->ctx.bytes;
    s->p2p_split = p->p2p_split;
    s->m2l_split = p->m2l_split;
    s->p2p_mutual = (p->p2p_mutual && p->p2p_dst != NULL) ? 1 : 0;
    s->react_particles = s->p2p_mutual ? p->p2p_react : 0;
    s->early_leaves = p->early_leaves;
    if (p->timing && p->ev_valid) {
        fmm_ctx *c = &p->ctx;
        FMM_CUDA(c, cudaEventSynchronize(p->ev[EV_END]));
        FMM_CUDA(c, cudaEventElapsedTime(&s->ms_p2m, p->ev[EV_P2M], p->ev[EV_M2M]));
        FMM_CUDA(c, cudaEventElapsedTime(&s->ms_m2m, p->ev[EV_M2M], p->ev[EV_UPEND]));
        FMM_CUDA(c, cudaEventElapsedTime(&s->ms_m2l, p->ev[EV_M2L], p->ev[EV_L2L]));
        FMM_CUDA(c, cudaEventElapsedTime(&s->ms_l2l, p->ev[EV_L2L], p->ev[EV_P2P]));
        FMM_CUDA(c, cudaEventElapsedTime(&s->ms_p2p, p->ev[EV_P2P], p->ev[EV_L2P]));
        FMM_CUDA(c, cudaEventElapsedTime(&s->ms_l2p, p->ev[EV_L2P], p->ev[EV_END]));
        s->timing_valid = 1;
    }
    return FMM_OK;
}

extern "C" int fmm_plan_export(fmm_plan_t *p, fmm_export_t *o)
{
    if (!p || !o) return FMM_EINVAL;
    fmm_ctx *c = &p->ctx;
    FMM_CUDA(c, cudaStreamSynchronize(c->stream));
    const size_t N = (size_t)p->N, nodes = (size_t)p->nodes;
    std::vector<int32_t> tmp;
    auto get_i32 = [&](const int32_t *dev, size_t count) -> int {
        tmp.resize(count);
        FMM_CUDA(c, cudaMemcpy(tmp.data(), dev, sizeof(int32_t) * count, cudaMemcpyDeviceToHost));
        return FMM_OK;
    };
    if (o->perm) {
        FMM_TRY(get_i32(p->perm, N));
        for (size_t k = 0; k < N; ++k) o->perm[k] = tmp[k];
    }
    if (o->node_lo) {
        FMM_TRY(get_i32(p->node_lo + 1, nodes));
        for (size_t k = 0; k < nodes; ++k) o->node_lo[k] = tmp[k];
    }
    if (o->node_hi) {
        FMM_TRY(get_i32(p->node_hi + 1, nodes));
        for (size_t k = 0; k < nodes; ++k) o->node_hi[k] = tmp[k];
    }
    if (o->bbox) FMM_CUDA(c, cudaMemcpy(o->bbox, p->bbox + 6, sizeof(double) * 6 * nodes, cudaMemcpyDeviceToHost));
    if (o->M) FMM_CUDA(c, cudaMemcpy(o->M, p->M + 4 * (size_t)p->P, sizeof(double) * 4 * (size_t)p->P * nodes, cudaMemcpyDeviceToHost));
    if (o->L) FMM_CUDA(c, cudaMemcpy(o->L, p->L + 6 * (size_t)p->P, sizeof(double) * 6 * (size_t)p->P * nodes, cudaMemcpyDeviceToHost));
    if (p->stop_level < 0) {
        if (o->p2p_off) FMM_CUDA(c, cudaMemcpy(o->p2p_off, p->p2p_off + 1, sizeof(int32_t) * (nodes + 1), cudaMemcpyDeviceToHost));
        if (o->m2l_off) FMM_CUDA(c, cudaMemcpy(o->m2l_off, p->m2l_off + 1, sizeof(int32_t) * (nodes + 1), cudaMemcpyDeviceToHost));
        if (o->p2p_src && p->n_p2p > 0)
            FMM_CUDA(c, cudaMemcpy(o->p2p_src, p->p2p_src, sizeof(int32_t) * (size_t)p->n_p2p, cudaMemcpyDeviceToHost));
        if (o->m2l_src && p->n_m2l > 0)
            FMM_CUDA(c, cudaMemcpy(o->m2l_src, p->m2l_src, sizeof(int32_t) * (size_t)p->n_m2l, cudaMemcpyDeviceToHost));
        return FMM_OK;
    }
    // FMM_TREE_STOP_AT_N0: inside the library a leaf S of level kappa-1 works through its slot 2S (fmm_internal.cuh).  The
    // export shows the tree of Alg 5.2: S is the leaf, its two slots are unused (range [0, 0), zeros), and the lists name S.
    std::vector<int32_t> lo(nodes + 1), hi(nodes + 1);
    FMM_CUDA(c, cudaMemcpy(lo.data(), p->node_lo, sizeof(int32_t) * (nodes + 1), cudaMemcpyDeviceToHost));
    FMM_CUDA(c, cudaMemcpy(hi.data(), p->node_hi, sizeof(int32_t) * (nodes + 1), cudaMemcpyDeviceToHost));
    const size_t leaves = (size_t)p->leaves;
    std::vector<char> early(nodes + 2, 0);  // early[S] for S on level kappa-1; early[2S] = early[2S+1] = 2: unused slot
    for (size_t S = leaves / 2; S < leaves; ++S)
        if (hi[S] - lo[S] <= p->N0) { early[S] = 1; early[2 * S] = early[2 * S + 1] = 2; }
    for (size_t i = 1; i <= nodes; ++i) {
        if (early[i] != 2) continue;
        if (o->node_lo) o->node_lo[i - 1] = 0;
        if (o->node_hi) o->node_hi[i - 1] = 0;
        if (o->bbox) memset(o->bbox + 6 * (i - 1), 0, sizeof(double) * 6);
        if (o->M) memset(o->M + 4 * (size_t)p->P * (i - 1), 0, sizeof(double) * 4 * (size_t)p->P);
        if (o->L) memset(o->L + 6 * (size_t)p->P * (i - 1), 0, sizeof(double) * 6 * (size_t)p->P);
    }
    auto name_of = [&](int32_t id) -> int32_t { return early[(size_t)id] == 2 ? id / 2 : id; };  // (only the left slot 2S is ever named)
    auto remap = [&](const int32_t *dev_off, const int32_t *dev_src, int64_t n, int32_t *out_off, int32_t *out_src) -> int {
        if (!out_off && !out_src) return FMM_OK;
        std::vector<int32_t> off(nodes + 2), src((size_t)(n > 0 ? n : 1)), row;
        FMM_CUDA(c, cudaMemcpy(off.data(), dev_off, sizeof(int32_t) * (nodes + 2), cudaMemcpyDeviceToHost));
        if (n > 0) FMM_CUDA(c, cudaMemcpy(src.data(), dev_src, sizeof(int32_t) * (size_t)n, cudaMemcpyDeviceToHost));
        int32_t at = 0;
        for (size_t t = 1; t <= nodes; ++t) {  // out_off[t - 1] = start of the row of node t, out_off[nodes] = length
            if (out_off) out_off[t - 1] = at;
            if (early[t] == 2) continue;  // unused slot
            row.assign(src.begin() + off[t], src.begin() + off[t + 1]);
            if (early[t] == 1)  // P2P (and the treecode's particle-cluster) rows of S are kept under its slot 2S
                row.insert(row.end(), src.begin() + off[2 * t], src.begin() + off[2 * t + 1]);
            for (auto &v : row) v = name_of(v);
            std::sort(row.begin(), row.end());  // ascending source id in the new names (D-4)
            if (out_src) memcpy(out_src + at, row.data(), sizeof(int32_t) * row.size());
            at += (int32_t)row.size();
        }
        if (out_off) out_off[nodes] = at;
        return FMM_OK;
    };
    FMM_TRY(remap(p->p2p_off, p->p2p_src, p->n_p2p, o->p2p_off, o->p2p_src));
    FMM_TRY(remap(p->m2l_off, p->m2l_src, p->n_m2l, o->m2l_off, o->m2l_src));
    return FMM_OK;
}

// ---------------------------------------------------------------------------------------
// a11: direct summation
// ---------------------------------------------------------------------------------------
extern "C" int fmm_direct(const fmm_particles_t *in, double gamma_bar, uint32_t flags, int64_t nt, const int64_t *tidx,
                          double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz,
                          fmm_alloc_fn alloc, fmm_free_fn free_, void *user, void *cuda_stream)
{
    if (check_particles(in) != FMM_OK || nt < 1 || !Ex || !Ey || !Ez || !Bx || !By || !Bz) return FMM_EINVAL;
    if (!tidx && nt != in->N) return FMM_EINVAL;
    if ((alloc == NULL) != (free_ == NULL)) return FMM_EINVAL;
    fmm_ctx ctx;
    ctx_init(&ctx, alloc, free_, user, cuda_stream);
    fmm_ctx *c = &ctx;
    int rc = FMM_OK;
    if (!(gamma_bar > 0.0) && !(flags & FMM_KERNEL_SOURCE_MOMENTUM)) {  // the source-momentum kernel has no gamma_bar
        rc = tree_gamma_bar(c, in->N, in->px, in->py, in->pz, &gamma_bar);
        if (rc == FMM_OK && !isfinite(gamma_bar)) rc = FMM_ENONFINITE;
    }
    double *w = NULL;
    if (rc == FMM_OK) {
        w = (double *)ctx_alloc(c, sizeof(double) * 4 * (size_t)in->N);
        if (!w) rc = FMM_ENOMEM;
    }
    const size_t N = (size_t)in->N;
    if (rc == FMM_OK) rc = pairs_source_weights(c, in->N, in->px, in->py, in->pz, in->q, in->q_scalar, w, w + N, w + 2 * N, w + 3 * N);
    const bool sm = (flags & FMM_KERNEL_SOURCE_MOMENTUM) != 0;
    if (rc == FMM_OK)
        rc = pairs_direct(c, in->N, in->x, in->y, in->z, w, w + N, w + 2 * N, w + 3 * N, sm ? in->px : NULL, sm ? in->py : NULL,
                          sm ? in->pz : NULL, gamma_bar, (flags & FMM_RAW_SUMS) ? 1 : 0, nt, tidx, Ex, Ey, Ez, Bx, By, Bz);
    ctx_free_all(c);
    return rc;
}

// a11 without any allocation: scratch in a file-scope device array of kernels_pairs.cu (see there)
extern "C" int fmm_direct_noalloc(const fmm_particles_t *in, double gamma_bar, uint32_t flags, int64_t nt, const int64_t *tidx,
                                  double *Ex, double *Ey, double *Ez, double *Bx, double *By, double *Bz, void *cuda_stream)
{
    if (check_particles(in) != FMM_OK || nt < 1 || !Ex || !Ey || !Ez || !Bx || !By || !Bz) return FMM_EINVAL;
    if (!tidx && nt != in->N) return FMM_EINVAL;
    fmm_ctx ctx;
    ctx_init(&ctx, NULL, NULL, NULL, cuda_stream);
    char msg[200];
    if (in->N > FMM_NOALLOC_MAX_N || nt > FMM_NOALLOC_MAX_N) {
        snprintf(msg, sizeof(msg), "fmm_direct_noalloc: N = %lld, n_targets = %lld exceed the fixed scratch (at most %d each); use fmm_direct",
                 (long long)in->N, (long long)nt, FMM_NOALLOC_MAX_N);
        ctx_set_error(&ctx, msg);
        return FMM_EINVAL;
    }
    const bool sm = (flags & FMM_KERNEL_SOURCE_MOMENTUM) != 0;
    if (!sm && !(gamma_bar > 0.0 && isfinite(gamma_bar))) {
        ctx_set_error(&ctx, "fmm_direct_noalloc: gamma_bar must be given (> 0, finite) with the mean-gamma kernel");
        return FMM_EINVAL;
    }
    return pairs_direct_noalloc(&ctx, in, sm, gamma_bar, (flags & FMM_RAW_SUMS) ? 1 : 0, nt, tidx, Ex, Ey, Ez, Bx, By, Bz);
}

// ---------------------------------------------------------------------------------------
// whole of Alg 5.12 from host memory
// ---------------------------------------------------------------------------------------
extern "C" int fmm_field_host(const fmm_particles_t *h, const fmm_params_t *prm, double *Ex, double *Ey, double *Ez,
                              double *Bx, double *By, double *Bz, fmm_stats_t *stats,
                              fmm_alloc_fn alloc, fmm_free_fn free_, void *user, void *cuda_stream)
{
    if (check_particles(h) != FMM_OK || !prm || !Ex || !Ey || !Ez || !Bx || !By || !Bz) return FMM_EINVAL;
    if ((alloc == NULL) != (free_ == NULL)) return FMM_EINVAL;
    fmm_ctx ctx;
    ctx_init(&ctx, alloc, free_, user, cuda_stream);
    fmm_ctx *c = &ctx;
    const size_t N = (size_t)h->N, bytes = sizeof(double) * N;
    const int nin = h->q ? 7 : 6;
    double *din = (double *)ctx_alloc(c, bytes * nin);
    double *dout = (double *)ctx_alloc(c, bytes * 6);
    fmm_plan_t *plan = NULL;
    int rc = (din && dout) ? FMM_OK : FMM_ENOMEM;
    auto body = [&]() -> int {
        const double *src[7] = {h->x, h->y, h->z, h->px, h->py, h->pz, h->q};
        for (int k = 0; k < nin; ++k)
            FMM_CUDA(c, cudaMemcpyAsync(din + k * N, src[k], bytes, cudaMemcpyHostToDevice, c->stream));
        fmm_particles_t d = *h;
        d.x = din; d.y = din + N; d.z = din + 2 * N;
        d.px = din + 3 * N; d.py = din + 4 * N; d.pz = din + 5 * N;
        d.q = h->q ? din + 6 * N : NULL;
        FMM_TRY(fmm_plan_create(&plan, &d, prm, alloc, free_, user, cuda_stream));
        FMM_TRY(fmm_eval(plan, dout, dout + N, dout + 2 * N, dout + 3 * N, dout + 4 * N, dout + 5 * N));
        double *dst[6] = {Ex, Ey, Ez, Bx, By, Bz};
        for (int k = 0; k < 6; ++k)
            FMM_CUDA(c, cudaMemcpyAsync(dst[k], dout + k * N, bytes, cudaMemcpyDeviceToHost, c->stream));
        FMM_CUDA(c, cudaStreamSynchronize(c->stream));
        if (stats) FMM_TRY(fmm_plan_stats(plan, stats));
        return FMM_OK;
    };
    if (rc == FMM_OK) rc = body();
    if (plan) fmm_plan_destroy(plan);
    cudaStreamSynchronize(c->stream);
    ctx_free_all(c);
    return rc;
}
