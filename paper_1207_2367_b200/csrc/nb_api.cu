// nb_api.cu -- the C-ABI of include/nb.h: argument checking, call-order state machine, buffer
// ownership and host<->device marshalling.  Every step of the path runs in the kernels of
// nb_force.cu / nb_step.cu / nb_energy.cu; nothing here computes on the host.
#include <math.h>
#include <new>
#include <string.h>

#include "nb_internal.cuh"

using namespace nb;

static double bits_to_double(long long b)
{
    double d;
    memcpy(&d, &b, sizeof(d));
    return d;
}

static bool is_pow2(double x)
{
    int e;
    return x > 0.0 && isfinite(x) && frexp(x, &e) == 0.5;
}

template <typename T>
static int dev_alloc(nb_ctx *ctx, T **p, size_t count, bool zero = true)
{
    NB_CUDA(ctx, cudaMalloc((void **)p, count * sizeof(T)));
    if (zero) NB_CUDA(ctx, cudaMemsetAsync(*p, 0, count * sizeof(T), ctx->stream));
    return NB_OK;
}

static void release(nb_ctx *ctx)
{
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    graph_release(ctx);
    gridres_release(ctx);
    if (ctx->h_ctl) cudaFreeHost(ctx->h_ctl);
    if (ctx->ctl) cudaFree(ctx->ctl);
    if (ctx->geom_cache) cudaFree(ctx->geom_cache);
    void *bufs[] = {ctx->mass, ctx->t, ctx->dt, ctx->r, ctx->v, ctx->a, ctx->j, ctx->s, ctx->c, ctx->jp,
                    ctx->active, ctx->user_idx, ctx->f1, ctx->stage, ctx->partials, ctx->d_tmin,
                    ctx->blk_count, ctx->red};
    for (void *b : bufs)
        if (b) cudaFree(b);
    if (ctx->h_sched) cudaFreeHost(ctx->h_sched);
    if (ctx->h_dbg) cudaFreeHost(ctx->h_dbg);
    delete ctx;
}

extern "C" const char *nb_version(void) { return "nb-b200 0.3 (sm_100a)"; }

extern "C" const char *nb_last_error(const nb_ctx *ctx) { return ctx ? ctx->err : "null context"; }

extern "C" void nb_free(nb_ctx *ctx) { release(ctx); }

#define NB_TRY(expr)                  \
    do {                              \
        const int rc_ = (expr);       \
        if (rc_ != NB_OK) return rc_; \
    } while (0)

// copy n doubles/ints from a [dev|host] pointer into a device buffer
static int copy_in(nb_ctx *ctx, void *dst_dev, const void *src, size_t bytes)
{
    NB_CUDA(ctx, cudaMemcpyAsync(dst_dev, src, bytes, cudaMemcpyDefault, ctx->stream));
    return NB_OK;
}
static int copy_out(nb_ctx *ctx, void *dst, const void *src_dev, size_t bytes)
{
    NB_CUDA(ctx, cudaMemcpyAsync(dst, src_dev, bytes, cudaMemcpyDefault, ctx->stream));
    return NB_OK;
}

// The staging buffer grows on demand: [n][3] copies need 9 n doubles, nb_get_derivs 12 Npad, a
// checkpoint 21 Npad.  Growing synchronises the stream (pending copies still use the old buffer).
int nb::reserve_stage(nb_ctx *ctx, size_t doubles)
{
    if (doubles <= ctx->stage_cap) return NB_OK;
    if (ctx->stage) { NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream)); cudaFree(ctx->stage); }
    ctx->stage = nullptr; ctx->stage_cap = 0;
    NB_CUDA(ctx, cudaMalloc((void **)&ctx->stage, doubles * sizeof(double)));
    ctx->stage_cap = doubles;
    return NB_OK;
}

static bool sliced(const nb_ctx *ctx) { return ctx->j_begin != 0 || ctx->j_end != ctx->N; }

extern "C" int nb_init(nb_ctx **out, int64_t N, const double *pos, const double *vel, const double *mass,
                       double eps, double eta, void *cuda_stream)
{
    if (!out) return NB_EINVAL;
    *out = nullptr;
    if (N < 1 || N > (int64_t)1 << 30 || !pos || !vel || !mass || !(eps >= 0.0) || !(eta > 0.0) || !isfinite(eps) ||
        !isfinite(eta))
        return NB_EINVAL;
    if (eps > 0.0 && !(eps * eps >= 2.2250738585072014e-308)) return NB_EINVAL;  // eps^2 must be normal
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return NB_ECUDA;  // no CPU fallback: without a device there is no library
    }
    nb_ctx *ctx = new (std::nothrow) nb_ctx();
    if (!ctx) return NB_ENOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->N = N;
    ctx->Npad = (N + TILE_ALIGN - 1) / TILE_ALIGN * TILE_ALIGN;
    ctx->eps = eps; ctx->eps2 = eps * eps; ctx->eta = eta; ctx->eta_init = 0.01;
    ctx->dt_min = ldexp(1.0, -25);
    ctx->dt_max = ldexp(1.0, -3);
    ctx->stream = (cudaStream_t)cuda_stream;
    int rc = NB_OK;
    auto fail = [&](int code) { release(ctx); return code; };
    if (cudaGetDevice(&ctx->device) != cudaSuccess) return fail(NB_ECUDA);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, ctx->device) != cudaSuccess) return fail(NB_ECUDA);
    if (prop.major < 10) return fail(NB_ECUDA);  // built for sm_100a only
    ctx->n_sm = prop.multiProcessorCount;

    const size_t P = (size_t)ctx->Npad;
    if ((rc = dev_alloc(ctx, &ctx->mass, P)) || (rc = dev_alloc(ctx, &ctx->t, P)) || (rc = dev_alloc(ctx, &ctx->dt, P)) ||
        (rc = dev_alloc(ctx, &ctx->r, 3 * P)) || (rc = dev_alloc(ctx, &ctx->v, 3 * P)) ||
        (rc = dev_alloc(ctx, &ctx->a, 3 * P)) || (rc = dev_alloc(ctx, &ctx->j, 3 * P)) ||
        (rc = dev_alloc(ctx, &ctx->s, 3 * P)) || (rc = dev_alloc(ctx, &ctx->c, 3 * P)) ||
        (rc = dev_alloc(ctx, &ctx->jp, REC * P)) || (rc = dev_alloc(ctx, &ctx->active, P)) ||
        (rc = dev_alloc(ctx, &ctx->user_idx, P)) || (rc = dev_alloc(ctx, &ctx->f1, 9 * P)) ||
        (rc = reserve_stage(ctx, 12 * P)) || (rc = dev_alloc(ctx, &ctx->d_tmin, 2)))
        return fail(rc);
    ctx->n_sched_blocks = (N + 2047) / 2048;
    if ((rc = dev_alloc(ctx, &ctx->blk_count, (size_t)ctx->n_sched_blocks + 1)) ||
        (rc = dev_alloc(ctx, &ctx->red, ((size_t)(N + 127) / 128 + 2) * 9)))
        return fail(rc);
    if (cudaHostAlloc((void **)&ctx->h_sched, sizeof(Sched), cudaHostAllocMapped) != cudaSuccess) return fail(NB_ENOMEM);
    if (cudaHostGetDevicePointer((void **)&ctx->d_sched, ctx->h_sched, 0) != cudaSuccess) return fail(NB_ECUDA);
    ctx->h_sched->t_next = 0.0; ctx->h_sched->n_active = 0;
    if (cudaHostAlloc((void **)&ctx->h_dbg, 2 * sizeof(int32_t), cudaHostAllocMapped) != cudaSuccess) return fail(NB_ENOMEM);
    if (cudaHostGetDevicePointer((void **)&ctx->d_dbg, ctx->h_dbg, 0) != cudaSuccess) return fail(NB_ECUDA);
    if ((rc = dev_alloc(ctx, &ctx->ctl, 1)) || (rc = dev_alloc(ctx, &ctx->geom_cache, (size_t)GEOM_CACHE_M + 1)))
        return fail(rc);
    if (cudaHostAlloc((void **)&ctx->h_ctl, sizeof(StepCtl), cudaHostAllocDefault) != cudaSuccess) return fail(NB_ENOMEM);
    memset(ctx->h_ctl, 0, sizeof(StepCtl));
    ctx->use_graph = N <= RES_AUTO_N ? 3 : (gridres_fits(ctx) ? 4 : 1);
    ctx->loop_auto = true;
    ctx->j_begin = 0; ctx->j_end = N;
    if ((rc = query_force_occupancy(ctx))) return fail(rc);

    // stage the caller's arrays on the device ([N][3] | [N][3] | [N]) and build the SoA state
    double *st = ctx->stage;
    if ((rc = copy_in(ctx, st, pos, 3 * (size_t)N * sizeof(double))) ||
        (rc = copy_in(ctx, st + 3 * P, vel, 3 * (size_t)N * sizeof(double))) ||
        (rc = copy_in(ctx, st + 6 * P, mass, (size_t)N * sizeof(double))) ||
        (rc = launch_load_state(ctx, st, st + 3 * P, st + 6 * P)))
        return fail(rc);
    if (cudaStreamSynchronize(ctx->stream) != cudaSuccess) return fail(NB_ECUDA);
    ctx->pred_valid = true; ctx->t_pred = 0.0; ctx->t_now = 0.0;
    *out = ctx;
    return NB_OK;
}

extern "C" int nb_set_limits(nb_ctx *ctx, double dt_min, double dt_max, double eta_init)
{
    if (!ctx) return NB_EINVAL;
    if (ctx->started) return set_err(ctx, NB_ESTATE, "nb_set_limits: only before nb_startup");
    if (!is_pow2(dt_min) || !is_pow2(dt_max) || dt_min > dt_max || !(eta_init > 0.0) || !isfinite(eta_init))
        return set_err(ctx, NB_EINVAL, "nb_set_limits: limits must be powers of two with dt_min <= dt_max, eta_init > 0");
    ctx->dt_min = dt_min; ctx->dt_max = dt_max; ctx->eta_init = eta_init;
    return NB_OK;
}

extern "C" int nb_startup(nb_ctx *ctx)
{
    if (!ctx) return NB_EINVAL;
    if (ctx->started) return set_err(ctx, NB_ESTATE, "nb_startup: already started");
    if (sliced(ctx))
        return set_err(ctx, NB_ESTATE, "nb_startup: a j-slice is set (nb_set_j_range); drive the start-up call by call "
                                       "(nb_force, exchange, nb_startup_commit)");
    // a context that steps will split small active sets over many j-pieces: take the partial-sum buffer
    // now (up to 0.5 GB at large N) rather than inside the first block step
    NB_TRY(reserve_partials(ctx, ctx->partials_limit));
    // predicted stream <- (r, v, a = 0) at t = 0 (all t_i = 0, derivatives 0: the predictor is the identity)
    NB_TRY(launch_predict(ctx, 0.0));
    NB_TRY(launch_force(ctx, nullptr, ctx->N, true)); // pass 1: a, jerk only (its snap would lack the m da term)
    NB_TRY(launch_startup_commit(ctx, 1));           // a_pred <- a
    NB_TRY(launch_force(ctx, nullptr, ctx->N));      // pass 2: a, jerk, snap
    NB_TRY(launch_startup_commit(ctx, 2));           // commit, crackle = 0, initial dt
    ctx->started = true; ctx->pred_valid = true; ctx->t_pred = 0.0; ctx->t_now = 0.0;
    ctx->have_block = false; ctx->evaluated = false; ctx->eval_partial = false;
    return NB_OK;
}

extern "C" int nb_startup_commit(nb_ctx *ctx, int pass)
{
    if (!ctx) return NB_EINVAL;
    if (ctx->started) return set_err(ctx, NB_ESTATE, "nb_startup_commit: already started");
    if (pass != 1 && pass != 2) return set_err(ctx, NB_EINVAL, "nb_startup_commit: pass is 1 or 2");
    if (ctx->n_eval != ctx->N) return set_err(ctx, NB_ESTATE, "nb_startup_commit: evaluate all N particles first (nb_force(NULL, N))");
    NB_TRY(launch_startup_commit(ctx, pass));
    if (pass == 2) {
        ctx->started = true; ctx->pred_valid = true; ctx->t_pred = 0.0; ctx->t_now = 0.0;
        ctx->have_block = false; ctx->evaluated = false; ctx->eval_partial = false;
    }
    return NB_OK;
}

extern "C" int nb_next_block(nb_ctx *ctx, double *t_next, int64_t *n_active)
{
    if (!ctx) return NB_EINVAL;
    if (!ctx->started) return set_err(ctx, NB_ESTATE, "nb_next_block: call nb_startup first");
    NB_TRY(launch_next_block(ctx));
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->t_next = ctx->h_sched->t_next;
    ctx->n_active = (int64_t)ctx->h_sched->n_active;
    ctx->have_block = true; ctx->evaluated = false; ctx->eval_partial = false;
    if (t_next) *t_next = ctx->t_next;
    if (n_active) *n_active = ctx->n_active;
    return NB_OK;
}

extern "C" int nb_get_active(nb_ctx *ctx, int32_t *idx)
{
    if (!ctx || !idx) return NB_EINVAL;
    if (!ctx->have_block) return set_err(ctx, NB_ESTATE, "nb_get_active: no block selected");
    return copy_out(ctx, idx, ctx->active, (size_t)ctx->n_active * sizeof(int32_t));
}

extern "C" int nb_predict(nb_ctx *ctx, double t)
{
    if (!ctx) return NB_EINVAL;
    if (!(t >= ctx->t_now) || !isfinite(t)) return set_err(ctx, NB_EINVAL, "nb_predict: t = %g is earlier than the current time %g", t, ctx->t_now);
    NB_TRY(launch_predict(ctx, t));
    ctx->pred_valid = true; ctx->t_pred = t; ctx->evaluated = false; ctx->eval_partial = false;
    return NB_OK;
}

extern "C" int nb_force(nb_ctx *ctx, const int32_t *active_idx, int64_t n_active, double *acc, double *jerk,
                        double *snap)
{
    if (!ctx) return NB_EINVAL;
    if (n_active < 0 || n_active > ctx->N) return set_err(ctx, NB_EINVAL, "nb_force: n_active = %lld outside [0, N]", (long long)n_active);
    if (!ctx->pred_valid) return set_err(ctx, NB_ESTATE, "nb_force: no predicted data");
    if (n_active == 0) { ctx->n_eval = 0; return NB_OK; }  // empty set: nothing to evaluate
    const int32_t *list = nullptr;
    bool sched_set = false;
    if (active_idx) {
        NB_TRY(copy_in(ctx, ctx->user_idx, active_idx, (size_t)n_active * sizeof(int32_t)));
        list = ctx->user_idx;
        if (ctx->debug) {
            NB_TRY(launch_check_indices(ctx, list, n_active));
            if (ctx->h_dbg[0] > 0)
                return set_err(ctx, NB_EINVAL, "nb_force: %d of the %lld entries of active_idx are outside [0, %lld); first at slot %d",
                               (int)ctx->h_dbg[0], (long long)n_active, (long long)ctx->N, (int)ctx->h_dbg[1]);
        }
    } else if (n_active == ctx->N) {
        list = nullptr;  // all particles, index order
        sched_set = ctx->have_block && ctx->n_active == ctx->N;
    } else {
        if (!ctx->have_block || n_active != ctx->n_active)
            return set_err(ctx, NB_ESTATE, "nb_force: active_idx is NULL but n_active = %lld is not the scheduler's %lld",
                           (long long)n_active, (long long)(ctx->have_block ? ctx->n_active : -1));
        list = ctx->active;
        sched_set = true;
    }
    NB_TRY(launch_force(ctx, list, n_active));
    ctx->n_eval = n_active;
    // over a proper j-slice these are partial sums: the corrector must not run on them (nb_set_forces)
    const bool block_eval = sched_set && ctx->t_pred == ctx->t_next;
    ctx->evaluated = block_eval && !sliced(ctx);
    ctx->eval_partial = block_eval && sliced(ctx);
    if ((acc || jerk || snap) && n_active > 0) {
        NB_TRY(reserve_stage(ctx, 9 * (size_t)n_active));
        NB_TRY(launch_unpack_f1(ctx, n_active));
        const size_t bytes = 3 * (size_t)n_active * sizeof(double);
        if (acc) NB_TRY(copy_out(ctx, acc, ctx->stage, bytes));
        if (jerk) NB_TRY(copy_out(ctx, jerk, ctx->stage + 3 * n_active, bytes));
        if (snap) NB_TRY(copy_out(ctx, snap, ctx->stage + 6 * n_active, bytes));
    }
    return NB_OK;
}

extern "C" int nb_correct_and_step(nb_ctx *ctx)
{
    if (!ctx) return NB_EINVAL;
    if (ctx->have_block && ctx->eval_partial)
        return set_err(ctx, NB_ESTATE, "nb_correct_and_step: the evaluated values are j-slice partials (nb_set_j_range); "
                                       "all-reduce nb_get_forces and store the sums with nb_set_forces first");
    if (!ctx->have_block || !ctx->evaluated)
        return set_err(ctx, NB_ESTATE, "nb_correct_and_step: needs nb_next_block, nb_predict(t_next) and nb_force on the scheduler's set");
    const int64_t m = ctx->n_active;
    NB_TRY(launch_correct(ctx, m == ctx->N ? nullptr : ctx->active, m, ctx->t_next));
    ctx->t_now = ctx->t_next;
    ctx->have_block = false; ctx->evaluated = false; ctx->eval_partial = false;
    ctx->n_steps += 1;
    int b = 0;
    while ((((int64_t)1) << (b + 1)) <= m) ++b;
    ctx->hist[b] += 1;
    return NB_OK;
}

static int one_block_step(nb_ctx *ctx)
{
    NB_TRY(launch_predict(ctx, ctx->t_next));
    ctx->pred_valid = true; ctx->t_pred = ctx->t_next;
    NB_TRY(launch_force(ctx, ctx->n_active == ctx->N ? nullptr : ctx->active, ctx->n_active));
    ctx->n_eval = ctx->n_active; ctx->evaluated = true;
    return nb_correct_and_step(ctx);
}

int nb::host_block_step(nb_ctx *ctx, double t_end, bool *stepped)
{
    *stepped = false;
    if (!ctx->have_block) NB_TRY(nb_next_block(ctx, nullptr, nullptr));
    if (ctx->t_next > t_end) return NB_OK;
    NB_TRY(one_block_step(ctx));
    *stepped = true;
    return NB_OK;
}

extern "C" int nb_run_until(nb_ctx *ctx, double t_end, int64_t *n_steps)
{
    if (!ctx) return NB_EINVAL;
    if (!isfinite(t_end)) return set_err(ctx, NB_EINVAL, "nb_run_until: bad t_end");
    if (sliced(ctx))   // before the implicit start-up: a refused call leaves the context untouched
        return set_err(ctx, NB_ESTATE, "nb_run_until: a j-shard is set (nb_set_j_range); drive the steps call by call and all-reduce nb_get_forces");
    if (!ctx->started) NB_TRY(nb_startup(ctx));
    if (ctx->use_graph == 3) return resident_run(ctx, t_end, INT64_MAX, n_steps);
    if (ctx->use_graph == 4) return gridres_run(ctx, t_end, INT64_MAX, n_steps);
    if (ctx->use_graph) return graph_run(ctx, t_end, INT64_MAX, n_steps);
    int64_t n = 0;
    for (;;) {
        if (!ctx->have_block) NB_TRY(nb_next_block(ctx, nullptr, nullptr));
        if (ctx->t_next > t_end) break;
        NB_TRY(one_block_step(ctx));
        ++n;
    }
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (n_steps) *n_steps = n;
    return NB_OK;
}

extern "C" int nb_run_steps(nb_ctx *ctx, int64_t n, double *log_t, int64_t *log_m, float *log_ms)
{
    if (!ctx || n < 0) return NB_EINVAL;
    if (sliced(ctx)) return set_err(ctx, NB_ESTATE, "nb_run_steps: a j-shard is set (nb_set_j_range)");
    if (!ctx->started) NB_TRY(nb_startup(ctx));
    if (ctx->use_graph && !log_t && !log_m && !log_ms) {
        if (n == 0) return NB_OK;
        if (ctx->use_graph == 3) return resident_run(ctx, bits_to_double(0x7fefffffffffffffLL), n, nullptr);
        if (ctx->use_graph == 4) return gridres_run(ctx, bits_to_double(0x7fefffffffffffffLL), n, nullptr);
        return graph_run(ctx, bits_to_double(0x7fefffffffffffffLL), n, nullptr);
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (log_ms) {
        NB_CUDA(ctx, cudaEventCreate(&e0));
        NB_CUDA(ctx, cudaEventCreate(&e1));
    }
    int rc = NB_OK;
    for (int64_t k = 0; k < n && rc == NB_OK; ++k) {
        if (log_ms) cudaEventRecord(e0, ctx->stream);
        if (!ctx->have_block) rc = nb_next_block(ctx, nullptr, nullptr);
        if (rc != NB_OK) break;
        const double tn = ctx->t_next;
        const int64_t m = ctx->n_active;
        rc = one_block_step(ctx);
        if (rc != NB_OK) break;
        if (log_t) log_t[k] = tn;
        if (log_m) log_m[k] = m;
        if (log_ms) {
            cudaEventRecord(e1, ctx->stream);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = set_err(ctx, NB_ECUDA, "nb_run_steps: event sync failed"); break; }
            cudaEventElapsedTime(&log_ms[k], e0, e1);
        }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (rc != NB_OK) return rc;
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return NB_OK;
}

extern "C" int nb_energy(nb_ctx *ctx, double out[9])
{
    if (!ctx || !out) return NB_EINVAL;
    // positions and velocities of every particle at the current time (the predictor is the identity
    // for particles already there, h = 0), written to a scratch copy of the record stream so that the
    // predicted data nb_force reads stay what the caller last set or predicted
    const size_t P = (size_t)ctx->Npad, N = (size_t)ctx->N;
    NB_TRY(reserve_stage(ctx, REC * P));
    NB_TRY(launch_predict(ctx, ctx->t_now, ctx->stage));
    if (P > N) NB_CUDA(ctx, cudaMemsetAsync(ctx->stage + REC * N, 0, REC * (P - N) * sizeof(double), ctx->stream));
    return launch_energy(ctx, ctx->stage, out);
}

extern "C" int nb_get_state(nb_ctx *ctx, double *pos, double *vel, double *t, double *dt)
{
    if (!ctx) return NB_EINVAL;
    const size_t P = (size_t)ctx->Npad, N = (size_t)ctx->N;
    NB_TRY(reserve_stage(ctx, 6 * P));
    if (pos) { NB_TRY(launch_pack3(ctx, ctx->r, ctx->stage)); NB_TRY(copy_out(ctx, pos, ctx->stage, 3 * N * sizeof(double))); }
    if (vel) { NB_TRY(launch_pack3(ctx, ctx->v, ctx->stage + 3 * P)); NB_TRY(copy_out(ctx, vel, ctx->stage + 3 * P, 3 * N * sizeof(double))); }
    if (t) NB_TRY(copy_out(ctx, t, ctx->t, N * sizeof(double)));
    if (dt) NB_TRY(copy_out(ctx, dt, ctx->dt, N * sizeof(double)));
    return NB_OK;
}

extern "C" int nb_get_derivs(nb_ctx *ctx, double *acc, double *jerk, double *snap, double *crackle)
{
    if (!ctx) return NB_EINVAL;
    const size_t P = (size_t)ctx->Npad, N = (size_t)ctx->N;
    double *dst[4] = {acc, jerk, snap, crackle};
    const double *src[4] = {ctx->a, ctx->j, ctx->s, ctx->c};
    NB_TRY(reserve_stage(ctx, 12 * P));
    for (int q = 0; q < 4; ++q)
        if (dst[q]) {
            NB_TRY(launch_pack3(ctx, src[q], ctx->stage + 3 * P * q));
            NB_TRY(copy_out(ctx, dst[q], ctx->stage + 3 * P * q, 3 * N * sizeof(double)));
        }
    return NB_OK;
}

extern "C" int nb_get_pred(nb_ctx *ctx, double *pos, double *vel, double *acc)
{
    if (!ctx) return NB_EINVAL;
    if (!ctx->pred_valid) return set_err(ctx, NB_ESTATE, "nb_get_pred: no predicted data");
    const size_t P = (size_t)ctx->Npad, N = (size_t)ctx->N;
    NB_TRY(reserve_stage(ctx, 9 * P));
    NB_TRY(launch_get_pred(ctx, ctx->stage, ctx->stage + 3 * P, ctx->stage + 6 * P));
    if (pos) NB_TRY(copy_out(ctx, pos, ctx->stage, 3 * N * sizeof(double)));
    if (vel) NB_TRY(copy_out(ctx, vel, ctx->stage + 3 * P, 3 * N * sizeof(double)));
    if (acc) NB_TRY(copy_out(ctx, acc, ctx->stage + 6 * P, 3 * N * sizeof(double)));
    return NB_OK;
}

extern "C" int nb_set_pred_acc(nb_ctx *ctx, const double *acc_pred)
{
    if (!ctx || !acc_pred) return NB_EINVAL;
    if (!ctx->pred_valid) return set_err(ctx, NB_ESTATE, "nb_set_pred_acc: no predicted data");
    NB_TRY(reserve_stage(ctx, 3 * (size_t)ctx->Npad));
    NB_TRY(copy_in(ctx, ctx->stage, acc_pred, 3 * (size_t)ctx->N * sizeof(double)));
    NB_TRY(launch_set_pred(ctx, nullptr, nullptr, ctx->stage, false, true));
    ctx->evaluated = false; ctx->eval_partial = false;
    return NB_OK;
}

extern "C" int nb_set_pred(nb_ctx *ctx, const double *pos, const double *vel, const double *acc)
{
    if (!ctx || !pos || !vel) return NB_EINVAL;
    const size_t P = (size_t)ctx->Npad, N = (size_t)ctx->N;
    NB_TRY(reserve_stage(ctx, 9 * P));
    NB_TRY(copy_in(ctx, ctx->stage, pos, 3 * N * sizeof(double)));
    NB_TRY(copy_in(ctx, ctx->stage + 3 * P, vel, 3 * N * sizeof(double)));
    if (acc) NB_TRY(copy_in(ctx, ctx->stage + 6 * P, acc, 3 * N * sizeof(double)));
    NB_TRY(launch_set_pred(ctx, ctx->stage, ctx->stage + 3 * P, ctx->stage + 6 * P, true, acc != nullptr));
    ctx->pred_valid = true; ctx->evaluated = false; ctx->eval_partial = false;
    return NB_OK;
}

extern "C" int nb_get_full_state(nb_ctx *ctx, double *state)
{
    if (!ctx || !state) return NB_EINVAL;
    NB_TRY(reserve_stage(ctx, 21 * (size_t)ctx->Npad));
    NB_TRY(launch_full_state(ctx, ctx->stage, false));
    return copy_out(ctx, state, ctx->stage, 21 * (size_t)ctx->N * sizeof(double));
}

extern "C" int nb_set_full_state(nb_ctx *ctx, const double *state)
{
    if (!ctx || !state) return NB_EINVAL;
    NB_TRY(reserve_stage(ctx, 21 * (size_t)ctx->Npad));
    NB_TRY(copy_in(ctx, ctx->stage, state, 21 * (size_t)ctx->N * sizeof(double)));
    NB_TRY(launch_full_state(ctx, ctx->stage, true));
    NB_TRY(launch_tmax(ctx));
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->t_now = ctx->h_sched->t_next;
    ctx->started = true; ctx->have_block = false; ctx->evaluated = false; ctx->eval_partial = false; ctx->pred_valid = false;
    return NB_OK;
}

extern "C" int nb_get_stats(nb_ctx *ctx, double out[4], int64_t hist[64])
{
    if (!ctx) return NB_EINVAL;
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (out) { out[0] = (double)ctx->n_steps; out[1] = ctx->n_pairs; out[2] = (double)ctx->n_launch; out[3] = ctx->t_now; }
    if (hist) memcpy(hist, ctx->hist, sizeof(ctx->hist));
    return NB_OK;
}

extern "C" int nb_set_tuning(nb_ctx *ctx, int split, int jlanes)
{
    if (!ctx) return NB_EINVAL;
    if (split < 0 || jlanes < 0 || jlanes > 32 || (jlanes & (jlanes - 1)))
        return set_err(ctx, NB_EINVAL, "nb_set_tuning: split >= 0, jlanes in {0,1,2,4,8,16,32}");
    ctx->force_split = split; ctx->force_jlanes = jlanes;
    return NB_OK;
}

extern "C" int nb_set_j_range(nb_ctx *ctx, int64_t j_begin, int64_t j_end)
{
    if (!ctx) return NB_EINVAL;
    if (j_begin < 0 || j_end > ctx->N || j_begin >= j_end || (j_begin % TILE_ALIGN) != 0 ||
        (j_end != ctx->N && (j_end % TILE_ALIGN) != 0))
        return set_err(ctx, NB_EINVAL, "nb_set_j_range: need 0 <= j_begin < j_end <= N, both multiples of %d (j_end may be N)", TILE_ALIGN);
    ctx->j_begin = j_begin; ctx->j_end = j_end;
    ctx->evaluated = false; ctx->eval_partial = false;
    return NB_OK;
}

extern "C" int nb_get_forces(nb_ctx *ctx, double *buf)
{
    if (!ctx || !buf) return NB_EINVAL;
    if (ctx->n_eval <= 0) return set_err(ctx, NB_ESTATE, "nb_get_forces: nothing evaluated");
    NB_TRY(reserve_stage(ctx, 9 * (size_t)ctx->n_eval));
    NB_TRY(launch_f1_contig(ctx, ctx->n_eval, ctx->stage, false));
    return copy_out(ctx, buf, ctx->stage, 9 * (size_t)ctx->n_eval * sizeof(double));
}

extern "C" int nb_set_forces(nb_ctx *ctx, const double *buf)
{
    if (!ctx || !buf) return NB_EINVAL;
    if (ctx->n_eval <= 0) return set_err(ctx, NB_ESTATE, "nb_set_forces: nothing evaluated");
    NB_TRY(reserve_stage(ctx, 9 * (size_t)ctx->n_eval));
    NB_TRY(copy_in(ctx, ctx->stage, buf, 9 * (size_t)ctx->n_eval * sizeof(double)));
    NB_TRY(launch_f1_contig(ctx, ctx->n_eval, ctx->stage, true));
    // the caller stores the sums over all j-slices: the set just evaluated is now complete
    if (ctx->eval_partial) { ctx->evaluated = true; ctx->eval_partial = false; }
    return NB_OK;
}

extern "C" int nb_set_precision(nb_ctx *ctx, int mode)
{
    if (!ctx) return NB_EINVAL;
    if (mode < 0 || mode > 2)
        return set_err(ctx, NB_EINVAL, "nb_set_precision: 0 (FP64), 1 (mixed SP/DP) or 2 (mixed, acceleration and jerk summed in double)");
    ctx->precision = mode;
    ctx->evaluated = false; ctx->eval_partial = false;
    return NB_OK;
}

extern "C" int nb_set_loop_mode(nb_ctx *ctx, int device_driven)
{
    if (!ctx) return NB_EINVAL;
    if (device_driven < 0 || device_driven > 4) return set_err(ctx, NB_EINVAL, "nb_set_loop_mode: 0, 1, 2, 3 or 4");
    if (device_driven == 4 && !gridres_fits(ctx))
        return set_err(ctx, NB_EINVAL, "nb_set_loop_mode: mode 4 (grid-resident loop) does not hold N = %lld in the shared memory of this device", (long long)ctx->N);
    if (device_driven == 3 && ctx->N > RES_MAX_N)
        return set_err(ctx, NB_EINVAL, "nb_set_loop_mode: mode 3 (cluster-resident loop) serves N <= %lld", (long long)RES_MAX_N);
    ctx->use_graph = device_driven;
    ctx->loop_auto = false;
    return NB_OK;
}

extern "C" int nb_get_loop_mode(nb_ctx *ctx, int *mode)
{
    if (!ctx || !mode) return NB_EINVAL;
    *mode = ctx->use_graph;
    return NB_OK;
}

extern "C" int nb_get_launch(nb_ctx *ctx, int64_t out[5])
{
    if (!ctx || !out) return NB_EINVAL;
    memcpy(out, ctx->last_launch, sizeof(ctx->last_launch));
    return NB_OK;
}

extern "C" int nb_probe_fp64_peak(nb_ctx *ctx, int64_t iters, double *flops, float *ms)
{
    if (!ctx || iters < 1) return NB_EINVAL;
    return launch_probe(ctx, iters, flops, ms);
}

extern "C" int nb_set_debug(nb_ctx *ctx, int on)
{
    if (!ctx) return NB_EINVAL;
    ctx->debug = on ? 1 : 0;
    return NB_OK;
}
