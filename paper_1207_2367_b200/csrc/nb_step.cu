// nb_step.cu -- the O(N) and O(m) kernels around the evaluation step:
//   predictor            Eq. 3-7      k_predict
//   next block / gather  Table 1 row 1    k_tmin, k_count_scan, k_scatter
//   corrector            Eq. 11-14      k_correct
//   new time step        Eq. 15-16     new_dt() inside k_correct
//   start-up             DESIGN.md reading G8            k_startup_commit
// All of them stream the SoA state once; they are HBM- or latency-bound.
#include "nb_internal.cuh"
#include "nb_force_dev.cuh"
#include "nb_step_dev.cuh"

namespace nb {

// ---------------------------------------------------------------------------------------
// load: caller layout [N][3] -> SoA planes, predicted records {r, v, 0, m}; t = dt = 0
__global__ void k_load_state(const int64_t N, const int64_t Npad, const double *__restrict__ pos,
                             const double *__restrict__ vel, const double *__restrict__ mass_in,
                             double *__restrict__ r, double *__restrict__ v, double *__restrict__ mass,
                             double *__restrict__ jp)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
    const double vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
    const double m = mass_in[i];
    r[i] = x; r[Npad + i] = y; r[2 * Npad + i] = z;
    v[i] = vx; v[Npad + i] = vy; v[2 * Npad + i] = vz;
    mass[i] = m;
    double2 *rec = reinterpret_cast<double2 *>(jp + i * REC);
    rec[0] = make_double2(x, y);
    rec[1] = make_double2(z, vx);
    rec[2] = make_double2(vy, vz);
    rec[3] = make_double2(0.0, 0.0);
    rec[4] = make_double2(0.0, m);
}

int launch_load_state(nb_ctx *ctx, const double *pos, const double *vel, const double *mass_in)
{
    const int64_t N = ctx->N;
    k_load_state<<<(unsigned)((N + 255) / 256), 256, 0, ctx->stream>>>(N, ctx->Npad, pos, vel, mass_in, ctx->r,
                                                                       ctx->v, ctx->mass, ctx->jp);
    NB_LAUNCH_CHECK(ctx, "k_load_state");
    return NB_OK;
}

__global__ void k_predict(const int64_t N, const int64_t Npad, const double t,
                          const double *__restrict__ ti, const double *__restrict__ mass,
                          const double *__restrict__ r, const double *__restrict__ v,
                          const double *__restrict__ a, const double *__restrict__ j,
                          const double *__restrict__ s, const double *__restrict__ c,
                          double *__restrict__ jp)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    predict_one(i, Npad, t, ti, mass, r, v, a, j, s, c, jp);
}

int launch_predict(nb_ctx *ctx, double t, double *records)
{
    const int64_t N = ctx->N;
    k_predict<<<(unsigned)((N + 255) / 256), 256, 0, ctx->stream>>>(N, ctx->Npad, t, ctx->t, ctx->mass, ctx->r,
                                                                    ctx->v, ctx->a, ctx->j, ctx->s, ctx->c,
                                                                    records ? records : ctx->jp);
    NB_LAUNCH_CHECK(ctx, "k_predict");
    return NB_OK;
}

// overwrite predicted data from caller-layout arrays (force-only use)
__global__ void k_set_pred(const int64_t N, const double *__restrict__ pos, const double *__restrict__ vel,
                           const double *__restrict__ acc, const bool pos_vel, const bool acc_valid,
                           double *__restrict__ jp)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    double *rec = jp + i * REC;
    if (pos_vel) {
#pragma unroll
        for (int d = 0; d < 3; ++d) { rec[d] = pos[3 * i + d]; rec[3 + d] = vel[3 * i + d]; }
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) rec[6 + d] = acc_valid ? acc[3 * i + d] : 0.0;
}

int launch_set_pred(nb_ctx *ctx, const double *pos, const double *vel, const double *acc, bool pos_vel,
                    bool acc_valid)
{
    const int64_t N = ctx->N;
    k_set_pred<<<(unsigned)((N + 255) / 256), 256, 0, ctx->stream>>>(N, pos, vel, acc, pos_vel, acc_valid, ctx->jp);
    NB_LAUNCH_CHECK(ctx, "k_set_pred");
    return NB_OK;
}

__global__ void k_get_pred(const int64_t N, const double *__restrict__ jp, double *__restrict__ pos,
                           double *__restrict__ vel, double *__restrict__ acc)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double *rec = jp + i * REC;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        pos[3 * i + d] = rec[d];
        vel[3 * i + d] = rec[3 + d];
        acc[3 * i + d] = rec[6 + d];
    }
}

int launch_get_pred(nb_ctx *ctx, double *pos, double *vel, double *acc)
{
    const int64_t N = ctx->N;
    k_get_pred<<<(unsigned)((N + 255) / 256), 256, 0, ctx->stream>>>(N, ctx->jp, pos, vel, acc);
    NB_LAUNCH_CHECK(ctx, "k_get_pred");
    return NB_OK;
}

__global__ void k_pack3(const int64_t N, const int64_t Npad, const double *__restrict__ soa,
                        double *__restrict__ aos)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    aos[3 * i] = soa[i];
    aos[3 * i + 1] = soa[Npad + i];
    aos[3 * i + 2] = soa[2 * Npad + i];
}

int launch_pack3(nb_ctx *ctx, const double *soa, double *aos)
{
    const int64_t N = ctx->N;
    k_pack3<<<(unsigned)((N + 255) / 256), 256, 0, ctx->stream>>>(N, ctx->Npad, soa, aos);
    NB_LAUNCH_CHECK(ctx, "k_pack3");
    return NB_OK;
}

// ---------------------------------------------------------------------------------------
// Debug range check of a caller-supplied index list (nb_set_debug): dbg = {number of entries outside
// [0, N), smallest offending slot}, in pinned mapped memory.
__global__ void k_check_indices(const int32_t *__restrict__ idx, const int64_t m, const int64_t N, int32_t *dbg)
{
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (int64_t)gridDim.x * blockDim.x) {
        const int32_t v = idx[k];
        if (v < 0 || (int64_t)v >= N) {
            atomicAdd(&dbg[0], 1);
            atomicMin(&dbg[1], (int32_t)k);
        }
    }
}

int launch_check_indices(nb_ctx *ctx, const int32_t *idx, int64_t m)
{
    ctx->h_dbg[0] = 0; ctx->h_dbg[1] = INT_MAX;
    int64_t g = (m + 255) / 256;
    if (g > 4 * ctx->n_sm) g = 4 * ctx->n_sm;
    k_check_indices<<<(unsigned)g, 256, 0, ctx->stream>>>(idx, m, ctx->N, ctx->d_dbg);
    NB_LAUNCH_CHECK(ctx, "k_check_indices");
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return NB_OK;
}

// ---------------------------------------------------------------------------------------
// Next block (Table 1 row 1).  Times are non-negative dyadic rationals, so
// t_i + dt_i is exact, equality is well defined, and the bit pattern of a non-negative double
// orders like the value: the minimum is an atomicMin on its 64-bit pattern.
__global__ void k_tmin(const int64_t N, const double *__restrict__ t, const double *__restrict__ dt,
                       unsigned long long *__restrict__ tmin_bits)
{
    double v = __longlong_as_double(0x7ff0000000000000LL);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
        v = fmin(v, t[i] + dt[i]);
    for (int off = 16; off > 0; off >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, off));
    __shared__ double sm[SCHED_THREADS / 32];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < SCHED_THREADS / 32 ? sm[threadIdx.x] : __longlong_as_double(0x7ff0000000000000LL);
        for (int off = 16; off > 0; off >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, off));
        if (threadIdx.x == 0) atomicMin(tmin_bits, (unsigned long long)__double_as_longlong(v));
    }
}

__device__ __forceinline__ int block_exclusive_scan(int v, int *total)
{
    // exclusive scan of one int per thread over a SCHED_THREADS-thread block
    __shared__ int warp_sum[SCHED_THREADS / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int incl = v;
    for (int off = 1; off < 32; off <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += n;
    }
    if (lane == 31) warp_sum[w] = incl;
    __syncthreads();
    if (w == 0) {
        int ws = lane < SCHED_THREADS / 32 ? warp_sum[lane] : 0;
        for (int off = 1; off < 32; off <<= 1) {
            const int n = __shfl_up_sync(0xffffffffu, ws, off);
            if (lane >= off) ws += n;
        }
        if (lane < SCHED_THREADS / 32) warp_sum[lane] = ws;  // inclusive over warps
    }
    __syncthreads();
    const int base = w ? warp_sum[w - 1] : 0;
    *total = warp_sum[SCHED_THREADS / 32 - 1];
    __syncthreads();
    return base + incl - v;
}

// per-block match counts; the last block to finish turns them into exclusive offsets and
// publishes (t_next, n_active) to the pinned host mirror
__global__ void __launch_bounds__(SCHED_THREADS)
    k_count_scan(const int64_t N, const double *__restrict__ t, const double *__restrict__ dt,
                 const unsigned long long *__restrict__ tmin_bits, int32_t *__restrict__ blk_count,
                 unsigned int *__restrict__ ticket, Sched *__restrict__ sched)
{
    const double tn = __longlong_as_double((long long)*tmin_bits);
    const int64_t base = (int64_t)blockIdx.x * SCHED_BLOCK + (int64_t)threadIdx.x * SCHED_ITEMS;
    int cnt = 0;
#pragma unroll
    for (int u = 0; u < SCHED_ITEMS; ++u) {
        const int64_t i = base + u;
        if (i < N && t[i] + dt[i] == tn) ++cnt;
    }
    int total;
    block_exclusive_scan(cnt, &total);
    __shared__ bool last;
    if (threadIdx.x == 0) {
        blk_count[blockIdx.x] = total;
        __threadfence();
        const unsigned int tk = atomicAdd(ticket, 1u);
        last = (tk == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    // exclusive scan of gridDim.x counts by this block, in chunks of SCHED_THREADS
    int carry = 0;
    for (int b0 = 0; b0 < (int)gridDim.x; b0 += SCHED_THREADS) {
        const int b = b0 + threadIdx.x;
        const int v = b < (int)gridDim.x ? ((volatile int32_t *)blk_count)[b] : 0;
        int tot;
        const int ex = block_exclusive_scan(v, &tot);
        if (b < (int)gridDim.x) blk_count[b] = carry + ex;
        carry += tot;
    }
    if (threadIdx.x == 0) {
        sched->t_next = tn;
        sched->n_active = carry;
        *ticket = 0;
    }
}

__global__ void __launch_bounds__(SCHED_THREADS)
    k_scatter(const int64_t N, const double *__restrict__ t, const double *__restrict__ dt,
              const unsigned long long *__restrict__ tmin_bits, const int32_t *__restrict__ blk_off,
              int32_t *__restrict__ active)
{
    const double tn = __longlong_as_double((long long)*tmin_bits);
    const int64_t base = (int64_t)blockIdx.x * SCHED_BLOCK + (int64_t)threadIdx.x * SCHED_ITEMS;
    bool hit[SCHED_ITEMS];
    int cnt = 0;
#pragma unroll
    for (int u = 0; u < SCHED_ITEMS; ++u) {
        const int64_t i = base + u;
        hit[u] = (i < N) && (t[i] + dt[i] == tn);
        cnt += hit[u] ? 1 : 0;
    }
    int total;
    int pos = blk_off[blockIdx.x] + block_exclusive_scan(cnt, &total);
#pragma unroll
    for (int u = 0; u < SCHED_ITEMS; ++u)
        if (hit[u]) active[pos++] = (int32_t)(base + u);
}

int launch_next_block(nb_ctx *ctx)
{
    const int64_t N = ctx->N;
    const int nb = (int)ctx->n_sched_blocks;
    NB_CUDA(ctx, cudaMemsetAsync(ctx->d_tmin, 0x7f, sizeof(unsigned long long), ctx->stream));
    int g = (int)((N + SCHED_THREADS - 1) / SCHED_THREADS);
    if (g > 4 * ctx->n_sm) g = 4 * ctx->n_sm;
    k_tmin<<<g, SCHED_THREADS, 0, ctx->stream>>>(N, ctx->t, ctx->dt, ctx->d_tmin);
    NB_LAUNCH_CHECK(ctx, "k_tmin");
    k_count_scan<<<nb, SCHED_THREADS, 0, ctx->stream>>>(N, ctx->t, ctx->dt, ctx->d_tmin, ctx->blk_count,
                                                        (unsigned int *)(ctx->d_tmin + 1), ctx->d_sched);
    NB_LAUNCH_CHECK(ctx, "k_count_scan");
    k_scatter<<<nb, SCHED_THREADS, 0, ctx->stream>>>(N, ctx->t, ctx->dt, ctx->d_tmin, ctx->blk_count, ctx->active);
    NB_LAUNCH_CHECK(ctx, "k_scatter");
    return NB_OK;
}

__global__ void k_tmax(const int64_t N, const double *__restrict__ t, unsigned long long *__restrict__ bits)
{
    double v = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
        v = fmax(v, t[i]);
    for (int off = 16; off > 0; off >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, off));
    if ((threadIdx.x & 31) == 0) atomicMax(bits, (unsigned long long)__double_as_longlong(v));
}
__global__ void k_publish_t(const unsigned long long *__restrict__ bits, Sched *__restrict__ sched)
{
    sched->t_next = __longlong_as_double((long long)*bits);
    sched->n_active = 0;
}

int launch_tmax(nb_ctx *ctx)
{
    NB_CUDA(ctx, cudaMemsetAsync(ctx->d_tmin, 0, sizeof(unsigned long long), ctx->stream));
    k_tmax<<<2 * ctx->n_sm, 256, 0, ctx->stream>>>(ctx->N, ctx->t, ctx->d_tmin);
    NB_LAUNCH_CHECK(ctx, "k_tmax");
    k_publish_t<<<1, 1, 0, ctx->stream>>>(ctx->d_tmin, ctx->d_sched);
    NB_LAUNCH_CHECK(ctx, "k_publish_t");
    return NB_OK;
}

__global__ void k_correct(const int m, const int64_t Npad, const int32_t *__restrict__ active,
                          const double t_next, const double eta, const double dt_min, const double dt_max,
                          const double *__restrict__ f1, double *__restrict__ ti, double *__restrict__ dti,
                          double *__restrict__ r, double *__restrict__ v, double *__restrict__ a,
                          double *__restrict__ j, double *__restrict__ s, double *__restrict__ c)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m) return;
    const int64_t i = active ? active[k] : k;
    correct_one(k, i, Npad, t_next, eta, dt_min, dt_max, f1, ti, dti, r, v, a, j, s, c);
}

int launch_correct(nb_ctx *ctx, const int32_t *active, int64_t m, double t_next)
{
    if (m <= 0) return NB_OK;
    k_correct<<<(unsigned)((m + 127) / 128), 128, 0, ctx->stream>>>((int)m, ctx->Npad, active, t_next, ctx->eta,
                                                                    ctx->dt_min, ctx->dt_max, ctx->f1, ctx->t,
                                                                    ctx->dt, ctx->r, ctx->v, ctx->a, ctx->j,
                                                                    ctx->s, ctx->c);
    NB_LAUNCH_CHECK(ctx, "k_correct");
    return NB_OK;
}

// ---------------------------------------------------------------------------------------
// Start-up S0 (paper silent; G8).  pass 1: a, jerk <- evaluation with a_pred = 0, and the
// predicted accelerations become a.  pass 2: a, jerk, snap <- evaluation with a_pred = a;
// crackle = 0; dt_i = pow2floor(eta_init min(|a|/|jerk|, sqrt(|a|/|snap|))), clamped.
__global__ void k_startup_commit(const int64_t N, const int64_t Npad, const int pass, const double eta_init,
                                 const double dt_min, const double dt_max, const double *__restrict__ f1,
                                 double *__restrict__ a, double *__restrict__ j, double *__restrict__ s,
                                 double *__restrict__ c, double *__restrict__ ti, double *__restrict__ dti,
                                 double *__restrict__ jp)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    double A[3], J[3], S[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        A[d] = f1[(0 + d) * Npad + i]; J[d] = f1[(3 + d) * Npad + i]; S[d] = f1[(6 + d) * Npad + i];
        a[d * Npad + i] = A[d]; j[d * Npad + i] = J[d];
    }
    if (pass == 1) {
        double *rec = jp + i * REC;
        rec[6] = A[0]; rec[7] = A[1]; rec[8] = A[2];
        return;
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) { s[d * Npad + i] = S[d]; c[d * Npad + i] = 0.0; }
    const double na = norm3_rn(A[0], A[1], A[2]), nj = norm3_rn(J[0], J[1], J[2]), ns = norm3_rn(S[0], S[1], S[2]);
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    double q = inf;
    if (nj > 0.0) q = __ddiv_rn(na, nj);
    if (ns > 0.0) {
        const double q2 = __dsqrt_rn(__ddiv_rn(na, ns));
        if (q2 < q) q = q2;
    }
    double dt;
    if (isinf(q)) dt = dt_max;
    else {
        const double x = __dmul_rn(eta_init, q);
        if (!(x > 0.0) || x < 2.2250738585072014e-308) dt = dt_min;
        else dt = pow2i(ilogb_pos_normal(x));
    }
    if (dt < dt_min) dt = dt_min;
    if (dt > dt_max) dt = dt_max;
    ti[i] = 0.0;
    dti[i] = dt;
}

int launch_startup_commit(nb_ctx *ctx, int pass)
{
    const int64_t N = ctx->N;
    k_startup_commit<<<(unsigned)((N + 255) / 256), 256, 0, ctx->stream>>>(N, ctx->Npad, pass, ctx->eta_init,
                                                                           ctx->dt_min, ctx->dt_max, ctx->f1, ctx->a,
                                                                           ctx->j, ctx->s, ctx->c, ctx->t, ctx->dt,
                                                                           ctx->jp);
    NB_LAUNCH_CHECK(ctx, "k_startup_commit");
    return NB_OK;
}

// ---------------------------------------------------------------------------------------
// checkpoint: [N][21] = {m, t, dt, r, v, a, jerk, snap, crackle}  <->  SoA planes
__global__ void k_full_state(const int64_t N, const int64_t Npad, double *__restrict__ st, const bool to_ctx,
                             double *__restrict__ mass, double *__restrict__ ti, double *__restrict__ dti,
                             double *__restrict__ r, double *__restrict__ v, double *__restrict__ a,
                             double *__restrict__ j, double *__restrict__ s, double *__restrict__ c)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    double *p = st + 21 * i;
    double *planes[6] = {r, v, a, j, s, c};
    if (to_ctx) {
        mass[i] = p[0]; ti[i] = p[1]; dti[i] = p[2];
#pragma unroll
        for (int q = 0; q < 6; ++q)
#pragma unroll
            for (int d = 0; d < 3; ++d) planes[q][d * Npad + i] = p[3 + 3 * q + d];
    } else {
        p[0] = mass[i]; p[1] = ti[i]; p[2] = dti[i];
#pragma unroll
        for (int q = 0; q < 6; ++q)
#pragma unroll
            for (int d = 0; d < 3; ++d) p[3 + 3 * q + d] = planes[q][d * Npad + i];
    }
}

int launch_full_state(nb_ctx *ctx, double *state, bool to_ctx)
{
    const int64_t N = ctx->N;
    k_full_state<<<(unsigned)((N + 255) / 256), 256, 0, ctx->stream>>>(N, ctx->Npad, state, to_ctx, ctx->mass, ctx->t,
                                                                       ctx->dt, ctx->r, ctx->v, ctx->a, ctx->j,
                                                                       ctx->s, ctx->c);
    NB_LAUNCH_CHECK(ctx, "k_full_state");
    return NB_OK;
}

// ---------------------------------------------------------------------------------------
// Device-driven block-step loop.  The same steps as above, but every
// size that depends on the active set is read from the control block StepCtl in device memory,
// so that the kernels of a step have fixed launch configurations and a batch of steps can be
// replayed as one CUDA graph without the host learning (t_next, m) in between.  One step is
//   k_g_gather_predict  : Table 1 row 1 + Eq. 3-7 in ONE pass over the particles: t_next is already
//                         known (the minimum was collected during the previous step), so a thread
//                         appends its particle to the active list if it is due (warp-aggregated
//                         atomic; the order of the list does not affect any result, G18), predicts
//                         it, and contributes t_i + dt_i of a particle that is NOT due to the minimum
//                         of the next step
//                         of the next step; the last block to finish publishes m and the geometry
//   k_force_persistent  : evaluation (nb_force.cu)
//   k_reduce_persistent : fixed-order sum of the j-split partials (nb_force.cu)
//   k_g_correct         : corrector and new dt for the active set, their share of the next minimum,
//                         bookkeeping
// All per-step scalars are double-buffered by the parity of the step (StepCtl).
__global__ void k_g_begin(StepCtl *ctl, const double t_end, const long long steps)
{
    ctl->tmin[0] = 0x7ff0000000000000ULL; ctl->tmin[1] = 0x7ff0000000000000ULL;
    ctl->cnt[0] = 0; ctl->cnt[1] = 0;
    ctl->done = 0; ctl->ticket = 0; ctl->work = 0;
    ctl->t_end = t_end; ctl->steps_left = steps; ctl->n_steps = 0; ctl->n_pairs = 0.0;
    for (int b = 0; b < 64; ++b) ctl->hist[b] = 0;
}

__global__ void __launch_bounds__(SCHED_THREADS)
    k_g_gather_predict(const int p, const int64_t N, const int64_t Npad, const double *__restrict__ t,
                       const double *__restrict__ dt, int32_t *__restrict__ active, StepCtl *__restrict__ ctl,
                       const double *__restrict__ mass, const double *__restrict__ r, const double *__restrict__ v,
                       const double *__restrict__ a, const double *__restrict__ j, const double *__restrict__ s,
                       const double *__restrict__ c, double *__restrict__ jp, const int n_sm, const int occ,
                       const int64_t partials_limit, const int force_split, const int force_jlanes,
                       ForceGeom *__restrict__ geom_cache)
{
    pdl_trigger();
    pdl_wait();
    // every block evaluates the same condition from values no kernel of this step modifies
    const double tn = __longlong_as_double((long long)ctl->tmin[p]);
    const bool done = ctl->done || ctl->steps_left <= 0 || !(tn <= ctl->t_end);
    if (done) {
        if (blockIdx.x == 0 && threadIdx.x == 0) ctl->done = 1;
        return;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) ctl->t_next = tn;
    const int64_t i = (int64_t)blockIdx.x * SCHED_THREADS + threadIdx.x;
    double vmin = __longlong_as_double(0x7ff0000000000000LL);
    bool hit = false;
    if (i < N) {
        const double due = t[i] + dt[i];
        hit = (due == tn);
        if (!hit) vmin = due;
        predict_one(i, Npad, tn, t, mass, r, v, a, j, s, c, jp);
    }
    // warp-aggregated append
    const unsigned mask = __ballot_sync(0xffffffffu, hit);
    if (mask) {
        const int lane = threadIdx.x & 31;
        const int leader = __ffs(mask) - 1;
        int base = 0;
        if (lane == leader) base = atomicAdd(&ctl->cnt[p], __popc(mask));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (hit) active[base + __popc(mask & ((1u << lane) - 1u))] = (int32_t)i;
    }
    block_min_to(vmin, &ctl->tmin[1 - p]);

    // the last block to finish knows m: it publishes (m, evaluation geometry).  The 65 split
    // candidates of choose_split are scored by one thread each (a single thread doing the 64-bit
    // divisions alone costs more than the rest of the step).
    __shared__ bool last;
    __shared__ ForceGeom sg;
    __shared__ SplitProblem sp;
    __shared__ long long scost[MAX_WAVES + 1];
    __shared__ int ssplit[MAX_WAVES + 1];
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        last = (atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    const int m = *((volatile int *)&ctl->cnt[p]);
    // the geometry is a function of m alone while the knobs stay put: block-step runs see the same
    // few set sizes again and again, so the answers for m <= GEOM_CACHE_M are remembered
    if (m <= GEOM_CACHE_M && geom_cache[m].S != 0) {
        if (threadIdx.x == 0) {
            ctl->ticket = 0;
            ctl->n_active = m;
            ctl->g = geom_cache[m];
        }
        return;
    }
    if (threadIdx.x == 0) {
        ctl->ticket = 0;
        sp = geom_begin(sg, m, Npad, n_sm, occ, partials_limit, force_jlanes);
    }
    __syncthreads();
    if (threadIdx.x <= MAX_WAVES) {
        int S;
        scost[threadIdx.x] = split_candidate(sp, threadIdx.x, &S);
        ssplit[threadIdx.x] = S;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long best = INT64_MAX;
        int best_s = 1;
        for (int w = 0; w <= MAX_WAVES; ++w)
            if (scost[w] < best) { best = scost[w]; best_s = ssplit[w]; }
        geom_finish(sg, sp, best_s, force_split);
        ctl->n_active = m;
        ctl->g = sg;
        if (m <= GEOM_CACHE_M) geom_cache[m] = sg;
    }
}

// Sum of the split partials, corrector and new dt for the active set, their share of the next minimum,
// and -- block 0 -- the bookkeeping of the step; that touches only fields which no block of this kernel
// reads (they read t_next, n_active, g, which the earlier kernels of the step published).
// One split: the evaluation wrote f1 itself, one thread corrects one particle.  Several splits: one WARP
// per active particle sums its nine components in the fixed order of part_layout / sum_splits_* (the order
// of k_reduce_thread / k_reduce_warp of the host-issued path), stores them to f1, and lane 0 corrects.
__global__ void __launch_bounds__(SCHED_THREADS)
    k_g_reduce_correct(const int p, const int64_t N, const int64_t Npad, const int32_t *__restrict__ active_list,
                       StepCtl *__restrict__ ctl, const double eta, const double dt_min, const double dt_max,
                       const double *__restrict__ partials, double *__restrict__ f1, double *__restrict__ ti,
                       double *__restrict__ dti, double *__restrict__ r, double *__restrict__ v,
                       double *__restrict__ a, double *__restrict__ j, double *__restrict__ s, double *__restrict__ c)
{
    pdl_trigger();
    pdl_wait();
    if (ctl->done) return;
    const int m = (int)ctl->n_active;
    const double tn = ctl->t_next;
    const int S = ctl->g.S;
    const int32_t *active = (m == N) ? nullptr : active_list;
    double vmin = __longlong_as_double(0x7ff0000000000000LL);
    if (S <= 1) {
        for (int k = blockIdx.x * SCHED_THREADS + threadIdx.x; k < m; k += gridDim.x * SCHED_THREADS) {
            const int64_t i = active ? active[k] : k;
            vmin = fmin(vmin, correct_one(k, i, Npad, tn, eta, dt_min, dt_max, f1, ti, dti, r, v, a, j, s, c));
        }
    } else {
        const PartLayout L = part_layout(S, ctl->g.mpad, Npad);
        const int lane = threadIdx.x & 31;
        const int nwarps = (gridDim.x * SCHED_THREADS) >> 5;
        for (int k = (blockIdx.x * SCHED_THREADS + threadIdx.x) >> 5; k < m; k += nwarps) {
            reduce_one(partials, S, L, k, lane, f1, Npad);
            if (lane == 0) {
                const int64_t i = active ? active[k] : k;
                vmin = fmin(vmin, correct_one(k, i, Npad, tn, eta, dt_min, dt_max, f1, ti, dti, r, v, a, j, s, c));
            }
        }
    }
    block_min_to(vmin, &ctl->tmin[1 - p]);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        ctl->t_now = tn;
        ctl->steps_left -= 1;
        ctl->n_steps += 1;
        ctl->n_pairs += (double)m * (double)N;
        int b = 0;
        while ((1LL << (b + 1)) <= (long long)m) ++b;
        ctl->hist[b] += 1;
        ctl->tmin[p] = 0x7ff0000000000000ULL;   // this step's minimum is consumed: slot p collects the one after next
        ctl->cnt[p] = 0;
        ctl->work = 0;
    }
}

int launch_graph_begin(nb_ctx *ctx, double t_end, int64_t steps)
{
    k_g_begin<<<1, 1, 0, ctx->stream>>>(ctx->ctl, t_end, (long long)steps);
    NB_LAUNCH_CHECK(ctx, "k_g_begin");
    int g = (int)((ctx->N + SCHED_THREADS - 1) / SCHED_THREADS);
    if (g > 4 * ctx->n_sm) g = 4 * ctx->n_sm;
    k_tmin<<<g, SCHED_THREADS, 0, ctx->stream>>>(ctx->N, ctx->t, ctx->dt, &ctx->ctl->tmin[0]);
    NB_LAUNCH_CHECK(ctx, "k_tmin");
    return NB_OK;
}

int enqueue_graph_gather_predict(nb_ctx *ctx, int parity)
{
    const unsigned np = (unsigned)((ctx->N + SCHED_THREADS - 1) / SCHED_THREADS);
    launch_chain(k_g_gather_predict, dim3(np), dim3(SCHED_THREADS), ctx->stream, ctx->use_graph == 2, (size_t)0, parity, ctx->N,
                 ctx->Npad, ctx->t, ctx->dt, ctx->active, ctx->ctl, ctx->mass, ctx->r, ctx->v, ctx->a, ctx->j, ctx->s,
                 ctx->c, ctx->jp, ctx->n_sm, ctx->occ[0], (int64_t)ctx->partials_limit, ctx->force_split,
                 ctx->force_jlanes, ctx->geom_cache);
    NB_LAUNCH_CHECK(ctx, "k_g_gather_predict");
    return NB_OK;
}

int enqueue_graph_correct(nb_ctx *ctx, int parity)
{
    // enough warps for one per active particle of a small set; large sets (one split) go thread per particle
    int64_t g = (ctx->N + SCHED_THREADS - 1) / SCHED_THREADS;
    if (g > 4 * ctx->n_sm) g = 4 * ctx->n_sm;
    launch_chain(k_g_reduce_correct, dim3((unsigned)g), dim3(SCHED_THREADS), ctx->stream, ctx->use_graph == 2, (size_t)0, parity, ctx->N,
                 ctx->Npad, ctx->active, ctx->ctl, ctx->eta, ctx->dt_min, ctx->dt_max, ctx->partials, ctx->f1, ctx->t, ctx->dt,
                 ctx->r, ctx->v, ctx->a, ctx->j, ctx->s, ctx->c);
    NB_LAUNCH_CHECK(ctx, "k_g_reduce_correct");
    return NB_OK;
}

}  // namespace nb
