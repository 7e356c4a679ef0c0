// nb_resident.cu -- the block-step loop resident on ONE thread-block cluster, state in shared memory
// (loop mode 3, N <= RES_MAX_N).
//
// For a small system most block steps advance a handful of particles (config 1, N = 1024: m < 8 in two
// steps out of three; PAPER.md:252 is about exactly these steps, Table 1 rows 1 and 4).  Such a step is a
// few thousand pair interactions; what it costs is latency: the graph-driven loop (nb_graph.cu) pays three
// kernel boundaries and a dozen dependent round trips to L2 per step (~23 us at N = 1024, measured).  Here ONE
// kernel, launched once per nb_run_until / nb_run_steps call as a single cluster of up to 16 CTAs, keeps
// the whole system on chip and runs every step until the time or step budget is used:
//
//   * CTA `rank` OWNS the particles [rank NL, (rank + 1) NL): their committed state (21 doubles each) and their
//     predicted records live in its shared memory for the whole run (loaded once, written back once).
//   * phase 1  gather + predict   Table 1 row 1 + Eq. 3-7 for the owned particles; the due ones go to the CTA's
//                                 list, whose length is broadcast to every CTA through distributed shared memory
//   * phase 2  evaluate           Eq. 8-10: every CTA evaluates ALL m active particles (their records read from the
//                                 owners' shared memory) against ITS OWN NL predicted records -- the paper's split of
//                                 the j-range with one split per CTA -- and stores the partial
//                                 (a, jerk, snap) into the owner's shared memory
//   * phase 3  reduce + correct   the owner sums the partials of its active particles in CTA-rank order, applies
//                                 Eq. 11-16 (correct_one), and broadcasts the minimum of t_i + dt_i it now holds
//   with one hardware cluster barrier (barrier.cluster, release / acquire) after each phase.
//
// The arithmetic is that of the other drivers (pair_body, predict_one, correct_one, new_dt); only the order
// in which the pair terms of one particle are added differs (per lane over the owner-CTA slice, butterfly over
// the lanes, then over the CTAs in rank order: fixed, so runs are bit-reproducible).  Results therefore agree
// with the other drivers to rounding (G18), not bit for bit; tests/test_gpu_graph.py checks identical time
// steps and positions to 1e-12 against the host-issued call sequence.
#include <cooperative_groups.h>

#include "nb_internal.cuh"
#include "nb_force_dev.cuh"
#include "nb_step_dev.cuh"
#include "nb_resident_dev.cuh"

namespace cg = cooperative_groups;

namespace nb {

constexpr int RES_THREADS = 512;    // 16 warps per CTA
constexpr int RES_WARPS = RES_THREADS / 32;
constexpr int RES_MAXC = 16;        // largest cluster
constexpr int RES_NL_MAX = 256;     // owned particles per CTA at most (N <= 2048 on 8 CTAs; 16 CTAs: 128 each)
constexpr int RES_PUSH_MIN = 16;    // each owner pushes the records of its first `push` due particles to every CTA: at least
                                    // this many, and as many more (up to all NL) as the shared memory left over holds
constexpr size_t RES_SMEM_BUDGET = 227 * 1024 - 2048;   // opt-in shared memory of a CTA on sm_100 less the static part

// Shared-memory plan of one CTA (NL = owned particles, a multiple of 32; doubles unless noted):
//   state  : t, dt, mass [NL]; r, v, a, jerk, snap, crackle [3][NL]      21 NL
//   rec    : predicted records [NL][REC]                                   10 NL
//   f1     : reduced (a, jerk, snap) of the owned active particles [9][NL]  9 NL
//   part   : partials [C][9][NL] (writer CTA, component, slot), written by every CTA of the cluster   9 C NL
//   irec   : records of the first `push` due particles of every CTA [16][push][REC], pushed by their owners
//            (a small active set is then evaluated without a read from remote shared memory)
//   tmin   : min(t_i + dt_i) of every CTA [16];  list: int32 local indices of the owned due particles [NL];
//   cnt    : int32 list length of every CTA [16]
struct ResPlan {
    int NL, C, push;
    size_t o_t, o_dt, o_m, o_r, o_v, o_a, o_j, o_s, o_c, o_rec, o_f1, o_part, o_irec, o_tmin, o_list, o_cnt, bytes;
};
__host__ __device__ inline ResPlan res_plan(const int64_t N, const int C)
{
    ResPlan p;
    p.C = C;
    int NL = (int)((N + C - 1) / C);
    NL = (NL + 31) & ~31;
    p.NL = NL;
    size_t o = 0;
    p.o_t = o; o += (size_t)NL * 8;
    p.o_dt = o; o += (size_t)NL * 8;
    p.o_m = o; o += (size_t)NL * 8;
    p.o_r = o; o += (size_t)3 * NL * 8;
    p.o_v = o; o += (size_t)3 * NL * 8;
    p.o_a = o; o += (size_t)3 * NL * 8;
    p.o_j = o; o += (size_t)3 * NL * 8;
    p.o_s = o; o += (size_t)3 * NL * 8;
    p.o_c = o; o += (size_t)3 * NL * 8;
    p.o_rec = o; o += (size_t)REC * NL * 8;
    p.o_f1 = o; o += (size_t)9 * NL * 8;
    p.o_part = o; o += (size_t)9 * C * NL * 8;
    {   // irec takes what is left after everything else (the three small arrays below: 16 doubles + NL + 16 ints)
        const size_t rest = o + (size_t)RES_MAXC * 8 + (size_t)NL * 4 + (size_t)RES_MAXC * 4 + 64;
        int push = rest < RES_SMEM_BUDGET ? (int)((RES_SMEM_BUDGET - rest) / ((size_t)RES_MAXC * REC * 8)) : 0;
        if (push > NL) push = NL;
        if (push < RES_PUSH_MIN) push = RES_PUSH_MIN;
        p.push = push;
    }
    p.o_irec = o; o += (size_t)RES_MAXC * p.push * REC * 8;
    p.o_tmin = o; o += (size_t)RES_MAXC * 8;
    p.o_list = o; o += (size_t)NL * 4;
    p.o_cnt = o; o += (size_t)RES_MAXC * 4;
    p.bytes = (o + 15) & ~(size_t)15;
    return p;
}

template <bool GUARD0, int MX>
__global__ void __launch_bounds__(RES_THREADS, 1)
    k_resident_loop(const int64_t N, const int64_t Npad, const double eps2, const double eta, const double dt_min,
                    const double dt_max, double *__restrict__ g_t, double *__restrict__ g_dt, const double *__restrict__ g_m,
                    double *__restrict__ g_r, double *__restrict__ g_v, double *__restrict__ g_a, double *__restrict__ g_j,
                    double *__restrict__ g_s, double *__restrict__ g_c, double *__restrict__ g_jp, StepCtl *__restrict__ ctl,
                    const int force_jlanes)
{
    extern __shared__ __align__(128) unsigned char smem[];
    cg::cluster_group cluster = cg::this_cluster();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int lgC = 31 - __clz(C);                                  // the cluster has 8 or 16 CTAs
    const ResPlan P = res_plan(N, C);
    const int NL = P.NL, PUSH = P.push;
    double *t = (double *)(smem + P.o_t), *dt = (double *)(smem + P.o_dt), *mass = (double *)(smem + P.o_m);
    double *r = (double *)(smem + P.o_r), *v = (double *)(smem + P.o_v), *a = (double *)(smem + P.o_a);
    double *j = (double *)(smem + P.o_j), *s = (double *)(smem + P.o_s), *c = (double *)(smem + P.o_c);
    double *rec = (double *)(smem + P.o_rec), *f1 = (double *)(smem + P.o_f1), *part = (double *)(smem + P.o_part);
    double *tmin = (double *)(smem + P.o_tmin), *irec = (double *)(smem + P.o_irec);
    int *list = (int *)(smem + P.o_list), *cnt = (int *)(smem + P.o_cnt);
    __shared__ int n_list;
    __shared__ long long hist[64];
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const int64_t first = (int64_t)rank * NL;                       // first owned particle
    const int64_t left = N - first;
    const int n_own = left <= 0 ? 0 : (left < NL ? (int)left : NL);

    // ---- load the owned slice (rows beyond N: mass 0 at the origin, never due)
    for (int i = tid; i < NL; i += RES_THREADS) {
        const bool live = i < n_own;
        const int64_t gi = first + i;
        t[i] = live ? g_t[gi] : 0.0; dt[i] = live ? g_dt[gi] : inf; mass[i] = live ? g_m[gi] : 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int64_t gq = d * Npad + gi;
            const int q = d * NL + i;
            r[q] = live ? g_r[gq] : 0.0; v[q] = live ? g_v[gq] : 0.0; a[q] = live ? g_a[gq] : 0.0;
            j[q] = live ? g_j[gq] : 0.0; s[q] = live ? g_s[gq] : 0.0; c[q] = live ? g_c[gq] : 0.0;
        }
#pragma unroll
        for (int d = 0; d < REC; ++d) rec[i * REC + d] = 0.0;
    }
    for (int b = tid; b < 64; b += RES_THREADS) hist[b] = 0;
    long long steps_left = ctl->steps_left;
    const double t_end = ctl->t_end;
    long long n_steps = 0;
    double n_pairs = 0.0, t_now = 0.0;
    __syncthreads();

    // minimum of t_i + dt_i over the owned particles -> tmin[rank] of every CTA
    // (one warp does it: a CTA owns at most RES_NL_MAX = 256 particles, eight per lane; the callers have just passed a
    // block barrier, so the corrected times are visible; no barrier inside)
    auto publish_min = [&]() {
        if (warp == 0) {
            double vmin = inf;
            for (int i = lane; i < n_own; i += 32) vmin = fmin(vmin, t[i] + dt[i]);
            for (int off = 16; off > 0; off >>= 1) vmin = fmin(vmin, __shfl_xor_sync(0xffffffffu, vmin, off));
            if (lane < C) cluster.map_shared_rank(tmin, lane)[rank] = vmin;
            if (lane == 0) n_list = 0;   // for the list of the next step (its phase 1 starts after the cluster barrier)
        }
    };
    publish_min();
    cluster.sync();
#ifdef NB_RES_TIMING   // development aid: cycles per phase, summed by one thread into unused histogram bins
    long long tph[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long tq = clock64();
#define NB_TICK(q) do { const long long now_ = clock64(); tph[q] += now_ - tq; tq = now_; } while (0)
#else
#define NB_TICK(q) do { } while (0)
#endif

    for (;;) {
        // ---- next block time: every thread of the cluster computes the same minimum
        double tn = (lane & (RES_MAXC - 1)) < C ? tmin[lane & (RES_MAXC - 1)] : inf;   // both half-warps hold the 16 minima
        for (int off = RES_MAXC / 2; off > 0; off >>= 1) tn = fmin(tn, __shfl_xor_sync(0xffffffffu, tn, off));
        if (steps_left <= 0 || !(tn <= t_end)) break;
        NB_TICK(0);

        // ---- phase 1: predict the owned particles (Eq. 3-7), list the due ones (Table 1 row 1)
        for (int i = tid; i < n_own; i += RES_THREADS) {          // (n_list was reset by publish_min, before the barrier)
            predict_one(i, NL, tn, t, mass, r, v, a, j, s, c, rec);
            if (t[i] + dt[i] == tn) list[atomicAdd(&n_list, 1)] = i;
        }
        __syncthreads();
        if (tid < C) cluster.map_shared_rank(cnt, tid)[rank] = n_list;
        {   // the records of the first PUSH due particles go to every CTA (remote stores, fire and forget)
            const int np = n_list < PUSH ? n_list : PUSH;
            for (int e = tid; e < C * np * (REC / 2); e += RES_THREADS) {   // 16-byte stores; C is a power of two
                const int o = e & (C - 1), w = e >> lgC, qq = w / (REC / 2), d = w - qq * (REC / 2);
                reinterpret_cast<double2 *>(cluster.map_shared_rank(irec, o) + ((size_t)rank * PUSH + qq) * REC)[d] =
                    reinterpret_cast<const double2 *>(rec + (size_t)list[qq] * REC)[d];
            }
        }
        NB_TICK(1);
        cluster.sync();
        NB_TICK(2);

        // ---- phase 2: all m active particles against the owned records; partials to the owners
        // inclusive prefix of the owners' list lengths, one per lane (lanes >= C hold the total): a warp scan
        int inc = lane < C ? cnt[lane] : 0;
#pragma unroll
        for (int off = 1; off < RES_MAXC; off <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, inc, off);
            if (lane >= off) inc += y;
        }
        const int m = __shfl_sync(0xffffffffu, inc, RES_MAXC - 1);
        int lj = 0;                                             // JL = 2^lj lanes per i: shifts, not divisions, below
        if (force_jlanes >= 1) { const int want = force_jlanes < JL_MAX ? force_jlanes : JL_MAX; while ((2 << lj) <= want) ++lj; }
        else { while ((2 << lj) <= JL_MAX && (m << (lj + 1)) <= RES_THREADS) ++lj; }
        const int JL = 1 << lj;
        const int slots = RES_THREADS >> lj;
        const int rot = (rank * m) >> lgC;                      // m <= 2048, rank < 16
        for (int k0 = 0; k0 < m; k0 += slots) {                 // warp-uniform trip count
            if (k0 + ((tid & ~31) >> lj) >= m) continue;           // a warp without a live slot has nothing to add
            const int k = k0 + (tid >> lj), jl = tid & (JL - 1);
            const bool live = k < m;
            // every CTA walks the slots in its own rotation, so that at any moment the 16 CTAs read the records of, and
            // store partial sums to, different owners instead of all pressing on the same few
            int kk = (live ? k : m - 1) + rot;
            if (kk >= m) kk -= m;
            int o, bo;                                          // owner CTA of slot kk and the first slot it owns:
            if (lj == 5) {                                      // one slot per warp (m <= 16): every lane asks the same
                o = __popc(__ballot_sync(0xffffffffu, lane < RES_MAXC && inc <= kk));   // owners wholly before slot kk
                bo = __shfl_sync(0xffffffffu, inc, o > 0 ? o - 1 : 0);
                if (o == 0) bo = 0;
            } else {
                o = 0; bo = 0;
#pragma unroll
                for (int q = 1; q < RES_MAXC; ++q) {
                    const int bq = __shfl_sync(0xffffffffu, inc, q - 1);
                    if (q < C && kk >= bq) { o = q; bo = bq; }
                }
            }
            const int qloc = kk - bo;                           // slot in the owner's list
            const double *ri;
            if (qloc < PUSH) ri = irec + ((size_t)o * PUSH + qloc) * REC;             // pushed by its owner in phase 1
            else ri = cluster.map_shared_rank(rec, o) + (size_t)cluster.map_shared_rank(list, o)[qloc] * REC;
            double rl[REC];                                     // the i-record in five 16-byte loads (local or remote)
#pragma unroll
            for (int d = 0; d < REC / 2; ++d) {
                const double2 w = reinterpret_cast<const double2 *>(ri)[d];
                rl[2 * d] = w.x; rl[2 * d + 1] = w.y;
            }
            ri = rl;
            Acc9 T;
            switch (JL) {
                case 1: T = res_eval<1, GUARD0, MX>(ri, rec, jl, NL, eps2); break;
                case 2: T = res_eval<2, GUARD0, MX>(ri, rec, jl, NL, eps2); break;
                case 4: T = res_eval<4, GUARD0, MX>(ri, rec, jl, NL, eps2); break;
                case 8: T = res_eval<8, GUARD0, MX>(ri, rec, jl, NL, eps2); break;
                case 16: T = res_eval<16, GUARD0, MX>(ri, rec, jl, NL, eps2); break;
                default: T = res_eval<32, GUARD0, MX>(ri, rec, jl, NL, eps2); break;
            }
            if (live && jl == 0) {
                // part[writer][component][slot]: the lanes of a warp hold consecutive slots of (mostly) one owner, so each
                // of the nine remote stores of a warp is one contiguous row in the owner's shared memory
                double *dst = cluster.map_shared_rank(part, o) + (size_t)rank * 9 * NL + qloc;
                dst[0 * NL] = T.ax; dst[1 * NL] = T.ay; dst[2 * NL] = T.az; dst[3 * NL] = T.jx; dst[4 * NL] = T.jy;
                dst[5 * NL] = T.jz; dst[6 * NL] = T.sx; dst[7 * NL] = T.sy; dst[8 * NL] = T.sz;
            }
        }
#ifdef NB_RES_TIMING
        {   // phase-2 cycles by floor(log2 m) -> bins 48 + b (development aid)
            const long long now_ = clock64();
            int b_ = 0;
            while ((1LL << (b_ + 1)) <= (long long)m) ++b_;
            if (rank == 0 && tid == 0 && b_ < 15) hist[48 + b_] += now_ - tq;
        }
#endif
        NB_TICK(3);
        cluster.sync();
        NB_TICK(4);

        // ---- phase 3: the owner sums the C partials of each of its active particles in rank order and
        // corrects it (Eq. 11-16).  One warp per particle: lanes 0..8 take one component each.
        const int n_mine = cnt[rank];
        if (n_mine <= RES_WARPS) {
            for (int q = warp; q < n_mine; q += RES_WARPS) {
                if (lane < 9) {
                    double acc = 0.0;
                    for (int o = 0; o < C; ++o) acc += part[((size_t)o * 9 + lane) * NL + q];
                    f1[lane * NL + q] = acc;
                }
                __syncwarp();
                correct_warp(lane, q, list[q], NL, tn, eta, dt_min, dt_max, f1, t, dt, r, v, a, j, s, c);
            }
        } else {
            // many active particles per CTA (a large step): one thread per (particle, component) for the sums, then one
            // thread per particle for the corrector (correct_one: the expressions and rounding order of correct_warp);
            // a warp taking several particles in turn would run their dependent chains one after the other
            for (int e = tid; e < n_mine * 9; e += RES_THREADS) {
                const int cc = e / n_mine, q = e - cc * n_mine;     // consecutive threads: consecutive slots
                double acc = 0.0;
                for (int o = 0; o < C; ++o) acc += part[((size_t)o * 9 + cc) * NL + q];
                f1[cc * NL + q] = acc;
            }
            __syncthreads();
            for (int q = tid; q < n_mine; q += RES_THREADS)
                correct_one(q, list[q], NL, tn, eta, dt_min, dt_max, f1, t, dt, r, v, a, j, s, c);
        }
        __syncthreads();
        steps_left -= 1; n_steps += 1; n_pairs += (double)m * (double)N; t_now = tn;
        if (tid == 0) {
            int b = 0;
            while ((1LL << (b + 1)) <= (long long)m) ++b;
            hist[b] += 1;
        }
        publish_min();
        NB_TICK(5);
        cluster.sync();
        NB_TICK(6);
    }
#ifdef NB_RES_TIMING
    if (rank == 0 && tid == 0)
        for (int q = 0; q < 8; ++q) hist[40 + q] += tph[q];
    __syncthreads();
#endif

    // ---- write the owned slice back: committed state and the last prediction
    __syncthreads();
    for (int i = tid; i < n_own; i += RES_THREADS) {
        const int64_t gi = first + i;
        g_t[gi] = t[i]; g_dt[gi] = dt[i];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int64_t gq = d * Npad + gi;
            const int q = d * NL + i;
            g_r[gq] = r[q]; g_v[gq] = v[q]; g_a[gq] = a[q]; g_j[gq] = j[q]; g_s[gq] = s[q]; g_c[gq] = c[q];
        }
        if (n_steps > 0) {
#pragma unroll
            for (int d = 0; d < REC; ++d) g_jp[gi * REC + d] = rec[i * REC + d];
        }
    }
    if (rank == 0 && tid == 0) {
        ctl->steps_left = steps_left; ctl->n_steps = n_steps; ctl->n_pairs = n_pairs; ctl->t_now = t_now;
        for (int b = 0; b < 64; ++b) ctl->hist[b] = hist[b];
        ctl->done = 1;
    }
    cluster.sync();   // no CTA leaves while another may still read its shared memory
}

// ---- host side ---------------------------------------------------------------------------
template <bool G0, int MX>
static cudaError_t launch_resident(nb_ctx *ctx, int n_cta)
{
    auto kern = k_resident_loop<G0, MX>;
    const ResPlan P = res_plan(ctx->N, n_cta);
    if (P.NL > RES_NL_MAX) return cudaErrorInvalidValue;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P.bytes);
    if (e != cudaSuccess) return e;
    if (n_cta > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_cta); cfg.blockDim = dim3(RES_THREADS);
    cfg.dynamicSmemBytes = P.bytes; cfg.stream = ctx->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)n_cta; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int n_clusters = 0;
    e = cudaOccupancyMaxActiveClusters(&n_clusters, kern, &cfg);
    if (e != cudaSuccess) return e;
    if (n_clusters < 1) return cudaErrorLaunchOutOfResources;
    return cudaLaunchKernelEx(&cfg, kern, ctx->N, ctx->Npad, ctx->eps2, ctx->eta, ctx->dt_min, ctx->dt_max, ctx->t, ctx->dt,
                              (const double *)ctx->mass, ctx->r, ctx->v, ctx->a, ctx->j, ctx->s, ctx->c, ctx->jp, ctx->ctl,
                              ctx->force_jlanes);
}

static cudaError_t launch_resident_any(nb_ctx *ctx, int n_cta)
{
    const int mx = ctx->precision == 1 ? 1 : (ctx->precision == 2 ? 3 : 0);
    const bool g0 = mx ? (float)ctx->eps2 < 1e-24f : ctx->eps == 0.0;   // as in nb_force.cu
    if (g0 && mx == 1) return launch_resident<true, 1>(ctx, n_cta);
    if (g0 && mx == 3) return launch_resident<true, 3>(ctx, n_cta);
    if (g0) return launch_resident<true, 0>(ctx, n_cta);
    if (mx == 1) return launch_resident<false, 1>(ctx, n_cta);
    if (mx == 3) return launch_resident<false, 3>(ctx, n_cta);
    return launch_resident<false, 0>(ctx, n_cta);
}

// Advance while the next block time is <= t_end and fewer than max_steps steps were taken: one launch.
int resident_run(nb_ctx *ctx, double t_end, int64_t max_steps, int64_t *n_steps)
{
    if (ctx->N > RES_MAX_N)
        return set_err(ctx, NB_EINVAL, "loop mode 3 (cluster-resident loop) serves N <= %lld; this context has N = %lld",
                       (long long)RES_MAX_N, (long long)ctx->N);
    {
        const int rc = launch_graph_begin(ctx, t_end, max_steps);   // seeds the control block (t_end, steps_left, counters)
        if (rc != NB_OK) return rc;
    }
    if (ctx->res_cluster == 0) ctx->res_cluster = RES_MAXC;
    cudaError_t e = launch_resident_any(ctx, ctx->res_cluster);
    if (e != cudaSuccess && ctx->res_cluster > 8) {   // no 16-CTA cluster on this part: the portable size
        cudaGetLastError();
        ctx->res_cluster = 8;
        e = launch_resident_any(ctx, 8);
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        if (ctx->loop_auto) {   // this device cannot host the cluster: the default falls back to the graph-driven loop
            ctx->use_graph = 1;
            return graph_run(ctx, t_end, max_steps, n_steps);
        }
        return set_err(ctx, NB_ECUDA, "launch of k_resident_loop failed: %s", cudaGetErrorString(e));
    }
    ctx->n_launch += 1;
    NB_CUDA(ctx, cudaMemcpyAsync(ctx->h_ctl, ctx->ctl, sizeof(StepCtl), cudaMemcpyDeviceToHost, ctx->stream));
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const StepCtl *h = ctx->h_ctl;
    if (h->n_steps > 0) {
        ctx->t_now = h->t_now;
        ctx->pred_valid = true; ctx->t_pred = h->t_now;
    }
    ctx->n_steps += h->n_steps;
    ctx->n_pairs += h->n_pairs;
    for (int b = 0; b < 64; ++b) ctx->hist[b] += h->hist[b];
    ctx->have_block = false; ctx->evaluated = false; ctx->eval_partial = false;
    if (n_steps) *n_steps = h->n_steps;
    return NB_OK;
}

}  // namespace nb
