// nb_resident.cu -- the block-step loop resident on ONE thread-block cluster (loop mode 3).
//
// For a small system most block steps advance a handful of particles (config 1, N = 1024: m < 8 in two
// steps out of three; PAPER.md:252 is about exactly these steps, Table 1 rows 1 and 4).  The arithmetic of
// such a step is a few microseconds of one SM; what it costs is the hand-over between its phases.  The
// graph-driven loop (nb_graph.cu) pays five kernel boundaries per step (~20 us).  Here ONE kernel,
// launched once per nb_run_until / nb_run_steps call as a single cluster of RES_CLUSTER CTAs, runs
// every step until the control block says done, and the phases of a step are separated by the hardware
// cluster barrier (barrier.cluster, release / acquire at cluster scope):
//
//   phase 1  gather + predict   Table 1 row 1 + Eq. 3-7: one pass over the particles (as k_g_gather_predict)
//   -- cluster barrier --
//   phase 2  evaluate           the SAME items (i-block, j-split) of the SAME geometry rule as the other
//                               drivers, each worked by a "virtual CTA" of this cluster (128 threads on a
//                               named barrier) through force_item
//   -- cluster barrier --
//   phase 3  reduce + correct   one warp per active particle: the split partials in the fixed order of
//                               part_layout / sum_splits_*, then correct_one (Eq. 11-16) by lane 0
//   -- cluster barrier --
//
// The state stays in global memory (L2-resident at these sizes); the predicted stream written in phase 1
// by generic stores is read in phase 2 by bulk copies (async proxy), hence the proxy fences around the
// first barrier.  Device functions, geometry and summation order are those of the other drivers, so the
// states are bit-identical (tests/test_gpu_graph.py).  One cluster is at most 16 SMs: the mode is offered
// for N <= RES_MAX_N only and chosen by default for N <= RES_AUTO_N, where the all-active steps are still
// cheap on 16 SMs.
#include "nb_internal.cuh"
#include "nb_force_dev.cuh"
#include "nb_step_dev.cuh"

namespace nb {

constexpr int RES_THREADS = 512;                      // 16 warps per CTA: 4 per SM sub-partition
constexpr int RES_WARPS = RES_THREADS / 32;
constexpr int RES_VC = RES_THREADS / NT_E;            // virtual evaluation CTAs per CTA
constexpr int RES_GEOM_SLOTS = 64;                    // per-CTA direct-mapped memory of geometries by set size

struct ResShared {
    double tile[RES_VC][2][TJ_E * REC];   // one two-stage ring of j-tiles per virtual CTA
    uint64_t full[RES_VC][2];
    ForceGeom geom[RES_GEOM_SLOTS];
    int geom_m[RES_GEOM_SLOTS];
    SplitProblem sp;
    ForceGeom g;
    long long scost[MAX_WAVES + 1];
    int ssplit[MAX_WAVES + 1];
    double red[RES_WARPS];
};

__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// min over the CTA of one value per thread -> atomicMin on the bits (times are non-negative)
__device__ __forceinline__ void res_block_min_to(double v, unsigned long long *dst, double *red)
{
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    for (int off = 16; off > 0; off >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, off));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < RES_WARPS ? red[threadIdx.x] : inf;
        for (int off = 16; off > 0; off >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, off));
        if (threadIdx.x == 0 && v < inf) atomicMin(dst, (unsigned long long)__double_as_longlong(v));
    }
}

// The geometry of a set size, identical to choose_geom(): remembered per CTA (block-step runs see the same few
// sizes again and again); on a miss the split candidates are scored by one thread each.  Called by all threads.
__device__ __forceinline__ ForceGeom res_geometry(ResShared &sh, const int m, const int64_t Npad, const int n_sm,
                                                  const int occ, const int64_t partials_limit,
                                                  const int force_split, const int force_jlanes)
{
    const int slot = m & (RES_GEOM_SLOTS - 1);
    __syncthreads();
    if (sh.geom_m[slot] != m) {
        if (threadIdx.x == 0) sh.sp = geom_begin(sh.g, m, Npad, n_sm, occ, partials_limit, force_jlanes);
        __syncthreads();
        if (threadIdx.x <= MAX_WAVES) {
            int S;
            sh.scost[threadIdx.x] = split_candidate(sh.sp, threadIdx.x, &S);
            sh.ssplit[threadIdx.x] = S;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            long long best = INT64_MAX;
            int best_s = 1;
            for (int w = 0; w <= MAX_WAVES; ++w)
                if (sh.scost[w] < best) { best = sh.scost[w]; best_s = sh.ssplit[w]; }
            geom_finish(sh.g, sh.sp, best_s, force_split);
            sh.geom[slot] = sh.g;
            sh.geom_m[slot] = m;
        }
        __syncthreads();
    }
    return sh.geom[slot];
}

template <bool GUARD0, int MX>
__global__ void __launch_bounds__(RES_THREADS, 1)
    k_resident_loop(const int64_t N, const int64_t Npad, const double eps2, const double eta, const double dt_min,
                    const double dt_max, double *t, double *dt, double *mass, double *r, double *v, double *a,
                    double *j, double *s, double *c, double *jp, int32_t *active_list, double *f1, double *partials,
                    StepCtl *ctl, const int n_sm, const int occ, const int64_t partials_limit,
                    const int force_split, const int force_jlanes)
{
    extern __shared__ __align__(128) unsigned char res_smem[];
    ResShared &sh = *reinterpret_cast<ResShared *>(res_smem);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_cta = gridDim.x, rank = blockIdx.x;            // the grid is one cluster
    const int gwarp = rank * RES_WARPS + warp, gwarps = n_cta * RES_WARPS;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);

    if (tid == 0) {
        for (int q = 0; q < RES_VC; ++q) { mbar_init(&sh.full[q][0], 1); mbar_init(&sh.full[q][1], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int q = tid; q < RES_GEOM_SLOTS; q += RES_THREADS) sh.geom_m[q] = -1;
    __syncthreads();
    unsigned tc = 0;                // tiles consumed so far through this thread's ring
    volatile StepCtl *vctl = ctl;
#ifdef NB_RES_TIMING   // development aid: cycles per phase of the step, summed by one thread into unused histogram bins
    long long tph[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long tq = clock64();
#define NB_TICK(q) do { const long long now_ = clock64(); tph[q] += now_ - tq; tq = now_; } while (0)
#else
#define NB_TICK(q) do { } while (0)
#endif

    for (int p = 0;; p ^= 1) {
        // ---- phase 1: gather + predict.  Every thread of the cluster evaluates the same condition from
        // values that nothing modifies before the second barrier of the step.
        const double tn = __longlong_as_double((long long)vctl->tmin[p]);
        if (vctl->steps_left <= 0 || !(tn <= vctl->t_end)) break;
        NB_TICK(0);
        double vmin = inf;
        for (int64_t base = (int64_t)gwarp * 32; base < N; base += (int64_t)gwarps * 32) {   // warp-uniform trip count
            const int64_t i = base + lane;
            bool hit = false;
            if (i < N) {
                const double due = t[i] + dt[i];
                hit = (due == tn);
                if (!hit) vmin = fmin(vmin, due);
                predict_one(i, Npad, tn, t, mass, r, v, a, j, s, c, jp);
            }
            // warp-aggregated append (the order of the list affects no result, G18)
            const unsigned mask = __ballot_sync(0xffffffffu, hit);
            if (mask) {
                const int leader = __ffs(mask) - 1;
                int slot0 = 0;
                if (lane == leader) slot0 = atomicAdd(&ctl->cnt[p], __popc(mask));
                slot0 = __shfl_sync(0xffffffffu, slot0, leader);
                if (hit) active_list[slot0 + __popc(mask & ((1u << lane) - 1u))] = (int32_t)i;
            }
        }
        res_block_min_to(vmin, &ctl->tmin[1 - p], sh.red);
        NB_TICK(1);
        fence_proxy_async();          // the records just stored are read by bulk copies (async proxy) below
        cluster_sync_all();
        fence_proxy_async();
        NB_TICK(2);

        // ---- phase 2: evaluate
        const int m = vctl->cnt[p];
        const ForceGeom g = res_geometry(sh, m, Npad, n_sm, occ, partials_limit, force_split, force_jlanes);
        NB_TICK(3);
        const int32_t *active = (m == N) ? nullptr : active_list;
        double *out = g.S > 1 ? partials : f1;
        const PartLayout L = part_layout(g.S, g.mpad, Npad);
        const long long items = (long long)g.n_ib * g.S;
        {
            const int vc = tid / NT_E, vt = tid % NT_E;        // virtual CTA of 128 threads, named barrier 1 + vc
            const int tiles_total = (int)(Npad / TJ_E);
            for (long long w = (long long)rank * RES_VC + vc; w < items; w += (long long)n_cta * RES_VC)
                force_item_jl<NT_E, TJ_E, GUARD0, MX, 12, 2>(g.JL, jp, jp, active, m, (int)(w % g.n_ib), (int)(w / g.n_ib),
                                                             tiles_total, g.tps, eps2, out, L.cstride, L.kstride, L.sstride,
                                                             sh.tile[vc], sh.full[vc], tc, vt, 1 + vc);
        }
        NB_TICK(4);
        cluster_sync_all();
        NB_TICK(5);

        // ---- phase 3: reduce + correct, one warp per active particle; the sum over the splits runs in the
        // order every driver uses (part_layout, sum_splits_*), so that all agree bit for bit.
        vmin = inf;
        for (int k = gwarp; k < m; k += gwarps) {
            if (g.S > 1) reduce_one(partials, g.S, L, k, lane, f1, Npad);
            if (lane == 0) {
                const int64_t i = active ? active[k] : k;
                vmin = fmin(vmin, correct_one(k, i, Npad, tn, eta, dt_min, dt_max, f1, t, dt, r, v, a, j, s, c));
            }
        }
        res_block_min_to(vmin, &ctl->tmin[1 - p], sh.red);
        if (rank == 0 && tid == 0) {      // bookkeeping: fields nobody reads before the next barrier
            ctl->t_now = tn;
            ctl->t_next = tn;
            ctl->n_active = m;
            ctl->steps_left -= 1;
            ctl->n_steps += 1;
            ctl->n_pairs += (double)m * (double)N;
            int b = 0;
            while ((1LL << (b + 1)) <= (long long)m) ++b;
            ctl->hist[b] += 1;
            ctl->tmin[p] = 0x7ff0000000000000ULL;   // consumed: slot p collects the minimum of the step after next
            ctl->cnt[p] = 0;
        }
        NB_TICK(6);
        cluster_sync_all();
        NB_TICK(7);
    }
#ifdef NB_RES_TIMING
    if (rank == 0 && tid == 0)
        for (int q = 0; q < 8; ++q) ctl->hist[40 + q] += tph[q];
#endif
    if (rank == 0 && tid == 0) ctl->done = 1;
}

// ---- host side ---------------------------------------------------------------------------
template <bool G0, int MX>
static cudaError_t launch_resident(nb_ctx *ctx, int n_cta)
{
    auto kern = k_resident_loop<G0, MX>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ResShared));
    if (e != cudaSuccess) return e;
    if (n_cta > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_cta); cfg.blockDim = dim3(RES_THREADS);
    cfg.dynamicSmemBytes = sizeof(ResShared); cfg.stream = ctx->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)n_cta; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int n_clusters = 0;
    e = cudaOccupancyMaxActiveClusters(&n_clusters, kern, &cfg);
    if (e != cudaSuccess) return e;
    if (n_clusters < 1) return cudaErrorLaunchOutOfResources;
    return cudaLaunchKernelEx(&cfg, kern, ctx->N, ctx->Npad, ctx->eps2, ctx->eta, ctx->dt_min, ctx->dt_max, ctx->t, ctx->dt,
                              ctx->mass, ctx->r, ctx->v, ctx->a, ctx->j, ctx->s, ctx->c, ctx->jp, ctx->active, ctx->f1,
                              ctx->partials, ctx->ctl, ctx->n_sm, ctx->occ[0], (int64_t)ctx->partials_limit,
                              ctx->force_split, ctx->force_jlanes);
}

static cudaError_t launch_resident_any(nb_ctx *ctx, int n_cta)
{
    const bool mx = ctx->precision == 1;
    const bool g0 = mx ? (float)ctx->eps2 < 1e-24f : ctx->eps == 0.0;   // as in nb_force.cu
    if (g0 && mx) return launch_resident<true, 1>(ctx, n_cta);
    if (g0) return launch_resident<true, 0>(ctx, n_cta);
    if (mx) return launch_resident<false, 1>(ctx, n_cta);
    return launch_resident<false, 0>(ctx, n_cta);
}

// Advance while the next block time is <= t_end and fewer than max_steps steps were taken: one launch.
int resident_run(nb_ctx *ctx, double t_end, int64_t max_steps, int64_t *n_steps)
{
    if (ctx->N > RES_MAX_N)
        return set_err(ctx, NB_EINVAL, "loop mode 3 (cluster-resident loop) serves N <= %lld; this context has N = %lld",
                       (long long)RES_MAX_N, (long long)ctx->N);
    {
        const int rc = reserve_partials(ctx, ctx->partials_limit);
        if (rc != NB_OK) return rc;
    }
    {
        const int rc = launch_graph_begin(ctx, t_end, max_steps);   // seeds the control block and tmin[0]
        if (rc != NB_OK) return rc;
    }
    if (ctx->res_cluster == 0) ctx->res_cluster = 16;
    cudaError_t e = launch_resident_any(ctx, ctx->res_cluster);
    if (e != cudaSuccess && ctx->res_cluster > 8) {   // no 16-SM cluster on this part: the portable size
        cudaGetLastError();
        ctx->res_cluster = 8;
        e = launch_resident_any(ctx, 8);
    }
    if (e != cudaSuccess) return set_err(ctx, NB_ECUDA, "launch of k_resident_loop failed: %s", cudaGetErrorString(e));
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
