// nb_gridres.cu -- the block-step loop resident on the WHOLE GPU, state in shared memory (loop mode 4,
// 2048 < N <= GR_NL_MAX x SMs, i.e. about 10^5 particles on a B200).
//
// The cluster-resident loop (nb_resident.cu) removes the kernel boundaries and the trips to L2 from a small
// block step, but one cluster holds only 2048 particles.  The same idea on all SMs: ONE cooperative kernel of one
// CTA per SM, launched once per run of small block steps.  CTA b OWNS the particles [b NL, (b + 1) NL): their
// committed state (21 doubles each) and their predicted records stay in its shared memory.  What the cluster does
// through distributed shared memory goes through three small buffers in global memory (L2-resident) here, and the
// cluster barrier becomes a grid barrier (one atomic and one polled line per CTA).  A step needs only TWO of them:
//
//   publish   (end of the previous step) every CTA finds the minimum of t_i + dt_i over ITS particles and the
//             particles that attain it (its candidates), predicts those to that time (Eq. 3-7) and writes
//             {minimum, count} and the candidates' records to global memory                        -- barrier --
//   select    every CTA reads the 148 headers: t_next = the least minimum (Table 1 row 1); the
//             active set is the union of the candidate lists of the CTAs whose minimum equals t_next -- their
//             records are already predicted to exactly that time.  No second exchange is needed.
//   predict   the owned particles to t_next (Eq. 3-7), into shared memory
//   evaluate  ALL m active particles against the OWNED records (Eq. 8-10; the paper's split of the j-range,
//             PAPER.md:108-114, one split per SM); partial (a, jerk, snap) to global memory        -- barrier --
//   correct   the owner sums the partials of each of its active particles over the CTAs in the fixed order of
//             sum_splits_warp, applies Eq. 11-16 (correct_warp), then publishes again.
//
// Large block steps stay with the streaming kernels: when the next step has m >= m_big active particles the kernel
// writes the state back and returns, the host runs that ONE step as nb_next_block -> nb_predict -> nb_force ->
// nb_correct_and_step (k_force at full occupancy; a step of that size is milliseconds, the switch ~50 us) and
// launches the kernel again.
//
// Arithmetic: pair_body, predict_one, correct_warp, new_dt of the other drivers.  The summation order of a small
// step is this loop's own (per lane over the owner's slice, butterfly over the lanes that share the i, then over
// the CTAs), fixed, so runs are bit-reproducible; it agrees with the other drivers to rounding (G18, G29).
#include "nb_internal.cuh"
#include "nb_resident_dev.cuh"

namespace nb {

constexpr int GR_THREADS = 512;
constexpr int GR_WARPS = GR_THREADS / 32;
constexpr int GR_MAXG = 192;          // CTAs (SMs) at most
constexpr int GR_NL_MAX = 704;        // owned particles per CTA at most (40 doubles + 4 bytes each in shared memory)

struct __align__(16) GrHdr {          // what a CTA publishes: its minimum of t_i + dt_i and how many particles attain it
    double tmin;
    int cnt, pad;
};

// Shared-memory plan of one CTA (NL = owned particles, a multiple of 32; doubles unless noted):
//   t, dt, mass [NL]; r, v, a, jerk, snap, crackle [3][NL]; rec [NL][REC]; f1 [9][NL] (reduced forces of the owned
//   active particles); list int32 [NL] (local indices of the candidates); htmin [G], hcnt int32 [G] (the headers);
//   base int32 [G + 1] (first slot of every CTA's candidates in the active list)
struct GridPlan {
    int NL, G;
    size_t o_t, o_dt, o_m, o_r, o_v, o_a, o_j, o_s, o_c, o_rec, o_f1, o_list, o_htmin, o_hcnt, o_base, bytes;
};
__host__ __device__ inline GridPlan grid_plan(const int64_t N, const int G)
{
    GridPlan p;
    p.G = G;
    int NL = (int)((N + G - 1) / G);
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
    p.o_htmin = o; o += (size_t)GR_MAXG * 8;
    p.o_list = o; o += (size_t)NL * 4;
    p.o_hcnt = o; o += (size_t)GR_MAXG * 4;
    p.o_base = o; o += (size_t)(GR_MAXG + 1) * 4;
    p.bytes = (o + 15) & ~(size_t)15;
    return p;
}

struct GridArgs {
    int64_t N, Npad;
    double eps2, eta, dt_min, dt_max;
    double *g_t, *g_dt;
    const double *g_m;
    double *g_r, *g_v, *g_a, *g_j, *g_s, *g_c, *g_jp;
    StepCtl *ctl;
    GrHdr *hdr;                 // [G]
    double *cand;               // [G][NL][REC] candidates' predicted records
    double *part;               // [m_big][9][G] partial sums of the active particles, one value per CTA
    unsigned long long *bar;    // grid barrier counter, zero at launch
    int32_t *active;            // the scheduler's list and its pinned mirror: filled when a large step is handed
    Sched *sched;               // to the call sequence, which then needs no search of its own
    double t_end;
    long long steps;            // step budget of this launch
    int m_big, force_jlanes;
};

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// All CTAs of the (cooperative, co-resident) grid.  The counter only grows: the k-th barrier waits for k G arrivals.
// Release / acquire at GPU scope: the block barrier orders this CTA's writes before thread 0's releasing add (which
// is cumulative), and thread 0's acquiring load before every later read of the CTA.
__device__ __forceinline__ void grid_barrier(unsigned long long *bar, unsigned long long &target, const int G)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        target += (unsigned long long)G;
        asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(bar) : "memory");
        while (ld_acquire_u64(bar) < target) { }
    }
    __syncthreads();
}

template <bool GUARD0, int MX>
__global__ void __launch_bounds__(GR_THREADS, 1) k_grid_loop(const GridArgs A)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = (int)gridDim.x, rank = (int)blockIdx.x;
    const GridPlan P = grid_plan(A.N, G);
    const int NL = P.NL;
    double *t = (double *)(smem + P.o_t), *dt = (double *)(smem + P.o_dt), *mass = (double *)(smem + P.o_m);
    double *r = (double *)(smem + P.o_r), *v = (double *)(smem + P.o_v), *a = (double *)(smem + P.o_a);
    double *j = (double *)(smem + P.o_j), *s = (double *)(smem + P.o_s), *c = (double *)(smem + P.o_c);
    double *rec = (double *)(smem + P.o_rec), *f1 = (double *)(smem + P.o_f1), *htmin = (double *)(smem + P.o_htmin);
    int *list = (int *)(smem + P.o_list), *base = (int *)(smem + P.o_base), *hcnt = (int *)(smem + P.o_hcnt);
    __shared__ int n_list;
    __shared__ int ctot[GR_MAXG / 32];
    __shared__ double red[GR_WARPS], rest[GR_WARPS];
    __shared__ unsigned long long moved_min;   // bits of the least t_i + dt_i among the particles corrected in this step
    __shared__ long long hist[64];
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const int64_t N = A.N, Npad = A.Npad;
    const int64_t first = (int64_t)rank * NL;
    const int64_t left = N - first;
    const int n_own = left <= 0 ? 0 : (left < NL ? (int)left : NL);
    double *my_cand = A.cand + (size_t)rank * NL * REC;

    // ---- load the owned slice (rows beyond N: mass 0 at the origin, never due)
    for (int i = tid; i < NL; i += GR_THREADS) {
        const bool live = i < n_own;
        const int64_t gi = first + i;
        t[i] = live ? A.g_t[gi] : 0.0; dt[i] = live ? A.g_dt[gi] : inf; mass[i] = live ? A.g_m[gi] : 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int64_t gq = d * Npad + gi;
            const int q = d * NL + i;
            r[q] = live ? A.g_r[gq] : 0.0; v[q] = live ? A.g_v[gq] : 0.0; a[q] = live ? A.g_a[gq] : 0.0;
            j[q] = live ? A.g_j[gq] : 0.0; s[q] = live ? A.g_s[gq] : 0.0; c[q] = live ? A.g_c[gq] : 0.0;
        }
#pragma unroll
        for (int d = 0; d < REC; ++d) rec[i * REC + d] = 0.0;
    }
    for (int b = tid; b < 64; b += GR_THREADS) hist[b] = 0;
    long long steps_left = A.steps;
    const double t_end = A.t_end;
    long long n_steps = 0;
    double n_pairs = 0.0, t_now = 0.0;
    unsigned long long bar_target = 0;
    int reason = 1;
    double tn_last = 0.0;
    __syncthreads();

    // publish: the minimum vmin of t_i + dt_i over the owned particles is known to every thread; the particles that
    // attain it (list), their records predicted to that time -> global memory, for every CTA to read after the barrier
    auto publish_at = [&](const double vmin) {
        for (int i = tid; i < n_own; i += GR_THREADS)
            if (t[i] + dt[i] == vmin) {
                const int q = atomicAdd(&n_list, 1);
                list[q] = i;
                // record of particle i at time vmin -> slot q of this CTA's candidates (predict_one writes to
                // out + i REC); rec keeps the prediction of the step just taken
                predict_one(i, NL, vmin, t, mass, r, v, a, j, s, c, my_cand + ((int64_t)q - i) * REC);
            }
        __syncthreads();
        if (tid == 0) { GrHdr h; h.tmin = vmin; h.cnt = n_list; h.pad = 0; A.hdr[rank] = h; }
    };
    // at the start: the minimum over all owned particles
    auto publish_first = [&]() {
        double vmin = inf;
        for (int i = tid; i < n_own; i += GR_THREADS) vmin = fmin(vmin, t[i] + dt[i]);
        for (int off = 16; off > 0; off >>= 1) vmin = fmin(vmin, __shfl_xor_sync(0xffffffffu, vmin, off));
        if (lane == 0) red[warp] = vmin;
        if (tid == 0) n_list = 0;
        __syncthreads();
        vmin = lane < GR_WARPS ? red[lane] : inf;
        for (int off = 16; off > 0; off >>= 1) vmin = fmin(vmin, __shfl_xor_sync(0xffffffffu, vmin, off));
        publish_at(vmin);
    };
    // after a step in which this CTA corrected particles (block barrier passed): the particles that were not due
    // (rest[], from before the evaluation) and the corrected ones (moved_min)
    auto publish_owner = [&]() {
        double vmin = lane < GR_WARPS ? rest[lane] : inf;
        for (int off = 16; off > 0; off >>= 1) vmin = fmin(vmin, __shfl_xor_sync(0xffffffffu, vmin, off));
        vmin = fmin(vmin, __longlong_as_double((long long)moved_min));
        publish_at(vmin);
    };
    publish_first();
    grid_barrier(A.bar, bar_target, G);
#ifdef NB_GR_TIMING   // development aid: cycles per phase of the steps with m < 64, summed by one thread into unused histogram bins
    long long tph[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tcur[8];
    long long tq = clock64();
#define NB_TICK(q) do { const long long now_ = clock64(); tcur[q] = now_ - tq; tq = now_; } while (0)
#else
#define NB_TICK(q) do { } while (0)
#endif

    for (;;) {
        // ---- select: every CTA computes the same next block time and the same slot offsets from the headers
        for (int b = tid; b < G; b += GR_THREADS) {   // one 16-byte load per header
            const longlong2 w = __ldcg(reinterpret_cast<const longlong2 *>(A.hdr + b));
            htmin[b] = __longlong_as_double(w.x);
            hcnt[b] = (int)(w.y & 0xffffffffLL);
        }
        __syncthreads();
        double tn = inf;
        for (int b = lane; b < G; b += 32) tn = fmin(tn, htmin[b]);
        for (int off = 16; off > 0; off >>= 1) tn = fmin(tn, __shfl_xor_sync(0xffffffffu, tn, off));
        // exclusive prefix of the counts of the CTAs whose minimum is t_next: warp w scans the 32 CTAs of chunk w,
        // then every entry adds the totals of the chunks before its own
        if (warp < GR_MAXG / 32) {
            const int b = warp * 32 + lane;
            const int cnt = (b < G && htmin[b] == tn) ? hcnt[b] : 0;
            int inc = cnt;
            for (int off = 1; off < 32; off <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, inc, off);
                if (lane >= off) inc += y;
            }
            if (b < G) base[b] = inc - cnt;
            if (lane == 31) ctot[warp] = inc;
        }
        __syncthreads();
        {
            int before = 0, total = 0;
#pragma unroll
            for (int w = 0; w < GR_MAXG / 32; ++w) {
                const int cw = ctot[w];
                if (w < (tid >> 5)) before += cw;
                total += cw;
            }
            if (tid < G) base[tid] += before;      // tid >> 5 is the chunk of entry tid
            if (tid == 0) base[G] = total;
        }
        __syncthreads();
        const int m = base[G];
        NB_TICK(0);
        if (steps_left <= 0 || !(tn <= t_end)) { reason = 1; break; }
        if (m >= A.m_big) { reason = 2; tn_last = tn; break; }   // a large step: the streaming kernels take it

        // lanes per i and the record of this thread's first slot: the load from the candidates buffer is issued
        // before the predictor so that its trip to L2 overlaps it
        int lj = 0;                                             // JL = 2^lj lanes per i: shifts, not divisions, below
        if (A.force_jlanes >= 1) { const int want = A.force_jlanes < JL_MAX ? A.force_jlanes : JL_MAX; while ((2 << lj) <= want) ++lj; }
        else { while ((2 << lj) <= JL_MAX && (m << (lj + 1)) <= GR_THREADS) ++lj; }
        const int JL = 1 << lj;
        const int slots = GR_THREADS >> lj;
        auto load_slot = [&](const int k0, double2 (&w)[REC / 2]) {
            const int k = k0 + (tid >> lj);
            const int kk = k < m ? k : m - 1;
            int lo = 0, hi = G - 1;                             // owner: the last CTA with base[o] <= kk (ties: the non-empty one)
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (base[mid] <= kk) lo = mid; else hi = mid - 1;
            }
            const double2 *src = reinterpret_cast<const double2 *>(A.cand + ((size_t)lo * NL + (kk - base[lo])) * REC);
#pragma unroll
            for (int d = 0; d < REC / 2; ++d) w[d] = __ldcg(src + d);
        };
        double2 w0[REC / 2];
        const bool first_live = ((tid & ~31) >> lj) < m;           // this warp has a live slot in the first round
        if (first_live) load_slot(0, w0);

        // ---- predict the owned particles (Eq. 3-7); on the way, the minimum of t_i + dt_i over the particles that are
        // NOT due now (it cannot change in this step): the owners' next publish starts from it
        {
            double vr = inf;
            for (int i = tid; i < n_own; i += GR_THREADS) {
                predict_one(i, NL, tn, t, mass, r, v, a, j, s, c, rec);
                const double x = t[i] + dt[i];
                if (x != tn) vr = fmin(vr, x);
            }
            for (int off = 16; off > 0; off >>= 1) vr = fmin(vr, __shfl_xor_sync(0xffffffffu, vr, off));
            if (lane == 0) rest[warp] = vr;
            if (tid == 0) { moved_min = 0x7ff0000000000000ULL; n_list = 0; }   // for the publish of this step
        }
        __syncthreads();
        NB_TICK(1);

        // ---- evaluate all m active particles against the owned records; one partial per CTA and component
        for (int k0 = 0; k0 < m; k0 += slots) {                 // warp-uniform trip count
            if (k0 + ((tid & ~31) >> lj) >= m) continue;           // a warp without a live slot has nothing to add
            const int k = k0 + (tid >> lj), jl = tid & (JL - 1);
            const bool live = k < m;
            if (k0 > 0) load_slot(k0, w0);
            double ri[REC];
#pragma unroll
            for (int d = 0; d < REC / 2; ++d) { ri[2 * d] = w0[d].x; ri[2 * d + 1] = w0[d].y; }
            Acc9 T;
            switch (JL) {
                case 1: T = res_eval<1, GUARD0, MX>(ri, rec, jl, NL, A.eps2); break;
                case 2: T = res_eval<2, GUARD0, MX>(ri, rec, jl, NL, A.eps2); break;
                case 4: T = res_eval<4, GUARD0, MX>(ri, rec, jl, NL, A.eps2); break;
                case 8: T = res_eval<8, GUARD0, MX>(ri, rec, jl, NL, A.eps2); break;
                case 16: T = res_eval<16, GUARD0, MX>(ri, rec, jl, NL, A.eps2); break;
                default: T = res_eval<32, GUARD0, MX>(ri, rec, jl, NL, A.eps2); break;
            }
            if (live && jl == 0) {
                double *dst = A.part + (size_t)k * 9 * G + rank;
                dst[0 * G] = T.ax; dst[1 * G] = T.ay; dst[2 * G] = T.az; dst[3 * G] = T.jx; dst[4 * G] = T.jy;
                dst[5 * G] = T.jz; dst[6 * G] = T.sx; dst[7 * G] = T.sy; dst[8 * G] = T.sz;
            }
        }
        NB_TICK(2);
        grid_barrier(A.bar, bar_target, G);
        NB_TICK(3);

        // ---- correct: the owner sums the G partials of each of its active particles (lane-strided, ascending,
        // then the xor butterfly: the order of sum_splits_warp) and applies Eq. 11-16 (one warp per particle).
        const int n_mine = (htmin[rank] == tn) ? base[rank + 1] - base[rank] : 0;
        // the sums: one warp per (particle, component), so that all loads of a sum are in flight together (one trip
        // to L2 instead of one per 32 CTAs); the additions and their order are those of sum_splits_warp
        for (int it = warp; it < n_mine * 9; it += GR_WARPS) {
            const int q = it / 9, cc = it - q * 9;
            const double *p0 = A.part + ((size_t)(base[rank] + q) * 9 + cc) * G;
            double vv[GR_MAXG / 32];
#pragma unroll
            for (int u = 0; u < GR_MAXG / 32; ++u) {
                const int sidx = lane + 32 * u;
                vv[u] = sidx < G ? __ldcg(p0 + sidx) : 0.0;
            }
            double x = 0.0;
#pragma unroll
            for (int u = 0; u < GR_MAXG / 32; ++u) x += vv[u];
            for (int off = 16; off > 0; off >>= 1) x += __shfl_xor_sync(0xffffffffu, x, off);
            if (lane == 0) f1[cc * NL + q] = x;
        }
        __syncthreads();
        for (int q = warp; q < n_mine; q += GR_WARPS) {
            const int i = list[q];
            correct_warp(lane, q, i, NL, tn, A.eta, A.dt_min, A.dt_max, f1, t, dt, r, v, a, j, s, c);
            // times are non-negative dyadic rationals: the bit pattern orders like the value
            if (lane == 0) atomicMin(&moved_min, (unsigned long long)__double_as_longlong(t[i] + dt[i]));
        }
        __syncthreads();
        NB_TICK(4);
        steps_left -= 1; n_steps += 1; n_pairs += (double)m * (double)N; t_now = tn;
        if (tid == 0) {
            int b = 0;
            while ((1LL << (b + 1)) <= (long long)m) ++b;
            hist[b] += 1;
        }
        if (n_mine > 0) publish_owner();   // nothing of a CTA without active particles changed: its header and candidates stand
        NB_TICK(5);
        grid_barrier(A.bar, bar_target, G);
        NB_TICK(6);
#ifdef NB_GR_TIMING
        if (m < 64) { for (int q = 0; q < 7; ++q) tph[q] += tcur[q]; tph[7] += 1; }
#endif
    }
#ifdef NB_GR_TIMING
    if (rank == 0 && tid == 0)
        for (int q = 0; q < 8; ++q) hist[40 + q] += tph[q];
    __syncthreads();
#endif

    // ---- a large step is next: its block time and active list go where nb_next_block would have put them
    // (owner-major order; no result depends on the order of the list, G18)
    if (reason == 2) {
        if (htmin[rank] == tn_last) {
            const int b0 = base[rank], cnt = base[rank + 1] - b0;
            for (int q = tid; q < cnt; q += GR_THREADS) A.active[b0 + q] = (int32_t)(first + list[q]);
        }
        if (rank == 0 && tid == 0) { A.sched->t_next = tn_last; A.sched->n_active = base[G]; }
    }

    // ---- write the owned slice back: committed state and (if a step was taken) the last prediction
    __syncthreads();
    for (int i = tid; i < n_own; i += GR_THREADS) {
        const int64_t gi = first + i;
        A.g_t[gi] = t[i]; A.g_dt[gi] = dt[i];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int64_t gq = d * Npad + gi;
            const int q = d * NL + i;
            A.g_r[gq] = r[q]; A.g_v[gq] = v[q]; A.g_a[gq] = a[q]; A.g_j[gq] = j[q]; A.g_s[gq] = s[q]; A.g_c[gq] = c[q];
        }
    }
    if (n_steps > 0) {   // the predicted stream of the last step taken
        for (int i = tid; i < n_own; i += GR_THREADS) {
#pragma unroll
            for (int d = 0; d < REC; ++d) A.g_jp[(first + i) * REC + d] = rec[i * REC + d];
        }
    }
    if (rank == 0 && tid == 0) {
        A.ctl->steps_left = steps_left; A.ctl->n_steps = n_steps; A.ctl->n_pairs = n_pairs; A.ctl->t_now = t_now;
        for (int b = 0; b < 64; ++b) A.ctl->hist[b] = hist[b];
        A.ctl->done = reason;
    }
}

// ---- host side ---------------------------------------------------------------------------
template <bool G0, int MX>
static cudaError_t launch_grid(nb_ctx *ctx, const GridArgs &args, int G, size_t bytes)
{
    auto kern = k_grid_loop<G0, MX>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, GR_THREADS, bytes);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    void *params[] = {(void *)&args};
    return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)G), dim3(GR_THREADS), params, bytes, ctx->stream);
}

bool gridres_fits(const nb_ctx *ctx)
{
    const int G = ctx->n_sm < GR_MAXG ? ctx->n_sm : GR_MAXG;
    return ctx->N > 0 && (ctx->N + G - 1) / G <= GR_NL_MAX;
}

void gridres_release(nb_ctx *ctx)
{
    if (ctx->gr_hdr) cudaFree(ctx->gr_hdr);
    if (ctx->gr_cand) cudaFree(ctx->gr_cand);
    if (ctx->gr_part) cudaFree(ctx->gr_part);
    if (ctx->gr_bar) cudaFree(ctx->gr_bar);
    ctx->gr_hdr = nullptr; ctx->gr_cand = nullptr; ctx->gr_part = nullptr; ctx->gr_bar = nullptr;
}

static int gridres_reserve(nb_ctx *ctx, int G, int NL)
{
    if (ctx->gr_hdr && ctx->gr_m_big_alloc == ctx->gr_m_big) return NB_OK;
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    gridres_release(ctx);
    NB_CUDA(ctx, cudaMalloc(&ctx->gr_hdr, (size_t)G * sizeof(GrHdr)));
    NB_CUDA(ctx, cudaMalloc((void **)&ctx->gr_cand, (size_t)G * NL * REC * sizeof(double)));
    NB_CUDA(ctx, cudaMalloc((void **)&ctx->gr_part, (size_t)ctx->gr_m_big * 9 * G * sizeof(double)));
    NB_CUDA(ctx, cudaMalloc((void **)&ctx->gr_bar, sizeof(unsigned long long)));
    ctx->gr_m_big_alloc = ctx->gr_m_big;
    return NB_OK;
}

// Advance while the next block time is <= t_end and fewer than max_steps steps were taken: small steps in the
// grid-resident kernel, a large one (m >= gr_m_big) through the host-issued call sequence, and so on.
int gridres_run(nb_ctx *ctx, double t_end, int64_t max_steps, int64_t *n_steps)
{
    if (!gridres_fits(ctx))
        return set_err(ctx, NB_EINVAL, "loop mode 4 (grid-resident loop) serves N <= %lld on this device; this context has N = %lld",
                       (long long)GR_NL_MAX * (ctx->n_sm < GR_MAXG ? ctx->n_sm : GR_MAXG), (long long)ctx->N);
    const int G = ctx->n_sm < GR_MAXG ? ctx->n_sm : GR_MAXG;
    const GridPlan P = grid_plan(ctx->N, G);
    if (ctx->gr_m_big < 1) ctx->gr_m_big = GR_M_BIG_DEFAULT;
    {
        const int rc = gridres_reserve(ctx, G, P.NL);
        if (rc != NB_OK) return rc;
    }
    const int mx = ctx->precision == 1 ? 1 : (ctx->precision == 2 ? 3 : 0);
    const bool g0 = mx ? (float)ctx->eps2 < 1e-24f : ctx->eps == 0.0;   // as in nb_force.cu
    int64_t total = 0;
    for (;;) {
        NB_CUDA(ctx, cudaMemsetAsync(ctx->gr_bar, 0, sizeof(unsigned long long), ctx->stream));
        GridArgs A;
        A.N = ctx->N; A.Npad = ctx->Npad; A.eps2 = ctx->eps2; A.eta = ctx->eta; A.dt_min = ctx->dt_min; A.dt_max = ctx->dt_max;
        A.g_t = ctx->t; A.g_dt = ctx->dt; A.g_m = ctx->mass; A.g_r = ctx->r; A.g_v = ctx->v; A.g_a = ctx->a; A.g_j = ctx->j;
        A.g_s = ctx->s; A.g_c = ctx->c; A.g_jp = ctx->jp; A.ctl = ctx->ctl; A.hdr = (GrHdr *)ctx->gr_hdr; A.cand = ctx->gr_cand;
        A.part = ctx->gr_part; A.bar = ctx->gr_bar; A.m_big = ctx->gr_m_big; A.force_jlanes = ctx->force_jlanes;
        A.active = ctx->active; A.sched = ctx->d_sched; A.t_end = t_end; A.steps = (long long)(max_steps - total);
        cudaError_t e;
        if (g0 && mx == 1) e = launch_grid<true, 1>(ctx, A, G, P.bytes);
        else if (g0 && mx == 3) e = launch_grid<true, 3>(ctx, A, G, P.bytes);
        else if (g0) e = launch_grid<true, 0>(ctx, A, G, P.bytes);
        else if (mx == 1) e = launch_grid<false, 1>(ctx, A, G, P.bytes);
        else if (mx == 3) e = launch_grid<false, 3>(ctx, A, G, P.bytes);
        else e = launch_grid<false, 0>(ctx, A, G, P.bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            if (ctx->loop_auto) {   // this device cannot co-schedule the grid: the default falls back to the graph-driven loop
                ctx->use_graph = 1;
                int64_t rest = 0;
                const int rc = graph_run(ctx, t_end, max_steps - total, &rest);
                if (n_steps) *n_steps = total + rest;
                return rc;
            }
            return set_err(ctx, NB_ECUDA, "launch of k_grid_loop failed: %s", cudaGetErrorString(e));
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
        total += h->n_steps;
        if (h->done != 2) break;
        // the large step that stopped the kernel: its block is already selected (t_next, list) -- straight to
        // predict, evaluate, correct
        ctx->t_next = ctx->h_sched->t_next;
        ctx->n_active = (int64_t)ctx->h_sched->n_active;
        ctx->have_block = true;
        bool stepped = false;
        const int rc = host_block_step(ctx, t_end, &stepped);
        if (rc != NB_OK) return rc;
        if (!stepped) break;
        total += 1;
        if (total >= max_steps) break;
    }
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (n_steps) *n_steps = total;
    return NB_OK;
}

}  // namespace nb
