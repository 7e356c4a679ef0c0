// nb_force.cu -- the evaluation step: acceleration, jerk and snap of the active particles
// against all predicted particles.  PAPER.md:72-81 (Eq. 8-10) with the Eq. 2 softening
// in every r_ij^2 (reading G3); split over j when the active set is
// small (the paper's "Bfactor") followed by a fixed-order reduction of the
// partial sums (Table 1 row 4).
//
// The kernel is bound by the FP64 pipe: per pair it issues
// 32 DFMA + 11 DMUL + 10 DADD = 53 FP64 instructions (85 flops) and one MUFU.RSQ64H.
//   - one i-particle per lane (or per group of JL lanes when m is small), its nine
//     predicted values and nine accumulators held in registers;
//   - the j-stream is read as packed 80-byte records staged through shared memory by 1-D
//     bulk copies (cp.async.bulk -> UBLKCP, completion on an mbarrier), two stages deep,
//     issued by one thread; every lane then reads the same record (LDS.128 broadcast);
//   - 1/sqrt(s): hardware seed on the upper word (rsqrt.approx.ftz.f64 -> MUFU.RSQ64H,
//     ~2^-21) refined by ONE third-order FP64 step y <- y + y e (1/2 + 3/8 e), e = 1 - s y^2,
//     relative error < 2^-60 before rounding;
//   - sums are blocked: one partial per j-tile is added to the running total, so the
//     rounding error grows with sqrt(tile) + sqrt(#tiles) instead of sqrt(N).
#include <stdarg.h>
#include <stdio.h>

#include "nb_internal.cuh"
#include "nb_force_dev.cuh"

namespace nb {

// grid.x: i-blocks, grid.y: j-splits; geometry passed by the host.
template <int JL, bool GUARD0, int MX = 0, int UNR = 12>
__global__ void __launch_bounds__(NT_E, MINB_E)
    k_force(const double *__restrict__ jp, const double *__restrict__ jstream,
            const int32_t *__restrict__ active, const int m, const int tiles_total, const int tiles_per_split, const double eps2,
            double *__restrict__ out, const size_t cstride, const size_t kstride, const size_t sstride)
{
    __shared__ __align__(128) double tile[2][TJ_E * REC];
    __shared__ __align__(8) uint64_t full[2];
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned tc = 0;
    force_item<NT_E, TJ_E, JL, GUARD0, MX, UNR>(jp, jstream, active, m, blockIdx.x, blockIdx.y, tiles_total, tiles_per_split,
                                                eps2, out, cstride, kstride, sstride, tile, full, tc);
}

// Persistent form for the device-driven block-step loop (nb_graph.cu): a fixed grid of
// resident CTAs; the set size and the geometry are read from the control block, where the gather
// kernel of the same step left them.  CTA b starts with work item b and then draws the next one
// from a counter in the control block (items of one launch take equally long, but CTAs do not start
// together: a fixed stride left a 2 % tail at m ~ 2e5).  Item w is (i-block w % n_ib, split
// w / n_ib), so concurrently running CTAs stream the same j-split.
// The lane count of a step is known only on the device, so the kernel holds all six force_item instantiations.
// Inlined into one body they share one register allocation (122 registers: a fifth of the warps lost, and a cap of
// 96 costs the pair loop its operand-reuse order).  So only the throughput path (one i per lane) is inline; the five
// lane-sharing instantiations of the small sets are NON-INLINED device functions with their own allocation.  They find
// the tile ring in the dynamic shared memory of the kernel, so their loads stay LDS.
constexpr size_t PERSIST_RING = 2 * TJ_E * REC * sizeof(double);
constexpr size_t PERSIST_SMEM = PERSIST_RING + 2 * sizeof(uint64_t) + sizeof(long long);

template <int JL, bool GUARD0, int MX, int UNR>
__device__ __noinline__ unsigned persistent_item(const double *__restrict__ jp, const int32_t *__restrict__ active, const int m,
                                                 const int ib, const int sp, const int tiles_total, const int tps,
                                                 const double eps2, double *__restrict__ out, const size_t cstride,
                                                 const size_t kstride, const size_t sstride, unsigned tc)
{
    extern __shared__ __align__(128) unsigned char persist_smem[];
    double (*tile)[TJ_E * REC] = reinterpret_cast<double (*)[TJ_E * REC]>(persist_smem);
    uint64_t *full = reinterpret_cast<uint64_t *>(persist_smem + PERSIST_RING);
    force_item<NT_E, TJ_E, JL, GUARD0, MX, UNR>(jp, jp, active, m, ib, sp, tiles_total, tps, eps2, out, cstride, kstride,
                                                sstride, tile, full, tc);
    return tc;
}

template <bool GUARD0, int MX = 0, int UNR = 12>
__global__ void __launch_bounds__(NT_E, 5)
    k_force_persistent(const double *__restrict__ jp, const int32_t *__restrict__ active_list, const int64_t N,
                       const int64_t Npad, const double eps2, double *__restrict__ f1,
                       double *__restrict__ partials, StepCtl *__restrict__ ctl)
{
    pdl_trigger();
    pdl_wait();
    if (ctl->done) return;
    extern __shared__ __align__(128) unsigned char persist_smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(persist_smem + PERSIST_RING);
    long long *next_item = reinterpret_cast<long long *>(persist_smem + PERSIST_RING + 2 * sizeof(uint64_t));
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int m = (int)ctl->n_active;
    const ForceGeom g = ctl->g;
    const int32_t *active = (m == N) ? nullptr : active_list;
    double *out = g.S > 1 ? partials : f1;
    const PartLayout L = part_layout(g.S, g.mpad, Npad);
    const int tiles_total = (int)(Npad / TJ_E);
    const long long items = (long long)g.n_ib * g.S;
    unsigned tc = 0;
    long long w = blockIdx.x;
    while (w < items) {
        const int ib = (int)(w % g.n_ib), sp = (int)(w / g.n_ib);
#define NB_PI(J) tc = persistent_item<J, GUARD0, MX, UNR>(jp, active, m, ib, sp, tiles_total, g.tps, eps2, out, L.cstride, L.kstride, L.sstride, tc)
        switch (g.JL) {
            case 1:   // the throughput path stays inline: its pair loop keeps the schedule of k_force<1>
                force_item<NT_E, TJ_E, 1, GUARD0, MX, UNR>(jp, jp, active, m, ib, sp, tiles_total, g.tps, eps2, out, L.cstride,
                                                           L.kstride, L.sstride, reinterpret_cast<double (*)[TJ_E * REC]>(persist_smem),
                                                           full, tc);
                break;
            case 2: NB_PI(2); break;
            case 4: NB_PI(4); break;
            case 8: NB_PI(8); break;
            case 16: NB_PI(16); break;
            default: NB_PI(32); break;
        }
#undef NB_PI
        if (threadIdx.x == 0) *next_item = (long long)gridDim.x + atomicAdd(&ctl->work, 1u);
        __syncthreads();
        w = *next_item;
        __syncthreads();
    }
}

// ---- partial-sum reduction (Table 1 row 4): f1[c][k] = sum over the splits, fixed order (part_layout) ---
// fewer than 32 splits: one thread per element, coalesced along k
__global__ void k_reduce_thread(const double *__restrict__ part, const int S, const int m,
                                const size_t cstride, const size_t sstride, double *__restrict__ f1,
                                const size_t f1stride)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (k >= m) return;
    f1[c * f1stride + k] = sum_splits_thread(part + c * cstride + k, S, sstride);
}
// 32 splits or more: one warp per element, the S values of an element are consecutive
__global__ void k_reduce_warp(const double *__restrict__ part, const int S, const int m,
                              const size_t cstride, const size_t kstride, double *__restrict__ f1,
                              const size_t f1stride)
{
    const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wid >= 9 * m) return;
    const int c = wid / m, k = wid - c * m;
    const double acc = sum_splits_warp(part + c * cstride + (size_t)k * kstride, S, lane);
    if (lane == 0) f1[c * f1stride + k] = acc;
}

// f1[c][k] -> stage[q][k][3]  (q = 0 acc, 1 jerk, 2 snap), the caller-facing [n][3] layout
__global__ void k_unpack_f1(const double *__restrict__ f1, const size_t f1stride, const int m,
                            double *__restrict__ stage)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m) return;
#pragma unroll
    for (int c = 0; c < 9; ++c) {
        const int q = c / 3, d = c % 3;
        stage[((size_t)q * m + k) * 3 + d] = f1[c * f1stride + k];
    }
}

// ---- host side ---------------------------------------------------------------------------
// The split search never asks for more than MAX_WAVES work items per SM, i.e. S * n_ib <= MAX_WAVES x SMs items of
// at most NT_E slots each; S <= 65535 splits of mpad <= m + 31 add the slack term.
static size_t partials_bound(const nb_ctx *ctx)
{
    int64_t items = (int64_t)MAX_WAVES * ctx->n_sm * NT_E + 32 * 65536;
    const int64_t by_n = (ctx->Npad / TJ_E) * (ctx->Npad + 32);   // S <= tiles, mpad <= Npad + 32
    if (by_n < items) items = by_n;
    return (size_t)(9 * items);
}

int query_force_occupancy(nb_ctx *ctx)
{
    int v = 0;
    NB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_force<1, false>, NT_E, 0));
    ctx->occ[0] = v > 0 ? v : 1;
    NB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, k_force_persistent<false>, NT_E, PERSIST_SMEM));
    ctx->occ[1] = v > 0 ? v : 1;
    ctx->partials_limit = partials_bound(ctx);
    return NB_OK;
}

int reserve_partials(nb_ctx *ctx, size_t need)
{
    if (need <= ctx->partials_cap) return NB_OK;
    if (ctx->partials) { NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream)); cudaFree(ctx->partials); }
    ctx->partials = nullptr; ctx->partials_cap = 0;
    size_t cap = need + need / 2;
    if (cap > ctx->partials_limit) cap = ctx->partials_limit;
    if (cap < need) cap = need;
    NB_CUDA(ctx, cudaMalloc(&ctx->partials, cap * sizeof(double)));
    ctx->partials_cap = cap;
    return NB_OK;
}

// Mixed precision relies on the self term being w * 0 with a finite w = m eps^-3 in float: below
// eps^2 ~ 1e-24 that product overflows, so the self pair is then excluded by the guard variant.
static bool mx_needs_guard(const nb_ctx *ctx) { return (float)ctx->eps2 < 1e-24f; }

template <int JL>
static void launch_lanes(nb_ctx *ctx, dim3 grid, const int32_t *active, int m, int tiles_total, int tps,
                         double *out, const PartLayout &L, bool no_snap)
{
    const double *jstream = ctx->jp + (size_t)ctx->j_begin * REC;   // j-shard (nb_set_j_range), else the whole stream
#define NB_KF(G0, MXP)                                                                                              \
    k_force<JL, G0, MXP><<<grid, NT_E, 0, ctx->stream>>>(ctx->jp, jstream, active, m, tiles_total, tps, ctx->eps2, out, \
                                                          L.cstride, L.kstride, L.sstride)
    const int mx = ctx->precision == 1 ? 1 : (ctx->precision == 2 ? 3 : 0);   // kernel template value (force_item)
    const bool g0 = mx ? mx_needs_guard(ctx) : ctx->eps == 0.0;
    if (g0 && mx == 1) NB_KF(true, 1);
    else if (mx == 1) NB_KF(false, 1);
    else if (g0 && mx == 3) NB_KF(true, 3);
    else if (mx == 3) NB_KF(false, 3);
    else if (JL == 1 && no_snap) {     // start-up pass 1 of a large system; small ones take the full body (same a, jerk)
        if (g0) NB_KF(true, 2);
        else NB_KF(false, 2);
    } else if (g0) NB_KF(true, 0);
    else NB_KF(false, 0);
#undef NB_KF
}

int launch_force(nb_ctx *ctx, const int32_t *active, int64_t m, bool no_snap)
{
    if (m <= 0) return NB_OK;
    // records of the j-shard, padded to whole tiles (records N..Npad-1 have zero mass)
    const int64_t jlen = (ctx->j_end == ctx->N ? ctx->Npad : ctx->j_end) - ctx->j_begin;
    const ForceGeom g = choose_geom(m, jlen, ctx->n_sm, ctx->occ[0], (int64_t)ctx->partials_limit,
                                    ctx->force_split, ctx->force_jlanes);
    const int64_t tiles = jlen / TJ_E;
    double *out = ctx->f1;
    if (g.S > 1) {
        const int rc = reserve_partials(ctx, (size_t)g.S * 9 * (size_t)g.mpad);
        if (rc != NB_OK) return rc;
        out = ctx->partials;
    }
    const PartLayout L = part_layout(g.S, g.mpad, ctx->Npad);
    dim3 grid((unsigned)g.n_ib, (unsigned)g.S, 1);
    switch (g.JL) {
        case 1: launch_lanes<1>(ctx, grid, active, (int)m, (int)tiles, g.tps, out, L, no_snap); break;
        case 2: launch_lanes<2>(ctx, grid, active, (int)m, (int)tiles, g.tps, out, L, no_snap); break;
        case 4: launch_lanes<4>(ctx, grid, active, (int)m, (int)tiles, g.tps, out, L, no_snap); break;
        case 8: launch_lanes<8>(ctx, grid, active, (int)m, (int)tiles, g.tps, out, L, no_snap); break;
        case 16: launch_lanes<16>(ctx, grid, active, (int)m, (int)tiles, g.tps, out, L, no_snap); break;
        default: launch_lanes<32>(ctx, grid, active, (int)m, (int)tiles, g.tps, out, L, no_snap); break;
    }
    NB_LAUNCH_CHECK(ctx, "k_force");
    if (g.S > 1) {
        if (g.S < 32) {
            dim3 gr((unsigned)((m + 127) / 128), 9, 1);
            k_reduce_thread<<<gr, 128, 0, ctx->stream>>>(out, g.S, (int)m, L.cstride, L.sstride, ctx->f1, (size_t)ctx->Npad);
        } else {
            const int64_t warps = 9 * m;
            k_reduce_warp<<<(unsigned)((warps + 7) / 8), 256, 0, ctx->stream>>>(out, g.S, (int)m, L.cstride, L.kstride, ctx->f1, (size_t)ctx->Npad);
        }
        NB_LAUNCH_CHECK(ctx, "k_reduce");
    }
    ctx->last_launch[0] = NT_E; ctx->last_launch[1] = g.JL; ctx->last_launch[2] = g.S;
    ctx->last_launch[3] = (int64_t)g.n_ib * g.S; ctx->last_launch[4] = TJ_E;
    ctx->n_pairs += (double)m * (double)(ctx->j_end - ctx->j_begin);
    return NB_OK;
}

// Device-driven loop: one wave of resident CTAs; everything returns at once when the control block says `done`.
int enqueue_force_persistent(nb_ctx *ctx)
{
    const unsigned gP = (unsigned)(ctx->n_sm * ctx->occ[1]);
#define NB_KP(G0, MXP)                                                                                      \
    launch_chain(k_force_persistent<G0, MXP>, dim3(gP), dim3(NT_E), ctx->stream, pdl, PERSIST_SMEM, ctx->jp, ctx->active, \
                 ctx->N, ctx->Npad, ctx->eps2, ctx->f1, ctx->partials, ctx->ctl)
    const int mx = ctx->precision == 1 ? 1 : (ctx->precision == 2 ? 3 : 0);
    const bool pdl = ctx->use_graph == 2;
    const bool g0 = mx ? mx_needs_guard(ctx) : ctx->eps == 0.0;
    if (g0 && mx == 1) NB_KP(true, 1);
    else if (g0 && mx == 3) NB_KP(true, 3);
    else if (g0) NB_KP(true, 0);
    else if (mx == 1) NB_KP(false, 1);
    else if (mx == 3) NB_KP(false, 3);
    else NB_KP(false, 0);
#undef NB_KP
    NB_LAUNCH_CHECK(ctx, "k_force_persistent");
    return NB_OK;
}

// f1 planes (stride Npad) <-> contiguous [9][m] (the buffer a j-sharded caller all-reduces)
__global__ void k_f1_contig(double *__restrict__ f1, const size_t f1stride, const int m, double *__restrict__ buf,
                            const bool to_f1)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (k >= m) return;
    if (to_f1) f1[c * f1stride + k] = buf[(size_t)c * m + k];
    else buf[(size_t)c * m + k] = f1[c * f1stride + k];
}

int launch_f1_contig(nb_ctx *ctx, int64_t m, double *buf, bool to_f1)
{
    if (m <= 0) return NB_OK;
    dim3 g((unsigned)((m + 255) / 256), 9, 1);
    k_f1_contig<<<g, 256, 0, ctx->stream>>>(ctx->f1, (size_t)ctx->Npad, (int)m, buf, to_f1);
    NB_LAUNCH_CHECK(ctx, "k_f1_contig");
    return NB_OK;
}

int launch_unpack_f1(nb_ctx *ctx, int64_t m)
{
    if (m <= 0) return NB_OK;
    k_unpack_f1<<<(unsigned)((m + 255) / 256), 256, 0, ctx->stream>>>(ctx->f1, (size_t)ctx->Npad, (int)m, ctx->stage);
    NB_LAUNCH_CHECK(ctx, "k_unpack_f1");
    return NB_OK;
}

int set_err(nb_ctx *ctx, int code, const char *fmt, ...)
{
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

}  // namespace nb
