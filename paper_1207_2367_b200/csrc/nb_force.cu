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

namespace nb {

struct Acc9 {
    double ax, ay, az, jx, jy, jz, sx, sy, sz;
};

__device__ __forceinline__ double rsqrt_seed(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    return y;
}

// One pair interaction, Eq. 8-10 in the factored form:
//   s = |dr|^2 + eps^2, w = m_j s^(-3/2), g = -3 (dr.dv)/s, b3 = -3 beta,
//   u = dv + g dr,  A0 = w dr,  A1 = w u,  A2 = w (da + 2 g u + b3 dr).
// q points at the packed record {x y z vx vy vz ax ay az m} of particle j in shared memory.
// SNAP = false (start-up pass 1, G8: only a and jerk are wanted; the snap of that pass would be
// discarded): the a_ij differences, r.a, beta and the snap accumulation are left out -- 31 instead
// of 53 FP64 instructions; a and jerk are computed by the same expressions.
template <bool GUARD0, bool SNAP = true>
__device__ __forceinline__ void pair_body(const double xi, const double yi, const double zi,
                                          const double vxi, const double vyi, const double vzi,
                                          const double axi, const double ayi, const double azi,
                                          const double *__restrict__ q, const double eps2, Acc9 &A)
{
    const double2 p0 = *reinterpret_cast<const double2 *>(q);
    const double2 p1 = *reinterpret_cast<const double2 *>(q + 2);
    const double2 p2 = *reinterpret_cast<const double2 *>(q + 4);
    const double2 p3 = *reinterpret_cast<const double2 *>(q + 6);
    const double2 p4 = *reinterpret_cast<const double2 *>(q + 8);
    // differences and the three dot products, component by component (z, y, x)
    const double dvz = p2.y - vzi, dvy = p2.x - vyi, dvx = p1.y - vxi;
    double vr = dvz * dvz;
    vr = fma(dvy, dvy, vr);
    vr = fma(dvx, dvx, vr);
    const double dz = p1.x - zi, daz = p4.x - azi;
    double s = fma(dz, dz, eps2);
    double rv = dz * dvz;
    vr = fma(dz, daz, vr);
    const double dy = p0.y - yi, day = p3.y - ayi;
    s = fma(dy, dy, s);
    rv = fma(dy, dvy, rv);
    vr = fma(dy, day, vr);
    const double dx = p0.x - xi, dax = p3.x - axi;
    s = fma(dx, dx, s);
    rv = fma(dx, dvx, rv);
    vr = fma(dx, dax, vr);
    const double mj = p4.y;
    double y0 = rsqrt_seed(s);
    if (GUARD0) {  // eps = 0: a coincident pair (the self term) contributes nothing (G12)
        if ((__double2hiint(s) | __double2loint(s)) == 0) y0 = 0.0;
    }
    // y = y0 (1 + e (1/2 + 3/8 e)), e = 1 - s y0^2: every instruction reads at most two registers
    const double y2 = y0 * y0;
    const double e = fma(-s, y2, 1.0);
    const double p = fma(e, 0.375, 0.5);
    const double ep1 = fma(e, p, 1.0);
    const double y = y0 * ep1;         // s^(-1/2)
    const double ri2 = y * y;          // 1/s
    const double my = mj * y;
    const double qq = ri2 * -3.0;
    const double w = my * ri2;         // m_j s^(-3/2)
    const double g = rv * qq;          // -3 alpha
    const double qv = qq * vr;
    const double gg = g * g;
    const double g2 = g + g;
    const double b3 = fma(gg, -1.0 / 3.0, qv);  // -3 beta = -3 (v^2 + r.a)/s - 3 alpha^2
    const double ux = fma(g, dx, dvx), uy = fma(g, dy, dvy), uz = fma(g, dz, dvz);
    A.ax = fma(w, dx, A.ax);
    A.ay = fma(w, dy, A.ay);
    A.az = fma(w, dz, A.az);
    A.jx = fma(w, ux, A.jx);
    A.jy = fma(w, uy, A.jy);
    A.jz = fma(w, uz, A.jz);
    if (!SNAP) return;  // everything that only feeds the snap above is dead code in this instantiation
    double tx = fma(g2, ux, dax), ty = fma(g2, uy, day), tz = fma(g2, uz, daz);
    tx = fma(b3, dx, tx);
    ty = fma(b3, dy, ty);
    tz = fma(b3, dz, tz);
    A.sx = fma(w, tx, A.sx);
    A.sy = fma(w, ty, A.sy);
    A.sz = fma(w, tz, A.sz);
}

// The same pair in the paper's mixed precision (reading G27): the nine
// differences are formed in double from the double records and rounded to float, everything
// else of Eq. 8-10 is float arithmetic (FFMA/FMUL on the FP32 pipe, MUFU.RSQ), and the pair
// terms are summed in float within one j-tile (the caller adds the tile sums in double).
// FP64-pipe work per pair: 9 DADD + 10 F2F instead of 53 instructions.
struct AccF {
    float ax, ay, az, jx, jy, jz, sx, sy, sz;
};
template <bool GUARD0>
__device__ __forceinline__ void pair_body_mx(const double xi, const double yi, const double zi,
                                             const double vxi, const double vyi, const double vzi,
                                             const double axi, const double ayi, const double azi,
                                             const double *__restrict__ q, const float eps2, AccF &A)
{
    const double2 p0 = *reinterpret_cast<const double2 *>(q);
    const double2 p1 = *reinterpret_cast<const double2 *>(q + 2);
    const double2 p2 = *reinterpret_cast<const double2 *>(q + 4);
    const double2 p3 = *reinterpret_cast<const double2 *>(q + 6);
    const double2 p4 = *reinterpret_cast<const double2 *>(q + 8);
    const float dx = (float)(p0.x - xi), dy = (float)(p0.y - yi), dz = (float)(p1.x - zi);
    const float dvx = (float)(p1.y - vxi), dvy = (float)(p2.x - vyi), dvz = (float)(p2.y - vzi);
    const float dax = (float)(p3.x - axi), day = (float)(p3.y - ayi), daz = (float)(p4.x - azi);
    const float mj = (float)p4.y;
    const float s = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
    const float rv = fmaf(dx, dvx, fmaf(dy, dvy, dz * dvz));
    const float vr = fmaf(dx, dax, fmaf(dy, day, fmaf(dz, daz, fmaf(dvx, dvx, fmaf(dvy, dvy, dvz * dvz)))));
    float y = rsqrtf(s);
    if (GUARD0) {  // eps = 0: the self term (s = 0) contributes nothing (G12)
        if (s == 0.0f) y = 0.0f;
    }
    const float P = y * y;             // 1/s
    const float w = (mj * y) * P;      // m_j s^(-3/2)
    const float qq = -3.0f * P;
    const float g = rv * qq;           // -3 alpha
    const float b3 = fmaf(g * g, -1.0f / 3.0f, qq * vr);  // -3 beta
    const float g2 = g + g;
    const float ux = fmaf(g, dx, dvx), uy = fmaf(g, dy, dvy), uz = fmaf(g, dz, dvz);
    A.ax = fmaf(w, dx, A.ax); A.ay = fmaf(w, dy, A.ay); A.az = fmaf(w, dz, A.az);
    A.jx = fmaf(w, ux, A.jx); A.jy = fmaf(w, uy, A.jy); A.jz = fmaf(w, uz, A.jz);
    float tx = fmaf(g2, ux, dax), ty = fmaf(g2, uy, day), tz = fmaf(g2, uz, daz);
    tx = fmaf(b3, dx, tx); ty = fmaf(b3, dy, ty); tz = fmaf(b3, dz, tz);
    A.sx = fmaf(w, tx, A.sx); A.sy = fmaf(w, ty, A.sy); A.sz = fmaf(w, tz, A.sz);
}

// ---- mbarrier / bulk-copy primitives (PTX, sm_90+; SASS: SYNCS.*, UBLKCP) ---------------
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// ---- the evaluation kernel -------------------------------------------------------------
// One work item = (i-block ib, j-split sp): NT/JL i-particles against tiles [sp*tps, sp*tps+nt).
// JLT = 1: one i per thread.  JLT = 0: JL (runtime, power of two <= 32) consecutive lanes share
// one i and stride through the tile.  `tc` counts the tiles this CTA has consumed so far: ring
// stage = tc & 1, mbarrier phase = (tc >> 1) & 1, so the ring carries over from item to item.
// MX: 0 = FP64, 1 = mixed precision (reading G27), 2 = FP64 acceleration and jerk only
template <int NT, int TJ, int JLT, bool GUARD0, int MX, int UNR>
__device__ __forceinline__ void force_item(const double *__restrict__ jp, const double *__restrict__ jstream,
                                           const int32_t *__restrict__ active, const int m, const int ib, const int sp, const int tiles_total,
                                           const int tiles_per_split, const int JL, const double eps2,
                                           double *__restrict__ out, const size_t cstride, const size_t sstride,
                                           double (*tile)[TJ * REC], uint64_t *full, unsigned &tc)
{
    constexpr int NS = 2;
    constexpr uint32_t TILE_BYTES = TJ * REC * sizeof(double);
    const int tid = threadIdx.x;
    const int slots = NT / JL;              // i-particles per CTA
    const int k = ib * slots + tid / JL;    // slot in the active list
    const int jl = tid % JL;                // j-lane
    const int t0 = sp * tiles_per_split;
    const int nt = min(tiles_per_split, tiles_total - t0);
    const char *src = reinterpret_cast<const char *>(jstream) + (size_t)t0 * TILE_BYTES;

    if (tid == 0) {
        for (int st = 0; st < NS && st < nt; ++st) {
            const unsigned sg = (tc + st) & 1u;
            mbar_expect_tx(&full[sg], TILE_BYTES);
            bulk_g2s(tile[sg], src + (size_t)st * TILE_BYTES, TILE_BYTES, &full[sg]);
        }
    }

    // i-particle: predicted r, v, a of active[k] (differences of PREDICTED data)
    const int kc = min(k, m - 1);
    const int i = active ? active[kc] : kc;
    const double *pi = jp + (size_t)i * REC;
    const double2 i0 = *reinterpret_cast<const double2 *>(pi);
    const double2 i1 = *reinterpret_cast<const double2 *>(pi + 2);
    const double2 i2 = *reinterpret_cast<const double2 *>(pi + 4);
    const double2 i3 = *reinterpret_cast<const double2 *>(pi + 6);
    const double i4 = pi[8];
    const double xi = i0.x, yi = i0.y, zi = i1.x, vxi = i1.y, vyi = i2.x, vzi = i2.y;
    const double axi = i3.x, ayi = i3.y, azi = i4;

    // a warp whose slots are all beyond m only keeps the barriers company
    const bool warp_idle = (ib * slots + (tid & ~31) / JL) >= m;

    Acc9 T = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int it = 0; it < nt; ++it) {
        const unsigned sg = tc & 1u;
        mbar_wait(&full[sg], (tc >> 1) & 1u);
        if (!warp_idle) {
            const double *q = tile[sg];
            if (MX == 1) {
                AccF A = {0, 0, 0, 0, 0, 0, 0, 0, 0};
                const float eps2f = (float)eps2;
                if (JLT) {
#pragma unroll 6
                    for (int jj = 0; jj < TJ; ++jj)
                        pair_body_mx<GUARD0>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + jj * REC, eps2f, A);
                } else {
#pragma unroll 2
                    for (int jj = jl; jj < TJ; jj += JL)
                        pair_body_mx<GUARD0>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + jj * REC, eps2f, A);
                }
                T.ax += (double)A.ax; T.ay += (double)A.ay; T.az += (double)A.az;
                T.jx += (double)A.jx; T.jy += (double)A.jy; T.jz += (double)A.jz;
                T.sx += (double)A.sx; T.sy += (double)A.sy; T.sz += (double)A.sz;
            } else {
                Acc9 A = {0, 0, 0, 0, 0, 0, 0, 0, 0};
                if (JLT) {
#pragma unroll UNR
                    for (int jj = 0; jj < TJ; ++jj)
                        pair_body<GUARD0, MX != 2>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + jj * REC, eps2, A);
                } else {
#pragma unroll 2
                    for (int jj = jl; jj < TJ; jj += JL)
                        pair_body<GUARD0, MX != 2>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + jj * REC, eps2, A);
                }
                T.ax += A.ax; T.ay += A.ay; T.az += A.az;
                T.jx += A.jx; T.jy += A.jy; T.jz += A.jz;
                T.sx += A.sx; T.sy += A.sy; T.sz += A.sz;
            }
        }
        __syncthreads();  // every warp is done reading tile[sg]
        if (tid == 0 && it + NS < nt) {
            mbar_expect_tx(&full[sg], TILE_BYTES);
            bulk_g2s(tile[sg], src + (size_t)(it + NS) * TILE_BYTES, TILE_BYTES, &full[sg]);
        }
        ++tc;
    }

    if (!JLT) {  // fixed-order butterfly over the JL lanes that share this i
        for (int off = JL >> 1; off > 0; off >>= 1) {
            T.ax += __shfl_xor_sync(0xffffffffu, T.ax, off);
            T.ay += __shfl_xor_sync(0xffffffffu, T.ay, off);
            T.az += __shfl_xor_sync(0xffffffffu, T.az, off);
            T.jx += __shfl_xor_sync(0xffffffffu, T.jx, off);
            T.jy += __shfl_xor_sync(0xffffffffu, T.jy, off);
            T.jz += __shfl_xor_sync(0xffffffffu, T.jz, off);
            T.sx += __shfl_xor_sync(0xffffffffu, T.sx, off);
            T.sy += __shfl_xor_sync(0xffffffffu, T.sy, off);
            T.sz += __shfl_xor_sync(0xffffffffu, T.sz, off);
        }
    }
    if (k < m && jl == 0) {
        double *o = out + (size_t)sp * sstride + k;
        o[0 * cstride] = T.ax; o[1 * cstride] = T.ay; o[2 * cstride] = T.az;
        o[3 * cstride] = T.jx; o[4 * cstride] = T.jy; o[5 * cstride] = T.jz;
        o[6 * cstride] = T.sx; o[7 * cstride] = T.sy; o[8 * cstride] = T.sz;
    }
}

// grid.x: i-blocks, grid.y: j-splits; geometry passed by the host.
template <int NT, int TJ, int MINB, int JLT, bool GUARD0, int MX = 0, int UNR = 12>
__global__ void __launch_bounds__(NT, MINB)
    k_force(const double *__restrict__ jp, const double *__restrict__ jstream,
            const int32_t *__restrict__ active, const int m, const int tiles_total, const int tiles_per_split, const int JLr, const double eps2,
            double *__restrict__ out, const size_t cstride, const size_t sstride)
{
    __shared__ __align__(128) double tile[2][TJ * REC];
    __shared__ __align__(8) uint64_t full[2];
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned tc = 0;
    force_item<NT, TJ, JLT, GUARD0, MX, UNR>(jp, jstream, active, m, blockIdx.x, blockIdx.y, tiles_total, tiles_per_split,
                                         JLT ? 1 : JLr, eps2, out, cstride, sstride, tile, full, tc);
}

// Persistent form for the device-driven block-step loop (nb_graph.cu): a fixed grid of
// resident CTAs; the set size and the geometry are read from the control block, where the gather
// kernel of the same step left them.  CTA b starts with work item b and then draws the next one
// from a counter in the control block (items of one launch take equally long, but CTAs do not start
// together: a fixed stride left a 2 % tail at m ~ 2e5).  Item w is (i-block w % n_ib, split
// w / n_ib), so concurrently running CTAs stream the same j-split.
template <int NT, int TJ, int MINB, int JLT, bool GUARD0, int MX = 0, int UNR = 12>
__global__ void __launch_bounds__(NT, MINB)
    k_force_persistent(const double *__restrict__ jp, const int32_t *__restrict__ active_list, const int64_t N,
                       const int64_t Npad, const double eps2, double *__restrict__ f1,
                       double *__restrict__ partials, StepCtl *__restrict__ ctl)
{
    pdl_trigger();
    pdl_wait();
    if (ctl->done || ctl->g.variant != (JLT ? 0 : 1)) return;
    __shared__ __align__(128) double tile[2][TJ * REC];
    __shared__ __align__(8) uint64_t full[2];
    __shared__ long long next_item;
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
    const size_t cstride = g.S > 1 ? (size_t)g.mpad : (size_t)Npad;
    const size_t sstride = 9 * (size_t)g.mpad;
    const int tiles_total = (int)(Npad / TJ);
    const long long items = (long long)g.n_ib * g.S;
    unsigned tc = 0;
    long long w = blockIdx.x;
    while (w < items) {
        force_item<NT, TJ, JLT, GUARD0, MX, UNR>(jp, jp, active, m, (int)(w % g.n_ib), (int)(w / g.n_ib), tiles_total,
                                                 g.tps, g.JL, eps2, out, cstride, sstride, tile, full, tc);
        if (threadIdx.x == 0) next_item = (long long)gridDim.x + atomicAdd(&ctl->work, 1u);
        __syncthreads();
        w = next_item;
        __syncthreads();
    }
}

// ---- partial-sum reduction (Table 1 row 4): f1[c][k] = sum_s part[s][c][k], s ascending ---
// thread-per-element version: coalesced along k, used when the number of splits is small
__global__ void k_reduce_thread(const double *__restrict__ part, const int S, const int m,
                                const size_t cstride, const size_t sstride, double *__restrict__ f1,
                                const size_t f1stride)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (k >= m) return;
    const double *p = part + c * cstride + k;
    double acc = 0.0;
    for (int s = 0; s < S; ++s) acc += p[(size_t)s * sstride];
    f1[c * f1stride + k] = acc;
}
// warp-per-element version: lane l sums splits l, l+32, ... then a fixed butterfly
__global__ void k_reduce_warp(const double *__restrict__ part, const int S, const int m,
                              const size_t cstride, const size_t sstride, double *__restrict__ f1,
                              const size_t f1stride)
{
    const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wid >= 9 * m) return;
    const int c = wid / m, k = wid - c * m;
    const double *p = part + c * cstride + k;
    double acc = 0.0;
    for (int s = lane; s < S; s += 32) acc += p[(size_t)s * sstride];
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
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

// Reduction for the device-driven loop: fixed grid, sizes read from the control block.  Element
// e = c * m + k; the sum over splits runs in ascending split order exactly as in k_reduce_thread
// (S < 32) or k_reduce_warp (S >= 32), so both drivers give bit-identical results.
__global__ void __launch_bounds__(256)
    k_reduce_persistent(const double *__restrict__ part, const StepCtl *__restrict__ ctl, double *__restrict__ f1,
                        const size_t f1stride)
{
    pdl_trigger();
    pdl_wait();
    if (ctl->done || ctl->g.S <= 1) return;
    const int S = ctl->g.S, m = (int)ctl->n_active;
    const size_t cstride = (size_t)ctl->g.mpad, sstride = 9 * (size_t)ctl->g.mpad;
    const long long total = 9LL * m;
    if (S < 32) {
        for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
            const int c = (int)(e / m), k = (int)(e - (long long)c * m);
            const double *p = part + c * cstride + k;
            double acc = 0.0;
            for (int s = 0; s < S; ++s) acc += p[(size_t)s * sstride];
            f1[c * f1stride + k] = acc;
        }
    } else {
        const int lane = threadIdx.x & 31;
        const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
        for (long long wid = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; wid < total; wid += nwarps) {
            const int c = (int)(wid / m), k = (int)(wid - (long long)c * m);
            const double *p = part + c * cstride + k;
            double acc = 0.0;
            for (int s = lane; s < S; s += 32) acc += p[(size_t)s * sstride];
            for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
            if (lane == 0) f1[c * f1stride + k] = acc;
        }
    }
}

// ---- host side ---------------------------------------------------------------------------
// The split search never asks for more than MAX_WAVES waves of CTAs, i.e. S * m <= MAX_WAVES x
// (resident CTAs) x (i-slots per CTA); S <= 65535 splits of mpad <= m + 31 add the slack term.
static size_t partials_bound(const nb_ctx *ctx)
{
    const int64_t a = (int64_t)ctx->n_sm * ctx->occ[0] * NT_A, b = (int64_t)ctx->n_sm * ctx->occ[1] * NT_B;
    int64_t items = (int64_t)MAX_WAVES * (a > b ? a : b) + 32 * 65536;
    const int64_t by_n = (ctx->Npad / TJ_B) * (ctx->Npad + 32);   // S <= tiles, mpad <= Npad + 32
    if (by_n < items) items = by_n;
    return (size_t)(9 * items);
}

int query_force_occupancy(nb_ctx *ctx)
{
    int v = 0;
    NB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                     &v, k_force<NT_A, TJ_A, MINB_A, 1, false>, NT_A, 0));
    ctx->occ[0] = v > 0 ? v : 1;
    NB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                     &v, k_force<NT_B, TJ_B, MINB_B, 0, false>, NT_B, 0));
    ctx->occ[1] = v > 0 ? v : 1;
    NB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                     &v, k_force_persistent<NT_A, TJ_A, MINB_A, 1, false>, NT_A, 0));
    ctx->occ[2] = v > 0 ? v : 1;
    NB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                     &v, k_force_persistent<NT_B, TJ_B, MINB_B, 0, false>, NT_B, 0));
    ctx->occ[3] = v > 0 ? v : 1;
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

template <int NT, int TJ, int MINB, int JLT>
static void launch_variant(nb_ctx *ctx, dim3 grid, const int32_t *active, int m, int tiles_total,
                           int tps, int JL, double *out, size_t cstride, size_t sstride, bool no_snap)
{
    const double *jstream = ctx->jp + (size_t)ctx->j_begin * REC;   // j-shard (nb_set_j_range), else the whole stream
#define NB_KF(G0, MXP)                                                                 \
    k_force<NT, TJ, MINB, JLT, G0, MXP><<<grid, NT, 0, ctx->stream>>>(ctx->jp, jstream, active, m, tiles_total, tps, JL, \
                                                                      ctx->eps2, out, cstride, sstride)
    const bool g0 = ctx->eps == 0.0, mx = ctx->precision == 1;
    if (g0 && mx) NB_KF(true, 1);
    else if (mx) NB_KF(false, 1);
    else if (g0 && no_snap) NB_KF(true, 2);
    else if (no_snap) NB_KF(false, 2);
    else if (g0) NB_KF(true, 0);
    else NB_KF(false, 0);
#undef NB_KF
}

int launch_force(nb_ctx *ctx, const int32_t *active, int64_t m, bool no_snap)
{
    if (m <= 0) return NB_OK;
    // records of the j-shard, padded to whole tiles (records N..Npad-1 have zero mass)
    const int64_t jlen = (ctx->j_end == ctx->N ? ctx->Npad : ctx->j_end) - ctx->j_begin;
    const ForceGeom g = choose_geom(m, jlen, ctx->n_sm, ctx->occ[0], ctx->occ[1], (int64_t)ctx->partials_limit,
                                    ctx->force_split, ctx->force_jlanes);
    const bool varA = g.variant == 0;
    const int TJ = varA ? TJ_A : TJ_B;
    const int64_t tiles = jlen / TJ;
    double *out = ctx->f1;
    size_t cstride = (size_t)ctx->Npad, sstride = 0;
    if (g.S > 1) {
        const int rc = reserve_partials(ctx, (size_t)g.S * 9 * (size_t)g.mpad);
        if (rc != NB_OK) return rc;
        out = ctx->partials; cstride = (size_t)g.mpad; sstride = 9 * (size_t)g.mpad;
    }
    dim3 grid((unsigned)g.n_ib, (unsigned)g.S, 1);
    if (varA)
        launch_variant<NT_A, TJ_A, MINB_A, 1>(ctx, grid, active, (int)m, (int)tiles, g.tps, 1, out, cstride, sstride, no_snap);
    else
        launch_variant<NT_B, TJ_B, MINB_B, 0>(ctx, grid, active, (int)m, (int)tiles, g.tps, g.JL, out, cstride, sstride, no_snap);
    NB_LAUNCH_CHECK(ctx, "k_force");
    if (g.S > 1) {
        if (g.S < 32) {
            dim3 gr((unsigned)((m + 127) / 128), 9, 1);
            k_reduce_thread<<<gr, 128, 0, ctx->stream>>>(out, g.S, (int)m, cstride, sstride, ctx->f1, (size_t)ctx->Npad);
        } else {
            const int64_t warps = 9 * m;
            k_reduce_warp<<<(unsigned)((warps + 7) / 8), 256, 0, ctx->stream>>>(out, g.S, (int)m, cstride, sstride, ctx->f1, (size_t)ctx->Npad);
        }
        NB_LAUNCH_CHECK(ctx, "k_reduce");
    }
    ctx->last_launch[0] = varA ? NT_A : NT_B; ctx->last_launch[1] = g.JL; ctx->last_launch[2] = g.S;
    ctx->last_launch[3] = (int64_t)g.n_ib * g.S; ctx->last_launch[4] = TJ;
    ctx->n_pairs += (double)m * (double)(ctx->j_end - ctx->j_begin);
    return NB_OK;
}

// Device-driven loop: both variants are enqueued with fixed grids (one wave of resident CTAs);
// the one the gather kernel did not select returns at once, as does everything when the control
// block says `done`.
int enqueue_force_persistent(nb_ctx *ctx)
{
    const unsigned gA = (unsigned)(ctx->n_sm * ctx->occ[2]), gB = (unsigned)(ctx->n_sm * ctx->occ[3]);
#define NB_KP(G0, MXP)                                                                                       \
    do {                                                                                                     \
        launch_chain(k_force_persistent<NT_A, TJ_A, MINB_A, 1, G0, MXP>, dim3(gA), dim3(NT_A), ctx->stream, pdl, \
                     ctx->jp, ctx->active, ctx->N, ctx->Npad, ctx->eps2, ctx->f1, ctx->partials, ctx->ctl);   \
        launch_chain(k_force_persistent<NT_B, TJ_B, MINB_B, 0, G0, MXP>, dim3(gB), dim3(NT_B), ctx->stream, pdl, \
                     ctx->jp, ctx->active, ctx->N, ctx->Npad, ctx->eps2, ctx->f1, ctx->partials, ctx->ctl);   \
    } while (0)
    const bool g0 = ctx->eps == 0.0, mx = ctx->precision == 1, pdl = ctx->use_graph == 2;
    if (g0 && mx) NB_KP(true, 1);
    else if (g0) NB_KP(true, 0);
    else if (mx) NB_KP(false, 1);
    else NB_KP(false, 0);
#undef NB_KP
    NB_LAUNCH_CHECK(ctx, "k_force_persistent");
    ctx->n_launch += 1;  // two kernels
    launch_chain(k_reduce_persistent, dim3((unsigned)(2 * ctx->n_sm)), dim3(256), ctx->stream, pdl, ctx->partials,
                 ctx->ctl, ctx->f1, (size_t)ctx->Npad);
    NB_LAUNCH_CHECK(ctx, "k_reduce_persistent");
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
