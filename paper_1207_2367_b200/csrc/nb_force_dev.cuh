// nb_force_dev.cuh -- device functions of the evaluation step, shared by the kernels of nb_force.cu
// (one launch per evaluation, persistent form for the graph-driven loop) and nb_resident.cu (the
// cluster-resident loop): the pair body (Eq. 8-10, with the Eq. 2 softening), the
// mbarrier / bulk-copy primitives and force_item, the work of one (i-block, j-split) item.  All
// drivers call the same functions with the same geometry, so their results are bit-identical.
#pragma once
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
//   s = |dr|^2 + eps^2,  y = s^(-1/2),  alpha = (dr.dv)/s,  beta = (|dv|^2 + dr.da)/s + alpha^2,
//   u = dv - 3 alpha dr,  A0 = w dr,  A1 = w u,  A2 = w (da - 6 alpha u - 3 beta dr),  w = m_j s^(-3/2).
// q points at the packed record {x y z vx vy vz ax ay az m} of particle j in shared memory.
//
// 51 FP64-pipe instructions (32 DFMA + 10 DMUL + 9 DADD) and one MUFU.RSQ64H:
//   * the factor 3 of "3 alpha", "3 beta" rides on the inverse square root: the Newton step produces
//     y' = sqrt(3) y (its three constants carry the sqrt(3)), so ri2 = y'^2 = 3/s, g = ri2 (dr.dv) = 3 alpha and
//     b3 = ri2 (|dv|^2 + dr.da) + g^2/3 = 3 beta come out directly and enter the FMAs negated (operand
//     modifiers are free);  w' = m_j y' ri2 = 3 sqrt(3) w, so the accumulators hold 3 sqrt(3) times the sums
//     and the caller scales them ONCE per item by PAIR_SCALE = 1/(3 sqrt(3)) (force_item);
//   * 2 g is an increment of the exponent field (integer pipe, exact for every normal g; g = 0 or
//     subnormal gives a value below 4.5e-308 whose product with u is far below one ulp of anything here).
// The statement ORDER below is not cosmetic.  The FP64 datapath reads one fresh 64-bit operand per cycle
// and SM sub-partition, so an instruction with three distinct register sources costs 3 cycles instead of 2
// unless one of them sits in the operand-reuse cache, i.e. the preceding FP64 instruction of the same warp
// read it in the same operand slot.  ptxas -O1 (this file's setting, _build.py)
// keeps close to the order written here; this order (found by a randomised search over dependency-respecting
// orders and operand orders, scored on the SASS by sum of max(2, fresh operands)) has 107 cycles of
// operand fetch per pair against 102 for the 51 instructions alone; the round-1 body had 124.
// SNAP = false (start-up pass 1, G8: only a and jerk are wanted): everything that only feeds the snap is
// dead code in that instantiation -- 29 FP64 instructions; a and jerk are computed by the same expressions.
constexpr double PAIR_SCALE = 0.19245008972987526;   // 1 / (3 sqrt(3))

__device__ __forceinline__ double twice(const double g)
{
    return __hiloint2double(__double2hiint(g) + 0x00100000, __double2loint(g));
}

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
    const double mj = p4.y;
    const double dy = p0.y - yi;
    const double dz = p1.x - zi;
    const double s0 = fma(dy, dy, eps2);
    const double dvz = p2.y - vzi;
    const double dvx = p1.y - vxi;
    const double daz = p4.x - azi;
    const double vr0 = dz * daz;
    const double dvy = p2.x - vyi;
    const double dax = p3.x - axi;
    const double dx = p0.x - xi;
    const double s1 = fma(dx, dx, s0);
    const double day = p3.y - ayi;
    const double s = fma(dz, dz, s1);                 // |dr|^2 + eps^2
    const double rv0 = dvy * dy;
    const double vr1 = fma(dy, day, vr0);
    const double vr2 = fma(dax, dx, vr1);
    const double rv1 = fma(dx, dvx, rv0);
    const double vr3 = fma(dvz, dvz, vr2);
    double y0 = rsqrt_seed(s);
    if (GUARD0) {  // eps = 0: a coincident pair (the self term) contributes nothing (G12)
        if ((__double2hiint(s) | __double2loint(s)) == 0) y0 = 0.0;
    }
    const double rv = fma(dz, dvz, rv1);              // dr.dv
    const double vr4 = fma(dvx, dvx, vr3);
    const double vr = fma(dvy, dvy, vr4);             // |dv|^2 + dr.da
    // y' = sqrt(3) y0 (1 + e (1/2 + 3/8 e)), e = 1 - s y0^2: one third-order step on the 2^-21 seed
    const double y2 = y0 * y0;
    const double e = fma(-s, y2, 1.0);
    const double p = fma(e, 0.649519052838329, 0.8660254037844386);      // sqrt(3) (3/8 e + 1/2)
    const double ep1 = fma(e, p, 1.7320508075688772);                    // sqrt(3) (1 + e (...))
    const double y = y0 * ep1;                        // sqrt(3) s^(-1/2)
    const double ri2 = y * y;                         // 3 / s
    const double g = ri2 * rv;                        // 3 alpha
    const double gg = g * g;
    const double qv = ri2 * vr;
    const double my = mj * y;
    const double uy = fma(dy, -g, dvy);               // u = dv - 3 alpha dr
    const double uz = fma(dz, -g, dvz);
    const double b3 = fma(gg, 1.0 / 3.0, qv);         // 3 beta
    const double t1y = fma(-b3, dy, day);
    const double ux = fma(-g, dx, dvx);
    const double g2 = twice(g);                       // 6 alpha
    const double t1x = fma(-b3, dx, dax);
    const double t1z = fma(dz, -b3, daz);
    const double ty = fma(uy, -g2, t1y);              // t = da - 6 alpha u - 3 beta dr
    const double tx = fma(ux, -g2, t1x);
    const double tz = fma(-g2, uz, t1z);
    const double w = ri2 * my;                        // 3 sqrt(3) m_j s^(-3/2)
    if (SNAP) A.sy = fma(w, ty, A.sy);
    A.az = fma(w, dz, A.az);
    if (SNAP) A.sz = fma(w, tz, A.sz);
    A.ay = fma(dy, w, A.ay);
    A.jz = fma(w, uz, A.jz);
    A.jx = fma(ux, w, A.jx);
    A.ax = fma(dx, w, A.ax);
    A.jy = fma(uy, w, A.jy);
    if (SNAP) A.sx = fma(w, tx, A.sx);
}

// The same pair in the paper's mixed precision (readings G27, G27b): the nine
// differences are formed in double from the double records and rounded to float, everything
// else of Eq. 8-10 is float arithmetic (FFMA/FMUL on the FP32 pipe, MUFU.RSQ).
//   ACC64 = false (reading G27, nb_set_precision 1): the pair terms are summed in float within one j-tile
//     (the caller adds the tile sums in double).  FP64-pipe work per pair: 9 DADD + 10 F2F.
//   ACC64 = true (reading G27b, nb_set_precision 2): the acceleration and jerk terms of every pair -- float
//     products, rounded once -- are converted and ADDED IN DOUBLE (6 DP additions: with the 9 differences the
//     15 double-precision operations PAPER.md:301 counts); the snap terms are summed in float as above.
struct AccF {
    float ax, ay, az, jx, jy, jz, sx, sy, sz;
};
template <bool GUARD0, bool ACC64 = false>
__device__ __forceinline__ void pair_body_mx(const double xi, const double yi, const double zi,
                                             const double vxi, const double vyi, const double vzi,
                                             const double axi, const double ayi, const double azi,
                                             const double *__restrict__ q, const float eps2, AccF &A, Acc9 &D)
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
    if (GUARD0) {  // eps = 0, or eps so small that m s^(-3/2) overflows a float (then w * 0 = NaN): the
                   // self term (dr = 0 exactly, s = eps^2) is excluded explicitly (G12)
        if (s == eps2) y = 0.0f;
    }
    const float P = y * y;             // 1/s
    const float w = (mj * y) * P;      // m_j s^(-3/2)
    const float qq = -3.0f * P;
    const float g = rv * qq;           // -3 alpha
    const float b3 = fmaf(g * g, -1.0f / 3.0f, qq * vr);  // -3 beta
    const float g2 = g + g;
    const float ux = fmaf(g, dx, dvx), uy = fmaf(g, dy, dvy), uz = fmaf(g, dz, dvz);
    if (ACC64) {
        D.ax += (double)(w * dx); D.ay += (double)(w * dy); D.az += (double)(w * dz);
        D.jx += (double)(w * ux); D.jy += (double)(w * uy); D.jz += (double)(w * uz);
    } else {
        A.ax = fmaf(w, dx, A.ax); A.ay = fmaf(w, dy, A.ay); A.az = fmaf(w, dz, A.az);
        A.jx = fmaf(w, ux, A.jx); A.jy = fmaf(w, uy, A.jy); A.jz = fmaf(w, uz, A.jz);
    }
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
// JL (compile time, a power of two <= 32) consecutive lanes share one i and stride through the tile:
// JL = 1 is one i per thread (m >= NT); JL > 1 keeps all lanes busy when the active set is small
// (the paper shrinks its thread blocks instead).  `tc` counts the tiles this CTA has
// consumed so far: ring stage = tc & 1, mbarrier phase = (tc >> 1) & 1, so the ring carries over
// from item to item.
// MX: 0 = FP64, 1 = mixed precision (reading G27), 2 = FP64 acceleration and jerk only,
//     3 = mixed precision with acceleration and jerk accumulated in double (reading G27b)
// The NT threads that work on an item are a whole CTA (VS = 0: tid = threadIdx.x, block barrier) or a
// "virtual CTA" of NT threads on the named barrier `bar_id` inside a larger CTA (VS = 2, the resident
// loop of nb_resident.cu).  The arithmetic and its order are the same.
// Output: element (component c, slot k, split sp) goes to out[c * cstride + k * kstride + sp * sstride]
// (PartLayout below).
template <int VS>
__device__ __forceinline__ void vcta_sync(const int bar_id, const int nthreads)
{
    if (VS == 0) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(nthreads) : "memory");
}

template <int NT, int TJ, int JL, bool GUARD0, int MX, int UNR, int VS = 0>
__device__ __forceinline__ void force_item(const double *__restrict__ jp, const double *__restrict__ jstream,
                                           const int32_t *__restrict__ active, const int m, const int ib, const int sp, const int tiles_total,
                                           const int tiles_per_split, const double eps2,
                                           double *__restrict__ out, const size_t cstride, const size_t kstride, const size_t sstride,
                                           double (*tile)[TJ * REC], uint64_t *full, unsigned &tc,
                                           const int tid_in = 0, const int bar_id = 0)
{
    static_assert(JL >= 1 && JL <= 32 && (JL & (JL - 1)) == 0, "lanes per i: a power of two within one warp");
    constexpr int NS = 2;
    constexpr uint32_t TILE_BYTES = TJ * REC * sizeof(double);
    constexpr int PER = TJ / JL;                          // pairs per thread and tile
    constexpr int UNRJ = JL == 1 ? UNR : (PER >= 24 ? 12 : PER);
    constexpr int UNRM = PER >= 6 ? 6 : PER;
    const int tid = VS == 0 ? (int)threadIdx.x : tid_in;
    constexpr int slots = NT / JL;          // i-particles per CTA
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
            const double *q = tile[sg] + jl * REC;
            if (MX == 1 || MX == 3) {
                AccF A = {0, 0, 0, 0, 0, 0, 0, 0, 0};
                const float eps2f = (float)eps2;
#pragma unroll UNRM
                for (int jj = 0; jj < PER; ++jj)
                    pair_body_mx<GUARD0, MX == 3>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + jj * (JL * REC), eps2f, A, T);
                if (MX == 1) {
                    T.ax += (double)A.ax; T.ay += (double)A.ay; T.az += (double)A.az;
                    T.jx += (double)A.jx; T.jy += (double)A.jy; T.jz += (double)A.jz;
                }
                T.sx += (double)A.sx; T.sy += (double)A.sy; T.sz += (double)A.sz;
            } else {
                Acc9 A = {0, 0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll UNRJ
                for (int jj = 0; jj < PER; ++jj)
                    pair_body<GUARD0, MX != 2>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + jj * (JL * REC), eps2, A);
                T.ax += A.ax; T.ay += A.ay; T.az += A.az;
                T.jx += A.jx; T.jy += A.jy; T.jz += A.jz;
                T.sx += A.sx; T.sy += A.sy; T.sz += A.sz;
            }
        }
        vcta_sync<VS>(bar_id, NT);  // every warp is done reading tile[sg]
        if (tid == 0 && it + NS < nt) {
            mbar_expect_tx(&full[sg], TILE_BYTES);
            bulk_g2s(tile[sg], src + (size_t)(it + NS) * TILE_BYTES, TILE_BYTES, &full[sg]);
        }
        ++tc;
    }

    if (MX == 0 || MX == 2) {  // the FP64 pair body accumulates 3 sqrt(3) times the sums (pair_body)
        T.ax *= PAIR_SCALE; T.ay *= PAIR_SCALE; T.az *= PAIR_SCALE;
        T.jx *= PAIR_SCALE; T.jy *= PAIR_SCALE; T.jz *= PAIR_SCALE;
        T.sx *= PAIR_SCALE; T.sy *= PAIR_SCALE; T.sz *= PAIR_SCALE;
    }
    if (JL > 1) {  // fixed-order butterfly over the JL lanes that share this i
#pragma unroll
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
        double *o = out + (size_t)sp * sstride + (size_t)k * kstride;
        o[0 * cstride] = T.ax; o[1 * cstride] = T.ay; o[2 * cstride] = T.az;
        o[3 * cstride] = T.jx; o[4 * cstride] = T.jy; o[5 * cstride] = T.jz;
        o[6 * cstride] = T.sx; o[7 * cstride] = T.sy; o[8 * cstride] = T.sz;
    }
}

// force_item for a lane count known only at run time (the geometry rule chooses it from m)
template <int NT, int TJ, bool GUARD0, int MX, int UNR, int VS = 0>
__device__ __forceinline__ void force_item_jl(const int JL, const double *__restrict__ jp, const double *__restrict__ jstream,
                                              const int32_t *__restrict__ active, const int m, const int ib, const int sp,
                                              const int tiles_total, const int tiles_per_split, const double eps2,
                                              double *__restrict__ out, const size_t cstride, const size_t kstride, const size_t sstride,
                                              double (*tile)[TJ * REC], uint64_t *full, unsigned &tc, const int tid_in = 0,
                                              const int bar_id = 0)
{
#define NB_ITEM(J) force_item<NT, TJ, J, GUARD0, MX, UNR, VS>(jp, jstream, active, m, ib, sp, tiles_total, tiles_per_split, eps2, \
                                                              out, cstride, kstride, sstride, tile, full, tc, tid_in, bar_id)
    switch (JL) {
        case 1: NB_ITEM(1); break;
        case 2: NB_ITEM(2); break;
        case 4: NB_ITEM(4); break;
        case 8: NB_ITEM(8); break;
        case 16: NB_ITEM(16); break;
        default: NB_ITEM(32); break;
    }
#undef NB_ITEM
}

// ---- where the split partials live, and their fixed-order sum (Table 1 row 4) ----
// One split: the evaluation writes f1[c][k] directly.  2..31 splits: part[sp][c][k] (split-major, coalesced
// along k for the many elements of a large set), summed by ONE thread per element in ascending split order.
// >= 32 splits (small sets): part[c][k][sp] (split-minor: the S values of an element are consecutive), summed by
// ONE warp per element: lane l adds the splits l, l + 32, ... in ascending order, then the xor butterfly
// 16, 8, 4, 2, 1.  Every driver sums through these two functions, so all agree bit for bit.
struct PartLayout {
    size_t cstride, kstride, sstride;
};
__host__ __device__ inline PartLayout part_layout(const int S, const int mpad, const int64_t Npad)
{
    PartLayout L;
    if (S <= 1) { L.cstride = (size_t)Npad; L.kstride = 1; L.sstride = 0; }
    else if (S < 32) { L.cstride = (size_t)mpad; L.kstride = 1; L.sstride = 9 * (size_t)mpad; }
    else { L.cstride = (size_t)mpad * S; L.kstride = (size_t)S; L.sstride = 1; }
    return L;
}
__device__ __forceinline__ double sum_splits_thread(const double *__restrict__ p, const int S, const size_t sstride)
{
    double acc = 0.0;
    for (int s = 0; s < S; ++s) acc += p[(size_t)s * sstride];
    return acc;
}
__device__ __forceinline__ double sum_splits_warp(const double *__restrict__ p, const int S, const int lane)
{
    double acc = 0.0;
#pragma unroll 4
    for (int s = lane; s < S; s += 32) acc += p[s];
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    return acc;
}

// All nine components of slot k, by one warp (all 32 lanes call it): f1[c][k] <- fixed-order sum over the splits.
// For S >= 32 the nine lane-strided sums advance together, so that a lane has nine (unrolled: eighteen) independent
// loads in flight instead of one component's at a time; per component the additions are those of sum_splits_warp,
// in the same order.
__device__ __forceinline__ void reduce_one(const double *__restrict__ part, const int S, const PartLayout &L, const int k,
                                           const int lane, double *__restrict__ f1, const int64_t Npad)
{
    if (S < 32) {
        if (lane < 9) f1[lane * Npad + k] = sum_splits_thread(part + lane * L.cstride + (size_t)k * L.kstride, S, L.sstride);
    } else {
        const double *p = part + (size_t)k * L.kstride;
        double acc[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll 2
        for (int s = lane; s < S; s += 32) {
#pragma unroll
            for (int cc = 0; cc < 9; ++cc) acc[cc] += p[cc * L.cstride + s];
        }
#pragma unroll
        for (int cc = 0; cc < 9; ++cc) {
            double a = acc[cc];
            for (int off = 16; off > 0; off >>= 1) a += __shfl_xor_sync(0xffffffffu, a, off);
            if (lane == 0) f1[cc * Npad + k] = a;
        }
    }
    __syncwarp();
}

}  // namespace nb
