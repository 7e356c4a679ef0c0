// nb_step_dev.cuh -- device functions of the O(N) / O(m) steps, shared by the kernels of nb_step.cu and the
// cluster-resident loop of nb_resident.cu: predictor (Eq. 3-7), corrector (Eq. 11-14) with the end-point
// derivatives (G6), the time-step rule (Eq. 15-16) and the block minimum.
#pragma once
#include "nb_internal.cuh"

namespace nb {

constexpr int SCHED_THREADS = 256;
constexpr int SCHED_ITEMS = 8;                        // consecutive particles per thread
constexpr int SCHED_BLOCK = SCHED_THREADS * SCHED_ITEMS;


// ---------------------------------------------------------------------------------------
// Predictor, Eq. 3-7 with the garbled dots read as the Taylor series (G1) and
// the interval h = t - t_i for every particle (G2), in Horner form:
//   r_p = r + h (v + h/2 (a + h/3 (j + h/4 (s + h/5 c))))
//   v_p = v + h (a + h/2 (j + h/3 (s + h/4 c)))
//   a_p = a + h (j + h/2 (s + h/3 c))
// Reads 19 + 1 doubles, writes one 80-byte record: 240 B per particle.
__device__ __forceinline__ void predict_one(const int64_t i, const int64_t Npad, const double t,
                                            const double *__restrict__ ti, const double *__restrict__ mass,
                                            const double *__restrict__ r, const double *__restrict__ v,
                                            const double *__restrict__ a, const double *__restrict__ j,
                                            const double *__restrict__ s, const double *__restrict__ c,
                                            double *__restrict__ jp)
{
    const double h = t - ti[i];
    const double h2 = h * 0.5, h3 = h * (1.0 / 3.0), h4 = h * 0.25, h5 = h * 0.2;
    double rp[3], vp[3], ap[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int64_t q = d * Npad + i;
        const double r0 = r[q], v0 = v[q], a0 = a[q], j0 = j[q], s0 = s[q], c0 = c[q];
        rp[d] = fma(h, fma(h2, fma(h3, fma(h4, fma(h5, c0, s0), j0), a0), v0), r0);
        vp[d] = fma(h, fma(h2, fma(h3, fma(h4, c0, s0), j0), a0), v0);
        ap[d] = fma(h, fma(h2, fma(h3, c0, s0), j0), a0);
    }
    double2 *rec = reinterpret_cast<double2 *>(jp + i * REC);
    rec[0] = make_double2(rp[0], rp[1]);
    rec[1] = make_double2(rp[2], vp[0]);
    rec[2] = make_double2(vp[1], vp[2]);
    rec[3] = make_double2(ap[0], ap[1]);
    rec[4] = make_double2(ap[2], mass[i]);
}

// ---------------------------------------------------------------------------------------
// Time-step rule, Eq. 15-16 with p = 6 (exponent read as 1/(p-3), G5),
// quantised to a power of two (G9).  This is an INTEGER decision taken in plain
// IEEE double, one correctly-rounded operation at a time (the *_rn intrinsics are never
// contracted into FMAs), in the order the formula is written, so that identical inputs give
// the identical step:  x = ((eta eta) eta) A1 / A4,  dt_q = 2^floor(ilogb(x)/3),
// dt = min(dt_q, 2 dt_old); growth only if t_next is a multiple of 2 dt_old; clamp.
__device__ __forceinline__ double norm3_rn(const double x, const double y, const double z)
{
    return __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z)));
}
__device__ __forceinline__ double pow2i(int k)  // 2^k for -1022 <= k <= 1023
{
    return __longlong_as_double((long long)(k + 1023) << 52);
}
__device__ __forceinline__ int ilogb_pos_normal(double x)
{
    return (int)((__double_as_longlong(x) >> 52) & 0x7ff) - 1023;
}
__device__ __forceinline__ int floordiv3(int e) { return e >= 0 ? e / 3 : -((-e + 2) / 3); }

static __device__ double new_dt(const double na, const double nj, const double ns, const double n3,
                         const double n4, const double n5, const double eta, const double dt_old,
                         const double t_next, const double dt_min, const double dt_max)
{
    const double A1 = __dsqrt_rn(__dadd_rn(__dmul_rn(na, ns), __dmul_rn(nj, nj)));
    const double A4 = __dsqrt_rn(__dadd_rn(__dmul_rn(n3, n5), __dmul_rn(n4, n4)));
    double dt_q;
    if (!(A4 > 0.0)) {
        dt_q = dt_max;
    } else {
        const double x = __ddiv_rn(__dmul_rn(__dmul_rn(__dmul_rn(eta, eta), eta), A1), A4);
        if (!(x > 0.0)) dt_q = dt_min;
        else if (isinf(x)) dt_q = dt_max;
        else if (x < 2.2250738585072014e-308) dt_q = dt_min;  // subnormal: far below any limit
        else dt_q = pow2i(floordiv3(ilogb_pos_normal(x)));
    }
    const double two_old = __dmul_rn(2.0, dt_old);
    double dt = dt_q < two_old ? dt_q : two_old;
    if (dt > dt_old) {
        const double q = __ddiv_rn(t_next, two_old);  // exact: power-of-two divisor
        if (q != rint(q)) dt = dt_old;
    }
    if (dt < dt_min) dt = dt_min;
    if (dt > dt_max) dt = dt_max;
    return dt;
}

// Corrector, Eq. 11-14: v first, r uses the corrected v.  Index 0 = stored
// values at t_i, index 1 = evaluated at t_i + h.  Then a^(3), a^(4), a^(5) at the END of the
// step from the quintic Hermite interpolant through (a, jerk, snap) at both ends (G6):
//   a3 =  3 [20 dA - h ( 8 j0 + 12 j1) + h^2 (3 s1 -   s0)] / h^3
//   a4 = 12 [30 dA - h (14 j0 + 16 j1) + h^2 (3 s1 - 2 s0)] / h^4
//   a5 = 60 [12 dA - 6 h (j0 + j1)     + h^2 (  s1 -   s0)] / h^5
// Commit: r, v <- corrected; a, jerk, snap <- evaluated (G16); crackle <- a3 (G7); t_i <- t_next.
__device__ __forceinline__ double correct_one(const int k, const int64_t i, const int64_t Npad, const double t_next,
                                              const double eta, const double dt_min, const double dt_max,
                                              const double *__restrict__ f1, double *__restrict__ ti,
                                              double *__restrict__ dti, double *__restrict__ r, double *__restrict__ v,
                                              double *__restrict__ a, double *__restrict__ j, double *__restrict__ s,
                                              double *__restrict__ c)
{
    const double h = dti[i];
    const double h2 = h * h, h3 = h2 * h;
    const double ih = 1.0 / h;  // exact: h is a power of two
    const double ih3 = ih * ih * ih, ih4 = ih3 * ih, ih5 = ih4 * ih;
    double A1[3], J1[3], S1[3], C3[3], C4[3], C5[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int64_t q = d * Npad + i;
        const double r0 = r[q], v0 = v[q], a0 = a[q], j0 = j[q], s0 = s[q];
        const double a1 = f1[(0 + d) * Npad + k], j1 = f1[(3 + d) * Npad + k], s1 = f1[(6 + d) * Npad + k];
        const double vc = v0 + (h * 0.5) * (a1 + a0) - (h2 * 0.1) * (j1 - j0) + (h3 * (1.0 / 120.0)) * (s1 + s0);
        const double rc = r0 + (h * 0.5) * (vc + v0) - (h2 * 0.1) * (a1 - a0) + (h3 * (1.0 / 120.0)) * (j1 + j0);
        const double dA = a1 - a0;
        C3[d] = 3.0 * (20.0 * dA - h * (8.0 * j0 + 12.0 * j1) + h2 * (3.0 * s1 - s0)) * ih3;
        C4[d] = 12.0 * (30.0 * dA - h * (14.0 * j0 + 16.0 * j1) + h2 * (3.0 * s1 - 2.0 * s0)) * ih4;
        C5[d] = 60.0 * (12.0 * dA - 6.0 * h * (j0 + j1) + h2 * (s1 - s0)) * ih5;
        A1[d] = a1; J1[d] = j1; S1[d] = s1;
        r[q] = rc; v[q] = vc; a[q] = a1; j[q] = j1; s[q] = s1; c[q] = C3[d];
    }
    ti[i] = t_next;
    const double dtn = new_dt(norm3_rn(A1[0], A1[1], A1[2]), norm3_rn(J1[0], J1[1], J1[2]), norm3_rn(S1[0], S1[1], S1[2]),
                              norm3_rn(C3[0], C3[1], C3[2]), norm3_rn(C4[0], C4[1], C4[2]), norm3_rn(C5[0], C5[1], C5[2]),
                              eta, h, t_next, dt_min, dt_max);
    dti[i] = dtn;
    return t_next + dtn;  // exact: dyadic rationals
}

__device__ __forceinline__ void block_min_to(double v, unsigned long long *dst)
{
    for (int off = 16; off > 0; off >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, off));
    __shared__ double smin[SCHED_THREADS / 32];
    if ((threadIdx.x & 31) == 0) smin[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < (blockDim.x >> 5) ? smin[threadIdx.x] : __longlong_as_double(0x7ff0000000000000LL);
        for (int off = 16; off > 0; off >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, off));
        if (threadIdx.x == 0 && v < __longlong_as_double(0x7ff0000000000000LL))
            atomicMin(dst, (unsigned long long)__double_as_longlong(v));
    }
}

}  // namespace nb
