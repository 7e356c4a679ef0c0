// nb_resident_dev.cuh -- device functions shared by the two on-chip block-step loops: the cluster-resident loop
// (nb_resident.cu, loop mode 3) and the grid-resident loop (nb_gridres.cu, loop mode 4).  Both keep the owned
// particles of a CTA in its shared memory, evaluate the active particles against the owned records (res_eval)
// and correct them with the corrector spread over a warp (correct_warp).
#pragma once
#include "nb_internal.cuh"
#include "nb_force_dev.cuh"
#include "nb_step_dev.cuh"

namespace nb {

// One active particle (record ri, read from its owner's shared memory) against the owned records
// jl, jl + JL, ...: the pair body of the other drivers; the JL lanes that share it are combined by the butterfly.
template <int JL, bool GUARD0, int MX>
__device__ __forceinline__ Acc9 res_eval(const double *ri, const double *rec, const int jl, const int NL, const double eps2)
{
    const double xi = ri[0], yi = ri[1], zi = ri[2], vxi = ri[3], vyi = ri[4], vzi = ri[5];
    const double axi = ri[6], ayi = ri[7], azi = ri[8];
    Acc9 T = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    const double *q = rec + jl * REC;
    const int per = NL / JL;
    if (MX == 1 || MX == 3) {
        const float eps2f = (float)eps2;
        for (int j0 = 0; j0 < per; j0 += 128) {        // float sums over at most 128 pair terms, as in force_item
            AccF A = {0, 0, 0, 0, 0, 0, 0, 0, 0};
            const int j1 = min(per, j0 + 128);
#pragma unroll 4
            for (int jj = j0; jj < j1; ++jj)
                pair_body_mx<GUARD0, MX == 3>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + (size_t)jj * (JL * REC), eps2f, A, T);
            if (MX == 1) {
                T.ax += (double)A.ax; T.ay += (double)A.ay; T.az += (double)A.az;
                T.jx += (double)A.jx; T.jy += (double)A.jy; T.jz += (double)A.jz;
            }
            T.sx += (double)A.sx; T.sy += (double)A.sy; T.sz += (double)A.sz;
        }
    } else {
        if (per == 2) {   // the usual case of a small system (64 records per CTA, 32 lanes per i): the two pairs overlap
            pair_body<GUARD0, true>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q, eps2, T);
            pair_body<GUARD0, true>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + (size_t)(JL * REC), eps2, T);
        } else {
#pragma unroll 8
            for (int jj = 0; jj < per; ++jj)
                pair_body<GUARD0, true>(xi, yi, zi, vxi, vyi, vzi, axi, ayi, azi, q + (size_t)jj * (JL * REC), eps2, T);
        }
    }
    if (MX == 0) {  // the FP64 pair body accumulates 3 sqrt(3) times the sums (pair_body)
        T.ax *= PAIR_SCALE; T.ay *= PAIR_SCALE; T.az *= PAIR_SCALE;
        T.jx *= PAIR_SCALE; T.jy *= PAIR_SCALE; T.jz *= PAIR_SCALE;
        T.sx *= PAIR_SCALE; T.sy *= PAIR_SCALE; T.sz *= PAIR_SCALE;
    }
    if (JL > 1) {
#pragma unroll
        for (int off = JL >> 1; off > 0; off >>= 1) {
            T.ax += __shfl_xor_sync(0xffffffffu, T.ax, off); T.ay += __shfl_xor_sync(0xffffffffu, T.ay, off);
            T.az += __shfl_xor_sync(0xffffffffu, T.az, off); T.jx += __shfl_xor_sync(0xffffffffu, T.jx, off);
            T.jy += __shfl_xor_sync(0xffffffffu, T.jy, off); T.jz += __shfl_xor_sync(0xffffffffu, T.jz, off);
            T.sx += __shfl_xor_sync(0xffffffffu, T.sx, off); T.sy += __shfl_xor_sync(0xffffffffu, T.sy, off);
            T.sz += __shfl_xor_sync(0xffffffffu, T.sz, off);
        }
    }
    return T;
}

// correct_one (nb_step_dev.cuh: Eq. 11-14, the end-point derivatives G6, the time-step rule Eq. 15-16) spread over
// a warp to shorten its dependent chain: lanes 0..2 take one component each, lanes 0..5 one of the six norms of
// Eq. 16 each, lane 0 the decision.  Same expressions, same rounding order as correct_one.
__device__ __forceinline__ void correct_warp(const int lane, const int k, const int i, const int NL, const double t_next,
                                             const double eta, const double dt_min, const double dt_max, const double *f1,
                                             double *ti, double *dti, double *r, double *v, double *a, double *j, double *s,
                                             double *c)
{
    const double h = dti[i];
    double val[6] = {0, 0, 0, 0, 0, 0};   // a1, j1, s1, a^(3), a^(4), a^(5) of this lane's component
    if (lane < 3) {
        const int d = lane;
        const double h2 = h * h, h3 = h2 * h;
        // 1 / h for h = 2^k, exactly, from the exponent field (an IEEE division is a few hundred cycles of dependent
        // instructions on the path every owner walks between two barriers): bits(2^-k) = (2046 << 52) - bits(2^k)
        const double ih = __longlong_as_double((2046LL << 52) - __double_as_longlong(h));
        const double ih3 = ih * ih * ih, ih4 = ih3 * ih, ih5 = ih4 * ih;
        const int q = d * NL + i;
        const double r0 = r[q], v0 = v[q], a0 = a[q], j0 = j[q], s0 = s[q];
        const double a1 = f1[(0 + d) * NL + k], j1 = f1[(3 + d) * NL + k], s1 = f1[(6 + d) * NL + k];
        const double vc = v0 + (h * 0.5) * (a1 + a0) - (h2 * 0.1) * (j1 - j0) + (h3 * (1.0 / 120.0)) * (s1 + s0);
        const double rc = r0 + (h * 0.5) * (vc + v0) - (h2 * 0.1) * (a1 - a0) + (h3 * (1.0 / 120.0)) * (j1 + j0);
        const double dA = a1 - a0;
        val[0] = a1; val[1] = j1; val[2] = s1;
        val[3] = 3.0 * (20.0 * dA - h * (8.0 * j0 + 12.0 * j1) + h2 * (3.0 * s1 - s0)) * ih3;
        val[4] = 12.0 * (30.0 * dA - h * (14.0 * j0 + 16.0 * j1) + h2 * (3.0 * s1 - 2.0 * s0)) * ih4;
        val[5] = 60.0 * (12.0 * dA - 6.0 * h * (j0 + j1) + h2 * (s1 - s0)) * ih5;
        r[q] = rc; v[q] = vc; a[q] = a1; j[q] = j1; s[q] = s1; c[q] = val[3];
    }
    double nrm = 0.0;
#pragma unroll
    for (int X = 0; X < 6; ++X) {
        const double x = __shfl_sync(0xffffffffu, val[X], 0), y = __shfl_sync(0xffffffffu, val[X], 1),
                     z = __shfl_sync(0xffffffffu, val[X], 2);
        if (lane == X) nrm = norm3_rn(x, y, z);
    }
    double n6[6];
#pragma unroll
    for (int X = 0; X < 6; ++X) n6[X] = __shfl_sync(0xffffffffu, nrm, X);
    if (lane == 0) {
        ti[i] = t_next;
        dti[i] = new_dt(n6[0], n6[1], n6[2], n6[3], n6[4], n6[5], eta, h, t_next, dt_min, dt_max);
    }
}

}  // namespace nb
