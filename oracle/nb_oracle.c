/*
 * nb_oracle.c -- CPU ORACLE for the HiGPUs hot path (arXiv 1207.2367).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_1207_2367_b200/csrc/ and neither side includes the other.
 *
 * What it is: a plain, slow, obviously-correct restatement of what the paper
 * computes, written from PAPER.md, one function per passage:
 *
 *   orc_force            Eq. 8-10 with the Eq. 2 softening
 *   orc_force_mixed      the same in the paper's mixed precision (reading G27)
 *   orc_predict          Eq. 3-7
 *   orc_correct_particle Eq. 11-14 + end-point derivatives of the
 *                        quintic Hermite interpolant (reading G6)
 *   orc_timestep         Eq. 15-16 + power-of-two quantisation
 *   orc_next_block       Table 1 row 1
 *   orc_energy           Eq. 2, Eq. 20
 *   orc_startup/orc_step/orc_run_until   the Hermite loop of PAPER.md:54-102 (P-E-C once)
 *
 * Arithmetic: every floating-point step is done in `long double` (x87 80-bit,
 * 64-bit mantissa) and rounded to double once when stored, EXCEPT the time-step
 * decision (orc_timestep / orc_initial_dt), which is an integer decision and is
 * taken in plain IEEE double, operation by operation (-ffp-contract=off), the
 * precision the CUDA path also takes it in.  There is no blocking, tiling, fusion
 * or reordering: loops run in index order; OpenMP only distributes independent i.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md section "Oracle pins".
 * Free choices of this build where the paper is silent (listed in DESIGN.md): the CHOICE of the
 * initial time-step rule and of eta_init (G8) -- the arithmetic of the stated rule is pinned by
 * hand-computed cases (tests/test_oracle_integrator.py::test_initial_dt_hand_cases); the
 * whole-trajectory values of config 1 are compared oracle <-> GPU only ("parity unpinned by the
 * paper": it prints no trajectory).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* The arithmetic type.  The oracle IS the long-double build (the default).  bench.py also times a second
 * build of this same file with -DORC_REAL=double -DORC_SQRT=sqrt -O3 -march=native, as a plain-double CPU
 * baseline for the throughput table only; no test compares against that build.                       */
#ifndef ORC_REAL
#define ORC_REAL long double
#define ORC_SQRT sqrtl
#endif
typedef ORC_REAL ld;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------------ */
/* Evaluation step.  PAPER.md:72-81, Eq. 8-10; softening of Eq. 2 enters every
 * r_ij^2 (reading G3).  r_ij = r_j - r_i, v_ij = v_j - v_i, a_ij = a_j - a_i on
 * PREDICTED data.  G = 1.  j = i is skipped by index.
 * idx == NULL means i = 0 .. n_idx-1.  Outputs are [n_idx][3].                 */
void orc_force(int64_t N, const double *rp, const double *vp, const double *ap,
               const double *mass, double eps, const int32_t *idx, int64_t n_idx,
               double *acc, double *jerk, double *snap)
{
    const ld eps2 = (ld)eps * (ld)eps;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < n_idx; ++k) {
        const int64_t i = idx ? (int64_t)idx[k] : k;
        ld A0[3] = {0, 0, 0}, A1[3] = {0, 0, 0}, A2[3] = {0, 0, 0};
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            ld r[3], v[3], a[3];
            for (int d = 0; d < 3; ++d) {
                r[d] = (ld)rp[3 * j + d] - (ld)rp[3 * i + d];
                v[d] = (ld)vp[3 * j + d] - (ld)vp[3 * i + d];
                a[d] = (ld)ap[3 * j + d] - (ld)ap[3 * i + d];
            }
            const ld s = r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + eps2; /* r_ij^2 (+eps^2) */
            const ld r3 = s * ORC_SQRT(s);                                  /* r_ij^3          */
            const ld rv = r[0] * v[0] + r[1] * v[1] + r[2] * v[2];
            const ld vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
            const ld ra = r[0] * a[0] + r[1] * a[1] + r[2] * a[2];
            const ld alpha = rv / s;                       /* alpha r^2 = r.v            */
            const ld beta = (vv + ra) / s + alpha * alpha; /* beta r^2 = v^2 + r.a + alpha^2 r^2 */
            const ld mj = (ld)mass[j];
            for (int d = 0; d < 3; ++d) {
                const ld a0 = mj * r[d] / r3;                                  /* Eq. 8  */
                const ld a1 = mj * v[d] / r3 - 3.0L * alpha * a0;              /* Eq. 9  */
                const ld a2 = mj * a[d] / r3 - 6.0L * alpha * a1 - 3.0L * beta * a0; /* Eq. 10 */
                A0[d] += a0;
                A1[d] += a1;
                A2[d] += a2;
            }
        }
        for (int d = 0; d < 3; ++d) {
            if (acc) acc[3 * k + d] = (double)A0[d];
            if (jerk) jerk[3 * k + d] = (double)A1[d];
            if (snap) snap[3 * k + d] = (double)A2[d];
        }
    }
}

/* ------------------------------------------------------------------------ */
/* Evaluation step in the paper's MIXED precision (section 5.7: "store predicted
 * positions, accelerations and derivatives [in double], while it computes partial results in
 * single precision mode using 32 bit registers"; 15 DP + 82 SP operations per pair,
 * PAPER.md:301).  Reading G27: the nine differences r_ij, v_ij, a_ij are formed in
 * double from the double predicted data and rounded to float; everything of Eq. 8-10 for the
 * pair (r^2 + eps^2, r^3, alpha, beta, the three pair terms) is float arithmetic, one rounded
 * operation at a time in the order written; the pair terms are summed over j in long double
 * (so that the sum itself adds no error: what is measured is the SP pair arithmetic).
 * scale (may be NULL) [n_idx][3] receives sum_j |pair term|_2 for acc, jerk, snap: the
 * magnitude any forward error bound of a float evaluation is relative to.              */
void orc_force_mixed(int64_t N, const double *rp, const double *vp, const double *ap,
                     const double *mass, double eps, const int32_t *idx, int64_t n_idx,
                     double *acc, double *jerk, double *snap, double *scale)
{
    const float eps2 = (float)eps * (float)eps;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < n_idx; ++k) {
        const int64_t i = idx ? (int64_t)idx[k] : k;
        ld A0[3] = {0, 0, 0}, A1[3] = {0, 0, 0}, A2[3] = {0, 0, 0}, sc[3] = {0, 0, 0};
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            float r[3], v[3], a[3];
            for (int d = 0; d < 3; ++d) {
                r[d] = (float)(rp[3 * j + d] - rp[3 * i + d]); /* DP difference, then SP */
                v[d] = (float)(vp[3 * j + d] - vp[3 * i + d]);
                a[d] = (float)(ap[3 * j + d] - ap[3 * i + d]);
            }
            const float s = r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + eps2;
            const float r3 = s * sqrtf(s);
            const float rv = r[0] * v[0] + r[1] * v[1] + r[2] * v[2];
            const float vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
            const float ra = r[0] * a[0] + r[1] * a[1] + r[2] * a[2];
            const float alpha = rv / s;
            const float beta = (vv + ra) / s + alpha * alpha;
            const float mj = (float)mass[j];
            float t0[3], t1[3], t2[3];
            for (int d = 0; d < 3; ++d) {
                t0[d] = mj * r[d] / r3;                                       /* Eq. 8  */
                t1[d] = mj * v[d] / r3 - 3.0f * alpha * t0[d];                /* Eq. 9  */
                t2[d] = mj * a[d] / r3 - 6.0f * alpha * t1[d] - 3.0f * beta * t0[d]; /* Eq. 10 */
                A0[d] += (ld)t0[d];
                A1[d] += (ld)t1[d];
                A2[d] += (ld)t2[d];
            }
            sc[0] += sqrtl((ld)t0[0] * t0[0] + (ld)t0[1] * t0[1] + (ld)t0[2] * t0[2]);
            sc[1] += sqrtl((ld)t1[0] * t1[0] + (ld)t1[1] * t1[1] + (ld)t1[2] * t1[2]);
            sc[2] += sqrtl((ld)t2[0] * t2[0] + (ld)t2[1] * t2[1] + (ld)t2[2] * t2[2]);
        }
        for (int d = 0; d < 3; ++d) {
            if (acc) acc[3 * k + d] = (double)A0[d];
            if (jerk) jerk[3 * k + d] = (double)A1[d];
            if (snap) snap[3 * k + d] = (double)A2[d];
            if (scale) scale[3 * k + d] = (double)sc[d];
        }
    }
}

/* ------------------------------------------------------------------------ */
/* Prediction step.  PAPER.md:58-69, Eq. 3-7, with the garbled dots read as the
 * Taylor series (G1) and the interval taken as t - t_j for every particle (G2). */
void orc_predict(int64_t N, double t, const double *ti, const double *r, const double *v,
                 const double *a, const double *j, const double *s, const double *c,
                 double *rp, double *vp, double *ap)
{
    for (int64_t i = 0; i < N; ++i) {
        const ld h = (ld)t - (ld)ti[i];
        const ld h2 = h * h, h3 = h2 * h, h4 = h3 * h, h5 = h4 * h;
        for (int d = 0; d < 3; ++d) {
            const int64_t q = 3 * i + d;
            rp[q] = (double)((ld)r[q] + (ld)v[q] * h + (ld)a[q] * h2 / 2.0L + (ld)j[q] * h3 / 6.0L +
                             (ld)s[q] * h4 / 24.0L + (ld)c[q] * h5 / 120.0L);
            vp[q] = (double)((ld)v[q] + (ld)a[q] * h + (ld)j[q] * h2 / 2.0L + (ld)s[q] * h3 / 6.0L +
                             (ld)c[q] * h4 / 24.0L);
            ap[q] = (double)((ld)a[q] + (ld)j[q] * h + (ld)s[q] * h2 / 2.0L + (ld)c[q] * h3 / 6.0L);
        }
    }
}

/* ------------------------------------------------------------------------ */
/* Correction step for ONE particle.  PAPER.md:83-91, Eq. 11-14 (v first, r uses
 * v_corr).  Index 0 = values stored at t_i, index 1 = evaluated at t_i + h.
 * Then the 3rd..5th derivatives of the acceleration at the END of the step from
 * the quintic Hermite interpolant through (a, jerk, snap) at both ends (G6).    */
void orc_correct_particle(double h_, const double *r0, const double *v0, const double *a0,
                          const double *j0, const double *s0, const double *a1, const double *j1,
                          const double *s1, double *r1, double *v1, double *c3, double *c4,
                          double *c5)
{
    const ld h = (ld)h_;
    const ld h2 = h * h, h3 = h2 * h, h4 = h3 * h, h5 = h4 * h;
    for (int d = 0; d < 3; ++d) {
        const ld A0 = a0[d], A1 = a1[d], J0 = j0[d], J1 = j1[d], S0 = s0[d], S1 = s1[d];
        const ld vc = (ld)v0[d] + h / 2.0L * (A1 + A0) - h2 / 10.0L * (J1 - J0) +
                      h3 / 120.0L * (S1 + S0); /* Eq. 11-12 */
        const ld rc = (ld)r0[d] + h / 2.0L * (vc + (ld)v0[d]) - h2 / 10.0L * (A1 - A0) +
                      h3 / 120.0L * (J1 + J0); /* Eq. 13-14 */
        v1[d] = (double)vc;
        r1[d] = (double)rc;
        const ld dA = A1 - A0;
        c3[d] = (double)(3.0L * (20.0L * dA - h * (8.0L * J0 + 12.0L * J1) + h2 * (3.0L * S1 - S0)) / h3);
        c4[d] = (double)(12.0L * (30.0L * dA - h * (14.0L * J0 + 16.0L * J1) + h2 * (3.0L * S1 - 2.0L * S0)) / h4);
        c5[d] = (double)(60.0L * (12.0L * dA - 6.0L * h * (J0 + J1) + h2 * (S1 - S0)) / h5);
    }
}

/* ------------------------------------------------------------------------ */
/* Time-step rule.  PAPER.md:93-102: generalized Aarseth criterion, Eq. 15-16 with
 * p = 6 (exponent read as 1/(p-3), G5), quantised to a power of two (G9):
 *   x = eta^3 A(1)/A(4);  dt_q = 2^floor(ilogb(x)/3)  (largest 2^k <= eta (A1/A4)^(1/3));
 *   dt = min(dt_q, 2 dt_old); growth only if t_next is a multiple of 2 dt_old;
 *   clamp to [dt_min, dt_max].  PLAIN DOUBLE on purpose (integer decision).     */
static double norm3(const double *x) { return sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]); }

static int floordiv3(int e) { return (e >= 0) ? e / 3 : -((-e + 2) / 3); }

double orc_timestep(const double *a, const double *j, const double *s, const double *c3,
                    const double *c4, const double *c5, double eta, double dt_old, double t_next,
                    double dt_min, double dt_max)
{
    const double A1 = sqrt(norm3(a) * norm3(s) + norm3(j) * norm3(j));    /* A^(1), Eq. 16 */
    const double A4 = sqrt(norm3(c3) * norm3(c5) + norm3(c4) * norm3(c4)); /* A^(4)         */
    double dt_q;
    if (!(A4 > 0.0)) {
        dt_q = dt_max;
    } else {
        const double x = eta * eta * eta * A1 / A4;
        if (!(x > 0.0)) dt_q = dt_min;
        else if (isinf(x)) dt_q = dt_max;
        else dt_q = ldexp(1.0, floordiv3(ilogb(x)));
    }
    double dt = dt_q < 2.0 * dt_old ? dt_q : 2.0 * dt_old;
    if (dt > dt_old && fmod(t_next, 2.0 * dt_old) != 0.0) dt = dt_old;
    if (dt < dt_min) dt = dt_min;
    if (dt > dt_max) dt = dt_max;
    return dt;
}

/* Start-up step (paper silent; reading G8; pinned by hand-computed cases):
 * dt = pow2floor(eta_init * min(|a|/|jerk|, sqrt(|a|/|snap|))), clamped.         */
double orc_initial_dt(const double *a, const double *j, const double *s, double eta_init,
                      double dt_min, double dt_max)
{
    const double na = norm3(a), nj = norm3(j), ns = norm3(s);
    double q = INFINITY;
    if (nj > 0.0) q = na / nj;
    if (ns > 0.0) {
        const double q2 = sqrt(na / ns);
        if (q2 < q) q = q2;
    }
    double dt;
    if (isinf(q)) dt = dt_max;
    else {
        const double x = eta_init * q;
        dt = (x > 0.0) ? ldexp(1.0, ilogb(x)) : dt_min;
    }
    if (dt < dt_min) dt = dt_min;
    if (dt > dt_max) dt = dt_max;
    return dt;
}

/* ------------------------------------------------------------------------ */
/* Diagnostics.  PAPER.md:40 (Eq. 2) and 138 (Eq. 20): out = E, K, W, P[3], L[3].
 * W = - sum_{i<j} m_i m_j / sqrt(r_ij^2 + eps^2).                              */
void orc_energy(int64_t N, const double *r, const double *v, const double *mass, double eps,
                double *out)
{
    const ld eps2 = (ld)eps * (ld)eps;
    ld K = 0, W = 0, P[3] = {0, 0, 0}, L[3] = {0, 0, 0};
    for (int64_t i = 0; i < N; ++i) {
        const ld m = mass[i];
        const ld x = r[3 * i], y = r[3 * i + 1], z = r[3 * i + 2];
        const ld vx = v[3 * i], vy = v[3 * i + 1], vz = v[3 * i + 2];
        K += 0.5L * m * (vx * vx + vy * vy + vz * vz);
        P[0] += m * vx; P[1] += m * vy; P[2] += m * vz;
        L[0] += m * (y * vz - z * vy);
        L[1] += m * (z * vx - x * vz);
        L[2] += m * (x * vy - y * vx);
    }
#pragma omp parallel
    {
        ld Wloc = 0;
#pragma omp for schedule(dynamic, 64)
        for (int64_t i = 0; i < N; ++i) {
            ld wi = 0;
            for (int64_t j = i + 1; j < N; ++j) {
                const ld dx = (ld)r[3 * j] - (ld)r[3 * i];
                const ld dy = (ld)r[3 * j + 1] - (ld)r[3 * i + 1];
                const ld dz = (ld)r[3 * j + 2] - (ld)r[3 * i + 2];
                wi += (ld)mass[j] / ORC_SQRT(dx * dx + dy * dy + dz * dz + eps2);
            }
            Wloc -= (ld)mass[i] * wi;
        }
#pragma omp critical
        W += Wloc;
    }
    out[0] = (double)(K + W); out[1] = (double)K; out[2] = (double)W;
    for (int d = 0; d < 3; ++d) { out[3 + d] = (double)P[d]; out[6 + d] = (double)L[d]; }
}

/* ------------------------------------------------------------------------ */
/* The integrator state and loop.                           */
typedef struct {
    int64_t N;
    double eps, eta, eta_init, dt_min, dt_max;
    double t_now;
    double *m, *t, *dt;               /* [N]    */
    double *r, *v, *a, *j, *s, *c;    /* [N][3] state at t_i */
    double *rp, *vp, *ap;             /* [N][3] predicted                     */
    double *a1, *j1, *s1;             /* [N][3] evaluated (active rows only)   */
    int32_t *active; int64_t n_active; double t_next;
    int started;
    /* statistics */
    int64_t n_steps; double n_pairs; int64_t hist[64];
} orc_state;

static double *dalloc(int64_t n) { return (double *)calloc((size_t)n, sizeof(double)); }

orc_state *orc_create(int64_t N, const double *pos, const double *vel, const double *mass,
                      double eps, double eta)
{
    orc_state *st = (orc_state *)calloc(1, sizeof(orc_state));
    st->N = N; st->eps = eps; st->eta = eta; st->eta_init = 0.01;
    st->dt_min = ldexp(1.0, -25);
    st->dt_max = ldexp(1.0, -3);
    st->m = dalloc(N); st->t = dalloc(N); st->dt = dalloc(N);
    st->r = dalloc(3 * N); st->v = dalloc(3 * N); st->a = dalloc(3 * N);
    st->j = dalloc(3 * N); st->s = dalloc(3 * N); st->c = dalloc(3 * N);
    st->rp = dalloc(3 * N); st->vp = dalloc(3 * N); st->ap = dalloc(3 * N);
    st->a1 = dalloc(3 * N); st->j1 = dalloc(3 * N); st->s1 = dalloc(3 * N);
    st->active = (int32_t *)calloc((size_t)N, sizeof(int32_t));
    memcpy(st->m, mass, (size_t)N * sizeof(double));
    memcpy(st->r, pos, (size_t)(3 * N) * sizeof(double));
    memcpy(st->v, vel, (size_t)(3 * N) * sizeof(double));
    return st;
}

void orc_destroy(orc_state *st)
{
    if (!st) return;
    free(st->m); free(st->t); free(st->dt);
    free(st->r); free(st->v); free(st->a); free(st->j); free(st->s); free(st->c);
    free(st->rp); free(st->vp); free(st->ap); free(st->a1); free(st->j1); free(st->s1);
    free(st->active); free(st);
}

void orc_set_limits(orc_state *st, double dt_min, double dt_max, double eta_init)
{
    st->dt_min = dt_min; st->dt_max = dt_max; st->eta_init = eta_init;
}

/* Start-up (G8): pass 1 with a_pred = 0 gives a, jerk; pass 2 with a_pred = a
 * gives snap; crackle = 0; then the initial step of every particle.            */
void orc_startup(orc_state *st)
{
    const int64_t N = st->N;
    memcpy(st->rp, st->r, (size_t)(3 * N) * sizeof(double));
    memcpy(st->vp, st->v, (size_t)(3 * N) * sizeof(double));
    memset(st->ap, 0, (size_t)(3 * N) * sizeof(double));
    orc_force(N, st->rp, st->vp, st->ap, st->m, st->eps, NULL, N, st->a, st->j, NULL);
    memcpy(st->ap, st->a, (size_t)(3 * N) * sizeof(double));
    orc_force(N, st->rp, st->vp, st->ap, st->m, st->eps, NULL, N, st->a, st->j, st->s);
    st->n_pairs += 2.0 * (double)N * (double)N;
    for (int64_t i = 0; i < N; ++i) {
        st->t[i] = 0.0;
        st->c[3 * i] = st->c[3 * i + 1] = st->c[3 * i + 2] = 0.0;
        st->dt[i] = orc_initial_dt(st->a + 3 * i, st->j + 3 * i, st->s + 3 * i, st->eta_init,
                                   st->dt_min, st->dt_max);
    }
    st->t_now = 0.0;
    st->started = 1;
}

/* Table 1 row 1: the particles due at the next block time.      */
double orc_next_block(orc_state *st)
{
    const int64_t N = st->N;
    double tn = INFINITY;
    for (int64_t i = 0; i < N; ++i) {
        const double x = st->t[i] + st->dt[i];
        if (x < tn) tn = x;
    }
    int64_t m = 0;
    for (int64_t i = 0; i < N; ++i)
        if (st->t[i] + st->dt[i] == tn) st->active[m++] = (int32_t)i;
    st->n_active = m; st->t_next = tn;
    return tn;
}

/* One block step: predict all (Eq. 3-7), evaluate the active set once (Eq. 8-10),
 * correct it (Eq. 11-14), new steps (Eq. 15-16).  Stored a, jerk, snap become the
 * evaluated values (G16); crackle becomes the interpolated a^(3)(t1) (G7).       */
void orc_step(orc_state *st)
{
    const int64_t N = st->N;
    orc_next_block(st);
    const double tn = st->t_next;
    const int64_t m = st->n_active;
    orc_predict(N, tn, st->t, st->r, st->v, st->a, st->j, st->s, st->c, st->rp, st->vp, st->ap);
    orc_force(N, st->rp, st->vp, st->ap, st->m, st->eps, st->active, m, st->a1, st->j1, st->s1);
    for (int64_t k = 0; k < m; ++k) {
        const int64_t i = st->active[k];
        double r1[3], v1[3], c3[3], c4[3], c5[3];
        const double h = st->dt[i];
        orc_correct_particle(h, st->r + 3 * i, st->v + 3 * i, st->a + 3 * i, st->j + 3 * i,
                             st->s + 3 * i, st->a1 + 3 * k, st->j1 + 3 * k, st->s1 + 3 * k, r1, v1,
                             c3, c4, c5);
        for (int d = 0; d < 3; ++d) {
            st->r[3 * i + d] = r1[d]; st->v[3 * i + d] = v1[d];
            st->a[3 * i + d] = st->a1[3 * k + d];
            st->j[3 * i + d] = st->j1[3 * k + d];
            st->s[3 * i + d] = st->s1[3 * k + d];
            st->c[3 * i + d] = c3[d];
        }
        st->t[i] = tn;
        st->dt[i] = orc_timestep(st->a + 3 * i, st->j + 3 * i, st->s + 3 * i, c3, c4, c5, st->eta,
                                 h, tn, st->dt_min, st->dt_max);
    }
    st->t_now = tn;
    st->n_steps += 1;
    st->n_pairs += (double)m * (double)N;
    int b = 0; while ((((int64_t)1) << (b + 1)) <= m) ++b;
    st->hist[b] += 1;
}

/* Repeat block steps while the next block time does not exceed t_end.
 * Optional log of (t_next, m) per step, up to log_cap entries.                  */
int64_t orc_run_until(orc_state *st, double t_end, double *log_t, int64_t *log_m, int64_t log_cap)
{
    int64_t n = 0;
    if (!st->started) orc_startup(st);
    for (;;) {
        orc_next_block(st);
        if (st->t_next > t_end) break;
        orc_step(st);
        if (n < log_cap) { if (log_t) log_t[n] = st->t_now; if (log_m) log_m[n] = st->n_active; }
        ++n;
    }
    return n;
}

/* accessors for the Python wrapper */
#define GETTER(name, field, count) \
    void orc_get_##name(const orc_state *st, double *out) { memcpy(out, st->field, (size_t)(count) * sizeof(double)); }
GETTER(mass, m, st->N) GETTER(t, t, st->N) GETTER(dt, dt, st->N)
GETTER(pos, r, 3 * st->N) GETTER(vel, v, 3 * st->N) GETTER(acc, a, 3 * st->N)
GETTER(jerk, j, 3 * st->N) GETTER(snap, s, 3 * st->N) GETTER(crackle, c, 3 * st->N)
GETTER(pos_pred, rp, 3 * st->N) GETTER(vel_pred, vp, 3 * st->N) GETTER(acc_pred, ap, 3 * st->N)
double orc_t_now(const orc_state *st) { return st->t_now; }
double orc_t_next(const orc_state *st) { return st->t_next; }
int64_t orc_n_active(const orc_state *st) { return st->n_active; }
void orc_get_active(const orc_state *st, int32_t *out) { memcpy(out, st->active, (size_t)st->n_active * sizeof(int32_t)); }
int64_t orc_n_steps(const orc_state *st) { return st->n_steps; }
double orc_n_pairs(const orc_state *st) { return st->n_pairs; }
void orc_get_hist(const orc_state *st, int64_t *out) { memcpy(out, st->hist, sizeof(st->hist)); }
/* Energy of the committed state; meaningful when all particles share one time. */
void orc_state_energy(const orc_state *st, double *out) { orc_energy(st->N, st->r, st->v, st->m, st->eps, out); }
