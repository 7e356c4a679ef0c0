"""Pins of the oracle's predictor, corrector, time-step rule, scheduler and energy
(oracle/nb_oracle.c).  Routes independent of the oracle's own formulas: polynomial
integration by numpy.polynomial, the Kepler closed form (Kepler's equation), hand-computed
time-step cases, scheduler invariants, convergence order and energy-vs-eta scaling."""
import math

import numpy as np
import pytest
from numpy.polynomial import Polynomial as P

from workloads import kepler_binary, plummer


# ---------------------------------------------------------------- predictor (Eq. 3-7)
def test_predictor_exact_for_cubic_acceleration(oracle):
    # a(t) cubic => r(t) quintic: Eq. 3-7 must reproduce the polynomial exactly (G1 reading:
    # 1/24 snap dt^4 + 1/120 crackle dt^5 in r; 1/6, 1/24 in v; 1/2, 1/6 in a).
    rng = np.random.default_rng(0)
    N = 5
    t0 = rng.choice([0.0, 0.125, 0.25, 0.375], size=N)
    t = 0.5
    R0 = rng.normal(size=(N, 3)); V0 = rng.normal(size=(N, 3))
    coef = rng.normal(size=(N, 3, 4))  # a(tau) = sum_k coef[k] tau^k, tau = t - t0
    a = coef[:, :, 0].copy(); j = coef[:, :, 1].copy(); s = 2 * coef[:, :, 2]; c = 6 * coef[:, :, 3]
    rp, vp, ap = oracle.predict(t, t0, R0, V0, a, j, s, c)
    for i in range(N):
        for d in range(3):
            pa = P(coef[i, d]); pv = pa.integ(1, k=[V0[i, d]]); pr = pv.integ(1, k=[R0[i, d]])
            tau = t - t0[i]
            assert ap[i, d] == pytest.approx(pa(tau), rel=1e-14, abs=1e-15)
            assert vp[i, d] == pytest.approx(pv(tau), rel=1e-14, abs=1e-15)
            assert rp[i, d] == pytest.approx(pr(tau), rel=1e-14, abs=1e-15)


def test_predictor_zero_interval_is_identity(oracle):
    rng = np.random.default_rng(1)
    x = [rng.normal(size=(4, 3)) for _ in range(6)]
    rp, vp, ap = oracle.predict(0.25, np.full(4, 0.25), *x)
    assert np.array_equal(rp, x[0]) and np.array_equal(vp, x[1]) and np.array_equal(ap, x[2])


# ---------------------------------------------------------------- corrector (Eq. 11-14) + G6
@pytest.mark.parametrize("deg", [3, 4, 5])
def test_corrector_exact_for_polynomial_acceleration(oracle, deg):
    # For a(t) a polynomial of degree <= 5 the quintic Hermite interpolant IS a(t):
    # v1 exact (Eq. 11-12 integrate the interpolant), a^(3,4,5)(t1) exact, r1 exact for degree <= 4.
    rng = np.random.default_rng(deg)
    h = 0.375
    r0 = rng.normal(size=3); v0 = rng.normal(size=3)
    coef = rng.normal(size=(3, deg + 1))
    pa = [P(coef[d]) for d in range(3)]
    a0 = np.array([p(0.0) for p in pa]); j0 = np.array([p.deriv(1)(0.0) for p in pa])
    s0 = np.array([p.deriv(2)(0.0) for p in pa])
    a1 = np.array([p(h) for p in pa]); j1 = np.array([p.deriv(1)(h) for p in pa])
    s1 = np.array([p.deriv(2)(h) for p in pa])
    r1, v1, c3, c4, c5 = oracle.correct_particle(h, r0, v0, a0, j0, s0, a1, j1, s1)
    for d in range(3):
        pv = pa[d].integ(1, k=[v0[d]]); pr = pv.integ(1, k=[r0[d]])
        assert v1[d] == pytest.approx(pv(h), rel=1e-13, abs=1e-14)
        assert c3[d] == pytest.approx(pa[d].deriv(3)(h), rel=1e-10, abs=1e-10)
        assert c4[d] == pytest.approx(pa[d].deriv(4)(h) if deg >= 4 else 0.0, rel=1e-9, abs=1e-9)
        assert c5[d] == pytest.approx(pa[d].deriv(5)(h) if deg >= 5 else 0.0, rel=1e-8, abs=1e-8)
        if deg <= 4:
            assert r1[d] == pytest.approx(pr(h), rel=1e-13, abs=1e-14)
        else:  # Eq. 13-14 truncate at h^7: the degree-5 term leaves an O(h^7) residue
            assert abs(r1[d] - pr(h)) < abs(coef[d, 5]) * h ** 7


# ---------------------------------------------------------------- time-step rule (Eq. 15-16)
def _vecs(A1, A4):
    # a = snap = (A1,0,0), jerk = 0  => A(1) = sqrt(|a||snap|) = A1; likewise A(4) = A4
    z = np.zeros(3)
    a = np.array([A1, 0, 0.0]); c = np.array([0, A4, 0.0])
    return a, z, a, c, z, c


def test_timestep_hand_cases(oracle):
    lo, hi = 2.0 ** -25, 2.0 ** -3
    # eta = 1: dt* = (A1/A4)^(1/3).  A1/A4 = 8^-2 exactly -> 2^-2, clamped to dt_max? no: old=2^-6
    f = lambda A1, A4, eta=1.0, old=2.0 ** -6, tn=1.0, lo=lo, hi=hi: oracle.timestep(*_vecs(A1, A4), eta, old, tn, lo, hi)
    assert f(1.0, 8.0 ** 6) == 2.0 ** -6                       # exactly 2^-6 stays
    assert f(1.0, 8.0 ** 6 * (1 + 2 ** -52)) == 2.0 ** -7      # just below 2^-6 -> floor to 2^-7
    assert f(1.0 + 2 ** -52, 8.0 ** 6) == 2.0 ** -6            # just above stays 2^-6
    assert f(1.0, 8.0 ** 9) == 2.0 ** -9                       # shrinking by several levels at once
    assert f(1.0, 8.0 ** 2, tn=1.0) == 2.0 ** -5               # growth limited to one doubling
    assert f(1.0, 8.0 ** 2, tn=1.0 + 2.0 ** -6) == 2.0 ** -6   # doubling refused: t not multiple of 2 dt_old
    assert f(1.0, 8.0 ** 2, old=hi, tn=1.0) == hi              # clamp at dt_max
    assert f(1.0, 8.0 ** 40, old=2.0 ** -24) == lo             # clamp at dt_min
    assert f(1.0, 0.0) == 2.0 ** -5                            # A(4) = 0 -> dt_max, then doubling rule
    # eta enters as eta^3 inside the floor: eta = 0.5 shifts one level exactly
    assert f(1.0, 8.0 ** 5, eta=0.5) == 2.0 ** -6
    # p = 6 => cube root (G5): A1/A4 = 2^-15 -> 2^-5; a square root would give 2^-8 (wrong)
    assert f(2.0 ** -15, 1.0, old=2.0 ** -5) == 2.0 ** -5


def test_timestep_uses_eq16_norm_combination(oracle):
    # A(1) = sqrt(|a||snap| + |jerk|^2): with |a| = |snap| = 0 only the jerk term survives.
    z = np.zeros(3)
    jerk = np.array([0.0, 3.0, 4.0])      # |jerk| = 5 -> A(1) = 5
    c4 = np.array([5.0 * 8.0 ** 4, 0, 0])  # A(4) = 5 * 8^4 -> x = 8^-4 -> dt = 2^-4
    assert oracle.timestep(z, jerk, z, z, c4, z, 1.0, 2.0 ** -4, 1.0, 2.0 ** -25, 2.0 ** -3) == 2.0 ** -4


# ---------------------------------------------------------------- start-up step (S0, reading G8)
def test_initial_dt_hand_cases(oracle):
    # S0 of SURVEY.md section 8(c): dt = pow2floor(eta_init * min(|a|/|jerk|, sqrt(|a|/|snap|))), clamped;
    # a zero denominator drops its term, both zero -> dt_max.  The paper is silent on the rule (G8), but
    # the arithmetic of the stated rule has hand-computable cases: every expected value below is a power
    # of two worked out by hand, with eta_init itself a power of two so that the products are exact.
    lo, hi = 2.0 ** -25, 2.0 ** -3
    ex, ey, ez = np.array([1.0, 0, 0]), np.array([0, 1.0, 0]), np.array([0, 0, 1.0])
    z = np.zeros(3)
    f = lambda a, j, s, eta=0.25, lo=lo, hi=hi: oracle.initial_dt(a, j, s, eta, lo, hi)
    big = 2.0 ** -40 * ez        # a tiny snap: sqrt(|a|/|snap|) = 2^20, never the minimum
    # jerk term: |a|/|jerk| = 2^-3 exactly -> 0.25 * 2^-3 = 2^-5 stays 2^-5 (floor keeps an exact power)
    assert f(ex, 8.0 * ey, big) == 2.0 ** -5
    assert f(ex, 8.0 * (1 + 2 ** -52) * ey, big) == 2.0 ** -6      # just below 2^-5 -> 2^-6
    assert f((1 + 2 ** -52) * ex, 8.0 * ey, big) == 2.0 ** -5      # just above stays 2^-5
    assert f(1.75 * ex, 8.0 * ey, big) == 2.0 ** -5                # mantissa 1.75: floor, not round (-> 2^-4 if rounded)
    # snap term wins and enters through a SQUARE ROOT: |a|/|snap| = 2^-10 -> sqrt = 2^-5 -> dt = 2^-7
    # (without the sqrt: 0.25 * 2^-10 = 2^-12; with max instead of min: 0.25 * 1 = 2^-2 -> clamp 2^-3)
    assert f(ex, ey, 2.0 ** 10 * ez) == 2.0 ** -7
    # jerk term wins over the snap term (min, not max; not the snap term alone):
    # |a|/|jerk| = 2^-6, sqrt(|a|/|snap|) = 2^-2 -> dt = 0.25 * 2^-6 = 2^-8
    assert f(ex, 64.0 * ey, 16.0 * ez) == 2.0 ** -8
    # the ratio is |a|/|jerk| (not its inverse): |a| = 2^-4, |jerk| = 1 -> 2^-4 -> dt = 2^-6
    assert f(2.0 ** -4 * ex, ey, big) == 2.0 ** -6
    # Euclidean norms of all three components: |a| = |(3,4,12)| = 13, |jerk| = |(0,5,12)|*8 = 104 -> 1/8
    assert f(np.array([3.0, 4.0, 12.0]), 8.0 * np.array([0.0, 5.0, 12.0]), big) == 2.0 ** -5
    # eta_init multiplies the ratio: halving it shifts exactly one level
    assert f(ex, 8.0 * ey, big, eta=0.125) == 2.0 ** -6
    # a zero denominator drops that term
    assert f(ex, z, 2.0 ** 10 * ez) == 2.0 ** -7                    # jerk = 0: snap term alone
    assert f(ex, 8.0 * ey, z) == 2.0 ** -5                          # snap = 0: jerk term alone
    assert f(ex, z, z) == hi                                        # both zero -> dt_max
    assert f(z, z, z) == hi                                         # a particle that feels nothing: dt_max, no 0/0
    # clamps
    assert f(ex, 2.0 ** -10 * ey, big) == hi                        # 0.25 * 2^10 -> clamp at dt_max
    assert f(ex, 2.0 ** 40 * ey, big) == lo                         # 0.25 * 2^-40 -> clamp at dt_min
    assert f(ex, 8.0 * ey, big, lo=2.0 ** -4, hi=2.0 ** -4) == 2.0 ** -4
    # |a| = 0 with a non-zero jerk: the candidate is 0 -> dt_min (no NaN, no log of 0)
    assert f(z, ey, ez) == lo


def test_startup_uses_the_initial_dt_rule_per_particle(oracle):
    # orc_startup assigns dt_i = initial_dt(a_i, jerk_i, snap_i): recompute every particle's step in numpy
    # (plain double: norms, ratio, sqrt, min, floor to a power of two by frexp) from the committed a, jerk, snap.
    pos, vel, m = plummer(96, seed=11)
    eta_init, lo, hi = 0.01, 2.0 ** -25, 2.0 ** -4
    it = oracle.Integrator(pos, vel, m, eps=1e-2, eta=0.45, dt_min=lo, dt_max=hi, eta_init=eta_init)
    na, nj, ns = (np.sqrt((x * x).sum(axis=1)) for x in (it.acc, it.jerk, it.snap))
    x = eta_init * np.minimum(na / nj, np.sqrt(na / ns))
    mant, ex = np.frexp(x)                         # x = mant * 2^ex, mant in [0.5, 1)
    want = np.clip(np.ldexp(0.5, ex), lo, hi)      # largest power of two <= x
    assert np.array_equal(it.dt, want)
    assert len(np.unique(it.dt)) > 2               # the case spans several levels


# ---------------------------------------------------------------- Kepler orbit (closed form)
def _kepler_rel(t, ecc):
    # start at apocentre on +x, a = 1, M = 1: mean anomaly pi + t; pericentre along -x
    Mn = math.pi + t
    E = Mn
    for _ in range(100):
        E -= (E - ecc * math.sin(E) - Mn) / (1 - ecc * math.cos(E))
    return np.array([-(math.cos(E) - ecc), -math.sqrt(1 - ecc * ecc) * math.sin(E), 0.0])


def _kepler_run(oracle, dt, t_end, ecc=0.5):
    pos, vel, m = kepler_binary(ecc)
    it = oracle.Integrator(pos, vel, m, eps=0.0, eta=0.45, dt_min=dt, dt_max=dt)  # shared fixed step
    e0 = it.energy()[0]
    it.run_until(t_end)
    assert np.all(it.t == t_end)
    return it, abs((it.energy()[0] - e0) / e0)


def test_kepler_sixth_order_and_closed_form(oracle):
    t_end = 6.25  # about one period (2 pi), a multiple of every dt used
    errs, perr = [], []
    for k in (5, 6, 7, 8):
        it, de = _kepler_run(oracle, 2.0 ** -k, t_end)
        errs.append(de)
        rel = it.pos[0] - it.pos[1]
        perr.append(np.abs(rel - _kepler_rel(t_end, 0.5)).max())
    # position error against Kepler's equation: 2^6 = 64 per halving = 6th order
    pr = [perr[i] / perr[i + 1] for i in range(3)]
    for r in pr:
        assert 50 < r < 90, (perr, pr)
    # the energy error converges at least as fast (it is super-convergent over a closed orbit)
    ratios = [errs[i] / errs[i + 1] for i in range(2)]
    for r in ratios:
        assert r > 50, (errs, ratios)
    assert perr[-1] < 1e-10 and errs[-1] < 1e-11     # orbit matches Kepler's equation


def test_shared_step_conserves_momentum_to_roundoff(oracle):
    pos, vel, m = plummer(64, seed=3)
    it = oracle.Integrator(pos, vel, m, eps=1e-2, eta=0.45, dt_min=2.0 ** -7, dt_max=2.0 ** -7)
    it.run_until(0.25)
    P = it.energy()[3:6]
    assert np.all(np.abs(P) < 1e-15)


# ---------------------------------------------------------------- scheduler (Table 1 row 1) + block steps
def test_block_step_invariants(oracle):
    pos, vel, m = plummer(128, seed=4)
    lo, hi = 2.0 ** -25, 2.0 ** -4
    it = oracle.Integrator(pos, vel, m, eps=1e-3, eta=0.45, dt_min=lo, dt_max=hi)
    seen_levels = set()
    for _ in range(400):
        tn, act = it.next_block()
        t, dt = it.t, it.dt
        # brute-force restatement of "the particles due next"
        nxt = t + dt
        assert tn == nxt.min()
        assert np.array_equal(act, np.nonzero(nxt == tn)[0].astype(np.int32))
        it.step()
        t, dt = it.t, it.dt
        assert np.all(t <= it.t_now) and it.t_now == tn
        assert np.all((dt >= lo) & (dt <= hi))
        mant, _ = np.frexp(dt)
        assert np.all(mant == 0.5)                       # powers of two
        assert np.all(np.mod(t, dt) == 0.0)              # commensurate: t_i / dt_i integer
        seen_levels.update(np.unique(dt).tolist())
        if math.fmod(it.t_now, hi) == 0.0:
            assert np.all(t == it.t_now)                 # synchronised at multiples of dt_max
    assert len(seen_levels) >= 3


def _paper_fig1_band():
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_fig1_energy_errors.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                eta, q, _, val = line.split()
                out[(float(eta), q)] = float(val)
    return out


def test_energy_error_scales_with_eta(oracle):
    pos, vel, m = plummer(256, seed=1)
    errs = {}
    for eta in (0.1, 0.2, 0.45):
        it = oracle.Integrator(pos, vel, m, eps=1e-3, eta=eta, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
        e0 = it.energy()[0]
        it.run_until(1.0)
        assert np.all(it.t == 1.0)
        errs[eta] = abs((it.energy()[0] - e0) / e0)
    assert errs[0.1] < errs[0.2] < errs[0.45]
    slope = math.log(errs[0.45] / errs[0.1]) / math.log(4.5)
    assert 3.0 < slope < 7.5, (errs, slope)
    # plausibility band from the values the paper prints (tests/golden/paper_fig1_energy_errors.txt,
    # PAPER.md:141): below 5e-9 at eta = 0.6 for N >= 2^15 in mixed precision; a 256-body FP64 run at the
    # smaller eta = 0.45 must not be two orders of magnitude worse than that, nor below the paper's floor
    band = _paper_fig1_band()
    assert band[(0.3, "dE_over_E")] < errs[0.45] < 100 * band[(0.6, "dE_over_E")]


# ---------------------------------------------------------------- energy (Eq. 2, Eq. 20)
def test_energy_closed_forms(oracle):
    # two bodies: E = 1/2 m1 v1^2 + 1/2 m2 v2^2 - m1 m2/sqrt(d^2 + eps^2)
    pos = np.array([[0.0, 0, 0], [3.0, 4.0, 0]]); vel = np.array([[1.0, 0, 0], [0, -2.0, 0]])
    m = np.array([2.0, 3.0])
    out = oracle.energy(pos, vel, m, 12.0)
    assert out[1] == pytest.approx(0.5 * 2 * 1 + 0.5 * 3 * 4)
    assert out[2] == pytest.approx(-6.0 / 13.0)
    assert out[0] == pytest.approx(out[1] + out[2])
    np.testing.assert_allclose(out[3:6], [2.0, -6.0, 0.0])
    np.testing.assert_allclose(out[6:9], [0, 0, 3.0 * (3.0 * -2.0 - 0.0)])
    # ring of n masses: W = -(n m^2 / (4 R)) sum_k 1/sin(pi k/n), L_z = n m R^2 w
    n, mm, R, w = 9, 0.2, 1.3, 0.7
    ph = 2 * np.pi * np.arange(n) / n
    pos = R * np.stack([np.cos(ph), np.sin(ph), 0 * ph], 1)
    vel = w * R * np.stack([-np.sin(ph), np.cos(ph), 0 * ph], 1)
    out = oracle.energy(pos, vel, np.full(n, mm), 0.0)
    assert out[2] == pytest.approx(-(n * mm * mm / (4 * R)) * sum(1 / math.sin(math.pi * k / n) for k in range(1, n)), rel=1e-13)
    assert out[8] == pytest.approx(n * mm * R * R * w, rel=1e-13)
    assert out[1] == pytest.approx(0.5 * n * mm * (w * R) ** 2, rel=1e-13)


def test_startup_two_pass(oracle):
    # Start-up (G8): after the two passes, stored a, jerk, snap equal one evaluation with a_pred = a.
    pos, vel, m = plummer(48, seed=6)
    it = oracle.Integrator(pos, vel, m, eps=1e-2, eta=0.45)
    a, j, s = oracle.force(pos, vel, it.acc, m, 1e-2)
    assert np.array_equal(a, it.acc) and np.array_equal(j, it.jerk) and np.array_equal(s, it.snap)
    assert np.all(it.crackle == 0) and np.all(it.t == 0)
    mant, _ = np.frexp(it.dt)
    assert np.all(mant == 0.5)
