"""Pins of the oracle's evaluation step (oracle/nb_oracle.c: orc_force), Eq. 8-10 of
PAPER.md:72-81 with the Eq. 2 softening.  None of these retypes Eq. 9-10: jerk and snap
are pinned by DIFFERENTIATING Eq. 8 along a prescribed motion (mpmath, 40 digits), by the
rigidly rotating ring (closed form) and by the pairwise antisymmetry invariants."""
import math

import mpmath as mp
import numpy as np
import pytest

from workloads import plummer

mp.mp.dps = 40


def _acc_of_t(t, k, R, V, A, J, M, eps):
    """Eq. 8 (softened, Eq. 2) for particle k when every particle moves on the prescribed
    polynomial path r(t) = R + V t + A t^2/2 + J t^3/6  (mpmath)."""
    n = len(M)
    pos = [[R[i][d] + V[i][d] * t + A[i][d] * t * t / 2 + J[i][d] * t ** 3 / 6 for d in range(3)]
           for i in range(n)]
    out = [mp.mpf(0)] * 3
    for j in range(n):
        if j == k:
            continue
        d = [pos[j][c] - pos[k][c] for c in range(3)]
        s = d[0] ** 2 + d[1] ** 2 + d[2] ** 2 + eps ** 2
        w = M[j] / (s * mp.sqrt(s))
        out = [out[c] + w * d[c] for c in range(3)]
    return out


@pytest.mark.parametrize("n,eps,seed", [(2, 0.0, 0), (2, 0.05, 1), (5, 0.01, 2), (8, 1e-3, 3)])
def test_jerk_snap_are_time_derivatives_of_eq8(oracle, n, eps, seed):
    rng = np.random.default_rng(seed)
    R = rng.normal(size=(n, 3)); V = rng.normal(size=(n, 3)); A = rng.normal(size=(n, 3))
    J = rng.normal(size=(n, 3))  # third derivative of the path: must NOT enter a, jerk, snap
    M = rng.uniform(0.1, 1.0, size=n)
    acc, jerk, snap = oracle.force(R, V, A, M, eps)
    Rm = [[mp.mpf(float(x)) for x in row] for row in R]
    Vm = [[mp.mpf(float(x)) for x in row] for row in V]
    Am = [[mp.mpf(float(x)) for x in row] for row in A]
    Jm = [[mp.mpf(float(x)) for x in row] for row in J]
    Mm = [mp.mpf(float(x)) for x in M]
    e = mp.mpf(eps)
    for k in range(n):
        for c in range(3):
            f = lambda t, c=c: _acc_of_t(t, k, Rm, Vm, Am, Jm, Mm, e)[c]
            a0 = f(mp.mpf(0)); a1 = mp.diff(f, 0, 1); a2 = mp.diff(f, 0, 2)
            scale_a = max(abs(float(x)) for x in acc[k]); scale_j = max(abs(float(x)) for x in jerk[k])
            scale_s = max(abs(float(x)) for x in snap[k])
            assert abs(acc[k, c] - float(a0)) <= 4e-16 * scale_a
            assert abs(jerk[k, c] - float(a1)) <= 4e-16 * scale_j
            assert abs(snap[k, c] - float(a2)) <= 4e-16 * scale_s


def test_two_body_closed_form(oracle):
    # a_1 = m_2 (r_2 - r_1) / (|r|^2 + eps^2)^(3/2): sign (attractive) and softening exponent.
    R = np.array([[0.0, 0.0, 0.0], [3.0, 4.0, 0.0]]); Z = np.zeros((2, 3)); M = np.array([2.0, 7.0])
    acc, jerk, snap = oracle.force(R, Z, Z, M, 0.0)
    np.testing.assert_allclose(acc[0], 7.0 * np.array([3.0, 4.0, 0.0]) / 125.0, rtol=1e-15)
    np.testing.assert_allclose(acc[1], -2.0 * np.array([3.0, 4.0, 0.0]) / 125.0, rtol=1e-15)
    assert np.all(jerk == 0) and np.all(snap == 0)
    eps = 12.0  # 3-4-5 and 5-12-13: s = 169, s^(3/2) = 2197
    acc, _, _ = oracle.force(R, Z, Z, M, eps)
    np.testing.assert_allclose(acc[0], 7.0 * np.array([3.0, 4.0, 0.0]) / 2197.0, rtol=1e-15)


@pytest.mark.parametrize("n", [3, 7, 16])
def test_rotating_ring_closed_form(oracle, n):
    # n equal masses m on a ring of radius Rr rotating rigidly with angular speed w (eps = 0):
    # |a| = m/(4 Rr^2) sum_k 1/sin(pi k/n) towards the centre; since the configuration only
    # rotates, a(t) = Rot(w t) a(0) => jerk = w z^ x a, snap = -w^2 a.
    m, Rr, w = 0.3, 1.7, 0.9
    ph = 2 * np.pi * np.arange(n) / n + 0.123
    R = Rr * np.stack([np.cos(ph), np.sin(ph), np.zeros(n)], 1)
    V = w * Rr * np.stack([-np.sin(ph), np.cos(ph), np.zeros(n)], 1)
    A = -w * w * R
    acc, jerk, snap = oracle.force(R, V, A, np.full(n, m), 0.0)
    amag = m / (4 * Rr * Rr) * sum(1.0 / math.sin(math.pi * k / n) for k in range(1, n))
    np.testing.assert_allclose(acc, -amag * R / Rr, rtol=0, atol=2e-14 * amag)  # inputs carry cos/sin rounding
    zxa = w * np.stack([-acc[:, 1], acc[:, 0], np.zeros(n)], 1)
    np.testing.assert_allclose(jerk, zxa, rtol=0, atol=1e-13 * amag * w)
    np.testing.assert_allclose(snap, -w * w * acc, rtol=0, atol=1e-12 * amag * w * w)


def test_pairwise_antisymmetry_invariants(oracle):
    # sum m a = sum m jerk = sum m snap = 0; torque and its first derivative vanish.
    pos, vel, m = plummer(96, seed=11)
    rng = np.random.default_rng(5)
    ap = rng.normal(size=pos.shape)
    acc, jerk, snap = oracle.force(pos, vel, ap, m, 1e-3)
    for x in (acc, jerk, snap):
        tot = (m[:, None] * x).sum(0)
        ref = (m[:, None] * np.abs(x)).sum()
        assert np.all(np.abs(tot) <= 1e-15 * ref)
    tq = (m[:, None] * np.cross(pos, acc)).sum(0)
    assert np.all(np.abs(tq) <= 1e-15 * (m[:, None] * np.abs(np.cross(pos, acc))).sum())
    dtq = (m[:, None] * (np.cross(pos, jerk) + np.cross(vel, acc))).sum(0)
    ref = (m[:, None] * (np.abs(np.cross(pos, jerk)) + np.abs(np.cross(vel, acc)))).sum()
    assert np.all(np.abs(dtq) <= 1e-15 * ref)


def test_subset_rows_equal_full_rows(oracle):
    pos, vel, m = plummer(64, seed=12)
    ap = np.zeros_like(pos)
    full = oracle.force(pos, vel, ap, m, 1e-2)
    idx = np.array([63, 0, 17, 17, 5], dtype=np.int32)
    sub = oracle.force(pos, vel, ap, m, 1e-2, idx)
    for f, s in zip(full, sub):
        assert np.array_equal(f[idx], s)


def test_self_term_is_skipped_and_N1_is_zero(oracle):
    z = np.zeros((1, 3))
    acc, jerk, snap = oracle.force(z + 1.0, z + 2.0, z + 3.0, np.array([5.0]), 0.0)
    assert np.all(acc == 0) and np.all(jerk == 0) and np.all(snap == 0)


# ---- the mixed-precision restatement (orc_force_mixed, reading G27) -----------
def test_mixed_oracle_is_the_fp64_result_to_single_precision(oracle):
    """Pinned to the (already pinned) FP64 evaluation: the same sums to a few float ulps of
    sum_j |pair term| -- and NOT better than that, i.e. the pair arithmetic really is SP."""
    pos, vel, m = plummer(1500, seed=14)
    rng = np.random.default_rng(6)
    ap = rng.normal(size=pos.shape)
    ref = oracle.force(pos, vel, ap, m, 1e-3)
    a, j, s, scale = oracle.force_mixed(pos, vel, ap, m, 1e-3)
    u = 2.0 ** -24
    for q, (x, y) in enumerate(zip(ref, (a, j, s))):
        err = np.abs(x - y).max(axis=1) / scale[:, q]
        assert err.max() <= 16 * u, (q, err.max())          # forward error of ~10 float operations
        assert np.median(err) >= 1e-3 * u                    # not a double evaluation in disguise
    # scale is what it says: sum_j |pair term|, >= |sum|
    for q, x in enumerate(ref):
        assert np.all(scale[:, q] >= np.linalg.norm(x, axis=1) * (1 - 1e-6))


def test_mixed_oracle_two_body_closed_form(oracle):
    # a = m2 d / (d^2 + eps^2)^(3/2) along x, to float precision; the DP difference keeps a small
    # separation exact even far from the origin (the reason the paper differences in DP)
    for x0 in (0.0, 1.0e4):
        d, eps = 3.0e-3, 1.0e-3
        pos = np.array([[x0, 0.0, 0.0], [x0 + d, 0.0, 0.0]])
        z = np.zeros((2, 3))
        a, j, s, _ = oracle.force_mixed(pos, z, z, np.array([0.25, 0.75]), eps)
        exact = 0.75 * d / (d * d + eps * eps) ** 1.5
        assert abs(a[0, 0] - exact) <= 4 * 2.0 ** -24 * exact
        assert np.all(j == 0) and np.all(s == 0) and a[0, 1] == 0 and a[0, 2] == 0
