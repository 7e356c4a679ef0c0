"""GPU parity of the evaluation step (a3, a4): nb_force through the C-ABI against the oracle's
plain long-double direct summation (oracle/nb_oracle.c: orc_force), same seeded inputs.
Tolerance: 1e-12 per component relative to the particle's vector norm (north_star; G17)."""
import numpy as np
import pytest
import torch

from parity import FORCE_TOL, dev, g17_err, gpu_force, host
from workloads import active_subset, config_inputs, kepler_binary, mean_field_acc, plummer, power_law_masses

pytestmark = pytest.mark.gpu


def _check(nb, oracle, pos, vel, accp, mass, eps, idx=None, tol=FORCE_TOL, **tune):
    (a, j, s), launch = gpu_force(nb, pos, vel, accp, mass, eps, idx, **tune)
    ra, rj, rs = oracle.force(pos, vel, accp if accp is not None else np.zeros_like(pos), mass, eps, idx)
    assert np.all(np.isfinite(a)) and np.all(np.isfinite(j)) and np.all(np.isfinite(s))
    errs = (g17_err(a, ra), g17_err(j, rj), g17_err(s, rs))
    assert max(errs) <= tol, (errs, launch)
    return errs, launch


@pytest.mark.parametrize("n,eps,seed", [(2, 0.0, 0), (3, 0.0, 1), (5, 1e-2, 2), (37, 1e-3, 3), (64, 1e-4, 4), (64, 0.0, 5)])
def test_brute_force_small(nb, oracle, n, eps, seed):
    rng = np.random.default_rng(seed)
    pos = rng.normal(size=(n, 3)); vel = rng.normal(size=(n, 3)); accp = rng.normal(size=(n, 3))
    mass = rng.uniform(0.1, 1.0, size=n)
    _check(nb, oracle, pos, vel, accp, mass, eps)


@pytest.mark.parametrize("N", [127, 128, 129, 1000, 4096 + 37])
def test_all_active_ragged(nb, oracle, N):
    pos, vel, m = plummer(N, seed=100 + N)
    _check(nb, oracle, pos, vel, mean_field_acc(pos), m, 1e-3)


def test_config3_smallest_point_all_active(nb, oracle):
    # BASELINE.json config 3, N = 2^14: every particle, element by element
    pos, vel, m, accp = config_inputs(3, 1 << 14)
    errs, launch = _check(nb, oracle, pos, vel, accp, m, 1e-3)
    assert launch["threads"] == 128 and launch["jlanes"] == 1


@pytest.mark.parametrize("m_act", [1, 2, 3, 5, 8, 16, 17, 31, 32, 33, 100, 127, 128, 129, 1000])
def test_active_subsets(nb, oracle, m_act):
    # spans every lane-sharing factor (JL = 8, 4, 2, 1), the one-warp variant and the 128-thread one
    N = 4096 + 37
    pos, vel, mass, accp = config_inputs(4, N)        # power-law masses (config 4 recipe)
    idx = active_subset(N, m_act, seed=40)
    _check(nb, oracle, pos, vel, accp, mass, 1e-4, idx)


def test_duplicate_and_unsorted_indices(nb, oracle):
    pos, vel, m = plummer(300, seed=9)
    idx = np.array([299, 0, 17, 17, 5, 299], dtype=np.int32)
    _check(nb, oracle, pos, vel, None, m, 1e-2, idx)


@pytest.mark.parametrize("split,jlanes", [(1, 0), (2, 0), (7, 0), (64, 0), (0, 1), (0, 2), (0, 8), (0, 32), (3, 16)])
def test_forced_split_and_lane_sharing(nb, oracle, split, jlanes):
    # every decomposition of the same sum is correct within the tolerance (G18)
    N = 2048 + 5
    pos, vel, m = plummer(N, seed=21)
    idx = active_subset(N, 9 if jlanes else 300, seed=3)
    errs, launch = _check(nb, oracle, pos, vel, mean_field_acc(pos), m, 1e-3, idx, split=split, jlanes=jlanes)
    if split:
        assert 1 <= launch["splits"] <= split and (split > 1) == (launch["splits"] > 1)
    if jlanes:
        assert launch["jlanes"] == jlanes


def test_results_do_not_depend_on_decomposition_beyond_rounding(nb):
    N = 3000
    pos, vel, m = plummer(N, seed=22)
    accp = mean_field_acc(pos)
    (a1, j1, s1), _ = gpu_force(nb, pos, vel, accp, m, 1e-3, split=1)
    (a2, j2, s2), _ = gpu_force(nb, pos, vel, accp, m, 1e-3, split=5)
    assert g17_err(a2, a1) < 1e-14 and g17_err(j2, j1) < 1e-14 and g17_err(s2, s1) < 1e-14
    (a3, j3, s3), _ = gpu_force(nb, pos, vel, accp, m, 1e-3, split=5)
    assert np.array_equal(a2, a3) and np.array_equal(j2, j3) and np.array_equal(s2, s3)  # bit-reproducible


def test_two_body_eps0_and_self_term(nb, oracle):
    # eps = 0: the self term (s = 0) contributes nothing (G12); closed form m r / |r|^3
    pos, vel, m = kepler_binary(0.5)
    (a, j, s), _ = gpu_force(nb, pos, vel, None, m, 0.0)
    d = pos[1] - pos[0]
    np.testing.assert_allclose(a[0], m[1] * d / np.linalg.norm(d) ** 3, rtol=1e-15)
    _check(nb, oracle, pos, vel, None, m, 0.0)


def test_single_particle_and_empty_set(nb):
    z = np.zeros((1, 3))
    (a, j, s), _ = gpu_force(nb, z + 1.0, z + 2.0, z + 3.0, np.array([5.0]), 0.0)
    assert np.all(a == 0) and np.all(j == 0) and np.all(s == 0)
    (a, j, s), _ = gpu_force(nb, z + 1.0, z + 2.0, z + 3.0, np.array([5.0]), 0.1)
    assert np.all(a == 0) and np.all(j == 0) and np.all(s == 0)
    pos, vel, m = plummer(64, seed=1)
    ctx = nb.nb_init(dev(pos), dev(vel), dev(m), 1e-3, 0.45)
    try:
        nb.nb_force(ctx, dev(np.zeros(0, dtype=np.int32), torch.int32), 0, None, None, None)  # no-op
    finally:
        nb.nb_free(ctx)


def test_host_pointers_give_the_same_result(nb):
    # [dev|host] arguments: numpy (pageable) and pinned tensors work like device tensors
    pos, vel, m = plummer(500, seed=5)
    accp = mean_field_acc(pos)
    (a_d, j_d, s_d), _ = gpu_force(nb, pos, vel, accp, m, 1e-3)
    ctx = nb.nb_init(pos, vel, m, 1e-3, 0.45)
    try:
        nb.nb_set_pred_acc(ctx, accp)
        idx = np.arange(500, dtype=np.int32)
        out = [torch.empty((500, 3), dtype=torch.float64).pin_memory() for _ in range(3)]
        nb.nb_force(ctx, idx, 500, *out)
        torch.cuda.synchronize()
    finally:
        nb.nb_free(ctx)
    assert np.array_equal(out[0].numpy(), a_d) and np.array_equal(out[1].numpy(), j_d) and np.array_equal(out[2].numpy(), s_d)


def test_error_codes(nb):
    pos, vel, m = plummer(64, seed=1)
    E = nb.NBError
    with pytest.raises(E) as e:
        nb.nb_init(dev(pos), dev(vel), dev(m), -1.0, 0.45)
    assert e.value.code == -1
    with pytest.raises(E):
        nb.nb_init(dev(pos), dev(vel), dev(m), 1e-3, 0.0)
    ctx = nb.nb_init(dev(pos), dev(vel), dev(m), 1e-3, 0.45)
    try:
        with pytest.raises(E) as e:
            nb.nb_force(ctx, None, 65, None, None, None)
        assert e.value.code == -1
        with pytest.raises(E) as e:
            nb.nb_force(ctx, None, 5, None, None, None)      # NULL list but no scheduler block
        assert e.value.code == -2
        with pytest.raises(E) as e:
            nb.nb_next_block(ctx)                             # before nb_startup
        assert e.value.code == -2
        with pytest.raises(E) as e:
            nb.nb_correct_and_step(ctx)
        assert e.value.code == -2
        with pytest.raises(E):
            nb.nb_set_limits(ctx, 0.3, 0.5)                   # not powers of two
        nb.nb_startup(ctx)
        with pytest.raises(E) as e:
            nb.nb_set_limits(ctx, 2.0 ** -20, 2.0 ** -4)      # after start-up
        assert e.value.code == -2
        assert "nb_set_limits" in nb.nb_last_error(ctx)
        with pytest.raises(E) as e:
            nb.nb_predict(ctx, -1.0)
        assert e.value.code == -1
    finally:
        nb.nb_free(ctx)


# ---------------------------------------------------------------- BASELINE.json full sizes, sampled
def _sample_rows(N, mass, pos, k=256, seed=7):
    rng = np.random.default_rng(seed)
    r = np.linalg.norm(pos, axis=1)
    special = [int(np.argmin(r)), int(np.argmax(r)), int(np.argmax(mass)), int(np.argmin(mass))]
    rest = rng.choice(N, size=k - len(special), replace=False)
    return np.unique(np.concatenate([special, rest])).astype(np.int32)


def test_config3_full_size_2p20_sampled(nb, oracle):
    # the launch configuration bench.py times: N = 2^20, all particles active, one evaluation;
    # 256 sampled rows (innermost, outermost, ...) against all N j in the oracle
    N = 1 << 20
    pos, vel, m, accp = config_inputs(3, N)
    (a, j, s), launch = gpu_force(nb, pos, vel, accp, m, 1e-3)
    # one i per lane; enough j-splits (4 or 5, depending on the resident CTAs per SM) that the piece the running
    # CTAs stream (<= 24 MB) stays L2-resident across the 8192 i-blocks
    assert launch["threads"] == 128 and launch["jlanes"] == 1
    assert 4 <= launch["splits"] <= 8 and launch["ctas"] == launch["splits"] * 8192
    rows = _sample_rows(N, m, pos)
    ra, rj, rs = oracle.force(pos, vel, accp, m, 1e-3, rows)
    errs = (g17_err(a[rows], ra), g17_err(j[rows], rj), g17_err(s[rows], rs))
    assert max(errs) <= FORCE_TOL, errs
    # property that holds at any size: pairwise antisymmetry => sum m a = sum m jerk = sum m snap = 0
    for x in (a, j, s):
        tot = np.abs((m[:, None] * x).sum(0)); ref = (m[:, None] * np.abs(x)).sum()
        assert np.all(tot <= 1e-13 * ref), (tot, ref)


@pytest.mark.parametrize("m_act", [64, 1024, 16384])
def test_config4_full_size_subsets(nb, oracle, m_act):
    # BASELINE.json config 4: N = 2^20, power-law masses, eps = 1e-4, random active subsets
    N = 1 << 20
    pos, vel, mass, accp = config_inputs(4)
    idx = active_subset(N, m_act, seed=40)
    (a, j, s), launch = gpu_force(nb, pos, vel, accp, mass, 1e-4, idx)
    sel = np.arange(m_act) if m_act <= 256 else np.random.default_rng(1).choice(m_act, 256, replace=False)
    ra, rj, rs = oracle.force(pos, vel, accp, mass, 1e-4, idx[sel])
    errs = (g17_err(a[sel], ra), g17_err(j[sel], rj), g17_err(s[sel], rs))
    assert max(errs) <= FORCE_TOL, (errs, launch)
    assert launch["ctas"] >= 148


@pytest.mark.parametrize("cfg,N,eps", [(3, 1 << 22, 1e-3), (5, 1 << 23, 1e-4)])
def test_largest_sizes_sampled_rows(nb, oracle, cfg, N, eps):
    # the largest N of BASELINE.json: top of the config 3 sweep (2^22) and config 5 (2^23, 8.4M particles).
    # 256 sampled active rows (innermost, outermost, ...) against ALL N predicted particles: the evaluation
    # runs split-j with thousands of CTAs over the whole 336 / 671 MB stream; the oracle needs ~10 s.
    if cfg == 3:
        pos, vel, m, accp = config_inputs(3, N)
    else:
        pos, vel, m, _ = config_inputs(5, N)
        from workloads import mean_field_acc
        accp = mean_field_acc(pos)
    rows = _sample_rows(N, m, pos)
    (a, j, s), launch = gpu_force(nb, pos, vel, accp, m, eps, rows)
    assert launch["splits"] > 1 and launch["ctas"] >= 148
    ra, rj, rs = oracle.force(pos, vel, accp, m, eps, rows)
    errs = (g17_err(a, ra), g17_err(j, rj), g17_err(s, rs))
    assert max(errs) <= FORCE_TOL, (errs, launch)
