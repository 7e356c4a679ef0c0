"""The evaluation step in the paper's mixed precision (nb_set_precision(ctx, 1 | 2); PAPER.md:287, 301,
DESIGN.md readings G27 and G27b) against the oracle's mixed restatement (oracle/nb_oracle.c:
orc_force_mixed: float pair terms, summed exactly) and against the FP64 oracle.
Mode 2 (G27b) adds the acceleration and jerk terms in double, so for those two the float tile sum drops
out of the bound: <= 32 u x sum|term|.

Tolerance (derived in DESIGN.md section 6.5): both sides round the nine differences to float and do
~10 float operations per pair term (different order, rsqrt instead of sqrt and divide, FMA on the
GPU): <= ~32 u of the term each, u = 2^-24.  The GPU also sums up to 128 pair terms of a j-tile in
float: <= 128 u of sum|term| in the worst case.  Bound used: |x_gpu - x_ref|_inf <= 256 u x
sum_j |pair term|_2 = 1.5e-5 x scale.
"""
import numpy as np
import pytest
import torch

from parity import dev, host
from workloads import active_subset, config_inputs, kepler_binary, plummer

pytestmark = pytest.mark.gpu

U = 2.0 ** -24
MIXED_TOL = 256 * U


def _gpu_force_mixed(nb, pos, vel, accp, m, eps, idx=None, mode=1):
    g = nb.NBody(dev(pos), dev(vel), dev(m), eps, 0.45)
    nb.nb_set_pred_acc(g.ctx, dev(accp))
    nb.nb_set_precision(g.ctx, mode)
    if idx is None:
        out = g.force()
    else:
        out = g.force(dev(idx, torch.int32))
    res = [host(x) for x in out]
    launch = nb.nb_get_launch(g.ctx)
    g.close()
    return res, launch


def _errs(x, ref, scale):
    return [float((np.abs(a - b).max(axis=1) / scale[:, q]).max()) for q, (a, b) in enumerate(zip(x, ref))]


@pytest.mark.parametrize("mode", [1, 2])
@pytest.mark.parametrize("n,eps", [(1000, 1e-3), (4500, 1e-4), (33, 1e-2)])
def test_mixed_force_all_active_matches_mixed_oracle(nb, oracle, n, eps, mode):
    pos, vel, m = plummer(n, seed=31)
    rng = np.random.default_rng(32)
    accp = rng.normal(size=pos.shape)
    (a, j, s), _ = _gpu_force_mixed(nb, pos, vel, accp, m, eps, mode=mode)
    ra, rj, rs, scale = oracle.force_mixed(pos, vel, accp, m, eps)
    e = _errs((a, j, s), (ra, rj, rs), scale)
    assert max(e) <= MIXED_TOL, e
    if mode == 2:
        assert max(e[:2]) <= 32 * U, e               # a, jerk: summed in double (G27b)
    # and it is close to the FP64 definition to single precision, not to double precision
    fa, fj, fs = oracle.force(pos, vel, accp, m, eps)
    e64 = _errs((a, j, s), (fa, fj, fs), scale)
    assert max(e64) <= MIXED_TOL and min(e64) > 1e-12, e64


@pytest.mark.parametrize("mode", [1, 2])
@pytest.mark.parametrize("m_act", [3, 64, 700])
def test_mixed_force_subsets_split_j(nb, oracle, m_act, mode):
    # small active sets: several lanes share one i, many j-splits
    n = 20000
    pos, vel, m, accp = config_inputs(4, n)
    idx = active_subset(n, m_act, 40)
    (a, j, s), launch = _gpu_force_mixed(nb, pos, vel, accp, m, 1e-4, idx, mode=mode)
    assert launch["splits"] > 1
    ra, rj, rs, scale = oracle.force_mixed(pos, vel, accp, m, 1e-4, idx)
    e = _errs((a, j, s), (ra, rj, rs), scale)
    assert max(e) <= MIXED_TOL, e
    if mode == 2:
        assert max(e[:2]) <= 32 * U, e


def test_mixed_eps0_self_term(nb, oracle):
    pos, vel, m = kepler_binary(0.3)
    z = np.zeros_like(pos)
    (a, j, s), _ = _gpu_force_mixed(nb, pos, vel, z, m, 0.0)
    ra, rj, rs, scale = oracle.force_mixed(pos, vel, z, m, 0.0)
    assert np.isfinite(a).all() and np.isfinite(j).all() and np.isfinite(s).all()
    for x, r, q in ((a, ra, 0), (j, rj, 1)):
        assert float((np.abs(x - r).max(axis=1) / scale[:, q]).max()) <= MIXED_TOL


def test_mixed_integration_energy_and_loop_identity(nb):
    """Config 1 shape, shortened: the mixed evaluation inside the FP64 Hermite loop.  Energy is
    conserved to single-precision force accuracy, and the device-driven loop equals the call
    sequence bit for bit in this mode too."""
    pos, vel, m = plummer(1024, seed=1)
    sts = []
    for graph, mode in ((1, 1), (0, 1), (1, 2), (0, 2)):
        g = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
        nb.nb_set_precision(g.ctx, mode)
        nb.nb_set_loop_mode(g.ctx, graph)
        g.startup()
        e0 = g.energy()
        g.run_until(0.25)
        e1 = g.energy()
        assert abs((e1[0] - e0[0]) / e0[0]) < 2e-7
        st = torch.empty((1024, 21), dtype=torch.float64, device="cuda")
        nb.nb_get_full_state(g.ctx, st); g.sync()
        sts.append(host(st))
        g.close()
    assert np.array_equal(sts[0], sts[1]) and np.array_equal(sts[2], sts[3])
