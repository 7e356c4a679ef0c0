"""The device-driven block-step loops (CUDA-graph batches, csrc/nb_graph.cu; the cluster-resident
loop, csrc/nb_resident.cu) against the host-driven call sequence nb_next_block -> nb_predict ->
nb_force -> nb_correct_and_step.

Both drivers run the same device functions with the same geometry rule and the same summation
order, so the committed state must be BIT-identical: positions, velocities, derivatives, times,
time steps, step count, pair count and the histogram of active-set sizes.  Parity of the
host-driven sequence against the oracle is in test_gpu_integrator.py; here the graph loop is
also compared with the oracle directly on config 1 (BASELINE.json configs[0], shortened).
"""
import numpy as np
import pytest
import torch

from parity import dev, host
from workloads import kepler_binary, plummer

pytestmark = pytest.mark.gpu


def _mk(nb, pos, vel, m, eps, eta, dt_min, dt_max, graph):
    """graph: False/0 = host-issued calls, True/1 = CUDA-graph batches, 2 = graph batches whose kernels
    are chained by programmatic dependent launch, 3 = one kernel resident on a thread-block cluster."""
    g = nb.NBody(dev(pos), dev(vel), dev(m), eps, eta, dt_min=dt_min, dt_max=dt_max)
    nb.nb_set_loop_mode(g.ctx, int(graph))
    return g


def _full(nb, g, n):
    st = torch.empty((n, 21), dtype=torch.float64, device="cuda")
    nb.nb_get_full_state(g.ctx, st)
    g.sync()
    return host(st)


@pytest.mark.parametrize("mode", [1, 2, 3])
@pytest.mark.parametrize("n,seed,eps,t_end", [(1024, 1, 1e-3, 0.25), (3000, 8, 1e-3, 0.0625), (77, 5, 1e-2, 0.5)])
def test_graph_loop_is_bit_identical_to_call_sequence(nb, n, seed, eps, t_end, mode):
    pos, vel, m = plummer(n, seed=seed)
    a = _mk(nb, pos, vel, m, eps, 0.45, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, eps, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    na = a.run_until(t_end)
    nb_ = b.run_until(t_end)
    assert na == nb_ and na > 10
    sa, sb = _full(nb, a, n), _full(nb, b, n)
    assert np.array_equal(sa, sb)                       # every one of the 21 doubles per particle
    ta, tb = a.stats(), b.stats()
    assert ta["n_steps"] == tb["n_steps"] and ta["n_pairs"] == tb["n_pairs"] and ta["t_now"] == tb["t_now"]
    assert list(ta["hist"]) == list(tb["hist"])
    # continue a second leg: the graph is replayed, not rebuilt, and the drivers still agree
    a.run_until(2 * t_end); b.run_until(2 * t_end)
    assert np.array_equal(_full(nb, a, n), _full(nb, b, n))
    assert np.array_equal(a.energy(), b.energy())
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3])
def test_graph_run_steps_counts_exactly(nb, mode):
    pos, vel, m = plummer(700, seed=21)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    for k in (1, 7, 64, 65, 130):                        # below, at and above the batch length
        a.run_steps(k, log=False)
        b.run_steps(k, log=False)
        assert a.stats()["n_steps"] == b.stats()["n_steps"]
        assert np.array_equal(_full(nb, a, 700), _full(nb, b, 700))
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3])
def test_graph_loop_then_single_calls(nb, mode):
    """Mixing drivers: a device-driven leg, then explicit calls, then a device-driven leg again."""
    pos, vel, m = plummer(500, seed=22)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    a.run_until(0.0625); b.run_until(0.0625)
    for g in (a, b):
        for _ in range(5):
            tn, n = g.next_block()
            g.predict(tn); nb.nb_force(g.ctx, None, n); g.correct_and_step()
    a.run_until(0.125); b.run_until(0.125)
    assert np.array_equal(_full(nb, a, 500), _full(nb, b, 500))
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3])
def test_graph_loop_all_active_and_eps0(nb, mode):
    # shared step: every block has m = N (index-order evaluation, variant A at N >= 128)
    pos, vel, m = plummer(512, seed=3)
    a = _mk(nb, pos, vel, m, 1e-2, 0.45, 2.0 ** -7, 2.0 ** -7, graph=mode)
    b = _mk(nb, pos, vel, m, 1e-2, 0.45, 2.0 ** -7, 2.0 ** -7, graph=False)
    assert a.run_until(0.125) == 16 and b.run_until(0.125) == 16
    assert np.array_equal(_full(nb, a, 512), _full(nb, b, 512))
    a.close(); b.close()
    # eps = 0 (GUARD0 kernels): Kepler binary, two particles
    pos, vel, m = kepler_binary(0.5)
    a = _mk(nb, pos, vel, m, 0.0, 0.1, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, 0.0, 0.1, 2.0 ** -25, 2.0 ** -4, graph=False)
    a.run_until(1.0); b.run_until(1.0)
    assert np.array_equal(_full(nb, a, 2), _full(nb, b, 2))
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3])
def test_graph_loop_respects_tuning_knobs(nb, mode):
    """nb_set_tuning changes kernel arguments of the captured nodes: the graph is re-captured."""
    pos, vel, m = plummer(600, seed=23)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    a.run_until(0.03125); b.run_until(0.03125)
    nb.nb_set_tuning(a.ctx, 1, 1); nb.nb_set_tuning(b.ctx, 1, 1)      # split-j off (Fig. 8 "Bfactor off")
    a.run_until(0.0625); b.run_until(0.0625)
    assert np.array_equal(_full(nb, a, 600), _full(nb, b, 600))
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3])
def test_graph_loop_matches_oracle_config1_quarter(nb, oracle, mode):
    pos, vel, m = plummer(1024, seed=1)
    g = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=mode)
    n = g.run_until(0.25)
    it = oracle.Integrator(pos, vel, m, eps=1e-3, eta=0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    k = it.run_until(0.25)[0]
    assert n == k
    r, v, t, dt = [host(x) for x in g.state()]
    assert np.array_equal(t, it.t) and np.array_equal(dt, it.dt)          # identical decisions
    err = (np.linalg.norm(r - it.pos, axis=1) / np.linalg.norm(it.pos, axis=1)).max()
    assert err < 1e-9
    g.close()


def test_graph_loop_large_ragged_n(nb):
    """N = 150 001 (not a multiple of any tile), batch of 64 steps replayed over many scheduler blocks; the
    first steps have m from a handful to tens of thousands: both evaluation variants, S > 1 and S = 1."""
    n = 150001
    pos, vel, m = plummer(n, seed=24)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=True)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    a.run_steps(12, log=False)
    b.run_steps(12, log=False)
    sa, sb = a.stats(), b.stats()
    assert sa["n_steps"] == sb["n_steps"] == 12 and sa["n_pairs"] == sb["n_pairs"] and sa["t_now"] == sb["t_now"]
    assert list(sa["hist"]) == list(sb["hist"]) and sa["hist"][4:].sum() > 0      # some large blocks among them
    assert np.array_equal(_full(nb, a, n), _full(nb, b, n))
    a.close(); b.close()


def test_resident_loop_limits_and_default(nb):
    """Mode 3 serves N <= 16384 and is the default driver for N <= 2048; above its limit it refuses loudly."""
    pos, vel, m = plummer(20000, seed=25)
    g = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    with pytest.raises(nb.NBError) as e:
        nb.nb_set_loop_mode(g.ctx, 3)
    assert e.value.code == nb.nb.NB_EINVAL
    g.close()
    # N = 6000 (several all-active variant-A steps on the cluster, multi-wave i-blocks): mode 3 == mode 0
    n = 6000
    pos, vel, m = plummer(n, seed=26)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=3)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    assert a.run_until(0.0625) == b.run_until(0.0625)
    assert np.array_equal(_full(nb, a, n), _full(nb, b, n))
    sa, sb = a.stats(), b.stats()
    assert sa["n_pairs"] == sb["n_pairs"] and list(sa["hist"]) == list(sb["hist"])
    a.close(); b.close()


def test_resident_loop_mixed_precision(nb):
    pos, vel, m = plummer(900, seed=27)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=3)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    nb.nb_set_precision(a.ctx, 1); nb.nb_set_precision(b.ctx, 1)
    assert a.run_until(0.0625) == b.run_until(0.0625)
    assert np.array_equal(_full(nb, a, 900), _full(nb, b, 900))
    a.close(); b.close()
