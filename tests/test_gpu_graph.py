"""The device-driven block-step loops (CUDA-graph batches, csrc/nb_graph.cu; the cluster-resident
loop, csrc/nb_resident.cu; the grid-resident loop, csrc/nb_gridres.cu) against the host-driven call sequence nb_next_block -> nb_predict ->
nb_force -> nb_correct_and_step.

The graph-driven loop (modes 1, 2) runs the same device functions with the same geometry rule and the
same summation order as the call sequence, so the committed state must be BIT-identical: positions,
velocities, derivatives, times, time steps, step count, pair count and the histogram of active-set
sizes.  The cluster-resident loop (mode 3) and the grid-resident loop (mode 4: all SMs, two grid barriers per
step, large steps handed to the call sequence) add the pair terms of a particle in their own fixed order
(G18: any order is correct), so it must reproduce times, time steps, step and pair counts
exactly and everything else to rounding (1e-12 of the particle's own magnitude), and be bit-reproducible
from run to run.  Parity of the
host-driven sequence against the oracle is in test_gpu_integrator.py; here the graph loop is
also compared with the oracle directly on config 1 (BASELINE.json configs[0], shortened).
"""
import numpy as np
import pytest
import torch

from parity import dev, host
from workloads import kepler_binary, plummer

pytestmark = pytest.mark.gpu


OWN_ORDER = (3, 4)   # loop modes with their own summation order


def _mk(nb, pos, vel, m, eps, eta, dt_min, dt_max, graph):
    """graph: False/0 = host-issued calls, True/1 = CUDA-graph batches, 2 = graph batches whose kernels
    are chained by programmatic dependent launch, 3 = one kernel resident on a thread-block cluster, 4 = one
    cooperative kernel resident on all SMs."""
    g = nb.NBody(dev(pos), dev(vel), dev(m), eps, eta, dt_min=dt_min, dt_max=dt_max)
    nb.nb_set_loop_mode(g.ctx, int(graph))
    return g


def _full(nb, g, n):
    st = torch.empty((n, 21), dtype=torch.float64, device="cuda")
    nb.nb_get_full_state(g.ctx, st)
    g.sync()
    return host(st)


def _same(sa, sb, mode, tol=1e-12):
    """Full states [n][21] = {m, t, dt, r, v, a, jerk, snap, crackle}: identical for the graph modes; for the
    resident loop m, t, dt identical and every 3-vector within tol of its own norm (crackle, a difference
    quotient of the evaluated values over h^3 that cancels heavily, within 1e-3)."""
    if mode not in OWN_ORDER:
        return bool(np.array_equal(sa, sb))
    if not np.array_equal(sa[:, :3], sb[:, :3]):
        return False
    for q in range(6):
        x, y = sa[:, 3 + 3 * q:6 + 3 * q], sb[:, 3 + 3 * q:6 + 3 * q]
        nrm = np.maximum(np.linalg.norm(y, axis=1, keepdims=True), 1e-300)
        if (np.abs(x - y) / nrm).max() > (1e-3 if q == 5 else tol * (10 ** q if q < 3 else 1e3)):
            return False
    return True


@pytest.mark.parametrize("mode", [1, 2, 3, 4])
@pytest.mark.parametrize("n,seed,eps,t_end", [(1024, 1, 1e-3, 0.25), (3000, 8, 1e-3, 0.0625), (77, 5, 1e-2, 0.5)])
def test_graph_loop_is_bit_identical_to_call_sequence(nb, n, seed, eps, t_end, mode):
    if mode == 3 and n > 2048:
        n = 2000                                        # the resident loop keeps at most 2048 particles on chip
    pos, vel, m = plummer(n, seed=seed)
    a = _mk(nb, pos, vel, m, eps, 0.45, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, eps, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    na = a.run_until(t_end)
    nb_ = b.run_until(t_end)
    assert na == nb_ and na > 10
    sa, sb = _full(nb, a, n), _full(nb, b, n)
    assert _same(sa, sb, mode)                          # modes 1, 2: every one of the 21 doubles per particle
    ta, tb = a.stats(), b.stats()
    assert ta["n_steps"] == tb["n_steps"] and ta["n_pairs"] == tb["n_pairs"] and ta["t_now"] == tb["t_now"]
    assert list(ta["hist"]) == list(tb["hist"])
    # continue a second leg: the graph is replayed, not rebuilt, and the drivers still agree
    a.run_until(2 * t_end); b.run_until(2 * t_end)
    assert _same(_full(nb, a, n), _full(nb, b, n), mode)
    if mode not in OWN_ORDER:
        assert np.array_equal(a.energy(), b.energy())
    else:
        assert abs(a.energy()[0] - b.energy()[0]) <= 1e-13 * abs(b.energy()[0])
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3, 4])
def test_graph_run_steps_counts_exactly(nb, mode):
    pos, vel, m = plummer(700, seed=21)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    for k in (1, 7, 64, 65, 130):                        # below, at and above the batch length
        a.run_steps(k, log=False)
        b.run_steps(k, log=False)
        assert a.stats()["n_steps"] == b.stats()["n_steps"]
        assert _same(_full(nb, a, 700), _full(nb, b, 700), mode)
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3, 4])
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
    assert _same(_full(nb, a, 500), _full(nb, b, 500), mode)
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3, 4])
def test_graph_loop_all_active_and_eps0(nb, mode):
    # shared step: every block has m = N (index-order evaluation, variant A at N >= 128)
    pos, vel, m = plummer(512, seed=3)
    a = _mk(nb, pos, vel, m, 1e-2, 0.45, 2.0 ** -7, 2.0 ** -7, graph=mode)
    b = _mk(nb, pos, vel, m, 1e-2, 0.45, 2.0 ** -7, 2.0 ** -7, graph=False)
    assert a.run_until(0.125) == 16 and b.run_until(0.125) == 16
    assert _same(_full(nb, a, 512), _full(nb, b, 512), mode)
    a.close(); b.close()
    # eps = 0 (GUARD0 kernels): Kepler binary, two particles
    pos, vel, m = kepler_binary(0.5)
    a = _mk(nb, pos, vel, m, 0.0, 0.1, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, 0.0, 0.1, 2.0 ** -25, 2.0 ** -4, graph=False)
    a.run_until(1.0); b.run_until(1.0)
    assert _same(_full(nb, a, 2), _full(nb, b, 2), mode)
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3, 4])
def test_graph_loop_respects_tuning_knobs(nb, mode):
    """nb_set_tuning changes kernel arguments of the captured nodes: the graph is re-captured."""
    pos, vel, m = plummer(600, seed=23)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    a.run_until(0.03125); b.run_until(0.03125)
    nb.nb_set_tuning(a.ctx, 1, 1); nb.nb_set_tuning(b.ctx, 1, 1)      # split-j off (Fig. 8 "Bfactor off")
    a.run_until(0.0625); b.run_until(0.0625)
    assert _same(_full(nb, a, 600), _full(nb, b, 600), mode)
    a.close(); b.close()


@pytest.mark.parametrize("mode", [1, 3, 4])
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
    """Mode 3 serves N <= 2048 and is the default driver up to N = 1024 (mode 4 above, while the system fits the
    shared memory of the device); above its limit it refuses loudly.  Two runs of it give bit-identical states
    (fixed summation order)."""
    pos, vel, m = plummer(3000, seed=25)
    g = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    with pytest.raises(nb.NBError) as e:
        nb.nb_set_loop_mode(g.ctx, 3)
    assert e.value.code == nb.nb.NB_EINVAL
    g.close()
    # N = 2048 (the limit: 128 particles per CTA; all-active steps among them) and a ragged N
    for n in (2048, 1531, 1000):
        pos, vel, m = plummer(n, seed=26)
        a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=3)
        a2 = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=3)
        b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
        d = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)   # default driver
        k = a.run_until(0.125)
        assert k == b.run_until(0.125) == a2.run_until(0.125) == d.run_until(0.125)
        sa = _full(nb, a, n)
        assert _same(sa, _full(nb, b, n), 3)
        assert np.array_equal(sa, _full(nb, a2, n))            # run-to-run bit-reproducible
        assert nb.nb_get_loop_mode(d.ctx) == (3 if n <= 1024 else 4)
        if n <= 1024:
            assert np.array_equal(sa, _full(nb, d, n))         # the default for this N is mode 3
        else:
            assert _same(_full(nb, d, n), _full(nb, b, n), 4)  # ... mode 4
        sa_, sb_ = a.stats(), b.stats()
        assert sa_["n_pairs"] == sb_["n_pairs"] and list(sa_["hist"]) == list(sb_["hist"]) and sa_["t_now"] == sb_["t_now"]
        for g in (a, a2, b, d):
            g.close()


def test_grid_resident_loop_limits_default_and_large_steps(nb):
    """Mode 4 holds up to 704 particles per SM and is the default driver above 2048 particles while the system fits;
    beyond that it refuses loudly.  At N = 20 011 (ragged: 136 particles per CTA on 148 SMs, the last CTAs partly
    or wholly empty) the first block steps range from a handful of particles to more than 2048, so the run crosses
    the hand-over of a large step to the call sequence and back several times.  Two runs are bit-identical."""
    n = 20011
    pos, vel, m = plummer(n, seed=27)
    a = _mk(nb, pos, vel, m, 1e-4, 0.45, 2.0 ** -25, 2.0 ** -4, graph=4)
    a2 = _mk(nb, pos, vel, m, 1e-4, 0.45, 2.0 ** -25, 2.0 ** -4, graph=4)
    b = _mk(nb, pos, vel, m, 1e-4, 0.45, 2.0 ** -25, 2.0 ** -4, graph=False)
    d = nb.NBody(dev(pos), dev(vel), dev(m), 1e-4, 0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)   # default driver
    k = a.run_until(2.0 ** -6)
    assert k == b.run_until(2.0 ** -6) == a2.run_until(2.0 ** -6) == d.run_until(2.0 ** -6) and k > 100
    sa = _full(nb, a, n)
    assert _same(sa, _full(nb, b, n), 4)
    assert np.array_equal(sa, _full(nb, a2, n))                # run-to-run bit-reproducible
    assert np.array_equal(sa, _full(nb, d, n))                 # the default for this N is mode 4
    sa_, sb_ = a.stats(), b.stats()
    assert sa_["n_pairs"] == sb_["n_pairs"] and list(sa_["hist"]) == list(sb_["hist"]) and sa_["t_now"] == sb_["t_now"]
    assert sb_["hist"][11:].sum() > 0 and sb_["hist"][:4].sum() > 0        # steps on both sides of the hand-over
    # an exact step budget that ends inside a run of small steps, then inside the hand-over
    for steps in (3, 40, 1):
        a.run_steps(steps, log=False); b.run_steps(steps, log=False)
        assert a.stats()["n_steps"] == b.stats()["n_steps"]
    assert _same(_full(nb, a, n), _full(nb, b, n), 4)
    # the predicted stream after a run is the prediction of the last step taken
    pa, pb = [host(x) for x in a.pred()], [host(x) for x in b.pred()]
    for x, y in zip(pa, pb):
        assert np.abs(x - y).max() <= 1e-12 * np.abs(y).max()
    for g in (a, a2, b, d):
        g.close()
    big = 704 * torch.cuda.get_device_properties(0).multi_processor_count + 1
    pos, vel, m = plummer(big, seed=28)
    g = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    with pytest.raises(nb.NBError) as e:
        nb.nb_set_loop_mode(g.ctx, 4)
    assert e.value.code == nb.nb.NB_EINVAL
    g.close()


def test_grid_resident_loop_matches_oracle(nb, oracle):
    """The default driver above N = 1024 against the oracle's Hermite loop directly (N = 4000, ragged over 148 CTAs):
    same number of block steps, identical t_i and dt_i (every time-step decision), positions within 1e-9."""
    n = 4000
    pos, vel, m = plummer(n, seed=30)
    g = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    assert nb.nb_get_loop_mode(g.ctx) == 4
    k = g.run_until(2.0 ** -6)
    it = oracle.Integrator(pos, vel, m, eps=1e-3, eta=0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    assert it.run_until(2.0 ** -6)[0] == k and k > 50
    r, v, t, dt = [host(x) for x in g.state()]
    assert np.array_equal(t, it.t) and np.array_equal(dt, it.dt)
    assert (np.linalg.norm(r - it.pos, axis=1) / np.linalg.norm(it.pos, axis=1)).max() < 1e-9
    assert (np.linalg.norm(v - it.vel, axis=1) / np.linalg.norm(it.vel, axis=1)).max() < 1e-8
    g.close()


def test_grid_resident_loop_every_step_large(nb):
    """A shared time step (dt_min = dt_max) at N = 4096 >= the hand-over threshold: EVERY block step has m = N and goes
    to the call sequence with the all-particles list; the grid-resident kernel only selects.  Bit-identical to mode 0."""
    n = 4096
    pos, vel, m = plummer(n, seed=29)
    a = _mk(nb, pos, vel, m, 1e-2, 0.45, 2.0 ** -8, 2.0 ** -8, graph=4)
    b = _mk(nb, pos, vel, m, 1e-2, 0.45, 2.0 ** -8, 2.0 ** -8, graph=False)
    assert a.run_until(2.0 ** -5) == 8 and b.run_until(2.0 ** -5) == 8
    assert np.array_equal(_full(nb, a, n), _full(nb, b, n))
    a.run_steps(3, log=False); b.run_steps(3, log=False)
    assert np.array_equal(_full(nb, a, n), _full(nb, b, n)) and a.stats()["n_pairs"] == b.stats()["n_pairs"]
    a.close(); b.close()


@pytest.mark.parametrize("mode", [3, 4])
def test_resident_loop_mixed_precision(nb, mode):
    """Mixed SP/DP pair arithmetic (reading G27) inside the resident loops: float rounding in another order moves
    individual time-step decisions, so only the integrated quantities are compared with the call sequence."""
    # config 1's system with a wide floor on the step (2^-12): single-precision forces can drive the 6th-order
    # step rule of a particle in a close encounter down to dt_min; that is a property of the
    # mode, not of the driver, and would only make this comparison long
    pos, vel, m = plummer(1024, seed=1)
    a = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -12, 2.0 ** -4, graph=mode)
    b = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -12, 2.0 ** -4, graph=False)
    nb.nb_set_precision(a.ctx, 1); nb.nb_set_precision(b.ctx, 1)
    a.startup(); b.startup()
    e0 = b.energy()[0]
    na, nb_ = a.run_until(0.125), b.run_until(0.125)
    assert abs(na - nb_) <= 0.1 * nb_ and nb_ > 50
    ea, eb = a.energy()[0], b.energy()[0]
    assert abs(ea - eb) <= 1e-6 * abs(eb) and abs(ea - e0) <= 1e-6 * abs(e0)
    ra, rb = _full(nb, a, 1024)[:, 3:6], _full(nb, b, 1024)[:, 3:6]
    assert (np.linalg.norm(ra - rb, axis=1) / np.linalg.norm(rb, axis=1)).max() < 1e-4
    a.close(); b.close()
