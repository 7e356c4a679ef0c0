"""GPU parity of the O(N)/O(m) steps and of whole trajectories against the oracle's Hermite
loop (oracle/nb_oracle.c), on the same seeded inputs, through the C-ABI.
  a1 next block / gather : bit-exact (t_next, ascending active list)
  a2 predictor           : <= 4 ulp-level relative error per component
  a5 corrector, a6 dt    : dt decisions identical; positions <= 1e-9 relative at t = 1 (north_star)
  a7 energy              : <= 1e-13 relative
"""
import math

import numpy as np
import pytest
import torch

from parity import dev, g17_err, host
from workloads import CONFIGS, config_inputs, kepler_binary, plummer

pytestmark = pytest.mark.gpu

TRAJ_TOL = 1e-9   # north_star: positions after 1 N-body time unit at N = 1024


def _mk(nb, pos, vel, m, eps, eta, dt_min, dt_max, eta_init=0.01):
    return nb.NBody(dev(pos), dev(vel), dev(m), eps, eta, dt_min=dt_min, dt_max=dt_max, eta_init=eta_init)


def _rel_pos_err(x_gpu, x_ref):
    return float((np.linalg.norm(x_gpu - x_ref, axis=1) / np.linalg.norm(x_ref, axis=1)).max())


def test_startup_matches_oracle(nb, oracle):
    pos, vel, m = plummer(300, seed=6)
    g = _mk(nb, pos, vel, m, 1e-2, 0.45, 2.0 ** -25, 2.0 ** -4)
    g.startup()
    it = oracle.Integrator(pos, vel, m, eps=1e-2, eta=0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    a, j, s, c = [host(x) for x in g.derivs()]
    assert g17_err(a, it.acc) < 1e-13 and g17_err(j, it.jerk) < 1e-13 and g17_err(s, it.snap) < 1e-13
    assert np.all(c == 0)
    _, _, t, dt = [host(x) for x in g.state()]
    assert np.all(t == 0) and np.array_equal(dt, it.dt)      # initial steps: identical decisions
    g.close()


def test_next_block_is_exact(nb, oracle):
    pos, vel, m = plummer(3000, seed=8)    # more than one scheduler block (2048 particles each)
    g = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4)
    g.startup()
    for _ in range(60):
        tn, n = g.next_block()
        _, _, t, dt = [host(x) for x in g.state()]
        nxt = t + dt
        assert tn == nxt.min()
        ref = np.nonzero(nxt == tn)[0].astype(np.int32)
        assert n == ref.size
        assert np.array_equal(host(g.active(n)), ref)          # ascending, bit-exact
        g.predict(tn); nb.nb_force(g.ctx, None, n); g.correct_and_step()
    g.close()


def test_predictor_matches_oracle(nb, oracle):
    pos, vel, m = plummer(700, seed=10)
    g = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4)
    g.run_until(0.2)                # particles now sit at different times with all derivatives set
    tn, n = g.next_block()
    g.predict(tn)
    r, v, t, _ = [host(x) for x in g.state()]
    a, j, s, c = [host(x) for x in g.derivs()]
    assert len(np.unique(t)) > 1
    rp, vp, ap = oracle.predict(tn, t, r, v, a, j, s, c)
    grp, gvp, gap = [host(x) for x in g.pred()]
    assert g17_err(grp, rp) < 1e-15 and g17_err(gvp, vp) < 1e-15 and g17_err(gap, ap) < 2e-15
    g.close()


def test_step_by_step_lockstep_with_oracle(nb, oracle):
    # every block step: same t_next, same active set, same new dt for every particle
    pos, vel, m = plummer(256, seed=1)
    lo, hi = 2.0 ** -25, 2.0 ** -4
    g = _mk(nb, pos, vel, m, 1e-3, 0.45, lo, hi)
    g.startup()
    it = oracle.Integrator(pos, vel, m, eps=1e-3, eta=0.45, dt_min=lo, dt_max=hi)
    n_steps = 0
    while True:
        tn, n = g.next_block()
        otn, oact = it.next_block()
        if tn > 0.25:
            break
        assert tn == otn and n == oact.size
        assert np.array_equal(host(g.active(n)), oact)
        g.predict(tn); nb.nb_force(g.ctx, None, n); g.correct_and_step()
        it.step()
        n_steps += 1
    r, v, t, dt = [host(x) for x in g.state()]
    assert np.array_equal(t, it.t) and np.array_equal(dt, it.dt)
    assert _rel_pos_err(r, it.pos) < 1e-12
    assert n_steps > 100
    g.close()


def test_config1_trajectory_parity(nb, oracle):
    # BASELINE.json config 1 in full: N = 1024, eps = 1e-3, eta = 0.45, dt_max = 1/16, to t = 1
    c = CONFIGS[1]
    pos, vel, m, _ = config_inputs(1)
    g = _mk(nb, pos, vel, m, c["eps"], c["eta"], c["dt_min"], c["dt_max"])
    g.startup()
    e0 = g.energy()
    n_gpu = g.run_until(c["t_end"])
    e1 = g.energy()
    it = oracle.Integrator(pos, vel, m, eps=c["eps"], eta=c["eta"], dt_min=c["dt_min"], dt_max=c["dt_max"])
    oe0 = it.energy()
    n_orc, _, _ = it.run_until(c["t_end"])
    oe1 = it.energy()
    r, v, t, dt = [host(x) for x in g.state()]
    assert np.all(t == c["t_end"]) and np.all(it.t == c["t_end"])        # synchronised at t = 1
    assert n_gpu == n_orc
    assert _rel_pos_err(r, it.pos) <= TRAJ_TOL
    assert _rel_pos_err(v, it.vel) <= 1e-8
    assert np.array_equal(dt, it.dt)            # every one of the 1.1e5 time-step decisions agrees (G23)
    st = g.stats()
    assert st["n_steps"] == n_gpu and np.array_equal(st["hist"], it.hist())
    assert st["n_pairs"] == it.n_pairs
    # energy: same initial value, same drift
    assert abs(e0[0] - oe0[0]) <= 1e-13 * abs(oe0[0])
    de_g = (e1[0] - e0[0]) / e0[0]; de_o = (oe1[0] - oe0[0]) / oe0[0]
    assert abs(de_g) < 1e-7 and abs(de_g - de_o) < 1e-11
    g.close()


def test_energy_matches_oracle(nb, oracle):
    for N, eps, seed in [(2, 0.0, 0), (129, 1e-2, 1), (5000, 1e-4, 2)]:
        pos, vel, m = plummer(N, seed=seed) if N > 2 else kepler_binary(0.3)
        g = _mk(nb, pos, vel, m, eps, 0.45, 2.0 ** -25, 2.0 ** -4)
        e = g.energy()
        ref = oracle.energy(pos, vel, m, eps)
        assert abs(e[1] - ref[1]) <= 1e-13 * abs(ref[1])
        assert abs(e[2] - ref[2]) <= 1e-13 * abs(ref[2])
        assert abs(e[0] - ref[0]) <= 1e-13 * (abs(ref[1]) + abs(ref[2]))
        scaleP = (m[:, None] * np.abs(vel)).sum()
        scaleL = (m[:, None] * np.abs(np.cross(pos, vel))).sum()
        assert np.all(np.abs(e[3:6] - ref[3:6]) <= 1e-14 * scaleP)
        assert np.all(np.abs(e[6:9] - ref[6:9]) <= 1e-14 * scaleL)
        g.close()


def test_kepler_closed_form_on_gpu(nb):
    # eps = 0, shared fixed step: the GPU integrator itself against Kepler's equation
    def kepler_rel(t, ecc):
        Mn = math.pi + t; E = Mn
        for _ in range(100):
            E -= (E - ecc * math.sin(E) - Mn) / (1 - ecc * math.cos(E))
        return np.array([-(math.cos(E) - ecc), -math.sqrt(1 - ecc * ecc) * math.sin(E), 0.0])
    pos, vel, m = kepler_binary(0.5)
    errs = []
    for k in (6, 7):
        g = _mk(nb, pos, vel, m, 0.0, 0.45, 2.0 ** -k, 2.0 ** -k)
        g.run_until(6.25)
        r, _, t, _ = [host(x) for x in g.state()]
        assert np.all(t == 6.25)
        errs.append(np.abs((r[0] - r[1]) - kepler_rel(6.25, 0.5)).max())
        g.close()
    assert 50 < errs[0] / errs[1] < 90 and errs[1] < 1e-8      # 6th order


def test_full_state_roundtrip_and_resume(nb):
    pos, vel, m = plummer(200, seed=12)
    lo, hi = 2.0 ** -25, 2.0 ** -4
    g = _mk(nb, pos, vel, m, 1e-3, 0.45, lo, hi)
    g.run_until(0.125)
    st = torch.empty((200, 21), dtype=torch.float64, device="cuda")
    nb.nb_get_full_state(g.ctx, st); g.sync()
    g.run_until(0.25)
    r1 = host(g.state()[0])
    h = _mk(nb, pos, vel, m, 1e-3, 0.45, lo, hi)
    nb.nb_set_full_state(h.ctx, st)
    assert h.stats()["t_now"] == 0.125
    h.run_until(0.25)
    assert np.array_equal(host(h.state()[0]), r1)           # checkpoint/resume is bit-exact
    g.close(); h.close()


def test_run_steps_log(nb):
    pos, vel, m = plummer(512, seed=13)
    g = _mk(nb, pos, vel, m, 1e-3, 0.45, 2.0 ** -25, 2.0 ** -4)
    lt, lm, ms = g.run_steps(8)
    assert np.all(np.diff(lt) > 0) and np.all(lm >= 1) and np.all(ms > 0)
    assert g.stats()["n_steps"] == 8
    g.close()


def test_shared_step_conserves_momentum(nb):
    # all particles on one level: pairwise antisymmetry makes the total momentum round-off only (G19)
    pos, vel, m = plummer(512, seed=3)
    g = _mk(nb, pos, vel, m, 1e-2, 0.45, 2.0 ** -7, 2.0 ** -7)
    g.run_until(0.25)
    P = g.energy()[3:6]
    assert np.all(np.abs(P) < 5e-15)
    g.close()


def test_config2_full_size_lockstep_with_oracle(nb, oracle):
    """BASELINE.json config 2 at its full size (N = 65 536, eps = 1e-4, eta = 0.45): start-up and the first
    block steps in lockstep with the oracle's Hermite loop -- same t_next, same active set, same new dt,
    positions to rounding.  (The whole run to t = 1 is 1.4e12 pairs: hours for the oracle; its
    conservation properties are checked in test_config2_short_run_properties.)"""
    c = CONFIGS[2]
    pos, vel, m, _ = config_inputs(2)
    g = _mk(nb, pos, vel, m, c["eps"], c["eta"], c["dt_min"], c["dt_max"])
    g.startup()
    it = oracle.Integrator(pos, vel, m, eps=c["eps"], eta=c["eta"], dt_min=c["dt_min"], dt_max=c["dt_max"])
    assert np.array_equal(host(g.state()[3]), it.dt)                  # initial steps: identical decisions
    for _ in range(40):
        tn, n = g.next_block()
        otn, oact = it.next_block()
        assert tn == otn and n == oact.size
        assert np.array_equal(host(g.active(n)), oact)
        g.predict(tn); nb.nb_force(g.ctx, None, n); g.correct_and_step()
        it.step()
    r, v, t, dt = [host(x) for x in g.state()]
    assert np.array_equal(t, it.t) and np.array_equal(dt, it.dt)
    assert _rel_pos_err(r, it.pos) < 1e-12
    g.close()


def test_config2_short_run_properties(nb):
    """Config 2 at full size through the device-driven loop for 1/32 time unit: the invariants that hold at
    any size -- every dt a power of two within the limits, t_i a multiple of dt_i, everybody synchronised at
    t_end (a multiple of dt_max), energy conserved to truncation level."""
    c = CONFIGS[2]
    pos, vel, m, _ = config_inputs(2)
    g = _mk(nb, pos, vel, m, c["eps"], c["eta"], c["dt_min"], c["dt_max"])
    g.startup()
    e0 = g.energy()
    t_end = c["dt_max"]                                                # 1/16
    n = g.run_until(t_end)
    e1 = g.energy()
    _, _, t, dt = [host(x) for x in g.state()]
    assert n > 500
    assert np.all(t == t_end)                                          # synchronised
    fr, ex = np.frexp(dt)
    assert np.all(fr == 0.5) and dt.min() >= c["dt_min"] and dt.max() <= c["dt_max"]
    assert np.all((t / dt) == np.rint(t / dt))
    assert abs((e1[0] - e0[0]) / e0[0]) < 1e-9
    st = g.stats()
    assert st["n_steps"] == n and st["hist"].sum() == n
    g.close()
