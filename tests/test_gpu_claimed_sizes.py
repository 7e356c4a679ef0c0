"""GPU-vs-oracle parity at the sizes and shapes BASELINE.json's configurations are claimed on, in the
launch configurations run_config.py / bench.py time:

  config 5  N = 2^23: start-up (two full-N passes), initial steps, the 8 block steps (scheduler bit-exact
            against a numpy restatement, evaluated rows against orc_force on the GPU's predicted stream),
            and the same 8 steps through the device-driven loop (bit-identical)
  config 4  N = 2^20, power-law masses, eps = 1e-4: m = 262 144 and m = N (a permutation)
  N1        Plummer + one heavy particle: lockstep with the oracle through both drivers
  N2        eta sweep: energy and angular-momentum errors against the oracle's
  a5        the interpolated crackle (G6, G7) against orc_correct_particle

The oracle computes sampled rows one by one (256 rows x 8.4M j take ~7 s on 16 host threads).
"""
import numpy as np
import pytest
import torch

from parity import FORCE_TOL, dev, g17_err, gpu_force, host
from workloads import CONFIGS, active_subset, config_inputs, plummer, plummer_with_heavy

pytestmark = pytest.mark.gpu


def _sample_rows(N, mass, pos, k=256, seed=7):
    rng = np.random.default_rng(seed)
    r = np.linalg.norm(pos, axis=1)
    special = [int(np.argmin(r)), int(np.argmax(r)), int(np.argmax(mass)), int(np.argmin(mass))]
    rest = rng.choice(N, size=k - len(special), replace=False)
    return np.unique(np.concatenate([special, rest])).astype(np.int32)


def _pow2floor_initial_dt(a, j, s, eta_init, lo, hi):
    """numpy restatement of S0 for whole arrays: plain double, frexp floor."""
    na, nj, ns = (np.sqrt((x * x).sum(axis=1)) for x in (a, j, s))
    with np.errstate(divide="ignore", invalid="ignore"):
        q1 = np.where(nj > 0, na / nj, np.inf)
        q2 = np.where(ns > 0, np.sqrt(na / ns), np.inf)
    x = eta_init * np.minimum(q1, q2)
    _, ex = np.frexp(np.where(np.isfinite(x) & (x > 0), x, 1.0))
    dt = np.where(np.isinf(x), hi, np.where(x > 0, np.ldexp(0.5, ex), lo))
    return np.clip(dt, lo, hi)


def test_config5_startup_and_eight_block_steps_at_full_size(nb, oracle):
    c = CONFIGS[5]
    N, eps = c["N"], c["eps"]
    pos, vel, m, _ = config_inputs(5)
    g = nb.NBody(dev(pos), dev(vel), dev(m), eps, c["eta"], dt_min=c["dt_min"], dt_max=c["dt_max"])
    g.startup()                                              # 2 x 7.0e13 pairs
    a, j, s, cr = [host(x) for x in g.derivs()]
    t = torch.empty(N, dtype=torch.float64, device="cuda"); dt = torch.empty_like(t)
    nb.nb_get_state(g.ctx, None, None, t, dt); g.sync()
    t0, dt0 = host(t), host(dt)
    assert np.all(t0 == 0) and np.all(cr == 0)
    # pass 2 is one evaluation with a_pred = a (G8): the oracle, fed the GPU's committed a, on sampled rows
    rows = _sample_rows(N, m, pos)
    ra, rj, rs = oracle.force(pos, vel, a, m, eps, rows)
    errs = (g17_err(a[rows], ra), g17_err(j[rows], rj), g17_err(s[rows], rs))
    assert max(errs) <= FORCE_TOL, errs
    # initial steps: identical to the oracle's rule on the same a, jerk, snap (sampled rows one by one,
    # all N through the numpy restatement)
    for i in rows:
        assert dt0[i] == oracle.initial_dt(a[i], j[i], s[i], 0.01, c["dt_min"], c["dt_max"])
    assert np.array_equal(dt0, _pow2floor_initial_dt(a, j, s, 0.01, c["dt_min"], c["dt_max"]))
    del cr

    state0 = torch.empty((N, 21), dtype=torch.float64, device="cuda")
    nb.nb_get_full_state(g.ctx, state0); g.sync()

    # the 8 block steps, call by call
    rng = np.random.default_rng(55)
    log = []
    for _ in range(c["n_block_steps"]):
        tn, n = g.next_block()
        nb.nb_get_state(g.ctx, None, None, t, dt); g.sync()
        nxt = host(t) + host(dt)
        assert tn == nxt.min()
        ref = np.nonzero(nxt == tn)[0].astype(np.int32)
        assert n == ref.size
        act = host(g.active(n))
        assert np.array_equal(act, ref)                      # ascending, bit-exact
        g.predict(tn)
        rp, vp, ap = [host(x) for x in g.pred()]
        f = g.force(None, n)
        fa, fj, fs = [host(x) for x in f]
        k = min(n, 48)
        sel = np.unique(np.concatenate([[0, n - 1], rng.choice(n, size=k, replace=False)]))
        oa, oj, os_ = oracle.force(rp, vp, ap, m, eps, act[sel])
        errs = (g17_err(fa[sel], oa), g17_err(fj[sel], oj), g17_err(fs[sel], os_))
        assert max(errs) <= FORCE_TOL, (n, errs)
        g.correct_and_step()
        log.append((tn, n))
        del rp, vp, ap
    assert len({n for _, n in log}) > 4                      # the steps span very different set sizes
    st_host = torch.empty((N, 21), dtype=torch.float64, device="cuda")
    nb.nb_get_full_state(g.ctx, st_host); g.sync()

    # the same 8 steps from the same state through the device-driven loop (what run_config times)
    nb.nb_set_full_state(g.ctx, state0)
    g.run_steps(c["n_block_steps"], log=False)
    st_dev = torch.empty((N, 21), dtype=torch.float64, device="cuda")
    nb.nb_get_full_state(g.ctx, st_dev); g.sync()
    assert torch.equal(st_host, st_dev)
    g.close()


@pytest.mark.parametrize("m_act", [262144, 1 << 20])
def test_config4_large_subsets(nb, oracle, m_act):
    # BASELINE.json config 4 at its two largest set sizes: power-law masses, eps = 1e-4, variant A over
    # several waves; m = N is the whole seeded permutation (every particle, random order)
    N = 1 << 20
    pos, vel, mass, accp = config_inputs(4)
    idx = active_subset(N, m_act, seed=40)
    (a, j, s), launch = gpu_force(nb, pos, vel, accp, mass, 1e-4, idx)
    assert launch["threads"] == 128 and launch["ctas"] > 148 * 4
    sel = np.random.default_rng(2).choice(m_act, 252, replace=False)
    heavy, light = int(np.argmax(mass[idx])), int(np.argmin(mass[idx]))
    sel = np.unique(np.concatenate([[0, m_act - 1, heavy, light], sel]))
    ra, rj, rs = oracle.force(pos, vel, accp, mass, 1e-4, idx[sel])
    errs = (g17_err(a[sel], ra), g17_err(j[sel], rj), g17_err(s[sel], rs))
    assert max(errs) <= FORCE_TOL, (errs, launch)
    if m_act == N:   # every particle once: antisymmetry => mass-weighted sums vanish
        mm = mass[idx][:, None]
        for x in (a, j, s):
            tot = np.abs((mm * x).sum(0)); ref = (mm * np.abs(x)).sum()
            assert np.all(tot <= 1e-13 * ref), (tot, ref)


def test_heavy_particle_lockstep_with_oracle_both_drivers(nb, oracle):
    # SURVEY.md 8(f) N1 / PAPER.md:254: one particle of 5 % of the mass; the stars bound to it take the
    # smallest steps and small blocks dominate.  >= 300 block steps: every t_next, active set and new dt
    # identical to the oracle's, host-issued calls; then the same steps through the device-driven loop.
    n, eps, eta = 1024, 1e-4, 0.45
    lo, hi = 2.0 ** -25, 2.0 ** -4
    pos, vel, m = plummer_with_heavy(n, seed=9, heavy_frac=0.05)
    assert m[0] == 0.05 and abs(m.sum() - 1.0) < 1e-14
    it = oracle.Integrator(pos, vel, m, eps=eps, eta=eta, dt_min=lo, dt_max=hi)
    g = nb.NBody(dev(pos), dev(vel), dev(m), eps, eta, dt_min=lo, dt_max=hi)
    g.startup()
    st0 = torch.empty((n, 21), dtype=torch.float64, device="cuda")
    nb.nb_get_full_state(g.ctx, st0); g.sync()
    steps, sizes = 320, []
    for _ in range(steps):
        tn, k = g.next_block()
        otn, oact = it.next_block()
        assert tn == otn and k == oact.size
        assert np.array_equal(host(g.active(k)), oact)
        g.predict(tn); nb.nb_force(g.ctx, None, k); g.correct_and_step()
        it.step()
        sizes.append(k)
    assert np.median(sizes) < 16                             # small blocks dominate
    r, v, t, dt = [host(x) for x in g.state()]
    assert np.array_equal(t, it.t) and np.array_equal(dt, it.dt)
    err = (np.linalg.norm(r - it.pos, axis=1) / np.maximum(np.linalg.norm(it.pos, axis=1), 1e-3)).max()
    assert err < 1e-11
    st_host = torch.empty_like(st0)
    nb.nb_get_full_state(g.ctx, st_host); g.sync()
    # graph-driven loop from the same start: bit-identical to the call sequence
    nb.nb_set_loop_mode(g.ctx, 1)
    nb.nb_set_full_state(g.ctx, st0)
    g.run_steps(steps, log=False)
    st_dev = torch.empty_like(st0)
    nb.nb_get_full_state(g.ctx, st_dev); g.sync()
    assert torch.equal(st_host, st_dev)
    # cluster-resident loop (the default driver at this N; its own summation order): the same steps and time
    # steps, positions to rounding
    nb.nb_set_loop_mode(g.ctx, 3)
    nb.nb_set_full_state(g.ctx, st0)
    g.run_steps(steps, log=False)
    st_res = torch.empty_like(st0)
    nb.nb_get_full_state(g.ctx, st_res); g.sync()
    a, b = host(st_res), host(st_host)
    assert np.array_equal(a[:, :3], b[:, :3])                # m, t, dt
    err = (np.linalg.norm(a[:, 3:6] - b[:, 3:6], axis=1) / np.maximum(np.linalg.norm(b[:, 3:6], axis=1), 1e-3)).max()
    assert err < 1e-11
    g.close()


@pytest.mark.parametrize("eta", [0.1, 0.2, 0.45, 0.6, 1.0])
def test_eta_sweep_energy_and_angular_momentum_against_oracle(nb, oracle, eta):
    # SURVEY.md 8(f) N2 / PAPER.md:136-153 (Eq. 20, Fig. 1): the relative energy error and the angular-momentum
    # error at t = 1 for several eta, GPU loop + nb_energy against the oracle's loop + orc_energy.
    n, eps = 256, 1e-3
    lo, hi = 2.0 ** -25, 2.0 ** -4
    pos, vel, m = plummer(n, seed=1)
    it = oracle.Integrator(pos, vel, m, eps=eps, eta=eta, dt_min=lo, dt_max=hi)
    oe0 = it.energy()
    n_orc, _, _ = it.run_until(1.0)
    oe1 = it.energy()
    g = nb.NBody(dev(pos), dev(vel), dev(m), eps, eta, dt_min=lo, dt_max=hi)
    g.startup()
    e0 = g.energy()
    n_gpu = g.run_until(1.0)
    e1 = g.energy()
    _, _, t, dt = [host(x) for x in g.state()]
    assert n_gpu == n_orc
    assert np.all(t == 1.0) and np.array_equal(dt, it.dt)    # every time-step decision identical
    E0, L0 = oe0[0], np.linalg.norm(oe0[6:9])
    dE_g, dE_o = (e1[0] - e0[0]) / E0, (oe1[0] - oe0[0]) / E0
    dL_g, dL_o = (e1[6:9] - e0[6:9]) / L0, (oe1[6:9] - oe0[6:9]) / L0
    assert abs(dE_g - dE_o) <= 1e-11, (dE_g, dE_o)
    assert np.abs(dL_g - dL_o).max() <= 1e-11, (dL_g, dL_o)
    # and the error itself behaves as the paper's Fig. 1 says: tiny at small eta, growing with eta
    assert abs(dE_g) < {0.1: 1e-10, 0.2: 2e-9, 0.45: 1e-7, 0.6: 1e-6, 1.0: 1e-4}[eta]
    g.close()


def test_crackle_and_corrected_state_against_oracle_corrector(nb, oracle):
    # a5 + G6/G7: after a block step the committed r, v and the stored crackle a^(3)(t1) of every active
    # particle equal orc_correct_particle fed the GPU's own pre-step state and evaluated a, jerk, snap;
    # the new dt equals orc_timestep on the oracle's a^(3..5).
    n, eps, eta = 700, 1e-3, 0.45
    lo, hi = 2.0 ** -25, 2.0 ** -4
    pos, vel, m = plummer(n, seed=21)
    g = nb.NBody(dev(pos), dev(vel), dev(m), eps, eta, dt_min=lo, dt_max=hi)
    g.startup()
    g.run_until(0.125)                   # past the first steps: crackle of the previous step is in use
    checked = 0
    for _ in range(40):
        tn, k = g.next_block()
        r0, v0, _, dt0 = [host(x) for x in g.state()]
        a0, j0, s0, _ = [host(x) for x in g.derivs()]
        act = host(g.active(k))
        g.predict(tn)
        a1, j1, s1 = [host(x) for x in g.force(None, k)]
        g.correct_and_step()
        r1, v1, t1, dt1 = [host(x) for x in g.state()]
        an, jn, sn, cn = [host(x) for x in g.derivs()]
        for q, i in enumerate(act):
            h = dt0[i]
            orr, orv, c3, c4, c5 = oracle.correct_particle(h, r0[i], v0[i], a0[i], j0[i], s0[i], a1[q], j1[q], s1[q])
            assert np.allclose(r1[i], orr, rtol=0, atol=4e-16 * max(1.0, np.abs(orr).max()))
            assert np.allclose(v1[i], orv, rtol=0, atol=4e-16 * max(1.0, np.abs(orv).max()))
            assert np.array_equal(an[i], a1[q]) and np.array_equal(jn[i], j1[q]) and np.array_equal(sn[i], s1[q])  # G16
            # a^(3) = 3 [20 dA - h (8 j0 + 12 j1) + h^2 (3 s1 - s0)] / h^3 cancels heavily: the two sides may
            # differ by a few roundings of the LARGEST term
            scale = 3.0 * (20 * np.abs(a1[q] - a0[i]) + h * (8 * np.abs(j0[i]) + 12 * np.abs(j1[q]))
                           + h * h * (3 * np.abs(s1[q]) + np.abs(s0[i]))) / h ** 3
            assert np.all(np.abs(cn[i] - c3) <= 8 * 2.0 ** -53 * scale), (cn[i], c3, scale)
            assert t1[i] == tn
            want = oracle.timestep(a1[q], j1[q], s1[q], c3, c4, c5, eta, h, tn, lo, hi)
            checked += 1
            if dt1[i] != want:   # only possible within rounding distance of a power-of-8 boundary (G23)
                pytest.fail("dt decision differs for particle %d: gpu %g oracle %g" % (i, dt1[i], want))
    assert checked > 200
    g.close()
