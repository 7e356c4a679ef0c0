"""Call-order state machine and argument checking of the C-ABI (include/nb.h):
the cases where a refused call must leave the context untouched, the debug index check, and the
calls that must not disturb data they do not own."""
import numpy as np
import pytest
import torch

from parity import dev, host
from workloads import mean_field_acc, plummer

pytestmark = pytest.mark.gpu


def _ctx(nb, n=1000, seed=42, eps=1e-3):
    pos, vel, m = plummer(n, seed=seed)
    g = nb.NBody(dev(pos), dev(vel), dev(m), eps, 0.45, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    return g, pos, vel, m


def test_j_slice_refusals_leave_the_context_untouched(nb):
    g, *_ = _ctx(nb)
    nb.nb_set_j_range(g.ctx, 128, 1000)
    for call in (lambda: g.run_until(0.1), lambda: g.run_steps(3, log=False), lambda: g.startup()):
        with pytest.raises(nb.NBError) as e:
            call()
        assert e.value.code == nb.nb.NB_ESTATE
    # not started: nb_set_limits is still allowed (it refuses once a start-up has been committed)
    nb.nb_set_limits(g.ctx, 2.0 ** -20, 2.0 ** -5)
    with pytest.raises(nb.NBError):
        g.next_block()                                        # needs a started context
    # with the slice removed the context starts normally
    nb.nb_set_j_range(g.ctx, 0, 1000)
    g.startup()
    tn, k = g.next_block()
    assert tn > 0 and k >= 1
    g.close()


def test_corrector_refuses_slice_partials_until_the_sums_are_stored(nb):
    g, *_ = _ctx(nb)
    g.startup()
    tn, k = g.next_block()
    g.predict(tn)
    nb.nb_force(g.ctx, None, k)
    full = torch.empty(9 * k, dtype=torch.float64, device="cuda")
    nb.nb_get_forces(g.ctx, full)
    # two slices: each evaluation alone must not reach the corrector
    parts = []
    for jb, je in ((0, 512), (512, 1000)):
        nb.nb_set_j_range(g.ctx, jb, je)
        nb.nb_force(g.ctx, None, k)
        with pytest.raises(nb.NBError) as e:
            g.correct_and_step()
        assert e.value.code == nb.nb.NB_ESTATE and "partials" in str(e.value)
        buf = torch.empty(9 * k, dtype=torch.float64, device="cuda")
        nb.nb_get_forces(g.ctx, buf)
        parts.append(buf)
    tot = parts[0] + parts[1]
    assert torch.allclose(tot, full, rtol=1e-13, atol=0)
    nb.nb_set_forces(g.ctx, tot)
    g.correct_and_step()                                      # now complete
    assert g.stats()["n_steps"] == 1
    g.close()


def test_debug_index_check(nb):
    g, pos, vel, m = _ctx(nb)
    good = torch.tensor([0, 5, 999, 5], dtype=torch.int32, device="cuda")
    out = [torch.empty((4, 3), dtype=torch.float64, device="cuda") for _ in range(3)]
    nb.nb_force(g.ctx, good, 4, *out); g.sync()
    ref = host(out[0]).copy()
    nb.nb_set_debug(g.ctx, 1)
    nb.nb_force(g.ctx, good, 4, *out); g.sync()               # valid lists pass unchanged
    assert np.array_equal(host(out[0]), ref)
    for bad, slot in (([0, 5, 1000, 7], 2), ([3, -1, 2, 1], 1), ([1 << 30, 0, 0, -5], 0)):
        idx = torch.tensor(bad, dtype=torch.int32, device="cuda")
        with pytest.raises(nb.NBError) as e:
            nb.nb_force(g.ctx, idx, 4, *out)
        assert e.value.code == nb.nb.NB_EINVAL and ("slot %d" % slot) in str(e.value)
    # host-side lists are checked the same way
    with pytest.raises(nb.NBError):
        nb.nb_force(g.ctx, np.array([0, 1, 2, 1000], dtype=np.int32), 4, *out)
    nb.nb_set_debug(g.ctx, 0)
    nb.nb_force(g.ctx, good, 4, *out); g.sync()
    assert np.array_equal(host(out[0]), ref)                  # the context is still usable
    g.close()


def test_energy_leaves_caller_set_predicted_data_alone(nb):
    g, pos, vel, m = _ctx(nb, n=777)
    nb.nb_set_pred_acc(g.ctx, dev(mean_field_acc(pos)))
    f1 = [host(x) for x in g.force()]
    e = g.energy()
    assert np.isfinite(e).all()
    f2 = [host(x) for x in g.force()]
    for x, y in zip(f1, f2):
        assert np.array_equal(x, y)                           # snap still sees the caller's a_j
    assert np.abs(f1[2]).max() > 0
    g.close()


def test_mixed_mode_with_tiny_softening_has_no_nan(nb):
    # m eps^-3 overflows a float for eps below ~1e-12: the self pair must be excluded explicitly
    for eps in (1e-14, 1e-30):
        g, pos, vel, m = _ctx(nb, n=300, eps=eps)
        nb.nb_set_precision(g.ctx, 1)
        a, j, s = [host(x) for x in g.force()]
        assert np.isfinite(a).all() and np.isfinite(j).all() and np.isfinite(s).all()
        nb.nb_set_precision(g.ctx, 0)
        a64 = host(g.force()[0])
        assert np.abs(a - a64).max() <= 1e-4 * np.abs(a64).max()
        g.close()


def test_energy_eps0_coincident_pair_is_finite(nb):
    pos = np.array([[0.0, 0, 0], [0.0, 0, 0], [1.0, 0, 0]])
    vel = np.zeros((3, 3)); m = np.array([0.25, 0.25, 0.5])
    g = nb.NBody(dev(pos), dev(vel), dev(m), 0.0, 0.45)
    e = g.energy()
    assert np.isfinite(e).all()
    assert e[2] == pytest.approx(-(0.25 * 0.5 + 0.25 * 0.5), rel=1e-14)   # the coincident pair adds nothing (G12)
    g.close()
