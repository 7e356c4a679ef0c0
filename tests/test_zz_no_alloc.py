"""nb_force_static (include/nb.h): the evaluation for callers that cannot allocate -- scratch in a fixed
`static __device__` array, no context, no cudaMalloc.  Checked against the existing path (nb_init + nb_set_pred_acc +
nb_force) within the force tolerance of the other GPU tests (G17, 1e-12), on calls made one after the other so
that a call sees the array as the previous one left it.  This file is named to be collected last."""
import numpy as np
import pytest
import torch

from parity import FORCE_TOL, dev, g17_err, gpu_force, host
from workloads import mean_field_acc, plummer

pytestmark = pytest.mark.gpu


def _static(nb, pos, vel, accp, mass, eps, idx=None):
    n = mass.shape[0] if idx is None else len(idx)
    out = [torch.full((n, 3), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)]
    nb.nb_force_static(dev(pos), dev(vel), None if accp is None else dev(accp), dev(mass), eps,
                       None if idx is None else dev(idx, torch.int32), n, *out, stream=torch.cuda.current_stream())
    torch.cuda.synchronize()
    return [host(o) for o in out]


def _case(N, seed, m, eps=1e-3):
    pos, vel, mass = plummer(N, seed=seed)
    accp = mean_field_acc(pos)
    idx = None if m is None else np.random.default_rng(seed).permutation(N)[:m].astype(np.int32)
    return pos, vel, accp, mass, eps, idx


def _agree(nb, case):
    pos, vel, accp, mass, eps, idx = case
    ref, _ = gpu_force(nb, pos, vel, accp, mass, eps, idx)
    got = _static(nb, pos, vel, accp, mass, eps, idx)
    for x, r in zip(got, ref):
        assert np.isfinite(x).all()
        assert g17_err(x, r) <= FORCE_TOL
    return got


def test_two_calls_in_a_row_match_the_existing_path(nb):
    # call 1: every particle of a ragged N (3 padding records short of a tile), one split or few
    a = _agree(nb, _case(3965, 11, None))
    # call 2 right after it: smaller N, 37 active (32 lanes per i, hundreds of j-splits): reads records and
    # partial sums where call 1 left other data
    b = _agree(nb, _case(1500, 12, 37))
    # and the first one again: same bits as before (fixed summation order, nothing stale picked up)
    a2 = _static(nb, *_case(3965, 11, None))
    for x, y in zip(a, a2):
        assert np.array_equal(x, y)
    assert b[0].shape == (37, 3)


@pytest.mark.parametrize("N,m,eps", [(4096, 1, 1e-3), (2500, 700, 1e-4), (640, 640, 0.0), (20000, 150, 1e-3)])
def test_set_sizes_and_eps_zero(nb, N, m, eps):
    _agree(nb, _case(N, 20 + m, None if m == N else m, eps))


def test_matches_the_oracle(nb, oracle):
    pos, vel, accp, mass, eps, idx = _case(1000, 31, 90)
    got = _static(nb, pos, vel, accp, mass, eps, idx)
    ref = oracle.force(pos, vel, accp, mass, eps, idx=idx)
    for x, r in zip(got, ref):
        assert g17_err(x, r) <= FORCE_TOL


def test_optional_arguments(nb):
    pos, vel, accp, mass, eps, idx = _case(777, 41, 50)
    ref, _ = gpu_force(nb, pos, vel, None, mass, eps, idx)            # a_pred = 0 after nb_init
    n = len(idx)
    jerk = torch.full((n, 3), float("nan"), dtype=torch.float64, device="cuda")
    nb.nb_force_static(dev(pos), dev(vel), None, dev(mass), eps, dev(idx, torch.int32), n, None, jerk, None)
    torch.cuda.synchronize()
    assert g17_err(host(jerk), ref[1]) <= FORCE_TOL
    nb.nb_force_static(dev(pos), dev(vel), None, dev(mass), eps, None, 0)   # empty set: set-up only


def test_sizes_beyond_the_array_are_refused(nb):
    N = nb.NB_STATIC_MAX_N + 1
    z = torch.zeros((N, 3), dtype=torch.float64, device="cuda")
    mass = torch.ones(N, dtype=torch.float64, device="cuda")
    out = torch.zeros((N, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(nb.NBError) as e:
        nb.nb_force_static(z, z, None, mass, 1e-3, None, N, out)
    assert e.value.code == nb.nb.NB_EINVAL and "NB_STATIC_MAX_N" in str(e.value)
    with pytest.raises(nb.NBError):
        nb.nb_force_static(z[:10], z[:10], None, mass[:10], 1e-3, None, 5, out[:5])   # NULL list needs n_active == N
    with pytest.raises(TypeError):
        nb.nb_force_static(np.zeros((4, 3)), np.zeros((4, 3)), None, np.ones(4), 1e-3, None, 4)   # host arrays


def test_largest_size_fits(nb):
    N = nb.NB_STATIC_MAX_N
    pos, vel, mass = plummer(N, seed=51)
    idx = np.arange(0, N, 257, dtype=np.int32)
    ref, _ = gpu_force(nb, pos, vel, None, mass, 1e-3, idx)
    got = _static(nb, pos, vel, None, mass, 1e-3, idx)
    for x, r in zip(got, ref):
        assert g17_err(x, r) <= FORCE_TOL
    full = _static(nb, pos, vel, None, mass, 1e-3, None)              # m = N: one split, 9 N sums in the array
    for q in range(3):
        assert g17_err(full[q][idx], ref[q]) <= FORCE_TOL


def test_runs_under_stream_capture(nb):
    """What the entry point is for: a capture in global mode refuses cudaMalloc and friends, so a graph that
    captures, instantiates and replays proves the call allocated nothing.  Replayed twice on changed inputs."""
    pos, vel, accp, mass, eps, idx = _case(2000, 61, 64)
    p, v, a, m_, ix = dev(pos), dev(vel), dev(accp), dev(mass), dev(idx, torch.int32)
    out = [torch.zeros((len(idx), 3), dtype=torch.float64, device="cuda") for _ in range(3)]
    nb.nb_force_static(p, v, a, m_, eps, ix, len(idx), *out, stream=torch.cuda.current_stream())   # set-up + kernels loaded
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        nb.nb_force_static(p, v, a, m_, eps, ix, len(idx), *out, stream=torch.cuda.current_stream())
    for scale in (1.0, 1.5):
        p.copy_(dev(pos * scale))
        for o in out:
            o.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        ref, _ = gpu_force(nb, pos * scale, vel, accp, mass, eps, idx)
        for x, r in zip(out, ref):
            assert g17_err(host(x), r) <= FORCE_TOL
