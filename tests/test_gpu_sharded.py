"""j-sharded evaluation (nb_set_j_range, nb_get_forces / nb_set_forces, nb_startup_commit;
SURVEY.md 8(f) N4) on ONE GPU: the `world` ranks are separate contexts driven one
after the other, and the test does the all-reduce by adding their buffers -- no kernel of one rank
waits on another.  Checks: slice partials sum to the oracle's full evaluation (<= 1e-12, G17);
the sharded block-step loop follows the unsharded one to rounding; all ranks stay BIT-identical.
"""
import numpy as np
import pytest
import torch

from parity import dev, g17_err, host
from paper_1207_2367_b200.sharded import ShardedNBody, j_range
from workloads import mean_field_acc, plummer

pytestmark = pytest.mark.gpu


def _unpack(buf, n):
    x = host(buf).reshape(9, n)
    return x[0:3].T.copy(), x[3:6].T.copy(), x[6:9].T.copy()


@pytest.mark.parametrize("world", [2, 3])
def test_slice_partials_sum_to_full_force(nb, oracle, world):
    n = 3000
    pos, vel, m = plummer(n, seed=41)
    accp = mean_field_acc(pos)
    total = torch.zeros(9 * n, dtype=torch.float64, device="cuda")
    for r in range(world):
        g = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45)
        nb.nb_set_pred_acc(g.ctx, dev(accp))
        nb.nb_set_j_range(g.ctx, *j_range(n, r, world))
        nb.nb_force(g.ctx, None, n)
        buf = torch.empty(9 * n, dtype=torch.float64, device="cuda")
        nb.nb_get_forces(g.ctx, buf); g.sync()
        total += buf
        g.close()
    a, j, s = _unpack(total, n)
    ra, rj, rs = oracle.force(pos, vel, accp, m, 1e-3)
    assert max(g17_err(a, ra), g17_err(j, rj), g17_err(s, rs)) <= 1e-12


def test_j_range_argument_checks(nb):
    pos, vel, m = plummer(1000, seed=42)
    g = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45)
    for bad in ((0, 100), (64, 1000), (128, 128), (-128, 256), (0, 1001)):
        with pytest.raises(nb.NBError):
            nb.nb_set_j_range(g.ctx, *bad)
    nb.nb_set_j_range(g.ctx, 128, 1000)
    with pytest.raises(nb.NBError):
        g.run_until(0.1)                      # the exchange is the caller's: no library-side loop
    g.close()


def test_sharded_loop_follows_the_unsharded_one_and_ranks_stay_identical(nb):
    n, world, t_end = 1500, 2, 0.0625
    pos, vel, m = plummer(n, seed=43)
    kw = dict(dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    ranks = [ShardedNBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, rank=r, world=world, reduce=None, **kw)
             for r in range(world)]

    def evaluate(k):                                          # the all-reduce, done by the test
        bufs = [rk.partial(k) for rk in ranks]
        tot = bufs[0].clone()
        for b in bufs[1:]:
            tot += b
        for rk in ranks:
            rk.finish(tot)

    for rk in ranks:
        nb.nb_predict(rk.g.ctx, 0.0)
    evaluate(n)
    for rk in ranks:
        nb.nb_startup_commit(rk.g.ctx, 1)
    evaluate(n)
    for rk in ranks:
        nb.nb_startup_commit(rk.g.ctx, 2)
    steps = 0
    while True:
        nxt = [nb.nb_next_block(rk.g.ctx) for rk in ranks]
        assert nxt[0] == nxt[1]                               # replicated scheduler: same (t_next, m)
        tn, k = nxt[0]
        if tn > t_end:
            break
        for rk in ranks:
            nb.nb_predict(rk.g.ctx, tn)
        evaluate(k)
        for rk in ranks:
            nb.nb_correct_and_step(rk.g.ctx)
        steps += 1

    ref = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, **kw)
    assert ref.run_until(t_end) == steps
    st = []
    for g in [rk.g for rk in ranks] + [ref]:
        x = torch.empty((n, 21), dtype=torch.float64, device="cuda")
        nb.nb_get_full_state(g.ctx, x); g.sync()
        st.append(host(x))
    assert np.array_equal(st[0], st[1])                       # ranks: bit-identical replicas
    assert np.array_equal(st[0][:, 1:3], st[2][:, 1:3])       # same t_i and dt_i as the single-GPU run
    r_sh, r_ref = st[0][:, 3:6], st[2][:, 3:6]
    err = (np.linalg.norm(r_sh - r_ref, axis=1) / np.linalg.norm(r_ref, axis=1)).max()
    assert err < 1e-11                                        # only the summation order differs
    for rk in ranks:
        rk.close()
    ref.close()


def test_sharded_world1_equals_plain_context(nb):
    n = 700
    pos, vel, m = plummer(n, seed=44)
    kw = dict(dt_min=2.0 ** -25, dt_max=2.0 ** -4)
    a = ShardedNBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, rank=0, world=1, reduce=lambda buf: None, **kw)
    a.startup()
    na = a.run_until(0.03125)
    b = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, **kw)
    nb.nb_set_loop_mode(b.ctx, 0)
    assert b.run_until(0.03125) == na
    xa = torch.empty((n, 21), dtype=torch.float64, device="cuda"); xb = torch.empty_like(xa)
    nb.nb_get_full_state(a.g.ctx, xa); nb.nb_get_full_state(b.ctx, xb); a.g.sync(); b.sync()
    assert np.array_equal(host(xa), host(xb))
    a.close(); b.close()


def test_sharded_driver_over_nccl_single_rank(nb):
    """The default exchange of ShardedNBody (torch.distributed.all_reduce on the NCCL backend) with a
    one-rank process group on this GPU: same states as the plain context, bit for bit."""
    import socket
    import torch.distributed as dist
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % port, rank=0, world_size=1)
    try:
        n = 900
        pos, vel, m = plummer(n, seed=45)
        kw = dict(dt_min=2.0 ** -25, dt_max=2.0 ** -4)
        a = ShardedNBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, **kw)       # rank/world from the process group
        assert (a.rank, a.world, a.j_begin, a.j_end) == (0, 1, 0, n)
        a.startup()
        na = a.run_until(0.03125)
        b = nb.NBody(dev(pos), dev(vel), dev(m), 1e-3, 0.45, **kw)
        nb.nb_set_loop_mode(b.ctx, 0)
        assert b.run_until(0.03125) == na and na > 10
        xa = torch.empty((n, 21), dtype=torch.float64, device="cuda"); xb = torch.empty_like(xa)
        nb.nb_get_full_state(a.g.ctx, xa); nb.nb_get_full_state(b.ctx, xb); a.g.sync(); b.sync()
        assert np.array_equal(host(xa), host(xb))
        a.close(); b.close()
    finally:
        dist.destroy_process_group()
