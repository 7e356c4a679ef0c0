"""Host side of the j-sharded multi-GPU path (Table 1 row 7)
on CPU: slice arithmetic, and the exchange step over two and three gloo ranks."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_1207_2367_b200.sharded import TILE, j_range  # noqa: E402


@pytest.mark.parametrize("N", [1, 127, 128, 129, 1000, 65536, 8388608, 1048576 + 77])
@pytest.mark.parametrize("world", [1, 2, 3, 8])
def test_j_range_partitions_whole_tiles(N, world):
    rs = [j_range(N, r, world) for r in range(world)]
    assert rs[0][0] == 0 and max(e for _, e in rs) == N
    for (b0, e0), (b1, e1) in zip(rs, rs[1:]):
        assert e0 == b1 or (b1 == N and e1 == N)             # contiguous; surplus ranks are empty
    for b, e in rs:
        assert b <= e and (e % TILE == 0 or e == N)
        assert b % TILE == 0 or (b == N and e == N)            # an empty slice sits at N
    sizes = [(e - b + TILE - 1) // TILE for b, e in rs]
    assert max(sizes) - min(sizes) <= 1                       # balanced to one tile


def test_j_range_rejects_bad_rank():
    with pytest.raises(ValueError):
        j_range(100, 2, 2)


def _port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_step_sums_slice_forces_to_the_full_evaluation(world):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(_port()),
           os.path.join("tests", "_sharded_worker.py"), "700"]
    p = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=300,
                       env=dict(os.environ, OMP_NUM_THREADS="2"))
    assert p.returncode == 0, p.stderr[-2000:]
    (line,) = [json.loads(l) for l in p.stdout.splitlines() if l.startswith("{")]
    assert line["world"] == world and line["n"] == 100
    assert line["ranges"][0][0] == 0 and line["ranges"][-1][1] == 700
    assert line["err"] < 1e-15                                # only the summation order differs
