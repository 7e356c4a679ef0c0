"""N > 1 path of bench.py on CPU: "replicas only".  Two gloo ranks check the
max-over-ranks timing and the whole-job value; the reference arm runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _torchrun(args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_port())] + args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout, env=env)


def _json_lines(out):
    return [json.loads(l) for l in out.splitlines() if l.startswith("{")]


def test_max_over_ranks_and_whole_job_value():
    p = _torchrun([os.path.join("tests", "_multirank_worker.py")])
    assert p.returncode == 0, p.stderr[-2000:]
    (line,) = _json_lines(p.stdout)
    assert line["world"] == 2 and line["ms_max"] == 200.0             # the slower rank decides
    assert line["value"] == 2 * 3 * 1e6 / 0.2                         # units of ALL ranks / max time


def test_reference_arm_runs_on_rank0_only():
    p = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--particles", "2048", "--steps", "1", "--warmup", "0"])
    assert p.returncode == 0, p.stderr[-2000:]
    lines = _json_lines(p.stdout)
    assert len(lines) == 1                                            # rank 1 exits 0 without work
    r = lines[0]
    assert r["impl"] == "reference" and r["cpu_baseline"]["kind"] == "oracle" and r["value"] > 0
    assert r["e2e"]["h2d_bytes_per_step"] == 0 and r["e2e"]["value"] == r["value"]
    assert r["metric"] == "fp64_pair_interactions_per_s" and r["n_gpus"] == 2
