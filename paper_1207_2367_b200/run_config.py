"""Run one of the five BASELINE.json configurations through the C-ABI and print one JSON line.

  python -m paper_1207_2367_b200.run_config --config 1|2|3|4|5 [--n N] [--t-end T] [--steps K]

Inputs are the seeded synthetic recipes of workloads/ (DESIGN.md section 4).  Timing is by CUDA
events on the context stream (force-only configs) or host wall clock around the device loop
(integrations), as DESIGN.md section 8 states.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOPS = 85.0
PEAK = 148 * 64 * 2 * 1.965e9


def _dev(x, dtype=None):
    import torch
    return torch.as_tensor(x, dtype=dtype).cuda().contiguous()


def _timed_force(nb, ctx, idx, n, reps):
    import torch
    best = None
    for _ in range(reps + 1):
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(); nb.nb_force(ctx, idx, n); e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)   # first call is the warm-up unless reps == 0
    return best


def run_integration(nb, cfg, c, N, t_end, n_steps):
    import torch
    from workloads import config_inputs
    pos, vel, m, _ = config_inputs(cfg, N)
    g = nb.NBody(_dev(pos), _dev(vel), _dev(m), c["eps"], c["eta"], dt_min=c["dt_min"], dt_max=c["dt_max"])
    t0 = time.perf_counter(); g.startup(); g.sync(); t_start = time.perf_counter() - t0
    e0 = g.energy()
    out = {"config": cfg, "name": c["name"], "N": N, "eps": c["eps"], "eta": c["eta"],
           "startup_s": t_start, "startup_pairs_per_s": 2.0 * N * N / t_start, "E0": float(e0[0])}
    if n_steps:                                   # config 5: a fixed number of block steps
        lt, lm, ms = g.run_steps(n_steps)
        out["steps"] = [{"t": float(t), "m": int(mm), "ms": float(x), "pairs_per_s": float(mm) * N / (x * 1e-3)}
                        for t, mm, x in zip(lt, lm, ms)]
    else:
        t0 = time.perf_counter(); n = g.run_until(t_end); wall = time.perf_counter() - t0
        st = g.stats()
        e1 = g.energy()
        pairs = st["n_pairs"] - 2.0 * N * N
        hist = {int(b): int(v) for b, v in enumerate(st["hist"]) if v}
        _, _, t, dt = g.state()
        out.update({"t_end": t_end, "block_steps": int(n), "wall_s": wall, "block_step_ms": wall / max(n, 1) * 1e3,
                    "pairs": pairs, "pairs_per_s": pairs / wall, "tflops_85": pairs / wall * FLOPS / 1e12,
                    "dE_over_E": float((e1[0] - e0[0]) / e0[0]),
                    "dL": float(np.linalg.norm(e1[6:9] - e0[6:9])), "dP": float(np.linalg.norm(e1[3:6] - e0[3:6])),
                    "active_hist_log2": hist, "synchronised": bool((t == t_end).all().item()),
                    "dt_levels_log2": [int(np.log2(x)) for x in (float(dt.min().item()), float(dt.max().item()))]})
    g.close()
    return out


def run_force(nb, cfg, c, Ns, ms_list):
    import torch
    from workloads import active_subset, config_inputs
    rows = []
    for N in Ns:
        pos, vel, m, accp = config_inputs(cfg, N)
        g = nb.NBody(_dev(pos), _dev(vel), _dev(m), c["eps"], 0.45)
        nb.nb_set_pred_acc(g.ctx, _dev(accp))
        for mm in (ms_list or [N]):
            idx = None if mm == N else _dev(active_subset(N, mm, c.get("subset_seed", 40)), torch.int32)
            reps = 0 if mm * N > 4e12 else (1 if mm * N > 5e11 else 3)
            ms = _timed_force(nb, g.ctx, idx, mm, reps)
            pr = float(mm) * N / (ms * 1e-3)
            rows.append({"N": N, "m": mm, "ms": ms, "pairs_per_s": pr, "tflops_85": pr * FLOPS / 1e12,
                         "tflops_97": pr * 97.0 / 1e12, "frac_fp64_peak_85": pr * FLOPS / PEAK,
                         "launch": {k: int(v) for k, v in nb.nb_get_launch(g.ctx).items()}})
            print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
        g.close()
    return {"config": cfg, "name": c["name"], "eps": c["eps"], "rows": rows}


def run_probe(nb):
    """DFMA peak and operand-fetch probes on a tiny context."""
    import subprocess
    z = np.zeros((128, 3)); z[:, 0] = np.arange(128)
    g = nb.NBody(_dev(z), _dev(z), _dev(np.ones(128)), 1e-3, 0.45)
    try:
        mhz = float(subprocess.run(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i", "0"],
                                   capture_output=True, text=True).stdout.split()[0])
    except Exception:
        mhz = 1965.0
    f, ms = nb.nb_probe_fp64_peak(g.ctx, 1 << 17)
    names = {0: "1 register + immediates", 1: "3 distinct registers", 2: "3 registers, one shared by 3 consecutive DFMAs",
             3: "2 distinct registers (a*a+c)"}
    out = {"sm_mhz_assumed": mhz, "dfma_peak_tflops": f / 1e12, "nominal_tflops": PEAK / 1e12,
           "cycles_per_warp_inst_per_smsp": {names[k]: nb.nb_probe_fp64_operands(g.ctx, k, 20000, mhz) for k in range(4)}}
    g.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=None, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--probe", action="store_true", help="FP64 pipe probes only (DESIGN.md section 6.3)")
    ap.add_argument("--n", type=int, default=None, help="override N (smaller dry runs)")
    ap.add_argument("--t-end", type=float, default=None)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--max-n", type=int, default=None, help="config 3: largest N of the sweep to run")
    a = ap.parse_args()
    import paper_1207_2367_b200 as nb
    from workloads import CONFIGS
    if a.probe or a.config is None:
        print(json.dumps(run_probe(nb)), flush=True)
        return
    c = CONFIGS[a.config]
    if c["kind"] == "integrate":
        N = a.n or c["N"]
        steps = a.steps if a.steps is not None else c.get("n_block_steps")
        out = run_integration(nb, a.config, c, N, a.t_end if a.t_end is not None else c.get("t_end"), steps)
    elif a.config == 3:
        Ns = [a.n] if a.n else [n for n in c["N"] if not a.max_n or n <= a.max_n]
        out = run_force(nb, 3, c, Ns, None)
    else:
        N = a.n or c["N"]
        out = run_force(nb, 4, c, [N], [mm for mm in c["m"] if mm <= N])
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
