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
PRECISION = 0   # nb_set_precision mode of this run (--precision)
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


def _timed_force_b2b(nb, ctx, idx, n, reps, batch=8):
    """Device-side cost of one evaluation: `batch` calls enqueued behind a first one, so that the GPU never waits
    for the host (what a call costs inside a block-step loop); _timed_force times ONE call on an idle stream and
    therefore includes the host's enqueue latency (10-15 us)."""
    import torch
    best = None
    for _ in range(reps + 1):
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        nb.nb_force(ctx, idx, n)
        e0.record()
        for _b in range(batch):
            nb.nb_force(ctx, idx, n)
        e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / batch
        best = ms if best is None else min(best, ms)
    return best


def run_integration(nb, cfg, c, N, t_end, n_steps, loop=None):
    import torch
    from workloads import config_inputs
    pos, vel, m, _ = config_inputs(cfg, N)
    g = nb.NBody(_dev(pos), _dev(vel), _dev(m), c["eps"], c["eta"], dt_min=c["dt_min"], dt_max=c["dt_max"])
    if loop is not None:
        nb.nb_set_loop_mode(g.ctx, loop)
    nb.nb_set_precision(g.ctx, PRECISION)
    t0 = time.perf_counter(); g.startup(); g.sync(); t_start = time.perf_counter() - t0
    e0 = g.energy()
    out = {"config": cfg, "name": c["name"], "N": N, "eps": c["eps"], "eta": c["eta"], "loop_mode": nb.nb_get_loop_mode(g.ctx),
           "startup_s": t_start, "startup_pairs_per_s": 2.0 * N * N / t_start, "E0": float(e0[0])}
    if n_steps:                                   # config 5: a fixed number of block steps
        st0 = torch.empty((N, 21), dtype=torch.float64, device="cuda")
        nb.nb_get_full_state(g.ctx, st0); g.sync()
        lt, lm, ms = g.run_steps(n_steps)         # per-step log: host-issued calls, CUDA events per step
        out["steps"] = [{"t": float(t), "m": int(mm), "ms": float(x), "pairs_per_s": float(mm) * N / (float(x) * 1e-3)}
                        for t, mm, x in zip(lt, lm, ms)]
        # the same steps again from the same state through the device-driven loop, timed as a whole
        # (twice: the first run also captures and instantiates the CUDA graph of this context)
        for _ in range(2):
            nb.nb_set_full_state(g.ctx, st0); g.sync()
            t0 = time.perf_counter(); g.run_steps(n_steps, log=False); g.sync(); w = time.perf_counter() - t0
        out["host_issued_total_ms"] = float(sum(ms))
        out["device_loop_total_ms"] = w * 1e3
    else:
        g.run_until(0.0); g.sync()   # first launch of the driver (graph capture, exchange buffers, module load) outside the timed part
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
        nb.nb_set_precision(g.ctx, PRECISION)
        for mm in (ms_list or [N]):
            idx = None if mm == N else _dev(active_subset(N, mm, c.get("subset_seed", 40)), torch.int32)
            reps = 0 if mm * N > 4e12 else (1 if mm * N > 5e11 else 3)
            ms = _timed_force(nb, g.ctx, idx, mm, reps)
            pr = float(mm) * N / (ms * 1e-3)
            rows.append({"N": N, "m": mm, "ms": ms, "pairs_per_s": pr, "tflops_85": pr * FLOPS / 1e12,
                         "tflops_97": pr * 97.0 / 1e12, "frac_fp64_peak_85": pr * FLOPS / PEAK,
                         "launch": {k: int(v) for k, v in nb.nb_get_launch(g.ctx).items()}})
            if mm * N <= 2e10:   # small sets: also the device-side cost without the host's enqueue latency
                b2b = _timed_force_b2b(nb, g.ctx, idx, mm, 2)
                rows[-1].update({"ms_back_to_back": b2b, "pairs_per_s_back_to_back": float(mm) * N / (b2b * 1e-3),
                                 "frac_fp64_peak_85_back_to_back": float(mm) * N / (b2b * 1e-3) * FLOPS / PEAK})
            print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
        g.close()
    return {"config": cfg, "name": c["name"], "eps": c["eps"], "rows": rows}


def run_splitj_sweep(nb, N, ms_list):
    """SURVEY.md section 8(f) N1 / PAPER.md:256, Fig. 8: evaluation time versus the number m of active
    particles with the j-split chosen automatically ("Bfactor on") and with one split and one lane
    per i ("Bfactor off": one thread block per TpB i-particles), same inputs."""
    import torch
    from workloads import active_subset, config_inputs
    pos, vel, m, accp = config_inputs(4, N)
    g = nb.NBody(_dev(pos), _dev(vel), _dev(m), 1e-4, 0.45)
    nb.nb_set_pred_acc(g.ctx, _dev(accp))
    rows = []
    for mm in ms_list:
        idx = None if mm == N else _dev(active_subset(N, mm, 40), torch.int32)
        reps = 0 if mm * N > 4e12 else (1 if mm * N > 5e11 else 3)
        nb.nb_set_tuning(g.ctx, 0, 0)
        on = _timed_force(nb, g.ctx, idx, mm, reps)
        lon = {k: int(v) for k, v in nb.nb_get_launch(g.ctx).items()}
        nb.nb_set_tuning(g.ctx, 1, 1)
        off = _timed_force(nb, g.ctx, idx, mm, 0 if mm * N > 1e11 else reps)
        loff = {k: int(v) for k, v in nb.nb_get_launch(g.ctx).items()}
        rows.append({"N": N, "m": mm, "ms_split_auto": on, "ms_split_off": off, "gain": off / on,
                     "pairs_per_s_auto": float(mm) * N / (on * 1e-3), "pairs_per_s_off": float(mm) * N / (off * 1e-3),
                     "launch_auto": lon, "launch_off": loff})
        print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
    g.close()
    return {"experiment": "splitj_on_off", "rows": rows}


def run_heavy(nb, N, frac, t_end, eps=1e-4, eta=0.45):
    """SURVEY.md 8(f) N1 / PAPER.md:254: Plummer + one heavy particle; small blocks dominate."""
    from workloads import plummer_with_heavy
    pos, vel, m = plummer_with_heavy(N, seed=9, heavy_frac=frac)
    out = {"experiment": "heavy_particle", "N": N, "heavy_frac": frac, "eps": eps, "eta": eta, "t_end": t_end}
    for mode in (None, 1, 0):   # the library's default driver for this N, the graph-driven loop, host-issued calls
        g = nb.NBody(_dev(pos), _dev(vel), _dev(m), eps, eta, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
        if mode is not None:
            nb.nb_set_loop_mode(g.ctx, mode)
        g.startup(); g.sync()
        g.run_until(0.0); g.sync()   # first launch (graph capture, buffers) outside the timed part
        e0 = g.energy()
        t0 = time.perf_counter(); n = g.run_until(t_end); wall = time.perf_counter() - t0
        st = g.stats(); e1 = g.energy()
        pairs = st["n_pairs"] - 2.0 * N * N
        key = {None: "default_loop_mode_%d" % nb.nb_get_loop_mode(g.ctx), 1: "graph_loop", 0: "host_loop"}[mode]
        out[key] = {"block_steps": int(n), "wall_s": wall, "block_step_us": wall / max(n, 1) * 1e6,
                    "pairs": pairs, "pairs_per_s": pairs / wall, "dE_over_E": float((e1[0] - e0[0]) / e0[0])}
        if mode is None:
            out["active_hist_log2"] = {int(b): int(v) for b, v in enumerate(st["hist"]) if v}
            _, _, _, dt = g.state()
            out["dt_levels_log2"] = [int(np.log2(float(dt.min().item()))), int(np.log2(float(dt.max().item())))]
        g.close()
    return out


def run_fig1(nb, Ns, etas, t_end=4.5, every=0.5, eps=1e-4):
    """SURVEY.md 8(f) N2 / PAPER.md:136-153 (section 5.1, Eq. 20, Fig. 1) in FP64: mean relative energy and
    angular-momentum errors over the run, sampled every `every` Henon time units up to t_end = 4.5
    (9.96 of the paper's time units, G11), versus eta."""
    from workloads import plummer
    rows = []
    for N in Ns:
        pos, vel, m = plummer(N, seed=1500 + int(np.log2(N)))
        for eta in etas:
            g = nb.NBody(_dev(pos), _dev(vel), _dev(m), eps, eta, dt_min=2.0 ** -25, dt_max=2.0 ** -4)
            nb.nb_set_precision(g.ctx, PRECISION)
            g.startup(); g.sync()
            e0 = g.energy(); L0 = np.linalg.norm(e0[6:9])
            dE, dL = [], []
            t0 = time.perf_counter(); steps = 0
            k = 1
            while k * every <= t_end + 1e-12:
                steps += g.run_until(k * every)
                e = g.energy()
                dE.append(abs((e[0] - e0[0]) / e0[0])); dL.append(np.linalg.norm(e[6:9] - e0[6:9]) / L0)
                k += 1
            wall = time.perf_counter() - t0
            st = g.stats()
            rows.append({"N": N, "eta": eta, "mean_dE_over_E": float(np.mean(dE)), "final_dE_over_E": float(dE[-1]),
                         "mean_dL_over_L": float(np.mean(dL)), "L0": float(L0), "block_steps": int(steps),
                         "pairs": st["n_pairs"] - 2.0 * N * N, "wall_s": wall})
            print(json.dumps(rows[-1]), file=sys.stderr, flush=True)
            g.close()
    return {"experiment": "fig1_energy_vs_eta", "precision": ["fp64", "mixed", "mixed2"][PRECISION], "eps": eps, "t_end": t_end, "sample_every": every, "rows": rows}


def run_probe(nb):
    """DFMA-only peak probe on a tiny context (the measured denominator beside the derived FP64 peak)."""
    z = np.zeros((128, 3)); z[:, 0] = np.arange(128)
    g = nb.NBody(_dev(z), _dev(z), _dev(np.ones(128)), 1e-3, 0.45)
    f, ms = nb.nb_probe_fp64_peak(g.ctx, 1 << 17)
    g.close()
    return {"dfma_peak_tflops": f / 1e12, "nominal_tflops": PEAK / 1e12, "ms": ms}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=None, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--probe", action="store_true", help="DFMA-only FP64 peak probe (DESIGN.md section 7)")
    ap.add_argument("--n", type=int, default=None, help="override N (smaller dry runs)")
    ap.add_argument("--t-end", type=float, default=None)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--max-n", type=int, default=None, help="config 3: largest N of the sweep to run")
    ap.add_argument("--experiment", default=None, choices=["splitj", "heavy", "fig1"],
                    help="the 'next' rows of SURVEY.md 8(f): split-j on/off sweep, heavy-particle run, Fig. 1 in FP64")
    ap.add_argument("--etas", default="0.3,0.45,0.6,0.8,1.0")
    ap.add_argument("--ns", default=None, help="comma-separated N list for --experiment fig1")
    ap.add_argument("--ms", default=None, help="comma-separated active-set sizes for --config 4 (default: the config's five)")
    ap.add_argument("--heavy-frac", type=float, default=0.05)
    ap.add_argument("--loop", type=int, default=None, choices=[0, 1, 2, 3, 4], help="4: grid-resident loop (N <= ~100k); 0: host-driven loop, 1: device-driven graph batches, 2: the same with programmatic dependent launch, 3: cluster-resident loop (N <= 2048); default: 3 for N <= 1024, 4 while the system fits the shared memory, else 1")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed", "mixed2"],
                    help="evaluation arithmetic: fp64 (default), the paper's mixed SP/DP scheme (PAPER.md:287, reading G27), "
                         "or the same with acceleration and jerk summed in double (reading G27b: the 15 DP operations of PAPER.md:301)")
    a = ap.parse_args()
    import paper_1207_2367_b200 as nb
    from workloads import CONFIGS
    global PRECISION
    PRECISION = {"fp64": 0, "mixed": 1, "mixed2": 2}[a.precision]
    if a.experiment == "splitj":
        N = a.n or (1 << 20)
        ms = [1, 2, 4, 8, 16, 32, 64, 128, 256, 1024, 4096, 16384, 65536, 262144]
        print(json.dumps(run_splitj_sweep(nb, N, [x for x in ms if x <= N])), flush=True)
        return
    if a.experiment == "heavy":
        print(json.dumps(run_heavy(nb, a.n or 65536, a.heavy_frac, a.t_end if a.t_end is not None else 0.25)), flush=True)
        return
    if a.experiment == "fig1":
        Ns = [int(x) for x in a.ns.split(",")] if a.ns else [1 << 15]
        print(json.dumps(run_fig1(nb, Ns, [float(x) for x in a.etas.split(",")],
                                  t_end=a.t_end if a.t_end is not None else 4.5)), flush=True)
        return
    if a.probe or a.config is None:
        print(json.dumps(run_probe(nb)), flush=True)
        return
    c = CONFIGS[a.config]
    if c["kind"] == "integrate":
        N = a.n or c["N"]
        steps = a.steps if a.steps is not None else c.get("n_block_steps")
        out = run_integration(nb, a.config, c, N, a.t_end if a.t_end is not None else c.get("t_end"), steps, a.loop)
        out["loop"] = {None: "default (mode %d)" % out.pop("loop_mode"), 0: "host", 1: "graph", 2: "graph+pdl", 3: "cluster-resident", 4: "grid-resident"}[a.loop]
    elif a.config == 3:
        Ns = [a.n] if a.n else [n for n in c["N"] if not a.max_n or n <= a.max_n]
        out = run_force(nb, 3, c, Ns, None)
    else:
        N = a.n or c["N"]
        ms = [int(x) for x in a.ms.split(",")] if a.ms else c["m"]
        out = run_force(nb, 4, c, [N], [mm for mm in ms if mm <= N])
    out["precision"] = a.precision
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
