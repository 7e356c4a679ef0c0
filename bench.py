#!/usr/bin/env python
"""bench.py -- the headline measurement of the HiGPUs hot path on B200.

Workload (default): BASELINE.json configs[2] at N = 2^20 -- Plummer sphere, equal masses,
eps = 1e-3, every particle active -- run as a COMPLETE Hermite block step, i.e. one pass of all
hot-path rows: next block / gather (a1), predictor for all N (a2), evaluation of acc+jerk+snap
of all N against all N (a3) in as many j-splits as keep the streamed piece L2-resident, summed in
fixed order (a4; the launch geometry is read back from the library and printed in
roofline.launch), corrector (a5) and new time steps (a6).  All particles share one time level (dt_min = dt_max), so each step is exactly one
full-N evaluation: N^2 = 1.0995e12 pair interactions.  north_star quotes the metric (FP64 pair
interactions/s, Tflop/s vs FP64 peak) on this full-N evaluation at N >= 1M.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--particles N]
                  [--workload step|force] [--no-cpu-baseline] [--no-e2e]

One JSON line on stdout (rank 0).  `--impl reference` times the CPU oracle (oracle/) on a
bounded sample of the same workload.  Multi-GPU: replicas only -- each
rank runs the same workload; value = units of all ranks / max-over-ranks device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# roofline.traffic comes from an ncu capture (bench.py cannot run under ncu itself): the JSON beside the
# ncu summary records which library version and launch geometry it was taken on, and the figure is
# reported only when both match what this run launched.
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "k_force_traffic.json")
FLOPS_PER_PAIR = 85.0        # 32 DFMA x 2 + 11 DMUL + 10 DADD, counted in the SASS
FLOPS_PER_PAIR_PAPER = 97.0  # the paper's convention (Table 2)
# FP64 ALU peak derived from unit counts and clocks: 148 SMs x 64 FP64
# lanes x 2 flop x 1.965 GHz (clocks.max.sm).  MEASURED_PEAKS.json has no FP64 entry.
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
METRIC = "fp64_pair_interactions_per_s"
UNIT = "interactions/s"
EPS = 1e-3
DT_SHARED = 2.0 ** -10


def ncu_traffic(N, launch, version):
    """(bytes per launch or None, note): dram__bytes_read.sum + dram__bytes_write.sum of the evaluation kernel
    from the committed ncu capture, valid only for the same library version, N and launch geometry."""
    try:
        with open(TRAFFIC_JSON) as f:
            rec = json.load(f)
    except Exception as e:
        return None, "no capture record (%s)" % e
    for c in rec.get("captures", []):
        if c.get("N") == N and c.get("nb_version") == version and c.get("launch") == launch:
            return int(c["dram_bytes_read"] + c["dram_bytes_write"]), \
                "bytes per launch, dram__bytes_read.sum + dram__bytes_write.sum of the ncu --set full capture in %s" % c.get("source")
    return None, "the committed ncu capture (%s) is of another library version / launch geometry than this run's (%s, %s)" % (
        os.path.relpath(TRAFFIC_JSON, ROOT), version, launch)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--particles", dest="n", type=int, default=1 << 20, help="particles (default 2^20, the configs[2] point north_star names)")
    ap.add_argument("--workload", default="step", choices=["step", "force"],
                    help="step: full block step (default); force: nb_force only (profiling aid)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-block-step", action="store_true", help="skip the block-step wall-time legs (configs 1 and 2)")
    return ap.parse_args()


def workload_name(N):
    k = int(round(np.log2(N)))
    return "config3_plummer_N2p%d_eps1e-3_all_active_full_block_step" % k


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(x: float, world: int, device="cuda") -> float:
    """MAX over ranks of a per-rank time (torch.distributed; NCCL on GPUs, gloo in the CPU tests)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def whole_job_value(units_per_rank_step: float, steps: int, world: int, ms_max: float) -> float:
    """Replicas only: every rank processes the same units; value = all ranks' units / max time."""
    return world * steps * units_per_rank_step / (ms_max * 1e-3)


# --------------------------------------------------------------------------------------------
def cpu_oracle_sample(pos, vel, accp, m, seconds_target=12.0):
    """Time the oracle's force evaluation, as it stands, on a bounded sample of i-rows x all N j."""
    import oracle.nb_oracle as orc
    N = m.shape[0]
    T = orc.num_threads()
    rng = np.random.default_rng(123)
    # calibrate on 2 rows per thread, then size the sample for ~seconds_target
    rows = rng.choice(N, size=min(N, 2 * T), replace=False).astype(np.int32)
    t0 = time.perf_counter(); orc.force(pos, vel, accp, m, EPS, rows); t1 = time.perf_counter()
    rate = rows.size * N / (t1 - t0)
    n_rows = int(min(N, max(T, seconds_target * rate / N)))
    n_rows = max(T, (n_rows // T) * T)
    rows = rng.choice(N, size=n_rows, replace=False).astype(np.int32)
    t0 = time.perf_counter(); orc.force(pos, vel, accp, m, EPS, rows); t1 = time.perf_counter()
    # the same on ONE core, on 1/8 of the rows (all cores and one core)
    one = None
    if T > 1:
        r1 = rows[:max(1, n_rows // 8)]
        orc.set_num_threads(1)
        s0 = time.perf_counter(); orc.force(pos, vel, accp, m, EPS, r1); s1 = time.perf_counter()
        orc.set_num_threads(T)
        one = r1.size * N / (s1 - s0)
    # the same source built with double arithmetic, -O3 -march=native (4x the rows: it is ~10x faster)
    plain = None
    try:
        rows4 = rng.choice(N, size=min(N, 4 * n_rows), replace=False).astype(np.int32)
        plain, _ = orc.force_plain_double_rate(pos, vel, accp, m, EPS, rows4)
    except Exception:
        plain = None
    return dict(value=n_rows * N / (t1 - t0), unit=UNIT, cores=T, kind="oracle", value_one_core=one,
                value_plain_double_O3_native=plain,
                sample="orc_force (long-double direct summation, a3 only: a1/a2/a5/a6 are O(N), <0.1%% of a step): "
                       "%d i-rows x %d j in %.1f s" % (n_rows, N, t1 - t0)), n_rows, (t1 - t0)


def run_reference(args):
    """--impl reference: the CPU oracle on the box's host cores, same metric/config; each step is
    a bounded sample (R i-rows x all N j) of the full-N evaluation."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle.nb_oracle as orc
    from workloads import config_inputs
    N = args.n
    pos, vel, m, accp = config_inputs(3, N)
    T = orc.num_threads()
    rng = np.random.default_rng(123)
    rows = rng.choice(N, size=min(N, 2 * T), replace=False).astype(np.int32)
    t0 = time.perf_counter(); orc.force(pos, vel, accp, m, EPS, rows); t1 = time.perf_counter()
    rate = rows.size * N / (t1 - t0)
    per_step_s = min(20.0, 120.0 / max(1, args.steps + args.warmup))
    n_rows = int(min(N, max(T, per_step_s * rate / N)))
    n_rows = max(T, (n_rows // T) * T)
    rows = rng.choice(N, size=n_rows, replace=False).astype(np.int32)
    for _ in range(args.warmup):
        orc.force(pos, vel, accp, m, EPS, rows)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.force(pos, vel, accp, m, EPS, rows)
    dt = time.perf_counter() - t0
    value = args.steps * n_rows * N / dt
    sample = "each step = orc_force on %d sampled i-rows x all %d j (of the %d x %d pairs of a full step)" % (n_rows, N, N, N)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / max(1, args.steps) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64 (long double accumulation)",
        "data": "synthetic", "config": {"workload": workload_name(N), "N": N, "eps": EPS, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": T, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "tflops_85": value * FLOPS_PER_PAIR / 1e12,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1207_2367_b200 as nb
    from workloads import config_inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    N = args.n
    K, W = args.steps, max(args.warmup, 0)
    pos, vel, m, accp = config_inputs(3, N)      # same seeded inputs on every rank (replicas)
    dev = lambda x: torch.as_tensor(x).cuda().contiguous()
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    g = nb.NBody(dev(pos), dev(vel), dev(m), EPS, 0.45, dt_min=DT_SHARED, dt_max=DT_SHARED)
    ctx = g.ctx
    ev = lambda: torch.cuda.Event(enable_timing=True)
    force_ms, sect = [], {"next_block": [], "predict": [], "force": [], "correct": []}

    def step(timed):
        """One full block step through the C-ABI; section events only on timed steps."""
        flush.zero_()                                   # L2 flush between iterations
        if args.workload == "force":
            es = [ev(), ev()]
            es[0].record(); nb.nb_force(ctx, None, N); es[1].record()
            if timed:
                force_ms.append(es)
            return
        es = [ev() for _ in range(5)]
        es[0].record()
        tn, n = nb.nb_next_block(ctx)
        assert n == N, "bench expects every particle active (shared level)"
        es[1].record()
        nb.nb_predict(ctx, tn)
        es[2].record()
        nb.nb_force(ctx, None, n)
        es[3].record()
        nb.nb_correct_and_step(ctx)
        es[4].record()
        if timed:
            force_ms.append((es[2], es[3]))
            for k, (a, b) in zip(("next_block", "predict", "force", "correct"), zip(es[:-1], es[1:])):
                sect[k].append((a, b))

    if args.workload == "step":
        g.startup()                                     # two full-N passes (start-up S0)
    else:
        nb.nb_set_pred_acc(ctx, dev(accp))
    for _ in range(W):
        step(False)
    barrier()
    launches0 = nb.nb_get_stats(ctx)["n_launch"]
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    t_start, t_end = ev(), ev()
    t_start.record()
    for _ in range(K):
        step(True)
    t_end.record()
    barrier()
    clk = clocks.stop() if rank == 0 else None
    ms_total = t_start.elapsed_time(t_end)
    launches = nb.nb_get_stats(ctx)["n_launch"] - launches0
    launch = {k: int(v) for k, v in nb.nb_get_launch(ctx).items()}   # what the last evaluation launched
    kern_ms = float(np.mean([a.elapsed_time(b) for a, b in force_ms])) if force_ms else float("nan")
    sections = {k: float(np.mean([a.elapsed_time(b) for a, b in v])) for k, v in sect.items() if v}
    ms_total = max_over_ranks(ms_total, world)
    pairs_per_step = float(N) * float(N)
    value = whole_job_value(pairs_per_step, K, world, ms_total)

    # energy drift over the run as a sanity check that the steps did real work
    diag = {}
    if args.workload == "step":
        st = nb.nb_get_stats(ctx)
        diag = {"t_now": st["t_now"], "block_steps_total": st["n_steps"], "pairs_total": st["n_pairs"]}

    # ---- e2e: same step through the C-ABI with HOST buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e and args.workload == "step":
        h_state = torch.empty((N, 21), dtype=torch.float64).pin_memory()
        nb.nb_get_full_state(ctx, h_state); torch.cuda.synchronize()
        h_out = torch.empty((N, 21), dtype=torch.float64).pin_memory()
        barrier()
        t0 = time.perf_counter()
        for _ in range(K):
            nb.nb_set_full_state(ctx, h_state)          # H2D: 21 doubles per particle
            tn, n = nb.nb_next_block(ctx)
            nb.nb_predict(ctx, tn)
            nb.nb_force(ctx, None, n)
            nb.nb_correct_and_step(ctx)
            nb.nb_get_full_state(ctx, h_out)            # D2H: 21 doubles per particle
            torch.cuda.synchronize()
            h_state, h_out = h_out, h_state
        barrier()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, world)
        e2e = {"value": whole_job_value(pairs_per_step, K, world, dt * 1e3), "unit": UNIT,
               "h2d_bytes_per_step": int(N * 21 * 8), "d2h_bytes_per_step": int(N * 21 * 8),
               "ms_per_step": dt / K * 1e3,
               "api": "nb_set_full_state(host) -> nb_next_block -> nb_predict -> nb_force -> nb_correct_and_step -> nb_get_full_state(host)"}

    probe_tf = None
    if rank == 0:
        f, _ = nb.nb_probe_fp64_peak(ctx, 1 << 16)
        probe_tf = f / 1e12
    g.close()

    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        cpu, _, _ = cpu_oracle_sample(pos, vel, accp, m)

    # the other half of BASELINE.json's metric, "block-step wall time": BASELINE.json configs[0] in full
    # (N = 1024 to t = 1) and the first 1/16 time unit of configs[1] (N = 65 536), device-driven loop
    block_step = None
    if rank == 0 and args.workload == "step" and not args.no_block_step:
        block_step = block_step_wall_time(nb, dev)

    if rank == 0:
        achieved = FLOPS_PER_PAIR * pairs_per_step / (kern_ms * 1e-3) / 1e12
        traffic, traffic_note = ncu_traffic(N, launch, nb.nb_version())
        kname = "k_force<%d,%d> variant %s, FP64, %d j-lane(s) per i" % (
            launch["threads"], launch["tile"], "A" if launch["threads"] == 128 else "B", launch["jlanes"])
        algorithmic = 80.0 * N * 2 + 72.0 * N * (launch["splits"] if launch["splits"] > 1 else 1)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(N) if args.workload == "step" else "config3_force_only_N%d" % N,
                       "N": N, "eps": EPS, "pairs_per_step": pairs_per_step, "shared_dt": DT_SHARED,
                       "parallelism": "replicas x%d" % world,
                       "l2": "flushed between steps (256 MiB memset inside the timed region); state 176 MB + stream 84 MB"},
            "tflops_85": value * FLOPS_PER_PAIR / 1e12, "tflops_97_paper_convention": value * FLOPS_PER_PAIR_PAPER / 1e12,
            "fp64_peak_frac_85": value / world * FLOPS_PER_PAIR / 1e12 / FP64_PEAK_TFLOPS,
            "roofline": {"bound": "alu", "kernel": kname, "achieved": achieved,
                         "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP64_PEAK_TFLOPS,
                         "frac_vs_probe": (achieved / probe_tf) if probe_tf else None,
                         "traffic": traffic, "traffic_note": traffic_note,
                         "algorithmic_bytes": algorithmic,
                         "kernel_ms": kern_ms,
                         "launch": dict(launch, grid=[launch["ctas"] // max(launch["splits"], 1), launch["splits"]],
                                        reduction="fixed-order sum of the split partials" if launch["splits"] > 1 else "none (one split)",
                                        version=nb.nb_version()),
                         "peak_source": "derived: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (DESIGN.md section 7); "
                                        "MEASURED_PEAKS.json has no FP64 entry",
                         "dfma_probe_tflops": probe_tf, "flops_per_pair": FLOPS_PER_PAIR,
                         "pipe_ceiling_frac": 85.0 / 106.0},
            "sections_ms": sections, "clocks": clk, "gpu_launches": int(launches),
            "e2e": e2e, "cpu_baseline": cpu, "block_step_wall_time": block_step, "diag": diag,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


LOOP_NAMES = {0: "host-issued calls", 1: "device-driven CUDA-graph batches", 2: "CUDA-graph batches with programmatic dependent launch",
              3: "cluster-resident loop (one kernel for the whole run, state in the shared memory of one cluster)",
              4: "grid-resident loop (one cooperative kernel on all SMs, state in shared memory; large steps by the streaming kernels)"}


def block_step_wall_time(nb, dev):
    """Wall time per block step of the Hermite loop (nb_run_until, device-driven) on the seeded inputs of
    BASELINE.json configs[0] (whole run) and configs[1] (first dt_max = 1/16 time unit)."""
    import torch
    from workloads import CONFIGS, config_inputs
    out = []
    for cfg, t_end in ((1, 1.0), (2, 1.0 / 16)):
        c = CONFIGS[cfg]
        pos, vel, m, _ = config_inputs(cfg)
        g = nb.NBody(dev(pos), dev(vel), dev(m), c["eps"], c["eta"], dt_min=c["dt_min"], dt_max=c["dt_max"])
        g.startup(); g.sync()
        e0 = g.energy()
        loop = LOOP_NAMES[nb.nb_get_loop_mode(g.ctx)]   # the library's default driver for this N (include/nb.h)
        g.run_until(0.0)                       # first launch (graph capture, buffers) outside the timed part
        torch.cuda.synchronize()
        t0 = time.perf_counter(); n = g.run_until(t_end); torch.cuda.synchronize(); wall = time.perf_counter() - t0
        e1 = g.energy()
        pairs = g.stats()["n_pairs"] - 2.0 * float(c["N"]) ** 2
        out.append({"workload": "config%d_%s_to_t=%g" % (cfg, c["name"], t_end), "N": c["N"], "block_steps": int(n),
                    "us_per_block_step": wall / max(n, 1) * 1e6, "wall_s": wall, "interactions_per_s": pairs / wall,
                    "dE_over_E": float((e1[0] - e0[0]) / e0[0]), "loop": loop})
        g.close()
    return out


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
