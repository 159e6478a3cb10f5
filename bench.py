#!/usr/bin/env python
"""Benchmark of the superphoton transport hot path (one JSON line on stdout; contract in DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--ns NS] [--impl reference]

A step is one pass of the whole path of SURVEY.md 8(a) over one synthetic workload: device tables (S0), weights,
zone counts and prefix sum (S1-S4), emission (S5), tracking with absorption and scattering (S6-S10, S12), Compton
events (S11) in id-range batches (S13), and the spectrum scaling.  `value` is superphotons/s (emitted + scattered,
the paper's own count) with the fluid grid already resident in HBM; `e2e` is the same through the
C-ABI with HOST buffers (pinned grid in, spectrum out) inside the timed region.

Default workload: BASELINE.json configs[2] (2-D Kerr torus, N_s = 1e7) -- the single-GPU stand-in for the GRMHD
run on which the paper quotes its superphotons/s; `--config` selects another.
`--impl reference` times the CPU oracle (as it stands) on a bounded id sub-range of the same workload.
Under torchrun (N > 1) each rank runs the same workload with its own Philox seed (weak scaling: histories are
independent, no data-path collective); the tallies are summed once at the end.
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
sys.path.insert(0, ROOT)

from paper_2602_13198_b200 import workloads as wl  # noqa: E402
from paper_2602_13198_b200.shard import rank_seed, reduce_tally  # noqa: E402

METRIC = "superphotons/s tracked (incl. scattering)"
UNIT = "superphotons/s"
# algorithmic FP64 flop per geodesic step: dadd + dmul + 2 dfma predicated-on thread instructions
# of ALL tracker launches of a step divided by the in-grid steps they committed, counted with ncu on each config at
# the N_s and with the pass schedule this file times (profiles/r02_final.md, r02_flops_cfg*.csv), then frozen.  Since
# round 2 the figure depends on the config: a bounded step of the cold pass (configs 2, 3) needs neither gather nor
# plasma state nor opacity, a step in hot plasma needs all of them.  "track": average over the in-grid steps of
# track_kernel (all passes); "escape": free-flight step of escape_kernel.
FLOP_PER_STEP = {0: {"track": 681.1, "escape": 208.4}, 1: {"track": 705.8, "escape": 208.4},
                 2: {"track": 516.3, "escape": 368.2}, 3: {"track": 560.0, "escape": 368.2},
                 4: {"track": 700.3, "escape": 368.2}}
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant launch from one ncu capture; a constant of that capture
# (its command and N_s are named in TRAFFIC_SOURCE), not a quantity measured in this run.  The run itself reports the
# ALGORITHMIC bytes per launch beside it (roofline.algorithmic_bytes_per_launch).
TRAFFIC_BYTES_PER_LAUNCH = {2: 2.897e9 + 2.832e9}
TRAFFIC_SOURCE = {2: "profiles/r02_final.md (ncu --set full of this workload, cfg2 at N_s=1e7): hot tracker pass of the largest "
                     "scattering generation, 59 ms: reads 1.6e7 records of 160 B, writes as many hand-over / free-flight / "
                     "scattered records: DRAM traffic = algorithmic record bytes, the gather is served by L1/L2"}
# N_s at which FLOP_PER_STEP was counted (with the automatic pass schedule); at any other N_s, or with --phase-pairs /
# --k-cold set, bounded and full steps mix differently and the constant is off by up to ~35 %: the line then says so
FLOP_COUNTED_AT_NS = {0: 1e5, 1: 1e6, 2: 1e7, 3: 1e7, 4: 1e7}
# algorithmic record bytes of the SAME launch TRAFFIC_BYTES_PER_LAUNCH was captured on (cfg2, hot pass of the largest
# generation): 1.6e7 records of 160 B read, as many written
TRAFFIC_LAUNCH_RECORD_BYTES = {2: 2 * 1.6e7 * 160.0}
_WORKLOADS = {0: ("cfg0 thin synchrotron sphere 32x16", 1e5), 1: ("cfg1 scattering sphere 32x16", 1e6),
              2: ("cfg2 Kerr FM torus 256x256", 1e7), 3: ("cfg3 3-D perturbed torus 192x128x128", 1e7),
              4: ("cfg4 Kerr torus x1e3 density (analog scattering)", 1e6)}


def workload_name(cfg: int, ns=None) -> str:
    """Name of the workload with the N_s actually run (BASELINE.json's N_s of the config unless --ns overrides it)."""
    name, default_ns = _WORKLOADS[cfg]
    return f"{name}, Ns={(ns or default_ns):.0e}".replace("e+0", "e").replace("e+", "e")


WORKLOAD_NAMES = {c: workload_name(c) for c in _WORKLOADS}


def make_workload(cfg: int, ns: float | None, seed: int):
    kw = {"seed": seed}
    if ns:
        kw["Ns"] = ns
    p, prim = wl.CONFIGS[cfg](**kw)
    return p, prim


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region (profiling recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(p, prim, n_sample_primaries: int, threads: int = 0):
    """Time the CPU oracle (as it stands) on the first n primaries + all their descendants."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from oracle_binding import Oracle
    o = Oracle(p, prim)
    t0 = time.perf_counter()
    n = o.prepare()
    t1 = time.perf_counter()
    m = min(n, n_sample_primaries)
    used = o.run(0, m, threads)
    t2 = time.perf_counter()
    s = o.stats()
    tracked = s["n_primary"] + s["n_spawned"]
    return {"tracked": tracked, "run_s": t2 - t1, "prepare_s": t1 - t0, "cores": used, "n_sample": m,
            "steps": s["n_steps_total"]}


def run_reference(args, rank, world):
    if rank != 0:
        return
    p, prim = make_workload(args.config, args.ns, 1)
    # bounded sample per step: sized from a quick probe so that K+W steps end within a few minutes
    probe = oracle_sample(p, prim, 2000)
    rate = probe["tracked"] / max(probe["run_s"], 1e-6)
    per_primary = probe["tracked"] / max(probe["n_sample"], 1)
    target_s = min(20.0, 150.0 / max(1, args.steps + args.warmup))
    n_sample = int(max(500, rate * target_s / per_primary))
    times, tracked = [], 0
    for it in range(args.warmup + args.steps):
        r = oracle_sample(p, prim, n_sample)
        if it >= args.warmup:
            times.append(r["run_s"] + r["prepare_s"]); tracked = r["tracked"]; cores = r["cores"]
    ms = 1e3 * float(np.mean(times))
    value = tracked / (ms * 1e-3)
    wname = workload_name(args.config, args.ns)
    sample = f"first {n_sample} primaries of {wname} + all descendants per step (oracle prepare included)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": wname, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=sorted(wl.CONFIGS))
    ap.add_argument("--ns", type=float, default=None, help="override N_s of the config")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", dest="other_configs", action="store_false",
                    help="skip the other_configs list (cfg3 full grid, cfg4 at 1e7, cfg1, cfg0) printed after the headline")
    ap.add_argument("--phase-pairs", type=int, default=-1, help="hot/cold tracker pass pairs per generation (-1: library default)")
    ap.add_argument("--k-cold", type=int, default=4, help="cold steps after which a hot pass hands a superphoton over")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2602_13198_b200 import binding as gm

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")   # > 126 MB L2
    peak_meas, _ = gm.fp64_peak()
    peak = peak_meas / 1e12

    def measure(cfg: int, ns, steps: int, warmup: int, with_cpu_baseline: bool, min_timed_s: float = 0.0):
        """All of the bench line for one workload: device-timed steps, e2e steps, roofline, clocks.
        min_timed_s > 0: as many timed steps as fill that time (small workloads: a step of a few ms ends before
        the 200 ms clock sampler fires once; a sub-line without clock samples is no measurement)."""
        t_gen = time.perf_counter()
        p, prim = make_workload(cfg, ns, rank_seed(1, rank))
        gen_s = time.perf_counter() - t_gen
        g = gm.GPUMonty(p)
        g.set_phase_passes(args.phase_pairs, args.k_cold)
        host_grid = torch.from_numpy(prim).pin_memory()
        dev_grid = host_grid.cuda()
        nb = p["n_th"] * p["n_nu"]
        d_spec = torch.zeros(2, nb, dtype=torch.float64, device="cuda")

        def step(e2e: bool):
            g.build_tables(stream)
            g.set_grid(host_grid if e2e else dev_grid, stream)
            g.prepare(stream)
            g.run(stream=stream)
            if e2e:
                return g.spectrum()
            g.spectrum_device(d_spec[0], d_spec[1], stream)
            return None

        def timed(e2e: bool, nsteps: int):
            ms = []
            for _ in range(nsteps):
                flush.fill_(1.0)                                  # L2 flush between timed iterations
                if world > 1:
                    dist.barrier()
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                step(e2e)
                e1.record(stream)
                torch.cuda.synchronize()
                ms.append(e0.elapsed_time(e1))
            return ms

        for _ in range(warmup):
            step(False)
        torch.cuda.synchronize()
        if min_timed_s > 0.0:
            probe_ms = float(np.mean(timed(False, 2)))          # includes the L2 flush only as untimed work between steps
            steps = int(min(500, max(steps, np.ceil(min_timed_s * 1e3 / max(probe_ms, 1e-3)))))
        g.timing(True)
        clocks = ClockSampler(local)
        clocks.start()
        ms_dev = timed(False, steps)
        clk = clocks.stop()
        tm = g.timing(False)
        st = g.stats()
        tracked = st["n_primary"] + st["n_spawned"]
        ms_e2e = timed(True, steps)

        t_dev = torch.tensor([float(np.mean(ms_dev)), float(np.mean(ms_e2e))], device="cuda", dtype=torch.float64)
        cnt = torch.tensor([float(tracked)], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(t_dev, op=dist.ReduceOp.MAX)
            dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
            reduce_tally([torch.from_numpy(a).cuda() for a in g.tally()], dist)   # combined spectrum of the N runs
        ms_step, ms_step_e2e = float(t_dev[0]), float(t_dev[1])
        total = float(cnt[0])
        value = total / (ms_step * 1e-3)
        n_track_launches = max(1, tm["track"][1])
        steps_track = st["n_steps_total"] - st["n_steps_free"]      # steps taken inside track_kernel (this rank, last timed step)
        flops = steps_track * FLOP_PER_STEP[cfg]["track"]
        esc_ms = tm["escape"][0] / steps
        esc_tflops = st["n_steps_free"] * FLOP_PER_STEP[cfg]["escape"] / max(esc_ms * 1e-3, 1e-9) / 1e12
        track_ms_per_step = tm["track"][0] / steps
        achieved = flops / (track_ms_per_step * 1e-3) / 1e12
        launches = sum(v[1] for v in tm.values()) // max(1, steps)
        # algorithmic bytes of the dominant kernel per launch: every input record read once (160 B), every
        # hand-over / free-flight / scattered record written once (160 B), 4 (2-D) or 8 (3-D) 64-byte zone lines
        # gathered per in-grid step (served by L1/L2 except on the 201 MB grid of cfg 3)
        lpl = max(1, n_track_launches // max(1, steps))
        rec_bytes = (tracked + st["n_spawned"]) * 160.0 / lpl
        gather_bytes = steps_track * (8 if p["n3"] > 1 else 4) * 64.0 / lpl
        flop_valid = (args.phase_pairs < 0 and args.k_cold == 4 and (ns or _WORKLOADS[cfg][1]) == FLOP_COUNTED_AT_NS[cfg])
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": workload_name(cfg, ns),
                       "superphotons_per_step_per_gpu": tracked, "primaries": st["n_primary"], "spawned": st["n_spawned"],
                       "geodesic_steps": st["n_steps_total"], "geodesic_steps_free_flight": st["n_steps_free"],
                       "l2": "flushed between timed steps (256 MB write)", "host_generation_s": gen_s,
                       "multi_gpu": "one independent seeded run per rank, tallies summed once" if world > 1 else "single GPU"},
            "e2e": {"value": total / (ms_step_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(prim.nbytes),
                    "d2h_bytes_per_step": int(nb * 8 * 3), "ms_per_step": ms_step_e2e},
            "gpu_launches": int(launches),
            "clocks": clk,
            "roofline": {"bound": "alu", "kernel": "track_kernel", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                         "frac": achieved / peak, "traffic": TRAFFIC_BYTES_PER_LAUNCH.get(cfg),
                         "traffic_source": TRAFFIC_SOURCE.get(cfg),
                         # like for like with `traffic`: record bytes of the launch the capture was taken on, and their ratio
                         "traffic_launch_algorithmic_record_bytes": TRAFFIC_LAUNCH_RECORD_BYTES.get(cfg),
                         "traffic_over_algorithmic": (TRAFFIC_BYTES_PER_LAUNCH[cfg] / TRAFFIC_LAUNCH_RECORD_BYTES[cfg]
                                                      if cfg in TRAFFIC_LAUNCH_RECORD_BYTES else None),
                         # this run, averaged over ALL tracker launches of a step (not comparable with `traffic`):
                         # record bytes (DRAM) and the zone lines the gathers ask for (served by L1/L2 on the 2-D grids)
                         "avg_record_bytes_per_launch": rec_bytes, "avg_l2_gather_bytes_per_launch": gather_bytes,
                         "flop_per_step_valid": bool(flop_valid),
                         "peak_source": "DFMA-chain microbenchmark run in this process (gm_fp64_peak); nominal 2*64*148*1.965 GHz = 37.2",
                         "flop_per_step": FLOP_PER_STEP[cfg]["track"], "track_ms_per_step": track_ms_per_step,
                         "flop_per_step_note": "algorithmic flop of THIS implementation (ncu-counted, profiles/r02_final.md); "
                                               "round 1 needed 693.7 (cfg2) / 808.5 (cfg3) per step for the same histories",
                         "escape_kernel": {"achieved": esc_tflops, "frac": esc_tflops / peak, "ms_per_step": esc_ms,
                                           "flop_per_step": FLOP_PER_STEP[cfg]["escape"]},
                         "track_launches_per_step": lpl,
                         "track_share_of_step": track_ms_per_step / ms_step,
                         "kernel_ms_per_step": {k: v[0] / steps for k, v in tm.items()}},
        }
        if with_cpu_baseline and world == 1 and rank == 0:
            pr = oracle_sample(p, prim, 20000)        # probe (also pays the one-off oracle table build)
            pr = oracle_sample(p, prim, 20000)
            rate = pr["tracked"] / max(pr["run_s"], 1e-6)
            n_sample = int(max(20000, rate * 15.0 / (pr["tracked"] / max(1, pr["n_sample"]))))
            r = oracle_sample(p, prim, n_sample)
            r1 = oracle_sample(p, prim, max(2000, n_sample // (4 * max(1, r["cores"]))), threads=1)   # ~4 s on one thread
            out["cpu_baseline"] = {"value": r["tracked"] / r["run_s"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                                   "sample": f"first {r['n_sample']} primaries + descendants ({r['tracked']} superphotons, "
                                             f"{r['run_s']:.1f} s, oracle prepare {r['prepare_s']:.1f} s not counted)",
                                   "one_thread": {"value": r1["tracked"] / r1["run_s"], "unit": UNIT, "cores": r1["cores"],
                                                  "sample": f"first {r1['n_sample']} primaries + descendants "
                                                            f"({r1['tracked']} superphotons, {r1['run_s']:.1f} s)"}}
        g.close()
        del dev_grid, host_grid
        torch.cuda.empty_cache()
        return out

    out = measure(args.config, args.ns, args.steps, args.warmup, not args.no_cpu_baseline)
    if args.other_configs and world == 1:
        # the other BASELINE.json configs, driver-timed in the same run (3 warm-up + 3 timed steps each, same rules);
        # nothing is cached across runs: every grid is generated here (host_generation_s states the cost)
        others = []
        for cfg, ns in ((3, None), (4, 1e7), (1, None), (0, None)):
            if cfg == args.config and not args.ns:
                continue
            r = measure(cfg, ns, 3, 3, False, min_timed_s=1.2)
            others.append({"workload": r["config"]["workload"], "value": r["value"], "unit": UNIT,
                           "ms_per_step": r["ms_per_step"], "steps": r["steps"], "e2e_value": r["e2e"]["value"],
                           "flop_per_step_valid": r["roofline"]["flop_per_step_valid"],
                           "superphotons_per_step": r["config"]["superphotons_per_step_per_gpu"],
                           "tracker_frac_of_fp64_peak": r["roofline"]["frac"], "tracker_tflops": r["roofline"]["achieved"],
                           "track_share_of_step": r["roofline"]["track_share_of_step"],
                           "gpu_launches": r["gpu_launches"], "host_generation_s": r["config"]["host_generation_s"],
                           "clocks": r["clocks"]})
        out["other_configs"] = others
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
