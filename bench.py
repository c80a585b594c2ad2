#!/usr/bin/env python
"""bench.py -- TNLM enhancement (TNLM-E) throughput on B200, one JSON line on rank 0.

Contract (task statement): `python bench.py --gpus N --steps K --warmup W`; for N > 1 the driver
launches it under torch.distributed.run, one rank per GPU (NCCL).  A "step" is ONE full pass of the
hot path: tnlm_enhance on BASELINE.json configs[2] ("config3": 10 phases x 128 x 256 x 256, 3^3
patch, 5^3 window, h=0.05, mu=0.5, 10 Gauss-Jacobi sweeps with weights refreshed each sweep) on a
seeded synthetic thorax stack.  The metric is BASELINE.json's: voxel-offset updates per second.

  value     device-timed (CUDA events), inputs resident in HBM, max over ranks, whole job
  e2e       same metric through tnlm_enhance_host: pinned HOST buffers, H2D + D2H inside the timed region
  roofline  FP32-pipe ("alu") roofline of the sweep kernel, HBM figures beside it
  cpu_baseline  the oracle as it stands on the host cores, on a bounded sample of the same workload

`--impl reference` times the CPU oracle (the only "reference implementation" this paper has) and
prints the same line with "impl": "reference".  Multi-GPU: whole stacks are sharded over ranks
(independent scans), no data-path collective -> "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tnlm_voxel_offset_updates_per_sec"
UNIT = "updates/s"
SM_LANES = 128                       # FP32 lanes per SM (4 SMSP x 32), B200_PROFILING.md / B300_MICROARCH.md
NOMINAL_SM_MHZ = 1965.0              # clocks.max.sm of this pool's B200s (MEASURED_PEAKS.json)
FALLBACK_HBM_GBS = 6650.0            # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tnlm", choices=["tnlm", "reference"])
    ap.add_argument("--config", default="config3")
    ap.add_argument("--variant", type=int, default=0, help="0 auto, 1 generic, 2 tiled")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            d = json.load(fh)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", NOMINAL_SM_MHZ)),
                "source": "MEASURED_PEAKS.json"}
    except Exception:
        return {"hbm_gbs": FALLBACK_HBM_GBS, "sm_max_mhz": NOMINAL_SM_MHZ, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons every 200 ms while the timed region runs."""
    FIELDS = ["clocks.sm", "clocks.max.sm", "power.draw", "clocks_event_reasons.hw_slowdown",
              "clocks_event_reasons.hw_thermal_slowdown", "clocks_event_reasons.sw_thermal_slowdown",
              "clocks_event_reasons.sw_power_cap"]

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={','.join(self.FIELDS)}", "--format=csv,noheader,nounits",
                 "-i", str(self.index), "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < len(self.FIELDS):
                continue
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); power.append(float(r[2]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------
def oracle_sample_rate(cfg, g, seconds, threads_note=True):
    """Times the oracle (as it stands) on a bounded random sample of output voxels of ONE sweep of
    this workload; every sweep is identical work, so updates/s carries over to the K-sweep job."""
    import numpy as np
    from oracle import tnlm_oracle as O
    h, mu = np.float32(cfg.h), np.float32(cfg.mu)
    per_voxel = 2 * cfg.n_offsets
    rng = np.random.default_rng(99)
    n0 = 2000
    idx = rng.integers(0, g.size, n0)
    t = time.perf_counter()
    O.jacobi_step_at(g, g, cfg.patch_radius, cfg.search_radius, h, mu, idx)
    rate0 = n0 / max(time.perf_counter() - t, 1e-6)
    n = int(max(n0, min(rate0 * seconds, 5e7)))
    idx = rng.integers(0, g.size, n)
    t = time.perf_counter()
    O.jacobi_step_at(g, g, cfg.patch_radius, cfg.search_radius, h, mu, idx)
    dt = time.perf_counter() - t
    return {"value": n * per_voxel / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"one Eq. 8 sweep at {n} random output voxels ({n * per_voxel:.3g} voxel-offset updates, "
                      f"{dt:.1f} s) of the {cfg.name} stack; oracle/tnlm_oracle.c, OpenMP, fp64",
            "host_cpus": os.cpu_count()}


def run_reference(args, cfg):
    """`--impl reference`: the oracle, rank 0 only, same metric/config; a step = one bounded sample."""
    info_rank = int(os.environ.get("RANK", "0"))
    if info_rank != 0:
        return 0
    import numpy as np
    from tnlm_inputs import make_stack
    from oracle import tnlm_oracle as O
    g = make_stack(cfg)
    h, mu = np.float32(cfg.h), np.float32(cfg.mu)
    per_voxel = 2 * cfg.n_offsets
    rng = np.random.default_rng(99)
    idx = rng.integers(0, g.size, 2000)
    t = time.perf_counter()
    O.jacobi_step_at(g, g, cfg.patch_radius, cfg.search_radius, h, mu, idx)
    rate = 2000 / max(time.perf_counter() - t, 1e-6)
    budget = 150.0 / max(args.steps + args.warmup, 1)           # whole run within a few minutes
    n = int(max(2000, rate * min(budget, 10.0)))
    idx = rng.integers(0, g.size, n)
    for _ in range(args.warmup):
        O.jacobi_step_at(g, g, cfg.patch_radius, cfg.search_radius, h, mu, idx)
    t = time.perf_counter()
    for _ in range(args.steps):
        O.jacobi_step_at(g, g, cfg.patch_radius, cfg.search_radius, h, mu, idx)
    dt = time.perf_counter() - t
    value = args.steps * n * per_voxel / dt
    sample = (f"each step = one Eq. 8 sweep at {n} random output voxels ({n * per_voxel:.3g} updates) of the "
              f"{cfg.name} stack; oracle/tnlm_oracle.c, OpenMP, fp64")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args.gpus),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def workload_config(cfg, n_gpus):
    return {"workload": f"{cfg.name}: TNLM-E, {cfg.n_phase} phases x {cfg.nz}x{cfg.ny}x{cfg.nx} fp32 thorax phantom "
                        f"(seed {cfg.seed}+rank), patch {(2 * cfg.patch_radius + 1)}^3, window "
                        f"{(2 * cfg.search_radius + 1)}^3, h={cfg.h}, mu={cfg.mu}, {cfg.n_iter} Gauss-Jacobi sweeps, "
                        f"weights recomputed each sweep",
            "updates_per_step_per_gpu": cfg.updates_per_sweep * cfg.n_iter,
            "parallelism": f"dp{n_gpus} (one independent stack per GPU, no collective)",
            "l2_policy": "inputs larger than L2 (3 x 335 MB stacks per step vs 126 MB L2); no explicit flush"}


def main():
    args = parse_args()
    from tnlm_inputs import CONFIGS, make_stack
    cfg = CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, cfg)

    import numpy as np
    import torch
    import paper_1201_2450_b200 as T
    from paper_1201_2450_b200 import dist as D

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the TNLM path has no CPU fallback")
    T.lib()
    info = D.rank_info()
    torch.cuda.set_device(info.local_rank)
    info = D.init("nccl")
    dev = torch.device("cuda", info.local_rank)
    peaks = measured_peaks()

    # one independent, differently seeded stack per rank (weak scaling)
    rcfg = cfg.scaled(seed=cfg.seed + info.rank)
    g_host_np = make_stack(rcfg)
    p = T.TnlmParams.make(cfg.shape, cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)
    g = torch.from_numpy(g_host_np).to(dev)
    f_out = torch.empty_like(g)
    ws = torch.empty(T.workspace_bytes(p), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    updates_per_step = cfg.updates_per_sweep * cfg.n_iter
    launches_per_step = cfg.n_iter * T.launches_per_sweep(p)

    def step():
        T.tnlm_enhance(p, g, cfg.n_iter, f_out=f_out, ws=ws, stream=stream, variant=args.variant)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    # ---- device-timed region -------------------------------------------------------------
    sampler = ClockSampler(info.local_rank)
    if info.rank == 0:
        sampler.start()
    D.barrier(info)
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    D.barrier(info)
    elapsed_ms = D.max_over_ranks(info, ev0.elapsed_time(ev1), device=dev)
    clocks = sampler.stop() if info.rank == 0 else None
    value = info.world * args.steps * updates_per_step / (elapsed_ms * 1e-3)

    # ---- FP32 probe (register-resident FFMA loop) for the measured pipe peak -------------
    sink = torch.zeros(4, device=dev)
    T.probe_fp32(2000, sink, stream)
    torch.cuda.synchronize()
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pe0.record(stream)
    n_ffma = T.probe_fp32(40000, sink, stream)
    pe1.record(stream)
    torch.cuda.synchronize()
    probe_slots_per_s = n_ffma / (pe0.elapsed_time(pe1) * 1e-3)

    # ---- end-to-end through tnlm_enhance_host (pinned host buffers) ----------------------
    e2e = None
    if not args.no_e2e:
        g_pin = torch.from_numpy(g_host_np).pin_memory()
        out_pin = torch.empty(cfg.shape, dtype=torch.float32).pin_memory()
        dev_ws = torch.empty(T.host_workspace_bytes(p), dtype=torch.uint8, device=dev)
        T.tnlm_enhance_host(p, g_pin, cfg.n_iter, f_out_host=out_pin, dev_ws=dev_ws, stream=stream)   # warm
        D.barrier(info)
        torch.cuda.synchronize()
        n_e2e = max(1, min(args.steps, 3))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            T.tnlm_enhance_host(p, g_pin, cfg.n_iter, f_out_host=out_pin, dev_ws=dev_ws, stream=stream)
        torch.cuda.synchronize()
        dt = D.max_over_ranks(info, time.perf_counter() - t0, device=dev)
        assert torch.equal(out_pin, f_out.cpu()), "host path and device path disagree"
        e2e = {"value": info.world * n_e2e * updates_per_step / dt, "unit": UNIT,
               "h2d_bytes_per_step": g_pin.numel() * 4, "d2h_bytes_per_step": out_pin.numel() * 4,
               "ms_per_step": 1e3 * dt / n_e2e, "steps": n_e2e,
               "api": "tnlm_enhance_host (C ABI, pinned host buffers, copies + sync inside the timed region)"}
        del dev_ws

    if info.rank != 0:
        D.finalize(info)
        return 0

    # ---- roofline of the dominant (sweep) kernel ------------------------------------------
    n_launch = args.steps * cfg.n_iter
    launch_ms = elapsed_ms / n_launch                  # CUDA events over the timed region / sweeps
    props = torch.cuda.get_device_properties(dev)
    sms = props.multi_processor_count
    A = 5 + 6 * cfg.patch_radius                       # FP32-pipe slots per voxel-offset update
    achieved = cfg.updates_per_sweep * A / (launch_ms * 1e-3)
    peak = sms * SM_LANES * peaks["sm_max_mhz"] * 1e6
    alg_bytes = 3 * g.numel() * 4                      # read f, read g, write f_out
    traffic = None          # dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the committed ncu capture
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as fh:
            for row in csv.DictReader(fh):
                if row["kernel"] == T.kernel_name(p) and cfg.name == "config3":
                    traffic = int(row["dram_bytes_per_launch"])
    except Exception:
        pass
    roofline = {
        "bound": "alu", "kernel": T.kernel_name(p), "achieved": achieved / 1e12, "peak": peak / 1e12,
        "unit": "Tslot/s (FP32-pipe lane-operations; A = 5+6d slots per voxel-offset update)",
        "frac": achieved / peak, "traffic": traffic,
        "peak_source": f"{sms} SMs x {SM_LANES} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz (sm_max_mhz, {peaks['source']})",
        "launch_ms": launch_ms, "slots_per_update": A,
        "ffma_probe_tslots": probe_slots_per_s / 1e12, "frac_of_ffma_probe": achieved / probe_slots_per_s,
        "frac_at_observed_clock": (achieved / (sms * SM_LANES * clocks["sm_mhz"] * 1e6)) if clocks and clocks.get("sm_mhz") else None,
        "hbm": {"algorithmic_bytes_per_launch": alg_bytes, "achieved_gbs": alg_bytes / (launch_ms * 1e-3) / 1e9,
                "peak_gbs": peaks["hbm_gbs"], "frac": alg_bytes / (launch_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                "peak_source": peaks["source"]},
    }

    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline = oracle_sample_rate(cfg, g_host_np, args.cpu_seconds)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": info.world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": elapsed_ms / args.steps,
        "s_per_enhancement": elapsed_ms * 1e-3 / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(cfg, info.world), "clocks": clocks, "e2e": e2e,
        "gpu_launches": args.steps * launches_per_step, "roofline": roofline, "cpu_baseline": cpu_baseline,
        "impl": "tnlm", "kernel": T.kernel_name(p),
    }
    print(json.dumps(line), flush=True)
    D.finalize(info)
    return 0


if __name__ == "__main__":
    sys.exit(main())
