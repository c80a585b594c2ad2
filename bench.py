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
(independent scans), no data-path collective -> "scaling": "weak".  `--scaling strong` instead splits ONE
stack into z-slabs over the ranks (halo exchange per sweep) and prints "scaling": "strong".
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

VARIANT_NAMES = {1: "jacobi_generic_kernel", 2: "tnlm_tiled_kernel"}
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
    ap.add_argument("--config", default="config3",
                    help="config1..config4: one enhancement per step; config5: the (patch, window) sweep of "
                         "BASELINE.json configs[4], one step = the eight enhancements, per-point figures in 'points'")
    ap.add_argument("--variant", type=int, default=0, help="kernel variant: 0 auto, 1 generic, 2 tiled, 3 paired (shared memory), 4 paired with TMEM operands")
    ap.add_argument("--ref", default="same", choices=["same", "separate"],
                    help="separate: every sweep takes its weights from a second stack (tnlm_jacobi_step(ref=...), "
                         "the TNLM-R form of the call, PAPER.md:198) instead of from the iterate; no e2e leg")
    ap.add_argument("--metrics", action="store_true",
                    help="also evaluate the paper's SRR (Eq. 10) and CNR on the enhanced stack and time the TV kernel")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak: one independent stack per GPU (the contract's line); strong: ONE stack split into z-slabs "
                         "over the ranks, each storing slab + halo only, halo exchange per sweep (dist.enhance_z_slabs_local)")
    ap.add_argument("--loopback-world", type=int, default=0,
                    help="with --scaling strong on ONE GPU: time the slab of every rank of a W-rank split one after the other "
                         "(halo planes filled locally, no exchange) and print the slowest rank's time: the compute side of the "
                         "strong-scaling curve, not a multi-GPU measurement")
    ap.add_argument("--tnlmr", action="store_true",
                    help="time the TNLM-R path (include/tnlmr.h) instead: the paper's phantom geometry (PAPER.md:245: 10 phases x "
                         "128^3 voxels, 30 views per phase, 512^2 detector), analytic ellipsoid projections, a step = one outer "
                         "iteration (3 CGLS iterations + sweep + clamp); prints its own JSON line")
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


def workload_config(cfg, n_gpus, sweep=False):
    what = (f"{cfg.name}: TNLM-E, {cfg.n_phase} phases x {cfg.nz}x{cfg.ny}x{cfg.nx} fp32 thorax phantom "
            f"(seed {cfg.seed}+rank), ")
    if sweep:
        what += (f"parameter sweep patch {{3^3, 5^3}} x window {{3^3, 5^3, 7^3, 9^3}}, h={cfg.h}, mu={cfg.mu}, "
                 f"{cfg.n_iter} Gauss-Jacobi sweeps per point, weights recomputed each sweep")
        per_step = sum(cfg.scaled(search_radius=M).updates_per_sweep for _ in (1, 2) for M in (1, 2, 3, 4)) * cfg.n_iter
    else:
        what += (f"patch {(2 * cfg.patch_radius + 1)}^3, window {(2 * cfg.search_radius + 1)}^3, h={cfg.h}, mu={cfg.mu}, "
                 f"{cfg.n_iter} Gauss-Jacobi sweeps, weights recomputed each sweep")
        per_step = cfg.updates_per_sweep * cfg.n_iter
    stack_mb = cfg.n_phase * cfg.voxels_per_phase * 4 / 1e6
    return {"workload": what, "updates_per_step_per_gpu": per_step,
            "parallelism": f"dp{n_gpus} (one independent stack per GPU, no collective)",
            "l2_policy": f"inputs larger than L2 (3 x {stack_mb:.0f} MB stacks per step vs 126 MB L2); no explicit flush"
                         if 3 * stack_mb > 126 else
                         f"3 x {stack_mb:.0f} MB stacks fit the 126 MB L2: the bench writes a 256 MB buffer between steps"}


def kernel_label(T, p, variant):
    """Name of the kernel the timed call launches (AUTO and PAIRED resolve through the library)."""
    if variant in VARIANT_NAMES:
        return VARIANT_NAMES[variant]
    return T.kernel_name(p)


def committed_traffic(kernel, cfg_name):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` at `cfg_name`, from the committed ncu
    capture (profiles/traffic.csv); None if that pair was not captured."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as fh:
            for row in csv.DictReader(fh):
                if row["kernel"] == kernel and row.get("config", "config3") == cfg_name:
                    return int(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


def roofline_block(T, p, cfg, variant, launch_ms, sms, peaks, clocks, probe_slots_per_s, stack_elems):
    """FP32-pipe ("alu") roofline of the sweep kernel; DESIGN.md section 5 defines the unit and the peak."""
    d = cfg.patch_radius
    A = 5 + 6 * d                                      # FP32-pipe slots per voxel-offset update
    A_shared = (3 + 6 * d) / 2 + 2                     # the same with the paper's mutual-weight sharing
    rate = cfg.updates_per_sweep / (launch_ms * 1e-3)  # updates/s of one launch
    peak = sms * SM_LANES * peaks["sm_max_mhz"] * 1e6
    alg_bytes = 3 * stack_elems * 4                    # read f, read g, write f_out
    kernel = kernel_label(T, p, variant)
    out = {
        "bound": "alu", "kernel": kernel, "achieved": rate * A / 1e12, "peak": peak / 1e12,
        "unit": "Tslot/s (FP32-pipe lane-operations; A = 5+6d slots per voxel-offset update)",
        "frac": rate * A / peak, "traffic": committed_traffic(kernel, cfg.name),
        "frac_vs_A_shared": rate * A_shared / peak, "slots_per_update": A, "slots_per_update_shared": A_shared,
        "peak_source": f"{sms} SMs x {SM_LANES} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz (sm_max_mhz, {peaks['source']})",
        "launch_ms": launch_ms,
        "hbm": {"algorithmic_bytes_per_launch": alg_bytes, "achieved_gbs": alg_bytes / (launch_ms * 1e-3) / 1e9,
                "peak_gbs": peaks["hbm_gbs"], "frac": alg_bytes / (launch_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                "peak_source": peaks["source"]},
    }
    out["issue_model"] = ("packed FP32 instructions hold the issue port for two cycles: the sweep kernels are bound by issue slots "
                          "(pair_tm at config 3: 18.5 slots per update against A = 11, 0.91 slots per cycle; profiles/r02_issue_model.md)")
    if probe_slots_per_s:
        out["ffma_probe_tslots"] = probe_slots_per_s / 1e12
        out["frac_of_ffma_probe"] = rate * A / probe_slots_per_s
    if clocks and clocks.get("sm_mhz"):
        out["frac_at_observed_clock"] = rate * A / (sms * SM_LANES * clocks["sm_mhz"] * 1e6)
    return out


def quality_metrics(T, torch, cfg, g, f):
    """SRR of Eq. 10 against the clean phantom and the tumour CNR of PAPER.md:265 (kernels of the library), and the
    TV kernel against the HBM roofline (algorithmic bytes of one tnlm_tv_diff = 2 stacks x 4 B per voxel)."""
    from tnlm_inputs import make_stack
    star = torch.from_numpy(make_stack(cfg, clean=True)).to(g.device)
    p = T.TnlmParams.make(cfg.shape, cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)
    for _ in range(3):
        T.tnlm_tv_diff(p, g, star)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n = 10
    e0.record()
    for _ in range(n):                       # operands alternate: two stacks each, larger than L2 from config 3 on
        T.tnlm_tv_diff(p, g, star)
        T.tnlm_tv_diff(p, f, star)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / (2 * n)
    gbs = 2 * g.numel() * 4 / (ms * 1e-3) / 1e9
    srr = T.tnlm_srr(p, g, f, star).cpu().numpy()
    P, Z, Y, X = cfg.shape
    cz, cy, cx = (Z - 1) / 2, (Y - 1) / 2, (X - 1) / 2
    tz = int(round(cz - cfg.si_amplitude / 2 + cfg.si_amplitude)); ty = int(round(cy - 0.03 * Y)); tx = int(round(cx + 0.20 * X))
    r = max(2, int(cfg.tumour_radius) // 2)
    roi = (tz - r, tz + r + 1, ty - r, ty + r + 1, tx - r, tx + r + 1)            # inside the tumour at phase 0
    bg = (tz - r, tz + r + 1, ty + 3 * r + 2, ty + 5 * r + 3, tx - r, tx + r + 1)  # lung next to it
    c0 = T.tnlm_cnr(p, g, 0, roi, bg).cpu().numpy()
    c1 = T.tnlm_cnr(p, f, 0, roi, bg).cpu().numpy()
    peaks = measured_peaks()
    return {"tv_diff_ms": ms, "tv_diff_gbs": gbs, "hbm_peak_gbs": peaks["hbm_gbs"], "hbm_roofline_frac": gbs / peaks["hbm_gbs"],
            "srr_min": float(srr.min()), "srr_max": float(srr.max()), "cnr_input": float(c0[4]), "cnr_enhanced": float(c1[4]),
            "roi": roi, "roi_bg": bg}


def run_strong(args, cfg, T, D, info, dev, peaks):
    """ONE stack of `cfg` split into z-slabs over the ranks: a step is one
    TNLM-E run through dist.enhance_z_slabs_local with tnlm_jacobi_step_slab as the slab sweep.  Device-timed with
    CUDA events, max over ranks; value = the one stack's updates / that time."""
    import torch
    from tnlm_inputs import make_stack
    g_np = make_stack(cfg)                                     # every rank paints the same stack and keeps its slab
    p = T.TnlmParams.make(cfg.shape, cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)
    P, Z, Y, X = cfg.shape
    halo, zt = cfg.search_radius + cfg.patch_radius, T.z_tile(p)
    L = D.slab_layout(Z, info.rank, info.world, halo, zt)
    g_own = torch.from_numpy(g_np[:, L.a:L.b].copy()).to(dev)
    p_loc = T.TnlmParams.make((P, L.nz_local, Y, X), cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)
    ws = torch.empty(T.workspace_bytes(p_loc), dtype=torch.uint8, device=dev)
    launches = [0]

    def sweep_slab(f, g, z0, z1, out):
        if z1 > z0:
            T.tnlm_jacobi_step_slab(p_loc, f, g, z0, z1, f_out=out, ws=ws, variant=args.variant)
            launches[0] += 1

    def step():
        return D.enhance_z_slabs_local(info, g_own, cfg.n_iter, halo, zt, Z, sweep_slab)

    if args.loopback_world > 0:
        return run_loopback(args, cfg, T, D, dev, peaks, g_np)
    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        f, _ = step()
    torch.cuda.synchronize()
    if info.world == 1:                                         # the split form must reproduce tnlm_enhance bit for bit
        want = T.tnlm_enhance(p, torch.from_numpy(g_np).to(dev), cfg.n_iter)
        assert torch.equal(f.owned(), want), "z-slab form and tnlm_enhance disagree"
        del want
    sampler = ClockSampler(info.local_rank)
    if info.rank == 0:
        sampler.start()
    D.barrier(info)
    torch.cuda.synchronize()
    launches[0] = 0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    D.barrier(info)
    ms = D.max_over_ranks(info, e0.elapsed_time(e1), device=dev)
    clocks = sampler.stop() if info.rank == 0 else None
    halo_bytes = D.sum_over_ranks(info, D.halo_bytes_per_sweep(L, info, (P, Y, X)), device=dev)
    if info.rank == 0:
        updates = cfg.updates_per_sweep * cfg.n_iter
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        A = 5 + 6 * cfg.patch_radius
        value = args.steps * updates / (ms * 1e-3)
        conf = workload_config(cfg, info.world)
        conf["workload"] = conf["workload"].replace("+rank", "")
        conf["parallelism"] = (f"z{info.world}: one stack split into {info.world} z-slabs, each rank stores slab + {halo} halo planes "
                               f"(+ tile-alignment padding); per sweep the boundary planes go to the z-neighbours by send/recv on a "
                               f"side stream while the interior is computed")
        conf["updates_per_step_per_gpu"] = updates / info.world
        conf["halo_bytes_per_sweep_all_ranks"] = int(halo_bytes)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": info.world, "steps": args.steps, "warmup": warmup,
                "ms_per_step": ms / args.steps, "s_per_enhancement": ms * 1e-3 / args.steps, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": conf,
                "clocks": clocks, "e2e": None, "gpu_launches": launches[0],
                "roofline": {"bound": "alu", "kernel": kernel_label(T, p, args.variant),
                             "achieved": value * A / 1e12, "peak": info.world * sms * SM_LANES * peaks["sm_max_mhz"] * 1e6 / 1e12,
                             "unit": "Tslot/s over all ranks", "frac": value * A / (info.world * sms * SM_LANES * peaks["sm_max_mhz"] * 1e6),
                             "traffic": None},
                "cpu_baseline": None, "impl": "tnlm", "kernel": kernel_label(T, p, args.variant), "variant": args.variant}
        print(json.dumps(line), flush=True)
    D.finalize(info)
    return 0


def run_tnlmr(args, T, dev):
    """One TNLM-R outer iteration per step at the paper's phantom geometry (context for PAPER.md Table 2: 66.9 s per
    iteration on a Tesla C1060 with unknown d, M).  Not the north-star metric; reported beside it."""
    import numpy as np
    import torch
    from tnlm_inputs import projections as PJ
    P, n_cgls, d, M, h, mu = 10, 3, 1, 2, 0.05, 0.5
    geom = PJ.paper_geometry(128, 30, 512)
    ang, y, clean = PJ.make_projection_stack(geom, P, noise=0.02, seed=5)
    g = T.TnlmrGeometry.make(P, geom.vol_shape, geom.n_view, geom.nv, geom.nu, geom.voxel, geom.du, geom.dv, geom.sid, geom.sdd)
    p = T.TnlmParams.make((P,) + geom.vol_shape, d, M, h, mu)
    yd = torch.from_numpy(y).to(dev)
    f = torch.zeros((P,) + geom.vol_shape, dtype=torch.float32, device=dev)
    out = torch.empty_like(f)
    ws = torch.empty(T.tnlmr_workspace_bytes(g, p), dtype=torch.uint8, device=dev)
    proj = torch.empty_like(yd)
    for _ in range(2):
        T.tnlmr_reconstruct(g, p, ang, yd, f, 1, n_cgls, f_out=out, ws=ws)
    torch.cuda.synchronize()

    def timed(fn, n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    ms_iter = timed(lambda: T.tnlmr_reconstruct(g, p, ang, yd, f, 1, n_cgls, f_out=out, ws=ws), args.steps)
    ms_fp = timed(lambda: T.tnlmr_project(g, ang, f, y=proj), 3)
    ms_bp = timed(lambda: T.tnlmr_backproject(g, ang, yd, f=out), 3)
    ms_sweep = timed(lambda: T.tnlm_jacobi_step(p, f, f, f_out=out), 3)
    rec = T.tnlmr_reconstruct(g, p, ang, yd, f, 7, n_cgls, ws=ws)          # the paper ran 7 iterations
    cg = T.tnlmr_cgls(g, ang, yd, torch.zeros_like(f), 7 * n_cgls)
    cl = torch.from_numpy(clean).to(dev)
    err = lambda a: float(torch.linalg.vector_norm(a - cl) / torch.linalg.vector_norm(cl))
    rays = P * geom.n_view * geom.nv * geom.nu
    print(json.dumps({"workload": "TNLM-R, PAPER.md:245 geometry: 10 phases x 128^3 voxels (0.2 cm), 30 views per phase, 512x512 detector, "
                                  "analytic ellipsoid projections + noise, start f = 0, 3 CGLS iterations per outer iteration, 3^3 patch, 5^3 window",
                      "ms_per_outer_iteration": ms_iter, "paper_s_per_iteration_c1060": 66.91,
                      "ms_project_all_phases": ms_fp, "ms_backproject_all_phases": ms_bp, "ms_tnlm_sweep": ms_sweep,
                      "rays_per_projection": rays, "grays_per_s_project": rays / (ms_fp * 1e-3) / 1e9,
                      "rel_error_vs_phantom_after_7_iterations": err(rec), "rel_error_cgls_only_21_iterations": err(cg),
                      "kernel_launches_per_outer_iteration": 2 + 2 + n_cgls * 8 + 3}), flush=True)
    return 0


def run_loopback(args, cfg, T, D, dev, peaks, g_np):
    """Compute side of the strong-scaling curve on one GPU: for each rank of a W-rank z-slab split, the time of its
    sweeps (boundary + interior launches on its local arrays) with the halo planes filled from its own data instead of
    an exchange.  The slowest rank bounds the job; the exchange (halo bytes below) is not included."""
    import torch
    W = args.loopback_world
    P, Z, Y, X = cfg.shape
    p = T.TnlmParams.make(cfg.shape, cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)
    halo, zt = cfg.search_radius + cfg.patch_radius, T.z_tile(p)
    rows = []
    for rank in range(W):
        info = D.RankInfo(rank, 0, W)
        L = D.slab_layout(Z, rank, W, halo, zt)
        g_own = torch.from_numpy(g_np[:, L.a:L.b].copy()).to(dev)
        p_loc = T.TnlmParams.make((P, L.nz_local, Y, X), cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)
        ws = torch.empty(T.workspace_bytes(p_loc), dtype=torch.uint8, device=dev)

        def sweep_slab(f, g, z0, z1, out):
            if z1 > z0:
                T.tnlm_jacobi_step_slab(p_loc, f, g, z0, z1, f_out=out, ws=ws, variant=args.variant)

        def local_fill(_info, stack, L_):
            stack[:, L_.lo - L_.halo:L_.lo] = stack[:, L_.lo:L_.lo + 1]
            stack[:, L_.hi:L_.hi + L_.halo] = stack[:, L_.hi - 1:L_.hi]

        for _ in range(2):
            D.enhance_z_slabs_local(info, g_own, cfg.n_iter, halo, zt, Z, sweep_slab, exchange=local_fill)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            D.enhance_z_slabs_local(info, g_own, cfg.n_iter, halo, zt, Z, sweep_slab, exchange=local_fill)
        e1.record()
        torch.cuda.synchronize()
        rows.append({"rank": rank, "planes": L.b - L.a, "local_planes": L.nz_local, "ms_per_enhancement": e0.elapsed_time(e1) / args.steps,
                     "halo_bytes_sent_per_sweep": D.halo_bytes_per_sweep(L, info, (P, Y, X))})
    slow = max(r["ms_per_enhancement"] for r in rows)
    print(json.dumps({"loopback_world": W, "config": cfg.name, "kernel": kernel_label(T, p, args.variant),
                      "slowest_rank_ms_per_enhancement": slow,
                      "projected_updates_per_s_excluding_exchange": cfg.updates_per_sweep * cfg.n_iter / (slow * 1e-3),
                      "ranks": rows, "note": "one GPU, ranks timed one after the other, halo planes filled locally"}), flush=True)
    return 0


def main():
    args = parse_args()
    from tnlm_inputs import CONFIGS, make_stack
    cfg = CONFIGS[args.config]
    sweep_mode = args.config == "config5"
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
    warmup = max(args.warmup, 3)
    if args.tnlmr:
        rc = run_tnlmr(args, T, dev)
        D.finalize(info)
        return rc
    if args.scaling == "strong":
        if sweep_mode or args.ref != "same":
            raise SystemExit("--scaling strong covers config1..config4 with ref = f")
        return run_strong(args, cfg, T, D, info, dev, peaks)

    # one independent, differently seeded stack per rank (weak scaling)
    rcfg = cfg.scaled(seed=cfg.seed + info.rank)
    g_host_np = make_stack(rcfg)
    g = torch.from_numpy(g_host_np).to(dev)
    f_out = torch.empty_like(g)
    stream = torch.cuda.current_stream()
    # the points of a step: (config with its d, M; params; workspace)
    point_cfgs = [cfg.scaled(patch_radius=d, search_radius=M) for d in (1, 2) for M in (1, 2, 3, 4)] if sweep_mode else [cfg]
    points = []
    for c in point_cfgs:
        p = T.TnlmParams.make(c.shape, c.patch_radius, c.search_radius, c.h, c.mu)
        points.append((c, p))
    ws = torch.empty(max(T.workspace_bytes(p) for _, p in points), dtype=torch.uint8, device=dev)
    updates_per_step = sum(c.updates_per_sweep * c.n_iter for c, _ in points)
    launches_per_step = sum(c.n_iter * T.launches_per_sweep(p) for c, p in points)
    stack_mb = g.numel() * 4 / 1e6
    flush = torch.empty(64 * 1024 * 1024, dtype=torch.float32, device=dev) if 3 * stack_mb <= 126 else None

    sep = args.ref == "separate"
    if sep:   # weights from a lightly smoothed copy of the stack, as an outer TNLM-R iteration would pass
        ref_stack = (0.5 * g + 0.25 * torch.roll(g, 1, 3) + 0.25 * torch.roll(g, -1, 3)).contiguous()
        f_tmp = torch.empty_like(g)
        args.no_e2e = True

    def step(record=None):
        for k, (c, p) in enumerate(points):
            if record is not None:
                record[k][0].record(stream)
            if sep:
                src, dst = g, (f_out if c.n_iter % 2 == 1 else f_tmp)
                for _ in range(c.n_iter):
                    T.tnlm_jacobi_step(p, src, g, ref=ref_stack, f_out=dst, ws=ws, stream=stream, variant=args.variant)
                    src, dst = dst, (f_tmp if dst is f_out else f_out)
            else:
                T.tnlm_enhance(p, g, c.n_iter, f_out=f_out, ws=ws, stream=stream, variant=args.variant)
            if record is not None:
                record[k][1].record(stream)
        if flush is not None:
            flush.zero_()                               # small stacks: evict them from L2 between steps

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()

    # ---- device-timed region -------------------------------------------------------------
    sampler = ClockSampler(info.local_rank)
    if info.rank == 0:
        sampler.start()
    D.barrier(info)
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    per_point = [[[torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)] for _ in points]
                 for _ in range(args.steps)]
    ev0.record(stream)
    for s_i in range(args.steps):
        step(per_point[s_i])
    ev1.record(stream)
    torch.cuda.synchronize()
    D.barrier(info)
    elapsed_ms = D.max_over_ranks(info, ev0.elapsed_time(ev1), device=dev)
    clocks = sampler.stop() if info.rank == 0 else None
    value = info.world * args.steps * updates_per_step / (elapsed_ms * 1e-3)
    # time inside the enhancement calls only (excludes the L2 flush of small configs), per point
    point_ms = [sum(per_point[s_i][k][0].elapsed_time(per_point[s_i][k][1]) for s_i in range(args.steps)) / args.steps
                for k in range(len(points))]
    if flush is not None:
        value = info.world * updates_per_step / (D.max_over_ranks(info, sum(point_ms), device=dev) * 1e-3)

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

    # ---- end-to-end through tnlm_enhance_host (pinned host buffers), the same number of steps --------
    e2e = None
    if not args.no_e2e:
        g_pin = torch.from_numpy(g_host_np).pin_memory()
        out_pin = torch.empty(cfg.shape, dtype=torch.float32).pin_memory()
        dev_ws = torch.empty(max(T.host_workspace_bytes(p) for _, p in points), dtype=torch.uint8, device=dev)

        def e2e_step():
            for c, p in points:
                T.tnlm_enhance_host(p, g_pin, c.n_iter, f_out_host=out_pin, dev_ws=dev_ws, stream=stream)

        e2e_step()                                      # warm
        D.barrier(info)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            e2e_step()
        torch.cuda.synchronize()
        dt = D.max_over_ranks(info, time.perf_counter() - t0, device=dev)
        if args.variant == 0:
            assert torch.equal(out_pin, f_out.cpu()), "host path and device path disagree"
        e2e = {"value": info.world * args.steps * updates_per_step / dt, "unit": UNIT,
               "h2d_bytes_per_step": g_pin.numel() * 4 * len(points), "d2h_bytes_per_step": out_pin.numel() * 4 * len(points),
               "ms_per_step": 1e3 * dt / args.steps, "steps": args.steps,
               "api": "tnlm_enhance_host (C ABI, pinned host buffers, copies + sync inside the timed region)"}
        del dev_ws

    quality = None
    if args.metrics and info.rank == 0:
        c, p = points[0] if not sweep_mode else points[1]
        f_enh = T.tnlm_enhance(p, g, c.n_iter, ws=ws, stream=stream)
        quality = quality_metrics(T, torch, c.scaled(seed=rcfg.seed), g, f_enh)

    if info.rank != 0:
        D.finalize(info)
        return 0

    # ---- roofline of the dominant (sweep) kernel ------------------------------------------
    props = torch.cuda.get_device_properties(dev)
    sms = props.multi_processor_count
    point_lines = []
    for (c, p), ms in zip(points, point_ms):
        launch_ms = ms / c.n_iter                      # CUDA events around the enhancement / its sweeps
        rl = roofline_block(T, p, c, args.variant, launch_ms, sms, peaks, clocks, probe_slots_per_s, g.numel())
        point_lines.append({"patch": 2 * c.patch_radius + 1, "window": 2 * c.search_radius + 1, "n_iter": c.n_iter,
                            "updates_per_s": c.updates_per_sweep * c.n_iter / (ms * 1e-3), "s_per_enhancement": ms * 1e-3,
                            "ms_per_sweep": launch_ms, "roofline": rl})
    # the headline roofline block: the single point, or (sweep) the point that takes the largest share of the step
    top = max(range(len(points)), key=lambda k: point_ms[k])
    roofline = point_lines[top]["roofline"]
    if sweep_mode:
        roofline = dict(roofline, note=f"dominant point of the sweep (patch {point_lines[top]['patch']}^3, window "
                                       f"{point_lines[top]['window']}^3, {100 * point_ms[top] / sum(point_ms):.0f} % of the step); "
                                       f"every point's block is in 'points'")

    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline = oracle_sample_rate(points[top][0], g_host_np, args.cpu_seconds)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": info.world, "steps": args.steps,
        "warmup": warmup, "ms_per_step": elapsed_ms / args.steps,
        "s_per_enhancement": sum(point_ms) * 1e-3 / len(points), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(cfg, info.world, sweep_mode), "clocks": clocks, "e2e": e2e,
        "gpu_launches": args.steps * launches_per_step, "roofline": roofline, "cpu_baseline": cpu_baseline,
        "impl": "tnlm", "kernel": roofline["kernel"], "variant": args.variant, "ref": args.ref,
    }
    if sep:
        line["config"]["workload"] += "; weights of every sweep from a SEPARATE stack (tnlm_jacobi_step(ref=...))"
        line["kernel"] = roofline["kernel"] = roofline["kernel"] + " (separate ref: candidate tile)"
        roofline["traffic"] = None
    if sweep_mode:
        line["points"] = point_lines
    if quality:
        line["quality"] = quality
    print(json.dumps(line), flush=True)
    D.finalize(info)
    return 0


if __name__ == "__main__":
    sys.exit(main())
