"""Parameter sweep of BASELINE.json configs[4] ("config5"): patch in {3^3, 5^3} x window in {3^3, 5^3, 7^3, 9^3}
on the 20-phase 256 x 256 x 128 thorax phantom (seed 4), h = 0.05, mu = 0.5, n_iter sweeps each.

    python -m paper_1201_2450_b200.sweep [--iters 5] [--config config5] [--nz 128]

Prints one JSON line per (patch, window) point: voxel-offset updates/s (CUDA events around tnlm_enhance),
seconds per enhancement, ms per sweep and the fraction of the FP32-pipe roofline
(A = 5 + 6d lane-operations per update, peak = SMs x 128 lanes x clocks.max.sm).
Argument marshalling only: every step runs in libtnlm.so's kernels on the current CUDA device.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="config5")
    ap.add_argument("--iters", type=int, default=None, help="Gauss-Jacobi sweeps per point (default: the config's)")
    ap.add_argument("--nz", type=int, default=None, help="override the number of planes (smaller = quicker)")
    ap.add_argument("--sm-mhz", type=float, default=1965.0)
    ap.add_argument("--metrics", action="store_true", help="time the TV/SRR/CNR kernels on the config instead (HBM roofline)")
    ap.add_argument("--hbm-gbs", type=float, default=6457.4, help="measured HBM copy bandwidth (MEASURED_PEAKS.json)")
    args = ap.parse_args()

    import torch
    import paper_1201_2450_b200 as T
    from tnlm_inputs import CONFIGS, make_stack

    if not torch.cuda.is_available():
        raise SystemExit("the sweep needs a CUDA device: the TNLM path has no CPU fallback")
    cfg = CONFIGS[args.config]
    if args.nz:
        cfg = cfg.scaled(nz=args.nz)
    n_iter = args.iters or cfg.n_iter
    g = torch.from_numpy(make_stack(cfg)).cuda()
    out = torch.empty_like(g)
    if args.metrics:
        return metrics(args, cfg, g, T, torch, make_stack)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    peak = sms * 128 * args.sm_mhz * 1e6
    stream = torch.cuda.current_stream()
    for d in (1, 2):
        for M in (1, 2, 3, 4):
            p = T.TnlmParams.make(cfg.shape, d, M, cfg.h, cfg.mu)
            ws = torch.empty(T.workspace_bytes(p), dtype=torch.uint8, device=g.device)
            T.tnlm_enhance(p, g, 1, f_out=out, ws=ws, stream=stream)          # warm-up
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            T.tnlm_enhance(p, g, n_iter, f_out=out, ws=ws, stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            sec = e0.elapsed_time(e1) * 1e-3
            updates = 2 * g.numel() * (2 * M + 1) ** 3 * n_iter
            print(json.dumps({"config": cfg.name, "shape": list(cfg.shape), "patch": 2 * d + 1, "window": 2 * M + 1,
                              "n_iter": n_iter, "kernel": T.kernel_name(p), "updates_per_s": updates / sec,
                              "s_per_enhancement": sec, "ms_per_sweep": 1e3 * sec / n_iter,
                              "roofline_frac": updates / sec * (5 + 6 * d) / peak, "finite": bool(torch.isfinite(out).all())}),
                  flush=True)
            del ws


def metrics(args, cfg, g, T, torch, make_stack):
    """SRR (Eq. 10) and tumour CNR before/after enhancement, and the TV kernel against the HBM roofline:
    algorithmic bytes of one tnlm_tv_diff = 2 stacks x 4 B per voxel (every operand voxel read once)."""
    star = torch.from_numpy(make_stack(cfg, clean=True)).cuda()
    p = T.TnlmParams.make(cfg.shape, cfg.patch_radius, cfg.search_radius, cfg.h, cfg.mu)
    f = T.tnlm_enhance(p, g, args.iters or cfg.n_iter)
    for _ in range(3):
        T.tnlm_tv_diff(p, g, star)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n = 10
    e0.record()
    for _ in range(n):                       # operands alternate, 2 x 335 MB each: larger than L2
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
    print(json.dumps({"config": cfg.name, "shape": list(cfg.shape), "tv_diff_ms": ms, "tv_diff_gbs": gbs,
                      "hbm_peak_gbs": args.hbm_gbs, "hbm_roofline_frac": gbs / args.hbm_gbs,
                      "srr_per_phase": [float(v) for v in srr], "cnr_input": float(c0[4]), "cnr_enhanced": float(c1[4]),
                      "roi": roi, "roi_bg": bg}), flush=True)


if __name__ == "__main__":
    main()
