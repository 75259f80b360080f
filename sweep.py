"""BASELINE.json config 5: bandwidth sweep of the per-iteration kernels through the C ABI.

    python sweep.py [--sizes 128x128x64,256x256x100,...] [--reps 20] [--batch B]
                    [--kernels force,iteration,smooth,pyramid,texture] [--json out.json]

For every size: the fused warp+force+update entry point for all six variants, the Gaussian
smoothing at sigma 1.0 and 2.0 (3 components), restrict and prolong.  Inputs are the seeded blob
phantom and a random smooth field with max |u| = 8 voxels (phantoms.sweep_inputs).  `iteration[...]` rows time one
whole [force ; smooth] iteration inside a registration (40 iterations, one level, sigma 1); with --batch B > 1 the
passive and double-force iteration rows are repeated through demons_register_batch with B pairs per call (time per
pair: what the batch axis does for sizes whose launches cannot fill 148 SMs).  Reported per
kernel: median over `reps` samples of 10 back-to-back launches (CUDA events) after 3 warm-ups, effective GB/s = algorithmic
bytes (DESIGN.md byte table) / time, and % of the measured HBM peak.  The same command with
--reps 1 --warmups 1 --inner 1 (every entry point launched twice) is what the ncu captures under profiles/ run.  S and M are separate allocations here, so the L2
access-policy window of the gathering kernels covers M alone (bench.py's pair shares one allocation and
gets both images).  The CPU oracle's time per call for the same entry points is measured by bench.py's
cpu_baseline leg (this script never loads the oracle).  A measurement script, like bench.py: it sits beside it, not
in the library package.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
SEEDS = {(128, 128, 64): 500, (256, 256, 100): 501, (512, 512, 160): 502, (512, 512, 256): 503}
# algorithmic bytes per voxel of each entry point as implemented
# variant 1 through the standalone entry point: |grad M|^2 pass (4 in, 4 out) + fused pass (u 12, S 4, M 4,
# |grad M|^2 4 in, 12 out); inside a registration the first pass runs once per level, not per iteration
FORCE_BYTES = {0: 32.0, 1: 44.0, 2: 52.0, 3: 52.0, 4: 52.0, 5: 96.0}
VARIANT_NAMES = ["passive", "evolved_passive", "active", "double", "adjusted_double", "inverse_consistent"]


def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"


WARMUPS, INNER, PAUSE_S = 3, 10, 0.3


def median_ms(torch, stream, fn, reps, inner=None):
    """Median over `reps` samples of (CUDA-event time of `inner` back-to-back launches) / inner: the
    queue stays full, so the host's launch latency is not in the number."""
    inner = INNER if inner is None else inner
    time.sleep(PAUSE_S)  # every row starts from the same power state (a long sweep runs into the board's power cap)
    for _ in range(WARMUPS):
        fn()
    torch.cuda.synchronize()
    times = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(inner):
            fn()
        e1.record(stream)
        e1.synchronize()
        times.append(e0.elapsed_time(e1) / inner)
    return float(np.median(times))


def run(sizes, kernels, reps, device="cuda:0", batch=1):
    import torch
    from paper_0909_0928_b200 import binding as B
    from paper_0909_0928_b200 import build, phantoms
    build.build()
    B.lib()
    peak, peak_kind = hbm_peak()
    stream = torch.cuda.Stream(device=device)
    rows = []
    for dims in sizes:
        N = dims[0] * dims[1] * dims[2]
        S, M, u = phantoms.sweep_inputs(dims, SEEDS.get(tuple(dims), 599))
        dS, dM, du = (torch.from_numpy(a).to(device) for a in (S, M, u))
        dub = (-du).contiguous()
        out, outb = torch.empty_like(du), torch.empty_like(du)
        met = torch.zeros(3, dtype=torch.float64, device=device)

        def add(name, ms, nbytes):
            gbs = nbytes / (ms * 1e-3) / 1e9
            rows.append({"dims": "x".join(map(str, dims)), "kernel": name, "ms": ms, "alg_bytes": nbytes,
                         "gbs": gbs, "pct_of_peak": 100.0 * gbs / peak, "pct_of_nominal_8TBs": 100.0 * gbs / 8000.0})

        if "force" in kernels:
            for variant in range(6):
                eng = B.Demons(dims, variant=variant, alpha=0.4 if variant == 4 else 1.0, device=device)
                ic = variant == 5
                ms = median_ms(torch, stream, lambda: B.demons_warp_force(
                    eng.ctx, dims, dS, dM, du, out, dub if ic else None, outb if ic else None, met, stream), reps)
                add(f"warp_force[{VARIANT_NAMES[variant]}]", ms, FORCE_BYTES[variant] * N)
                eng.close()
        if "texture" in kernels:
            # S9: hardware linear filtering (9-bit weights) against the software trilinear of the same pass
            eng = B.Demons(dims, variant=0, device=device)
            B.demons_warp_force(eng.ctx, dims, dS, dM, du, out, None, None, met, stream)
            torch.cuda.synchronize()
            soft = out.clone()
            B.demons_set_option(eng.ctx, "texture", 1)
            ms = median_ms(torch, stream, lambda: B.demons_warp_force(
                eng.ctx, dims, dS, dM, du, out, None, None, met, stream), reps)
            torch.cuda.synchronize()
            err = (out - soft).abs()
            add("warp_force[passive, texture unit]", ms, FORCE_BYTES[0] * N)
            rows[-1]["max_abs_err_vs_software_voxel"] = float(err.max())
            rows[-1]["mean_abs_err_vs_software_voxel"] = float(err.mean())
            rows[-1]["frac_outside_1e-4"] = float((err > 1e-4).float().mean())
            eng.close()
        eng = B.Demons(dims, variant=0, device=device)
        if "smooth" in kernels:
            for sigma in (1.0, 2.0):
                ms = median_ms(torch, stream, lambda: B.demons_smooth(eng.ctx, dims, du, out, 3, sigma, stream), reps)
                add(f"smooth[sigma={sigma}]", ms, 24.0 * N)
        if "pyramid" in kernels:
            cd = B.demons_level_dims(eng.ctx, 1)
            coarse = torch.empty((cd[2], cd[1], cd[0]), dtype=torch.float32, device=device)
            uc = torch.randn((3, cd[2], cd[1], cd[0]), dtype=torch.float32, device=device)
            ms = median_ms(torch, stream, lambda: B.demons_restrict(eng.ctx, dims, dS, coarse, stream), reps)
            add("restrict", ms, 4.5 * N)
            ms = median_ms(torch, stream, lambda: B.demons_prolong(eng.ctx, cd, uc, dims, out, stream), reps)
            add("prolong", ms, 13.5 * N)
        eng.close()
        if "iteration" in kernels:
            # one whole iteration INSIDE a registration ([force ; smooth], sigma 1, per-level CUDA graph): what the
            # standalone rows cannot show -- there the metric totals are finalised by the force kernel's last block (a
            # fence, a ticket and a serial sum at the tail of the kernel), here by k_metrics_final beside the smoother
            its = 40
            for variant in range(6):
                eng = B.Demons(dims, variant=variant, alpha=0.4 if variant == 4 else 1.0, sigma=1.0, device=device)
                ic = variant == 5
                out.copy_(du)  # the registrations continue from the sweep's field (max |u| = 8), one after another
                if ic:
                    outb.copy_(dub)
                torch.cuda.synchronize()
                ms = median_ms(torch, stream, lambda: B.demons_register(
                    eng.ctx, dS, dM, out, outb if ic else None, [its], 0.0, None, None, stream), max(3, reps // 4), inner=1) / its
                # force bytes inside a registration: variant 1 without the per-level |grad M|^2 pass; variant 5 starts
                # from the caller's fields here, i.e. the two-field form (96 B/voxel, both fields smoothed: 48)
                fb = {0: 32.0, 1: 36.0, 2: 52.0, 3: 52.0, 4: 52.0, 5: 96.0}[variant]
                add(f"iteration[{VARIANT_NAMES[variant]}]", ms, (fb + (48.0 if ic else 24.0)) * N)
                eng.close()
            if batch > 1 and batch * N < (1 << 29):
                # the same iteration with `batch` pairs per call (demons_register_batch): ms per pair and iteration
                bS = torch.stack([torch.roll(dS, k, dims=2) for k in range(batch)]).contiguous()
                bM = torch.stack([torch.roll(dM, k, dims=2) for k in range(batch)]).contiguous()
                bu0 = torch.stack([torch.roll(du, k, dims=3) for k in range(batch)]).contiguous()
                bu = torch.empty_like(bu0)
                for variant in (0, 3):
                    eng = B.Demons(dims, variant=variant, sigma=1.0, device=device, nbatch=batch)
                    bu.copy_(bu0)
                    torch.cuda.synchronize()
                    ms = median_ms(torch, stream, lambda: B.demons_register_batch(
                        eng.ctx, batch, bS, bM, bu, None, [its], 0.0, None, None, stream), max(3, reps // 4), inner=1) / (its * batch)
                    fb = {0: 32.0, 3: 52.0}[variant]
                    add(f"iteration[{VARIANT_NAMES[variant]}, B={batch}]", ms, (fb + 24.0) * N)
                    eng.close()
                del bS, bM, bu0, bu
    return rows, peak, peak_kind


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--sizes", default="128x128x64,256x256x100,512x512x160,512x512x256")
    ap.add_argument("--kernels", default="force,iteration,smooth,pyramid,texture")
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--json", default=None)
    ap.add_argument("--batch", type=int, default=1, help="also time the iteration rows with this many pairs per call")
    ap.add_argument("--warmups", type=int, default=3)
    ap.add_argument("--inner", type=int, default=10, help="back-to-back launches per timed sample")
    args = ap.parse_args()
    global WARMUPS, INNER
    WARMUPS, INNER = args.warmups, args.inner
    sizes = [tuple(int(v) for v in s.split("x")) for s in args.sizes.split(",")]
    rows, peak, kind = run(sizes, set(args.kernels.split(",")), args.reps, batch=args.batch)
    print(f"# HBM peak {peak:.1f} GB/s ({kind}); effective GB/s = algorithmic bytes / median time")
    print(f"{'dims':>12} {'kernel':<34} {'ms':>9} {'GB/s':>9} {'% peak':>7} {'% 8TB/s':>8}")
    for r in rows:
        extra = ""
        if "max_abs_err_vs_software_voxel" in r:
            extra = (f"  |u'(tex) - u'(software)|: max {r['max_abs_err_vs_software_voxel']:.3e} mean "
                     f"{r['mean_abs_err_vs_software_voxel']:.3e} voxel, {100 * r['frac_outside_1e-4']:.1f}% outside 1e-4")
        print(f"{r['dims']:>12} {r['kernel']:<34} {r['ms']:9.4f} {r['gbs']:9.1f} {r['pct_of_peak']:7.1f} "
              f"{r['pct_of_nominal_8TBs']:8.1f}{extra}")
    if args.json:
        with open(args.json, "w") as fh:
            json.dump({"peak_gbs": peak, "peak_kind": kind, "rows": rows}, fh, indent=1)


if __name__ == "__main__":
    main()
