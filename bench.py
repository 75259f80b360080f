"""Benchmark of the demons hot path on B200 (contract: one JSON line on stdout from rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one full registration of BASELINE.json config 2: the 256x256x100 lung-CT-shaped
phantom pair, passive-force demons (Eq.(1)), single scale, 300 iterations, sigma = 1 -- every
iteration runs the fused warp+gradient+force+update kernel (with the SSD / relative-norm
reduction) and the Gaussian smoothing of the field.  `value` is Gvoxel-iterations/s with the
inputs resident in HBM; `e2e` is the same through demons_register_host with pinned HOST buffers.
The multi-level variants of configs 3-4 (restrict / prolong included) are timed after the main
region and reported under "variants" (with the 3D error at 1,000 seeded points against the known
field, the final SSD and, for config 4, the inverse-consistency error); "batch" times
demons_register_batch on config 3 (B = 1, 4, 16 pairs per call); "evaluation" holds the accuracy
protocol for the timed config-2 registration.

"roofline" is per kernel, and the kernel durations are MEASURED IN THIS RUN from inside the replayed graph: with the
library's "profile" = 2 option one iteration in the middle of every 20-iteration graph chunk carries CUDA event-record
nodes (before the force kernel, between force and smoother, after the smoother); `avg_ms` is their mean over three
registrations (45 replays).  `frac` depends on nothing under profiles/.  Beside it, as cross-checks only: the share of
the iteration from the event-bracketed no-graph pass ("share_events_no_graph"), the committed ncu share
("share_ncu_committed") and "stale_share" = true when the committed share is more than 0.05 away from this run's.
"achieved" = ALGORITHMIC bytes / that duration (an effective bandwidth: each array element once);
"hbm_measured" = the DRAM bytes ncu counted for that kernel (profiles/r0N_ncu_traffic.csv) / the same
duration -- real HBM traffic, lower, because part of the field is still in L2 between the two kernels.
Both are given as fractions of the measured copy peak (MEASURED_PEAKS.json) and of the nominal 8 TB/s.

S and M live in one device allocation so that the library's L2 access-policy window keeps both resident.
N > 1: N independent replicas, one process per GPU (launched here when not already under torchrun).
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

DIMS = (256, 256, 100)
SPACING = (0.97, 0.97, 2.5)
ITERS = [300]
SIGMA = 1.0
METRIC = "demons Gvoxel-iter/s (passive force, 256x256x100, 300 iterations, sigma 1; ms_per_step = ms per registration)"
UNIT = "Gvoxel-iter/s"
FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0   # BASELINE.json north_star: "the B200's ~8 TB/s peak"


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return FALLBACK_HBM_GBS, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


def committed_csv(name):
    """kernel class -> value from a two-column csv under profiles/ (written from the committed ncu captures;
    the commands that made them are in the .md files beside them)."""
    out = {}
    try:
        with open(os.path.join(ROOT, "profiles", name)) as fh:
            for line in fh:
                parts = line.strip().split(",")
                if len(parts) == 2 and parts[0] != "kernel":
                    out[parts[0]] = float(parts[1])
    except Exception:
        pass
    return out


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons while the timed region runs (NVML)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._halt = threading.Event()

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake_slowdown",
                nv.nvmlClocksThrottleReasonApplicationsClocksSetting: "applications_clocks_setting",
            }
            while not self._halt.is_set():
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
                time.sleep(0.02)
        except Exception as e:  # no NVML: report that, do not fail the bench
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def stop(self):
        self._halt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def oracle_sample(S, M, iters):
    """The oracle as it stands on the host cores: `iters` iterations of the same workload."""
    from oracle import oracle as O
    O.build()
    t0 = time.perf_counter()
    O.register(0, 1.0, SIGMA, S, M, [iters])
    return time.perf_counter() - t0


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the workload."""
    from paper_0909_0928_b200 import phantoms, replicas
    rank, _, world = replicas.env_world()
    if rank != 0:
        return
    S, M, _ = phantoms.lung_pair(DIMS, 202)
    sample_iters = 2
    N = DIMS[0] * DIMS[1] * DIMS[2]
    for _ in range(args.warmup):
        oracle_sample(S, M, 1)
    t = 0.0
    for _ in range(args.steps):
        t += oracle_sample(S, M, sample_iters)
    value = args.steps * sample_iters * N / t / 1e9
    cores = 1
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config2: lung phantom 256x256x100, passive, single scale, sigma 1",
                   "sample": f"each step = {sample_iters} of the 300 iterations on the full volume pair"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{args.steps} x {sample_iters} iterations of the 300, full 256x256x100 pair "
                                   f"(single thread; the host offers {os.cpu_count()} cores)"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def device_pair(torch, S, M, device):
    """S and M in ONE device allocation, M right behind S: the library's L2 access-policy window
    (demons.h, option "l2_persist") then keeps both images resident instead of M alone."""
    both = torch.empty((2,) + S.shape, dtype=torch.float32, device=device)
    both[0].copy_(torch.from_numpy(S))
    both[1].copy_(torch.from_numpy(M))
    return both[0], both[1]


def time_registrations(torch, B, eng, dS, dM, du, dub, iters, steps, warmup, stream, replicas):
    """W untimed + K timed registrations; events on the launching stream; returns seconds."""
    def one():
        with torch.cuda.stream(stream):
            du.zero_()
            if dub is not None:
                dub.zero_()
        B.demons_register(eng.ctx, dS, dM, du, dub, iters, 0.0, None, None, stream)

    for _ in range(warmup):
        one()
    torch.cuda.synchronize()
    replicas.barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = B.demons_launch_count(eng.ctx)
    ev0.record(stream)
    for _ in range(steps):
        one()
    ev1.record(stream)
    torch.cuda.synchronize()
    replicas.barrier()
    return ev0.elapsed_time(ev1) * 1e-3, B.demons_launch_count(eng.ctx) - l0


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start the N ranks here
    (one process per GPU, rendezvous on 127.0.0.1) and pass their output through."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")          # the communicator lines (comm ... nranks N) print at INFO only
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    return subprocess.call(cmd, env=env)


def stub_main(args):
    """--stub: the N > 1 plumbing (rank discovery, barrier, max-over-ranks timing, one JSON line from rank 0)
    on CPU with the gloo backend and a sleep in place of the GPU step; tests/test_replicas.py runs it."""
    from paper_0909_0928_b200 import replicas
    rank, _, world = replicas.env_world()
    replicas.init("gloo")
    replicas.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time.sleep(0.01 * (rank + 1))
    secs = time.perf_counter() - t0
    replicas.barrier()
    agg = replicas.aggregate(float(args.steps), secs)
    ranks = int(round(replicas.sum_over_ranks(1.0)))
    if rank == 0:
        print(json.dumps({"metric": "stub steps/s", "value": agg["value"], "unit": "steps/s", "n_gpus": ranks,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * agg["seconds"] / args.steps,
                          "scaling": "weak", "stub": True, "units": agg["units"]}), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def time_oracle(fn, min_reps=1):
    t0 = time.perf_counter()
    for _ in range(min_reps):
        fn()
    return (time.perf_counter() - t0) / min_reps


def cpu_baseline_details(S, M):
    """the oracle, as it stands, one host thread: config 1 whole; configs 3 and 4 as one
    sampled iteration per level x the iteration counts (labelled sampled); config 5 ms per call per kernel at
    128x128x64 and 256x256x100.  About half a minute of CPU."""
    from oracle import oracle as O
    from paper_0909_0928_b200 import phantoms
    O.build()
    out = {}
    S1, M1, _ = phantoms.config1_pair()
    t = time_oracle(lambda: O.register(0, 1.0, 1.0, S1, M1, [50]))
    out["config1_passive_64x64x32_50it"] = {"s_per_registration": t, "gvoxel_iter_per_s": 50 * S1.size / t / 1e9, "sampled": False}
    # configs 3 / 4: one iteration on each level, scaled by the 100 iterations per level
    S4, M4, _ = phantoms.lung_pair((256, 256, 110), 404)
    for name, variant, alpha, Sx, Mx in (("config3_active", 2, 1.0, S, M), ("config3_double", 3, 1.0, S, M),
                                         ("config3_adjusted_a0.4", 4, 0.4, S, M),
                                         ("config4_inverse_consistent", 5, 1.0, S4, M4)):
        Sl, Ml, total, vox = Sx, Mx, 0.0, 0
        for _ in range(3):
            u0 = np.zeros((3,) + Sl.shape, np.float32)
            total += 100 * time_oracle(lambda: O.register(variant, alpha, 1.0, Sl, Ml, [1], u0=u0,
                                                          ub0=u0 if variant == 5 else None))
            vox += 100 * Sl.size
            Sl, Ml = O.restrict(Sl), O.restrict(Ml)
        out[name] = {"s_per_registration": total, "gvoxel_iter_per_s": vox / total / 1e9, "sampled": True,
                     "sample": "1 iteration per level x 100"}
    # config 5: per-kernel ms per call
    per_kernel = {}
    for dims, seed in (((128, 128, 64), 500), ((256, 256, 100), 501)):
        Sb, Mb, ub = phantoms.sweep_inputs(dims, seed)
        key = "x".join(map(str, dims))
        row = {}
        for variant, nm in enumerate(["passive", "evolved_passive", "active", "double", "adjusted_double", "inverse_consistent"]):
            row[f"warp_force[{nm}]"] = 1e3 * time_oracle(lambda: O.warp_force(variant, 0.4 if variant == 4 else 1.0, Sb, Mb, ub,
                                                                              -ub if variant == 5 else None))
        for sigma in (1.0, 2.0):
            row[f"smooth[sigma={sigma}]"] = 1e3 * time_oracle(lambda: O.smooth(ub, sigma))
        row["restrict"] = 1e3 * time_oracle(lambda: O.restrict(Sb))
        uc = np.zeros((3,) + O.coarse_shape(Sb.shape), np.float32)
        row["prolong"] = 1e3 * time_oracle(lambda: O.prolong(uc, Sb.shape))
        per_kernel[key] = row
    out["config5_ms_per_call"] = per_kernel
    return out


def texture_error_vs_oracle(torch, B, device, stream):
    """S9: the texture-unit option's precision loss against the ORACLE at 128x128x64 (config-5
    inputs), with the software path beside it.  Reported, never gated."""
    from oracle import oracle as O
    from paper_0909_0928_b200 import phantoms
    dims = (128, 128, 64)
    S, M, u = phantoms.sweep_inputs(dims, 500)
    ref = torch.from_numpy(O.warp_force(0, 1.0, S, M, u, None)[0]).to(device)
    dS, dM, du = (torch.from_numpy(a).to(device) for a in (S, M, u))
    out = torch.empty_like(du)
    eng = B.Demons(dims, variant=0, device=device)
    res = {}
    torch.cuda.synchronize()
    for name, opt in (("software_trilinear", 0), ("texture_unit", 1)):
        B.demons_set_option(eng.ctx, "texture", opt)
        B.demons_warp_force(eng.ctx, dims, dS, dM, du, out, None, None, None, stream)
        torch.cuda.synchronize()
        e = (out - ref).abs()
        res[name] = {"max_abs_err_voxel": float(e.max()), "mean_abs_err_voxel": float(e.mean()),
                     "frac_outside_1e-4+1e-5|ref|": float((e > 1e-4 + 1e-5 * ref.abs()).float().mean())}
    eng.close()
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the per-variant, batch and cpu_baseline legs")
    ap.add_argument("--stub", action="store_true", help="CPU stand-in for the GPU step (tests of the N > 1 plumbing)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        sys.exit(relaunch_under_torchrun(args))
    if args.stub:
        stub_main(args)
        return
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    from paper_0909_0928_b200 import binding as B
    from paper_0909_0928_b200 import build, phantoms, replicas

    build.build()
    B.lib()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    rank, local_rank, world = replicas.env_world()
    assert world == args.gpus, f"--gpus {args.gpus} but {world} rank(s) are running"
    torch.cuda.set_device(local_rank)
    device = f"cuda:{local_rank}"
    replicas.init("nccl")
    N = DIMS[0] * DIMS[1] * DIMS[2]

    S, M, _d_known = phantoms.lung_pair(DIMS, replicas.replica_seed(202, rank))
    dS, dM = device_pair(torch, S, M, device)
    du = torch.zeros((3,) + S.shape, dtype=torch.float32, device=device)
    eng = B.Demons(DIMS, SPACING, B.PASSIVE, 1.0, SIGMA, levels=1, device=device, queue=True)
    stream = torch.cuda.Stream(device=device)
    torch.cuda.synchronize()

    # ---- device-resident timing (the headline `value`) ----
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    secs, launches = time_registrations(torch, B, eng, dS, dM, du, None, ITERS, args.steps, args.warmup, stream,
                                        replicas)
    clocks = sampler.stop()
    units = args.steps * sum(ITERS) * N
    agg = replicas.aggregate(units, secs, device)
    ranks_reporting = int(round(replicas.sum_over_ranks(1.0, device)))
    final_u_absmax = float(du.abs().max())
    # BASELINE.json config 2: 3D error at 1,000 seeded interior points against the known field
    # (PAPER.md L222 protocol) and the correlation coefficient (L234), through the C ABI
    evaluation = None
    if rank == 0:
        pts = phantoms.eval_points(DIMS, np.random.default_rng(2020), 1000)
        truth = phantoms.true_inverse_at(_d_known, pts).astype(np.float32)
        dpts = torch.from_numpy(pts.astype(np.float32)).to(device)
        dtruth = torch.from_numpy(truth).to(device)
        derr = torch.zeros(1000, dtype=torch.float64, device=device)
        dcc = torch.zeros(1, dtype=torch.float64, device=device)
        zero = torch.zeros_like(du)
        torch.cuda.synchronize()  # the tensors above were filled on torch's stream; the library runs on `stream`
        B.demons_point_error(eng.ctx, DIMS, du, 1000, dpts, dtruth, derr, stream)
        B.demons_cc(eng.ctx, DIMS, dS, dM, du, None, dcc, stream)
        torch.cuda.synchronize()
        err_after, cc_after = derr.cpu().numpy().copy(), float(dcc[0])
        B.demons_point_error(eng.ctx, DIMS, zero, 1000, dpts, dtruth, derr, stream)
        B.demons_cc(eng.ctx, DIMS, dS, dM, zero, None, dcc, stream)
        torch.cuda.synchronize()
        err_before, cc_before = derr.cpu().numpy(), float(dcc[0])
        del zero
        evaluation = {"points": 1000, "err_mm_mean_before": float(err_before.mean()), "err_mm_sd_before": float(err_before.std()),
                      "err_mm_mean_after": float(err_after.mean()), "err_mm_sd_after": float(err_after.std()),
                      "cc_before": cc_before, "cc_after": cc_after,
                      "note": "single-scale passive demons cannot capture the 12-voxel motion of config 2 in 300 "
                              "iterations (SURVEY.md 8d); parity and throughput are what this bench grades"}

    # ---- end to end through the C ABI with pinned host buffers ----
    hS, hM = torch.from_numpy(S).pin_memory(), torch.from_numpy(M).pin_memory()
    hu = torch.zeros((3,) + S.shape, dtype=torch.float32).pin_memory()
    B.demons_set_option(eng.ctx, "zero_start", 1)  # zero initial field set on the device: inputs are S and M
    def one_host():
        B.demons_register_host(eng.ctx, hS, hM, hu, None, ITERS, 0.0, None, None, stream)
    for _ in range(2):
        one_host()
    torch.cuda.synchronize()
    replicas.barrier()
    t0 = time.perf_counter()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        one_host()
    ev1.record(stream)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    e2e_secs = max(ev0.elapsed_time(ev1) * 1e-3, wall)
    e2e_serial = replicas.aggregate(units, e2e_secs, device)
    # the same K registrations as ONE queue call: the upload of pair k + 1 and the download of field k - 1 ride beside
    # registration k (every step's S and M still go up and its field still comes down, inside the timed region)
    hu2 = torch.zeros_like(hu).pin_memory()
    def one_queue(k):
        B.demons_register_host_queue(eng.ctx, [hS] * k, [hM] * k, [hu if i % 2 == 0 else hu2 for i in range(k)], None, ITERS,
                                     0.0, None, None, stream)
    one_queue(2)
    torch.cuda.synchronize()
    replicas.barrier()
    t0 = time.perf_counter()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    one_queue(args.steps)
    ev1.record(stream)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    e2e = replicas.aggregate(units, max(ev0.elapsed_time(ev1) * 1e-3, wall), device)
    B.demons_set_option(eng.ctx, "zero_start", 0)
    h2d = 2 * N * 4  # S and M (the zero initial field is set on the device: option "zero_start")
    d2h = 3 * N * 4

    # ---- per-kernel device time inside one more registration ("profile" option: events around every kernel) ----
    B.demons_set_option(eng.ctx, "profile", 1)
    du.zero_()
    torch.cuda.synchronize()
    l0 = B.demons_launch_count(eng.ctx)
    B.demons_register(eng.ctx, dS, dM, du, None, ITERS, 0.0, None, None, stream)
    torch.cuda.synchronize()
    prof = B.demons_get_profile(eng.ctx)
    launches_per_iter = (B.demons_launch_count(eng.ctx) - l0) / sum(ITERS)
    # ---- the same kernels timed INSIDE the replayed graph ("profile" = 2: event-record nodes around one iteration in
    # the middle of every 20-iteration chunk): this, and nothing read from profiles/, is what `frac` is computed from
    B.demons_set_option(eng.ctx, "profile", 2)
    ingraph = {"force": {"ms": 0.0, "groups": 0}, "smooth": {"ms": 0.0, "groups": 0}, "warp": {"ms": 0.0, "groups": 0}}
    for _ in range(3):
        du.zero_()
        torch.cuda.synchronize()
        B.demons_register(eng.ctx, dS, dM, du, None, ITERS, 0.0, None, None, stream)
        torch.cuda.synchronize()
        got = B.demons_get_profile(eng.ctx)
        for k in ingraph:
            ingraph[k]["ms"] += got[k]["ms"]
            ingraph[k]["groups"] += got[k]["groups"]
    B.demons_set_option(eng.ctx, "profile", 0)
    assert ingraph["force"]["groups"] > 0 and ingraph["smooth"]["groups"] > 0, "in-graph timing returned nothing"
    smooth_launches = launches_per_iter - 2  # per iteration: the force kernel, k_metrics_final (side branch), the smoother
    bytes_per_voxel = {"force": 32.0, "smooth": 24.0 if smooth_launches <= 1 else 72.0}
    kernel_names = {"force": "k_force_fixed_lc<0,4> (fused warp+gradient+force+update+metrics, lane-consecutive cells)",
                    "smooth": "k_smooth_tma<3> (TMA-fed single pass, 3 components)" if smooth_launches <= 1
                    else "k_smooth_axis x3 (separable fallback, 3 components)"}
    peak, peak_src = measured_peak()
    # cross-checks only (side fields): ncu's share of the iteration and DRAM bytes per launch from committed captures
    ncu_share = committed_csv("r03_kernel_shares.csv") or committed_csv("r02_kernel_shares.csv")
    ncu_bytes = committed_csv("r03_ncu_traffic.csv") or committed_csv("r02_ncu_traffic.csv")
    per_kernel = {}
    ms_per_iter = 1e3 * agg["seconds"] / (args.steps * sum(ITERS))
    node_gap_ms = ingraph["warp"]["ms"] / max(ingraph["warp"]["groups"], 1)   # the empty bracket of "profile" = 2
    ingraph_iter = sum(ingraph[k]["ms"] / ingraph[k]["groups"] for k in ("force", "smooth"))
    for k in ("force", "smooth"):
        ms_raw = prof[k]["ms"] / max(prof[k]["groups"], 1)
        share_ev = prof[k]["ms"] / max(prof["force"]["ms"] + prof["smooth"]["ms"], 1e-9)
        ms = ingraph[k]["ms"] / ingraph[k]["groups"]
        share_ingraph = ms / ingraph_iter
        gbs = bytes_per_voxel[k] * N / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
        entry = {"kernel": kernel_names[k], "avg_ms": ms,
                 "avg_ms_how": "measured in this run: CUDA event-record nodes inside the replayed level graph around one "
                               f"iteration per 20-iteration chunk, mean of {ingraph[k]['groups']} replays (includes the "
                               "node-to-node launch gaps on both sides of the kernel)",
                 "share_ingraph": share_ingraph, "avg_ms_share_x_iteration": share_ingraph * ms_per_iter,
                 "event_node_gap_ms": node_gap_ms,
                 "share_events_no_graph": share_ev, "share_ncu_committed": ncu_share.get(k),
                 "avg_ms_event_bracketed_no_graph": ms_raw, "alg_bytes_per_voxel": bytes_per_voxel[k],
                 "achieved_gbs": gbs, "achieved_kind": "effective (algorithmic bytes / time)",
                 "frac": gbs / peak, "frac_of_nominal": gbs / NOMINAL_HBM_GBS}
        if k in ncu_bytes and ms > 0:
            dram = ncu_bytes[k] / (ms * 1e-3) / 1e9
            entry["hbm_measured"] = {"dram_bytes_per_launch": ncu_bytes[k], "gbs": dram, "frac": dram / peak,
                                     "frac_of_nominal": dram / NOMINAL_HBM_GBS,
                                     "note": "committed ncu dram__bytes_read + dram__bytes_write of this kernel / the "
                                             "duration measured in this run"}
        per_kernel[k] = entry
    # the committed ncu shares are only a cross-check; say so loudly when they no longer describe this build
    stale_share = bool(ncu_share) and any(abs(ncu_share.get(k, per_kernel[k]["share_ingraph"]) - per_kernel[k]["share_ingraph"]) > 0.05
                                          for k in per_kernel)
    dom = max(("force", "smooth"), key=lambda k: per_kernel[k]["avg_ms"])
    it_gbs = (bytes_per_voxel["force"] + bytes_per_voxel["smooth"]) * N / (ms_per_iter * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": per_kernel[dom]["kernel"], "achieved": per_kernel[dom]["achieved_gbs"],
                "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": per_kernel[dom]["frac"],
                "frac_of_nominal": per_kernel[dom]["frac_of_nominal"], "nominal_peak": NOMINAL_HBM_GBS,
                "traffic": ncu_bytes.get(dom),
                "stale_share": stale_share,
                "ingraph_iteration_ms": ingraph_iter, "event_node_gap_ms": node_gap_ms,
                "note": "frac uses the raw in-graph interval, record-node gaps included (event_node_gap_ms = an empty "
                        "bracket measured the same way): the timed iteration is longer than the untimed one "
                        "(whole_iteration.ms), so frac is a lower bound",
                "whole_iteration": {"ms": ms_per_iter, "alg_bytes_per_voxel": bytes_per_voxel["force"] + bytes_per_voxel["smooth"],
                                    "achieved_gbs": it_gbs, "frac": it_gbs / peak, "frac_of_nominal": it_gbs / NOMINAL_HBM_GBS,
                                    "note": "driver-timed: no attribution involved"},
                "per_kernel": per_kernel}

    line = {
        "metric": METRIC, "value": agg["value"] / 1e9, "unit": UNIT, "n_gpus": ranks_reporting, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * agg["seconds"] / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "config2: lung-CT-shaped phantom 256x256x100 fp32, spacing 0.97x0.97x2.5, passive "
                               "force, single scale, 300 iterations, sigma 1.0",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "working set 210 MB (S, M, u, u') > 126 MB L2; no flush between steps",
                   "graphs": True,
                   "layout": "S and M in one device allocation (the L2 persisting window covers both images)"},
        "clocks": clocks,
        "e2e": {"value": e2e["value"] / 1e9, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": 1e3 * e2e["seconds"] / args.steps,
                "api": "demons_register_host_queue: the K steps as one call on pinned host buffers, transfers of "
                       "neighbouring registrations overlapped with the compute (wall clock around the call)",
                "serial": {"value": e2e_serial["value"] / 1e9, "ms_per_step": 1e3 * e2e_serial["seconds"] / args.steps,
                           "api": "K demons_register_host calls, each: upload, register, download, synchronise"}},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "final_u_absmax_voxel": final_u_absmax,
        "evaluation": evaluation,
    }
    eng.close()

    if rank == 0 and world == 1 and not args.no_extras:
        line["variants"] = bench_variants(torch, B, phantoms, replicas, S, M, _d_known, device, stream)
        line["batch"] = bench_batch(torch, B, replicas, S, M, device, stream)
        sample_iters = 6
        t = oracle_sample(S, M, sample_iters)
        cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else os.cpu_count()
        line["cpu_baseline"] = {"value": sample_iters * N / t / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{sample_iters} of the 300 iterations on the full 256x256x100 pair "
                                          f"({t:.1f} s, single thread; the host offers {cores} cores)",
                                "host_cores": cores, "details": cpu_baseline_details(S, M),
                                "texture_option_error_vs_oracle_128x128x64": texture_error_vs_oracle(torch, B, device, stream)}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def bench_batch(torch, B, replicas, S, M, device, stream):
    """demons_register_batch on BASELINE.json config 3's geometry (256x256x100, three levels x 100, passive):
    B pairs per call.  The two coarse levels of a single registration cannot fill 148 SMs; a batch does."""
    out = {}
    iters = [100, 100, 100]
    dims = DIMS
    for nb in (1, 4, 16):
        eng = B.Demons(dims, SPACING, B.PASSIVE, 1.0, SIGMA, levels=3, device=device, nbatch=nb)
        dS = torch.empty((nb,) + S.shape, dtype=torch.float32, device=device)
        dM = torch.empty_like(dS)
        for k in range(nb):   # the same pair, rolled along x by k voxels: distinct data, same statistics
            dS[k].copy_(torch.from_numpy(np.roll(S, k, axis=2)))
            dM[k].copy_(torch.from_numpy(np.roll(M, k, axis=2)))
        du = torch.zeros((nb, 3) + S.shape, dtype=torch.float32, device=device)
        torch.cuda.synchronize()

        def one():
            B.demons_register_batch(eng.ctx, nb, dS, dM, du, None, iters, 0.0, None, None, stream)

        for _ in range(2):
            one()
        torch.cuda.synchronize()
        reps = 3
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = B.demons_launch_count(eng.ctx)
        ev0.record(stream)
        for _ in range(reps):
            one()
        ev1.record(stream)
        torch.cuda.synchronize()
        secs = ev0.elapsed_time(ev1) * 1e-3 / reps
        voxel_iters = 0
        for l in range(3):
            d = B.demons_level_dims(eng.ctx, l)
            voxel_iters += d[0] * d[1] * d[2] * 100
        out[f"B={nb}"] = {"ms_per_call": 1e3 * secs, "ms_per_pair": 1e3 * secs / nb,
                          "gvoxel_iter_per_s": nb * voxel_iters / secs / 1e9,
                          "launches_per_call": (B.demons_launch_count(eng.ctx) - l0) // reps}
        eng.close()
        del dS, dM, du
    return out


def bench_variants(torch, B, phantoms, replicas, S, M, d_known, device, stream):
    """BASELINE.json config 3 (variants 0-4 on the 256x256x100 pair) and config 4 (inverse consistent on
    the 256x256x110 pair, seed 404): three-level pyramid, 100 iterations per level."""
    out = {}
    iters = [100, 100, 100]
    cases = [(0, 1.0, "passive"), (1, 1.0, "evolved_passive"), (2, 1.0, "active"), (3, 1.0, "double"),
             (4, 0.4, "adjusted_double_a0.4"), (4, 1.0, "adjusted_double_a1.0"), (5, 1.0, "inverse_consistent_256x256x110")]
    pair = {}
    for variant, alpha, name in cases:
        dims = (256, 256, 110) if variant == 5 else DIMS
        if dims not in pair:
            Sx, Mx, dx = (S, M, d_known) if dims == DIMS else phantoms.lung_pair(dims, 404)
            pts = phantoms.eval_points(dims, np.random.default_rng(2020), 1000)
            pair = {dims: (*device_pair(torch, Sx, Mx, device),
                           torch.from_numpy(pts.astype(np.float32)).to(device),
                           torch.from_numpy(phantoms.true_inverse_at(dx, pts).astype(np.float32)).to(device))}
        dS, dM, dpts, dtruth = pair[dims]
        derr = torch.zeros(1000, dtype=torch.float64, device=device)
        eng = B.Demons(dims, SPACING, variant, alpha, SIGMA, levels=3, device=device)
        du = torch.zeros((3, dims[2], dims[1], dims[0]), dtype=torch.float32, device=device)
        dub = torch.zeros_like(du) if variant == 5 else None
        secs, launches = time_registrations(torch, B, eng, dS, dM, du, dub, iters, 3, 2, stream, replicas)
        voxel_iters = 0
        for l in range(3):
            d = B.demons_level_dims(eng.ctx, l)
            voxel_iters += d[0] * d[1] * d[2] * 100
        dval = torch.zeros(2, dtype=torch.float64, device=device)
        torch.cuda.synchronize()  # derr / dval were filled on torch's stream; the library runs on `stream`
        B.demons_point_error(eng.ctx, dims, du, 1000, dpts, dtruth, derr, stream)
        B.demons_ssd(eng.ctx, dims, dS, dM, du, dub, dval, stream)
        torch.cuda.synchronize()
        e = derr.cpu().numpy()
        out[name] = {"ms_per_registration": 1e3 * secs / 3, "gvoxel_iter_per_s": 3 * voxel_iters / secs / 1e9,
                     "launches_per_registration": launches // 3, "final_ssd": float(dval[0]),
                     "err_mm_mean": float(e.mean()), "err_mm_sd": float(e.std())}
        if variant == 5:
            # config 4 report: |u_f(x) + u_b(x + u_f(x))|; u_f alone is half of the symmetric motion
            # (no composite field is formed, reading A14), so its point error against the full truth is large
            B.demons_ic_error(eng.ctx, dims, du, dub, dval, stream)
            torch.cuda.synchronize()
            out[name]["ic_error_voxel_mean"] = float(dval[0])
            out[name]["ic_error_voxel_max"] = float(dval[1])
        eng.close()
    return out


if __name__ == "__main__":
    main()
