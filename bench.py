#!/usr/bin/env python
"""bench.py -- PD slice-iterations/s and stack reconstruction time of the B200 hot path (arXiv 2006.09808).

    python bench.py --gpus N --steps K --warmup W            # the CUDA path (one rank per GPU under torchrun)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands, on the host cores

A "step" is one pass of the whole hot path (all iterations of the PD solve) over one
batch of synthetic input of the named workload.  Default workload: C3 = BASELINE.json configs[3] (128 slices x 8 coil
field maps of 256x256, 200 iterations, lambda 0.005), the largest 256x256 configuration, which fits one GPU; inputs
(0.5 GB) and state (1.6 GB) exceed the 126 MB L2, so no explicit flush is needed between timed steps.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for the meaning of every key.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2006_09808_b200 import shard, synth  # noqa: E402  (input generator and host-side sharding helpers only)

METRIC = "pd_slice_iterations_per_s"
UNIT = "slice-iterations/s"
WORKLOADS = {"C0": 0, "C1": 1, "C2": 2, "C3": 3, "C4": 4, "NS": 5,
             "E1": 6, "E2": 7, "E3": 8}   # E1-E3: stand-ins in the paper's own matrix sizes (256x258, 128x132)

# Algorithmic HBM bytes per pixel of a slice and launch of each kernel class of the streaming variant:
# what the pass must read and write once, spectra counted at 4 B/px/slice (one float2 per pixel of a slice PAIR).
KERNEL_BYTES_PER_PX = {
    "resident": 48.0,     # one launch = the whole path: the streaming floor per slice-ITERATION (x iterations below)
    # literal path (W set, or PD_OPT_FOURIER_DUAL = 0): cols + dual_rows + cols + fd_rows, 80 B/px/slice-iteration
    "dual_rows": 24.0,    # Z r4 w4 + phi r4 + W r4 + p r4 w4
    "dipole_cols": 8.0,   # Z r4 + Z w4
    # W = identity, Fourier-domain dual (pd_streaming_fd.cuh): two launches per iteration, 64 B/px/slice-iteration
    "fd_cols": 20.0,      # Z r4 w4 + phi^ r4 + p^ r4 w4
    "fd_rows": 40.0,      # Z r4 w4 + chi_n r4 + chi_{n-1} r4 + chi_{n+1} w4 + qx r4 w4 + qy r4 w4 + M r4 (36 without a mask)
}
# DRAM bytes per pixel of a slice per launch measured by ncu (dram__bytes_read.sum + dram__bytes_write.sum of one
# `--set full` capture over the whole batch): (kernel, line length, masked) -> B/px
NCU_DRAM_BYTES_PER_PX = {
    ("fd_rows", 512, False): 35.3,   # profiles/r02/ncu_sfd_rows_c4.md: 1.347 + 1.025 GB over 256 slices of 512x512 (36 algorithmic)
    ("fd_cols", 512, False): 19.4,   # profiles/r02/ncu_sfd_cols_c4.md: 0.812 + 0.487 GB (20 algorithmic)
    ("fd_rows", 256, True): 39.7,    # profiles/r02/ncu_sfd_rows_c3.md: 1.636 + 1.029 GB over 1024 slices of 256x256 (40 algorithmic)
    ("fd_cols", 256, True): 19.3,    # profiles/r02/ncu_sfd_cols_c3.md: 0.806 + 0.490 GB (20 algorithmic)
}
PATH_FLOOR_BYTES_PER_PX = 48.0  # streaming floor per slice-iteration (12 words)

# What ncu measured on the resident kernel of THIS build (profiles/r02/, one `--set full` capture of the kernel alone on
# C2 and one metrics-only pass over every launch of a hybrid C3 step); quoted beside the live numbers, never timed here.
NCU_RESIDENT = {
    "source": "profiles/r02/ncu_resident_tm_c2.md (kernel alone on C2, hybrid tail off), profiles/r02/dram_bytes_C3_hybrid_step.md",
    "issue_slots_busy_pct": 38.7, "fma_pipe_pct": 39.3, "l1tex_pct": 54.8, "l2_pct": 11.4, "dram_pct": 0.06,
    "shared_wavefronts_pct_of_peak": 55.5,          # 596.1 M wavefronts / (120 SMs x 8.96 M active cycles), 1 wavefront/clk/SM
    "l2_bytes_per_pixel_pair_iteration": 51.7,      # lts__t_sectors 677.3 M x 32 B / (32 pairs x 200 iterations x 65536)
    "warps_per_scheduler": 4.0, "cycles_per_issue": 10.33,
}
# dram__bytes_read.sum + dram__bytes_write.sum summed over every launch of one step (resident kernel + streaming tail)
NCU_DRAM_BYTES_PER_STEP = {("C3", 47): 81401493248.0}   # (workload, hybrid_tail_pairs) -> bytes (profiles/r02/dram_bytes_C3_hybrid_step.md)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            pk = json.load(f)
        return float(pk["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_sm_mhz():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f).get("sm_max_mhz", 1965.0))
    return 1965.0


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.tmp.flush()
        self.tmp.seek(0)
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.tmp.read().splitlines():
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 9:
                continue
            try:
                sm.append(float(parts[1]))
                mx.append(float(parts[2]))
                power.append(float(parts[3]))
            except ValueError:
                continue
            for name, val in zip(names, parts[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        self.tmp.close()
        os.unlink(self.tmp.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=float(max(power)))
        return out


def oracle_module():
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import pd_oracle  # test infrastructure; only the cpu_baseline / --impl reference legs reach this line
    pd_oracle.lib()
    return pd_oracle


def time_oracle(cfg, data, nsample):
    """The oracle as it stands (float instantiation, one thread) on the first `nsample` batch entries."""
    orc = oracle_module()
    t0 = time.perf_counter()
    out = orc.solve(data["field"][:nsample], data["mask"][:nsample], lambda_=cfg.lam, sigma=cfg.sigma, tau=cfg.tau,
                    theta=cfg.theta, max_iters=cfg.iters, tol=cfg.tol, precision="f32", want_hist=False)
    dt = time.perf_counter() - t0
    return float(out["iters_done"].sum()) / dt, dt, int(out["iters_done"].sum())


def time_oracle_all_cores(cfg, data, nsample):
    """Parallel-for over slices OUTSIDE the oracle (one single-threaded oracle call per slice on a thread pool; the
    ctypes call releases the GIL), on every host core."""
    from concurrent.futures import ThreadPoolExecutor
    orc = oracle_module()
    ncores = os.cpu_count() or 1

    def one(b):
        out = orc.solve(data["field"][b:b + 1], data["mask"][b:b + 1], lambda_=cfg.lam, sigma=cfg.sigma, tau=cfg.tau,
                        theta=cfg.theta, max_iters=cfg.iters, tol=cfg.tol, precision="f32", want_hist=False)
        return int(out["iters_done"].sum())
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=ncores) as ex:
        its = sum(ex.map(one, range(nsample)))
    dt = time.perf_counter() - t0
    return its / dt, dt, its, ncores


def oracle_sample_size(cfg):
    """Batch entries giving roughly 10-30 s of single-core oracle work (about 8e-7 s per pixel-iteration measured)."""
    per_slice = 8e-7 * cfg.nx * cfg.ny * (cfg.iters if cfg.tol <= 0 else min(cfg.iters, 80))
    return int(max(1, min(cfg.batch, round(20.0 / per_slice))))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0   # under torchrun only rank 0 runs the reference arm
    cid = WORKLOADS[args.workload]
    cfg = synth.CONFIGS[cid]
    nsample = max(1, oracle_sample_size(cfg) // 4)        # one step = a bounded sample, so K+W steps end in minutes
    nslices = -(-nsample // cfg.ncoils)
    data = synth.generate(cid, nslices=nslices)
    for _ in range(args.warmup):
        time_oracle(cfg, data, min(nsample, 1))
    t0 = time.perf_counter()
    its = 0
    for _ in range(args.steps):
        _, _, n = time_oracle(cfg, data, nsample)
        its += n
    dt = time.perf_counter() - t0
    value = its / dt
    sample = "first %d of %d batch entries of %s, all %d iterations, per step" % (nsample, cfg.batch, cfg.name, cfg.iters)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(cfg, args.workload, cfg.batch, 1),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def run_prepost(args):
    """--prepost: the steps either side of the iteration (NEXT-4) on the shape of the chosen workload: pd_preprocess
    (automatic scale: max pass + main pass) and pd_combine_coils, CUDA events on the launch stream, HBM roofline from the
    algorithmic bytes (16 + 28 B per pixel; 8 ncoils + 4 B per output pixel).  Its own JSON line."""
    import torch
    from paper_2006_09808_b200 import binding
    torch.cuda.set_device(0)
    binding.lib()
    cfg = synth.CONFIGS[WORKLOADS[args.workload]]
    nsl = max(1, min(cfg.nslices, 4))
    e = synth.echo_pair(cfg.cid, nslices=nsl)
    rep = cfg.nslices // nsl
    s0 = torch.from_numpy(e["s0"]).cuda().repeat(rep, 1, 1).contiguous()
    s1 = torch.from_numpy(e["s1"]).cuda().repeat(rep, 1, 1).contiguous()
    batch, ny, nx = s0.shape
    npix = batch * ny * nx
    f = torch.empty((batch, ny, nx), device="cuda")
    w, m = torch.empty_like(f), torch.empty_like(f)
    wmax = torch.zeros(1, device="cuda")
    out = torch.empty((batch // cfg.ncoils, ny, nx), device="cuda")
    flush = torch.empty(64 * 1024 * 1024, device="cuda") if npix * 44 <= 2 * 126e6 else None
    peak, peak_src = load_peaks()

    def timed(fn):
        for _ in range(args.warmup):
            fn()
        tot = 0.0
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(args.steps):
            if flush is not None:
                flush.fill_(1.0)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            tot += e0.elapsed_time(e1)
        return tot / args.steps

    sampler = ClockSampler(0)
    ms_pre = timed(lambda: binding.preprocess(s0, s1, e["fscale"], 0.3, field=f, weight=w, mask=m, wmax=wmax))
    ms_pre_given = timed(lambda: binding.preprocess(s0, s1, e["fscale"], 0.3, wscale=1.0, field=f, weight=w, mask=m))
    ms_comb = timed(lambda: binding.combine_coils(f, w, cfg.ncoils, out))
    clocks = sampler.stop()

    def roof(ms, nbytes, launches):
        gbs = nbytes / (ms * 1e-3) / 1e9
        return {"ms": ms, "launches": launches, "algorithmic_bytes": nbytes, "bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s",
                "frac": gbs / peak, "peak_source": peak_src}
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import pd_prepost_oracle as po
    t0 = time.perf_counter()
    po.field_map(e["s0"], e["s1"], e["fscale"]); po.weight(e["s0"], e["s1"]); po.mask_f32(e["s0"], e["s1"], 0.3)
    dt = time.perf_counter() - t0
    line = {"metric": "prepost_pixels_per_s", "value": npix / (ms_pre * 1e-3), "unit": "pixels/s (pd_preprocess, automatic scale)", "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_pre, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "%s shape: %d maps of %dx%d, %d coils (synth.echo_pair of %d slices tiled x%d)"
                                   % (args.workload, batch, ny, nx, cfg.ncoils, nsl, rep),
                       "l2": "flushed between steps" if flush is not None else "working set exceeds the 126 MB L2"},
            "preprocess_auto_scale": roof(ms_pre, 44.0 * npix, 2), "preprocess_given_scale": roof(ms_pre_given, 28.0 * npix, 1),
            "combine_coils": roof(ms_comb, (8.0 * cfg.ncoils + 4.0) * (npix // cfg.ncoils), 1),
            "cpu_baseline": {"value": e["s0"].size / dt, "unit": "pixels/s", "cores": 1, "kind": "oracle (numpy, float64)",
                             "sample": "%d maps, %.2f s" % (e["s0"].shape[0], dt)},
            "gpu_launches": 4 * args.steps, "clocks": clocks}
    print(json.dumps(line), flush=True)
    return 0


def run_volume(args):
    """--volume: the true 3-D variant (NEXT-2) on 8 coil volumes of 256 x 256 x 64 (the voxel count of 512 slices of 256^2),
    100 iterations; voxel-iterations/s, HBM roofline of the whole step from its algorithmic bytes (DESIGN.md 5.7:
    the bytes its seven passes must move, two volumes per complex transform: q-update 32, y 8, z with the p-update 22, y 8, x back + chi-update + x forward 4 + 28 + 4 = 106 B per voxel and iteration with a mask).  Its own JSON line."""
    import torch
    from paper_2006_09808_b200 import binding
    torch.cuda.set_device(0)
    binding.lib()
    nx, ny, nz, nvol, iters = 256, 256, 64, 8, 100
    case = synth.volume_case(nx, ny, nz, nvol=2, seed=9)
    f = torch.from_numpy(case["field"]).cuda().repeat(nvol // 2, 1, 1, 1).contiguous()
    m = torch.from_numpy(case["mask"]).cuda().repeat(nvol // 2, 1, 1, 1).contiguous()
    lam = 0.02 * float(np.abs(case["field"]).max())
    out = torch.empty_like(f)
    plan = binding.Plan3D(nx, ny, nz, nvol, 2, lam, 0.25, 0.25, 1.0)
    if args.weighted:   # W set: the literal iteration, K applied twice (12 launches per iteration)
        gen = torch.Generator(device="cuda").manual_seed(200609808)
        plan.set_weight(0.2 + 0.8 * torch.rand(f.shape, device="cuda", generator=gen))
    peak, peak_src = load_peaks()
    for _ in range(args.warmup):
        plan.solve(f, m, out, iters)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        plan.solve(f, m, out, iters)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    clocks = sampler.stop()
    launches = plan.last_launch_count
    plan.destroy()
    nvox = nvol * nz * ny * nx
    bytes_per_voxel_it = 172.0 if args.weighted else 106.0   # literal: 2 x (8 + 8 + 10 + 8 + 8) + 56 (q- and p-update) + 32
    gbs = bytes_per_voxel_it * nvox * iters / (ms * 1e-3) / 1e9
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import pd3_oracle as o3
    t0 = time.perf_counter()
    o3.solve3(case["field"][0], case["mask"][0], lambda_=lam, sigma=0.25, tau=0.25, max_iters=4)
    dt = time.perf_counter() - t0
    line = {"metric": "pd3_voxel_iterations_per_s", "value": nvox * iters / (ms * 1e-3), "unit": "voxel-iterations/s", "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "V1: %d coil volumes of %dx%dx%d (synth.volume_case), %d iterations, B0 along z, mask%s"
                                   % (nvol, nx, ny, nz, iters, ", random W in [0.2, 1] (literal iteration)" if args.weighted else ""),
                       "l2": "working set (%.1f GB) exceeds the 126 MB L2" % (44.0 * nvox / 1e9)},
            "roofline": {"kernel": "whole step (%d launches per iteration)" % (12 if args.weighted else 5), "bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s",
                         "frac": gbs / peak, "algorithmic_bytes_per_voxel_iteration": bytes_per_voxel_it, "peak_source": peak_src,
                         # dram__bytes_read.sum + dram__bytes_write.sum over the five kernels of one iteration (profiles/r02/ncu_volume.md)
                         "traffic": None if args.weighted else 100.3 * nvox * iters},
            "cpu_baseline": {"value": nz * ny * nx * 4 / dt, "unit": "voxel-iterations/s", "cores": os.cpu_count(), "kind": "oracle (numpy float64, numpy.fft)",
                             "sample": "1 volume, 4 iterations, %.1f s" % dt},
            "gpu_launches": launches * args.steps, "clocks": clocks}
    print(json.dumps(line), flush=True)
    return 0


def flops_per_slice_it_ns(cfg):
    P = cfg.nx * cfg.ny
    return P * (10.0 * math.log2(P) + 32.0)


def workload_config(cfg, name, batch_per_gpu, ngpus):
    return {"workload": "%s: %s" % (name, cfg.name), "nx": cfg.nx, "ny": cfg.ny, "batch_per_gpu": batch_per_gpu,
            "slices": cfg.nslices, "coils": cfg.ncoils, "iterations": cfg.iters, "tol": cfg.tol, "lambda": cfg.lam,
            "sigma": cfg.sigma, "tau": cfg.tau, "theta": cfg.theta, "B0": cfg.b0_dir,
            "parallelism": "batch-sharded x%d, no collective" % ngpus,
            "l2": "inputs+state per step exceed the 126 MB L2 (no flush needed)" if batch_per_gpu * cfg.nx * cfg.ny * 32 > 2 * 126e6
                  else "working set fits L2: a 256 MB buffer is overwritten between timed steps"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C3", choices=sorted(WORKLOADS))
    ap.add_argument("--variant", default="auto", choices=["auto", "streaming", "resident"],
                    help="auto: the library's own choice (resident cluster kernel for square slices <= 256, else streaming)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the north-star single-coil stack timing")
    ap.add_argument("--weighted", action="store_true",
                    help="set a non-trivial data weight W (seeded uniform [0.2, 1]): the literal path of PAPER.md:49, "
                         "two K applications per iteration (SURVEY.md 8(f) NEXT-1)")
    ap.add_argument("--hybrid-tail", type=int, default=-1,
                    help="PD_OPT_HYBRID_TAIL: slice pairs run by the streaming kernels beside the resident clusters "
                         "(-1 automatic, 0 off)")
    ap.add_argument("--no-graph-loop", action="store_true",
                    help="PD_OPT_GRAPH_LOOP = 0: plain launches from the host instead of the graphed device-side loop "
                         "(used for the ncu launch lists)")
    ap.add_argument("--volume", action="store_true", help="time the true 3-D variant (NEXT-2, pd_solve3d); own JSON line")
    ap.add_argument("--prepost", action="store_true",
                    help="time pd_preprocess and pd_combine_coils (NEXT-4) on the workload's shape instead of the solve; own JSON line")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if (args.prepost or args.volume) and int(os.environ.get("RANK", "0")) != 0:
        return 0   # single-GPU lines: under torchrun rank 0 alone runs and prints them
    if args.prepost:
        return run_prepost(args)
    if args.volume:
        return run_volume(args)

    import torch
    import torch.distributed as dist
    from paper_2006_09808_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.lib()

    cid = WORKLOADS[args.workload]
    cfg = synth.CONFIGS[cid]
    # weak scaling: every rank reconstructs its own stack of the workload's size (slices are independent)
    data = synth.generate(cid, first_slice=shard.weak_first_slice(cfg.nslices, rank))
    batch = cfg.batch
    P = cfg.nx * cfg.ny
    field = torch.from_numpy(data["field"]).cuda()
    # a config whose mask is all ones ("Mask: all ones", C0 and C4) passes mask = NULL, the ABI's way of saying M = 1
    mask_is_one = bool((data["mask"] == 1.0).all())
    mask = None if mask_is_one else torch.from_numpy(data["mask"]).cuda()
    chi = torch.empty_like(field)
    b0 = binding.B0_Y if cfg.b0_dir == "y" else binding.B0_X
    plan = binding.Plan(cfg.nx, cfg.ny, batch, b0, cfg.lam, cfg.sigma, cfg.tau, cfg.theta)
    if args.variant != "auto":
        plan.set_option(binding.OPT_VARIANT, {"streaming": binding.VARIANT_STREAMING, "resident": binding.VARIANT_RESIDENT}[args.variant])
    plan.set_option(binding.OPT_HYBRID_TAIL, args.hybrid_tail)
    if args.no_graph_loop:
        plan.set_option(binding.OPT_GRAPH_LOOP, 0)
    weight = None
    if args.weighted:
        gen = torch.Generator(device="cuda").manual_seed(200609808 + rank)
        weight = 0.2 + 0.8 * torch.rand(field.shape, device="cuda", generator=gen)
        plan.set_weight(weight)
    plan_info = plan.info()
    plan_info["weighted"] = bool(args.weighted)
    plan_info["mask"] = "none (all ones)" if mask_is_one else "per slice"
    pow2 = {64, 128, 256, 512}
    if not (cfg.nx in pow2 and cfg.ny in pow2):
        plan_info["kernels"] = ("general-length row kernels (dense two-stage line DFT, shared-memory bound, literal iteration; DESIGN.md 5.4)"
                                + (" + tuned column kernel" if cfg.ny in pow2 else ""))
    plan_info["hybrid_tail_pairs"] = plan.hybrid_tail()
    plan_info["hybrid_rho_measured_at_plan_time"] = plan.hybrid_rho()
    small = batch * P * 32 <= 2 * 126e6
    flush = torch.empty(64 * 1024 * 1024, device="cuda") if small else None

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(nsteps, host=False, h=None):
        """K steps bracketed by barrier+sync; device time (CUDA events on the launch stream), max over ranks."""
        barrier()
        total = 0.0
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if flush is None:
            e0.record()
            for _ in range(nsteps):
                if host:
                    plan.solve_host(h[0], h[1], h[2], cfg.iters, cfg.tol)
                else:
                    plan.solve(field, mask, chi, cfg.iters, cfg.tol)
            e1.record()
            torch.cuda.synchronize()
            total = e0.elapsed_time(e1)
        else:
            for _ in range(nsteps):   # small working set: flush L2 between steps, time each step separately
                flush.fill_(1.0)
                e0.record()
                if host:
                    plan.solve_host(h[0], h[1], h[2], cfg.iters, cfg.tol)
                else:
                    plan.solve(field, mask, chi, cfg.iters, cfg.tol)
                e1.record()
                torch.cuda.synchronize()
                total += e0.elapsed_time(e1)
        barrier()
        return shard.max_over_ranks(total, "cuda")

    def total_iters():
        it, _, _ = plan.stats()
        return shard.sum_over_ranks(float(it.sum()), "cuda"), it

    # ---- device-resident measurement (inputs already in HBM)
    timed(args.warmup)
    sampler = ClockSampler(local) if rank == 0 else None
    ms = timed(args.steps)
    clocks = sampler.stop() if sampler else None
    slice_its, its_local = total_iters()
    value = slice_its * args.steps / (ms * 1e-3)
    launches = plan.last_launch_count * args.steps

    # ---- per-kernel device time, live, same K steps with CUDA events around every launch
    plan.set_option(binding.OPT_KERNEL_TIMING, 1)
    ktot = {}
    ms_evt = 0.0
    for _ in range(args.steps):
        ms_evt += timed(1)
        for k, (t, c) in plan.kernel_times().items():
            a = ktot.setdefault(k, [0.0, 0])
            a[0] += t
            a[1] += c
    plan.set_option(binding.OPT_KERNEL_TIMING, 0)
    peak, peak_src = load_peaks()
    dom = max(KERNEL_BYTES_PER_PX, key=lambda k: ktot.get(k, [0.0, 0])[0])
    dom_ms, dom_n = ktot[dom]
    ksum = sum(v[0] for v in ktot.values())
    slice_its_local = float(its_local.sum())
    # FP32 peak of the CUDA cores: NOMINAL (148 SMs x 128 lanes x 2 flop) at the SM clock sampled during the timed region
    sm_mhz = (clocks or {}).get("sm_mhz") or load_sm_mhz()
    alu_peak = 148 * 128 * 2 * sm_mhz * 1e6 / 1e12
    alu_src = "nominal: 148 SMs x 128 FP32 lanes x 2 flop x %.0f MHz (SM clock sampled during the timed region)" % sm_mhz
    flops_per_slice_it = P * (10.0 * math.log2(P) + 32.0)   # algorithmic, two K applications per iteration
    common = {"kernel": dom, "avg_launch_us": 1e3 * dom_ms / dom_n, "share_of_step": dom_ms / ksum,
              "kernel_ms_per_step": {k: v[0] / args.steps for k, v in ktot.items()}, "step_ms_with_events": ms_evt / args.steps}
    if dom == "resident":
        # One launch runs every iteration of every slice (with the hybrid schedule the bracket also covers the streaming
        # tail on the second stream).  HBM is touched at load and store only, so the bound SURVEY.md 8(d) names is
        # max(shared memory, FP32 pipe): report the FP32 fraction, the ncu percentages beside it.
        flops = flops_per_slice_it * slice_its_local
        achieved = flops / (dom_ms / dom_n * 1e-3) / 1e12
        # the ncu pass was taken at the tail the plan chose on that box; a plan whose measured rho gives a tail within 4
        # pairs of it is the same step to 5 % (the tail's share of the traffic is proportional to its pairs)
        tail_now = plan_info.get("hybrid_tail_pairs", 0)
        traffic = None
        for (wl, tl), byts in NCU_DRAM_BYTES_PER_STEP.items():
            if wl == args.workload and abs(tl - tail_now) <= 4:
                traffic = byts * (tail_now / tl if tl else 1.0)
        roofline = dict(common, bound="alu", achieved=achieved, peak=alu_peak, unit="TFLOP/s", frac=achieved / alu_peak,
                        traffic=traffic, peak_source=alu_src, flops_per_launch=flops,
                        flops_model="P (10 log2 P + 32) per slice-iteration (SURVEY.md 8(d)); the Fourier-domain dual executes "
                                    "about 0.58 of that (one FFT round trip per iteration instead of two)",
                        ncu=NCU_RESIDENT,
                        vs_streaming_floor={"what": "the same step against a perfect streaming kernel at 48 B/px/slice-iteration "
                                                    "(no such bytes move: the state is on chip)",
                                            "frac": PATH_FLOOR_BYTES_PER_PX * P * slice_its_local / (dom_ms / dom_n * 1e-3) / 1e9 / peak})
    else:
        # units one launch processes: every active slice once; averaged over the launches of the solve (a stopped slice
        # is skipped by later launches), = batch when no tolerance is set
        avg_active_slices = slice_its_local / max(cfg.iters, 1)
        per_px = KERNEL_BYTES_PER_PX[dom] - (4.0 if (dom == "fd_rows" and mask_is_one) else 0.0)
        bytes_per_launch = per_px * P * avg_active_slices
        achieved = bytes_per_launch / (dom_ms / dom_n * 1e-3) / 1e9
        ncu_px = NCU_DRAM_BYTES_PER_PX.get((dom, cfg.nx if dom == "fd_rows" else cfg.ny, not mask_is_one))
        traffic = ncu_px * P * avg_active_slices if ncu_px is not None else None
        roofline = dict(common, bound="hbm", achieved=achieved, peak=peak, unit="GB/s", frac=achieved / peak, traffic=traffic,
                        peak_source=peak_src, bytes_per_launch=bytes_per_launch)
    step_s = (ms / args.steps) * 1e-3
    path_bytes = PATH_FLOOR_BYTES_PER_PX * P * slice_its_local
    roofline_path = {"bound": "hbm", "what": "whole path at the 48 B/px/slice-iteration streaming floor", "unit": "GB/s",
                     "achieved": path_bytes / step_s / 1e9, "peak": peak}
    roofline_path["frac"] = roofline_path["achieved"] / peak
    # FP32 view of the whole step (all kernels, launch gaps included)
    alu_ach = flops_per_slice_it * slice_its_local / step_s / 1e12
    roofline_alu = {"bound": "alu", "what": "whole path, algorithmic flops P(10 log2 P + 32) per slice-iteration",
                    "unit": "TFLOP/s", "achieved": alu_ach, "peak": alu_peak, "frac": alu_ach / alu_peak, "peak_source": alu_src}

    # ---- end to end through the C ABI with HOST buffers (pinned), H2D and D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        hf = torch.from_numpy(data["field"]).pin_memory()
        hm = None if mask_is_one else torch.from_numpy(data["mask"]).pin_memory()
        hc = torch.empty_like(hf).pin_memory()
        timed(1, host=True, h=(hf, hm, hc))
        ms_h = timed(args.steps, host=True, h=(hf, hm, hc))
        e2e = {"value": slice_its * args.steps / (ms_h * 1e-3), "unit": UNIT, "ms_per_step": ms_h / args.steps,
               "h2d_bytes_per_step": int(hf.numel() * 4 + (0 if hm is None else hm.numel() * 4)), "d2h_bytes_per_step": int(hc.numel() * 4),
               "api": "pd_solve_host (pinned host buffers)"}
        del hf, hm, hc

    # ---- north-star stack (128 slices x 256x256, one field map per slice, 200 iterations): whole-stack recon ms
    extra = None
    if not args.no_extra and not args.weighted and rank == 0 and cid == 3:
        ns = synth.CONFIGS[5]
        f2, m2, c2 = field[::cfg.ncoils].contiguous(), mask[::cfg.ncoils].contiguous(), torch.empty_like(field[::cfg.ncoils])
        plan2 = binding.Plan(ns.nx, ns.ny, ns.batch, b0, ns.lam, ns.sigma, ns.tau, ns.theta)
        if args.variant != "auto":
            plan2.set_option(binding.OPT_VARIANT, {"streaming": binding.VARIANT_STREAMING, "resident": binding.VARIANT_RESIDENT}[args.variant])
        plan2.set_option(binding.OPT_HYBRID_TAIL, args.hybrid_tail)
        for _ in range(3):
            plan2.solve(f2, m2, c2, ns.iters, 0.0)
        torch.cuda.synchronize()
        times = []
        fl = torch.empty(64 * 1024 * 1024, device="cuda")
        for _ in range(max(args.steps, 5)):
            fl.fill_(0.0)   # 256 MB write: flushes L2 between repetitions
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            plan2.solve(f2, m2, c2, ns.iters, 0.0)
            b.record()
            torch.cuda.synchronize()
            times.append(a.elapsed_time(b))
        t_ns = float(np.median(times))
        extra = {"workload": "NS: 128 slices x 256x256, 1 field map per slice, 200 iterations (BASELINE.json north_star target)",
                 "stack_recon_ms": t_ns, "slice_iterations_per_s": ns.batch * ns.iters / (t_ns * 1e-3),
                 "hbm_floor_frac": PATH_FLOOR_BYTES_PER_PX * ns.nx * ns.ny * ns.batch * ns.iters / (t_ns * 1e-3) / 1e9 / peak,
                 "fp32_frac": flops_per_slice_it_ns(ns) * ns.batch * ns.iters / (t_ns * 1e-3) / 1e12 / alu_peak,
                 "hybrid_tail_pairs": plan2.hybrid_tail()}
        plan2.destroy()

    if rank == 0:
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            nsample = max(1, oracle_sample_size(cfg) // 2)
            v, dt, n = time_oracle(cfg, data, nsample)
            nall = min(batch, nsample * (os.cpu_count() or 1))
            va, dta, na, ncores = time_oracle_all_cores(cfg, data, nall)
            cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                   "sample": "first %d of %d batch entries of the same inputs, %d slice-iterations in %.1f s, float instantiation"
                             % (nsample, batch, n, dt),
                   "all_cores": {"value": va, "unit": UNIT, "cores": ncores, "kind": "oracle, parallel-for over slices outside it",
                                 "sample": "first %d of %d batch entries, %d slice-iterations in %.1f s" % (nall, batch, na, dta)},
                   "host_cores_available": os.cpu_count()}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": dict(workload_config(cfg, args.workload, batch, world), **plan_info),
            "stack_recon_ms": ms / args.steps, "slice_iterations_per_step": slice_its,
            "roofline": roofline, "roofline_path": roofline_path, "roofline_alu": roofline_alu, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": launches, "clocks": clocks, "north_star_stack": extra,
            "paper_context": "paper reports 4-15x GPU over CPU on unnamed hardware (PAPER.md:118); not comparable",
        }
        print(json.dumps(line), flush=True)
    plan.destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
