#!/usr/bin/env python
"""bench.py -- IDG filter throughput on B200 (BASELINE.json metric: Gvoxel-iter/s, HBM fraction).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one complete idg_filter call (all n iterations, every row of SURVEY.md section 8(a))
on the workload cube.  Default workload: BASELINE.json configs[3], the 1024x1024x512 fp32 cube
with n = 20 and the paper's default parameters (the HBM-roofline config; it fits one GPU).
`value` is timed with CUDA events on the launching stream with the cube resident in HBM; `e2e`
is the same call through idg_filter_host with pinned HOST buffers (H2D + D2H inside the timed
region).  For N > 1 (torchrun) every rank filters its own cube (independent replicas, no
data-path collective): weak scaling, time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "idg_filter_throughput"
UNIT = "Gvoxel-iter/s"
BYTES_PER_VOXEL_ITER = 8.0          # 4 B read + 4 B written per voxel-iteration, un-fused

WORKLOADS = {
    # name: (nz, ny, nx), n_iter, generator
    "cfg3_1024x1024x512_n20": ((512, 1024, 1024), 20, "large"),
    "cfg2_512x512x256_n20": ((256, 512, 512), 20, "survey"),
    "cfg0_100x100x67_n10": ((67, 100, 100), 10, "modelb"),
    "cfg4_256x128x128x64_n10": ((64, 128, 128), 10, "batch"),      # 256 cubes, per-cube parameters
}
BATCH = 256
# reference filters (PAPER.md:402-405 timing parameters); --filter idg is the contract's metric
FILTERS = {"idg": None, "box": ("box", (3, 3, 3)), "box_aniso": ("box", (3, 5, 5)),
           "gauss": ("gauss", (3.0, 3.0, 3.0), (0.0, 0.0, 0.0)), "gauss_aniso": ("gauss", (2.0, 3.0, 3.0), (0.0, 0.0, 0.0)),
           "gauss_rot": ("gauss", (2.0, 3.0, 3.0), (10.0, 20.0, 30.0)),
           "mask_sums": ("quality",),
           "wavelet_haar": ("wavelet", 0, (0.5, 0.8, 1.1)), "wavelet_legall": ("wavelet", 1, (1.0, 1.4, 1.7))}   # PAPER.md:222                 # Eq. 13-14 over the whole cube: reads 2 cubes
DEFAULT_WORKLOAD = "cfg3_1024x1024x512_n20"


def make_cube(name: str, seed_offset: int = 0, threads=None):
    from paper_1609_03782_b200 import synth
    shape, n, gen = WORKLOADS[name]
    if gen == "large":
        c = synth.large_cube(seed=3000 + seed_offset, shape=shape, threads=threads)
    elif gen == "survey":
        c = synth.survey_field(shape, seed=2000 + seed_offset, n_discs=6, threads=threads)
    elif gen == "batch":                      # one cube of the batch (reference arm / oracle sample)
        c = synth.modelb_like(shape, seed=4000 + seed_offset, snr=32.0, threads=threads)
    else:
        c = synth.modelb_like(shape, seed=1000 + seed_offset, snr=32.0, threads=threads)
    return c, n


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic_bytes(kernel_tag: str):
    """dram read+write bytes per launch of the dominant kernel from the committed ncu summary."""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    try:
        for line in open(p):
            k, _, v = line.partition(" = ")              # the key itself holds '=' signs ("fuse=4")
            if k.strip() == kernel_tag:
                return float(v.split()[0])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, f"/tmp/idg_clocks_{os.getpid()}.csv"

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        try:
            for line in open(self.path):
                f = [s.strip() for s in line.split(",")]
                if len(f) < 8:
                    continue
                try:
                    sm.append(float(f[1]))
                    mx.append(float(f[2]))
                except ValueError:
                    continue
                for nme, v in zip(names, f[4:8]):
                    if v.lower().startswith("active"):
                        reasons.add(nme)
            os.remove(self.path)
        except Exception:
            pass
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_rate(cube: np.ndarray, n_iter: int, target_s: float, prm: dict):
    """Time the oracle, as it stands, on a bounded sample: the first planes of the workload cube."""
    import oracle
    cores = oracle.set_threads(os.cpu_count() or 1)
    nz, ny, nx = cube.shape
    probe = cube[: min(nz, 4)]
    t0 = time.perf_counter()
    oracle.idg_filter_oracle(probe, 2, **prm)
    rate = probe.size * 2 / max(time.perf_counter() - t0, 1e-6)          # voxel-iter/s, rough
    planes = int(max(2, min(nz, target_s * rate / (ny * nx * n_iter))))
    sample = cube[:planes]
    t0 = time.perf_counter()
    oracle.idg_filter_oracle(sample, n_iter, **prm)
    dt = time.perf_counter() - t0
    if dt < target_s / 3 and planes < nz:       # the 4-plane probe underestimates the rate: size the sample again
        planes = int(min(nz, planes * target_s / max(dt, 1e-6)))
        sample = cube[:planes]
        t0 = time.perf_counter()
        oracle.idg_filter_oracle(sample, n_iter, **prm)
        dt = time.perf_counter() - t0
    desc = f"first {planes} of {nz} planes ({nx}x{ny}x{planes} voxels), n={n_iter}, fp64, {dt:.1f} s"
    return sample.size * n_iter / dt / 1e9, cores, desc, dt


def run_reference(args) -> None:
    """--impl reference: the fp64 oracle on the host cores (rank 0 only), bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1609_03782_b200.binding import Params
    cube, n = make_cube(args.workload)
    prm = Params().f32()
    import oracle
    cores = oracle.set_threads(os.cpu_count() or 1)
    nz, ny, nx = cube.data.shape
    # size the per-step sample so that steps + warm-up end within a few minutes
    _, _, _, _ = oracle_rate(cube.data, n, 1.0, prm)                       # warms caches and threads
    r, _, _, _ = oracle_rate(cube.data, n, 2.0, prm)
    budget = 150.0 / max(1, args.steps + args.warmup)
    planes = int(max(2, min(nz, budget * r * 1e9 / (ny * nx * n))))
    sample = cube.data[:planes]
    for _ in range(args.warmup):
        oracle.idg_filter_oracle(sample, n, **prm)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.idg_filter_oracle(sample, n, **prm)
    dt = (time.perf_counter() - t0) / args.steps
    v = sample.size * n / dt / 1e9
    desc = f"first {planes} of {nz} planes ({nx}x{ny}x{planes} voxels) per step, n={n}, fp64 oracle"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "n_iter": n, "params": "K=1.5 tau=0.0325 C=5 (PAPER.md:187)",
                   "sample": desc},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def max_over_ranks(ms: float, world: int, device) -> float:
    """Slowest rank's time (the contract's max over ranks); a collective every rank must enter."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(voxel_iters_per_rank: float, world: int, ms_step_max: float) -> float:
    """Whole-job throughput: the units all ranks processed / the slowest rank's time, in G/s."""
    return world * voxel_iters_per_rank / (ms_step_max * 1e-3) / 1e9


def run_ours(args) -> None:
    import torch
    import torch.distributed as dist
    from paper_1609_03782_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the IDG filter has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()                                   # fail loudly if the extension is missing
    B.idg_set_option(B.IDG_OPT_FUSE, args.fuse)
    B.idg_set_option(B.IDG_OPT_ZCHUNK, args.zchunk)
    B.idg_set_option(B.IDG_OPT_TILE, args.tile)

    threads = max(1, (os.cpu_count() or 1) // max(1, world))
    batched = WORKLOADS[args.workload][2] == "batch"
    filt = FILTERS[args.filter]
    if batched:
        from paper_1609_03782_b200 import synth
        shape, n, _ = WORKLOADS[args.workload]
        data = synth.batch_cubes(BATCH, seed=4000 + 1000 * rank, shape=shape, threads=threads)
        plist = [B.Params(*[float(v) for v in row]) for row in synth.batch_params(BATCH, seed=4000 + 1000 * rank)]
        nz, ny, nx = shape
        N = BATCH * nz * ny * nx
        args.no_e2e = True                    # the host-buffer entry point takes one cube
    else:
        cube, n = make_cube(args.workload, seed_offset=rank, threads=threads)
        data = cube.data
        nz, ny, nx = data.shape
        N = nz * ny * nx
    p = B.Params()                            # PAPER.md:187 defaults; rms = 1 by construction
    host_in = torch.from_numpy(data).pin_memory()
    d_in = host_in.cuda(non_blocking=True)
    d_out = torch.empty_like(d_in)
    ws = B.alloc_workspace(nx, ny, nz, BATCH if batched else 1)
    stream = torch.cuda.current_stream()
    if filt is not None:
        if batched:
            raise SystemExit("--filter box/gauss runs on single-cube workloads")
        n = 1                                 # one pass; throughput in Gvoxel/s
        args.no_e2e = True
        if filt[0] == "quality":              # the "filtered" cube: a box-smoothed copy
            B.idg_box_filter(d_in, 3, 3, 3, out=d_out, stream=stream)
            q_sums = torch.empty(8, dtype=torch.float64, device="cuda")

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        if filt is not None:
            if filt[0] == "quality":
                B.idg_mask_sums(d_in, d_out, None, 3.0, 1.5, None, sums=q_sums, stream=stream)
            elif filt[0] == "wavelet":
                B.idg_wavelet_filter(d_in, filt[1], filt[2], 1.0, out=d_out, stream=stream)
            elif filt[0] == "box":
                B.idg_box_filter(d_in, *filt[1], out=d_out, stream=stream)
            else:
                B.idg_gaussian_filter(d_in, filt[1], filt[2], out=d_out, stream=stream)
        elif batched:
            B.idg_filter_batched(d_in, n, plist, out=d_out, workspace=ws, stream=stream)
        else:
            B.idg_filter(d_in, n, p, out=d_out, workspace=ws, stream=stream)

    for _ in range(max(3, args.warmup)):
        step()
    launches_per_step = B.idg_last_launch_count()
    plan = B.idg_last_plan()
    fuse = -(-n // launches_per_step)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else {}
    ms_step = max_over_ranks(ms, world, "cuda") / args.steps
    value = aggregate_value(N * n, world, ms_step)

    # end to end through the C-ABI host entry point: pinned host buffers, copies inside the timed region
    e2e_value = None
    if not args.no_e2e:
        host_out = torch.empty_like(host_in).pin_memory()
        dev = torch.empty(B.host_buffers_bytes(nx, ny, nz), dtype=torch.uint8, device="cuda")
        for _ in range(2):
            B.idg_filter_host(host_in, n, p, out_host=host_out, dev_buffers=dev, stream=stream)
        barrier()
        e_steps = max(2, min(args.steps, 5))
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(e_steps):
            B.idg_filter_host(host_in, n, p, out_host=host_out, dev_buffers=dev, stream=stream)
        e1.record(stream)
        barrier()
        e_ms = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3)
        e2e_value = aggregate_value(N * n, world, max_over_ranks(e_ms, world, "cuda") / e_steps)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak_gbs()
    ms_launch = ms_step / launches_per_step
    if filt is not None and filt[0] == "wavelet":      # many small passes: the roofline unit is the whole filter
        ms_launch, fuse = ms_step, 1
    achieved = BYTES_PER_VOXEL_ITER * N * fuse / (ms_launch * 1e-3) / 1e9     # algorithmic GB/s per launch
    kernel_tag = f"{plan} {args.workload}"
    if filt is not None:                      # reference filter: its own metric, oracle timed on a small block
        import oracle
        cores = oracle.set_threads(os.cpu_count() or 1)
        blk = data[:min(nz, 48), :min(ny, 256), :min(nx, 256)]
        t0 = time.perf_counter()
        if filt[0] == "quality":
            from oracle import quality_oracle
            blk = data
            t0 = time.perf_counter()
            quality_oracle.mask_sums_oracle(blk, blk, None, 3.0, 1.5)
        elif filt[0] == "wavelet":
            blk = data[:min(nz, 128)]
            t0 = time.perf_counter()
            oracle.wavelet_filter_oracle(blk, filt[1], filt[2], 1.0)
        elif filt[0] == "box":
            oracle.box_filter_oracle(blk, *filt[1])
        else:
            oracle.gaussian_filter_oracle(blk, filt[1], filt[2])
        dt = time.perf_counter() - t0
        cpu_v, sample = blk.size / dt / 1e9, f"{blk.shape[2]}x{blk.shape[1]}x{blk.shape[0]} block, oracle as it stands, fp64, {dt:.1f} s"
        metric, unit, params = f"{args.filter}_throughput", "Gvoxel/s", str(filt[1:])
    else:
        first = data[0] if batched else data
        cpu_v, cores, sample, _ = oracle_rate(first, n, 15.0, (plist[0] if batched else p).f32())
        metric, unit = METRIC, UNIT
        params = ("per-cube K, tau, C_j (synth.batch_params)" if batched
                  else "K=1.5 tau=0.0325 Cx=Cy=Cz=5 rms=1 (PAPER.md:187, :406)")
    line = {
        "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "shape_xyz": [nx, ny, nz], "n_iter": n,
                   "params": params, "batch": BATCH if batched else 1,
                   "fused_iterations_per_launch": fuse, "parallelism": f"replicas x{world}",
                   "l2": f"input + output ({2 * N * 4 / 1e6:.0f} MB per call) against the 126 MB L2: "
                         + ("larger, no flush needed" if 2 * N * 4 > 252e6 else "NOT larger -- warm-L2 number"),
                   "paper_context": "GTX860M OpenGL 0.90, i7 8 threads 0.036 Gvoxel-iter/s (PAPER.md:408-414)"},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": ncu_traffic_bytes(kernel_tag),
                     "kernel": plan, "ms_per_launch": ms_launch,
                     "algorithmic_bytes_per_launch": BYTES_PER_VOXEL_ITER * N * fuse,
                     "peak_source": peak_src,
                     "note": "algorithmic bytes = 8 B x voxels x fused iterations (what an un-fused sweep must "
                             "move); temporal fusion moves fewer DRAM bytes, so frac can exceed 1 -- see traffic"},
        "cpu_baseline": {"value": cpu_v, "unit": unit, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": e2e_value, "unit": unit, "h2d_bytes_per_step": N * 4, "d2h_bytes_per_step": N * 4,
                "api": "idg_filter_host (pinned host buffers)"},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks,
    }
    if filt is None:
        # after temporal fusion the IDG kernels sit between the DRAM and the FP32 ceilings: report the second too
        lane_ops = 10.0 * value * 1e9 / 1e12                       # 10 FP32 lane-ops per voxel-iteration
        peak_ops = 148 * 128 * 1.965e9 / 1e12
        line["roofline"]["alu"] = {"achieved": lane_ops, "peak": peak_ops, "unit": "T lane-op/s", "frac": lane_ops / peak_ops,
                                   "note": "useful voxel-iterations only; halo recomputation (x 1.2 at T = 2 to x 1.45 at T = 4) comes on top"}
    if filt is not None and filt[0] == "gauss" and any(filt[2]):     # rotated Gaussian: bound by FP32, not by HBM
        r = B.idg_gaussian_radii(filt[1], filt[2])[0]
        flops = 2.0 * (2 * r + 1) ** 3 * N
        peak_tf = 148 * 128 * 2 * 1.965e9 / 1e12          # SMs x FP32 lanes x 2 flop x max clock (B200_PROFILING.md)
        line["roofline"] = {"bound": "alu", "achieved": flops / (ms_launch * 1e-3) / 1e12, "peak": peak_tf,
                            "unit": "TFLOP/s", "frac": flops / (ms_launch * 1e-3) / 1e12 / peak_tf, "traffic": None,
                            "kernel": plan, "ms_per_launch": ms_launch,
                            "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--filter", default="idg", choices=sorted(FILTERS),
                    help="idg (the contract's metric) or a reference filter: one pass, Gvoxel/s")
    ap.add_argument("--fuse", type=int, default=0, help="iterations fused per launch (0 = library default)")
    ap.add_argument("--zchunk", type=int, default=0, help="planes per CTA along z (0 = library default)")
    ap.add_argument("--tile", type=int, default=0, help="TMA kernel tile variant (0 = library default)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
