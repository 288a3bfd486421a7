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
    # configs[1]: S/N 22 and 62 cubes x 8 K values; a step = the whole exploration, one batched 16-cube call per n = 1..40
    "cfg1_sweep_2x8x40": ((67, 100, 100), 40, "sweep"),
}
BATCH = 256
L2_BYTES = 126e6                    # B200 L2 (B200_PROFILING.md)
L2_PEAK_GBS = 6300 * 1.965          # ~6300 B/clk chip-wide LTS cap x 1.965 GHz (B300_MICROARCH.md, L2 cache) = 12.4 TB/s
# reference filters (PAPER.md:402-405 timing parameters); --filter idg is the contract's metric
FILTERS = {"idg": None, "box": ("box", (3, 3, 3)), "box_aniso": ("box", (3, 5, 5)),
           "gauss": ("gauss", (3.0, 3.0, 3.0), (0.0, 0.0, 0.0)), "gauss_aniso": ("gauss", (2.0, 3.0, 3.0), (0.0, 0.0, 0.0)),
           "gauss5": ("gauss", (5.0, 5.0, 5.0), (0.0, 0.0, 0.0)), "gauss7": ("gauss", (7.0, 7.0, 7.0), (0.0, 0.0, 0.0)),
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


def ncu_counters(plan: str, workload: str) -> dict:
    """Per-launch ncu counters of the dominant kernel of (plan, workload) from the committed table
    profiles/ncu_per_launch.txt (each entry names its source note and commit); {} when this plan on this workload
    has never been captured -- then the line carries no traffic figure rather than someone else's."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_per_launch.txt")) as f:
            for e in json.load(f)["entries"]:
                if e["plan"] == plan and e["workload"] == workload:
                    return e
    except Exception:
        pass
    return {}


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


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


class OracleBuffers:
    """fp64 input, output and scratch of the oracle for `planes` planes of a cube, allocated and touched once, so that
    a timed call measures the oracle's arithmetic and not the page faults of fresh multi-GB allocations."""

    def __init__(self, cube: np.ndarray, planes: int):
        self.a = np.ascontiguousarray(cube[:planes], dtype=np.float64)
        self.out = np.zeros_like(self.a)
        self.scratch = np.zeros_like(self.a)

    def run(self, n_iter: int, prm: dict) -> float:
        import oracle
        t0 = time.perf_counter()
        oracle.idg_filter_oracle_into(self.a, n_iter, self.out, self.scratch, **prm)
        return time.perf_counter() - t0


def oracle_rate(cube: np.ndarray, n_iter: int, target_s: float, prm: dict, threads=None):
    """Time the oracle, as it stands, on a bounded sample: the first planes of the workload cube (buffers preallocated
    and touched; the fp32 -> fp64 conversion of the input is outside the timed region)."""
    import oracle
    cores = oracle.set_threads(threads or os.cpu_count() or 1)
    nz, ny, nx = cube.shape
    probe = OracleBuffers(cube, min(nz, 8))
    probe.run(2, prm)                                                      # threads and caches warm
    rate = probe.a.size * 2 / max(probe.run(2, prm), 1e-6)                 # voxel-iter/s, rough
    planes = int(max(2, min(nz, target_s * rate / (ny * nx * n_iter))))
    buf = OracleBuffers(cube, planes)
    dt = buf.run(n_iter, prm)
    if dt < target_s / 3 and planes < nz:       # the small probe underestimates the rate: size the sample again
        planes = int(min(nz, planes * target_s / max(dt, 1e-6)))
        buf = OracleBuffers(cube, planes)
        dt = buf.run(n_iter, prm)
    desc = (f"first {planes} of {nz} planes ({nx}x{ny}x{planes} voxels), n={n_iter}, fp64, {dt:.1f} s "
            "(buffers preallocated; conversion to fp64 not timed)")
    return buf.a.size * n_iter / dt / 1e9, cores, desc, dt


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
    buf = OracleBuffers(cube.data, planes)
    for _ in range(args.warmup):
        buf.run(n, prm)
    dt = sum(buf.run(n, prm) for _ in range(args.steps)) / args.steps
    sample = buf.a
    v = sample.size * n / dt / 1e9
    desc = (f"first {planes} of {nz} planes ({nx}x{ny}x{planes} voxels) per step, n={n}, fp64 oracle "
            "(buffers preallocated; conversion to fp64 not timed)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "n_iter": n, "params": "K=1.5 tau=0.0325 C=5 (PAPER.md:187)",
                   "sample": desc},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "cpu_model": cpu_model()},
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
    from paper_1609_03782_b200 import synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the IDG filter has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()                                   # fail loudly if the extension is missing
    B.idg_set_option(B.IDG_OPT_KERNEL, args.kernel)
    B.idg_set_option(B.IDG_OPT_FUSE, args.fuse)
    B.idg_set_option(B.IDG_OPT_ZCHUNK, args.zchunk)
    B.idg_set_option(B.IDG_OPT_TILE, args.tile)

    threads = max(1, (os.cpu_count() or 1) // max(1, world))
    shape, n, gen = WORKLOADS[args.workload]
    batched, sweep = gen == "batch", gen == "sweep"
    filt = FILTERS[args.filter]
    nz, ny, nx = shape
    nb = 1
    if batched:
        nb = BATCH
        data = synth.batch_cubes(nb, seed=4000 + 1000 * rank, shape=shape, threads=threads)
        plist = [B.Params(*[float(v) for v in row]) for row in synth.batch_params(nb, seed=4000 + 1000 * rank)]
    elif sweep:                               # configs[1]: 2 cubes x 8 K
        two = [synth.modelb_like(shape, seed=1001 + 10 * rank, snr=22.0, threads=threads).data,
               synth.modelb_like(shape, seed=1002 + 10 * rank, snr=62.0, threads=threads).data]
        data = np.stack([two[i] for i in (0, 1) for _ in synth.K_SWEEP])
        plist = [B.Params(K=float(K)) for _ in (0, 1) for K in synth.K_SWEEP]
        nb = len(plist)
    else:
        cube, n = make_cube(args.workload, seed_offset=rank, threads=threads)
        data = cube.data
    N = nb * nz * ny * nx
    if nb > 1:
        args.no_e2e = True                    # the host-buffer entry point takes one cube
    p = B.Params()                            # PAPER.md:187 defaults; rms = 1 by construction
    host_in = torch.from_numpy(data).pin_memory()
    d_in = host_in.cuda(non_blocking=True)
    d_out = torch.empty_like(d_in)
    ws = B.alloc_workspace(nx, ny, nz, nb)
    stream = torch.cuda.current_stream()
    if filt is not None:
        if nb > 1:
            raise SystemExit("--filter box/gauss runs on single-cube workloads")
        n = 1                                 # one pass; throughput in Gvoxel/s
        args.no_e2e = True
        if filt[0] == "quality":              # the "filtered" cube: a box-smoothed copy
            B.idg_box_filter(d_in, 3, 3, 3, out=d_out, stream=stream)
            q_sums = torch.empty(8, dtype=torch.float64, device="cuda")
    voxel_iters = N * (n * (n + 1) // 2 if sweep else n)      # per step

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    launches = [0]

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
            launches[0] = B.idg_last_launch_count()
        elif sweep:                           # every n from scratch, one batched call each
            launches[0] = 0
            for k in range(1, n + 1):
                B.idg_filter_batched(d_in, k, plist, out=d_out, workspace=ws, stream=stream)
                launches[0] += B.idg_last_launch_count()
        elif batched:
            B.idg_filter_batched(d_in, n, plist, out=d_out, workspace=ws, stream=stream)
            launches[0] = B.idg_last_launch_count()
        else:
            B.idg_filter(d_in, n, p, out=d_out, workspace=ws, stream=stream)
            launches[0] = B.idg_last_launch_count()

    warm = max(3, args.warmup)
    for _ in range(warm):
        step()
    launches_per_step = launches[0]
    plan = B.idg_last_plan()
    fuse = max(1, -(-n // launches_per_step)) if not sweep else 1
    barrier()

    # L2 rule: a working set (input + output of a call) that fits the 126 MB L2 is timed COLD -- a 512 MB scratch
    # write between the timed calls, outside the events -- and the back-to-back (warm) figure is reported beside it.
    fits_l2 = 2 * N * 4 <= 2 * L2_BYTES
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device="cuda") if fits_l2 else None

    def timed(steps: int, flush: bool) -> float:
        e0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps if flush else 1)]
        e1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps if flush else 1)]
        if not flush:
            e0[0].record(stream)
            for _ in range(steps):
                step()
            e1[0].record(stream)
        else:
            for i in range(steps):
                flush_buf.fill_(i & 0xff)
                e0[i].record(stream)
                step()
                e1[i].record(stream)
        barrier()
        return sum(a.elapsed_time(b) for a, b in zip(e0, e1))

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms = timed(args.steps, fits_l2)
    clocks = sampler.stop() if rank == 0 else {}
    ms_step = max_over_ranks(ms, world, "cuda") / args.steps
    value = aggregate_value(voxel_iters, world, ms_step)
    l2_note = {"working_set_mb": 2 * N * 4 / 1e6, "timed": "larger than L2: back to back, no flush needed"}
    if fits_l2:
        ms_warm = max_over_ranks(timed(args.steps, False), world, "cuda") / args.steps
        l2_note = {"working_set_mb": 2 * N * 4 / 1e6, "timed": "cold: 512 MB scratch write between timed calls (value)",
                   "warm_ms_per_step": ms_warm, "warm_value": aggregate_value(voxel_iters, world, ms_warm),
                   "cold_ms_per_step": ms_step}
    extra = {}
    if sweep:                                 # the same exploration run incrementally: 40 single-iteration calls (pin P11)
        cur = d_in.clone()

        def inc():
            cur.copy_(d_in)
            for _ in range(n):
                B.idg_filter_batched(cur, 1, plist, out=cur, workspace=ws, stream=stream)
        for _ in range(2):
            inc()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            inc()
        e1.record(stream)
        barrier()
        ms_inc = max_over_ranks(e0.elapsed_time(e1), world, "cuda") / args.steps
        extra["incremental_sweep"] = {"ms_per_sweep": ms_inc, "value": aggregate_value(N * n, world, ms_inc), "unit": UNIT,
                                      "what": f"{n} single-iteration batched calls in place (warm), {nb} cubes", "plan": B.idg_last_plan()}

    # end to end through the C-ABI host entry point: pinned host buffers, copies inside the timed region
    e2e_value, e2e_floor = None, None
    if not args.no_e2e:
        host_out = torch.empty_like(host_in).pin_memory()
        dev = torch.empty(B.host_buffers_bytes(nx, ny, nz), dtype=torch.uint8, device="cuda")
        for _ in range(2):
            B.idg_filter_host(host_in, n, p, out_host=host_out, dev_buffers=dev, stream=stream)
        barrier()
        e_steps = max(2, min(args.steps, 5))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(e_steps):
            B.idg_filter_host(host_in, n, p, out_host=host_out, dev_buffers=dev, stream=stream)
        e1.record(stream)
        barrier()
        e_ms = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3)
        e2e_value = aggregate_value(voxel_iters, world, max_over_ranks(e_ms, world, "cuda") / e_steps)
        # its floor, measured: the same bytes over the same link with no kernel at all -- upload of the cube and
        # download of a cube on two streams at once, in the slabs the pipeline uses
        s_up, s_dn = torch.cuda.Stream(), torch.cuda.Stream()
        slabs = 16 if N * 4 >= (64 << 20) else 1
        zs = -(-nz // slabs)
        d_tmp = d_out

        def copies():
            for z in range(0, nz, zs):
                with torch.cuda.stream(s_up):
                    d_in[z:z + zs].copy_(host_in[z:z + zs], non_blocking=True)
                with torch.cuda.stream(s_dn):
                    host_out[z:z + zs].copy_(d_tmp[z:z + zs], non_blocking=True)
        copies()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e_steps):
            copies()
        barrier()
        f_ms = max_over_ranks((time.perf_counter() - t0) * 1e3, world, "cuda") / e_steps
        e2e_floor = {"ms_per_step": f_ms, "value": aggregate_value(voxel_iters, world, f_ms),
                     "what": f"copy-only pipeline: H2D and D2H of {N * 4 / 1e9:.2f} GB each, {slabs} slabs, two streams, no kernel",
                     "frac": f_ms / (max_over_ranks(e_ms, world, "cuda") / e_steps)}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak_gbs()
    roof_launches = launches_per_step
    if filt is not None and filt[0] == "wavelet":      # many small passes: the roofline unit is the whole filter
        roof_launches, fuse = 1, 1
    ms_launch = ms_step / roof_launches
    alg_bytes = BYTES_PER_VOXEL_ITER * voxel_iters / roof_launches            # algorithmic bytes per launch
    if filt is None and "fuse=" in plan:               # iterations the dominant kernel fuses (a sweep mixes tails in)
        try:
            fuse = max(fuse, int(plan.split("fuse=")[1].split()[0]))
        except ValueError:
            pass
    if "idg_resident" in plan:
        fuse = n
    hbm_equiv = alg_bytes / (ms_launch * 1e-3) / 1e9
    ncu = ncu_counters(plan, args.workload)
    traffic = ncu.get("dram_bytes")
    import oracle
    if filt is not None:                      # reference filter: its own metric, oracle timed on a small block
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
        cpu_1 = None
        metric, unit, params = f"{args.filter}_throughput", "Gvoxel/s", str(filt[1:])
    else:
        first = data[0] if nb > 1 else data
        prm0 = (plist[0] if nb > 1 else p).f32()
        n_cpu = 10 if sweep else n
        cpu_v, cores, sample, _ = oracle_rate(first, n_cpu, 12.0, prm0)
        v1, _, s1, _ = oracle_rate(first, n_cpu, 5.0, prm0, threads=1)
        oracle.set_threads(os.cpu_count() or 1)
        cpu_1 = {"value": v1, "unit": UNIT, "cores": 1, "sample": s1}
        metric, unit = METRIC, UNIT
        params = ("per-cube K, tau, C_j (synth.batch_params)" if batched
                  else "K in {0.5,1,1.5,2,3,5,7.5,10} x S/N {22,62}, tau=0.0325 C=5, every n = 1..40 from scratch" if sweep
                  else "K=1.5 tau=0.0325 Cx=Cy=Cz=5 rms=1 (PAPER.md:187, :406)")

    # Which ceiling binds.  The temporally fused IDG kernels are bound by FP32 issue, not by HBM:
    # the roof is the SMs' instruction issue rate (148 SMs x 4 schedulers x 1.965 GHz, B200_PROFILING.md unit counts)
    # and `achieved` is the MEASURED warp-instruction count of this plan (ncu, profiles/ncu_per_launch.txt) over the
    # launch time measured live here.  hbm_equiv_frac keeps north_star's figure (8 B per voxel-iteration over the
    # copy bandwidth: > 1 means the fusion beats an un-fused sweep); dram_frac_actual is what really crosses the HBM pins.
    issue_peak = 148 * 4 * 1.965e9 / 1e12              # T warp-instructions / s
    fused_idg = filt is None and ("idg_tma" in plan or "idg_stream" in plan or "idg_resident" in plan) and fuse >= 2
    roof = {"bound": "hbm", "achieved": hbm_equiv, "peak": peak, "unit": "GB/s", "frac": hbm_equiv / peak,
            "traffic": traffic, "kernel": plan, "ms_per_launch": ms_launch,
            "algorithmic_bytes_per_launch": alg_bytes, "peak_source": peak_src}
    wi = ncu.get("warp_instructions")
    if fused_idg and wi:
        roof.update({"bound": "alu", "unit": "T warp-inst/s", "peak": issue_peak,
                     "achieved": (wi / (ms_launch * 1e-3) / 1e12) if wi else None,
                     "frac": (wi / (ms_launch * 1e-3) / 1e12 / issue_peak) if wi else None,
                     "peak_source": "derived: 148 SMs x 4 warp schedulers x 1.965 GHz (B200_PROFILING.md)",
                     "warp_instructions_per_launch": wi,
                     "useful_thread_inst_per_voxel_iter": (wi * 32 / (voxel_iters / roof_launches)) if wi else None})
    elif fused_idg:
        roof["note_bound"] = ("a fused IDG plan is bound by instruction issue, not HBM; no ncu instruction count of this plan on "
                              "this workload is committed, so only the HBM-equivalent figure is given")
    roof["hbm_equiv_gbs"] = hbm_equiv
    roof["hbm_equiv_frac"] = hbm_equiv / peak
    roof["hbm_peak_gbs"] = peak
    roof["dram_frac_actual"] = (traffic / (ms_launch * 1e-3) / 1e9 / peak) if traffic else None
    roof["counters_source"] = ({k: ncu[k] for k in ("source", "commit") if k in ncu} if ncu else
                               "no ncu capture of this plan on this workload is committed: traffic and the ALU figures are withheld")
    if fits_l2:
        l2b = ncu.get("l2_bytes")
        roof["l2"] = {"bytes_per_launch": l2b, "gbs": (l2b / (ms_launch * 1e-3) / 1e9) if l2b else None,
                      "peak_gbs": L2_PEAK_GBS, "frac": (l2b / (ms_launch * 1e-3) / 1e9 / L2_PEAK_GBS) if l2b else None,
                      "note": "L2 -> SM read bytes (l1tex__m_xbar2l1tex_read_bytes.sum) of the ncu capture over the launch time measured here"}
    roof["note"] = ("algorithmic bytes = 8 B x voxel-iterations of a launch (what an un-fused sweep must move); temporal "
                    "fusion moves fewer DRAM bytes, so hbm_equiv_frac can exceed 1 -- dram_frac_actual is the real HBM load")
    line = {
        "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps,
        "warmup": warm, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "shape_xyz": [nx, ny, nz], "n_iter": n,
                   "params": params, "batch": nb,
                   "fused_iterations_per_launch": fuse, "parallelism": f"replicas x{world}",
                   "l2": l2_note,
                   "paper_context": "GTX860M OpenGL 0.90, i7 8 threads 0.036 Gvoxel-iter/s (PAPER.md:408-414)", **extra},
        "roofline": roof,
        "cpu_baseline": {"value": cpu_v, "unit": unit, "cores": cores, "kind": "oracle", "sample": sample,
                         "single_thread": cpu_1, "cpu_model": cpu_model()},
        "e2e": {"value": e2e_value, "unit": unit, "h2d_bytes_per_step": N * 4, "d2h_bytes_per_step": N * 4,
                "api": "idg_filter_host (pinned host buffers)", "floor": e2e_floor},
        "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks,
    }
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
    ap.add_argument("--kernel", type=int, default=0, help="IDG_OPT_KERNEL (0 = library default plan)")
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
