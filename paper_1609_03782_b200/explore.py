"""Parameter exploration on the GPU: the paper's use of the filter (Table 3, Fig. 9).

    python -m paper_1609_03782_b200.explore [--snr 22] [--seed 1001] [--nmax 40] [--filter idg|pm]

For a ModelB-like synthetic cube (BASELINE.json configs[1]) the intensity-driven gradient filter is run for
every K of the sweep -- all K as one batched call with per-cube parameters -- up to n = nmax, incrementally from one
reported n to the next (f(I, n+m) = f(f(I, n), m), DESIGN.md pin P11; the iterations in between are fused on the
device), and at every reported n the quality diagnostics are evaluated on the device: rms of the filtered cube over signal-free
channels (idg_cube_stats), the masked sums over the ROI (idg_mask_sums) and F, sigma_F, F_M (idg_quality,
Eq. 12-18).  Prints one line per (K, n) of interest and the best run by F, like Table 1 / Table 3 of the paper.
Everything numerical runs in the library's CUDA kernels; this module only marshals arguments.
"""
from __future__ import annotations

import argparse
import math

import numpy as np
import torch

from . import binding as B
from . import synth


def explore(snr: float = 22.0, seed: int = 1001, nmax: int = 40, variant: str = "idg", ks=synth.K_SWEEP,
            report=(1, 5, 10, 20, 30, 40)) -> list:
    """Returns rows {K, n, rms_f, F, sigma_F, F_M}.  ROI: the whole field in x, y, the channels with signal;
    noise estimate: the first 8 channels (signal-free in this generator)."""
    B.lib()
    c = synth.modelb_like(seed=seed, snr=snr)
    nz, ny, nx = c.data.shape
    orig = torch.from_numpy(c.data).cuda()
    model = torch.from_numpy(c.model).cuda()
    noise_roi = (0, nx, 0, ny, 0, 8)
    chan = np.abs(c.model).reshape(nz, -1).max(axis=1) > 0.05 * np.abs(c.model).max()
    z0, z1 = int(np.argmax(chan)), int(nz - np.argmax(chan[::-1]))
    roi = (0, nx, 0, ny, z0, z1)
    # all K values as ONE batch (idg_filter_batched, per-cube parameters), and the iterations between two reported n in
    # one call (fused on the device): f(I, n + m) = f(f(I, n), m), DESIGN.md pin P11
    ks = [float(K) for K in ks]
    plist = [B.Params(K=K, rms=float(c.rms)) for K in ks]
    cur = orig.unsqueeze(0).repeat(len(ks), 1, 1, 1).contiguous()
    ws = B.alloc_workspace(nx, ny, nz, len(ks))
    sums = torch.empty(8, dtype=torch.float64, device="cuda")
    stats = torch.empty(8, dtype=torch.float64, device="cuda")
    rows, done = [], 0
    for n in sorted(m for m in set(report) | {nmax} if 1 <= m <= nmax):
        step = B.idg_filter_pm_batched if variant == "pm" else B.idg_filter_batched
        step(cur, n - done, plist, out=cur, workspace=ws)
        done = n
        if n not in report:
            continue
        for b, K in enumerate(ks):
            st = B.idg_cube_stats(cur[b], noise_roi, stats).cpu().numpy()
            rms_f = B.idg_stats_rms(st)[1]
            s = B.idg_mask_sums(orig, cur[b], model, 3.0 * c.rms, 3.0 * rms_f, roi, sums).cpu().numpy()
            q = B.idg_quality(s, c.rms, rms_f)
            rows.append({"K": K, "n": n, "rms_f": rms_f, **q})
    rows.sort(key=lambda r: (r["K"], r["n"]))
    return rows


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--snr", type=float, default=22.0)
    ap.add_argument("--seed", type=int, default=1001)
    ap.add_argument("--nmax", type=int, default=40)
    ap.add_argument("--filter", default="idg", choices=["idg", "pm"])
    a = ap.parse_args()
    rows = explore(a.snr, a.seed, a.nmax, a.filter)
    print(f"{'K':>5} {'n':>3} {'rms_f':>8} {'F':>8} {'sigma_F':>8} {'F_M':>7}")
    for r in rows:
        print(f"{r['K']:5.1f} {r['n']:3d} {r['rms_f']:8.4f} {r['F']:8.4f} {r['sigma_F']:8.4f} {r['F_M']:7.4f}")
    best = max(rows, key=lambda r: r["F"])
    print(f"best by F: K = {best['K']}, n = {best['n']}: F = {best['F']:.4f} +- {best['sigma_F']:.4f}, "
          f"F_M = {best['F_M']:.4f}")


if __name__ == "__main__":
    main()
