"""oracle/quality_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy statement of the paper's smoothing-quality diagnostics (Eq. 12-16, and
PAPER.md:344-355, Eq. 17-18), written from the paper only; same access rules as the rest of oracle/.

    M_i(x,y,z) = 1 if I_i >= 3 rms_i else 0,  i = o (original), f (filtered)          (Eq. 14)
    S_oo = sum I_o M_o,   S_of = sum I_o M_f     (sums over a ROI sub-cube)            (Eq. 13)
    F    = |S_of| / |S_oo|                                                             (Eq. 12)
    sigma_S_oi = sqrt(N_i) rms_i,  N_i = independent voxels in M_i                     (Eq. 16)
    sigma_F = sqrt(sigma_S_of^2 / S_oo^2 + S_of^2 sigma_S_oo^2 / S_oo^4)               (Eq. 15)
    S_mf = sum I_m M_f,   S_m = sum I_m,   F_M = |S_mf| / |S_m|   (I_m = noiseless model)  (Eq. 17-18)

Readings where the paper is silent (Q1-Q4):
  Q1  the threshold 3 rms_i is passed in as an fp32 number per cube and compared with the fp32 voxel
      (I >= thr, NaN voxels never pass), so the mask is decided in the cube's own precision;
  Q2  the ROI is a half-open index box [x0,x1) x [y0,y1) x [z0,z1); sums are accumulated in fp64;
  Q3  "independent voxels": N_i = (voxels in M_i) / voxels_per_beam, voxels_per_beam >= 1 supplied by
      the caller (1 = every voxel independent);
  Q4  the noise level of a cube is estimated as the standard deviation about the mean over a
      (signal-free) ROI: rms = sqrt(sum x^2 / n - (sum x / n)^2).
"""
from __future__ import annotations

import math
from typing import Optional, Sequence

import numpy as np


def _roi(shape, roi: Optional[Sequence[int]]):
    nz, ny, nx = shape
    if roi is None:
        return slice(0, nz), slice(0, ny), slice(0, nx)
    x0, x1, y0, y1, z0, z1 = (int(v) for v in roi)
    if not (0 <= x0 <= x1 <= nx and 0 <= y0 <= y1 <= ny and 0 <= z0 <= z1 <= nz):
        raise ValueError("ROI outside the cube")
    return slice(z0, z1), slice(y0, y1), slice(x0, x1)


def mask_sums_oracle(orig: np.ndarray, filt: np.ndarray, model: Optional[np.ndarray], thr_o: float,
                     thr_f: float, roi: Optional[Sequence[int]] = None) -> dict:
    """The sums of Eq. 13 and 18 and the mask populations over the ROI; cubes are [z, y, x] fp32."""
    o = np.asarray(orig, dtype=np.float32)
    f = np.asarray(filt, dtype=np.float32)
    if o.shape != f.shape or o.ndim != 3:
        raise ValueError("orig and filt must be 3-D cubes of equal shape")
    s = _roi(o.shape, roi)
    o, f = o[s], f[s]
    m_o = o >= np.float32(thr_o)                                   # Eq. 14, reading Q1
    m_f = f >= np.float32(thr_f)
    o64 = o.astype(np.float64)
    out = {"S_oo": float(o64[m_o].sum()), "S_of": float(o64[m_f].sum()),
           "N_o": int(m_o.sum()), "N_f": int(m_f.sum()), "n_roi": int(o.size), "S_mf": 0.0, "S_m": 0.0}
    if model is not None:
        m = np.asarray(model, dtype=np.float32)[s].astype(np.float64)
        out["S_mf"] = float(m[m_f].sum())                          # Eq. 18
        out["S_m"] = float(m.sum())
    return out


def quality_oracle(sums: dict, rms_o: float, rms_f: float, voxels_per_beam: float = 1.0) -> dict:
    """F (Eq. 12), sigma_F (Eq. 15-16) and F_M (Eq. 17) from the sums."""
    S_oo, S_of = sums["S_oo"], sums["S_of"]
    F = abs(S_of) / abs(S_oo) if S_oo != 0.0 else math.nan
    sig_of = math.sqrt(sums["N_f"] / voxels_per_beam) * rms_f      # Eq. 16, reading Q3
    sig_oo = math.sqrt(sums["N_o"] / voxels_per_beam) * rms_o
    sigma_F = (math.sqrt(sig_of ** 2 / S_oo ** 2 + S_of ** 2 * sig_oo ** 2 / S_oo ** 4)
               if S_oo != 0.0 else math.nan)                        # Eq. 15
    F_M = abs(sums["S_mf"]) / abs(sums["S_m"]) if sums["S_m"] != 0.0 else math.nan
    return {"F": F, "sigma_F": sigma_F, "F_M": F_M}


def cube_stats_oracle(cube: np.ndarray, roi: Optional[Sequence[int]] = None) -> dict:
    """n, sum, sum of squares (fp64) over the ROI and the rms estimate of reading Q4."""
    a = np.asarray(cube, dtype=np.float32)
    a = a[_roi(a.shape, roi)].astype(np.float64)
    n, s1, s2 = int(a.size), float(a.sum()), float((a * a).sum())
    rms = math.sqrt(max(s2 / n - (s1 / n) ** 2, 0.0)) if n else math.nan
    return {"n": n, "sum": s1, "sumsq": s2, "rms": rms}


def histogram_oracle(cube: np.ndarray, lo: float, hi: float, nbins: int,
                     roi: Optional[Sequence[int]] = None, mask_thr: Optional[float] = None) -> np.ndarray:
    """Histogram of the voxel intensities of a ROI sub-cube (Fig. 6; the F-versus-threshold
    scan of PAPER.md:342 needs it).  Reading Q5: nbins equal bins over [lo, hi); the bin of a voxel is decided
    in fp32 like the mask of Eq. 14: b = floor((v - lo) * (nbins / (hi - lo))) with every operand and operation
    in fp32; voxels outside [lo, hi) and NaN are not counted; with mask_thr only voxels v >= mask_thr count."""
    a = np.asarray(cube, dtype=np.float32)
    a = a[_roi(a.shape, roi)].ravel()
    lo32, hi32 = np.float32(lo), np.float32(hi)
    if not (hi32 > lo32) or nbins < 1:
        raise ValueError("need hi > lo and nbins >= 1")
    scale = np.float32(np.float32(nbins) / np.float32(hi32 - lo32))
    counts = np.zeros(int(nbins), dtype=np.int64)
    keep = (a >= lo32) & (a < hi32)
    if mask_thr is not None:
        keep &= a >= np.float32(mask_thr)
    v = a[keep]
    b = np.floor((v - lo32).astype(np.float32) * scale).astype(np.int64)
    b = np.minimum(b, nbins - 1)                         # (v - lo) * scale can round up to nbins just below hi
    np.add.at(counts, b, 1)
    return counts
