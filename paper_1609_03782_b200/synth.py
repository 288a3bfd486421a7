"""Seeded synthetic HI cubes standing in for the paper's data.

This module serves BOTH the CUDA path and the oracle with inputs and holds none
of the filter's arithmetic: it only draws noise, evaluates a toy galaxy model and
returns fp32 cubes indexed [z (velocity)][y (Dec)][x (RA)].  The recipe (DESIGN.md
section 4) follows the paper's ModelA/B/C description: Gaussian noise of rms 1,
correlated spatially by the 88"x70" beam on 20" pixels (4.4 x 3.5 px FWHM),
independent per 8.25 km/s channel, plus an inclined rotating exponential disc, a
companion and a faint tidal tail.  numpy/scipy only; deterministic per seed and
independent of the thread count.
"""
from __future__ import annotations

import math
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np
from scipy import ndimage

FWHM_TO_SIGMA = 1.0 / (2.0 * math.sqrt(2.0 * math.log(2.0)))   # PAPER.md:142 (Eq. 2)
BEAM_FWHM_X = 4.4       # px along RA   (88" / 20")
BEAM_FWHM_Y = 3.5       # px along Dec  (70" / 20")
CHANNEL_KMS = 8.25
SIGMA_V_KMS = 10.0


@dataclass
class Disc:
    """Inclined, rotating exponential disc (one emission component)."""
    x0: float
    y0: float
    z0: float
    h: float = 12.0            # scale length [px]
    incl_deg: float = 50.0
    pa_rad: float = 0.0
    vrot: float = 150.0        # flat rotation [km/s]
    vsys: float = 0.0          # offset from channel z0 [km/s]
    sigma_v: float = SIGMA_V_KMS
    amp: float = 1.0           # central brightness before beam convolution
    q_floor: float = 0.0       # intrinsic flattening (thick disc): q = sqrt(cos^2 i + q0^2 sin^2 i)


@dataclass
class Tail:
    """Straight faint filament between two points (x, y, v_kms relative to channel z0)."""
    p0: Tuple[float, float, float]
    p1: Tuple[float, float, float]
    z0: float
    width: float = 2.0
    sigma_v: float = SIGMA_V_KMS
    snr: float = 1.0           # beam-convolved peak S/N of the tail ("peak S/N 1")


@dataclass
class Source:
    """Components scaled together so that the beam-convolved peak equals `peak_snr`."""
    peak_snr: float
    discs: List[Disc] = field(default_factory=list)
    tails: List[Tail] = field(default_factory=list)


def _threads(n: Optional[int]) -> int:
    return max(1, n if n else min(16, os.cpu_count() or 1))


def beam_noise(shape: Sequence[int], seed: int, threads: Optional[int] = None) -> np.ndarray:
    """rms-1 Gaussian noise, beam-correlated in (y, x), independent per channel z. fp32 [nz,ny,nx]."""
    nz, ny, nx = (int(s) for s in shape)
    sx, sy = BEAM_FWHM_X * FWHM_TO_SIGMA, BEAM_FWHM_Y * FWHM_TO_SIGMA
    fx = np.fft.rfftfreq(nx)[None, :]
    fy = np.fft.fftfreq(ny)[:, None]
    H = np.exp(-2.0 * math.pi ** 2 * (sx * sx * fx * fx + sy * sy * fy * fy))   # periodic Gaussian beam
    out = np.empty((nz, ny, nx), dtype=np.float32)
    s1 = np.zeros(nz)
    s2 = np.zeros(nz)

    def one(z: int) -> None:
        rng = np.random.default_rng([int(seed), 0x6E6F6973, z])
        w = rng.standard_normal((ny, nx))
        c = np.fft.irfft2(np.fft.rfft2(w) * H, s=(ny, nx))
        s1[z] = c.sum()
        s2[z] = (c * c).sum()
        out[z] = c

    with ThreadPoolExecutor(_threads(threads)) as ex:
        list(ex.map(one, range(nz)))
    n = float(nz) * ny * nx
    mean = s1.sum() / n
    std = math.sqrt(max(s2.sum() / n - mean * mean, 1e-300))
    out *= np.float32(1.0 / std)
    return out


def _disc_box(d: Disc, shape: Sequence[int]) -> Tuple[slice, slice, slice]:
    nz, ny, nx = shape
    r = 8.0 * d.h + 3 * BEAM_FWHM_X
    dv = (abs(d.vrot) + abs(d.vsys) + 4.5 * d.sigma_v) / CHANNEL_KMS + 1
    lo = lambda c, e, n: int(max(0, math.floor(c - e)))
    hi = lambda c, e, n: int(min(n, math.ceil(c + e) + 1))
    return (slice(lo(d.z0, dv, nz), hi(d.z0, dv, nz)),
            slice(lo(d.y0, r, ny), hi(d.y0, r, ny)),
            slice(lo(d.x0, r, nx), hi(d.x0, r, nx)))


def _eval_disc(d: Disc, box: Tuple[slice, slice, slice]) -> np.ndarray:
    zs, ys, xs = box
    z = np.arange(zs.start, zs.stop, dtype=np.float64)[:, None, None]
    y = np.arange(ys.start, ys.stop, dtype=np.float64)[None, :, None] - d.y0
    x = np.arange(xs.start, xs.stop, dtype=np.float64)[None, None, :] - d.x0
    cp, sp = math.cos(d.pa_rad), math.sin(d.pa_rad)
    xr = cp * x + sp * y            # along the major axis
    yr = -sp * x + cp * y           # along the minor axis
    inc = math.radians(d.incl_deg)
    q = math.sqrt(math.cos(inc) ** 2 + (d.q_floor * math.sin(inc)) ** 2)
    R = np.sqrt(xr * xr + (yr / q) ** 2)
    sigma = np.exp(-R / d.h)
    with np.errstate(invalid="ignore", divide="ignore"):
        cosphi = np.where(R > 0, xr / R, 0.0)
    vlos = d.vsys + d.vrot * math.sin(inc) * cosphi
    vz = (z - d.z0) * CHANNEL_KMS
    return d.amp * sigma * np.exp(-0.5 * ((vz - vlos) / d.sigma_v) ** 2)


def _tail_box(t: Tail, shape: Sequence[int]) -> Tuple[slice, slice, slice]:
    nz, ny, nx = shape
    e = 4 * t.width + 3 * BEAM_FWHM_X
    xs = (min(t.p0[0], t.p1[0]) - e, max(t.p0[0], t.p1[0]) + e)
    ys = (min(t.p0[1], t.p1[1]) - e, max(t.p0[1], t.p1[1]) + e)
    ev = 4.5 * t.sigma_v
    zs = (t.z0 + (min(t.p0[2], t.p1[2]) - ev) / CHANNEL_KMS, t.z0 + (max(t.p0[2], t.p1[2]) + ev) / CHANNEL_KMS)
    c = lambda a, n: (int(max(0, math.floor(a[0]))), int(min(n, math.ceil(a[1]) + 1)))
    return slice(*c(zs, nz)), slice(*c(ys, ny)), slice(*c(xs, nx))


def _eval_tail(t: Tail, box: Tuple[slice, slice, slice]) -> np.ndarray:
    zs, ys, xs = box
    z = np.arange(zs.start, zs.stop, dtype=np.float64)[:, None, None]
    y = np.arange(ys.start, ys.stop, dtype=np.float64)[None, :, None]
    x = np.arange(xs.start, xs.stop, dtype=np.float64)[None, None, :]
    ax, ay = t.p1[0] - t.p0[0], t.p1[1] - t.p0[1]
    L2 = max(ax * ax + ay * ay, 1e-12)
    s = np.clip(((x - t.p0[0]) * ax + (y - t.p0[1]) * ay) / L2, 0.0, 1.0)   # position along the segment
    dx, dy = x - (t.p0[0] + s * ax), y - (t.p0[1] + s * ay)
    prof = np.exp(-0.5 * (dx * dx + dy * dy) / (t.width ** 2))
    vlos = t.p0[2] + s * (t.p1[2] - t.p0[2])
    vz = (z - t.z0) * CHANNEL_KMS
    return prof * np.exp(-0.5 * ((vz - vlos) / t.sigma_v) ** 2)


def _beam_smooth(a: np.ndarray) -> np.ndarray:
    sx, sy = BEAM_FWHM_X * FWHM_TO_SIGMA, BEAM_FWHM_Y * FWHM_TO_SIGMA
    a = ndimage.gaussian_filter1d(a, sx, axis=2, mode="constant", truncate=4.0)
    return ndimage.gaussian_filter1d(a, sy, axis=1, mode="constant", truncate=4.0)


def _union(boxes: List[Tuple[slice, slice, slice]]) -> Tuple[slice, slice, slice]:
    return tuple(slice(min(b[k].start for b in boxes), max(b[k].stop for b in boxes)) for k in range(3))


def add_source(model: np.ndarray, src: Source) -> float:
    """Add one source (discs scaled to peak_snr; each tail scaled to its own peak) in place.

    Returns the source's beam-convolved peak.
    """
    shape = model.shape
    if src.discs:
        boxes = [_disc_box(d, shape) for d in src.discs]
        ub = _union(boxes)
        acc = np.zeros(tuple(s.stop - s.start for s in ub))
        for d, b in zip(src.discs, boxes):
            rel = tuple(slice(b[k].start - ub[k].start, b[k].stop - ub[k].start) for k in range(3))
            acc[rel] += _eval_disc(d, b)
        acc = _beam_smooth(acc)
        m = float(acc.max())
        if m > 0:
            model[ub] += (acc * (src.peak_snr / m)).astype(np.float32)
    for t in src.tails:
        b = _tail_box(t, shape)
        if any(s.stop <= s.start for s in b):
            continue
        a = _beam_smooth(_eval_tail(t, b))
        m = float(a.max())
        if m > 0:
            model[b] += (a * (t.snr / m)).astype(np.float32)
    return src.peak_snr


# --------------------------------------------------------------------------------------
# BASELINE.json configs
# --------------------------------------------------------------------------------------

@dataclass
class Cube:
    data: np.ndarray            # fp32 [nz, ny, nx] = noise + model
    model: Optional[np.ndarray]  # fp32 noiseless model (None when keep_model=False)
    rms: float                  # noise rms of `data` (1.0 by construction)
    peak: float                 # max |data| / rms (keep < 64 for n = 40 runs)


def _finish(noise: np.ndarray, model: np.ndarray, keep_model: bool) -> Cube:
    noise += model
    peak = float(np.abs(noise).max())
    return Cube(noise, model if keep_model else None, 1.0, peak)


def _modelb_source(shape: Sequence[int], rng: np.random.Generator, snr: float) -> Source:
    """Disc + companion (1/5 mass, 35 px away) + tail of peak S/N 1 (BASELINE.json configs[0])."""
    nz, ny, nx = shape
    h = 12.0
    ang = rng.uniform(0.0, 2.0 * math.pi)
    x0 = nx / 2.0 - 0.35 * 35.0 * math.cos(ang)
    y0 = ny / 2.0 - 0.35 * 35.0 * math.sin(ang)
    z0 = (nz - 1) / 2.0
    main = Disc(x0, y0, z0, h=h, incl_deg=50.0, pa_rad=rng.uniform(0, math.pi), vrot=150.0)
    xc, yc = x0 + 35.0 * math.cos(ang), y0 + 35.0 * math.sin(ang)
    comp = Disc(xc, yc, z0, h=h / math.sqrt(5.0), incl_deg=50.0, pa_rad=rng.uniform(0, math.pi),
                vrot=100.0, vsys=40.0)
    tail = Tail((x0, y0, 0.0), (xc, yc, 40.0), z0, width=2.0, snr=1.0)
    return Source(snr, [main, comp], [tail])


def modelb_like(shape: Sequence[int] = (67, 100, 100), seed: int = 1000, snr: float = 32.0,
                keep_model: bool = True, threads: Optional[int] = None) -> Cube:
    """configs[0]/[1]/[4]: ModelA/B/C-like cube; shape is (nz, ny, nx)."""
    rng = np.random.default_rng([int(seed), 0x6D6F646C])
    model = np.zeros(tuple(shape), dtype=np.float32)
    add_source(model, _modelb_source(shape, rng, snr))
    return _finish(beam_noise(shape, seed, threads), model, keep_model)


def _field_sources(shape: Sequence[int], rng: np.random.Generator, n_discs: int,
                   thick: bool) -> List[Source]:
    nz, ny, nx = shape
    out: List[Source] = []
    for _ in range(n_discs):
        h = rng.uniform(8.0, 20.0)
        m = 3.0 * h
        x0, y0 = rng.uniform(m, nx - m), rng.uniform(m, ny - m)
        z0 = rng.uniform(0.25 * nz, 0.75 * nz)
        incl = rng.uniform(20.0, 80.0)
        pa = rng.uniform(0.0, math.pi)
        v = rng.uniform(80.0, 220.0)
        snr = math.exp(rng.uniform(math.log(5.0), math.log(40.0)))
        d = Disc(x0, y0, z0, h=h, incl_deg=incl, pa_rad=pa, vrot=v)
        L, a = rng.uniform(30.0, 50.0), rng.uniform(0.0, 2.0 * math.pi)
        t = Tail((x0, y0, 0.0), (x0 + L * math.cos(a), y0 + L * math.sin(a), rng.uniform(-40.0, 40.0)),
                 z0, width=2.0, snr=rng.uniform(0.5, 1.0))
        out.append(Source(snr, [d], [t]))
        if thick:   # extra-planar gas: thick, lagging, low-S/N component (BASELINE.json configs[3])
            out.append(Source(1.0, [Disc(x0, y0, z0, h=1.5 * h, incl_deg=incl, pa_rad=pa,
                                         vrot=0.8 * v, sigma_v=25.0, q_floor=0.3)], []))
    return out


def survey_field(shape: Sequence[int] = (256, 512, 512), seed: int = 2000, n_discs: int = 6,
                 thick: bool = False, keep_model: bool = False,
                 threads: Optional[int] = None) -> Cube:
    """configs[2] (6 discs) and configs[3] (shape (512,1024,1024), 20 discs, thick=True)."""
    rng = np.random.default_rng([int(seed), 0x6669656C])
    model = np.zeros(tuple(shape), dtype=np.float32)
    for s in _field_sources(shape, rng, n_discs, thick):
        add_source(model, s)
    return _finish(beam_noise(shape, seed, threads), model, keep_model)


def large_cube(seed: int = 3000, shape: Sequence[int] = (512, 1024, 1024),
               threads: Optional[int] = None) -> Cube:
    """configs[3]: 1024x1024x512, noise-dominated, 20 discs + extra-planar gas."""
    return survey_field(shape, seed, n_discs=20, thick=True, keep_model=False, threads=threads)


K_SWEEP = (0.5, 1.0, 1.5, 2.0, 3.0, 5.0, 7.5, 10.0)     # configs[1]; PAPER.md:187 range, :285 grid
TAU_SET = (0.0125, 0.0225, 0.0325)
C_SET = (4.0, 5.0, 6.0)                                  # PAPER.md:287-314 (Table 1 best C_j)


def batch_params(batch: int = 256, seed: int = 4000) -> np.ndarray:
    """configs[4] per-cube parameters, rows (K, tau, cx, cy, cz, rms), with tau*(cx+cy+cz) <= 0.5."""
    rng = np.random.default_rng([int(seed), 0x70617261])
    out = np.empty((batch, 6), dtype=np.float32)
    for b in range(batch):
        while True:
            K = K_SWEEP[rng.integers(len(K_SWEEP))]
            tau = TAU_SET[rng.integers(len(TAU_SET))]
            c = [C_SET[rng.integers(len(C_SET))] for _ in range(3)]
            if tau * sum(c) <= 0.5:
                break
        out[b] = (K, tau, c[0], c[1], c[2], 1.0)
    return out


def batch_cubes(batch: int = 256, seed: int = 4000, shape: Sequence[int] = (64, 128, 128),
                threads: Optional[int] = None) -> np.ndarray:
    """configs[4]: `batch` independent cubes (seeds seed+b, S/N uniform in [10, 60]). fp32 [B,nz,ny,nx]."""
    out = np.empty((batch,) + tuple(shape), dtype=np.float32)
    rng = np.random.default_rng([int(seed), 0x736E7273])
    snrs = rng.uniform(10.0, 60.0, size=batch)

    def one(b: int) -> None:
        out[b] = modelb_like(shape, seed + b, float(snrs[b]), keep_model=False, threads=1).data

    with ThreadPoolExecutor(_threads(threads)) as ex:
        list(ex.map(one, range(batch)))
    return out
