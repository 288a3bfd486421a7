"""oracle/ -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain fp64 CPU oracles for the intensity-driven gradient filter (PAPER.md:165-189,
section 3.3, Eq. 6-7) and for the box and Gaussian reference filters (PAPER.md:121-159,
sections 3.1-3.2, Eq. 1-3), written from the paper and independent of the CUDA path:
it imports nothing from ``paper_1609_03782_b200`` and the package imports nothing
from here.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may use it.

The arithmetic lives in ``idg_oracle.c`` (plain C, compiled by ``build()`` with
gcc); this module is the ctypes loader and argument marshalling only.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "idg_oracle.c"), os.path.join(_HERE, "ref_filters_oracle.c"),
        os.path.join(_HERE, "wavelet_oracle.c")]
_LIB = os.path.join(_HERE, "libidg_oracle.so")
_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """Compile the oracle's C sources into ``oracle/libidg_oracle.so`` (gcc, -O2, OpenMP)."""
    srcs = [s for s in _SRC if os.path.exists(s)]
    newest = max(os.path.getmtime(s) for s in srcs)
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
               "-ffp-contract=off", "-o", _LIB] + srcs + ["-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        lib.idg_oracle_f64.restype = ctypes.c_int
        lib.idg_oracle_f64.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                       ctypes.c_double, ctypes.c_double, ctypes.c_double, dp, dp]
        lib.idg_oracle_set_threads.restype = ctypes.c_int
        lib.idg_oracle_set_threads.argtypes = [ctypes.c_int]
        i_ = ctypes.c_int
        lib.wavelet_forward_oracle.restype = i_
        lib.wavelet_forward_oracle.argtypes = [dp, i_, i_, i_, i_, i_]
        lib.wavelet_inverse_oracle.restype = i_
        lib.wavelet_inverse_oracle.argtypes = [dp, i_, i_, i_, i_, i_]
        lib.wavelet_filter_oracle.restype = i_
        lib.wavelet_filter_oracle.argtypes = [dp, i_, i_, i_, i_, i_, dp, ctypes.c_double, dp]
        lib.pm_oracle_f64.restype = ctypes.c_int
        lib.pm_oracle_f64.argtypes = lib.idg_oracle_f64.argtypes
        ip = ctypes.POINTER(ctypes.c_int)
        lib.box_oracle_f64.restype = ctypes.c_int
        lib.box_oracle_f64.argtypes = [dp] + [ctypes.c_int] * 6 + [dp]
        lib.gaussian_radii_oracle.restype = ctypes.c_int
        lib.gaussian_radii_oracle.argtypes = [dp, dp, ip]
        lib.gaussian_kernel_oracle.restype = ctypes.c_int
        lib.gaussian_kernel_oracle.argtypes = [dp, dp, ip, dp]
        lib.gaussian_oracle_f64.restype = ctypes.c_int
        lib.gaussian_oracle_f64.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp]
        _lib = lib
    return _lib


def set_threads(n: int) -> int:
    """Set the OpenMP thread count of the oracle (timing only); returns the count in effect."""
    return int(_load().idg_oracle_set_threads(int(n)))


def idg_filter_oracle(cube: np.ndarray, n_iter: int, K: float = 1.5, tau: float = 0.0325,
                      cx: float = 5.0, cy: float = 5.0, cz: float = 5.0,
                      rms: float = 1.0) -> np.ndarray:
    """n_iter IDG updates (Eq. 7) of ``cube[z, y, x]`` in fp64.

    ``cube`` is indexed [z][y][x] (x = RA fastest); its values are
    converted exactly to fp64.  Parameters are used as the fp64 values given: callers
    comparing against the fp32 GPU path pass the fp32-rounded values (``np.float32(p)``)
    so both sides evaluate the same function.  Returns a new fp64 array.
    """
    a = np.ascontiguousarray(cube, dtype=np.float64)
    if a.ndim != 3:
        raise ValueError("cube must be 3-D [nz, ny, nx]")
    nz, ny, nx = a.shape
    out = np.empty_like(a)
    scratch = np.empty_like(a)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = _load().idg_oracle_f64(a.ctypes.data_as(dp), nx, ny, nz, int(n_iter),
                                float(K), float(tau), float(cx), float(cy), float(cz),
                                float(rms), out.ctypes.data_as(dp), scratch.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError(f"idg_oracle_f64 rejected its arguments (rc={rc})")
    return out


def idg_filter_oracle_into(a64: np.ndarray, n_iter: int, out: np.ndarray, scratch: np.ndarray, K: float = 1.5,
                           tau: float = 0.0325, cx: float = 5.0, cy: float = 5.0, cz: float = 5.0,
                           rms: float = 1.0) -> np.ndarray:
    """:func:`idg_filter_oracle` on caller-owned fp64 buffers (marshalling only, the same C routine): ``a64`` is the
    input already in fp64, ``out`` receives I_n, ``scratch`` is the second Jacobi buffer; all C-contiguous, same
    shape.  For timing the arithmetic without the conversion and the page faults of fresh multi-GB allocations."""
    for b in (a64, out, scratch):
        if b.dtype != np.float64 or not b.flags.c_contiguous or b.shape != a64.shape or b.ndim != 3:
            raise ValueError("buffers must be C-contiguous float64 arrays of one 3-D shape")
    nz, ny, nx = a64.shape
    dp = ctypes.POINTER(ctypes.c_double)
    rc = _load().idg_oracle_f64(a64.ctypes.data_as(dp), nx, ny, nz, int(n_iter), float(K), float(tau), float(cx),
                                float(cy), float(cz), float(rms), out.ctypes.data_as(dp), scratch.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError(f"idg_oracle_f64 rejected its arguments (rc={rc})")
    return out


def pm_filter_oracle(cube: np.ndarray, n_iter: int, K: float = 1.5, tau: float = 0.0325,
                     cx: float = 5.0, cy: float = 5.0, cz: float = 5.0, rms: float = 1.0) -> np.ndarray:
    """n_iter updates of the gradient-driven (Perona-Malik, Eq. 5) variant of Eq. 7 in fp64:
    conductance 1/(1 + |grad I|^2/(K^2 rms^2)) from central differences of the six neighbours."""
    a = np.ascontiguousarray(cube, dtype=np.float64)
    if a.ndim != 3:
        raise ValueError("cube must be 3-D [nz, ny, nx]")
    nz, ny, nx = a.shape
    out, scratch = np.empty_like(a), np.empty_like(a)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = _load().pm_oracle_f64(a.ctypes.data_as(dp), nx, ny, nz, int(n_iter), float(K), float(tau),
                               float(cx), float(cy), float(cz), float(rms), out.ctypes.data_as(dp),
                               scratch.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError(f"pm_oracle_f64 rejected its arguments (rc={rc})")
    return out


def _cube64(cube: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(cube, dtype=np.float64)
    if a.ndim != 3:
        raise ValueError("cube must be 3-D [nz, ny, nx]")
    return a


def _d3(v) -> "ctypes.Array":
    return (ctypes.c_double * 3)(*[float(t) for t in v])


def box_filter_oracle(cube: np.ndarray, wx: int, wy: int, wz: int) -> np.ndarray:
    """Box filter: mean over the wx x wy x wz neighbourhood (odd widths, x = RA) of
    ``cube[z, y, x]``; out-of-cube neighbours are the nearest in-cube voxel (reading F1)."""
    a = _cube64(cube)
    nz, ny, nx = a.shape
    out = np.empty_like(a)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = _load().box_oracle_f64(a.ctypes.data_as(dp), nx, ny, nz, int(wx), int(wy), int(wz),
                                out.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError(f"box_oracle_f64 rejected its arguments (rc={rc})")
    return out


def gaussian_radii_oracle(fwhm, theta=(0.0, 0.0, 0.0)) -> tuple:
    """Support radii (rx, ry, rz) of the sampled kernel (reading F3)."""
    r = (ctypes.c_int * 3)()
    if _load().gaussian_radii_oracle(_d3(fwhm), _d3(theta), r) != 0:
        raise ValueError("invalid Gaussian parameters")
    return int(r[0]), int(r[1]), int(r[2])


def gaussian_kernel_oracle(fwhm, theta=(0.0, 0.0, 0.0)) -> np.ndarray:
    """The normalised kernel of Eq. 1-3 as an array [2rz+1, 2ry+1, 2rx+1]; fwhm = (x, y, z) in voxels,
    theta = (theta_x, theta_y, theta_z) in degrees."""
    rx, ry, rz = gaussian_radii_oracle(fwhm, theta)
    k = np.empty((2 * rz + 1, 2 * ry + 1, 2 * rx + 1), dtype=np.float64)
    r = (ctypes.c_int * 3)(rx, ry, rz)
    dp = ctypes.POINTER(ctypes.c_double)
    if _load().gaussian_kernel_oracle(_d3(fwhm), _d3(theta), r, k.ctypes.data_as(dp)) != 0:
        raise ValueError("invalid Gaussian parameters")
    return k


def gaussian_filter_oracle(cube: np.ndarray, fwhm, theta=(0.0, 0.0, 0.0)) -> np.ndarray:
    """Gaussian filter (Eq. 1-3): direct 3-D convolution of ``cube[z, y, x]`` with the
    kernel of :func:`gaussian_kernel_oracle`; replicated faces (reading F1)."""
    a = _cube64(cube)
    nz, ny, nx = a.shape
    out = np.empty_like(a)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = _load().gaussian_oracle_f64(a.ctypes.data_as(dp), nx, ny, nz, _d3(fwhm), _d3(theta),
                                     out.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError(f"gaussian_oracle_f64 rejected its arguments (rc={rc})")
    return out


HAAR, LEGALL = 0, 1


def wavelet_transform_oracle(cube: np.ndarray, wavelet: int, levels: int, inverse: bool = False) -> np.ndarray:
    """Forward (or inverse) lifting transform to `levels` (Eq. 8-11), coefficients
    interleaved in place: c at even, d at odd lattice positions.  wavelet: HAAR or LEGALL."""
    a = np.array(cube, dtype=np.float64, order="C", copy=True)
    if a.ndim != 3:
        raise ValueError("cube must be 3-D [nz, ny, nx]")
    nz, ny, nx = a.shape
    dp = ctypes.POINTER(ctypes.c_double)
    fn = _load().wavelet_inverse_oracle if inverse else _load().wavelet_forward_oracle
    if fn(a.ctypes.data_as(dp), nx, ny, nz, int(wavelet), int(levels)) != 0:
        raise ValueError("wavelet oracle rejected its arguments")
    return a


def wavelet_filter_oracle(cube: np.ndarray, wavelet: int, thresholds, rms: float = 1.0) -> np.ndarray:
    """Wavelet thresholding filter: decompose to len(thresholds) levels, zero every
    coefficient with |v| < t_l * rms (detail bands of level l, approximation band with t_L), transform back."""
    a = _cube64(cube)
    nz, ny, nx = a.shape
    out = np.empty_like(a)
    t = np.ascontiguousarray(thresholds, dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = _load().wavelet_filter_oracle(a.ctypes.data_as(dp), nx, ny, nz, int(wavelet), int(t.size),
                                       t.ctypes.data_as(dp), float(rms), out.ctypes.data_as(dp))
    if rc != 0:
        raise ValueError(f"wavelet_filter_oracle rejected its arguments (rc={rc})")
    return out
