"""ctypes binding of libidg_b200.so (include/idg.h): argument marshalling only.

Same names as the C ABI.  torch supplies device memory and streams; every voxel
update runs in the library's CUDA kernels.  There is no CPU path: a missing
library or a CPU tensor raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence, Union

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libidg_b200.so")

IDG_OPT_KERNEL, IDG_OPT_FUSE, IDG_OPT_ZCHUNK, IDG_OPT_TILE, IDG_OPT_CTAS, IDG_OPT_HOST_SLABS, IDG_OPT_COOP = 0, 1, 2, 3, 4, 5, 6
KERNEL_AUTO, KERNEL_NAIVE, KERNEL_TILED, KERNEL_TMA, KERNEL_STREAM, KERNEL_RESIDENT = 0, 1, 2, 3, 4, 5

# every symbol include/idg.h declares (tests check the library exports them all)
SYMBOLS = ("idg_version", "idg_status_string", "idg_params_check", "idg_workspace_bytes",
           "idg_filter", "idg_filter_ws", "idg_filter_batched", "idg_filter_host",
           "idg_set_option", "idg_get_option", "idg_last_launch_count", "idg_last_plan",
           "idg_box_filter", "idg_gaussian_filter", "idg_gaussian_radii",
           "idg_mask_sums", "idg_cube_stats", "idg_quality", "idg_filter_pm",
           "idg_wavelet_transform", "idg_wavelet_filter", "idg_histogram", "idg_release_temporaries", "idg_stats_rms", "idg_gaussian_filter_static", "idg_filter_pm_batched")
WAVELET_HAAR, WAVELET_LEGALL53 = 0, 1


class IdgParams(ctypes.Structure):
    """struct idg_params: K, tau, cx, cy, cz, rms -- all fp32."""
    _fields_ = [("K", ctypes.c_float), ("tau", ctypes.c_float), ("cx", ctypes.c_float),
                ("cy", ctypes.c_float), ("cz", ctypes.c_float), ("rms", ctypes.c_float)]


@dataclass
class Params:
    """Paper defaults: K = 1.5, tau = 0.0325, Cx = Cy = Cz = 5."""
    K: float = 1.5
    tau: float = 0.0325
    cx: float = 5.0
    cy: float = 5.0
    cz: float = 5.0
    rms: float = 1.0

    def c(self) -> IdgParams:
        return IdgParams(self.K, self.tau, self.cx, self.cy, self.cz, self.rms)

    def f32(self) -> dict:
        """The fp32-rounded values the library sees, as Python floats (for the oracle)."""
        return {k: float(np.float32(getattr(self, k))) for k in ("K", "tau", "cx", "cy", "cz", "rms")}


class IdgRoi(ctypes.Structure):
    """struct idg_roi: half-open index box [x0,x1) x [y0,y1) x [z0,z1)."""
    _fields_ = [(n, ctypes.c_int) for n in ("x0", "x1", "y0", "y1", "z0", "z1")]


class IdgError(RuntimeError):
    def __init__(self, status: int):
        self.status = status
        super().__init__(f"idg status {status}: {status_string(status)}")


_lib: Optional[ctypes.CDLL] = None


def lib() -> ctypes.CDLL:
    """Load libidg_b200.so; fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1609_03782_b200.build` "
                               "(the IDG filter has no CPU or PyTorch fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, fp, ip, sz, i = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int
        pp = ctypes.POINTER(IdgParams)
        L.idg_version.restype = i
        L.idg_status_string.restype = ctypes.c_char_p
        L.idg_status_string.argtypes = [i]
        L.idg_params_check.restype = ctypes.c_uint
        L.idg_params_check.argtypes = [pp]
        L.idg_workspace_bytes.restype = sz
        L.idg_workspace_bytes.argtypes = [i, i, i, i]
        L.idg_filter.restype = i
        L.idg_filter.argtypes = [fp, i, i, i, i, pp, fp, vp]
        L.idg_filter_ws.restype = i
        L.idg_filter_ws.argtypes = [fp, i, i, i, i, pp, fp, vp, sz, vp]
        L.idg_filter_pm.restype = i
        L.idg_filter_pm.argtypes = [fp, i, i, i, i, pp, fp, vp, sz, vp]
        L.idg_filter_batched.restype = i
        L.idg_filter_batched.argtypes = [fp, i, i, i, i, ip, i, pp, fp, vp, sz, vp]
        L.idg_filter_pm_batched.restype = i
        L.idg_filter_pm_batched.argtypes = [fp, i, i, i, i, ip, i, pp, fp, vp, sz, vp]
        L.idg_filter_host.restype = i
        L.idg_filter_host.argtypes = [fp, i, i, i, i, pp, fp, vp, sz, vp]
        L.idg_set_option.restype = i
        L.idg_set_option.argtypes = [i, i]
        L.idg_get_option.restype = i
        L.idg_get_option.argtypes = [i]
        L.idg_last_launch_count.restype = i
        L.idg_release_temporaries.restype = i
        L.idg_release_temporaries.argtypes = []
        L.idg_last_plan.restype = ctypes.c_char_p
        f = ctypes.c_float
        L.idg_box_filter.restype = i
        L.idg_box_filter.argtypes = [fp, i, i, i, i, i, i, fp, vp]
        L.idg_gaussian_filter.restype = i
        L.idg_gaussian_filter.argtypes = [fp, i, i, i, f, f, f, f, f, f, fp, vp]
        L.idg_gaussian_filter_static.restype = i
        L.idg_gaussian_filter_static.argtypes = [fp, i, i, i, f, f, f, f, f, f, fp, vp]
        L.idg_gaussian_radii.restype = i
        L.idg_gaussian_radii.argtypes = [f, f, f, f, f, f, ctypes.POINTER(ctypes.c_int)]
        rp, d, dptr = ctypes.POINTER(IdgRoi), ctypes.c_double, ctypes.POINTER(ctypes.c_double)
        L.idg_mask_sums.restype = i
        L.idg_mask_sums.argtypes = [fp, fp, fp, i, i, i, rp, f, f, vp, vp]
        L.idg_cube_stats.restype = i
        L.idg_cube_stats.argtypes = [fp, i, i, i, rp, vp, vp]
        L.idg_histogram.restype = i
        L.idg_histogram.argtypes = [fp, i, i, i, rp, f, f, i, ctypes.POINTER(ctypes.c_float), vp, vp]
        L.idg_stats_rms.restype = i
        L.idg_stats_rms.argtypes = [dptr, dptr, dptr]
        L.idg_quality.restype = i
        L.idg_quality.argtypes = [dptr, d, d, d, dptr, dptr, dptr]
        L.idg_wavelet_transform.restype = i
        L.idg_wavelet_transform.argtypes = [fp, i, i, i, i, i, i, fp, vp]
        L.idg_wavelet_filter.restype = i
        L.idg_wavelet_filter.argtypes = [fp, i, i, i, i, i, ctypes.POINTER(ctypes.c_float), f, fp, vp]
        _lib = L
    return _lib


def _check(status: int) -> None:
    if status != 0:
        raise IdgError(status)


def _dev(t: torch.Tensor, name: str) -> int:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor (no CPU path)")
    if t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous float32 tensor")
    return t.data_ptr()


def _stream(stream: Optional[torch.cuda.Stream]) -> int:
    return (stream or torch.cuda.current_stream()).cuda_stream


def idg_version() -> int:
    return int(lib().idg_version())


def status_string(status: int) -> str:
    return lib().idg_status_string(int(status)).decode()


def idg_params_check(p: Params) -> int:
    c = p.c()
    return int(lib().idg_params_check(ctypes.byref(c)))


def idg_workspace_bytes(nx: int, ny: int, nz: int, batch: int = 1) -> int:
    return int(lib().idg_workspace_bytes(nx, ny, nz, batch))


def idg_set_option(key: int, value: int) -> None:
    _check(lib().idg_set_option(key, value))


def idg_get_option(key: int) -> int:
    return int(lib().idg_get_option(key))


def idg_release_temporaries() -> None:
    """Hand the library's cached stream-ordered temporaries back to the driver (idg.h)."""
    _check(lib().idg_release_temporaries())


def idg_last_launch_count() -> int:
    return int(lib().idg_last_launch_count())


def idg_last_plan() -> str:
    return lib().idg_last_plan().decode()


def alloc_workspace(nx: int, ny: int, nz: int, batch: int = 1, device="cuda") -> torch.Tensor:
    return torch.empty(idg_workspace_bytes(nx, ny, nz, batch), dtype=torch.uint8, device=device)


def idg_filter(cube: torch.Tensor, n_iter: int, params: Params = Params(),
               out: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
               stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_filter / idg_filter_ws on a [nz, ny, nx] CUDA tensor.  Asynchronous on `stream`."""
    if cube.dim() != 3:
        raise ValueError("cube must be [nz, ny, nx]")
    nz, ny, nx = cube.shape
    if out is None:
        out = torch.empty_like(cube)
    c = params.c()
    if workspace is None:
        rc = lib().idg_filter(_dev(cube, "cube"), nx, ny, nz, int(n_iter), ctypes.byref(c),
                              _dev(out, "out"), _stream(stream))
    else:
        rc = lib().idg_filter_ws(_dev(cube, "cube"), nx, ny, nz, int(n_iter), ctypes.byref(c),
                                 _dev(out, "out"), workspace.data_ptr(), workspace.numel(),
                                 _stream(stream))
    _check(rc)
    return out


def idg_filter_pm(cube: torch.Tensor, n_iter: int, params: Params = Params(),
                  out: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
                  stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_filter_pm (gradient-driven conductance, Eq. 5) on a [nz, ny, nx] CUDA tensor."""
    if cube.dim() != 3:
        raise ValueError("cube must be [nz, ny, nx]")
    nz, ny, nx = cube.shape
    if out is None:
        out = torch.empty_like(cube)
    if workspace is None:
        workspace = alloc_workspace(nx, ny, nz, 1, cube.device)
    c = params.c()
    _check(lib().idg_filter_pm(_dev(cube, "cube"), nx, ny, nz, int(n_iter), ctypes.byref(c), _dev(out, "out"),
                               workspace.data_ptr(), workspace.numel(), _stream(stream)))
    return out


def idg_filter_batched(cubes: torch.Tensor, n_iter: Union[int, Sequence[int]],
                       params: Sequence[Params], out: Optional[torch.Tensor] = None,
                       workspace: Optional[torch.Tensor] = None,
                       stream: Optional[torch.cuda.Stream] = None, variant: str = "idg") -> torch.Tensor:
    """idg_filter_batched (variant "pm": idg_filter_pm_batched) on a [B, nz, ny, nx] CUDA tensor with per-cube parameters."""
    if cubes.dim() != 4:
        raise ValueError("cubes must be [B, nz, ny, nx]")
    B, nz, ny, nx = cubes.shape
    if len(params) != B:
        raise ValueError("one Params per cube")
    if out is None:
        out = torch.empty_like(cubes)
    if workspace is None:
        workspace = alloc_workspace(nx, ny, nz, B, cubes.device)
    arr = (IdgParams * B)(*[p.c() for p in params])
    if isinstance(n_iter, int):
        n_ptr, n_all = None, n_iter
    else:
        if len(n_iter) != B:
            raise ValueError("one n_iter per cube")
        n_arr = (ctypes.c_int * B)(*[int(v) for v in n_iter])
        n_ptr, n_all = ctypes.cast(n_arr, ctypes.c_void_p), 0
    fn = lib().idg_filter_pm_batched if variant == "pm" else lib().idg_filter_batched
    rc = fn(_dev(cubes, "cubes"), nx, ny, nz, B, n_ptr, n_all, arr, _dev(out, "out"), workspace.data_ptr(),
            workspace.numel(), _stream(stream))
    _check(rc)
    return out


def idg_filter_pm_batched(cubes: torch.Tensor, n_iter: Union[int, Sequence[int]], params: Sequence[Params],
                          out: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
                          stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_filter_pm_batched: the gradient-driven variant (Eq. 5) on a [B, nz, ny, nx] CUDA tensor."""
    return idg_filter_batched(cubes, n_iter, params, out, workspace, stream, variant="pm")


def idg_filter_host(cube_host: torch.Tensor, n_iter: int, params: Params = Params(),
                    out_host: Optional[torch.Tensor] = None,
                    dev_buffers: Optional[torch.Tensor] = None,
                    stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_filter_host: HOST fp32 tensors in and out (pinned for full PCIe rate); synchronises."""
    if cube_host.is_cuda or cube_host.dtype != torch.float32 or not cube_host.is_contiguous():
        raise TypeError("cube_host must be a contiguous float32 CPU tensor")
    nz, ny, nx = cube_host.shape
    if out_host is None:
        out_host = torch.empty_like(cube_host, pin_memory=cube_host.is_pinned())
    c = params.c()
    dptr, dbytes = (dev_buffers.data_ptr(), dev_buffers.numel()) if dev_buffers is not None else (None, 0)
    rc = lib().idg_filter_host(cube_host.data_ptr(), nx, ny, nz, int(n_iter), ctypes.byref(c),
                               out_host.data_ptr(), dptr, dbytes, _stream(stream))
    _check(rc)
    return out_host


def idg_box_filter(cube: torch.Tensor, wx: int, wy: int, wz: int, out: Optional[torch.Tensor] = None,
                   stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_box_filter on a [nz, ny, nx] CUDA tensor (widths along x, y, z).  Asynchronous on `stream`."""
    if cube.dim() != 3:
        raise ValueError("cube must be [nz, ny, nx]")
    nz, ny, nx = cube.shape
    if out is None:
        out = torch.empty_like(cube)
    _check(lib().idg_box_filter(_dev(cube, "cube"), nx, ny, nz, int(wx), int(wy), int(wz), _dev(out, "out"),
                                _stream(stream)))
    return out


def idg_gaussian_filter(cube: torch.Tensor, fwhm: Sequence[float], theta: Sequence[float] = (0.0, 0.0, 0.0),
                        out: Optional[torch.Tensor] = None,
                        stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_gaussian_filter on a [nz, ny, nx] CUDA tensor; fwhm = (x, y, z) voxels, theta = (x, y, z) degrees."""
    if cube.dim() != 3:
        raise ValueError("cube must be [nz, ny, nx]")
    nz, ny, nx = cube.shape
    if out is None:
        out = torch.empty_like(cube)
    _check(lib().idg_gaussian_filter(_dev(cube, "cube"), nx, ny, nz, float(fwhm[0]), float(fwhm[1]),
                                     float(fwhm[2]), float(theta[0]), float(theta[1]), float(theta[2]),
                                     _dev(out, "out"), _stream(stream)))
    return out


def idg_gaussian_filter_static(cube: torch.Tensor, fwhm: Sequence[float], theta: Sequence[float],
                               out: Optional[torch.Tensor] = None,
                               stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_gaussian_filter_static: the rotated Gaussian filter with its weights in the library's static device array
    (no allocation inside the call when `out` is given; support radius <= 9, else IdgError status -8)."""
    if cube.dim() != 3:
        raise ValueError("cube must be [nz, ny, nx]")
    nz, ny, nx = cube.shape
    if out is None:
        out = torch.empty_like(cube)
    _check(lib().idg_gaussian_filter_static(_dev(cube, "cube"), nx, ny, nz, float(fwhm[0]), float(fwhm[1]),
                                            float(fwhm[2]), float(theta[0]), float(theta[1]), float(theta[2]),
                                            _dev(out, "out"), _stream(stream)))
    return out


def idg_gaussian_radii(fwhm: Sequence[float], theta: Sequence[float] = (0.0, 0.0, 0.0)) -> tuple:
    r = (ctypes.c_int * 3)()
    _check(lib().idg_gaussian_radii(float(fwhm[0]), float(fwhm[1]), float(fwhm[2]), float(theta[0]),
                                    float(theta[1]), float(theta[2]), r))
    return int(r[0]), int(r[1]), int(r[2])


def _roi(roi) -> Optional[IdgRoi]:
    return None if roi is None else IdgRoi(*[int(v) for v in roi])


SUM_KEYS = ("S_oo", "S_of", "N_o", "N_f", "S_mf", "S_m", "n_roi")


def idg_mask_sums(orig: torch.Tensor, filt: torch.Tensor, model: Optional[torch.Tensor], thr_o: float,
                  thr_f: float, roi=None, sums: Optional[torch.Tensor] = None,
                  stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_mask_sums on [nz, ny, nx] CUDA tensors; roi = (x0, x1, y0, y1, z0, z1) or None.
    Returns the device tensor of 8 doubles (asynchronous on `stream`)."""
    nz, ny, nx = orig.shape
    if filt.shape != orig.shape or (model is not None and model.shape != orig.shape):
        raise ValueError("cubes must have equal shapes")
    if sums is None:
        sums = torch.empty(8, dtype=torch.float64, device=orig.device)
    r = _roi(roi)
    _check(lib().idg_mask_sums(_dev(orig, "orig"), _dev(filt, "filt"),
                               None if model is None else _dev(model, "model"), nx, ny, nz,
                               None if r is None else ctypes.byref(r), float(thr_o), float(thr_f),
                               sums.data_ptr(), _stream(stream)))
    return sums


def idg_cube_stats(cube: torch.Tensor, roi=None, stats: Optional[torch.Tensor] = None,
                   stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_cube_stats: device tensor of 8 doubles (n, sum, sum of squares, 0...)."""
    nz, ny, nx = cube.shape
    if stats is None:
        stats = torch.empty(8, dtype=torch.float64, device=cube.device)
    r = _roi(roi)
    _check(lib().idg_cube_stats(_dev(cube, "cube"), nx, ny, nz, None if r is None else ctypes.byref(r),
                                stats.data_ptr(), _stream(stream)))
    return stats


def idg_stats_rms(stats: Sequence[float]) -> tuple:
    """idg_stats_rms on a HOST copy of the idg_cube_stats output: (mean, rms)."""
    arr = (ctypes.c_double * 8)(*[float(v) for v in list(stats)[:8]] + [0.0] * (8 - min(8, len(stats))))
    mean, rms = ctypes.c_double(), ctypes.c_double()
    _check(lib().idg_stats_rms(arr, ctypes.byref(mean), ctypes.byref(rms)))
    return mean.value, rms.value


def idg_histogram(cube: torch.Tensor, lo: float, hi: float, nbins: int, roi=None, mask_thr: Optional[float] = None,
                  counts: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_histogram: device tensor of nbins int64 counts over [lo, hi) for the ROI."""
    nz, ny, nx = cube.shape
    if counts is None:
        counts = torch.empty(int(nbins), dtype=torch.int64, device=cube.device)
    r = _roi(roi)
    thr = None if mask_thr is None else ctypes.byref(ctypes.c_float(float(mask_thr)))
    _check(lib().idg_histogram(_dev(cube, "cube"), nx, ny, nz, None if r is None else ctypes.byref(r), float(lo),
                               float(hi), int(nbins), thr, counts.data_ptr(), _stream(stream)))
    return counts


def idg_quality(sums: Sequence[float], rms_o: float, rms_f: float, voxels_per_beam: float = 1.0) -> dict:
    """idg_quality on a HOST copy of the sums: {"F", "sigma_F", "F_M"} (Eq. 12, 15-17)."""
    arr = (ctypes.c_double * 8)(*[float(v) for v in list(sums)[:8]] + [0.0] * (8 - min(8, len(sums))))
    out = [ctypes.c_double() for _ in range(3)]
    _check(lib().idg_quality(arr, float(rms_o), float(rms_f), float(voxels_per_beam),
                             *[ctypes.byref(o) for o in out]))
    return {"F": out[0].value, "sigma_F": out[1].value, "F_M": out[2].value}


def idg_wavelet_transform(cube: torch.Tensor, wavelet: int, levels: int, inverse: bool = False,
                          out: Optional[torch.Tensor] = None,
                          stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_wavelet_transform on a [nz, ny, nx] CUDA tensor (out may be the cube itself: in place)."""
    nz, ny, nx = cube.shape
    if out is None:
        out = torch.empty_like(cube)
    _check(lib().idg_wavelet_transform(_dev(cube, "cube"), nx, ny, nz, int(wavelet), int(levels), int(bool(inverse)),
                                       _dev(out, "out"), _stream(stream)))
    return out


def idg_wavelet_filter(cube: torch.Tensor, wavelet: int, thresholds: Sequence[float], rms: float = 1.0,
                       out: Optional[torch.Tensor] = None,
                       stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """idg_wavelet_filter: len(thresholds) levels, thresholds in units of rms."""
    nz, ny, nx = cube.shape
    if out is None:
        out = torch.empty_like(cube)
    t = (ctypes.c_float * max(1, len(thresholds)))(*[float(v) for v in thresholds])
    _check(lib().idg_wavelet_filter(_dev(cube, "cube"), nx, ny, nz, int(wavelet), len(thresholds), t, float(rms),
                                    _dev(out, "out"), _stream(stream)))
    return out


def host_buffers_bytes(nx: int, ny: int, nz: int) -> int:
    cube = (nx * ny * nz * 4 + 255) // 256 * 256
    return 2 * cube + idg_workspace_bytes(nx, ny, nz, 1)
