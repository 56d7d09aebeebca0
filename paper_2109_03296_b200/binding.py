"""Thin ctypes binding of libkbmod_b200.so (include/kbmod_b200.h): same names, argument marshalling
only.  Device buffers are torch CUDA tensors (torch is used for device memory and streams, nothing
else); host arrays are numpy.  There is no CPU fallback: if the library is missing or a call fails,
this raises."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkbmod_b200.so")

ALGO_AUTO, ALGO_DIRECT, ALGO_PRUNED = 0, 1, 2
MAX_T, MAX_K, MAX_PSF, MAX_STAMP_RADIUS = 64, 32, 31, 15

EXPORTS = ["kbmod_default_params", "kbmod_prepare_psi_phi", "kbmod_displacements",
           "kbmod_search_workspace_bytes", "kbmod_search", "kbmod_plan_stats", "kbmod_search_stats", "kbmod_search_phase_timing",
           "kbmod_search_phase_ms", "kbmod_coadd_stamps",
           "kbmod_eval_trajectories", "kbmod_sigmag_filter", "kbmod_stamp_moments", "kbmod_pipeline_host_arena_bytes",
           "kbmod_pipeline_host", "kbmod_pipeline_host_batch", "kbmod_measure_smem_gbs", "kbmod_last_error", "kbmod_version"]


class KbmodError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"kbmod_b200 error {code}: {msg}")
        self.code = code


class CParams(C.Structure):
    _fields_ = [("sigmag_enable", C.c_int), ("pct_lo", C.c_float), ("pct_hi", C.c_float),
                ("sigmag_coeff", C.c_float), ("n_sigma", C.c_float), ("filter_on", C.c_int),
                ("min_lh", C.c_float), ("min_obs", C.c_int), ("K", C.c_int), ("algo", C.c_int)]


@dataclass
class SearchParams:
    """kbmod_search_params; defaults are the paper's values."""
    sigmag_enable: int = 1
    pct_lo: float = 25.0
    pct_hi: float = 75.0
    sigmag_coeff: float = 0.7413
    n_sigma: float = 2.0
    filter_on: int = 0
    min_lh: float = 10.0
    min_obs: int = 1
    K: int = 8
    algo: int = ALGO_AUTO

    def c(self) -> CParams:
        return CParams(self.sigmag_enable, self.pct_lo, self.pct_hi, self.sigmag_coeff, self.n_sigma,
                       self.filter_on, self.min_lh, self.min_obs, self.K, self.algo)


_lib = None


def lib():
    """Loads the library (never builds it: build() in paper_2109_03296_b200.build does)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise KbmodError(-4, f"{LIB_PATH} is missing: run `python -m paper_2109_03296_b200.build`")
        L = C.CDLL(LIB_PATH)
        L.kbmod_last_error.restype = C.c_char_p
        L.kbmod_version.restype = C.c_int
        L.kbmod_search_workspace_bytes.restype = C.c_size_t
        L.kbmod_pipeline_host_arena_bytes.restype = C.c_size_t
        L.kbmod_default_params.restype = None
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise KbmodError(rc, lib().kbmod_last_error().decode())


def _dev(t, dtype=None, allow_none=False):
    """Device pointer of a contiguous CUDA tensor."""
    import torch
    if t is None:
        if allow_none:
            return C.c_void_p(0)
        raise ValueError("tensor required")
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("expected a CUDA torch tensor (no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _host(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data_as(C.c_void_p)


def _stream(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def kbmod_version() -> int:
    return int(lib().kbmod_version())


def kbmod_default_params() -> SearchParams:
    cp = CParams()
    lib().kbmod_default_params(C.byref(cp))
    return SearchParams(*[getattr(cp, f) for f, _ in CParams._fields_])


def kbmod_displacements(times, vx, vy):
    """(a2) host-only displacement table: returns dx, dy int32 [n_vel][T]."""
    t, tp = _host(times, np.float64)
    x, xp = _host(vx, np.float32)
    y, yp = _host(vy, np.float32)
    dx = np.empty((len(x), len(t)), np.int32)
    dy = np.empty((len(x), len(t)), np.int32)
    _check(lib().kbmod_displacements(tp, len(t), xp, yp, len(x), dx.ctypes.data_as(C.c_void_p),
                                     dy.ctypes.data_as(C.c_void_p)))
    return dx, dy


def kbmod_prepare_psi_phi(img, var, mask, psf, out=None, stream=None):
    """(a1) img, var [T][H][W] float32 CUDA, mask uint8 CUDA or None, psf numpy [k][k] or [T][k][k].
    Returns the psi/phi stack, float32 CUDA [T][H][W][2]."""
    import torch
    T, H, W = img.shape
    p, pp = _host(psf, np.float32)
    n_psf = 1 if p.ndim == 2 else p.shape[0]
    k = p.shape[-1]
    if out is None:
        out = torch.empty((T, H, W, 2), dtype=torch.float32, device=img.device)
    _check(lib().kbmod_prepare_psi_phi(_dev(img, torch.float32), _dev(var, torch.float32),
                                       _dev(mask, torch.uint8, allow_none=True), T, H, W, pp, n_psf, k,
                                       _dev(out, torch.float32), _stream(stream)))
    return out


def kbmod_search_workspace_bytes(T, H, W, n_vel, params: SearchParams) -> int:
    cp = params.c()
    return int(lib().kbmod_search_workspace_bytes(T, H, W, n_vel, C.byref(cp)))


def kbmod_search(psiphi, times, vx, vy, params: SearchParams, out=None, workspace=None, stream=None):
    """(a3)-(a5).  psiphi float32 CUDA [T][H][W][2].  Returns (lh, flux, vel_idx, n_obs), each [H][W][K]."""
    import torch
    T, H, W, two = psiphi.shape
    assert two == 2
    t, tp = _host(times, np.float64)
    x, xp = _host(vx, np.float32)
    y, yp = _host(vy, np.float32)
    assert len(t) == T and len(x) == len(y)
    K = params.K
    dev = psiphi.device
    if out is None:
        out = (torch.empty((H, W, K), dtype=torch.float32, device=dev),
               torch.empty((H, W, K), dtype=torch.float32, device=dev),
               torch.empty((H, W, K), dtype=torch.int32, device=dev),
               torch.empty((H, W, K), dtype=torch.int32, device=dev))
    nbytes = kbmod_search_workspace_bytes(T, H, W, len(x), params)
    if workspace is None:
        workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=dev)
    cp = params.c()
    _check(lib().kbmod_search(_dev(psiphi, torch.float32), T, H, W, tp, xp, yp, len(x), C.byref(cp),
                              _dev(out[0], torch.float32), _dev(out[1], torch.float32),
                              _dev(out[2], torch.int32), _dev(out[3], torch.int32), _dev(workspace),
                              C.c_size_t(workspace.numel()), _stream(stream)))
    kbmod_search.last_workspace = workspace
    return out


def kbmod_plan_stats(T, H, W, times, vx, vy, params: SearchParams):
    """Host-only: dict(too_scattered, staged_bytes_per_eval, n_groups, off_image_fraction) of the pruned kernel's plan."""
    t, tp = _host(times, np.float64)
    x, xp = _host(vx, np.float32)
    y, yp = _host(vy, np.float32)
    cp = params.c()
    out = (C.c_double * 4)()
    _check(lib().kbmod_plan_stats(T, H, W, tp, xp, yp, len(x), C.byref(cp), out))
    return dict(too_scattered=bool(out[0]), staged_bytes_per_eval=float(out[1]), n_groups=int(out[2]),
                off_image_fraction=float(out[3]))


def kbmod_search_stats(workspace):
    """[evaluated, nominal, launches, algo] of the last kbmod_search that used `workspace` (synchronises)."""
    out = (C.c_ulonglong * 4)()
    _check(lib().kbmod_search_stats(_dev(workspace), out))
    return [int(v) for v in out]


def kbmod_search_phase_timing(enable: bool):
    """Switches the per-phase CUDA-event timing of kbmod_search on or off for this host thread."""
    _check(lib().kbmod_search_phase_timing(C.c_int(1 if enable else 0)))


def kbmod_search_phase_ms():
    """dict of milliseconds per phase of the last timed kbmod_search on this thread (synchronises)."""
    out = (C.c_float * 4)()
    _check(lib().kbmod_search_phase_ms(out))
    return dict(planes=float(out[0]), gather=float(out[1]), exact=float(out[2]), finalize=float(out[3]))


def kbmod_coadd_stamps(img, mask, times, x0, y0, vx, vy, radius, epoch_mask=None, want_mean=True,
                       want_median=True, stream=None):
    """(a6).  img float32 CUDA [T][H][W]; x0, y0 int32 CUDA; vx, vy float32 CUDA; epoch_mask int64/uint64
    CUDA or None.  Returns (mean, median) float32 CUDA [n][2r+1][2r+1] (None where not wanted)."""
    import torch
    T, H, W = img.shape
    t, tp = _host(times, np.float64)
    n, S = x0.numel(), 2 * radius + 1
    mean = torch.empty((n, S, S), dtype=torch.float32, device=img.device) if want_mean else None
    med = torch.empty((n, S, S), dtype=torch.float32, device=img.device) if want_median else None
    _check(lib().kbmod_coadd_stamps(_dev(img, torch.float32), _dev(mask, torch.uint8, allow_none=True), T, H, W,
                                    tp, _dev(x0, torch.int32), _dev(y0, torch.int32), _dev(vx, torch.float32),
                                    _dev(vy, torch.float32), _dev(epoch_mask, allow_none=True), n, radius,
                                    _dev(mean, allow_none=True), _dev(med, allow_none=True), _stream(stream)))
    return mean, med


def kbmod_eval_trajectories(psiphi, times, x0, y0, vx, vy, params: SearchParams, stream=None):
    """Single-trajectory variant.  Returns a dict of CUDA tensors."""
    import torch
    T, H, W, _ = psiphi.shape
    t, tp = _host(times, np.float64)
    n, dev = x0.numel(), psiphi.device
    r = dict(psi_lc=torch.empty((n, T), dtype=torch.float32, device=dev),
             phi_lc=torch.empty((n, T), dtype=torch.float32, device=dev),
             valid=torch.empty(n, dtype=torch.int64, device=dev), kept=torch.empty(n, dtype=torch.int64, device=dev),
             lh=torch.empty(n, dtype=torch.float32, device=dev), flux=torch.empty(n, dtype=torch.float32, device=dev))
    cp = params.c()
    _check(lib().kbmod_eval_trajectories(_dev(psiphi, torch.float32), T, H, W, tp, _dev(x0, torch.int32),
                                         _dev(y0, torch.int32), _dev(vx, torch.float32), _dev(vy, torch.float32), n,
                                         C.byref(cp), _dev(r["psi_lc"]), _dev(r["phi_lc"]), _dev(r["valid"]),
                                         _dev(r["kept"]), _dev(r["lh"]), _dev(r["flux"]), _stream(stream)))
    return r


def kbmod_sigmag_filter(psi_lc, phi_lc, params: SearchParams, stream=None):
    """sigma-G on given lightcurves [n][T] float32 CUDA.  Returns dict(kept int64, lh, flux)."""
    import torch
    n, T = psi_lc.shape
    dev = psi_lc.device
    r = dict(kept=torch.empty(n, dtype=torch.int64, device=dev), lh=torch.empty(n, dtype=torch.float32, device=dev),
             flux=torch.empty(n, dtype=torch.float32, device=dev))
    cp = params.c()
    _check(lib().kbmod_sigmag_filter(_dev(psi_lc, torch.float32), _dev(phi_lc, torch.float32), n, T, C.byref(cp),
                                     _dev(r["kept"]), _dev(r["lh"]), _dev(r["flux"]), _stream(stream)))
    return r


def kbmod_stamp_moments(stamps, thresholds=None, stream=None):
    """Central moments (x, y, xy, xx, yy) of [n][S][S] stamps and the paper's keep / reject flag.
    Returns (moments float64 [n][5], keep uint8 [n])."""
    import torch
    s = _dev(stamps, torch.float32)
    n, S, S2 = stamps.shape
    if S != S2 or S % 2 != 1:
        raise KbmodError(-1, f"stamps must be [n][2r+1][2r+1], got {tuple(stamps.shape)}")
    mom = torch.empty((n, 5), dtype=torch.float64, device=stamps.device)
    keep = torch.empty((n,), dtype=torch.uint8, device=stamps.device)
    thr_arr, thr_ptr = (None, C.c_void_p(0)) if thresholds is None else _host(thresholds, np.float64)
    if thr_arr is not None and thr_arr.shape != (5,):
        raise KbmodError(-1, "thresholds must be 5 numbers: x, y, xy, xx, yy")
    _check(lib().kbmod_stamp_moments(s, C.c_int(n), C.c_int(S // 2), thr_ptr, _dev(mom), _dev(keep), _stream(stream)))
    return mom, keep


def kbmod_pipeline_host_batch(stacks, psf, times, vx, vy, params: SearchParams, outs, arena, stream=None):
    """`stacks`: list of (img, var, mask-or-None) CPU tensors of one shape; `outs`: list of 4-tuples of CPU tensors
    [H][W][K]; `arena`: uint8 CUDA tensor of at least 2 x kbmod_pipeline_host_arena_bytes (1 x for one stack).
    Copies overlap the searches; synchronises before returning."""
    n = len(stacks)
    T, H, W = stacks[0][0].shape
    p, pp = _host(psf, np.float32)
    n_psf = 1 if p.ndim == 2 else p.shape[0]
    t, tp = _host(times, np.float64)
    x, xp = _host(vx, np.float32)
    y, yp = _host(vy, np.float32)
    has_mask = stacks[0][2] is not None
    for st_ in stacks:
        assert tuple(st_[0].shape) == (T, H, W) and (st_[2] is not None) == has_mask
        for a in st_:
            assert a is None or (not a.is_cuda and a.is_contiguous())
    arr = lambda items: (C.c_void_p * n)(*[C.c_void_p(a.data_ptr()) for a in items])
    imgs, vars_ = arr([s_[0] for s_ in stacks]), arr([s_[1] for s_ in stacks])
    masks = arr([s_[2] for s_ in stacks]) if has_mask else None
    o = [arr([o_[j] for o_ in outs]) for j in range(4)]
    cp = params.c()
    _check(lib().kbmod_pipeline_host_batch(C.c_int(n), imgs, vars_, masks, T, H, W, pp, n_psf, p.shape[-1], tp, xp, yp, len(x),
                                           C.byref(cp), o[0], o[1], o[2], o[3], _dev(arena), C.c_size_t(arena.numel()),
                                           _stream(stream)))
    return outs


def kbmod_measure_smem_gbs(bytes_per_lane: int = 4, stream=None) -> float:
    """Measured shared-memory load bandwidth of the whole GPU in GB/s (roofline denominator; synchronises)."""
    out = C.c_double(0.0)
    _check(lib().kbmod_measure_smem_gbs(C.c_int(bytes_per_lane), C.byref(out), _stream(stream)))
    return float(out.value)


def kbmod_pipeline_host_arena_bytes(T, H, W, n_vel, params: SearchParams) -> int:
    cp = params.c()
    return int(lib().kbmod_pipeline_host_arena_bytes(T, H, W, n_vel, C.byref(cp)))


def kbmod_pipeline_host(img, var, mask, psf, times, vx, vy, params: SearchParams, out, arena, stream=None):
    """Whole path from HOST buffers: img, var (float32), mask (uint8 or None) are CPU torch tensors
    (pinned for full PCIe speed); `out` = 4 CPU tensors [H][W][K]; `arena` = uint8 CUDA tensor.
    Synchronises the stream before returning."""
    import torch
    T, H, W = img.shape
    p, pp = _host(psf, np.float32)
    n_psf = 1 if p.ndim == 2 else p.shape[0]
    t, tp = _host(times, np.float64)
    x, xp = _host(vx, np.float32)
    y, yp = _host(vy, np.float32)
    for a in (img, var, mask) + tuple(out):
        assert a is None or (not a.is_cuda and a.is_contiguous())
    cp = params.c()
    hp = lambda a: C.c_void_p(a.data_ptr()) if a is not None else C.c_void_p(0)
    _check(lib().kbmod_pipeline_host(hp(img), hp(var), hp(mask), T, H, W, pp, n_psf, p.shape[-1], tp, xp, yp, len(x),
                                     C.byref(cp), hp(out[0]), hp(out[1]), hp(out[2]), hp(out[3]), _dev(arena),
                                     C.c_size_t(arena.numel()), _stream(stream)))
    return out
