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

# every symbol include/kbmod_b200.h declares, with its C signature (restype, argtypes): ctypes then converts and
# range-checks every argument itself (a Python int for a size_t can no longer be truncated to a C int)
_P, _I, _Z, _D = C.c_void_p, C.c_int, C.c_size_t, C.c_double
SIGNATURES = {
    "kbmod_default_params": (None, [_P]),
    "kbmod_percentile_ranks": (_I, [_P, _I, _P, _P]),
    "kbmod_prepare_psi_phi": (_I, [_P, _P, _P, _I, _I, _I, _P, _I, _I, _P, _P]),
    "kbmod_displacements": (_I, [_P, _I, _P, _P, _I, _P, _P]),
    "kbmod_search_workspace_bytes": (_Z, [_I, _I, _I, _I, _P]),
    "kbmod_search_workspace_bytes_for": (_Z, [_I, _I, _I, _P, _P, _P, _I, _P, _I, _I]),
    "kbmod_search": (_I, [_P, _I, _I, _I, _P, _P, _P, _I, _P, _P, _P, _P, _P, _P, _Z, _P]),
    "kbmod_search_rows": (_I, [_P, _I, _I, _I, _P, _P, _P, _I, _P, _I, _I, _P, _P, _P, _P, _P, _Z, _P]),
    "kbmod_search_unfiltered_lh": (_I, [_P, _P, _P, _P]),
    "kbmod_plan_create": (_I, [_I, _I, _I, _P, _P, _P, _I, _P, _I, _I, C.POINTER(_P)]),
    "kbmod_plan_workspace_bytes": (_Z, [_P]),
    "kbmod_plan_info": (_I, [_P, _P]),
    "kbmod_plan_search": (_I, [_P, _P, _P, _P, _P, _P, _P, _Z, _P]),
    "kbmod_plan_unfiltered_lh": (_I, [_P, _P, _P, _P, _P]),
    "kbmod_plan_destroy": (None, [_P]),
    "kbmod_release_thread_state": (_I, []),
    "kbmod_plan_stats": (_I, [_I, _I, _I, _P, _P, _P, _I, _P, _P]),
    "kbmod_search_stats": (_I, [_P, _P]),
    "kbmod_search_phase_timing": (_I, [_I]),
    "kbmod_search_phase_ms": (_I, [_P]),
    "kbmod_coadd_stamps": (_I, [_P, _P, _I, _I, _I, _P, _P, _P, _P, _P, _P, _I, _I, _P, _P, _P]),
    "kbmod_coadd_stamps_filtered": (_I, [_P, _P, _I, _I, _I, _P, _P, _P, _P, _P, _P, _I, _I, _P, _P, _P, _P, _P, _P]),
    "kbmod_eval_trajectories": (_I, [_P, _I, _I, _I, _P, _P, _P, _P, _P, _I, _P, _P, _P, _P, _P, _P, _P, _P]),
    "kbmod_sigmag_filter": (_I, [_P, _P, _I, _I, _P, _P, _P, _P, _P]),
    "kbmod_sigmag_postfilter": (_I, [_P, _P, _I, _I, _P, _P, _P, _P, _P, _P, _P, _P]),
    "kbmod_sigmag_postfilter_static": (_I, [_P, _P, _I, _I, _P, _P, _P, _P, _P, _P, _P]),
    "kbmod_stamp_moments": (_I, [_P, _I, _I, _P, _P, _P, _P]),
    "kbmod_pipeline_host_arena_bytes": (_Z, [_I, _I, _I, _I, _P]),
    "kbmod_pipeline_host_arena_bytes_for": (_Z, [_I, _I, _I, _P, _P, _P, _I, _P]),
    "kbmod_pipeline_host": (_I, [_P, _P, _P, _I, _I, _I, _P, _I, _I, _P, _P, _P, _I, _P, _P, _P, _P, _P, _P, _Z, _P]),
    "kbmod_pipeline_host_batch": (_I, [_I, _P, _P, _P, _I, _I, _I, _P, _I, _I, _P, _P, _P, _I, _P, _P, _P, _P, _P, _P, _Z, _P]),
    "kbmod_measure_smem_gbs": (_I, [_I, _P, _P, _P]),
    "kbmod_measure_issue_rate": (_I, [_I, _P, _P, _P]),
    "kbmod_last_error": (C.c_char_p, []),
    "kbmod_version": (_I, []),
}
EXPORTS = list(SIGNATURES)


class KbmodError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"kbmod_b200 error {code}: {msg}")
        self.code = code


class CParams(C.Structure):
    _fields_ = [("sigmag_enable", C.c_int), ("pct_lo", C.c_float), ("pct_hi", C.c_float),
                ("sigmag_coeff", C.c_float), ("n_sigma", C.c_float), ("filter_on", C.c_int),
                ("min_lh", C.c_float), ("min_obs", C.c_int), ("K", C.c_int), ("algo", C.c_int),
                ("pct_interp", C.c_int)]


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
    pct_interp: int = 0

    def c(self) -> CParams:
        return CParams(self.sigmag_enable, self.pct_lo, self.pct_hi, self.sigmag_coeff, self.n_sigma,
                       self.filter_on, self.min_lh, self.min_obs, self.K, self.algo, self.pct_interp)


_lib = None


def lib():
    """Loads the library (never builds it: build() in paper_2109_03296_b200.build does)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise KbmodError(-4, f"{LIB_PATH} is missing: run `python -m paper_2109_03296_b200.build`")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)  # AttributeError if the library does not export what the header declares
            fn.restype, fn.argtypes = res, args
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


def _grid(times, vx, vy, T):
    """Host arrays of a search: times float64 [T], vx, vy float32 [n_vel]; shapes checked here."""
    t, tp = _host(times, np.float64)
    x, xp = _host(vx, np.float32)
    y, yp = _host(vy, np.float32)
    if t.ndim != 1 or len(t) != T:
        raise ValueError(f"times must be [T] = [{T}], got {t.shape}")
    if x.ndim != 1 or x.shape != y.shape:
        raise ValueError(f"vx, vy must be 1-D arrays of one length, got {x.shape}, {y.shape}")
    return (t, x, y), (tp, xp, yp)


def _check_out(out, shape):
    import torch
    want = (torch.float32, torch.float32, torch.int32, torch.int32)
    if len(out) != 4:
        raise ValueError("out must be (lh, flux, vel_idx, n_obs)")
    for o, dt in zip(out, want):
        if tuple(o.shape) != tuple(shape) or o.dtype != dt:
            raise ValueError(f"output tensors must be {tuple(shape)} {want}, got {tuple(o.shape)} {o.dtype}")


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


def kbmod_percentile_ranks(params: SearchParams, n: int):
    """Host-only: [(k, g)] for (pct_lo, 50, pct_hi) of n valid samples; g < 0 means "take s[k]"."""
    cp = params.c()
    k, g = (C.c_int * 3)(), (C.c_float * 3)()
    _check(lib().kbmod_percentile_ranks(C.byref(cp), n, k, g))
    return [(int(k[i]), float(g[i])) for i in range(3)]


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
    if p.ndim not in (2, 3) or p.shape[-1] != p.shape[-2]:
        raise ValueError(f"psf must be [k][k] or [T][k][k], got {p.shape}")
    n_psf = 1 if p.ndim == 2 else p.shape[0]
    k = p.shape[-1]
    if tuple(var.shape) != (T, H, W) or (mask is not None and tuple(mask.shape) != (T, H, W)):
        raise ValueError("img, var and mask must have one shape [T][H][W]")
    if out is None:
        out = torch.empty((T, H, W, 2), dtype=torch.float32, device=img.device)
    elif tuple(out.shape) != (T, H, W, 2):
        raise ValueError(f"out must be [T][H][W][2], got {tuple(out.shape)}")
    _check(lib().kbmod_prepare_psi_phi(_dev(img, torch.float32), _dev(var, torch.float32),
                                       _dev(mask, torch.uint8, allow_none=True), T, H, W, pp, n_psf, k,
                                       _dev(out, torch.float32), _stream(stream)))
    return out


def kbmod_search_workspace_bytes(T, H, W, n_vel, params: SearchParams) -> int:
    """Upper bound for any list of n_vel velocities (the stack padded by the image size on every side)."""
    cp = params.c()
    return int(lib().kbmod_search_workspace_bytes(T, H, W, n_vel, C.byref(cp)))


def kbmod_search_workspace_bytes_for(T, H, W, times, vx, vy, params: SearchParams, rows=None) -> int:
    """Exact workspace need of kbmod_search / kbmod_search_rows for this grid."""
    (t, x, y), (tp, xp, yp) = _grid(times, vx, vy, T)
    r0, r1 = (0, H) if rows is None else rows
    cp = params.c()
    n = int(lib().kbmod_search_workspace_bytes_for(T, H, W, tp, xp, yp, len(x), C.byref(cp), r0, r1))
    if n == 0:
        raise KbmodError(-1, lib().kbmod_last_error().decode())
    return n


def kbmod_search(psiphi, times, vx, vy, params: SearchParams, out=None, workspace=None, stream=None, rows=None):
    """(a3)-(a5).  psiphi float32 CUDA [T][H][W][2].  Returns (lh, flux, vel_idx, n_obs), each [H][W][K]; with
    rows=(row_begin, row_end) the search is restricted to that band of start rows and the outputs are
    [row_end - row_begin][W][K] (kbmod_search_rows)."""
    import torch
    T, H, W, two = psiphi.shape
    if two != 2:
        raise ValueError("psiphi must be [T][H][W][2]")
    (t, x, y), (tp, xp, yp) = _grid(times, vx, vy, T)
    K = params.K
    dev = psiphi.device
    r0, r1 = (0, H) if rows is None else (int(rows[0]), int(rows[1]))
    shape = (max(r1 - r0, 0), W, K)
    if out is None:
        out = (torch.empty(shape, dtype=torch.float32, device=dev), torch.empty(shape, dtype=torch.float32, device=dev),
               torch.empty(shape, dtype=torch.int32, device=dev), torch.empty(shape, dtype=torch.int32, device=dev))
    else:
        _check_out(out, shape)
    cp = params.c()
    if workspace is None:
        nbytes = int(lib().kbmod_search_workspace_bytes_for(T, H, W, tp, xp, yp, len(x), C.byref(cp), r0, r1))
        workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=dev)
    args = [_dev(psiphi, torch.float32), T, H, W, tp, xp, yp, len(x), C.byref(cp)]
    tail = [_dev(out[0], torch.float32), _dev(out[1], torch.float32), _dev(out[2], torch.int32),
            _dev(out[3], torch.int32), _dev(workspace), workspace.numel(), _stream(stream)]
    if rows is None:
        _check(lib().kbmod_search(*args, *tail))
    else:
        _check(lib().kbmod_search_rows(*args, r0, r1, *tail))
    kbmod_search.last_workspace = workspace
    return out


def kbmod_search_unfiltered_lh(workspace, vel_idx, stream=None):
    """Unfiltered sum-LH of the result slots of the last kbmod_search of this thread that used
    `workspace`.  vel_idx int32 CUDA [rows][W][K] -> float32 CUDA of the same shape."""
    import torch
    out = torch.empty(vel_idx.shape, dtype=torch.float32, device=vel_idx.device)
    _check(lib().kbmod_search_unfiltered_lh(_dev(workspace), _dev(vel_idx, torch.int32), _dev(out), _stream(stream)))
    return out


class Plan:
    """kbmod_plan: the geometry-only part of a search (host memory), shared by any number of searches / streams."""

    def __init__(self, T, H, W, times, vx, vy, params: SearchParams, rows=None):
        (t, x, y), (tp, xp, yp) = _grid(times, vx, vy, T)
        self.T, self.H, self.W, self.K, self.n_vel = T, H, W, params.K, len(x)
        self.rows = (0, H) if rows is None else (int(rows[0]), int(rows[1]))
        self._h = C.c_void_p(0)
        cp = params.c()
        _check(lib().kbmod_plan_create(T, H, W, tp, xp, yp, len(x), C.byref(cp), self.rows[0], self.rows[1], C.byref(self._h)))

    def workspace_bytes(self) -> int:
        return int(lib().kbmod_plan_workspace_bytes(self._h))

    def info(self):
        out = (C.c_double * 10)()
        _check(lib().kbmod_plan_info(self._h, out))
        return dict(algo=int(out[0]), n_groups=int(out[1]), staged_bytes_per_eval=float(out[2]),
                    off_image_fraction=float(out[3]), canvas=(int(out[4]), int(out[5])), too_scattered=bool(out[6]),
                    table_bytes=int(out[7]), gather_fraction=float(out[8]), workspace_bytes=int(out[9]))

    def search(self, psiphi, out=None, workspace=None, stream=None):
        import torch
        if tuple(psiphi.shape) != (self.T, self.H, self.W, 2):
            raise ValueError("psiphi does not have the plan's shape")
        dev = psiphi.device
        shape = (self.rows[1] - self.rows[0], self.W, self.K)
        if out is None:
            out = tuple(torch.empty(shape, dtype=dt, device=dev)
                        for dt in (torch.float32, torch.float32, torch.int32, torch.int32))
        else:
            _check_out(out, shape)
        if workspace is None:
            workspace = torch.empty(max(self.workspace_bytes(), 256), dtype=torch.uint8, device=dev)
        _check(lib().kbmod_plan_search(self._h, _dev(psiphi, torch.float32), _dev(out[0]), _dev(out[1]), _dev(out[2]),
                                       _dev(out[3]), _dev(workspace), workspace.numel(), _stream(stream)))
        self.last_workspace = workspace
        return out

    def unfiltered_lh(self, workspace, vel_idx, stream=None):
        import torch
        out = torch.empty(vel_idx.shape, dtype=torch.float32, device=vel_idx.device)
        _check(lib().kbmod_plan_unfiltered_lh(self._h, _dev(workspace), _dev(vel_idx, torch.int32), _dev(out),
                                              _stream(stream)))
        return out

    def destroy(self):
        if self._h:
            lib().kbmod_plan_destroy(self._h)
            self._h = C.c_void_p(0)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# the plan entry points under their C names (thin aliases of the Plan class)
def kbmod_plan_create(T, H, W, times, vx, vy, params: SearchParams, rows=None) -> Plan:
    return Plan(T, H, W, times, vx, vy, params, rows)


def kbmod_plan_workspace_bytes(plan: Plan) -> int:
    return plan.workspace_bytes()


def kbmod_plan_info(plan: Plan):
    return plan.info()


def kbmod_plan_search(plan: Plan, psiphi, out=None, workspace=None, stream=None):
    return plan.search(psiphi, out=out, workspace=workspace, stream=stream)


def kbmod_plan_unfiltered_lh(plan: Plan, workspace, vel_idx, stream=None):
    return plan.unfiltered_lh(workspace, vel_idx, stream=stream)


def kbmod_plan_destroy(plan: Plan):
    plan.destroy()


def kbmod_search_rows(psiphi, times, vx, vy, params: SearchParams, rows, out=None, workspace=None, stream=None):
    return kbmod_search(psiphi, times, vx, vy, params, out=out, workspace=workspace, stream=stream, rows=rows)


def kbmod_release_thread_state():
    """Frees the per-thread conveniences of the library (cached plan, timing events, batch copy streams)."""
    _check(lib().kbmod_release_thread_state())


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
    """[evaluated, nominal, launches, algo, reached_min_lh] of the last search that used `workspace` (synchronises)."""
    out = (C.c_ulonglong * 5)()
    _check(lib().kbmod_search_stats(_dev(workspace), out))
    return [int(v) for v in out]


def kbmod_search_phase_timing(enable: bool):
    """Switches the per-phase CUDA-event timing of kbmod_search on or off for this host thread."""
    _check(lib().kbmod_search_phase_timing(1 if enable else 0))


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


def kbmod_coadd_stamps_filtered(img, mask, times, x0, y0, vx, vy, radius, epoch_mask=None, thresholds=None,
                                want_mean=True, want_median=True, stream=None):
    """(a6) + the central-moment filter in one kernel.  Returns (mean, median, moments float64 [n][5],
    keep uint8 [n]); the moments are those of the median stamp, bit-identical to kbmod_stamp_moments(median)."""
    import torch
    T, H, W = img.shape
    t, tp = _host(times, np.float64)
    n, S = x0.numel(), 2 * radius + 1
    dev = img.device
    mean = torch.empty((n, S, S), dtype=torch.float32, device=dev) if want_mean else None
    med = torch.empty((n, S, S), dtype=torch.float32, device=dev) if want_median else None
    mom = torch.empty((n, 5), dtype=torch.float64, device=dev)
    keep = torch.empty((n,), dtype=torch.uint8, device=dev)
    thr_arr, thr_ptr = (None, C.c_void_p(0)) if thresholds is None else _host(thresholds, np.float64)
    if thr_arr is not None and thr_arr.shape != (5,):
        raise KbmodError(-1, "thresholds must be 5 numbers: x, y, xy, xx, yy")
    for a in (x0, y0, vx, vy):
        if a.numel() != n:
            raise ValueError("x0, y0, vx, vy must have one length")
    _check(lib().kbmod_coadd_stamps_filtered(_dev(img, torch.float32), _dev(mask, torch.uint8, allow_none=True), T, H, W,
                                             tp, _dev(x0, torch.int32), _dev(y0, torch.int32), _dev(vx, torch.float32),
                                             _dev(vy, torch.float32), _dev(epoch_mask, allow_none=True), n, radius,
                                             _dev(mean, allow_none=True), _dev(med, allow_none=True), thr_ptr, _dev(mom),
                                             _dev(keep), _stream(stream)))
    return mean, med, mom, keep


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


def kbmod_sigmag_postfilter(psi_lc, phi_lc, params: SearchParams, compact=True, stream=None):
    """The paper's post-filter: sigma-G on given lightcurves, then reject L' < min_lh.  Returns
    dict(kept, lh, flux, passed uint8 [n], survivors int32 [n] (first n_pass entries valid, ascending), n_pass
    uint64 [4] device counter ([0] = number of survivors))."""
    import torch
    n, T = psi_lc.shape
    if tuple(phi_lc.shape) != (n, T):
        raise ValueError("psi_lc and phi_lc must have one shape [n][T]")
    dev = psi_lc.device
    r = dict(kept=torch.empty(n, dtype=torch.int64, device=dev), lh=torch.empty(n, dtype=torch.float32, device=dev),
             flux=torch.empty(n, dtype=torch.float32, device=dev), passed=torch.empty(n, dtype=torch.uint8, device=dev))
    if compact:
        r["survivors"] = torch.empty(n, dtype=torch.int32, device=dev)
        r["n_pass"] = torch.empty(4, dtype=torch.int64, device=dev)
    cp = params.c()
    _check(lib().kbmod_sigmag_postfilter(_dev(psi_lc, torch.float32), _dev(phi_lc, torch.float32), n, T, C.byref(cp),
                                         _dev(r["kept"]), _dev(r["lh"]), _dev(r["flux"]), _dev(r["passed"]),
                                         _dev(r.get("survivors"), allow_none=True), _dev(r.get("n_pass"), allow_none=True),
                                         _stream(stream)))
    return r


POSTFILTER_STATIC_MAX_LC = 1 << 22


def kbmod_sigmag_postfilter_static(psi_lc, phi_lc, params: SearchParams, out=None, stream=None):
    """kbmod_sigmag_postfilter without device allocations inside the library call: the pass flags and compaction
    counters live in a static device array of the library (at most POSTFILTER_STATIC_MAX_LC lightcurves per call;
    calls that overlap on the GPU race on it).  `out`: optional dict of preallocated outputs (kept int64 [n], lh,
    flux float32 [n], survivors int32 [n], n_survivors int64 [1]); returned (allocated by torch if not given)."""
    import torch
    n, T = psi_lc.shape
    if tuple(phi_lc.shape) != (n, T):
        raise ValueError("psi_lc and phi_lc must have one shape [n][T]")
    dev = psi_lc.device
    r = out if out is not None else dict(
        kept=torch.empty(n, dtype=torch.int64, device=dev), lh=torch.empty(n, dtype=torch.float32, device=dev),
        flux=torch.empty(n, dtype=torch.float32, device=dev), survivors=torch.empty(n, dtype=torch.int32, device=dev),
        n_survivors=torch.empty(1, dtype=torch.int64, device=dev))
    for k, dt in (("kept", torch.int64), ("lh", torch.float32), ("flux", torch.float32), ("survivors", torch.int32)):
        if r[k].numel() < n or r[k].dtype != dt:
            raise ValueError(f"out[{k!r}] must hold {n} elements of {dt}")
    cp = params.c()
    _check(lib().kbmod_sigmag_postfilter_static(_dev(psi_lc, torch.float32), _dev(phi_lc, torch.float32), n, T,
                                                C.byref(cp), _dev(r["kept"]), _dev(r["lh"]), _dev(r["flux"]),
                                                _dev(r["survivors"]), _dev(r["n_survivors"]), _stream(stream)))
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
    _check(lib().kbmod_stamp_moments(s, n, S // 2, thr_ptr, _dev(mom), _dev(keep), _stream(stream)))
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
    for o_ in outs:
        for a in o_:
            assert tuple(a.shape) == (H, W, params.K) and not a.is_cuda and a.is_contiguous()
    _check(lib().kbmod_pipeline_host_batch(n, C.cast(imgs, C.c_void_p), C.cast(vars_, C.c_void_p),
                                           C.cast(masks, C.c_void_p) if masks is not None else None, T, H, W, pp, n_psf,
                                           p.shape[-1], tp, xp, yp, len(x), C.byref(cp), C.cast(o[0], C.c_void_p),
                                           C.cast(o[1], C.c_void_p), C.cast(o[2], C.c_void_p), C.cast(o[3], C.c_void_p),
                                           _dev(arena), arena.numel(), _stream(stream)))
    return outs


def kbmod_measure_smem_gbs(bytes_per_lane: int = 4, stream=None) -> float:
    """Measured shared-memory load bandwidth of the whole GPU in GB/s (roofline denominator; synchronises)."""
    import torch
    out = C.c_double(0.0)
    scratch = torch.zeros(4, dtype=torch.uint8, device="cuda")
    _check(lib().kbmod_measure_smem_gbs(bytes_per_lane, _dev(scratch), C.byref(out), _stream(stream)))
    return float(out.value)


def kbmod_measure_issue_rate(op: int, stream=None) -> float:
    """Warp-instructions per clock per SM of op = 0 FMNMX, 1 IADD3, 2 FADD, 3 the kernels' compare-exchange."""
    import torch
    out = C.c_double(0.0)
    scratch = torch.zeros(4, dtype=torch.uint8, device="cuda")
    _check(lib().kbmod_measure_issue_rate(op, _dev(scratch), C.byref(out), _stream(stream)))
    return float(out.value)


def kbmod_pipeline_host_arena_bytes(T, H, W, n_vel, params: SearchParams) -> int:
    """Upper bound for any list of n_vel velocities."""
    cp = params.c()
    return int(lib().kbmod_pipeline_host_arena_bytes(T, H, W, n_vel, C.byref(cp)))


def kbmod_pipeline_host_arena_bytes_for(T, H, W, times, vx, vy, params: SearchParams) -> int:
    """Exact arena need of kbmod_pipeline_host / one buffer of kbmod_pipeline_host_batch for this grid."""
    (t, x, y), (tp, xp, yp) = _grid(times, vx, vy, T)
    cp = params.c()
    n = int(lib().kbmod_pipeline_host_arena_bytes_for(T, H, W, tp, xp, yp, len(x), C.byref(cp)))
    if n == 0:
        raise KbmodError(-1, lib().kbmod_last_error().decode())
    return n


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
                                     arena.numel(), _stream(stream)))
    return out
