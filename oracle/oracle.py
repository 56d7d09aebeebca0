"""ctypes front end of oracle/kbmod_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It shares nothing with paper_2109_03296_b200 (the CUDA path) and never imports it.
Argument marshalling only; every step is computed in kbmod_oracle.c (see its header for the
PAPER.md citations of each step).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kbmod_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp; no fast-math, so every operation is separately rounded."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
                               "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_num_threads.restype = C.c_int
        _lib.oracle_pct_rank.restype = C.c_int
        _lib.oracle_pct_rank.argtypes = [C.c_float, C.c_int]
        _lib.oracle_pct_value.restype = C.c_float
        _lib.oracle_pct_value.argtypes = [C.POINTER(C.c_float), C.c_int, C.c_float, C.c_int]
    return _lib


@dataclass
class Params:
    """Paper defaults: 25th/75th percentiles, C = 0.7413, n = 2; 8 per pixel (L137)."""

    sigmag_enable: int = 1
    pct_lo: float = 25.0
    pct_hi: float = 75.0
    coeff: float = 0.7413
    n_sigma: float = 2.0
    filter_on: int = 0
    min_lh: float = -np.inf
    min_obs: int = 1
    K: int = 8
    pct_interp: int = 0  # 0 nearest-rank order statistics (R10), 1 linear interpolation (R23)


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def _c(a, dt):
    return None if a is None else np.ascontiguousarray(a, dtype=dt)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def pct_rank(q: float, n: int) -> int:
    return int(lib().oracle_pct_rank(C.c_float(q), n))


def pct_value(sorted_values, q: float, interp: int) -> float:
    """The q-th percentile of an ascending float32 array: nearest rank (interp=0, R10) or linear (interp=1, R23)."""
    s = np.ascontiguousarray(sorted_values, dtype=np.float32)
    return float(lib().oracle_pct_value(_p(s, C.c_float), len(s), C.c_float(q), interp))


def prepare_psi_phi(img, var, mask, psf):
    """O1. Returns psi, phi (float64 [T][H][W]), valid (uint8), psi_abs (float64)."""
    img, var = _c(img, np.float32), _c(var, np.float32)
    mask = _c(mask, np.uint8)
    psf = _c(psf, np.float32)
    T, H, W = img.shape
    n_psf = 1 if psf.ndim == 2 else psf.shape[0]
    k = psf.shape[-1]
    psi, phi = np.empty((T, H, W)), np.empty((T, H, W))
    valid, psi_abs = np.empty((T, H, W), np.uint8), np.empty((T, H, W))
    lib().oracle_prepare_psi_phi(_p(img, C.c_float), _p(var, C.c_float), _p(mask, C.c_uint8), T, H, W,
                                 _p(psf, C.c_float), n_psf, k, _p(psi, C.c_double), _p(phi, C.c_double),
                                 _p(valid, C.c_uint8), _p(psi_abs, C.c_double))
    return psi, phi, valid, psi_abs


def displacements(times, vx, vy):
    """O2. Returns dx, dy int32 [n_vel][T]."""
    times, vx, vy = _c(times, np.float64), _c(vx, np.float32), _c(vy, np.float32)
    T, nv = len(times), len(vx)
    dx, dy = np.empty((nv, T), np.int32), np.empty((nv, T), np.int32)
    lib().oracle_displacements(_p(times, C.c_double), T, _p(vx, C.c_float), _p(vy, C.c_float), nv,
                               _p(dx, C.c_int32), _p(dy, C.c_int32))
    return dx, dy


def interleave(psi, phi):
    """[T][H][W] psi, phi -> float32 [T][H][W][2] (the library's float2 layout)."""
    return np.ascontiguousarray(np.stack([psi, phi], axis=-1), dtype=np.float32)


def search_pixels(psiphi, times, vx, vy, px, py, p: Params):
    """O3-O6 on the listed start pixels. Returns lh, flux (float64 [n][K]), vel_idx, n_obs (int32 [n][K])."""
    psiphi = _c(psiphi, np.float32)
    T, H, W, _ = psiphi.shape
    times, vx, vy = _c(times, np.float64), _c(vx, np.float32), _c(vy, np.float32)
    px, py = _c(px, np.int32), _c(py, np.int32)
    n = len(px)
    lh, flux = np.empty((n, p.K)), np.empty((n, p.K))
    vel, nobs = np.empty((n, p.K), np.int32), np.empty((n, p.K), np.int32)
    lib().oracle_search_pixels(_p(psiphi, C.c_float), T, H, W, _p(times, C.c_double), _p(vx, C.c_float),
                               _p(vy, C.c_float), len(vx), _p(px, C.c_int32), _p(py, C.c_int32), n,
                               p.sigmag_enable, C.c_float(p.pct_lo), C.c_float(p.pct_hi), C.c_float(p.coeff),
                               C.c_float(p.n_sigma), p.filter_on, C.c_float(p.min_lh), p.min_obs, p.K, p.pct_interp,
                               _p(lh, C.c_double), _p(flux, C.c_double), _p(vel, C.c_int32), _p(nobs, C.c_int32))
    return lh, flux, vel, nobs


def search(psiphi, times, vx, vy, p: Params):
    """O3-O6 on every start pixel; outputs shaped [H][W][K]."""
    T, H, W, _ = psiphi.shape
    yy, xx = np.mgrid[0:H, 0:W]
    out = search_pixels(psiphi, times, vx, vy, xx.reshape(-1), yy.reshape(-1), p)
    return tuple(o.reshape(H, W, p.K) for o in out)


def eval_trajectories(psiphi, times, x0, y0, vx, vy, p: Params):
    """Single-trajectory variant. Returns dict of per-trajectory arrays."""
    psiphi = _c(psiphi, np.float32)
    T, H, W, _ = psiphi.shape
    times, vx, vy = _c(times, np.float64), _c(vx, np.float32), _c(vy, np.float32)
    x0, y0 = _c(x0, np.int32), _c(y0, np.int32)
    n = len(x0)
    psi_lc, phi_lc = np.empty((n, T), np.float32), np.empty((n, T), np.float32)
    valid, kept = np.empty(n, np.uint64), np.empty(n, np.uint64)
    lh, flux, nk = np.empty(n), np.empty(n), np.empty(n, np.int32)
    lib().oracle_eval_trajectories(_p(psiphi, C.c_float), T, H, W, _p(times, C.c_double), _p(x0, C.c_int32),
                                   _p(y0, C.c_int32), _p(vx, C.c_float), _p(vy, C.c_float), n, p.sigmag_enable,
                                   C.c_float(p.pct_lo), C.c_float(p.pct_hi), C.c_float(p.coeff),
                                   C.c_float(p.n_sigma), p.filter_on, p.min_obs, p.pct_interp, _p(psi_lc, C.c_float),
                                   _p(phi_lc, C.c_float), _p(valid, C.c_uint64), _p(kept, C.c_uint64),
                                   _p(lh, C.c_double), _p(flux, C.c_double), _p(nk, C.c_int32))
    return dict(psi_lc=psi_lc, phi_lc=phi_lc, valid=valid, kept=kept, lh=lh, flux=flux, n_kept=nk)


def sigmag_filter(psi_lc, phi_lc, p: Params):
    """The post-filter on given lightcurves. `passed` = has a result and L' >= p.min_lh."""
    psi_lc, phi_lc = _c(psi_lc, np.float32), _c(phi_lc, np.float32)
    n, T = psi_lc.shape
    kept, lh, flux, nk = np.empty(n, np.uint64), np.empty(n), np.empty(n), np.empty(n, np.int32)
    passed = np.empty(n, np.uint8)
    lib().oracle_sigmag_filter(_p(psi_lc, C.c_float), _p(phi_lc, C.c_float), n, T, p.sigmag_enable,
                               C.c_float(p.pct_lo), C.c_float(p.pct_hi), C.c_float(p.coeff), C.c_float(p.n_sigma),
                               p.filter_on, p.min_obs, p.pct_interp, C.c_float(p.min_lh), _p(kept, C.c_uint64),
                               _p(lh, C.c_double), _p(flux, C.c_double), _p(nk, C.c_int32), _p(passed, C.c_uint8))
    return dict(kept=kept, lh=lh, flux=flux, n_kept=nk, passed=passed)


def unfiltered_lh(psiphi, times, vx, vy, px, py, vel_idx):
    """Unfiltered sum-LH of every result slot: vel_idx int32 [n][K] -> float64 [n][K]."""
    psiphi = _c(psiphi, np.float32)
    T, H, W, _ = psiphi.shape
    times, vx, vy = _c(times, np.float64), _c(vx, np.float32), _c(vy, np.float32)
    px, py, vel_idx = _c(px, np.int32), _c(py, np.int32), _c(vel_idx, np.int32)
    n, K = vel_idx.shape
    out = np.empty((n, K))
    lib().oracle_unfiltered_lh(_p(psiphi, C.c_float), T, H, W, _p(times, C.c_double), _p(vx, C.c_float),
                               _p(vy, C.c_float), len(vx), _p(px, C.c_int32), _p(py, C.c_int32), n, K,
                               _p(vel_idx, C.c_int32), _p(out, C.c_double))
    return out


def coadd_stamps(img, mask, times, x0, y0, vx, vy, radius: int, epoch_mask=None):
    """O7. Returns mean, median float64 [n][2r+1][2r+1]."""
    img, mask = _c(img, np.float32), _c(mask, np.uint8)
    T, H, W = img.shape
    times, vx, vy = _c(times, np.float64), _c(vx, np.float32), _c(vy, np.float32)
    x0, y0 = _c(x0, np.int32), _c(y0, np.int32)
    em = _c(epoch_mask, np.uint64)
    n, S = len(x0), 2 * radius + 1
    mean, med = np.empty((n, S, S)), np.empty((n, S, S))
    lib().oracle_coadd_stamps(_p(img, C.c_float), _p(mask, C.c_uint8), T, H, W, _p(times, C.c_double),
                              _p(x0, C.c_int32), _p(y0, C.c_int32), _p(vx, C.c_float), _p(vy, C.c_float),
                              _p(em, C.c_uint64), n, radius, _p(mean, C.c_double), _p(med, C.c_double))
    return mean, med


PAPER_MOMENT_THRESHOLDS = (0.5, 0.5, 1.5, 36.5, 36.5)  # x, y, xy, xx, yy "strictly less than"


def stamp_moments(stamps, thresholds=PAPER_MOMENT_THRESHOLDS):
    """N2 (reading R22). stamps [n][S][S]. Returns moments float64 [n][5], keep uint8 [n]."""
    stamps = _c(stamps, np.float32)
    n, S, S2 = stamps.shape
    assert S == S2 and S % 2 == 1
    thr = np.ascontiguousarray(thresholds, dtype=np.float64)
    mom, keep = np.empty((n, 5), np.float64), np.empty(n, np.uint8)
    lib().oracle_stamp_moments(stamps.ctypes.data_as(C.c_void_p), C.c_int(n), C.c_int(S // 2),
                               thr.ctypes.data_as(C.c_void_p), mom.ctypes.data_as(C.c_void_p),
                               keep.ctypes.data_as(C.c_void_p))
    return mom, keep
