"""Seeded synthetic inputs shaped like the paper's DECam difference-image workloads.

This module serves BOTH the CUDA path and the oracle (tests, bench.py, smoke()).  It holds
none of the method's arithmetic: it only draws inputs (image / variance / mask stacks,
epoch times, PSF kernels, velocity grids, candidate trajectory lists).  It imports neither
`oracle/` nor the CUDA binding.

The DECam NEO Survey data of the paper (section 2.1-2.2) is not available;
these stacks stand in for it.  Shapes and cadence follow PAPER.md L37 (2K x 4K CCDs),
L39 (about 5 pointings per night, 5 minutes apart), L43/L47 (>= 4 nights, 20-25 pointings),
L69 (about 180 residual sources per difference image), L167 (92-526 px/day, +-pi/10 about
the ecliptic angle).  The five recipes are the ones BASELINE.json `configs` names; the
concrete numbers are SURVEY.md section 8d's and are restated in DESIGN.md.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

THETA_ECLIPTIC = 4.4  # rad; motion mostly along the 4096-pixel axis


# ----------------------------------------------------------------------------- inputs
@dataclass
class Stack:
    """An aligned difference-image stack: the library's input contract."""

    img: np.ndarray  # [T][H][W] float32
    var: np.ndarray  # [T][H][W] float32
    mask: np.ndarray  # [T][H][W] uint8 (non-zero = bad)
    times: np.ndarray  # [T] float64, days
    psf: np.ndarray  # [k][k] float32
    movers: list = field(default_factory=list)  # dicts: x0, y0, vx, vy, flux
    name: str = ""

    @property
    def shape(self):
        return self.img.shape


def gaussian_psf(sigma: float) -> np.ndarray:
    """Point-sampled Gaussian, radius ceil(3 sigma), unit sum (SURVEY 8c reading R4)."""
    r = int(math.ceil(3.0 * sigma))
    ax = np.arange(-r, r + 1, dtype=np.float64)
    g = np.exp(-0.5 * (ax / sigma) ** 2)
    k = np.outer(g, g)
    k /= k.sum()
    return k.astype(np.float32)


def velocity_grid(n_ang: int, n_spd: int, ang_lo: float, ang_hi: float, spd_lo: float, spd_hi: float):
    """Endpoint-exclusive (angle, speed) grid; vel_idx = a * n_spd + b (SURVEY 8c reading R6)."""
    a = ang_lo + np.arange(n_ang, dtype=np.float64) * (ang_hi - ang_lo) / n_ang
    s = spd_lo + np.arange(n_spd, dtype=np.float64) * (spd_hi - spd_lo) / n_spd
    vx = (s[None, :] * np.cos(a)[:, None]).reshape(-1).astype(np.float32)
    vy = (s[None, :] * np.sin(a)[:, None]).reshape(-1).astype(np.float32)
    return vx, vy


def night_times(per_night, gap_min: float = 5.0) -> np.ndarray:
    """Epoch times in days: night n has per_night[n] pointings `gap_min` minutes apart (L39)."""
    t = [n + j * gap_min / 1440.0 for n, c in enumerate(per_night) for j in range(c)]
    return np.asarray(t, dtype=np.float64)


def _inject(img, times, psf_sigma, x0, y0, vx, vy, flux):
    """Add flux * Gaussian(sigma) sampled at the sub-pixel true position in every epoch."""
    T, H, W = img.shape
    r = int(math.ceil(4.0 * psf_sigma))
    norm = 1.0 / (2.0 * math.pi * psf_sigma * psf_sigma)
    for t in range(T):
        dt = times[t] - times[0]
        xc, yc = x0 + vx * dt, y0 + vy * dt
        ix, iy = int(math.floor(xc + 0.5)), int(math.floor(yc + 0.5))
        xa, xb = max(ix - r, 0), min(ix + r + 1, W)
        ya, yb = max(iy - r, 0), min(iy + r + 1, H)
        if xa >= xb or ya >= yb:
            continue
        xs = np.arange(xa, xb, dtype=np.float64) - xc
        ys = np.arange(ya, yb, dtype=np.float64) - yc
        g = np.exp(-0.5 * (ys[:, None] ** 2 + xs[None, :] ** 2) / psf_sigma**2) * norm
        img[t, ya:yb, xa:xb] += (flux * g).astype(np.float32)


def _epochs_on_chip(times, H, W, x0, y0, vx, vy):
    dt = times - times[0]
    x, y = x0 + vx * dt, y0 + vy * dt
    return int(np.sum((x >= 0) & (x < W) & (y >= 0) & (y < H)))


# ----------------------------------------------------------------------------- configs
def config1_tiny(seed: int = 0) -> Stack:
    """BASELINE.json configs[0]: 64x64, T=5, sigma=1 noise, var=1, PSF sigma 1 (7x7), one mover."""
    rng = np.random.default_rng(seed)
    T, H, W = 5, 64, 64
    times = np.array([0.0, 0.5, 1.0, 1.5, 2.0])
    img = rng.standard_normal((T, H, W), dtype=np.float32)
    var = np.ones((T, H, W), dtype=np.float32)
    mask = np.zeros((T, H, W), dtype=np.uint8)
    mv = dict(x0=20.0, y0=30.0, vx=20.0, vy=5.0, flux=100.0)
    _inject(img, times, 1.0, **mv)
    return Stack(img, var, mask, times, gaussian_psf(1.0), [mv], "config1_tiny")


def config1_grid():
    return velocity_grid(16, 16, -math.pi / 4, math.pi / 4, 0.0, 40.0)


def config2_medium(seed: int = 1, size: int = 512, n_movers: int = 20) -> Stack:
    """BASELINE.json configs[1]: 512x512, T=10 uneven over 3 days, gradient variance, 1% mask."""
    rng = np.random.default_rng(seed)
    T, H, W = 10, size, size
    times = np.sort(np.concatenate([[0.0, 3.0], 3.0 * rng.random(T - 2)]))
    yy, xx = np.mgrid[0:H, 0:W]
    v2d = (0.5 + 1.5 * (xx + yy) / float(W + H - 2)).astype(np.float32)
    var = np.broadcast_to(v2d, (T, H, W)).copy()
    img = rng.standard_normal((T, H, W), dtype=np.float32) * np.sqrt(var)
    mask = (rng.random((T, H, W), dtype=np.float32) < 0.01).astype(np.uint8)
    movers = []
    while len(movers) < n_movers:
        spd, ang = rng.uniform(50.0, 300.0), rng.uniform(0.0, 2 * math.pi)
        mv = dict(x0=float(rng.integers(0, W)), y0=float(rng.integers(0, H)),
                  vx=spd * math.cos(ang), vy=spd * math.sin(ang), flux=rng.uniform(30.0, 200.0))
        if _epochs_on_chip(times, H, W, mv["x0"], mv["y0"], mv["vx"], mv["vy"]) >= 6:
            movers.append(mv)
            _inject(img, times, 1.5, **mv)
    return Stack(img, var, mask, times, gaussian_psf(1.5), movers, "config2_medium")


def config2_grid():
    return velocity_grid(64, 32, 0.0, 2 * math.pi, 50.0, 300.0)


def decam_stack(seed: int, per_night, H: int = 4096, W: int = 2048, n_movers: int = 200,
                flux_range=(500.0, 5000.0), flux_log: bool = True, n_stars: int = 500,
                psf_sigma: float = 1.8, name: str = "config3_decam") -> Stack:
    """BASELINE.json configs[2]/[3]: DECam-CCD-shaped difference stack (SURVEY 8d recipe).

    Sky variance 300 ADU with +-10 % per-epoch scatter and a +-5 % smooth gradient; 2 % masked
    (static discs, bad columns, per-epoch pixels); subtraction dipoles at fixed star positions;
    0.1 % single-epoch cosmic-ray pixels; injected movers.  H, W, n_stars scale down for tests.
    """
    rng = np.random.default_rng(seed)
    times = night_times(per_night)
    T = len(times)
    g_t = np.clip(rng.standard_normal(T), -2.0, 2.0)
    v_t = 300.0 * (1.0 + 0.1 * g_t)
    yy = np.arange(H, dtype=np.float32)[:, None] / max(H - 1, 1)
    xx = np.arange(W, dtype=np.float32)[None, :] / max(W - 1, 1)
    grad = (1.0 + 0.05 * (xx + yy - 1.0)).astype(np.float32)
    var = np.empty((T, H, W), dtype=np.float32)
    img = np.empty((T, H, W), dtype=np.float32)
    for t in range(T):
        var[t] = np.float32(v_t[t]) * grad
        img[t] = rng.standard_normal((H, W), dtype=np.float32) * np.sqrt(var[t])

    # --- mask: 1 % static discs, 0.5 % static bad columns, 0.5 % per-epoch pixels
    static = np.zeros((H, W), dtype=np.uint8)
    n_disc = max(1, int(round(0.01 * H * W / (math.pi * 63.0))))
    for _ in range(n_disc):
        cx, cy, r = rng.integers(0, W), rng.integers(0, H), rng.uniform(3.0, 12.0)
        ri = int(math.ceil(r))
        ya, yb, xa, xb = max(cy - ri, 0), min(cy + ri + 1, H), max(cx - ri, 0), min(cx + ri + 1, W)
        py, px = np.mgrid[ya:yb, xa:xb]
        static[ya:yb, xa:xb] |= ((px - cx) ** 2 + (py - cy) ** 2 <= r * r).astype(np.uint8)
    for c in rng.choice(W, size=max(1, int(round(0.005 * W))), replace=False):
        static[:, c] = 1
    mask = np.empty((T, H, W), dtype=np.uint8)
    for t in range(T):
        mask[t] = static | (rng.random((H, W), dtype=np.float32) < 0.005).astype(np.uint8)

    # --- subtraction residuals: dipoles at fixed star positions, +-5 sigma_pix peak (L69, L85)
    sx, sy = rng.uniform(0, W, n_stars), rng.uniform(0, H, n_stars)
    sep, ori = rng.uniform(1.0, 2.0, n_stars), rng.uniform(0, 2 * math.pi, n_stars)
    r = int(math.ceil(4.0 * psf_sigma)) + 2
    for t in range(T):
        amp = 5.0 * math.sqrt(v_t[t]) * (1.0 + 0.2 * rng.uniform(-1.0, 1.0, n_stars))
        for s in range(n_stars):
            ix, iy = int(round(sx[s])), int(round(sy[s]))
            xa, xb, ya, yb = max(ix - r, 0), min(ix + r + 1, W), max(iy - r, 0), min(iy + r + 1, H)
            if xa >= xb or ya >= yb:
                continue
            ux, uy = 0.5 * sep[s] * math.cos(ori[s]), 0.5 * sep[s] * math.sin(ori[s])
            xs = np.arange(xa, xb, dtype=np.float64)[None, :]
            ys = np.arange(ya, yb, dtype=np.float64)[:, None]
            gp = np.exp(-0.5 * ((xs - sx[s] - ux) ** 2 + (ys - sy[s] - uy) ** 2) / psf_sigma**2)
            gm = np.exp(-0.5 * ((xs - sx[s] + ux) ** 2 + (ys - sy[s] + uy) ** 2) / psf_sigma**2)
            img[t, ya:yb, xa:xb] += (amp[s] * (gp - gm)).astype(np.float32)

    # --- cosmic rays: 0.1 % of pixels per epoch, single pixel, 10-50 sigma_pix
    n_cr = int(round(0.001 * H * W))
    for t in range(T):
        idx = rng.integers(0, H * W, n_cr)
        a = rng.uniform(10.0, 50.0, n_cr).astype(np.float32)
        flat = img[t].reshape(-1)
        flat[idx] += a * np.sqrt(var[t].reshape(-1)[idx])

    # --- movers
    movers = []
    need = (T + 1) // 2
    while len(movers) < n_movers:
        spd = rng.uniform(92.0, 526.0)
        ang = THETA_ECLIPTIC + rng.uniform(-math.pi / 10, math.pi / 10)
        if flux_log:
            flux = math.exp(rng.uniform(math.log(flux_range[0]), math.log(flux_range[1])))
        else:
            flux = rng.uniform(*flux_range)
        mv = dict(x0=float(rng.integers(0, W)), y0=float(rng.integers(0, H)),
                  vx=spd * math.cos(ang), vy=spd * math.sin(ang), flux=flux)
        if _epochs_on_chip(times, H, W, mv["x0"], mv["y0"], mv["vx"], mv["vy"]) >= need:
            movers.append(mv)
            _inject(img, times, psf_sigma, **mv)
    return Stack(img, var, mask, times, gaussian_psf(psf_sigma), movers, name)


def config3_decam(seed: int = 2, H: int = 4096, W: int = 2048, **kw) -> Stack:
    return decam_stack(seed, (7, 6, 7, 6), H, W, name="config3_decam", **kw)


def config3_grid(n_ang: int = 128, n_spd: int = 64):
    return velocity_grid(n_ang, n_spd, THETA_ECLIPTIC - math.pi / 10, THETA_ECLIPTIC + math.pi / 10, 92.0, 526.0)


def paper_grid():
    """The paper's own search grid: 512 speed steps over 92-550 px/day x 256 angle steps within
    +-pi/10 of the ecliptic angle = 131072 velocities (about 1.1e12 trajectories on a 2K x 4K CCD, L133)."""
    return velocity_grid(256, 512, THETA_ECLIPTIC - math.pi / 10, THETA_ECLIPTIC + math.pi / 10, 92.0, 550.0)


def config4_heavy(seed: int = 3, H: int = 4096, W: int = 2048, n_movers: int = 1000, **kw) -> Stack:
    return decam_stack(seed, (9, 8, 8, 9, 8, 8), H, W, n_movers=n_movers, flux_range=(10.0, 100.0),
                       flux_log=False, name="config4_heavy", **kw)


def config4_grid(n_ang: int = 256, n_spd: int = 128):
    return config3_grid(n_ang, n_spd)


def config5_trajectories(seed: int, H: int, W: int, n: int = 100_000):
    """BASELINE.json configs[4]: random start pixels, speeds in [92,526) px/day, angle theta_e +- pi/10."""
    rng = np.random.default_rng(seed)
    x0 = rng.integers(0, W, n).astype(np.int32)
    y0 = rng.integers(0, H, n).astype(np.int32)
    spd = rng.uniform(92.0, 526.0, n)
    ang = THETA_ECLIPTIC + rng.uniform(-math.pi / 10, math.pi / 10, n)
    return x0, y0, (spd * np.cos(ang)).astype(np.float32), (spd * np.sin(ang)).astype(np.float32)


def outlier_lightcurves(seed: int, psi_lc: np.ndarray, phi_lc: np.ndarray, frac: float = 0.2, n_sig: float = 10.0):
    """configs[4]: replace `frac` of the epochs (i.i.d.) by psi += +-n_sig * sqrt(phi)."""
    rng = np.random.default_rng(seed)
    hit = rng.random(psi_lc.shape) < frac
    sign = np.where(rng.random(psi_lc.shape) < 0.5, -1.0, 1.0)
    out = psi_lc.astype(np.float32).copy()
    out[hit] += (sign[hit] * n_sig * np.sqrt(phi_lc[hit])).astype(np.float32)
    return out, hit


def random_stack(seed: int, T: int, H: int, W: int, psf_sigma: float = 1.0, mask_frac: float = 0.05,
                 t_span: float = 2.0) -> Stack:
    """Small generic noise stack for unit tests (ragged sizes, random masks, uneven times)."""
    rng = np.random.default_rng(seed)
    times = np.sort(np.concatenate([[0.0], t_span * rng.random(T - 1)])) if T > 1 else np.zeros(1)
    var = rng.uniform(0.5, 2.0, (T, H, W)).astype(np.float32)
    img = rng.standard_normal((T, H, W), dtype=np.float32) * np.sqrt(var)
    mask = (rng.random((T, H, W)) < mask_frac).astype(np.uint8)
    return Stack(img, var, mask, times.astype(np.float64), gaussian_psf(psf_sigma), [], f"random{seed}")
