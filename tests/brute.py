"""Numpy brute force used to PIN the oracle (tests only; tiny stacks).

Structurally different from oracle/kbmod_oracle.c: instead of walking one trajectory at a time
it builds, per velocity, the T shifted psi/phi planes ("shift and stack") and
evaluates every start pixel at once with array operations; percentiles come from np.sort.
"""
import math

import numpy as np


def shifted(plane, dx, dy, fill=0.0):
    """out[y, x] = plane[y + dy, x + dx] where on-image, else `fill`."""
    H, W = plane.shape
    out = np.full((H, W), fill, dtype=plane.dtype)
    ya, yb = max(0, -dy), min(H, H - dy)
    xa, xb = max(0, -dx), min(W, W - dx)
    if ya < yb and xa < xb:
        out[ya:yb, xa:xb] = plane[ya + dy:yb + dy, xa + dx:xb + dx]
    return out


def round_half_up(a):
    return np.floor(np.asarray(a, dtype=np.float64) + 0.5).astype(np.int64)


def rank(q, n):
    return min(max(int(math.ceil(float(q) * n / 100.0)) - 1, 0), n - 1)


def all_scores(psi, phi, times, vx, vy, sigmag=True, pct=(25.0, 75.0), coeff=0.7413, n_sigma=2.0,
               filter_on=0, min_obs=1):
    """Returns L, flux (float64 [n_vel][H][W], NaN = no result), n_kept and kept masks (uint64)."""
    psi = np.asarray(psi, np.float32)
    phi = np.asarray(phi, np.float32)
    T, H, W = psi.shape
    nv = len(vx)
    dt = np.asarray(times, np.float64) - times[0]
    L = np.full((nv, H, W), np.nan)
    F = np.full((nv, H, W), np.nan)
    NK = np.zeros((nv, H, W), np.int32)
    KEPT = np.zeros((nv, H, W), np.uint64)
    for v in range(nv):
        dx = round_half_up(np.float64(np.float32(vx[v])) * dt)
        dy = round_half_up(np.float64(np.float32(vy[v])) * dt)
        ps = np.stack([shifted(psi[t], int(dx[t]), int(dy[t])) for t in range(T)])
        ph = np.stack([shifted(phi[t], int(dx[t]), int(dy[t])) for t in range(T)])
        valid = ph > 0
        n = valid.sum(0)
        with np.errstate(divide="ignore", invalid="ignore"):
            f = (ps / np.sqrt(ph) if filter_on else ps / ph).astype(np.float32)
        kept = valid.copy()
        if sigmag:
            s = np.sort(np.where(valid, f, np.float32(np.inf)), axis=0)
            r_lo = np.vectorize(lambda m: rank(pct[0], m) if m > 0 else 0)(n)
            r_md = np.vectorize(lambda m: rank(50.0, m) if m > 0 else 0)(n)
            r_hi = np.vectorize(lambda m: rank(pct[1], m) if m > 0 else 0)(n)
            take = lambda r: np.take_along_axis(s, r[None].astype(np.int64), 0)[0]
            p_lo, p_md, p_hi = take(r_lo), take(r_md), take(r_hi)
            with np.errstate(invalid="ignore"):
                w = np.float32(n_sigma) * (np.float32(coeff) * (p_hi - p_lo).astype(np.float32)).astype(np.float32)
                lo, hi = (p_md - w).astype(np.float32), (p_md + w).astype(np.float32)
                kept = valid & (f >= lo[None]) & (f <= hi[None])
        sp = np.where(kept, ps.astype(np.float64), 0.0).sum(0)
        sf = np.where(kept, ph.astype(np.float64), 0.0).sum(0)
        ok = n >= max(1, min_obs)
        with np.errstate(divide="ignore", invalid="ignore"):
            L[v] = np.where(ok, sp / np.sqrt(sf), np.nan)
            F[v] = np.where(ok, sp / sf, np.nan)
        NK[v] = np.where(ok, kept.sum(0), 0)
        bits = np.zeros((H, W), np.uint64)
        for t in range(T):
            bits |= kept[t].astype(np.uint64) << np.uint64(t)
        KEPT[v] = np.where(ok, bits, np.uint64(0))
    return L, F, NK, KEPT


def topk(L, F, NK, K, min_lh=-np.inf):
    """Full sort of all candidates per pixel by (L desc, vel_idx asc)."""
    nv, H, W = L.shape
    lh = np.full((H, W, K), -np.inf)
    fl = np.zeros((H, W, K))
    vi = np.full((H, W, K), -1, np.int32)
    no = np.zeros((H, W, K), np.int32)
    for y in range(H):
        for x in range(W):
            c = [(-L[v, y, x], v) for v in range(nv) if not np.isnan(L[v, y, x]) and L[v, y, x] >= min_lh]
            c.sort()
            for k, (negl, v) in enumerate(c[:K]):
                lh[y, x, k], fl[y, x, k], vi[y, x, k], no[y, x, k] = -negl, F[v, y, x], v, NK[v, y, x]
    return lh, fl, vi, no
