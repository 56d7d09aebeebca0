"""GPU-vs-oracle comparison protocol.

Bit-exact: displacement tables, validity bitmaps, kept sets, (pixel, vel_idx) identity, n_obs.
Floating point: |L_gpu - L'| <= 1e-4 |L'| + 1e-5 * sum_kept|psi| / sqrt(sum_kept phi)  (north_star:
1e-4 relative in float32; the second term covers cancellation near L = 0), same form for flux.
Top-K sets must be equal except for members within that tolerance of the boundary (the K-th value
or min_lh).  The oracle always runs on the GPU-produced float32 psi/phi stack so that prep rounding
does not leak into search parity.
"""
import numpy as np

RTOL = 1e-4
ATOL_SCALE = 1e-5


def _bits(mask, T):
    m = np.asarray(mask).astype(np.uint64)
    return ((m[:, None] >> np.arange(T, dtype=np.uint64)[None, :]) & np.uint64(1)).astype(bool)


def score_tolerances(ev, T):
    """Per-trajectory absolute tolerances for L and flux from the oracle's own lightcurves."""
    kept = _bits(ev["kept"], T)
    ps = np.where(kept, np.abs(ev["psi_lc"].astype(np.float64)), 0.0).sum(1)
    ph = np.where(kept, ev["phi_lc"].astype(np.float64), 0.0).sum(1)
    with np.errstate(divide="ignore", invalid="ignore"):
        tl = RTOL * np.abs(ev["lh"]) + ATOL_SCALE * np.where(ph > 0, ps / np.sqrt(ph), 0.0)
        tf = RTOL * np.abs(ev["flux"]) + ATOL_SCALE * np.where(ph > 0, ps / ph, 0.0)
    return tl, tf


def check_entries(O, psiphi, times, vx, vy, p, px, py, g_lh, g_flux, g_vel, g_nobs):
    """Every filled GPU slot must be the oracle's evaluation of that (pixel, velocity): L, flux to
    tolerance, n_obs exactly, L' >= min_lh to tolerance, list sorted.  g_* are [n][K] numpy."""
    T = psiphi.shape[0]
    n, K = g_vel.shape
    filled = g_vel >= 0
    # unfilled slots carry the sentinels and sit behind the filled ones
    assert np.all(np.isneginf(g_lh[~filled])) and np.all(g_flux[~filled] == 0) and np.all(g_nobs[~filled] == 0)
    assert np.all(filled[:, :-1] >= filled[:, 1:]), "filled slots must be a prefix"
    ii, kk = np.nonzero(filled)
    if len(ii) == 0:
        return 0
    v = g_vel[ii, kk]
    assert v.max() < len(vx)
    ev = O.eval_trajectories(psiphi, times, px[ii], py[ii], vx[v], vy[v], p)
    tl, tf = score_tolerances(ev, T)
    dl = np.abs(g_lh[ii, kk].astype(np.float64) - ev["lh"])
    df = np.abs(g_flux[ii, kk].astype(np.float64) - ev["flux"])
    bad = ~(dl <= tl)
    assert not bad.any(), f"L mismatch at {np.nonzero(bad)[0][:5]}: gpu {g_lh[ii, kk][bad][:5]} oracle {ev['lh'][bad][:5]}"
    bad = ~(df <= tf)
    assert not bad.any(), f"flux mismatch: gpu {g_flux[ii, kk][bad][:5]} oracle {ev['flux'][bad][:5]}"
    assert np.array_equal(g_nobs[ii, kk], ev["n_kept"]), "n_obs (kept count) must be bit-exact"
    assert np.all(ev["lh"] + tl >= p.min_lh), "a returned trajectory is below min_lh"
    # order: L descending; equal L -> ascending velocity index
    a, b = g_lh[:, :-1], g_lh[:, 1:]
    both = filled[:, 1:]
    assert np.all((a >= b) | ~both), "top-K list not sorted"
    tie = both & (a == b)
    assert np.all(g_vel[:, :-1][tie] < g_vel[:, 1:][tie]), "ties must be ordered by velocity index"
    return len(ii)


def compare_topk(O, psiphi, times, vx, vy, p, px, py, gpu, ora):
    """gpu, ora: tuples (lh, flux, vel, nobs) of [n][K] numpy arrays for the same pixel list.
    Returns dict(n_pix, n_entries, n_exact_pix, n_tie_pix)."""
    g_lh, g_flux, g_vel, g_nobs = [np.asarray(a) for a in gpu]
    o_lh, o_flux, o_vel, o_nobs = [np.asarray(a) for a in ora]
    T = psiphi.shape[0]
    n, K = g_vel.shape
    n_entries = check_entries(O, psiphi, times, vx, vy, p, px, py, g_lh, g_flux, g_vel, g_nobs)
    same = np.all(g_vel == o_vel, axis=1)
    n_tie = 0
    for i in np.nonzero(~same)[0]:
        # the lists differ: only acceptable for members within tolerance of the boundary
        gs, os_ = set(g_vel[i][g_vel[i] >= 0].tolist()), set(o_vel[i][o_vel[i] >= 0].tolist())
        diff = sorted(gs ^ os_)
        if diff:
            ev = O.eval_trajectories(psiphi, times, np.full(len(diff), px[i]), np.full(len(diff), py[i]),
                                     vx[diff], vy[diff], p)
            tl, _ = score_tolerances(ev, T)
            full_g, full_o = (g_vel[i] >= 0).all(), (o_vel[i] >= 0).all()
            bounds = [float(p.min_lh)]
            if full_g:
                bounds.append(float(g_lh[i, K - 1]))
            if full_o:
                bounds.append(float(o_lh[i, K - 1]))
            for j, vv in enumerate(diff):
                near = any(abs(ev["lh"][j] - b) <= 2 * tl[j] + 1e-12 for b in bounds if np.isfinite(b))
                assert near, (f"pixel ({px[i]},{py[i]}): velocity {vv} (L'={ev['lh'][j]}) is in one top-K list only "
                              f"and not within tolerance of the boundary {bounds}; gpu {g_vel[i]} oracle {o_vel[i]}")
        else:
            # same members, different order: neighbours must be within tolerance of each other
            order_ok = np.abs(np.sort(g_lh[i])[::-1] - np.sort(o_lh[i])[::-1].astype(np.float32))
            assert np.all((order_ok <= 2 * RTOL * np.abs(o_lh[i]) + 1e-4) | ~np.isfinite(o_lh[i]))
        n_tie += 1
    return dict(n_pix=n, n_entries=n_entries, n_exact_pix=int(same.sum()), n_tie_pix=n_tie)


def oracle_params(O, sp):
    """SearchParams (binding) -> oracle.Params, field by field."""
    return O.Params(sigmag_enable=sp.sigmag_enable, pct_lo=sp.pct_lo, pct_hi=sp.pct_hi, coeff=sp.sigmag_coeff,
                    n_sigma=sp.n_sigma, filter_on=sp.filter_on, min_lh=sp.min_lh, min_obs=sp.min_obs, K=sp.K,
                    pct_interp=getattr(sp, "pct_interp", 0))


def check_prep(O, stack, g_psiphi, psf=None):
    """GPU psi/phi [T][H][W][2] (numpy float32) against the oracle: validity bit-exact,
    |dpsi| <= 1e-5 sum|P I w|, |dphi| <= 1e-5 phi."""
    psf = stack.psf if psf is None else psf
    psi, phi, valid, psi_abs = O.prepare_psi_phi(stack.img, stack.var, stack.mask, psf)
    g_psi, g_phi = g_psiphi[..., 0].astype(np.float64), g_psiphi[..., 1].astype(np.float64)
    inv = valid == 0
    assert np.all(g_psi[inv] == 0) and np.all(g_phi[inv] == 0), "invalid pixels must be (0, 0)"
    assert np.all(g_phi[~inv] > 0) or np.all(phi[~inv][g_phi[~inv] <= 0] <= 0), "validity bitmap differs"
    assert np.all(np.abs(g_psi - psi) <= 1e-5 * psi_abs + 1e-30), float(np.max(np.abs(g_psi - psi) / (psi_abs + 1e-30)))
    assert np.all(np.abs(g_phi - phi) <= 1e-5 * phi + 1e-30), float(np.max(np.abs(g_phi - phi) / (phi + 1e-30)))
    return int((~inv).sum())
