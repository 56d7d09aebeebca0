"""GPU parity tests of the round-2 entry points: row-band search, the explicit plan shared by several
streams (N3), interpolated percentiles and the unfiltered sum-LH (N4), the post-filter's reject flag and compacted
survivor list (N1), the moment filter fused into the coadd kernel (N2), thread-state release.  Every expected value
is the oracle's; protocol in tests/parity.py."""
import numpy as np
import pytest

from paper_2109_03296_b200 import synth
from tests import parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def kb():
    import torch
    import paper_2109_03296_b200 as kb_
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (there is no CPU fallback)"
    kb_.binding.lib()
    return kb_


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _prep(kb, st):
    return kb.kbmod_prepare_psi_phi(_cuda(st.img), _cuda(st.var), _cuda(st.mask) if st.mask is not None else None, st.psf)


@pytest.fixture(scope="module")
def decam_small(kb):
    st = synth.decam_stack(21, (7, 6, 7, 6), H=700, W=520, n_movers=40, n_stars=50)
    return st, _prep(kb, st)


# ------------------------------------------------------------------------------------------- N3: row bands, plans
@pytest.mark.parametrize("algo,min_lh", [("pruned", 10.0), ("direct", 10.0), ("direct", -np.inf)])
def test_row_bands_concatenate_to_the_full_search(kb, oracle, decam_small, algo, min_lh):
    """start pixels partitioned into row bands, every band searched on its own (as one rank of a multi-GPU
    run would), results concatenated -- must equal the full search bit for bit; one band is also checked against the
    oracle directly.  Band edges are not multiples of the 32-row tile."""
    import torch
    st, d = decam_small
    T, H, W = st.img.shape
    vx, vy = synth.config3_grid(64, 32)
    sp = kb.SearchParams(K=8, min_obs=13, min_lh=min_lh, algo=kb.ALGO_PRUNED if algo == "pruned" else kb.ALGO_DIRECT)
    full = [o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    edges = [0, 37, 300, 301, 655, H]
    parts = [[o.clone() for o in kb.kbmod_search_rows(d, st.times, vx, vy, sp, rows=(a, b))] for a, b in zip(edges[:-1], edges[1:])]
    for k in range(4):
        assert torch.equal(torch.cat([p[k] for p in parts], dim=0), full[k])
    assert int((full[2] >= 0).sum()) > 100
    # the band [301, 655) against the oracle, every pixel of 40 of its rows
    a, b = edges[3], edges[4]
    yy, xx = np.mgrid[a:a + 40, 0:W]
    px, py = xx.reshape(-1).astype(np.int32), yy.reshape(-1).astype(np.int32)
    psiphi = d.cpu().numpy()
    op = parity.oracle_params(oracle, sp)
    ora = oracle.search_pixels(psiphi, st.times, vx, vy, px, py, op)
    g = [o.cpu().numpy()[py - a, px] for o in parts[3]]
    parity.compare_topk(oracle, psiphi, st.times, vx, vy, op, px, py, g, ora)
    # an empty band is legal
    e = kb.kbmod_search_rows(d, st.times, vx, vy, sp, rows=(10, 10))
    assert tuple(e[0].shape) == (0, W, 8)


def test_one_plan_many_streams(kb, decam_small):
    """N3 (60 CCDs per pointing group, one grid and one set of times): ONE plan, three stacks
    searched concurrently on three streams with three workspaces; each result equals the one-call kbmod_search."""
    import torch
    st, d0 = decam_small
    T, H, W = st.img.shape
    vx, vy = synth.config3_grid(64, 32)
    sp = kb.SearchParams(K=4, min_obs=13, min_lh=10.0)
    stacks = [d0] + [_prep(kb, synth.decam_stack(30 + i, (7, 6, 7, 6), H=H, W=W, n_movers=20, n_stars=30)) for i in range(2)]
    ref = [[o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)] for d in stacks]
    plan = kb.Plan(T, H, W, st.times, vx, vy, sp)
    assert plan.info()["algo"] == kb.ALGO_PRUNED
    streams = [torch.cuda.Stream() for _ in stacks]
    wss = [torch.empty(plan.workspace_bytes(), dtype=torch.uint8, device="cuda") for _ in stacks]
    torch.cuda.synchronize()
    outs = [plan.search(d, workspace=w, stream=s) for d, w, s in zip(stacks, wss, streams)]
    torch.cuda.synchronize()
    for r, o in zip(ref, outs):
        for a, b in zip(r, o):
            assert torch.equal(a, b)
    assert not torch.equal(outs[0][2], outs[1][2])
    plan.destroy()


def test_release_thread_state_then_search_again(kb, decam_small):
    """The per-thread conveniences (cached plan, phase-timing events, batch copy streams) have an owner:
    kbmod_release_thread_state() frees them and the next calls rebuild what they need."""
    import torch
    st, d = decam_small
    T, H, W = st.img.shape
    vx, vy = synth.config3_grid(32, 16)
    sp = kb.SearchParams(K=2, min_obs=13, min_lh=10.0)
    kb.kbmod_search_phase_timing(True)
    a = [o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    assert kb.kbmod_search_phase_ms()["gather"] > 0
    pin = lambda x: torch.from_numpy(np.ascontiguousarray(x)).pin_memory()
    outs = [tuple(torch.empty((H, W, 2), dtype=dt).pin_memory() for dt in (torch.float32, torch.float32, torch.int32, torch.int32))
            for _ in range(2)]
    arena = torch.empty(2 * kb.kbmod_pipeline_host_arena_bytes_for(T, H, W, st.times, vx, vy, sp), dtype=torch.uint8, device="cuda")
    hin = (pin(st.img), pin(st.var), pin(st.mask))
    kb.kbmod_pipeline_host_batch([hin, hin], st.psf, st.times, vx, vy, sp, outs, arena)
    kb.kbmod_release_thread_state()
    kb.kbmod_release_thread_state()
    with pytest.raises(kb.KbmodError):
        kb.kbmod_search_phase_ms()                      # the timing events are gone
    b = kb.kbmod_search(d, st.times, vx, vy, sp)          # plan rebuilt
    kb.kbmod_pipeline_host_batch([hin, hin], st.psf, st.times, vx, vy, sp, outs, arena)   # streams rebuilt
    kb.kbmod_search_phase_timing(False)
    for x, y in zip(a, b):
        assert torch.equal(x, y)
    assert torch.equal(outs[0][2].cuda(), b[2]) and torch.equal(outs[1][0].cuda(), b[0])


# ------------------------------------------------------------------------------------------- N4: variants
@pytest.mark.parametrize("algo", ["direct", "pruned"])
@pytest.mark.parametrize("T,pct", [(26, (25.0, 75.0)), (10, (10.0, 90.0)), (7, (25.0, 75.0))])
def test_search_interpolated_percentiles(kb, oracle, algo, T, pct):
    """Reading R23 (pct_interp = 1): the search with linear-interpolated percentiles against the oracle, every pixel,
    both kernels (the pruned kernel's kept-count bound m(n) changes with the definition)."""
    st = synth.random_stack(600 + T, T, 40, 90, mask_frac=0.08, t_span=2.0)
    rng = np.random.default_rng(600 + T)
    st.img[rng.random(st.img.shape) < 0.02] *= 15.0
    vx = rng.uniform(-15, 15, 50).astype(np.float32)
    vy = rng.uniform(-15, 15, 50).astype(np.float32)
    d = _prep(kb, st)
    psiphi = d.cpu().numpy()
    H, W = 40, 90
    yy, xx = np.mgrid[0:H, 0:W]
    px, py = xx.reshape(-1).astype(np.int32), yy.reshape(-1).astype(np.int32)
    sp = kb.SearchParams(K=4, min_obs=max(1, T // 2), min_lh=2.5, pct_lo=pct[0], pct_hi=pct[1], pct_interp=1,
                         algo=kb.ALGO_PRUNED if algo == "pruned" else kb.ALGO_DIRECT)
    g = [o.cpu().numpy().reshape(H * W, -1) for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    op = parity.oracle_params(oracle, sp)
    assert op.pct_interp == 1
    ora = oracle.search_pixels(psiphi, st.times, vx, vy, px, py, op)
    r = parity.compare_topk(oracle, psiphi, st.times, vx, vy, op, px, py, g, ora)
    assert r["n_entries"] > 500
    # the definition matters: nearest rank gives different kept sets on a good share of the trajectories
    g0 = kb.kbmod_search(d, st.times, vx, vy, kb.SearchParams(**{**sp.__dict__, "pct_interp": 0}))
    if T != 7 or pct != (25.0, 75.0):   # (n = 5, 9 put the positions on integers: test_oracle_pins)
        assert (g0[3].cpu().numpy().reshape(H * W, -1) != g[3]).mean() > 0.01


def test_interpolated_percentiles_lightcurve_tools(kb, oracle):
    rng = np.random.default_rng(610)
    n, T = 50000, 26
    phi = rng.uniform(0.5, 2.0, (n, T)).astype(np.float32)
    psi = (rng.standard_normal((n, T)) * np.sqrt(phi)).astype(np.float32)
    phi[rng.random((n, T)) < 0.1] = 0.0
    psi, _ = synth.outlier_lightcurves(T, psi, phi, 0.15, 9.0)
    for fon in (0, 1):
        sp = kb.SearchParams(K=1, min_obs=3, pct_interp=1, filter_on=fon)
        g = {k: v.cpu().numpy() for k, v in kb.kbmod_sigmag_filter(_cuda(psi), _cuda(phi), sp).items()}
        o = oracle.sigmag_filter(psi, phi, parity.oracle_params(oracle, sp))
        assert np.array_equal(g["kept"].view(np.uint64), o["kept"])
        has = o["n_kept"] > 0
        tl, _ = parity.score_tolerances(dict(o, psi_lc=psi, phi_lc=phi), T)
        assert np.all(np.abs(g["lh"][has] - o["lh"][has]) <= tl[has])


@pytest.mark.parametrize("algo,rows", [("pruned", None), ("direct", None), ("pruned", (100, 333))])
def test_unfiltered_lh_beside_filtered(kb, oracle, decam_small, algo, rows):
    """the unfiltered sum-LH next to sum-LH' for every returned trajectory; equals the oracle's
    plain sum over all valid epochs (and is >= what an outlier-free lightcurve gives after the clip: not asserted)."""
    st, d = decam_small
    T, H, W = st.img.shape
    vx, vy = synth.config3_grid(64, 32)
    sp = kb.SearchParams(K=8, min_obs=13, min_lh=10.0, algo=kb.ALGO_PRUNED if algo == "pruned" else kb.ALGO_DIRECT)
    lh, flux, vel, nobs = kb.kbmod_search(d, st.times, vx, vy, sp, rows=rows)
    raw = kb.kbmod_search_unfiltered_lh(kb.kbmod_search.last_workspace, vel).cpu().numpy()
    r0, r1 = rows or (0, H)
    v = vel.cpu().numpy()
    yy, xx = np.mgrid[r0:r1, 0:W]
    has = (v[..., 0] >= 0)
    px, py = xx[has].astype(np.int32), yy[has].astype(np.int32)
    assert len(px) > 100
    o = oracle.unfiltered_lh(d.cpu().numpy(), st.times, vx, vy, px, py, v[has])
    g = raw[has]
    filled = v[has] >= 0
    assert np.all(np.isneginf(g[~filled])) and np.all(np.isneginf(o[~filled]))
    assert np.all(np.abs(g[filled] - o[filled]) <= 1e-4 * np.abs(o[filled]) + 1e-5)
    assert np.all(np.isneginf(raw[~has]))
    # the explicit-plan form gives the same numbers
    plan = kb.Plan(T, H, W, st.times, vx, vy, sp, rows=rows)
    out = plan.search(d)
    raw2 = plan.unfiltered_lh(plan.last_workspace, out[2]).cpu().numpy()
    assert np.array_equal(raw2, raw)
    plan.destroy()


# ------------------------------------------------------------------------------------------- N1: post-filter
@pytest.mark.parametrize("n,T", [(1_000_000, 26), (5000, 10), (77, 50), (1, 5), (300_001, 20)])
def test_sigmag_postfilter_reject_flag_and_survivor_list(kb, oracle, n, T):
    """"reject the trajectory if the recomputed likelihood (sum LH') is less than 10".  Flags against
    the oracle; the compacted survivor list must be exactly the ascending indices of the passing lightcurves."""
    rng = np.random.default_rng(700 + T)
    phi = rng.uniform(0.5, 2.0, (n, T)).astype(np.float32)
    psi = ((rng.standard_normal((n, T)) + rng.uniform(0, 5, (n, 1))) * np.sqrt(phi)).astype(np.float32)
    phi[rng.random((n, T)) < 0.1] = 0.0
    psi, _ = synth.outlier_lightcurves(T, psi, phi, 0.1, 10.0)
    sp = kb.SearchParams(K=1, min_obs=max(1, T // 2), min_lh=10.0)
    g = {k: v.cpu().numpy() for k, v in kb.kbmod_sigmag_postfilter(_cuda(psi), _cuda(phi), sp).items()}
    o = oracle.sigmag_filter(psi, phi, parity.oracle_params(oracle, sp))
    assert np.array_equal(g["kept"].view(np.uint64), o["kept"])
    tl, _ = parity.score_tolerances(dict(o, psi_lc=psi, phi_lc=phi), T)
    solid = (o["n_kept"] == 0) | (np.abs(o["lh"] - 10.0) > 2 * tl + 1e-6)   # L' within float32 rounding of 10: either way
    assert np.array_equal(g["passed"][solid], o["passed"][solid]) and solid.mean() > 0.999
    n_pass = int(g["n_pass"][0])
    assert n_pass == int(g["passed"].sum())
    assert np.array_equal(g["survivors"][:n_pass], np.nonzero(g["passed"])[0].astype(np.int32))
    if n >= 5000:
        assert 0.02 * n < n_pass < 0.98 * n
    # min_lh = -inf keeps every lightcurve that has a result; no compaction asked for: no list
    r = kb.kbmod_sigmag_postfilter(_cuda(psi), _cuda(phi), kb.SearchParams(K=1, min_obs=max(1, T // 2), min_lh=-np.inf), compact=False)
    assert np.array_equal(r["passed"].cpu().numpy().astype(bool), o["n_kept"] > 0) and "survivors" not in r


# ------------------------------------------------------------------------------------------- N2: fused moments
@pytest.mark.parametrize("T,radius", [(26, 10), (5, 3), (50, 15), (10, 0)])
def test_coadd_with_fused_moment_filter(kb, oracle, T, radius):
    """median stamp -> central moments.  The fused kernel's moments and keep flags equal
    kbmod_stamp_moments of its own median stamps bit for bit, its stamps equal kbmod_coadd_stamps', and the moments
    agree with the oracle's moments of the oracle's median stamps."""
    import torch
    H, W = 90, 120
    st = synth.random_stack(800 + T, T, H, W, mask_frac=0.05, t_span=2.0)
    rng = np.random.default_rng(800 + T)
    n = 400
    x0 = rng.integers(0, W, n).astype(np.int32); y0 = rng.integers(0, H, n).astype(np.int32)
    vx = rng.uniform(-10, 10, n).astype(np.float32); vy = rng.uniform(-10, 10, n).astype(np.float32)
    for i in range(0, n, 3):   # a source on every third trajectory, so that some stamps pass
        for t in range(T):
            dt = st.times[t] - st.times[0]
            cx, cy = int(np.floor(x0[i] + vx[i] * dt + 0.5)), int(np.floor(y0[i] + vy[i] * dt + 0.5))
            ax = np.arange(-6, 7)
            blob = 40.0 * np.exp(-0.5 * (ax[None, :] ** 2 + ax[:, None] ** 2) / 1.5 ** 2)
            ya, yb, xa, xb = max(cy - 6, 0), min(cy + 7, H), max(cx - 6, 0), min(cx + 7, W)
            if ya < yb and xa < xb:
                st.img[t, ya:yb, xa:xb] += blob[ya - cy + 6:yb - cy + 6, xa - cx + 6:xb - cx + 6].astype(np.float32)
    thr = oracle.PAPER_MOMENT_THRESHOLDS if radius == 10 else (0.4, 0.4, 0.8, 0.25 * radius * radius + 0.5, 0.25 * radius * radius + 0.5)
    args = (_cuda(st.img), _cuda(st.mask), st.times, _cuda(x0), _cuda(y0), _cuda(vx), _cuda(vy), radius)
    mean, med, mom, keep = kb.kbmod_coadd_stamps_filtered(*args, thresholds=None if radius == 10 else thr)
    mean0, med0 = kb.kbmod_coadd_stamps(*args)
    assert torch.equal(mean, mean0) and torch.equal(med, med0)
    mom1, keep1 = kb.kbmod_stamp_moments(med, None if radius == 10 else thr)
    assert torch.equal(mom.view(torch.int64), mom1.view(torch.int64)) and torch.equal(keep, keep1)
    _, od = oracle.coadd_stamps(st.img, st.mask, st.times, x0, y0, vx, vy, radius)
    assert np.array_equal(med.cpu().numpy(), od.astype(np.float32))
    o_mom, o_keep = oracle.stamp_moments(od.astype(np.float32), thr)
    nan = np.isnan(o_mom).any(1)
    assert np.allclose(mom.cpu().numpy()[~nan], o_mom[~nan], rtol=1e-11, atol=1e-11)
    t = np.asarray(thr)
    dist = np.minimum(np.abs(np.abs(o_mom[:, :3]) - t[:3]).min(1), np.abs(o_mom[:, 3:] - t[3:]).min(1))
    solid = ~nan & (dist > 1e-9)
    assert np.array_equal(keep.cpu().numpy()[solid], o_keep[solid])
    if radius in (3, 10):
        assert 0 < int(o_keep.sum()) < n
    # moments alone (no stamp output)
    _, _, mom2, keep2 = kb.kbmod_coadd_stamps_filtered(*args, thresholds=None if radius == 10 else thr, want_mean=False,
                                                       want_median=False)
    assert torch.equal(mom2.view(torch.int64), mom.view(torch.int64)) and torch.equal(keep2, keep)
