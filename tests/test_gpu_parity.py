"""GPU parity tests proper: the CUDA path (through the C ABI) against the oracle, element by element,
on the same seeded inputs.  Sizes span several tiles and a ragged tail; protocol in tests/parity.py."""
import math

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


def _prep(kb, st, psf=None):
    out = kb.kbmod_prepare_psi_phi(_cuda(st.img), _cuda(st.var), _cuda(st.mask) if st.mask is not None else None,
                                   st.psf if psf is None else psf)
    return out


def _search_and_compare(kb, O, psiphi_d, times, vx, vy, sp, pixels=None):
    T, H, W, _ = psiphi_d.shape
    out = kb.kbmod_search(psiphi_d, times, vx, vy, sp)
    g = [o.cpu().numpy() for o in out]
    psiphi = psiphi_d.cpu().numpy()
    if pixels is None:
        yy, xx = np.mgrid[0:H, 0:W]
        px, py = xx.reshape(-1).astype(np.int32), yy.reshape(-1).astype(np.int32)
    else:
        px, py = pixels
    op = parity.oracle_params(O, sp)
    ora = O.search_pixels(psiphi, times, vx, vy, px, py, op)
    gsel = [a[py, px] for a in g]
    return parity.compare_topk(O, psiphi, times, vx, vy, op, px, py, gsel, ora)


# ------------------------------------------------------------------------------------------- prep
@pytest.mark.parametrize("seed,T,H,W,sigma", [(11, 3, 37, 70, 1.0), (12, 2, 130, 65, 1.8), (13, 1, 9, 5, 1.5)])
def test_prep_random(kb, oracle, seed, T, H, W, sigma):
    st = synth.random_stack(seed, T, H, W, psf_sigma=sigma, mask_frac=0.08)
    st.var[0, 0, 0] = 0.0  # var <= 0 and non-finite pixels are bad pixels (reading R19)
    st.img[0, min(3, H - 1), min(4, W - 1)] = np.nan
    st.var[0, min(5, H - 1), 1] = np.inf
    g = _prep(kb, st).cpu().numpy()
    assert parity.check_prep(oracle, st, g) > 0


def test_prep_per_epoch_asymmetric_psf(kb, oracle):
    st = synth.random_stack(14, 3, 40, 50, mask_frac=0.03)
    rng = np.random.default_rng(5)
    psf = rng.random((3, 5, 5)).astype(np.float32)  # asymmetric: tells correlation from convolution (R2)
    g = _prep(kb, st, psf).cpu().numpy()
    parity.check_prep(oracle, st, g, psf)


def test_prep_no_mask_and_max_psf(kb, oracle):
    st = synth.random_stack(15, 1, 50, 80, mask_frac=0.0)
    st.mask = None
    psf = synth.gaussian_psf(5.0)  # 31 x 31, the largest supported
    assert psf.shape == (31, 31)
    g = _prep(kb, st, psf).cpu().numpy()
    parity.check_prep(oracle, st, g, psf)


def test_prep_config1(kb, oracle):
    st = synth.config1_tiny()
    parity.check_prep(oracle, st, _prep(kb, st).cpu().numpy())


# ------------------------------------------------------------------------------------------- search
def test_search_config1_tiny(kb, oracle):
    """BASELINE configs[0]: every pixel, K=1, sigma-G on; the injected mover is recovered (L177 window)."""
    st = synth.config1_tiny()
    vx, vy = synth.config1_grid()
    d = _prep(kb, st)
    for min_lh in (-np.inf, 10.0):
        sp = kb.SearchParams(K=1, min_obs=3, min_lh=min_lh, algo=kb.ALGO_DIRECT)
        r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp)
        assert r["n_pix"] == 64 * 64
    lh, flux, vel, nobs = [o.cpu().numpy() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    y, x = np.unravel_index(np.argmax(lh[..., 0]), lh.shape[:2])
    v = vel[y, x, 0]
    assert abs(x - 20) <= 5 and abs(y - 30) <= 5 and abs(vx[v] - 20) <= 5 and abs(vy[v] - 5) <= 5
    assert 35 < lh[y, x, 0] < 70


@pytest.mark.parametrize("seed,T,H,W,K,sig,fon,min_lh,min_obs", [
    (21, 7, 45, 70, 4, 1, 0, -np.inf, 1),
    (22, 10, 33, 37, 8, 1, 1, -np.inf, 4),
    (23, 5, 20, 100, 3, 0, 0, -np.inf, 2),
    (24, 12, 40, 40, 2, 1, 0, 1.5, 6),
    (25, 26, 24, 40, 8, 1, 0, -np.inf, 13),
    (26, 1, 10, 10, 2, 1, 0, -np.inf, 1),
    (27, 3, 17, 19, 32, 1, 0, -np.inf, 1),
])
def test_search_random(kb, oracle, seed, T, H, W, K, sig, fon, min_lh, min_obs):
    st = synth.random_stack(seed, T, H, W, mask_frac=0.06, t_span=1.5)
    rng = np.random.default_rng(seed)
    nv = 40
    vx = rng.uniform(-25, 25, nv).astype(np.float32)
    vy = rng.uniform(-25, 25, nv).astype(np.float32)
    vx[0] = vy[0] = 0.0
    vx[1], vy[1] = 1e4, 0.0  # leaves the chip after the first epoch
    d = _prep(kb, st)
    sp = kb.SearchParams(sigmag_enable=sig, filter_on=fon, min_lh=min_lh, min_obs=min_obs, K=K, algo=kb.ALGO_DIRECT)
    r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp)
    assert r["n_entries"] > 0


def test_search_all_zero_psi(kb, oracle):
    """All-zero psi gives L' = 0 and flux' = 0 (a legal score, not the sentinel) -- SURVEY 8c pin 2."""
    import torch
    T, H, W = 4, 12, 16
    d = torch.zeros((T, H, W, 2), device="cuda")
    d[..., 1] = 0.5
    vx, vy = np.array([0, 1, 2], np.float32), np.array([0, 0, 1], np.float32)
    sp = kb.SearchParams(K=2, min_lh=-np.inf, algo=kb.ALGO_DIRECT)
    lh, flux, vel, nobs = [o.cpu().numpy() for o in kb.kbmod_search(d, np.arange(T) * 0.5, vx, vy, sp)]
    assert np.all(lh == 0) and np.all(flux == 0) and np.all(vel[..., 0] == 0) and np.all(vel[..., 1] == 1)


def test_search_empty_velocity_list(kb):
    import torch
    d = torch.ones((2, 8, 8, 2), device="cuda")
    sp = kb.SearchParams(K=3, algo=kb.ALGO_DIRECT)
    lh, flux, vel, nobs = kb.kbmod_search(d, np.array([0.0, 1.0]), np.zeros(0, np.float32), np.zeros(0, np.float32), sp)
    assert torch.all(torch.isneginf(lh)) and torch.all(vel == -1) and torch.all(nobs == 0) and torch.all(flux == 0)


@pytest.mark.parametrize("min_lh", [10.0, -np.inf])
def test_search_config2_medium_every_pixel(kb, oracle, min_lh):
    """BASELINE configs[1] (512x512, T=10, 64 x 32 velocities over the full circle, K=8, 1% mask) as SURVEY 8c
    prescribes: EVERY pixel, both kernels, mode (A) min_lh = 10 and mode (B) min_lh = -inf.  The full 2 pi angle
    grid is the one configuration whose velocity groups scatter in all directions."""
    st = synth.config2_medium()
    vx, vy = synth.config2_grid()
    d = _prep(kb, st)
    psiphi = d.cpu().numpy()
    T, H, W = st.img.shape
    yy, xx = np.mgrid[0:H, 0:W]
    px, py = xx.reshape(-1).astype(np.int32), yy.reshape(-1).astype(np.int32)
    op = oracle.Params(K=8, min_obs=5, min_lh=min_lh)
    ora = oracle.search_pixels(psiphi, st.times, vx, vy, px, py, op)      # 5.4e9 evaluations
    for algo in (kb.ALGO_DIRECT, kb.ALGO_PRUNED, kb.ALGO_AUTO):
        sp = kb.SearchParams(K=8, min_obs=5, min_lh=min_lh, algo=algo)
        g = [o.cpu().numpy().reshape(H * W, -1) for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
        r = parity.compare_topk(oracle, psiphi, st.times, vx, vy, op, px, py, g, ora)
        assert r["n_pix"] == H * W and r["n_exact_pix"] > 0.999 * H * W, r
        used = kb.kbmod_search_stats(kb.kbmod_search.last_workspace)[3]
        assert used == (kb.ALGO_DIRECT if algo == kb.ALGO_DIRECT or (algo == kb.ALGO_AUTO and not np.isfinite(min_lh))
                        else kb.ALGO_PRUNED)
        if not np.isfinite(min_lh):
            assert r["n_entries"] == H * W * 8      # every pixel returns K results


# ------------------------------------------------------------------------------------------- lightcurves
def _random_trajectories(rng, n, H, W, vmax):
    return (rng.integers(0, W, n).astype(np.int32), rng.integers(0, H, n).astype(np.int32),
            rng.uniform(-vmax, vmax, n).astype(np.float32), rng.uniform(-vmax, vmax, n).astype(np.float32))


@pytest.mark.parametrize("T,fon,min_obs", [(5, 0, 1), (10, 1, 3), (26, 0, 13), (50, 0, 1), (64, 0, 20), (3, 0, 1)])
def test_eval_trajectories(kb, oracle, T, fon, min_obs):
    st = synth.random_stack(30 + T, T, 60, 75, mask_frac=0.1, t_span=3.0)
    d = _prep(kb, st)
    psiphi = d.cpu().numpy()
    rng = np.random.default_rng(T)
    x0, y0, vx, vy = _random_trajectories(rng, 5000, 60, 75, 12.0)
    sp = kb.SearchParams(filter_on=fon, min_obs=min_obs, K=1)
    g = {k: v.cpu().numpy() for k, v in
         kb.kbmod_eval_trajectories(d, st.times, _cuda(x0), _cuda(y0), _cuda(vx), _cuda(vy), sp).items()}
    o = oracle.eval_trajectories(psiphi, st.times, x0, y0, vx, vy, parity.oracle_params(oracle, sp))
    assert np.array_equal(g["valid"].view(np.uint64), o["valid"])      # positions + validity: bit-exact
    assert np.array_equal(g["psi_lc"], o["psi_lc"]) and np.array_equal(g["phi_lc"], o["phi_lc"])
    assert np.array_equal(g["kept"].view(np.uint64), o["kept"])        # float32 decisions: bit-exact
    tl, tf = parity.score_tolerances(o, T)
    has = o["n_kept"] > 0
    assert has.sum() > 1000
    assert np.all(np.abs(g["lh"][has] - o["lh"][has]) <= tl[has])
    assert np.all(np.abs(g["flux"][has] - o["flux"][has]) <= tf[has])
    assert np.all(np.isneginf(g["lh"][~has])) and np.all(g["flux"][~has] == 0)


@pytest.mark.parametrize("T", [4, 9, 26, 50])
def test_sigmag_filter_with_outliers(kb, oracle, T):
    """BASELINE configs[4]: rerun sigma-G on lightcurves with 20% of epochs replaced by 10-sigma outliers."""
    rng = np.random.default_rng(40 + T)
    n = 20000
    phi = rng.uniform(0.5, 2.0, (n, T)).astype(np.float32)
    psi = (rng.standard_normal((n, T)) * np.sqrt(phi)).astype(np.float32)
    phi[rng.random((n, T)) < 0.1] = 0.0  # invalid epochs
    psi, hit = synth.outlier_lightcurves(T, psi, phi, 0.2, 10.0)
    sp = kb.SearchParams(K=1, min_obs=2)
    g = {k: v.cpu().numpy() for k, v in kb.kbmod_sigmag_filter(_cuda(psi), _cuda(phi), sp).items()}
    o = oracle.sigmag_filter(psi, phi, parity.oracle_params(oracle, sp))
    assert np.array_equal(g["kept"].view(np.uint64), o["kept"])
    has = o["n_kept"] > 0
    o2 = dict(o, psi_lc=psi, phi_lc=phi)
    tl, tf = parity.score_tolerances(o2, T)
    assert np.all(np.abs(g["lh"][has] - o["lh"][has]) <= tl[has])
    assert np.all(np.abs(g["flux"][has] - o["flux"][has]) <= tf[has])


# ------------------------------------------------------------------------------------------- coadd
@pytest.mark.parametrize("T,radius,use_sel,use_mask", [(5, 10, False, True), (26, 10, True, True), (10, 3, True, False),
                                                      (50, 15, False, True), (1, 0, False, True), (64, 2, True, True)])
def test_coadd_stamps(kb, oracle, T, radius, use_sel, use_mask):
    import torch
    H, W = 70, 90
    st = synth.random_stack(50 + T, T, H, W, mask_frac=0.1, t_span=2.0)
    st.img[0, 5, 5] = np.inf
    rng = np.random.default_rng(T)
    n = 300
    x0, y0, vx, vy = _random_trajectories(rng, n, H, W, 15.0)
    x0[:4], y0[:4] = [0, W - 1, 0, W - 1], [0, 0, H - 1, H - 1]  # stamps hanging over the corners
    sel = rng.integers(0, 2 ** min(T, 62), n, dtype=np.int64) if use_sel else None
    mask = st.mask if use_mask else None
    gm, gd = kb.kbmod_coadd_stamps(_cuda(st.img), _cuda(mask) if use_mask else None, st.times, _cuda(x0), _cuda(y0),
                                   _cuda(vx), _cuda(vy), radius, _cuda(sel) if use_sel else None)
    om, od = oracle.coadd_stamps(st.img, mask, st.times, x0, y0, vx, vy, radius,
                                 sel.view(np.uint64) if use_sel else None)
    gm, gd = gm.cpu().numpy(), gd.cpu().numpy()
    assert np.array_equal(gd, od.astype(np.float32))  # a median is one sample or the mean of two: exact in float32
    assert np.all(np.abs(gm - om) <= 1e-5 * np.abs(om) + 1e-5)


# ------------------------------------------------------------------------------------------- errors
def test_error_codes(kb):
    import torch
    d = torch.zeros((2, 8, 8, 2), device="cuda")
    t = np.array([0.0, 1.0])
    v = np.zeros(1, np.float32)
    with pytest.raises(kb.KbmodError) as e:
        kb.kbmod_search(d, t, v, v, kb.SearchParams(K=33))
    assert e.value.code == -2
    with pytest.raises(kb.KbmodError) as e:
        kb.kbmod_search(d, t, v, v, kb.SearchParams(K=0))
    assert e.value.code == -1
    with pytest.raises(kb.KbmodError) as e:
        kb.kbmod_search(d, t, v, v, kb.SearchParams(K=1), workspace=torch.empty(256, dtype=torch.uint8, device="cuda")[:0])
    assert e.value.code in (-1, -3)
    with pytest.raises(kb.KbmodError) as e:
        kb.kbmod_prepare_psi_phi(d[..., 0].contiguous(), d[..., 0].contiguous(), None, np.ones((4, 4), np.float32))
    assert e.value.code == -1
    with pytest.raises(TypeError):
        kb.kbmod_search(d.cpu(), t, v, v, kb.SearchParams(K=1))  # no CPU fallback
    for bad_v, bad_t in ((np.array([np.inf], np.float32), t), (np.array([np.nan], np.float32), t), (v, np.array([0.0, np.nan]))):
        with pytest.raises(kb.KbmodError) as e:
            kb.kbmod_search(d, bad_t, bad_v, v, kb.SearchParams(K=1))
        assert e.value.code == -1


# ------------------------------------------------------------------------------------------- pruned search
@pytest.mark.parametrize("seed,T,H,W,K,sig,fon,min_lh,min_obs", [
    (61, 7, 45, 70, 4, 1, 0, 2.0, 1),
    (62, 10, 33, 137, 8, 1, 1, 1.0, 4),
    (63, 5, 20, 100, 3, 0, 0, 2.5, 2),
    (64, 26, 50, 90, 8, 1, 0, 3.0, 13),
    (65, 50, 40, 70, 16, 1, 0, 3.5, 25),
    (66, 64, 17, 65, 2, 1, 0, 4.0, 1),
    (67, 3, 16, 64, 32, 1, 0, -1.0, 1),
])
def test_search_pruned_random(kb, oracle, seed, T, H, W, K, sig, fon, min_lh, min_obs):
    """The pruned kernel (TMA-staged bound + exact re-evaluation) against the oracle, every pixel; low
    thresholds so that a large share of the trajectories goes through both phases."""
    st = synth.random_stack(seed, T, H, W, mask_frac=0.06, t_span=1.5)
    rng = np.random.default_rng(seed)
    nv = 70  # not a multiple of the group size
    vx = rng.uniform(-25, 25, nv).astype(np.float32)
    vy = rng.uniform(-25, 25, nv).astype(np.float32)
    vx[0] = vy[0] = 0.0
    vx[1], vy[1] = 1e4, 0.0    # leaves the chip after the first epoch: its group cannot be staged
    vx[2], vy[2] = 3e9, -3e9   # displacement beyond int32
    d = _prep(kb, st)
    sp = kb.SearchParams(sigmag_enable=sig, filter_on=fon, min_lh=min_lh, min_obs=min_obs, K=K, algo=kb.ALGO_PRUNED)
    r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp)
    assert r["n_entries"] > 0
    ws = kb.kbmod_search.last_workspace
    ev, nominal, launches, algo, _ = kb.kbmod_search_stats(ws)
    assert algo == kb.ALGO_PRUNED and nominal == H * W * nv and 0 < ev <= nominal


def test_search_pruned_config1(kb, oracle):
    st = synth.config1_tiny()
    vx, vy = synth.config1_grid()
    d = _prep(kb, st)
    sp = kb.SearchParams(K=1, min_obs=3, min_lh=10.0, algo=kb.ALGO_PRUNED)
    r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp)
    assert r["n_entries"] > 50


def test_search_pruned_equals_direct_decam_shaped(kb):
    """Property that holds at any size: both kernels return identical arrays (same evaluation function,
    order-independent top-K).  DECam-shaped stack scaled to 1024x600 with artefacts, masks and movers."""
    import torch
    st = synth.decam_stack(5, (7, 6, 7, 6), H=1024, W=600, n_movers=40, n_stars=60)
    vx, vy = synth.config3_grid()  # the full 128 x 64 grid: dense enough for every velocity group to be staged
    d = _prep(kb, st)
    outs = {}
    for name, algo in (("direct", kb.ALGO_DIRECT), ("pruned", kb.ALGO_PRUNED)):
        sp = kb.SearchParams(K=8, min_obs=13, min_lh=10.0, algo=algo)
        outs[name] = [o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    ev, nominal, _, algo, _ = kb.kbmod_search_stats(kb.kbmod_search.last_workspace)
    assert algo == kb.ALGO_PRUNED and ev < 0.05 * nominal, (ev, nominal)
    for a, b in zip(outs["direct"], outs["pruned"]):
        assert torch.equal(a, b)
    assert int((outs["pruned"][2] >= 0).sum()) > 100  # the movers are found


@pytest.fixture(scope="module")
def c3(kb):
    """BASELINE configs[2] (2048x4096x26) and its psi/phi stack on the GPU, shared by the full-size tests."""
    st = synth.config3_decam()
    d = _prep(kb, st)
    return st, d, d.cpu().numpy()


def protocol_pixels(st, rng, n_windows=64, n_mask_adjacent=1000, n_border=2000, mover_window=2, n_random=0):
    """The pixel sample SURVEY 8c prescribes for the full-size configurations: all pixels of `n_windows` random 32x32
    windows, windows on EVERY injected mover start, `n_mask_adjacent` pixels next to a statically masked pixel (bad
    columns, disc edges), the four borders."""
    T, H, W = st.img.shape
    px, py = [], []
    wy, wx = np.mgrid[0:32, 0:32]
    for _ in range(n_windows):
        x0, y0 = int(rng.integers(0, W - 32)), int(rng.integers(0, H - 32))
        px.append(x0 + wx.reshape(-1)); py.append(y0 + wy.reshape(-1))
    k = mover_window
    my, mx = np.mgrid[-k:k + 1, -k:k + 1]
    for m in st.movers:
        px.append(np.clip(int(m["x0"]) + mx.reshape(-1), 0, W - 1))
        py.append(np.clip(int(m["y0"]) + my.reshape(-1), 0, H - 1))
    static = (st.mask != 0).all(axis=0)                      # masked in every epoch: discs and bad columns
    grown = static.copy()
    grown[1:, :] |= static[:-1, :]; grown[:-1, :] |= static[1:, :]
    grown[:, 1:] |= static[:, :-1]; grown[:, :-1] |= static[:, 1:]
    ay, ax = np.nonzero(grown & ~static)
    pick = rng.choice(len(ay), min(n_mask_adjacent, len(ay)), replace=False)
    px.append(ax[pick]); py.append(ay[pick])
    bx, by = rng.integers(0, W, n_border), rng.integers(0, H, n_border)
    px += [bx[:n_border // 2], np.zeros(n_border // 2, int), np.full(n_border // 2, W - 1), bx[n_border // 2:]]
    py += [np.zeros(n_border // 2, int), by[:n_border // 2], by[n_border // 2:], np.full(n_border - n_border // 2, H - 1)]
    px.append(np.array([0, W - 1, 0, W - 1])); py.append(np.array([0, 0, H - 1, H - 1]))
    if n_random:
        px.append(rng.integers(0, W, n_random)); py.append(rng.integers(0, H, n_random))
    return np.concatenate(px).astype(np.int32), np.concatenate(py).astype(np.int32)


def test_search_config3_full_size_protocol_mode_a(kb, oracle, c3):
    """BASELINE configs[2] at full size in the launch configuration bench.py times (AUTO -> pruned, min_lh = 10,
    K = 8), on the sample SURVEY 8c prescribes: 64 random 32x32 windows, 5x5 windows on all 200 mover starts, 1000
    mask-adjacent pixels, the four borders, and pixels where the search returned something: > 10^5 start pixels x
    all 8192 velocities in the oracle."""
    st, d, psiphi = c3
    vx, vy = synth.config3_grid()
    T, H, W = st.img.shape
    rng = np.random.default_rng(3)
    px, py = protocol_pixels(st, rng, n_random=20000)
    sp = kb.SearchParams(K=8, min_obs=13, min_lh=10.0, algo=kb.ALGO_AUTO)
    out = kb.kbmod_search(d, st.times, vx, vy, sp)
    ev, nominal, _, algo, _ = kb.kbmod_search_stats(kb.kbmod_search.last_workspace)
    assert algo == kb.ALGO_PRUNED and nominal == H * W * len(vx) and ev < 0.05 * nominal
    g = [o.cpu().numpy() for o in out]
    # ... and 6000 pixels where the search returned something (the pixel LIST may come from anywhere; every expected
    # value is the oracle's)
    has_y, has_x = np.nonzero(g[2][..., 0] >= 0)
    pick = rng.choice(len(has_y), min(6000, len(has_y)), replace=False)
    px, py = np.concatenate([px, has_x[pick].astype(np.int32)]), np.concatenate([py, has_y[pick].astype(np.int32)])
    assert len(px) >= 100_000
    op = parity.oracle_params(oracle, sp)
    ora = oracle.search_pixels(psiphi, st.times, vx, vy, px, py, op)
    r = parity.compare_topk(oracle, psiphi, st.times, vx, vy, op, px, py, [a[py, px] for a in g], ora)
    assert r["n_entries"] > 20000 and r["n_exact_pix"] > 0.999 * len(px), r
    # recovery (PAPER.md L177 window: 5 px, 5 px/day): the best result near a bright injected mover is the mover
    found = 0
    bright = [m for m in st.movers if m["flux"] > 1500]
    for m in bright:
        x, y = int(m["x0"]), int(m["y0"])
        v = g[2][max(y - 2, 0):y + 3, max(x - 2, 0):x + 3, 0]
        l = g[0][max(y - 2, 0):y + 3, max(x - 2, 0):x + 3, 0]
        if (v >= 0).any():
            vb = v.reshape(-1)[np.argmax(np.where(v >= 0, l, -np.inf))]
            found += int(abs(vx[vb] - m["vx"]) <= 5 and abs(vy[vb] - m["vy"]) <= 5)
    # (the injected velocities are random, not grid points: a mover between grid velocities drifts off its nearest
    # trajectory by a few pixels over three days; the paper itself recovers 22 of 26 known objects, L177)
    assert found >= 0.6 * len(bright), (found, len(bright))


def test_search_config3_full_size_mode_b_direct(kb, oracle, c3):
    """SURVEY 8d mode (B): min_lh = -inf, every pixel returns K results, every trajectory gets the full filter --
    the direct kernel at full size (2048x4096x26 x 8192 velocities) on > 10^4 sampled pixels incl. borders, mover
    starts and mask-adjacent pixels."""
    st, d, psiphi = c3
    vx, vy = synth.config3_grid()
    T, H, W = st.img.shape
    px, py = protocol_pixels(st, np.random.default_rng(33), n_windows=4, n_mask_adjacent=500, n_border=1000, mover_window=1,
                             n_random=3000)
    assert len(px) >= 10_000
    sp = kb.SearchParams(K=8, min_obs=13, min_lh=-np.inf, algo=kb.ALGO_AUTO)
    r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp, pixels=(px, py))
    ev, nominal, _, algo, _ = kb.kbmod_search_stats(kb.kbmod_search.last_workspace)
    assert algo == kb.ALGO_DIRECT and ev == nominal == H * W * len(vx)
    assert r["n_exact_pix"] > 0.99 * len(px), r


def test_search_paper_grid_full_size_sampled(kb, oracle, c3):
    """The paper's own operating point (512 speed x 256 angle steps = 131072 velocities; L133: of order
    10^12 trajectories per 2Kx4K stack) on the configs[2] stack: oracle on > 2000 sampled pixels x all velocities."""
    st, d, psiphi = c3
    vx, vy = synth.paper_grid()
    assert len(vx) == 131072
    T, H, W = st.img.shape
    px, py = protocol_pixels(st, np.random.default_rng(34), n_windows=1, n_mask_adjacent=200, n_border=200, mover_window=0,
                             n_random=500)
    assert len(px) >= 2000
    sp = kb.SearchParams(K=8, min_obs=13, min_lh=10.0, algo=kb.ALGO_AUTO)
    r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp, pixels=(px, py))
    ev, nominal, _, algo, _ = kb.kbmod_search_stats(kb.kbmod_search.last_workspace)
    assert algo == kb.ALGO_PRUNED and nominal == H * W * 131072
    assert r["n_exact_pix"] > 0.99 * len(px) and r["n_entries"] > 100, r


def test_pipeline_host_batch_against_the_oracle_full_size(kb, oracle, c3):
    """The call bench.py's e2e figure times, at full size: the HOST result arrays of kbmod_pipeline_host_batch (two
    stacks: both arena halves) against the oracle on sampled pixels."""
    import torch
    st, d, psiphi = c3
    vx, vy = synth.config3_grid()
    T, H, W = st.img.shape
    sp = kb.SearchParams(K=8, min_obs=13, min_lh=10.0)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_in = (pin(st.img), pin(st.var), pin(st.mask))
    outs = [tuple(torch.empty((H, W, 8), dtype=dt).pin_memory() for dt in (torch.float32, torch.float32, torch.int32, torch.int32))
            for _ in range(2)]
    arena = torch.empty(2 * kb.kbmod_pipeline_host_arena_bytes_for(T, H, W, st.times, vx, vy, sp), dtype=torch.uint8, device="cuda")
    kb.kbmod_pipeline_host_batch([h_in, h_in], st.psf, st.times, vx, vy, sp, outs, arena)
    del arena
    for a, b in zip(outs[0], outs[1]):
        assert torch.equal(a, b)
    px, py = protocol_pixels(st, np.random.default_rng(35), n_windows=2, n_mask_adjacent=300, n_border=400, mover_window=2,
                             n_random=1000)
    g = [o.numpy()[py, px] for o in outs[1]]
    op = parity.oracle_params(oracle, sp)
    # (the pipeline's own psi/phi stack is the same kernel's output as `d`: the prep parity tests cover it)
    ora = oracle.search_pixels(psiphi, st.times, vx, vy, px, py, op)
    r = parity.compare_topk(oracle, psiphi, st.times, vx, vy, op, px, py, g, ora)
    assert r["n_entries"] > 1000 and r["n_exact_pix"] > 0.99 * len(px), r


# ------------------------------------------------------------------------------------------- round-1 additions
def test_search_pruned_queue_overflow_path(kb, oracle, monkeypatch):
    """A survivor queue of 64 entries (test hook KBMOD_B200_QUEUE_CAP) overflows at once: almost every
    (tile, group, warp) item goes through the overflow bitmap and exact_overflow_kernel.  Same results."""
    import torch
    st = synth.random_stack(81, 9, 70, 150, mask_frac=0.05, t_span=1.5)
    rng = np.random.default_rng(81)
    vx = rng.uniform(-20, 20, 40).astype(np.float32)
    vy = rng.uniform(-20, 20, 40).astype(np.float32)
    d = _prep(kb, st)
    sp = kb.SearchParams(K=4, min_obs=3, min_lh=2.0, algo=kb.ALGO_PRUNED)
    ref = [o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    monkeypatch.setenv("KBMOD_B200_QUEUE_CAP", "64")
    small = [o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    monkeypatch.delenv("KBMOD_B200_QUEUE_CAP")
    for a, b in zip(ref, small):
        assert torch.equal(a, b)
    r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp)
    assert r["n_entries"] > 100


def test_search_phase_timing_api(kb):
    st = synth.config1_tiny()
    vx, vy = synth.config1_grid()
    d = _prep(kb, st)
    kb.kbmod_search_phase_timing(True)
    try:
        for algo, keys in ((kb.ALGO_PRUNED, ("planes", "gather", "exact", "finalize")), (kb.ALGO_DIRECT, ("gather",))):
            kb.kbmod_search(d, st.times, vx, vy, kb.SearchParams(K=1, min_obs=3, min_lh=10.0, algo=algo))
            ms = kb.kbmod_search_phase_ms()
            assert all(ms[k] > 0.0 for k in keys), ms
            assert all(v >= 0.0 for v in ms.values())
    finally:
        kb.kbmod_search_phase_timing(False)


def test_search_pruned_equals_direct_heavy_shaped(kb):
    """BASELINE configs[3] shape (T = 50 over 6 nights, K = 16, min_obs = 25, sub-threshold movers) scaled to
    512x320 with a 64 x 32 slice of the velocity grid: both kernels must return identical arrays."""
    import torch
    st = synth.decam_stack(7, (9, 8, 8, 9, 8, 8), H=512, W=320, n_movers=60, flux_range=(10.0, 100.0), flux_log=False,
                           n_stars=30, name="heavy_small")
    vx, vy = synth.config3_grid(64, 32)
    d = _prep(kb, st)
    outs = {}
    for name, algo in (("direct", kb.ALGO_DIRECT), ("pruned", kb.ALGO_PRUNED)):
        sp = kb.SearchParams(K=16, min_obs=25, min_lh=6.0, algo=algo)
        outs[name] = [o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    for a, b in zip(outs["direct"], outs["pruned"]):
        assert torch.equal(a, b)
    assert int((outs["pruned"][2] >= 0).sum()) > 10  # (50, 50) percentiles keep only values equal to the median


def test_config5_full_size_coadd_and_refilter(kb, oracle):
    """BASELINE configs[4] at full size: 10^5 candidate trajectories on the 2048x4096x26 stack, 21x21 mean and
    median stamps (oracle on a sample of 1500 trajectories), lightcurves with 20 % of the epochs replaced by
    10-sigma outliers, sigma-G rerun (oracle on all 10^5): kept sets bit-exact, >= 99 % of the outliers dropped
    among lightcurves that keep enough clean epochs."""
    st = synth.config3_decam()
    T, H, W = st.img.shape
    n = 100_000
    x0, y0, vx, vy = synth.config5_trajectories(4, H, W, n)
    img, mask = _cuda(st.img), _cuda(st.mask)
    gm, gd = kb.kbmod_coadd_stamps(img, mask, st.times, _cuda(x0), _cuda(y0), _cuda(vx), _cuda(vy), 10)
    pick = np.random.default_rng(5).choice(n, 1500, replace=False)
    om, od = oracle.coadd_stamps(st.img, st.mask, st.times, x0[pick], y0[pick], vx[pick], vy[pick], 10)
    gm, gd = gm[_cuda(pick)].cpu().numpy(), gd[_cuda(pick)].cpu().numpy()
    assert np.array_equal(gd, od.astype(np.float32))
    assert np.all(np.abs(gm - om) <= 1e-5 * np.abs(om) + 1e-4)
    # lightcurves of the same candidates
    d = _prep(kb, st)
    sp = kb.SearchParams(K=1, min_obs=13)
    ev = {k: v.cpu().numpy() for k, v in
          kb.kbmod_eval_trajectories(d, st.times, _cuda(x0), _cuda(y0), _cuda(vx), _cuda(vy), sp).items()}
    psi, hit = synth.outlier_lightcurves(6, ev["psi_lc"], ev["phi_lc"], 0.2, 10.0)
    g = {k: v.cpu().numpy() for k, v in kb.kbmod_sigmag_filter(_cuda(psi), _cuda(ev["phi_lc"]), sp).items()}
    o = oracle.sigmag_filter(psi, ev["phi_lc"], parity.oracle_params(oracle, sp))
    assert np.array_equal(g["kept"].view(np.uint64), o["kept"])
    has = o["n_kept"] > 0
    tl, tf = parity.score_tolerances(dict(o, psi_lc=psi, phi_lc=ev["phi_lc"]), T)
    assert np.all(np.abs(g["lh"][has] - o["lh"][has]) <= tl[has])
    assert np.all(np.abs(g["flux"][has] - o["flux"][has]) <= tf[has])
    valid = ev["phi_lc"] > 0
    kept = ((o["kept"][:, None] >> np.arange(T, dtype=np.uint64)[None, :]) & np.uint64(1)).astype(bool)
    few = has & ((hit & valid).sum(1) <= 5) & (valid.sum(1) >= 20)  # the 25/75 percentiles stay on clean epochs
    dropped = (hit & valid & ~kept)[few].sum() / max(1, (hit & valid)[few].sum())
    assert few.sum() > 10_000 and dropped >= 0.99, (int(few.sum()), float(dropped))


def test_search_config4_full_size_sampled(kb, oracle):
    """BASELINE configs[3] at full size (2048x4096x50, 256 x 128 velocities, K = 16, min_obs = 25) through the
    AUTO -> pruned path at the paper's threshold: oracle on > 2x10^4 pixels (random windows, the borders,
    mask-adjacent pixels and 3x3 windows on all 1000 injected mover starts; their fluxes are sub-threshold by
    construction: what is checked is parity)."""
    st = synth.config4_heavy()
    vx, vy = synth.config4_grid()
    d = _prep(kb, st)
    T, H, W = st.img.shape
    # SURVEY 8c sample: 32x32 windows, 3x3 windows on all 1000 mover starts, mask-adjacent pixels, borders: > 2x10^4
    px, py = protocol_pixels(st, np.random.default_rng(4), n_windows=8, n_mask_adjacent=500, n_border=1000, mover_window=1,
                             n_random=1500)
    assert len(px) >= 20_000
    sp = kb.SearchParams(K=16, min_obs=25, min_lh=10.0, algo=kb.ALGO_AUTO)
    r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp, pixels=(px, py))
    ev, nominal, _, algo, _ = kb.kbmod_search_stats(kb.kbmod_search.last_workspace)
    assert algo == kb.ALGO_PRUNED and nominal == H * W * len(vx) and ev < 0.2 * nominal
    assert r["n_pix"] == len(px)


@pytest.mark.parametrize("T,H,W,nv,K", [(1, 9, 7, 1, 1), (2, 33, 65, 3, 2), (1, 40, 130, 17, 4), (4, 5, 300, 33, 3)])
def test_search_pruned_degenerate_shapes(kb, oracle, T, H, W, nv, K):
    """One or two epochs (the producer's table ring wraps inside a single region burst), a single velocity, images
    smaller than one 64x32 tile: the pruned path against the oracle, every pixel."""
    st = synth.random_stack(90 + T + H, T, H, W, mask_frac=0.05, t_span=1.0)
    rng = np.random.default_rng(90 + T)
    vx = rng.uniform(-30, 30, nv).astype(np.float32)
    vy = rng.uniform(-30, 30, nv).astype(np.float32)
    d = _prep(kb, st)
    sp = kb.SearchParams(min_lh=0.5, min_obs=1, K=K, algo=kb.ALGO_PRUNED)
    r = _search_and_compare(kb, oracle, d, st.times, vx, vy, sp)
    assert r["n_pix"] == H * W
    _, nominal, _, algo, _ = kb.kbmod_search_stats(kb.kbmod_search.last_workspace)
    assert algo == kb.ALGO_PRUNED and nominal == H * W * nv


@pytest.mark.parametrize("T", [1, 2, 3, 5, 7, 12, 26, 50, 64])
def test_search_pruned_equals_direct_with_clamped_terms(kb, T):
    """Very bright pixels (up to 10^8 sigma) make the fixed-point terms of the bound planes clamp; very faint and
    very noisy epochs spread phi over six decades.  The pruned path must still equal the direct kernel exactly."""
    import torch
    H, W = 70, 140
    st = synth.random_stack(200 + T, T, H, W, mask_frac=0.03, t_span=2.0)
    rng = np.random.default_rng(200 + T)
    hot = rng.random((T, H, W)) < 0.01
    st.img[hot] *= (10.0 ** rng.uniform(1, 8, int(hot.sum()))).astype(np.float32)
    st.var *= (10.0 ** rng.uniform(-3, 3, (T, 1, 1))).astype(np.float32)
    vx = rng.uniform(-15, 15, 48).astype(np.float32)
    vy = rng.uniform(-15, 15, 48).astype(np.float32)
    d = _prep(kb, st)
    outs = {}
    for name, algo in (("direct", kb.ALGO_DIRECT), ("pruned", kb.ALGO_PRUNED)):
        sp = kb.SearchParams(K=4, min_obs=1, min_lh=5.0, algo=algo)
        outs[name] = [o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    for a, b in zip(outs["direct"], outs["pruned"]):
        assert torch.equal(a, b)
    assert int((outs["pruned"][2] >= 0).sum()) > 100


@pytest.mark.parametrize("n_sigma,pct,fon,sig", [(0.5, (25.0, 75.0), 0, 1), (1.4, (10.0, 90.0), 0, 1), (3.0, (40.0, 60.0), 1, 1),
                                               (2.0, (25.0, 75.0), 0, 0), (1.36, (50.0, 50.0), 0, 1)])
def test_search_pruned_equals_direct_filter_parameters(kb, n_sigma, pct, fon, sig):
    """The number of epochs the bound may count on, m(n), depends on the filter parameters (n_sigma * C below 1:
    only the median is certain to be kept; filter off: all n).  Pruned must equal direct for each."""
    import torch
    st = synth.random_stack(300, 12, 60, 100, mask_frac=0.1, t_span=2.0)
    rng = np.random.default_rng(300)
    st.img[rng.random(st.img.shape) < 0.02] *= 30.0
    vx = rng.uniform(-12, 12, 40).astype(np.float32)
    vy = rng.uniform(-12, 12, 40).astype(np.float32)
    d = _prep(kb, st)
    outs = {}
    for name, algo in (("direct", kb.ALGO_DIRECT), ("pruned", kb.ALGO_PRUNED)):
        sp = kb.SearchParams(sigmag_enable=sig, pct_lo=pct[0], pct_hi=pct[1], n_sigma=n_sigma, filter_on=fon, K=3, min_obs=4,
                             min_lh=3.0, algo=algo)
        outs[name] = [o.clone() for o in kb.kbmod_search(d, st.times, vx, vy, sp)]
    for a, b in zip(outs["direct"], outs["pruned"]):
        assert torch.equal(a, b)
    assert int((outs["pruned"][2] >= 0).sum()) > 10  # (50, 50) percentiles keep only values equal to the median


# ------------------------------------------------------------------------------------------- N2: stamp moments
def _moments_agree(g_mom, g_keep, o_mom, o_keep, thr):
    g_mom, g_keep = g_mom.cpu().numpy(), g_keep.cpu().numpy()
    nan = np.isnan(o_mom).any(1)
    assert np.array_equal(np.isnan(g_mom).any(1), nan)
    assert np.allclose(g_mom[~nan], o_mom[~nan], rtol=1e-11, atol=1e-11)  # double on both sides, other summation order
    # the flag is a threshold on a double: compare it except where a moment sits within 1e-9 of its threshold
    t = np.asarray(thr)
    dist = np.minimum(np.abs(np.abs(o_mom[:, :3]) - t[:3]).min(1), np.abs(o_mom[:, 3:] - t[3:]).min(1))
    solid = ~nan & (dist > 1e-9)
    assert np.array_equal(g_keep[solid], o_keep[solid]) and np.all(g_keep[nan] == 0)
    return int(solid.sum())


@pytest.mark.parametrize("radius", [0, 1, 3, 10, 15])
def test_stamp_moments_random(kb, oracle, radius):
    rng = np.random.default_rng(400 + radius)
    S = 2 * radius + 1
    n = 3000
    ax = np.arange(-radius, radius + 1)
    st = rng.standard_normal((n, S, S)).astype(np.float32)
    amp = rng.uniform(0, 60, n)[:, None, None]
    cx, cy = rng.uniform(-1.5, 1.5, n)[:, None, None], rng.uniform(-1.5, 1.5, n)[:, None, None]
    st += (amp * np.exp(-0.5 * ((ax[None, None, :] - cx) ** 2 + (ax[None, :, None] - cy) ** 2) / 1.6**2)).astype(np.float32)
    st[5] = 4.25                 # constant stamp
    st[6, 0, 0] = np.nan         # non-finite pixel
    st[7, S - 1, S - 1] = np.inf
    thr = (0.5, 0.5, 1.5, 36.5, 36.5) if radius == 10 else (0.3, 0.3, 0.5, 0.3 * radius * radius + 0.5, 0.3 * radius * radius + 0.5)
    g_mom, g_keep = kb.kbmod_stamp_moments(_cuda(st), None if radius == 10 else thr)
    o_mom, o_keep = oracle.stamp_moments(st, thr)
    assert _moments_agree(g_mom, g_keep, o_mom, o_keep, thr) > n - 20
    if radius >= 3:
        assert 0 < int(o_keep.sum()) < n


def test_stamp_moments_on_coadded_stamps(kb, oracle):
    """The step as the paper chains it (L141): median stamps of candidate trajectories, then the moment filter.
    Candidates on injected movers (true velocity) must pass, candidates on empty sky mostly fail."""
    st = synth.decam_stack(9, (7, 6, 7, 6), H=768, W=512, n_movers=60, n_stars=40)
    T, H, W = st.img.shape
    mv = [m for m in st.movers if m["flux"] > 1500]
    n_sky = 2000
    rng = np.random.default_rng(9)
    x0 = np.concatenate([[int(m["x0"]) for m in mv], rng.integers(0, W, n_sky)]).astype(np.int32)
    y0 = np.concatenate([[int(m["y0"]) for m in mv], rng.integers(0, H, n_sky)]).astype(np.int32)
    vx = np.concatenate([[m["vx"] for m in mv], rng.uniform(-300, 300, n_sky)]).astype(np.float32)
    vy = np.concatenate([[m["vy"] for m in mv], rng.uniform(-300, 300, n_sky)]).astype(np.float32)
    _, med = kb.kbmod_coadd_stamps(_cuda(st.img), _cuda(st.mask), st.times, _cuda(x0), _cuda(y0), _cuda(vx), _cuda(vy), 10)
    g_mom, g_keep = kb.kbmod_stamp_moments(med)
    o_mom, o_keep = oracle.stamp_moments(med.cpu().numpy())
    _moments_agree(g_mom, g_keep, o_mom, o_keep, oracle.PAPER_MOMENT_THRESHOLDS)
    k = g_keep.cpu().numpy().astype(bool)
    assert len(mv) >= 10 and k[:len(mv)].mean() > 0.8, (len(mv), k[:len(mv)].mean())
    assert k[len(mv):].mean() < 0.5


def test_sigmag_refilter_one_million_candidates(kb, oracle):
    """N1 (the CPU post-filter rejects ~10^6 trajectories in ~60 s on 30 cores): sigma-G on 10^6
    candidate lightcurves of 26 epochs, both lightcurve choices (R9), every kept set against the oracle."""
    rng = np.random.default_rng(77)
    n, T = 1_000_000, 26
    phi = rng.uniform(5e-5, 1.2e-4, (n, T)).astype(np.float32)
    psi = (rng.standard_normal((n, T)).astype(np.float32) + np.float32(1.5)) * np.sqrt(phi)
    phi[rng.random((n, T)) < 0.08] = 0.0
    psi, _ = synth.outlier_lightcurves(8, psi, phi, 0.1, 8.0)
    d_psi, d_phi = _cuda(psi), _cuda(phi)
    for fon in (0, 1):
        sp = kb.SearchParams(K=1, min_obs=13, filter_on=fon)
        g = {k: v.cpu().numpy() for k, v in kb.kbmod_sigmag_filter(d_psi, d_phi, sp).items()}
        o = oracle.sigmag_filter(psi, phi, parity.oracle_params(oracle, sp))
        assert np.array_equal(g["kept"].view(np.uint64), o["kept"])
        has = o["n_kept"] > 0
        tl, tf = parity.score_tolerances(dict(o, psi_lc=psi, phi_lc=phi), T)
        assert has.sum() > 900_000
        assert np.all(np.abs(g["lh"][has] - o["lh"][has]) <= tl[has])
        assert np.all(np.abs(g["flux"][has] - o["flux"][has]) <= tf[has])
        assert np.all(np.isneginf(g["lh"][~has]))


def test_measured_smem_peak_is_plausible(kb):
    """The roofline denominator bench.py measures live: within 25 % of SMs x 128 B/clk x max SM clock."""
    import torch
    props = torch.cuda.get_device_properties(0)
    theo = props.multi_processor_count * 128 * 1.965  # GB/s at 1965 MHz
    for width in (4, 8, 16):
        gbs = kb.kbmod_measure_smem_gbs(width)
        assert 0.6 * theo < gbs < 1.1 * theo, (width, gbs, theo)


def test_pipeline_host_batch_equals_single_calls(kb):
    """Five stacks of one shape through kbmod_pipeline_host_batch (copies overlapped with the searches, two arena
    halves reused) must give exactly what five kbmod_pipeline_host calls give."""
    import torch
    T, H, W, K = 8, 96, 130, 4
    rng = np.random.default_rng(500)
    vx = rng.uniform(-20, 20, 50).astype(np.float32)
    vy = rng.uniform(-20, 20, 50).astype(np.float32)
    sts = [synth.random_stack(500 + i, T, H, W, mask_frac=0.05, t_span=1.5) for i in range(5)]
    for s_ in sts:
        s_.img[rng.random(s_.img.shape) < 0.02] *= 20.0
        s_.times = sts[0].times
    sp = kb.SearchParams(K=K, min_obs=3, min_lh=4.0)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    stacks = [(pin(s_.img), pin(s_.var), pin(s_.mask)) for s_ in sts]
    mk_out = lambda: tuple(torch.empty((H, W, K), dtype=dt).pin_memory() for dt in (torch.float32, torch.float32, torch.int32, torch.int32))
    per = kb.kbmod_pipeline_host_arena_bytes(T, H, W, len(vx), sp)
    arena = torch.empty(2 * per, dtype=torch.uint8, device="cuda")
    singles = []
    for stk in stacks:
        o = mk_out()
        kb.kbmod_pipeline_host(*stk, sts[0].psf, sts[0].times, vx, vy, sp, o, arena)
        singles.append([t.clone() for t in o])
    outs = [mk_out() for _ in stacks]
    kb.kbmod_pipeline_host_batch(stacks, sts[0].psf, sts[0].times, vx, vy, sp, outs, arena)
    for a, b in zip(singles, outs):
        for x, y in zip(a, b):
            assert torch.equal(x, y)
    assert any(int((o[2] >= 0).sum()) > 0 for o in outs)
    assert not torch.equal(outs[0][2], outs[1][2])  # different stacks, different results
