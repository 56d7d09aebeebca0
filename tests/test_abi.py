"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/kbmod_b200.h
declares, and its host-only logic (displacement table, argument validation, workspace sizing) is right.
No compute entry point is called here (no GPU)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2109_03296_b200 import binding, synth
from paper_2109_03296_b200 import build as kb_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    kb_build.build()
    return binding.lib()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "kbmod_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kbmod_[a-z_]+)\s*\(", src)))


def test_exports_every_declared_symbol(lib):
    names = declared_functions()
    assert len(names) >= 13
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/kbmod_b200.h but not exported"
    assert set(binding.EXPORTS) == set(names)
    for n in names:  # the Python binding carries the same names
        assert hasattr(binding, n) or n == "kbmod_last_error"
    assert binding.kbmod_version() >= 100


def test_default_params_are_the_papers(lib):
    p = binding.kbmod_default_params()
    assert (p.sigmag_enable, p.pct_lo, p.pct_hi, p.n_sigma, p.min_lh, p.K) == (1, 25.0, 75.0, 2.0, 10.0, 8)
    assert abs(p.sigmag_coeff - 0.7413) < 1e-7


@pytest.mark.parametrize("cfg", ["c1", "c2", "c3", "c4", "half"])
def test_displacement_table_bit_exact(lib, oracle, cfg):
    """(a2) is integer work: the library's table equals the oracle's, entry by entry (reading R5)."""
    if cfg == "c1":
        t, (vx, vy) = np.array([0, .5, 1, 1.5, 2.]), synth.config1_grid()
    elif cfg == "c2":
        t, (vx, vy) = synth.config2_medium(size=16, n_movers=0).times, synth.config2_grid()
    elif cfg == "c3":
        t, (vx, vy) = synth.night_times((7, 6, 7, 6)), synth.config3_grid()
    elif cfg == "c4":
        t, (vx, vy) = synth.night_times((9, 8, 8, 9, 8, 8)), synth.config4_grid()
    else:  # exact halves, negative and positive; times with a non-zero zero point, unsorted
        t = np.array([10.0, 10.5, 9.5, 11.0])
        vx = np.array([5, -5, 3, -3, 2.5, 0], np.float32)
        vy = np.array([-1, 1, -7, 7, 0, 1e-8], np.float32)
    dx, dy = binding.kbmod_displacements(t, vx, vy)
    ox, oy = oracle.displacements(t, vx, vy)
    assert np.array_equal(dx, ox) and np.array_equal(dy, oy)
    if cfg == "half":
        assert dx[0].tolist() == [0, 3, -2, 5] and dx[1].tolist() == [0, -2, 3, -5]  # round half up


def test_workspace_and_validation_without_gpu(lib):
    sp = binding.SearchParams(K=8)
    n1 = binding.kbmod_search_workspace_bytes(26, 4096, 2048, 8192, sp)
    n2 = binding.kbmod_search_workspace_bytes(26, 4096, 2048, 16384, sp)
    assert 0 < n1 < n2 and n1 % 256 == 0
    assert binding.kbmod_search_workspace_bytes(65, 10, 10, 1, sp) == 0  # T > 64 unsupported
    cp = sp.c()
    # argument validation happens before any CUDA call, so it is testable here
    rc = lib.kbmod_search(None, 5, 8, 8, None, None, None, 0, C.byref(cp), None, None, None, None, None,
                          C.c_size_t(0), None)
    assert rc == -1 and b"NULL" in lib.kbmod_last_error()
    rc = lib.kbmod_displacements(None, 1, None, None, 0, None, None)
    assert rc == -1
    one = (C.c_float * 4)()
    rc = lib.kbmod_prepare_psi_phi(one, one, None, 1, 2, 2, one, 1, 2, one, None)
    assert rc == -1 and b"odd" in lib.kbmod_last_error()
    rc = lib.kbmod_prepare_psi_phi(one, one, None, 65, 2, 2, one, 1, 1, one, None)
    assert rc == -2


def test_binding_refuses_cpu_tensors(lib):
    import torch
    with pytest.raises(TypeError):
        binding.kbmod_prepare_psi_phi(torch.zeros(1, 4, 4), torch.ones(1, 4, 4), None, np.ones((1, 1), np.float32))


def test_planner_host_logic_without_gpu(lib):
    """The pruned kernel's host planner (k-d velocity grouping, staging geometry, on-image masks) runs without a GPU
    through kbmod_plan_stats: the numbers DESIGN.md quotes for the benchmark configurations."""
    import math
    import paper_2109_03296_b200 as kb
    from paper_2109_03296_b200 import synth
    sp = kb.SearchParams()
    c3 = kb.kbmod_plan_stats(26, 4096, 2048, synth.night_times((7, 6, 7, 6)), *synth.config3_grid(), sp)
    assert not c3["too_scattered"] and c3["n_groups"] == 512
    assert 0.5 < c3["staged_bytes_per_eval"] < 0.65 and 0.10 < c3["off_image_fraction"] < 0.18
    c4 = kb.kbmod_plan_stats(50, 4096, 2048, synth.night_times((9, 8, 8, 9, 8, 8)), *synth.config4_grid(), sp)
    assert c4["n_groups"] == 2048 and 0.2 < c4["off_image_fraction"] < 0.3
    c1 = kb.kbmod_plan_stats(5, 64, 64, synth.config1_tiny().times, *synth.config1_grid(), sp)
    assert c1["n_groups"] == 16 and c1["off_image_fraction"] == 0.0  # 40 px/day x 2 d stays inside one 64x64 tile's regions
    # velocities all over the sky at a long baseline: groups are bisected until every staged region fits the ring
    rng = np.random.default_rng(0)
    vx, vy = rng.uniform(-3000, 3000, 200).astype(np.float32), rng.uniform(-3000, 3000, 200).astype(np.float32)
    sc = kb.kbmod_plan_stats(10, 512, 512, np.linspace(0, 5, 10), vx, vy, sp)
    assert sc["n_groups"] > math.ceil(200 / 16) and sc["off_image_fraction"] > 0.5
    # bad arguments are refused on the host
    with pytest.raises(kb.KbmodError):
        kb.kbmod_plan_stats(65, 64, 64, np.zeros(65), vx, vy, sp)


def test_percentile_positions_match_the_oracle_for_user_percentiles(lib, oracle):
    """The library's own percentile table (DevParams.rk_* / fr_*), read through the host-only kbmod_percentile_ranks,
    against the oracle for the paper's 25 / 75 and for user percentiles, both percentile definitions: the value the
    table picks from a sorted array must be the oracle's percentile of that array, bit for bit."""
    rng = np.random.default_rng(9)
    for lo, hi in ((25.0, 75.0), (10.0, 90.0), (0.0, 100.0), (33.3, 66.7), (50.0, 50.0), (5.0, 95.0)):
        for interp in (0, 1):
            sp = binding.SearchParams(pct_lo=lo, pct_hi=hi, pct_interp=interp)
            for n in range(1, 65):
                s = np.sort(rng.standard_normal(n).astype(np.float32))
                for (k, g), q in zip(binding.kbmod_percentile_ranks(sp, n), (lo, 50.0, hi)):
                    assert 0 <= k < n
                    if g < 0:
                        got = s[k]
                        if not interp:
                            assert k == oracle.pct_rank(q, n)
                    else:
                        assert interp and k + 1 < n and 0.0 <= g < 1.0
                        got = np.float32(s[k] + np.float32(np.float32(g) * np.float32(s[k + 1] - s[k])))
                    assert got == np.float32(oracle.pct_value(s, q, interp)), (lo, hi, interp, n, q)
    assert [k for k, _ in binding.kbmod_percentile_ranks(binding.SearchParams(), 26)] == [6, 12, 19]


def test_plan_without_gpu_and_row_bands_tile_the_image(lib):
    """kbmod_plan_create is host-only work (no CUDA context needed): kernel choice, velocity groups, padded-stack
    geometry, workspace size.  Row bands (one CCD shards over GPUs by start-pixel rows, results
    concatenate): the bands' plans cover every start row exactly once and each needs less workspace than the whole."""
    import paper_2109_03296_b200 as kb
    times = synth.night_times((7, 6, 7, 6))
    vx, vy = synth.config3_grid()
    sp = kb.SearchParams(K=8, min_obs=13)
    T, H, W = 26, 4096, 2048
    full = kb.Plan(T, H, W, times, vx, vy, sp)
    fi = full.info()
    assert fi["algo"] == kb.ALGO_PRUNED and fi["n_groups"] == 512 and not fi["too_scattered"]
    # motion about theta = 4.4 rad is towards -x, -y: the stack is padded on the low sides only, by the largest displacement
    dx, dy = kb.kbmod_displacements(times, vx, vy)
    assert fi["canvas"] == (W - dx.min() + max(dx.max(), 0), H - dy.min() + max(dy.max(), 0))
    assert dx.max() <= 0 and dy.max() <= 0 and -dx.min() == 919 and -dy.min() == 1567   # max |d| = (919, 1567)
    assert 0 < full.workspace_bytes() < kb.kbmod_search_workspace_bytes(T, H, W, len(vx), sp)
    assert full.workspace_bytes() == kb.kbmod_search_workspace_bytes_for(T, H, W, times, vx, vy, sp)
    n = 4
    edges = [H * r // n for r in range(n + 1)]
    covered = np.zeros(H, int)
    for r in range(n):
        band = kb.Plan(T, H, W, times, vx, vy, sp, rows=(edges[r], edges[r + 1]))
        bi = band.info()
        assert bi["algo"] == fi["algo"] and bi["n_groups"] == fi["n_groups"] and bi["canvas"] == fi["canvas"]
        assert band.workspace_bytes() < full.workspace_bytes()
        covered[band.rows[0]:band.rows[1]] += 1
        # bands towards +y keep more of their trajectories on the image than bands towards -y (the motion is towards -y)
        if r:
            assert bi["off_image_fraction"] <= prev + 1e-12
        prev = bi["off_image_fraction"]
        band.destroy()
    assert np.all(covered == 1)
    # direct kernel when nothing can be pruned; an empty band is legal
    assert kb.Plan(T, H, W, times, vx, vy, kb.SearchParams(min_lh=-np.inf)).info()["algo"] == kb.ALGO_DIRECT
    assert kb.Plan(T, H, W, times, vx, vy, sp, rows=(100, 100)).workspace_bytes() > 0
    with pytest.raises(kb.KbmodError):
        kb.Plan(T, H, W, times, vx, vy, sp, rows=(10, H + 1))
    with pytest.raises(kb.KbmodError):  # a canvas beyond 2^32 pixels: T = 64 with displacements in every direction
        kb.Plan(64, 4096, 2048, np.linspace(0, 10, 64), np.array([900, -900], np.float32), np.array([900, -900], np.float32), sp)
    full.destroy()
    kb.kbmod_release_thread_state()   # frees the plan kbmod_search_workspace_bytes_for cached; callable without a GPU
    kb.kbmod_release_thread_state()   # idempotent
