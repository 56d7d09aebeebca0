"""kbmod_sigmag_postfilter_static: the post-filter entry point that allocates nothing (its scratch is a static device
array inside the library, include/kbmod_b200.h).  Its outputs must equal those of kbmod_sigmag_postfilter -- the same
kernels' arithmetic on caller-owned scratch -- bit for bit, on two calls in a row (the second call finds the first call's
flags and counters in the array).  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _lightcurves(seed, n, T, frac_bright):
    """configs[4]-like lightcurves: noise at the DECam variance level, some with a real signal, 20 % of the epochs of
    every tenth lightcurve replaced by outliers, 5 % invalid epochs."""
    rng = np.random.default_rng(seed)
    phi = rng.uniform(0.02, 0.05, (n, T)).astype(np.float32)
    psi = (rng.standard_normal((n, T)) * np.sqrt(phi)).astype(np.float32)
    bright = rng.random(n) < frac_bright
    psi[bright] += (rng.uniform(2.0, 6.0, (int(bright.sum()), 1)) * np.sqrt(phi[bright])).astype(np.float32)
    out = (rng.random((n, T)) < 0.2) & (np.arange(n)[:, None] % 10 == 0)
    psi[out] += (10.0 * np.sqrt(phi[out])).astype(np.float32)
    phi[rng.random((n, T)) < 0.05] = 0.0
    return psi, phi


def test_postfilter_static_equals_postfilter_twice():
    import torch
    import paper_2109_03296_b200 as kb

    assert torch.cuda.is_available()
    dev = torch.device("cuda:0")
    sp = kb.SearchParams(K=1, min_obs=13, min_lh=10.0)
    # two calls in a row with different sizes and contents: the second is smaller, so stale flags of the first call sit
    # right behind its range in the shared array
    for call, (seed, n) in enumerate(((11, 300_007), (12, 120_011))):
        psi, phi = _lightcurves(seed, n, 26, 0.3)
        d_psi, d_phi = torch.from_numpy(psi).to(dev), torch.from_numpy(phi).to(dev)
        ref = kb.kbmod_sigmag_postfilter(d_psi, d_phi, sp)
        got = kb.kbmod_sigmag_postfilter_static(d_psi, d_phi, sp)
        torch.cuda.synchronize()
        n_ref, n_got = int(ref["n_pass"][0].item()), int(got["n_survivors"][0].item())
        assert n_ref == int(ref["passed"].sum().item())
        assert 0 < n_ref < n, "the case must have both survivors and rejections"
        assert n_got == n_ref, (call, n_got, n_ref)
        assert torch.equal(got["survivors"][:n_got], ref["survivors"][:n_ref])
        assert torch.equal(got["kept"], ref["kept"])
        # same kernel, same inputs: bit-identical (the tolerance of the parity tests, 1e-4 relative, holds a fortiori)
        assert torch.equal(got["lh"].view(torch.int32), ref["lh"].view(torch.int32))
        assert torch.equal(got["flux"].view(torch.int32), ref["flux"].view(torch.int32))


def test_postfilter_static_limits():
    import torch
    import paper_2109_03296_b200 as kb

    dev = torch.device("cuda:0")
    sp = kb.SearchParams(K=1, min_obs=1, min_lh=10.0)
    # beyond the static array: rejected with a clear error, nothing launched
    n = kb.binding.POSTFILTER_STATIC_MAX_LC + 1
    z = torch.zeros((n, 1), dtype=torch.float32, device=dev)
    with pytest.raises(kb.KbmodError, match="KBMOD_POSTFILTER_STATIC_MAX_LC"):
        kb.kbmod_sigmag_postfilter_static(z, z, sp)
    # an empty list: zero survivors
    e = torch.zeros((0, 26), dtype=torch.float32, device=dev)
    r = kb.kbmod_sigmag_postfilter_static(e, e, sp)
    torch.cuda.synchronize()
    assert int(r["n_survivors"][0].item()) == 0
