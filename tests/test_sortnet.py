"""The generated compare-exchange networks of csrc/sortnet_gen.cuh, checked on the CPU: the header is parsed (not the
generator re-run), every network is applied to 0/1 vectors of every density (the zero-one principle), to random
permutations and to floats with ties, infinities, signed zeros and denormals; the output must be sorted and must be
exactly the multiset it was given."""
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HDR = os.path.join(ROOT, "paper_2109_03296_b200", "csrc", "sortnet_gen.cuh")


def networks():
    src = open(HDR).read()
    out = {}
    for m in re.finditer(r"struct SortNet<(\d+)> \{.*?static __device__ __forceinline__ void sort\(.*?\) \{(.*?)\n    \}", src, re.S):
        out[int(m.group(1))] = [(int(a), int(b)) for a, b in re.findall(r"KB_CE\((\d+),(\d+)\)", m.group(2))]
    sizes = [int(x) for x in re.search(r"#define KB_SORTNET_SIZES (.*)", src).group(1).split(",")]
    assert sorted(out) == sizes
    return out


def apply(net, a):
    """a: float32 [cases][n]; the kernel's compare-exchange on every row at once."""
    a = a.copy()
    for i, j in net:
        lo, hi = np.minimum(a[:, i], a[:, j]), np.maximum(a[:, i], a[:, j])
        a[:, i], a[:, j] = lo, hi
    return a


def test_header_compare_exchange_is_min_max():
    src = open(HDR).read()
    assert "fminf(a[i], a[j])" in src and "fmaxf(a[i], a[j])" in src


def test_every_network_sorts():
    rng = np.random.default_rng(0)
    for n, net in networks().items():
        assert all(0 <= i < j < n for i, j in net)
        cases = []
        for ones in range(n + 1):  # every density of 0/1 inputs: near-sorted and unbalanced ones included
            for _ in range(300):
                v = np.zeros(n, np.float32)
                v[rng.choice(n, ones, replace=False)] = 1.0
                cases.append(v)
        if n <= 12:
            cases = [np.array([(b >> k) & 1 for k in range(n)], np.float32) for b in range(1 << n)]
        for _ in range(2000):
            cases.append(rng.permutation(n).astype(np.float32))
            cases.append(rng.integers(0, 4, n).astype(np.float32))                      # many ties
            x = rng.standard_normal(n).astype(np.float32) * np.float32(10.0) ** rng.integers(-40, 38)
            x[rng.random(n) < 0.15] = np.inf                                            # the padding of invalid epochs
            x[rng.random(n) < 0.05] = -np.inf
            x[rng.random(n) < 0.05] = 0.0
            x[rng.random(n) < 0.05] = -0.0
            cases.append(x)
        with np.errstate(over="ignore"):
            a = np.stack(cases).astype(np.float32)
        with np.errstate(over="ignore"):
            s = apply(net, a)
        assert np.all(s[:, :-1] <= s[:, 1:]), n
        # the multiset of values is preserved (numpy's min / max may pick either zero of a +0 / -0 pair: compare values)
        assert np.array_equal(np.sort(s, axis=1), np.sort(a, axis=1)), n
