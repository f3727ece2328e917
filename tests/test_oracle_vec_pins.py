"""Pins of the oracle's vectorised-operator functions (sections 3.2.4 / 4.2.5; eq. 3): the vectorised
combinators written out as explicit loops over rows of d scalars, and finite differences of those loops."""
import numpy as np
import pytest

import oracle

RNG = np.random.default_rng(252)
F = {"add": lambda a, b: a + b, "mul": lambda a, b: a * b, "min": np.minimum, "max": np.maximum}
E = {"add": 0.0, "mul": 1.0, "min": np.inf, "max": -np.inf}


def rbi_vec_loop(op, w, is_, vss):
    """reduce_by_index with map2 (.) on whole rows: the loop of P:L335 with vector elements."""
    hist = np.full((w, vss.shape[1]), E[op])
    for i, k in enumerate(is_):
        if 0 <= k < w:
            hist[k] = F[op](hist[k], vss[i])
    return hist


def scan_vec_loop(op, xss):
    out = xss.copy()
    for i in range(1, len(xss)):
        out[i] = F[op](out[i - 1], xss[i])
    return out


@pytest.mark.parametrize("op", ["add", "mul", "min", "max"])
def test_vectorised_forward_is_the_row_loop(op):
    n, d, w = 120, 5, 7
    is_ = RNG.integers(-1, w + 1, size=n)
    vss = RNG.uniform(0.5, 1.5, (n, d))
    np.testing.assert_allclose(oracle.rbi_forward_vec(op, w, is_, vss), rbi_vec_loop(op, w, is_, vss), rtol=1e-12)


@pytest.mark.parametrize("op", ["add", "mul"])
def test_vectorised_rbi_vjp_by_central_differences(op):
    n, d, w, h = 12, 3, 4, 1e-6
    is_ = RNG.integers(-1, w + 1, size=n)
    vss = RNG.uniform(0.5, 1.5, (n, d))
    hb = RNG.standard_normal((w, d))
    want = np.zeros((n, d))
    for i in range(n):
        for c in range(d):
            p, m = vss.copy(), vss.copy()
            p[i, c] += h
            m[i, c] -= h
            want[i, c] = np.sum((rbi_vec_loop(op, w, is_, p) - rbi_vec_loop(op, w, is_, m)) / (2 * h) * hb)
    np.testing.assert_allclose(oracle.vjp_rbi_vec(op, w, is_, vss, hb), want, rtol=1e-6, atol=1e-8)


def test_vectorised_min_is_one_hot_per_bin_and_column():
    n, d, w = 200, 4, 6
    is_ = RNG.integers(0, w, size=n)
    vss = np.round(RNG.standard_normal((n, d)), 1)          # ties: the lowest index wins, per column
    hb = RNG.standard_normal((w, d))
    got = oracle.vjp_rbi_vec("min", w, is_, vss, hb)
    want = np.zeros((n, d))
    for c in range(d):
        for k in range(w):
            idx = np.flatnonzero(is_ == k)
            if idx.size:
                want[idx[np.argmin(vss[idx, c])], c] = hb[k, c]
    np.testing.assert_array_equal(got, want)


@pytest.mark.parametrize("op", ["add", "mul"])
def test_vectorised_scan_vjp_by_central_differences(op):
    n, d, h = 9, 3, 1e-6
    xss = RNG.uniform(0.5, 1.5, (n, d))
    yb = RNG.standard_normal((n, d))
    want = np.zeros((n, d))
    for i in range(n):
        for c in range(d):
            p, m = xss.copy(), xss.copy()
            p[i, c] += h
            m[i, c] -= h
            want[i, c] = np.sum((scan_vec_loop(op, p) - scan_vec_loop(op, m)) / (2 * h) * yb)
    np.testing.assert_allclose(oracle.vjp_scan_vec(op, xss, yb), want, rtol=1e-6, atol=1e-8)
