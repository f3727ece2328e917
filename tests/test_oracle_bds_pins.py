"""Pins of the oracle's block-diagonal (non-redundant BDS) scan rule: an operator that applies a small
operator to each of k blocks of its element has a Jacobian of k DIFFERENT diagonal blocks, and its scan VJP is k scans
with the scaled-down operator.  Checked against the tuple operator written out directly: dense Jacobians by finite
differences, never against the oracle itself or the CUDA path."""
import numpy as np
import pytest

import oracle

RNG = np.random.default_rng(20231003)


def linrec(P, x):      # (A, B) (+) (a, b) = (a A, a B + b)
    return np.array([x[0] * P[0], x[0] * P[1] + x[1]])


def matmul2(R, X):
    return (R.reshape(2, 2) @ X.reshape(2, 2)).ravel()


SMALL = {"linrec": (linrec, 2, np.array([1.0, 0.0]), 0), "matmul": (matmul2, 4, np.eye(2).ravel(), 2)}


def tuple_op(name, k):
    f, a, _, _ = SMALL[name]
    return lambda R, X: np.concatenate([f(R[c * a:(c + 1) * a], X[c * a:(c + 1) * a]) for c in range(k)])


def scan_inclusive(name, k, xss):
    f, (_, a, e, _) = tuple_op(name, k), SMALL[name]
    acc, out = np.tile(e, k), []
    for x in xss:
        acc = f(acc, x)
        out.append(acc)
    return np.array(out)


@pytest.mark.parametrize("name,k", [("linrec", 3), ("matmul", 2)])
def test_jacobian_of_the_tuple_operator_is_block_diagonal_with_different_blocks(name, k):
    f, a = tuple_op(name, k), SMALL[name][1]
    R, X = RNG.uniform(0.5, 1.5, k * a), RNG.uniform(0.5, 1.5, k * a)
    h, J = 1e-6, np.empty((k * a, k * a))
    for j in range(k * a):
        rp, rm = R.copy(), R.copy()
        rp[j] += h
        rm[j] -= h
        J[:, j] = (f(rp, X) - f(rm, X)) / (2 * h)
    blocks = [J[c * a:(c + 1) * a, c * a:(c + 1) * a] for c in range(k)]
    off = J.copy()
    for c in range(k):
        off[c * a:(c + 1) * a, c * a:(c + 1) * a] = 0.0
    assert np.max(np.abs(off)) < 1e-9                                   # block-diagonal
    assert not np.allclose(blocks[0], blocks[1], atol=1e-3)             # the blocks differ: BDS, not RBDS


@pytest.mark.parametrize("name,k", [("linrec", 3), ("matmul", 2)])
def test_vjp_is_k_scans_of_the_small_operator(name, k):
    a, q = SMALL[name][1], SMALL[name][3]
    n = 7
    xss = RNG.uniform(0.5, 1.2, (n, k * a))
    ybar = RNG.standard_normal((n, k * a))
    got = oracle.vjp_scan_vec(name, xss, ybar, q=q)
    flat, fd, h = xss.ravel(), np.empty(n * k * a), 1e-6
    for i in range(flat.size):
        xp, xm = flat.copy(), flat.copy()
        xp[i] += h
        xm[i] -= h
        fd[i] = np.sum((scan_inclusive(name, k, xp.reshape(n, -1)) - scan_inclusive(name, k, xm.reshape(n, -1))) * ybar) / (2 * h)
    np.testing.assert_allclose(got.ravel(), fd, rtol=2e-6, atol=1e-7)


def test_arity_one_is_unchanged():
    xss, ybar = RNG.uniform(0.5, 1.5, (9, 3)), RNG.standard_normal((9, 3))
    got = oracle.vjp_scan_vec("mul", xss, ybar)
    for c in range(3):
        np.testing.assert_array_equal(got[:, c], oracle.vjp_scan("mul", xss[:, c], ybar[:, c]))
