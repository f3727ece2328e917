"""Pins of the oracle's exclusive-scan functions (oracle/__init__.py, "exclusive scan") against the definition written
out as a plain loop, closed forms and central finite differences -- never against the oracle itself or the CUDA path.
scan^exc: ys_0 = e, ys_i = x_0 (.) ... (.) x_{i-1} (the paper's Fig. 2)."""
import numpy as np
import pytest

import oracle

RNG = np.random.default_rng(20231003)


def op_fn(opname, q):
    if opname == "add":
        return lambda a, b: a + b
    if opname == "mul":
        return lambda a, b: a * b
    if opname == "min":
        return np.minimum
    if opname == "max":
        return np.maximum
    if opname == "linrec":      # (A, B) (+) (a, b) = (a A, a B + b)  (BASELINE config 3)
        return lambda P, x: np.array([x[0] * P[0], x[0] * P[1] + x[1]])
    return lambda R, X: (R.reshape(q, q) @ X.reshape(q, q)).ravel()


def neutral(opname, q):
    return {"add": np.array([0.0]), "mul": np.array([1.0]), "min": np.array([np.inf]), "max": np.array([-np.inf]),
            "linrec": np.array([1.0, 0.0])}.get(opname, np.eye(q).ravel() if q else None)


def fold_exclusive(opname, q, xs):
    """The definition, one element at a time."""
    f, acc = op_fn(opname, q), neutral(opname, q)
    out = []
    for x in xs:
        out.append(acc)
        acc = f(acc, x)
    return np.array(out).reshape(xs.shape)


def make(opname, q, n):
    if opname == "matmul":
        return RNG.uniform(-1.0, 1.0, (n, q * q)) / np.sqrt(q)
    if opname == "linrec":
        return np.stack([RNG.uniform(0.5, 1.2, n), RNG.standard_normal(n)], axis=1)
    if opname in ("min", "max"):
        return RNG.permutation(n).astype(np.float64) + 0.25          # distinct values: smooth points
    return RNG.uniform(0.6, 1.4, n)


CASES = [("add", 0), ("mul", 0), ("min", 0), ("max", 0), ("linrec", 0), ("matmul", 2), ("matmul", 3)]


@pytest.mark.parametrize("opname,q", CASES)
@pytest.mark.parametrize("n", [0, 1, 2, 11])
def test_forward_is_the_definition(opname, q, n):
    xs = make(opname, q, n)
    got = oracle.scan_exclusive_forward(opname, xs, q)
    want = fold_exclusive(opname, q, xs) if n else xs
    np.testing.assert_allclose(got, want, rtol=1e-13, atol=0.0)
    if n:
        assert np.array_equal(got.reshape(n, -1)[0], neutral(opname, q))


def test_add_is_the_strict_suffix_sum():
    yb = RNG.standard_normal(40)
    got = oracle.vjp_scan_exclusive("add", RNG.standard_normal(40), yb)
    want = np.concatenate([np.cumsum(yb[::-1])[::-1][1:], [0.0]])      # sum of ys_bar_j over j > i
    np.testing.assert_allclose(got, want, rtol=1e-13, atol=1e-15)


def test_mul_closed_form_without_zeros_and_with_one_zero():
    xs = RNG.uniform(0.5, 1.5, 12)
    yb = RNG.standard_normal(12)
    ys = np.concatenate([[1.0], np.cumprod(xs)[:-1]])
    want = np.array([np.sum(yb[i + 1:] * ys[i + 1:]) / xs[i] for i in range(12)])
    np.testing.assert_allclose(oracle.vjp_scan_exclusive("mul", xs, yb), want, rtol=1e-12)
    xs[4] = 0.0                                                         # outputs 5.. are 0; only x_4 and x_0..3 matter
    got = oracle.vjp_scan_exclusive("mul", xs, yb)
    assert not got[5:].any()
    pre = np.concatenate([[1.0], np.cumprod(xs[:4])])                   # ys_0..4
    rest = np.concatenate([[1.0], np.cumprod(xs[5:])[:-1]])             # ys_j / (ys_4 x_4) for j = 5..
    assert got[4] == pytest.approx(pre[4] * np.sum(yb[5:] * rest), rel=1e-12)


@pytest.mark.parametrize("opname,q", CASES)
def test_gradient_by_central_differences_of_the_definition(opname, q):
    n = 9
    xs = make(opname, q, n)
    yb = RNG.standard_normal(xs.shape)
    got = oracle.vjp_scan_exclusive(opname, xs, yb, q)
    flat = xs.ravel()
    fd = np.empty_like(flat)
    h = 1e-6
    for i in range(flat.size):
        xp, xm = flat.copy(), flat.copy()
        xp[i] += h
        xm[i] -= h
        fp, fm = fold_exclusive(opname, q, xp.reshape(xs.shape)), fold_exclusive(opname, q, xm.reshape(xs.shape))
        d = np.where(np.isfinite(fp), fp, 0.0) - np.where(np.isfinite(fm), fm, 0.0)       # ys_0 = +-inf for min / max
        fd[i] = np.sum(d * yb) / (2 * h)
    np.testing.assert_allclose(got.ravel(), fd, rtol=2e-6, atol=1e-7)
    assert not got.reshape(n, -1)[-1].any()                             # x_{n-1} enters no output


def test_edge_sizes():
    assert oracle.vjp_scan_exclusive("add", [], []).size == 0
    assert oracle.vjp_scan_exclusive("mul", [3.0], [5.0]).tolist() == [0.0]
    assert oracle.scan_exclusive_forward("linrec", np.zeros((1, 2))).tolist() == [[1.0, 0.0]]
