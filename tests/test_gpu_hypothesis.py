"""CUDA path against the oracle on randomly drawn problems (hypothesis): sizes, histogram widths,
operators, key skew and the share of ignored keys are drawn, not listed -- the listed shapes of test_gpu_parity.py cover
the tile boundaries, these cover what nobody thought of listing."""
import numpy as np
import pytest
import torch
from hypothesis import given, settings, strategies as st

import oracle
from paper_2310_03568_b200 import binding as B

pytestmark = pytest.mark.gpu
SET = dict(max_examples=60, deadline=None, derandomize=True)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def nrel(got, ref):
    got = np.asarray(got, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    assert got.shape == ref.shape and np.all(np.isfinite(got))
    den, err = np.max(np.abs(ref)), np.max(np.abs(got - ref))
    return (0.0 if err == 0.0 else np.inf) if den == 0.0 else err / den


def draw_keys(rng, n, w, skew):
    if skew:  # a few hot bins hold most of the elements
        hot = rng.integers(0, w, size=max(1, min(w, 5)))
        is_ = np.where(rng.random(n) < 0.7, hot[rng.integers(0, hot.size, size=n)], rng.integers(0, w, size=n))
    else:
        is_ = rng.integers(0, w, size=n)
    oob = rng.random(n) < 0.03
    is_ = np.where(oob, rng.choice([-1, -7, w, w + 9, -(2**40), 2**40], size=n), is_)
    return is_.astype(np.int64)


@settings(**SET)
@given(n=st.integers(1, 60000), w=st.one_of(st.integers(1, 1100), st.integers(1100, 13000), st.integers(13000, 140000)),
       opname=st.sampled_from(["add", "min", "max", "mul"]), skew=st.booleans(), seed=st.integers(0, 2**20))
def test_rbi_vjp_on_drawn_problems(n, w, opname, skew, seed):
    rng = np.random.default_rng(seed)
    is_ = draw_keys(rng, n, w, skew)
    hb = rng.standard_normal(w).astype(np.float32)
    if opname == "mul":
        vs = (0.9 + 0.2 * rng.random(n)).astype(np.float32)
        vs[rng.random(n) < 0.02] = 0.0
    else:
        vs = np.round(rng.standard_normal(n), 1).astype(np.float32)  # ties
    got = B.vjp_reduce_by_index(B.Op.of(opname), w, dev(is_), dev(vs), dev(hb)).cpu().numpy()
    if opname == "add":
        assert np.array_equal(got.astype(np.float64), oracle.vjp_rbi_add(w, is_, hb))
    elif opname in ("min", "max"):
        assert np.array_equal(got.astype(np.float64), oracle.vjp_rbi_minmax(opname, w, is_, vs, hb)[0])  # a copy: bit-identical
    else:
        assert nrel(got, oracle.vjp_rbi_mul(w, is_, vs, hb)[0]) <= 1e-4


@settings(**SET)
@given(n=st.integers(1, 40000), name=st.sampled_from(["add", "mul", "linrec", "min", "max", "matmul2", "matmul3", "matmul5"]),
       seed=st.integers(0, 2**20))
def test_scan_vjp_on_drawn_problems(n, name, seed):
    rng = np.random.default_rng(seed)
    q = int(name[-1]) if name.startswith("matmul") else 0
    dtype = torch.float64 if name == "mul" else torch.float32
    npdt = np.float64 if name == "mul" else np.float32
    if q:
        a = rng.standard_normal((n, q, q))
        xs = np.linalg.qr(a)[0].reshape(n, q * q).astype(npdt)       # orthogonal factors: unit gain
    elif name == "linrec":
        xs = np.stack([0.9 + 0.1 * rng.random(n), rng.standard_normal(n)], axis=1).astype(npdt)
    elif name == "mul":
        xs = (0.99 + 0.02 * rng.random(n)).astype(npdt)
        xs[rng.random(n) < 1e-3] = 0.0
    else:
        xs = np.round(rng.standard_normal(n), 1).astype(npdt)
    yb = rng.standard_normal(xs.shape).astype(npdt)
    got = B.vjp_scan(B.Op.of(name, dtype), dev(xs), dev(yb)).cpu().numpy()
    ref = oracle.vjp_scan("matmul" if q else name, xs, yb, q=q)
    if name in ("min", "max"):
        assert np.array_equal(got != 0, np.asarray(ref) != 0)
    assert nrel(got, ref) <= (1e-10 if name == "mul" else 1e-4)
