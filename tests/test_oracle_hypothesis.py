"""Property tests of the oracle on randomly drawn shapes (hypothesis): what must hold for ANY input --
the VJP is linear in the output adjoint, <J v, w> = <v, J^T w> against a forward difference of the primal, adjoints of
ignored keys are exactly 0, and the min/max rule puts every bin's adjoint on exactly one element of that bin."""
import numpy as np
from hypothesis import given, settings, strategies as st

import oracle

SET = dict(max_examples=40, deadline=None, derandomize=True)


@settings(**SET)
@given(n=st.integers(1, 300), op=st.sampled_from(["add", "mul", "linrec"]), seed=st.integers(0, 2**20))
def test_scan_vjp_is_linear_in_the_output_adjoint(n, op, seed):
    rng = np.random.default_rng(seed)
    d = 2 if op == "linrec" else 1
    xs = 0.5 + rng.random((n, d)) if d > 1 else 0.5 + rng.random(n)
    a, b = rng.standard_normal(xs.shape), rng.standard_normal(xs.shape)
    va, vb = oracle.vjp_scan(op, xs, a), oracle.vjp_scan(op, xs, b)
    vab = oracle.vjp_scan(op, xs, 2.0 * a - 3.0 * b)
    assert np.allclose(vab, 2.0 * va - 3.0 * vb, rtol=1e-10, atol=1e-10)


@settings(**SET)
@given(n=st.integers(1, 200), op=st.sampled_from(["add", "mul", "linrec"]), seed=st.integers(0, 2**20))
def test_scan_vjp_is_the_transpose_of_the_forward_derivative(n, op, seed):
    rng = np.random.default_rng(seed)
    d = 2 if op == "linrec" else 1
    shape = (n, d) if d > 1 else (n,)
    xs = 0.8 + 0.4 * rng.random(shape)
    v, w = rng.standard_normal(shape), rng.standard_normal(shape)
    h = 1e-6
    jv = (oracle.scan_forward(op, xs + h * v) - oracle.scan_forward(op, xs - h * v)) / (2 * h)   # J v by central differences
    lhs = float(np.sum(jv * w))
    rhs = float(np.sum(v * oracle.vjp_scan(op, xs, w)))
    assert abs(lhs - rhs) <= 1e-5 * (1.0 + abs(lhs) + abs(rhs)) * max(1.0, float(np.max(np.abs(jv))))


@settings(**SET)
@given(n=st.integers(1, 400), w=st.integers(1, 50), seed=st.integers(0, 2**20))
def test_rbi_minmax_adjoint_goes_to_exactly_one_member_of_each_bin(n, w, seed):
    rng = np.random.default_rng(seed)
    is_ = rng.integers(-3, w + 3, size=n, dtype=np.int64)
    vs = np.round(rng.standard_normal(n), 1)          # rounding forces ties
    hb = 1.0 + rng.random(w)                          # strictly positive: a non-zero adjoint marks the receiver
    for op in ("min", "max"):
        vb, arg, ext = oracle.vjp_rbi_minmax(op, w, is_, vs, hb)
        inr = (is_ >= 0) & (is_ < w)
        assert np.all(vb[~inr] == 0.0)                 # ignored keys: exactly 0 (Q3)
        for k in range(w):
            members = np.flatnonzero(is_ == k)
            if members.size == 0:
                assert arg[k] == n
                continue
            best = vs[members].min() if op == "min" else vs[members].max()
            first = members[np.flatnonzero(vs[members] == best)[0]]   # lowest index among the ties (Q4)
            assert arg[k] == first and ext[k] == best
            assert vb[first] == hb[k] and np.count_nonzero(vb[members]) == 1


@settings(**SET)
@given(n=st.integers(1, 300), w=st.integers(1, 40), seed=st.integers(0, 2**20), zero_rate=st.sampled_from([0.0, 0.05, 0.3]))
def test_rbi_mul_adjoint_is_the_product_of_the_others(n, w, seed, zero_rate):
    rng = np.random.default_rng(seed)
    is_ = rng.integers(-2, w + 2, size=n, dtype=np.int64)
    vs = 0.5 + rng.random(n)
    vs[rng.random(n) < zero_rate] = 0.0
    hb = rng.standard_normal(w)
    vb = oracle.vjp_rbi_mul(w, is_, vs, hb)[0]
    for i in range(n):
        k = is_[i]
        if k < 0 or k >= w:
            assert vb[i] == 0.0
            continue
        others = np.flatnonzero((is_ == k) & (np.arange(n) != i))
        ref = hb[k] * np.prod(vs[others])
        assert abs(vb[i] - ref) <= 1e-12 * (1.0 + abs(ref))
