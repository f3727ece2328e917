"""Pins for the CPU oracle (oracle/vjp_oracle.c): everything here checks the oracle against
something OTHER than itself -- hand-worked fixtures, closed forms the paper states, numpy
library routines, brute force on tiny inputs, finite differences (exact for the multilinear
operators), the dot-product identity <Jv,w> = <v,J^T w>, and PPAD's rule (Fig. 11) with a
numerically differentiated operator.  No GPU, no CUDA package."""
import json
import os

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
RNG = np.random.default_rng(20231003)


# ------------------------------------------------------------------ hand-worked fixtures
def _cases():
    with open(os.path.join(HERE, "golden", "hand_worked.json")) as f:
        return json.load(f)["cases"]


@pytest.mark.parametrize("case", _cases(), ids=lambda c: c["name"])
def test_hand_worked(case):
    if case["kind"] == "scan":
        got = oracle.vjp_scan(case["op"], case["xs"], case["ys_bar"], q=case["q"])
        np.testing.assert_allclose(got, np.asarray(case["xs_bar"], dtype=float), rtol=0, atol=1e-12)
    elif case["kind"] == "sort":
        sk, perm = oracle.rbi_sort_perm(case["w"], case["is"])
        assert sk.tolist() == case["sorted_keys"] and perm.tolist() == case["perm"]
    else:
        op, w = case["op"], case["w"]
        if op == "add":
            got = oracle.vjp_rbi_add(w, case["is"], case["hist_bar"])
        elif op in ("min", "max"):
            got, arg, _ = oracle.vjp_rbi_minmax(op, w, case["is"], case["vs"], case["hist_bar"])
            assert arg.tolist() == case["arg"]
        elif op == "mul":
            got, zeros, prod = oracle.vjp_rbi_mul(w, case["is"], case["vs"], case["hist_bar"])
            assert zeros.tolist() == case["zeros"]
            np.testing.assert_allclose(prod, case["prod_nz"], rtol=0, atol=1e-12)
        else:
            got = oracle.vjp_rbi_general(op, w, case["is"], case["vs"], case["hist_bar"], S=case["S"])
        np.testing.assert_allclose(got, np.asarray(case["vs_bar"], dtype=float), rtol=0, atol=1e-12)
        # the general rule (eq. 5) must reproduce every specialised rule
        if op != "satadd":
            gen = oracle.vjp_rbi_general(op, w, case["is"], case["vs"], case["hist_bar"])
            np.testing.assert_allclose(gen, np.asarray(case["vs_bar"], dtype=float), rtol=0, atol=1e-12)


# ------------------------------------------------------------------ independent numpy primal scans
def np_scan(op, xs, q=0):
    xs = np.asarray(xs, dtype=np.float64)
    if op == "add":
        return np.cumsum(xs)
    if op == "mul":
        return np.cumprod(xs)
    if op == "min":
        return np.minimum.accumulate(xs)
    if op == "max":
        return np.maximum.accumulate(xs)
    out = np.empty_like(xs)
    if op == "linrec":          # y_i = (prod a, value of the recurrence b_i + a_i * B_{i-1})
        A, B = 1.0, 0.0
        for i, (a, b) in enumerate(xs):
            A, B = a * A, a * B + b
            out[i] = (A, B)
        return out
    if op == "matmul":
        R = np.eye(q)
        o2 = out.reshape(xs.shape[0], q * q)
        for i in range(xs.shape[0]):
            R = R @ xs[i].reshape(q, q)
            o2[i] = R.reshape(-1)
        return out
    raise ValueError(op)


SCAN_CASES = [("add", 0, 1), ("mul", 0, 1), ("linrec", 0, 2), ("matmul", 1, 1), ("matmul", 2, 4),
              ("matmul", 3, 9), ("matmul", 5, 25)]


def _scan_inputs(op, d, n, rng):
    xs = rng.uniform(0.5, 1.5, size=(n, d)) * rng.choice([-1.0, 1.0], size=(n, d))
    yb = rng.standard_normal((n, d))
    if d == 1:
        xs, yb = xs[:, 0], yb[:, 0]
    return xs, yb


@pytest.mark.parametrize("op,q,d", SCAN_CASES + [("min", 0, 1), ("max", 0, 1)])
def test_scan_forward_matches_numpy(op, q, d):
    xs, _ = _scan_inputs(op, d, 37, RNG)
    want = np_scan(op, xs, q)
    assert np.abs(oracle.scan_forward(op, xs, q=q) - want).max() <= 1e-13 * (1.0 + np.abs(want).max())


def _dense_jacobian_fd(op, q, xs, h=1e-3):
    """J[out, in] by central differences of the INDEPENDENT numpy primal.  All scan operators
    tested here are linear in every single input scalar, so central differences are exact."""
    flat = xs.reshape(-1).copy()
    m = flat.size
    J = np.empty((m, m))
    for j in range(m):
        p, mn = flat.copy(), flat.copy()
        p[j] += h
        mn[j] -= h
        J[:, j] = (np_scan(op, p.reshape(xs.shape), q) - np_scan(op, mn.reshape(xs.shape), q)).reshape(-1) / (2 * h)
    return J


@pytest.mark.parametrize("op,q,d", SCAN_CASES)
@pytest.mark.parametrize("n", [1, 2, 3, 8, 17])
def test_scan_vjp_equals_dense_jacobian_transpose(op, q, d, n):
    if d * n > 260:
        n = 260 // d
    xs, yb = _scan_inputs(op, d, n, RNG)
    J = _dense_jacobian_fd(op, q, xs)
    want = (J.T @ yb.reshape(-1)).reshape(xs.shape)
    got = oracle.vjp_scan(op, xs, yb, q=q)
    scale = np.abs(want).max() + 1.0
    assert np.abs(got - want).max() / scale < 1e-8


def test_scan_mul_with_zeros_against_dense_jacobian():
    for zpos in ([0], [5], [11], [3, 7], [0, 11]):
        xs, yb = _scan_inputs("mul", 1, 12, RNG)
        xs[zpos] = 0.0
        J = _dense_jacobian_fd("mul", 0, xs)
        np.testing.assert_allclose(oracle.vjp_scan("mul", xs, yb), J.T @ yb, rtol=0, atol=1e-8)


def test_scan_add_closed_form_reverse_cumsum():
    yb = RNG.standard_normal(1000)
    np.testing.assert_allclose(oracle.vjp_scan("add", RNG.standard_normal(1000), yb),
                               np.cumsum(yb[::-1])[::-1], rtol=1e-13, atol=1e-12)


def test_scan_mul_no_zero_closed_form():
    # without zeros  xb_i = sum_{j>=i} yb_j * y_j / x_i
    xs = RNG.uniform(0.9, 1.1, 200)
    yb = RNG.standard_normal(200)
    ys = np.cumprod(xs)
    want = np.cumsum((yb * ys)[::-1])[::-1] / xs
    np.testing.assert_allclose(oracle.vjp_scan("mul", xs, yb), want, rtol=1e-11, atol=1e-11)


def test_scan_mul_everything_right_of_a_zero():
    xs = RNG.uniform(0.9, 1.1, 50)
    xs[20] = 0.0
    yb = RNG.standard_normal(50)
    got = oracle.vjp_scan("mul", xs, yb)
    assert np.all(got[21:] == 0.0)               # y_j = 0 for j >= 20, so r_{i-1} = 0 for i > 20
    ys = np.cumprod(xs)
    tail = np.cumprod(np.r_[1.0, xs[21:]])       # x_20's adjoint sees the products to its right
    np.testing.assert_allclose(got[20], ys[19] * np.sum(yb[20:] * tail), rtol=1e-12)


def test_linrec_brute_force_and_reduction_to_add():
    n = 40
    xs, yb = _scan_inputs("linrec", 2, n, RNG)
    a = xs[:, 0]
    got = oracle.vjp_scan("linrec", xs, yb)
    # b_bar_m = sum_{j>=m} Bbar_j * prod_{m<t<=j} a_t
    want_b = np.array([sum(yb[j, 1] * np.prod(a[m + 1:j + 1]) for j in range(m, n)) for m in range(n)])
    np.testing.assert_allclose(got[:, 1], want_b, rtol=1e-11, atol=1e-11)
    ones = xs.copy()
    ones[:, 0] = 1.0                              # a == 1: B is a plain prefix sum of b
    got1 = oracle.vjp_scan("linrec", ones, yb)
    np.testing.assert_allclose(got1[:, 1], np.cumsum(yb[::-1, 1])[::-1], rtol=1e-12, atol=1e-12)


def test_matmul_reductions():
    n = 30
    # q = 1 is the scalar product scan
    xs, yb = _scan_inputs("mul", 1, n, RNG)
    np.testing.assert_allclose(oracle.vjp_scan("matmul", xs, yb, q=1), oracle.vjp_scan("mul", xs, yb), rtol=1e-13)
    # diagonal matrices: q independent scalar product scans
    q = 3
    dg = RNG.uniform(0.5, 1.5, (n, q))
    X = np.zeros((n, q, q))
    X[:, np.arange(q), np.arange(q)] = dg
    G = RNG.standard_normal((n, q, q))
    got = oracle.vjp_scan("matmul", X.reshape(n, -1), G.reshape(n, -1), q=q).reshape(n, q, q)
    for c in range(q):
        ys = np.cumprod(dg[:, c])
        want = np.cumsum((G[:, c, c] * ys)[::-1])[::-1] / dg[:, c]
        np.testing.assert_allclose(got[:, c, c], want, rtol=1e-11)


def test_matmul_rotations_reduce_to_scan_add():
    # 2x2 rotations commute: prefix product = rotation by the cumulative angle, so the adjoint of
    # the angles is a reverse prefix sum of <Ybar_j, Rot'(phi_j)>.
    n = 64
    th = RNG.uniform(-1, 1, n)
    rot = lambda t: np.stack([np.cos(t), -np.sin(t), np.sin(t), np.cos(t)], axis=-1)
    drot = lambda t: np.stack([-np.sin(t), -np.cos(t), np.cos(t), -np.sin(t)], axis=-1)
    G = RNG.standard_normal((n, 4))
    xb = oracle.vjp_scan("matmul", rot(th), G, q=2)
    phi = np.cumsum(th)
    dphi = np.sum(G * drot(phi), axis=1)
    want = np.cumsum(dphi[::-1])[::-1]
    got = np.sum(xb * drot(th), axis=1)           # chain rule through X_i = Rot(theta_i)
    np.testing.assert_allclose(got, want, rtol=1e-11, atol=1e-11)


def _num_jac(f, x, h=1e-4):
    x = np.asarray(x, dtype=float)
    cols = []
    for j in range(x.size):
        p, m = x.copy(), x.copy()
        p[j] += h
        m[j] -= h
        cols.append((f(p) - f(m)) / (2 * h))
    return np.stack(cols, axis=1)                 # [out, in]


@pytest.mark.parametrize("op,q,d", [c for c in SCAN_CASES if c[0] != "add"])
def test_scan_vjp_equals_ppad_rule(op, q, d):
    """PPAD's rule (Fig. 11) evaluated sequentially with the operator differentiated
    NUMERICALLY: x_hat_i = xb_i + (d op(x_i, u_{i+1})/d x_i)^T x_hat_{i+1}, then
    u_bar_i = (d op(x_{i-1}, u_i)/d u_i)^T x_hat_i -- an independent derivation of the same VJP."""
    n = 9
    us, xb = _scan_inputs(op, d, n, RNG)
    us2, xb2 = us.reshape(n, d), xb.reshape(n, d)

    def opf(a, b):
        return np_scan(op, np.stack([a, b]).reshape((2,) + us.shape[1:]), q)[-1].reshape(-1)

    x = np_scan(op, us, q).reshape(n, d)
    x_hat = np.zeros((n, d))
    x_hat[n - 1] = xb2[n - 1]
    for i in range(n - 2, -1, -1):
        J1 = _num_jac(lambda t: opf(t, us2[i + 1]), x[i])
        x_hat[i] = xb2[i] + J1.T @ x_hat[i + 1]
    want = np.zeros((n, d))
    want[0] = x_hat[0]
    for i in range(1, n):
        J2 = _num_jac(lambda t: opf(x[i - 1], t), us2[i])
        want[i] = J2.T @ x_hat[i]
    got = oracle.vjp_scan(op, us, xb, q=q).reshape(n, d)
    np.testing.assert_allclose(got, want, rtol=1e-7, atol=1e-7)


@pytest.mark.parametrize("op,q,d", SCAN_CASES)
def test_scan_dot_product_identity(op, q, d):
    """<J v, w> = <v, J^T w>, J v from central differences of the oracle's own PRIMAL (which is
    pinned to numpy above)."""
    n = 300
    xs, w = _scan_inputs(op, d, n, RNG)
    if op != "add":
        xs = 1.0 + 0.05 * (xs - np.sign(xs))      # keep long products bounded
        if op == "matmul":
            xs = (np.eye(q).reshape(-1)[None, :] + 0.05 * RNG.standard_normal((n, q * q))).reshape(xs.shape)
    v = RNG.standard_normal(xs.shape)
    h = 1e-5
    Jv = (oracle.scan_forward(op, xs + h * v, q=q) - oracle.scan_forward(op, xs - h * v, q=q)) / (2 * h)
    lhs = np.sum(Jv * w)
    rhs = np.sum(v * oracle.vjp_scan(op, xs, w, q=q))
    assert abs(lhs - rhs) <= 1e-6 * (abs(lhs) + abs(rhs) + 1.0)


def test_scan_min_max_one_hot_first_occurrence():
    xs = np.array([3.0, 1.0, 2.0, 1.0, 0.5, 0.5, 4.0])
    yb = np.arange(1.0, 8.0)
    # prefix minima are attained at indices 0,1,1,1,4,4,4 (first occurrence keeps it)
    np.testing.assert_array_equal(oracle.vjp_scan("min", xs, yb), [1, 2 + 3 + 4, 0, 0, 5 + 6 + 7, 0, 0])
    np.testing.assert_array_equal(oracle.vjp_scan("max", -xs, yb), [1, 2 + 3 + 4, 0, 0, 5 + 6 + 7, 0, 0])


# ------------------------------------------------------------------ reduce-by-index
def _rbi_inputs(n, w, rng, oob=True):
    lo, hi = (-3, w + 3) if oob else (0, w)
    return rng.integers(lo, hi, size=n), rng.standard_normal(n), rng.standard_normal(w)


def test_rbi_forward_matches_numpy_ufunc_at():
    n, w = 500, 13
    is_, vs, _ = _rbi_inputs(n, w, RNG)
    ok = (is_ >= 0) & (is_ < w)
    for op, ufunc, neutral in (("add", np.add, 0.0), ("mul", np.multiply, 1.0),
                               ("min", np.minimum, np.inf), ("max", np.maximum, -np.inf)):
        want = np.full(w, neutral)
        ufunc.at(want, is_[ok], vs[ok])
        np.testing.assert_allclose(oracle.reduce_by_index_forward(op, w, is_, vs), want, rtol=1e-12, atol=1e-12)
    S = 1.5
    pos = np.abs(vs)
    want = np.minimum(np.bincount(is_[ok], weights=pos[ok], minlength=w), S)
    np.testing.assert_allclose(oracle.reduce_by_index_forward("satadd", w, is_, pos, S=S), want, rtol=1e-12)


def test_rbi_add_closed_form_gather():
    n, w = 1000, 17
    is_, _, hb = _rbi_inputs(n, w, RNG)
    ok = (is_ >= 0) & (is_ < w)
    got = oracle.vjp_rbi_add(w, is_, hb)
    np.testing.assert_array_equal(got, np.where(ok, hb[np.clip(is_, 0, w - 1)], 0.0))
    cnt = np.bincount(is_[ok], minlength=w)
    np.testing.assert_allclose(got.sum(), np.sum(cnt * hb), rtol=1e-12)


@pytest.mark.parametrize("op", ["min", "max"])
def test_rbi_minmax_against_numpy(op):
    n, w = 2000, 23
    is_, vs, hb = _rbi_inputs(n, w, RNG)
    vs = np.round(vs, 1)                          # many ties
    is_[is_ == 5] = 6                             # an empty bin
    ok = (is_ >= 0) & (is_ < w)
    got, arg, ext = oracle.vjp_rbi_minmax(op, w, is_, vs, hb)
    uf, neutral = (np.minimum, np.inf) if op == "min" else (np.maximum, -np.inf)
    want_ext = np.full(w, neutral)
    uf.at(want_ext, is_[ok], vs[ok])
    np.testing.assert_array_equal(ext, want_ext)
    for k in range(w):
        hits = np.flatnonzero(ok & (is_ == k) & (vs == want_ext[k]))
        assert arg[k] == (hits[0] if hits.size else n)                                  # lowest index
    assert arg[5] == n and np.isinf(ext[5])
    nz = np.flatnonzero(got)
    assert set(nz) <= set(arg[arg < n])
    np.testing.assert_array_equal(got[arg[arg < n]], hb[arg < n])


def test_rbi_minmax_first_element_equal_to_neutral_wins():
    got, arg, ext = oracle.vjp_rbi_minmax("min", 1, [0, 0], [np.inf, np.inf], [2.0])
    assert arg.tolist() == [0] and got.tolist() == [2.0, 0.0]                           # min^L (n,inf)(0,inf) = (0,inf)


def test_rbi_mul_brute_force_product_of_others_and_zero_cases():
    n, w = 300, 11
    is_, vs, hb = _rbi_inputs(n, w, RNG)
    vs[RNG.random(n) < 0.03] = 0.0
    ok = (is_ >= 0) & (is_ < w)
    got, zeros, prod = oracle.vjp_rbi_mul(w, is_, vs, hb)
    want = np.zeros(n)
    for i in range(n):
        if ok[i]:
            others = [vs[j] for j in range(n) if j != i and is_[j] == is_[i]]
            want[i] = np.prod(others) * hb[is_[i]]
    np.testing.assert_allclose(got, want, rtol=1e-10, atol=1e-13)
    np.testing.assert_array_equal(zeros, np.bincount(is_[ok & (vs == 0)], minlength=w))
    # Fig. 3's three-way return sweep from the lifted primal's outputs
    for i in range(n):
        if not ok[i]:
            fig3 = 0.0
        elif zeros[is_[i]] == 0:
            fig3 = prod[is_[i]] / vs[i] * hb[is_[i]]
        elif zeros[is_[i]] == 1 and vs[i] == 0:
            fig3 = prod[is_[i]] * hb[is_[i]]
        else:
            fig3 = 0.0
        assert abs(fig3 - got[i]) <= 1e-10 * (1 + abs(got[i]))
    assert {0, 1}.issubset(set(np.minimum(zeros, 2).tolist()))


@pytest.mark.parametrize("op", ["add", "mul", "min", "max"])
def test_general_rule_equals_specialised_rules(op):
    n, w = 4000, 37
    is_, vs, hb = _rbi_inputs(n, w, RNG)
    if op in ("min", "max"):
        vs = np.round(vs, 2)
    if op == "mul":
        vs = RNG.uniform(0.8, 1.2, n)
        vs[RNG.random(n) < 0.01] = 0.0
    gen = oracle.vjp_rbi_general(op, w, is_, vs, hb)
    if op == "add":
        spec = oracle.vjp_rbi_add(w, is_, hb)
    elif op == "mul":
        spec = oracle.vjp_rbi_mul(w, is_, vs, hb)[0]
    else:
        spec = oracle.vjp_rbi_minmax(op, w, is_, vs, hb)[0]
    np.testing.assert_allclose(gen, spec, rtol=1e-12, atol=1e-300)


def test_general_rule_l_r_are_segmented_exclusive_scans_of_the_sorted_values():
    # Fig. 4: ls / rs come from segmented exclusive scans over the stably sorted values.
    n, w = 1000, 9
    is_, vs, hb = _rbi_inputs(n, w, RNG)
    _, ls, rs = oracle.vjp_rbi_general("add", w, is_, vs, hb, with_lr=True)
    sk, perm = oracle.rbi_sort_perm(w, is_)
    svs = vs[perm]
    for k in range(w):
        seg = np.flatnonzero(sk == k)
        excl = np.r_[0.0, np.cumsum(svs[seg])[:-1]]
        np.testing.assert_allclose(ls[perm[seg]], excl, rtol=1e-12, atol=1e-12)
        rexcl = np.r_[0.0, np.cumsum(svs[seg][::-1])[:-1]][::-1]
        np.testing.assert_allclose(rs[perm[seg]], rexcl, rtol=1e-12, atol=1e-12)


def test_sort_perm_is_numpy_stable_argsort_of_clamped_keys():
    n, w = 5000, 29
    is_ = RNG.integers(-5, w + 5, size=n)
    clamped = np.where((is_ >= 0) & (is_ < w), is_, w)
    sk, perm = oracle.rbi_sort_perm(w, is_)
    want = np.argsort(clamped, kind="stable")
    np.testing.assert_array_equal(perm, want)
    np.testing.assert_array_equal(sk, clamped[want])


def test_satadd_closed_form_and_limits():
    n, w, S = 6000, 20, 150.0
    is_ = RNG.integers(-2, w + 2, size=n)
    vs = RNG.random(n)
    hb = RNG.standard_normal(w)
    ok = (is_ >= 0) & (is_ < w)
    tot = np.bincount(is_[ok], weights=vs[ok], minlength=w)
    assert (tot < S).any() and (tot > S).any()
    # non-negative values: saturation is monotone, so the adjoint passes iff the bin total < S
    want = np.where(ok, hb[np.clip(is_, 0, w - 1)] * (tot[np.clip(is_, 0, w - 1)] < S), 0.0)
    np.testing.assert_array_equal(oracle.vjp_rbi_general("satadd", w, is_, vs, hb, S=S), want)
    # S = inf is plain '+'
    np.testing.assert_array_equal(oracle.vjp_rbi_general("satadd", w, is_, vs, hb, S=np.inf),
                                  oracle.vjp_rbi_add(w, is_, hb))


@pytest.mark.parametrize("op,S", [("add", 0), ("mul", 0), ("min", 0), ("max", 0), ("satadd", 12.0)])
def test_rbi_dot_product_identity(op, S):
    n, w = 400, 15
    is_ = RNG.integers(-2, w + 2, size=n)
    vs = RNG.uniform(0.1, 1.0, n)                 # distinct values: min/max differentiable; satadd away from the kink
    hb = RNG.standard_normal(w)
    v = RNG.standard_normal(n)
    h = 1e-7
    f = lambda x: oracle.reduce_by_index_forward(op, w, is_, x, S=S)
    Jv = (f(vs + h * v) - f(vs - h * v)) / (2 * h)
    lhs = float(np.sum(Jv * hb))
    if op == "add":
        g = oracle.vjp_rbi_add(w, is_, hb)
    elif op == "mul":
        g = oracle.vjp_rbi_mul(w, is_, vs, hb)[0]
    elif op in ("min", "max"):
        g = oracle.vjp_rbi_minmax(op, w, is_, vs, hb)[0]
    else:
        g = oracle.vjp_rbi_general(op, w, is_, vs, hb, S=S)
    rhs = float(np.sum(v * g))
    assert abs(lhs - rhs) <= 1e-5 * (abs(lhs) + abs(rhs) + 1.0)


def test_reduce_is_rbi_with_one_bin():
    # reduce = reduce-by-index with w = 1 (Fig. 2 vs Fig. 4): '+' replicates ybar
    n = 100
    vs = RNG.standard_normal(n)
    got = oracle.vjp_rbi_general("add", 1, np.zeros(n, dtype=np.int64), vs, [3.5])
    np.testing.assert_array_equal(got, np.full(n, 3.5))


def test_edge_cases():
    assert oracle.vjp_scan("add", [], []).size == 0
    np.testing.assert_array_equal(oracle.vjp_scan("mul", [7.0], [2.0]), [2.0])          # xb[0] = rb[0]
    assert oracle.vjp_rbi_add(4, [], [1, 2, 3, 4]).size == 0
    np.testing.assert_array_equal(oracle.vjp_rbi_add(2, [-1, 2, 9], [1.0, 2.0]), [0, 0, 0])
    got, arg, _ = oracle.vjp_rbi_minmax("min", 3, [7, -1], [1.0, 2.0], [1.0, 2.0, 3.0])
    assert arg.tolist() == [2, 2, 2] and not got.any()
