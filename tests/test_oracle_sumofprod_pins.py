"""Pins of the oracle's sumOfProd functions (invertible-operator rule, sections 3.3 and 4.2.4; Fig. 6)
against what the paper and the mathematics fix.  P:Lnnn = line of PAPER.md."""
import numpy as np
import pytest

import oracle

RNG = np.random.default_rng(318)


def pairs(n):
    return RNG.uniform(-1.5, 1.5, size=(n, 2))


def test_operator_is_associative_commutative_with_neutral_00():
    a, b, c = pairs(3)
    np.testing.assert_allclose(oracle.sop_apply(a, b), oracle.sop_apply(b, a), rtol=1e-14)
    np.testing.assert_allclose(oracle.sop_apply(oracle.sop_apply(a, b), c), oracle.sop_apply(a, oracle.sop_apply(b, c)),
                               rtol=1e-13, atol=1e-14)
    np.testing.assert_array_equal(oracle.sop_apply(a, [0.0, 0.0]), a)
    # the printed definition: (p1 + p2 + s1*s2, s1 + s2)
    np.testing.assert_allclose(oracle.sop_apply([1.0, 2.0], [3.0, 5.0]), [1 + 3 + 2 * 5, 7.0])


def test_inverse_property_3():
    # P:L286 (3): if z = a (.) b then a = z (.)_inv b and b = z (.)_inv a
    for _ in range(20):
        a, b = pairs(2)
        z = oracle.sop_apply(a, b)
        np.testing.assert_allclose(oracle.sop_inv(z, b), a, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(oracle.sop_inv(z, a), b, rtol=1e-12, atol=1e-13)
    # the printed inverse: (p - p2 - (s - s2)*s2, s - s2)
    np.testing.assert_allclose(oracle.sop_inv([14.0, 7.0], [3.0, 5.0]), [14 - 3 - 2 * 5, 2.0])


def test_near_homomorphism_sum_of_pairwise_products():
    # map f> as |> reduce sumOfProd (0,0) |> f<  =  sum_{i<j} a_i a_j, with f>(a) = (0,a), f<(p,_) = p
    a = RNG.standard_normal(40)
    vs = np.stack([np.zeros(40), a], axis=1)
    hist = oracle.rbi_sop_forward(1, np.zeros(40, dtype=np.int64), vs)
    brute = sum(a[i] * a[j] for i in range(40) for j in range(i + 1, 40))
    assert hist[0, 0] == pytest.approx(brute, rel=1e-12)
    assert hist[0, 1] == pytest.approx(a.sum(), rel=1e-13)


def closed_form_hist(w, is_, vs):
    h = np.zeros((w, 2))
    for k in range(w):
        m = is_ == k
        p, s = vs[m, 0], vs[m, 1]
        h[k] = [p.sum() + (s.sum() ** 2 - (s ** 2).sum()) / 2.0, s.sum()]
    return h


@pytest.mark.parametrize("n,w", [(0, 3), (1, 1), (50, 4), (400, 17)])
def test_forward_is_the_closed_form_per_bin(n, w):
    is_ = RNG.integers(-1, w + 1, size=n)
    vs = pairs(n)
    np.testing.assert_allclose(oracle.rbi_sop_forward(w, is_, vs), closed_form_hist(w, is_, vs), rtol=1e-11, atol=1e-12)


@pytest.mark.parametrize("general", [False, True])
def test_vjp_equals_dense_jacobian_transpose_by_central_differences(general):
    # the histogram is quadratic in the inputs: central differences are exact up to rounding
    n, w, h = 14, 3, 1e-5
    is_ = RNG.integers(-1, w + 1, size=n)
    vs = pairs(n)
    hb = RNG.standard_normal((w, 2))
    want = np.zeros((n, 2))
    for i in range(n):
        for c in range(2):
            vp, vm = vs.copy(), vs.copy()
            vp[i, c] += h
            vm[i, c] -= h
            d = (oracle.rbi_sop_forward(w, is_, vp) - oracle.rbi_sop_forward(w, is_, vm)) / (2 * h)
            want[i, c] = np.sum(d * hb)
    np.testing.assert_allclose(oracle.vjp_rbi_sop(w, is_, vs, hb, general=general), want, rtol=1e-7, atol=1e-8)


def test_invertible_rule_equals_general_rule_and_the_closed_form():
    # both rules give vs_bar_i = (Pbar_k, Pbar_k * (S_k - s_i) + Sbar_k); out-of-range keys get exactly 0
    n, w = 500, 9
    is_ = RNG.integers(-2, w + 2, size=n)
    vs = pairs(n)
    hb = RNG.standard_normal((w, 2))
    a = oracle.vjp_rbi_sop(w, is_, vs, hb, general=False)
    b = oracle.vjp_rbi_sop(w, is_, vs, hb, general=True)
    np.testing.assert_allclose(a, b, rtol=1e-11, atol=1e-12)
    S = closed_form_hist(w, is_, vs)[:, 1]
    ok = (is_ >= 0) & (is_ < w)
    want = np.zeros((n, 2))
    k = is_[ok]
    want[ok, 0] = hb[k, 0]
    want[ok, 1] = hb[k, 0] * (S[k] - vs[ok, 1]) + hb[k, 1]
    np.testing.assert_allclose(a, want, rtol=1e-11, atol=1e-12)
    assert not a[~ok].any() and not b[~ok].any()
