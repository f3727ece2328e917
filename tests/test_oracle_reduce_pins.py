"""Pins of the oracle's `reduce` functions (oracle/vjp_oracle.c, section "reduce") against what the paper
and the mathematics fix -- never against the oracle itself and never against the CUDA path.

P:Lnnn = line of PAPER.md.  Section 3: general rule eq. 2 + Fig. 2; '+' P:L166-171;
min/max P:L174-186; '*' Fig. 3."""
import numpy as np
import pytest

import oracle

RNG = np.random.default_rng(20231003)


def satadd_fold(xs, S):
    acc = 0.0
    for x in xs:
        acc = min(acc + x, S)
    return acc


# ------------------------------------------------------------------ primal ------------------

@pytest.mark.parametrize("n", [0, 1, 2, 17, 1000])
def test_reduce_forward_is_the_numpy_reduction(n):
    xs = RNG.uniform(0.5, 1.5, n)
    assert oracle.reduce_forward("add", xs) == pytest.approx(np.sum(xs), rel=1e-13, abs=0.0 if n else 0.0)
    assert oracle.reduce_forward("mul", xs) == pytest.approx(np.prod(xs), rel=1e-12)
    assert oracle.reduce_forward("min", xs) == (np.min(xs) if n else np.inf)
    assert oracle.reduce_forward("max", xs) == (np.max(xs) if n else -np.inf)
    S = 0.4 * n
    assert oracle.reduce_forward("satadd", xs, S=S) == pytest.approx(satadd_fold(xs, S), rel=1e-13)


# ------------------------------------------------------------------ specialised rules -------

def test_add_replicates_y_bar():
    # as_bar = replicate n y_bar
    xb, _, _ = oracle.vjp_reduce("add", RNG.standard_normal(37), -2.25)
    np.testing.assert_array_equal(xb, np.full(37, -2.25))
    assert oracle.vjp_reduce("add", [], 1.0)[0].size == 0


@pytest.mark.parametrize("opname", ["min", "max"])
def test_minmax_is_one_hot_at_the_smallest_index_of_the_extremum(opname):
    # 0 for i != k, y_bar for k; duplicates -> the smallest index
    for n in (1, 2, 9, 500):
        xs = np.round(RNG.standard_normal(n), 1)            # rounding forces ties
        k_ref = int(np.argmin(xs) if opname == "min" else np.argmax(xs))   # numpy: first occurrence
        xb, k, e = oracle.vjp_reduce(opname, xs, 3.0)
        assert k == k_ref and e == xs[k_ref]
        want = np.zeros(n)
        want[k_ref] = 3.0
        np.testing.assert_array_equal(xb, want)


def test_minmax_edge_cases():
    # all elements equal to the neutral value: min^L((n,inf),(0,inf)) = (0,inf) -- index 0 takes it
    xb, k, e = oracle.vjp_reduce("min", [np.inf, np.inf, np.inf], 1.0)
    assert k == 0 and e == np.inf and xb.tolist() == [1.0, 0.0, 0.0]
    xb, k, e = oracle.vjp_reduce("max", [-np.inf, -np.inf], 1.0)
    assert k == 0 and xb.tolist() == [1.0, 0.0]
    # -0.0 == +0.0 under "<": a tie, the lower index wins (Q6)
    assert oracle.vjp_reduce("min", [0.0, -0.0], 1.0)[1] == 0
    # empty array: k = n, nothing is written ("discards the updates of out of bounds indices")
    xb, k, e = oracle.vjp_reduce("min", [], 1.0)
    assert xb.size == 0 and k == 0 and e == np.inf


def brute_force_product_of_others(xs):
    return np.array([np.prod(np.delete(xs, i)) for i in range(len(xs))])


@pytest.mark.parametrize("zeros_at", [(), (3,), (0,), (11,), (2, 7), (0, 5, 11)])
def test_mul_is_the_product_of_the_others_in_all_three_zero_cases(zeros_at):
    # d y / d a_i = l_i * r_i; Fig. 3: no zero -> (y/a) y_bar; exactly one zero ->
    # only that element gets y^{>0} y_bar; more -> 0
    xs = RNG.uniform(0.5, 2.0, 12) * RNG.choice([-1.0, 1.0], 12)
    for z in zeros_at:
        xs[z] = 0.0
    yb = 1.75
    xb, nz, pnz = oracle.vjp_reduce("mul", xs, yb)
    np.testing.assert_allclose(xb, brute_force_product_of_others(xs) * yb, rtol=1e-12, atol=0.0)
    assert nz == len(zeros_at)
    assert pnz == pytest.approx(np.prod(xs[xs != 0.0]), rel=1e-13)
    # the three cases of Fig. 3 written out
    if len(zeros_at) == 0:
        np.testing.assert_allclose(xb, (np.prod(xs) / xs) * yb, rtol=1e-12)
    elif len(zeros_at) == 1:
        want = np.zeros(12)
        want[zeros_at[0]] = pnz * yb
        np.testing.assert_allclose(xb, want, rtol=1e-12, atol=0.0)
    else:
        assert not xb.any()


# ------------------------------------------------------------------ general rule ------------

def test_general_rule_ls_rs_are_the_two_exclusive_scans():
    # Fig. 2: ls = scan^exc, rs = reverse (scan^exc (reverse as))
    xs = RNG.uniform(0.5, 1.5, 50)
    _, ls, rs = oracle.vjp_reduce_general("add", xs, 1.0, with_lr=True)
    np.testing.assert_allclose(ls, np.concatenate([[0.0], np.cumsum(xs)[:-1]]), rtol=1e-13)
    np.testing.assert_allclose(rs, np.concatenate([np.cumsum(xs[::-1])[:-1][::-1], [0.0]]), rtol=1e-13)
    _, ls, rs = oracle.vjp_reduce_general("mul", xs, 1.0, with_lr=True)
    np.testing.assert_allclose(ls, np.concatenate([[1.0], np.cumprod(xs)[:-1]]), rtol=1e-12)
    np.testing.assert_allclose(rs, np.concatenate([np.cumprod(xs[::-1])[:-1][::-1], [1.0]]), rtol=1e-12)
    _, ls, rs = oracle.vjp_reduce_general("min", xs, 1.0, with_lr=True)
    np.testing.assert_array_equal(ls, np.concatenate([[np.inf], np.minimum.accumulate(xs)[:-1]]))
    np.testing.assert_array_equal(rs, np.concatenate([np.minimum.accumulate(xs[::-1])[:-1][::-1], [np.inf]]))


@pytest.mark.parametrize("opname", ["add", "mul", "min", "max"])
def test_general_rule_equals_the_specialised_rules(opname):
    # section 3.2: the specialised rules are instances of eq. 2
    for n in (1, 2, 13, 300):
        xs = np.round(RNG.uniform(0.5, 1.5, n), 2) if opname in ("min", "max") else RNG.uniform(0.5, 1.5, n)
        if opname == "mul" and n > 5:
            xs[3] = 0.0
        got = oracle.vjp_reduce_general(opname, xs, 0.7)
        want = oracle.vjp_reduce(opname, xs, 0.7)[0]
        np.testing.assert_allclose(got, want, rtol=1e-12, atol=0.0)


def test_general_rule_satadd_closed_form():
    # min(a+b, S) on non-negative reals: y = min(sum, S); d y / d a_i = 1 iff sum < S
    xs = RNG.uniform(0.0, 1.0, 64)
    tot = float(np.sum(xs))
    np.testing.assert_array_equal(oracle.vjp_reduce_general("satadd", xs, 2.5, S=tot + 1.0), np.full(64, 2.5))
    np.testing.assert_array_equal(oracle.vjp_reduce_general("satadd", xs, 2.5, S=tot - 1.0), np.zeros(64))
    # S = inf: satadd is '+'
    np.testing.assert_array_equal(oracle.vjp_reduce_general("satadd", xs, 2.5, S=np.inf),
                                  oracle.vjp_reduce("add", xs, 2.5)[0])


@pytest.mark.parametrize("opname,S", [("add", 0.0), ("mul", 0.0), ("satadd", 1e9), ("min", 0.0), ("max", 0.0)])
def test_gradient_by_central_differences(opname, S):
    # y_bar * dy/da_i by central differences of the plain fold (smooth points: distinct values, no saturation)
    n = 11
    xs = RNG.uniform(0.6, 1.4, n) + 0.01 * np.arange(n)
    yb, h = 1.3, 1e-6
    fd = np.empty(n)
    for i in range(n):
        xp, xm = xs.copy(), xs.copy()
        xp[i] += h
        xm[i] -= h
        fd[i] = yb * (oracle.reduce_forward(opname, xp, S=S) - oracle.reduce_forward(opname, xm, S=S)) / (2 * h)
    np.testing.assert_allclose(oracle.vjp_reduce_general(opname, xs, yb, S=S), fd, rtol=1e-6, atol=1e-8)
    if opname != "satadd":
        np.testing.assert_allclose(oracle.vjp_reduce(opname, xs, yb)[0], fd, rtol=1e-6, atol=1e-8)


@pytest.mark.parametrize("opname", ["add", "mul", "min", "max", "satadd"])
def test_reduce_is_reduce_by_index_with_one_bin(opname):
    # a reduce is a reduce_by_index whose keys are all 0 (Fig. 2 vs Fig. 4 with w = 1) -- this ties the new
    # functions to the reduce-by-index ones, which have their own pins (test_oracle_pins.py)
    n = 200
    xs = RNG.uniform(0.0, 1.5, n)
    xs[RNG.random(n) < 0.02] = 0.0
    keys = np.zeros(n, dtype=np.int64)
    S = 0.45 * n
    assert oracle.reduce_forward(opname, xs, S=S) == oracle.reduce_by_index_forward(opname, 1, keys, xs, S=S)[0]
    np.testing.assert_array_equal(oracle.vjp_reduce_general(opname, xs, 1.5, S=S),
                                  oracle.vjp_rbi_general(opname, 1, keys, xs, [1.5], S=S))
