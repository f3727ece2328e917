"""GPU parity of the reduce VJP (NEXT row f2; section 3 of the paper) against the f64 CPU oracle.  Bars as
everywhere: bit-exact for indices, zero counts and pure copies; normwise 1e-4 (f32) / 1e-10 (f64) otherwise."""
import numpy as np
import pytest
import torch

import oracle
from paper_2310_03568_b200 import binding as B
from paper_2310_03568_b200 import workloads as W

pytestmark = pytest.mark.gpu

import os

SIZES = [1, 2, 3, 5, 511, 2047, 2049, 4097, 65537, 300007, 1 << 21]
if os.environ.get("VJP_TEST_MAX_N"):
    SIZES = [n for n in SIZES if n <= int(os.environ["VJP_TEST_MAX_N"])]


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def nrel(got, ref):
    got = np.asarray(got, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    assert got.shape == ref.shape and np.all(np.isfinite(got))
    den, err = np.max(np.abs(ref)), np.max(np.abs(got - ref))
    return (0.0 if err == 0.0 else np.inf) if den == 0.0 else err / den


def satadd_S(xs, want_saturated):
    tot = float(np.sum(xs.astype(np.float64)))
    return float(np.float32(tot * (0.5 if want_saturated else 1.5) + 1.0))


@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("opname", ["add", "min", "max", "mul", "satadd"])
def test_reduce_forward_matches_oracle(opname, n):
    d = W.f2_reduce(opname, n=n, seed=n % 7)
    S = satadd_S(d["xs"], True)
    got = B.reduce_forward(B.Op.of(opname, S=S), dev(d["xs"])).cpu().numpy()[0]
    ref = oracle.reduce_forward(opname, d["xs"], S=S)
    if opname in ("min", "max"):
        assert got == ref
    else:
        # f64 accumulation inside the kernel: only the final rounding to f32 (and the cancellation of a
        # zero-mean sum, measured against the sum of magnitudes) remains
        scale = float(np.sum(np.abs(d["xs"].astype(np.float64)))) if opname == "add" else abs(ref)
        assert abs(got - ref) <= 1e-6 * max(scale, 1e-30)


def test_reduce_forward_of_an_empty_array_is_the_neutral_element():
    x = torch.zeros(4, device="cuda")[:0]
    for name, e in (("add", 0.0), ("mul", 1.0), ("min", np.inf), ("max", -np.inf), ("satadd", 0.0)):
        assert B.reduce_forward(B.Op.of(name, S=1.0), x).item() == e
    assert B.reduce_forward(B.Op.of("add", torch.float64), x.double()).item() == 0.0


@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_reduce_add_vjp_replicates_y_bar(n, dtype):
    yb = torch.tensor([1.625], dtype=dtype, device="cuda")
    got = B.vjp_reduce(B.Op.of("add", dtype), None, yb, n=n).cpu().numpy()
    ref, _, _ = oracle.vjp_reduce("add", np.zeros(n), 1.625)
    assert np.array_equal(got.astype(np.float64), ref)


@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("opname", ["min", "max"])
def test_reduce_minmax_vjp_bit_exact(opname, n):
    d = W.f2_reduce(opname, n=n, seed=1)
    op = B.Op.of(opname)
    got = B.vjp_reduce(op, dev(d["xs"]), dev(d["y_bar"])).cpu().numpy()
    ref, k, e = oracle.vjp_reduce(opname, d["xs"], float(d["y_bar"][0]))
    ai, av = B.reduce_lifted(op, dev(d["xs"]))
    assert ai.item() == k and float(av.item()) == e                      # smallest index on ties
    assert np.array_equal(got.astype(np.float64), ref)                   # a pure copy


@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("nzeros", [0, 1, 2])
def test_reduce_mul_vjp_three_zero_cases(nzeros, n):
    d = W.f2_reduce("mul", n=n, seed=2)
    xs = d["xs"].copy()
    for z in range(min(nzeros, n)):
        xs[(n // 3 + z * (n // 2 + 1)) % n] = 0.0
    op = B.Op.of("mul")
    got = B.vjp_reduce(op, dev(xs), dev(d["y_bar"])).cpu().numpy()
    ref, rz, rp = oracle.vjp_reduce("mul", xs, float(d["y_bar"][0]))
    ai, av = B.reduce_lifted(op, dev(xs))
    assert ai.item() == rz                                               # zero count bit-exact
    assert abs(float(av.item()) - rp) <= 1e-4 * abs(rp)
    assert nrel(got, ref) <= 1e-4


@pytest.mark.parametrize("n", [1, 5, 4097, 300007])
@pytest.mark.parametrize("saturated", [False, True])
def test_reduce_satadd_general_rule(saturated, n):
    d = W.f2_reduce("satadd", n=n, seed=3)
    S = satadd_S(d["xs"], saturated)
    got = B.vjp_reduce(B.Op.of("satadd", S=S), dev(d["xs"]), dev(d["y_bar"])).cpu().numpy()
    ref = oracle.vjp_reduce_general("satadd", d["xs"], float(d["y_bar"][0]), S=S)
    assert np.array_equal(got.astype(np.float64), ref)                   # every adjoint is y_bar or 0


@pytest.mark.parametrize("n", [1, 5, 4097, 100003])
@pytest.mark.parametrize("opname", ["add", "min", "max", "mul"])
def test_reduce_general_rule_with_specialisable_operators(opname, n):
    """eq. 2: force_general routes the common operators through the two exclusive scans."""
    d = W.f2_reduce(opname, n=n, seed=4)
    xs = d["xs"].copy()
    if opname == "mul" and n > 3:
        xs[n // 2] = 0.0
    got = B.vjp_reduce(B.Op.of(opname, force_general=True), dev(xs), dev(d["y_bar"])).cpu().numpy()
    ref = oracle.vjp_reduce_general(opname, xs, float(d["y_bar"][0]))
    if opname == "mul":
        assert nrel(got, ref) <= 1e-4
    else:
        assert np.array_equal(got.astype(np.float64), ref)


@pytest.mark.parametrize("opname", ["add", "min", "mul", "satadd"])
def test_reduce_vjp_accumulate(opname):
    n = 100003
    d = W.f2_reduce(opname, n=n, seed=5)
    S = satadd_S(d["xs"], False)
    prior = np.random.default_rng(8).standard_normal(n).astype(np.float32)
    out = dev(prior)
    B.vjp_reduce(B.Op.of(opname, S=S, accumulate=True), dev(d["xs"]), dev(d["y_bar"]), out=out)
    yb = float(d["y_bar"][0])
    con = oracle.vjp_reduce_general("satadd", d["xs"], yb, S=S) if opname == "satadd" else oracle.vjp_reduce(opname, d["xs"], yb)[0]
    got = out.cpu().numpy()
    if opname == "mul":
        assert nrel(got.astype(np.float64) - prior, con) <= 1e-4
    else:
        assert np.array_equal(got, (prior.astype(np.float64) + con).astype(np.float32))


def test_reduce_rejects_bad_arguments():
    x = torch.ones(8, device="cuda")
    yb = torch.ones(1, device="cuda")
    with pytest.raises(B.VjpError):
        B.vjp_reduce(B.Op.of("linrec"), x, yb)
    with pytest.raises(B.VjpError):
        B.vjp_reduce(B.Op.of("min", torch.float64), x.double(), yb.double())
    with pytest.raises(B.VjpError):
        B.vjp_reduce(B.Op.of("mul"), None, yb, n=8)      # xs is required unless op is '+'
    with pytest.raises(B.VjpError):
        B.vjp_reduce(B.Op.of("mul"), x, torch.ones(2, device="cuda"))
    assert B.vjp_reduce(B.Op.of("mul"), x[:0], yb).numel() == 0


@pytest.mark.parametrize("opname", ["add", "min", "max", "mul", "satadd"])
def test_f2_reduce_full_size(opname):
    d = W.f2_reduce(opname)
    S = satadd_S(d["xs"], True)
    yb = float(d["y_bar"][0])
    op = B.Op.of(opname, S=S)
    got = B.vjp_reduce(op, dev(d["xs"]), dev(d["y_bar"])).cpu().numpy()
    if opname == "satadd":
        ref = oracle.vjp_reduce_general("satadd", d["xs"], yb, S=S)
    else:
        ref, ri, rv = oracle.vjp_reduce(opname, d["xs"], yb)
    if opname == "mul":
        assert nrel(got, ref) <= 1e-4
        ai, av = B.reduce_lifted(op, dev(d["xs"]))
        assert ai.item() == ri and abs(float(av.item()) - rv) <= 1e-4 * abs(rv)
    else:
        assert np.array_equal(got.astype(np.float64), ref)
        if opname in ("min", "max"):
            ai, _ = B.reduce_lifted(op, dev(d["xs"]))
            assert ai.item() == ri == (1 << 24) // 3
