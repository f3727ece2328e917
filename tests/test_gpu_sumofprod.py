"""GPU parity of reduce-by-index with the invertible operator sumOfProd (NEXT row f1; sections 3.3 / 4.2.4, Fig. 6)
against the f64 CPU oracle: primal, invertible-operator rule, general rule.  Normwise 1e-4 (f32); keys out of range
get exactly (0, 0); the p component of vs_bar is a pure copy of hist_bar (bit-exact)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2310_03568_b200 import binding as B
from paper_2310_03568_b200 import workloads as W

pytestmark = pytest.mark.gpu

SHAPES = [(1, 1), (5, 3), (1000, 1), (4097, 7), (100003, 1024), (100003, 20000), (1 << 18, 70000)]


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def nrel(got, ref):
    got = np.asarray(got, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    assert got.shape == ref.shape and np.all(np.isfinite(got))
    den, err = np.max(np.abs(ref)), np.max(np.abs(got - ref))
    return (0.0 if err == 0.0 else np.inf) if den == 0.0 else err / den


@pytest.mark.parametrize("n,w", SHAPES)
@pytest.mark.parametrize("dist", ["uniform", "zipf"])
def test_sumofprod_forward_matches_oracle(dist, n, w):
    d = W.f1_rbi_sumofprod(n=n, w=w, dist=dist)
    got = B.rbi_sumofprod_forward(w, dev(d["is_"]), dev(d["vs"])).cpu().numpy()
    ref = oracle.rbi_sop_forward(w, d["is_"], d["vs"])
    assert nrel(got[:, 1], ref[:, 1]) <= 1e-4      # S
    assert nrel(got[:, 0], ref[:, 0]) <= 1e-4      # P (closed form in three sums)


@pytest.mark.parametrize("n,w", SHAPES)
@pytest.mark.parametrize("dist", ["uniform", "zipf"])
@pytest.mark.parametrize("general", [0, 1, 2])
def test_sumofprod_vjp_matches_oracle(general, dist, n, w):
    d = W.f1_rbi_sumofprod(n=n, w=w, dist=dist)
    got = B.vjp_rbi_sumofprod(w, dev(d["is_"]), dev(d["vs"]), dev(d["hist_bar"]), general=general).cpu().numpy()
    ref = oracle.vjp_rbi_sop(w, d["is_"], d["vs"], d["hist_bar"], general=general)
    assert np.array_equal(got[:, 0].astype(np.float64), ref[:, 0])          # Pbar copied, 0 out of range
    assert nrel(got[:, 1], ref[:, 1]) <= 1e-4
    oob = (d["is_"] < 0) | (d["is_"] >= w)
    assert not got[oob].any()


@pytest.mark.parametrize("general", [0, 1, 2])
def test_sumofprod_vjp_accumulate_and_empty(general):
    n, w = 50021, 333
    d = W.f1_rbi_sumofprod(n=n, w=w)
    prior = np.random.default_rng(4).standard_normal((n, 2)).astype(np.float32)
    out = dev(prior).view(-1)
    B.vjp_rbi_sumofprod(w, dev(d["is_"]), dev(d["vs"]), dev(d["hist_bar"]), general=general, accumulate=True, out=out)
    ref = oracle.vjp_rbi_sop(w, d["is_"], d["vs"], d["hist_bar"], general=general)
    assert nrel(out.cpu().numpy().reshape(n, 2).astype(np.float64) - prior, ref) <= 1e-4
    e = torch.zeros(0, dtype=torch.int64, device="cuda")
    assert B.vjp_rbi_sumofprod(w, e, torch.zeros(0, device="cuda"), dev(d["hist_bar"]), general=general).numel() == 0
    h = B.rbi_sumofprod_forward(3, e, torch.zeros(0, device="cuda")).cpu().numpy()
    assert h.shape == (3, 2) and not h.any()                                  # neutral (0, 0)


@pytest.mark.parametrize("w,dist", [(1 << 10, "uniform"), (1 << 10, "zipf"), (1 << 16, "uniform")])
def test_f1_sumofprod_full_size(w, dist):
    d = W.f1_rbi_sumofprod(w=w, dist=dist)
    is_, vs, hb = dev(d["is_"]), dev(d["vs"]), dev(d["hist_bar"])
    ref = oracle.vjp_rbi_sop(w, d["is_"], d["vs"], d["hist_bar"])
    for general in (0, 1, 2):
        got = B.vjp_rbi_sumofprod(w, is_, vs, hb, general=general).cpu().numpy()
        assert np.array_equal(got[:, 0].astype(np.float64), ref[:, 0])
        assert nrel(got[:, 1], ref[:, 1]) <= 1e-4
    hist = B.rbi_sumofprod_forward(w, is_, vs).cpu().numpy()
    href = oracle.rbi_sop_forward(w, d["is_"], d["vs"])
    assert nrel(hist[:, 0], href[:, 0]) <= 1e-4 and nrel(hist[:, 1], href[:, 1]) <= 1e-4
