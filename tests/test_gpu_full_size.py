"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: the C oracle
is fast enough to produce every output of every configuration, so the comparison is element by
element here too (no sampling).  Same bars as test_gpu_parity.py."""
import numpy as np
import pytest
import torch

import oracle
from paper_2310_03568_b200 import binding as B
from paper_2310_03568_b200 import workloads as W

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def nrel(got, ref):
    got = np.asarray(got, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    assert got.shape == ref.shape and np.all(np.isfinite(got))
    den, err = np.max(np.abs(ref)), np.max(np.abs(got - ref))
    return (0.0 if err == 0.0 else np.inf) if den == 0.0 else err / den


def test_c1_rbi_add_full():
    d = W.c1_rbi_add()
    got = B.vjp_reduce_by_index(B.Op.of("add"), d["w"], dev(d["is_"]), None, dev(d["hist_bar"])).cpu().numpy()
    assert np.array_equal(got.astype(np.float64), oracle.vjp_rbi_add(d["w"], d["is_"], d["hist_bar"]))


@pytest.mark.parametrize("dist", ["uniform", "zipf"])
@pytest.mark.parametrize("w", [1 << 10, 1 << 16])
def test_c2_rbi_min_full(w, dist):
    d = W.c2_rbi_min(w=w, dist=dist)
    op = B.Op.of("min")
    got = B.vjp_reduce_by_index(op, w, dev(d["is_"]), dev(d["vs"]), dev(d["hist_bar"])).cpu().numpy()
    ref, rarg, rext = oracle.vjp_rbi_minmax("min", w, d["is_"], d["vs"], d["hist_bar"])
    arg, ext = B.rbi_argext(op, w, dev(d["is_"]), dev(d["vs"]))
    assert np.array_equal(arg.cpu().numpy(), rarg)                      # indices bit-exact, ties -> lowest
    assert np.array_equal(ext.cpu().numpy().astype(np.float64), rext)
    assert np.array_equal(got.astype(np.float64), ref)                  # a pure copy: bit-exact
    hist = B.reduce_by_index_forward(op, w, dev(d["is_"]), dev(d["vs"])).cpu().numpy()
    assert np.array_equal(hist.astype(np.float64), rext)


@pytest.mark.parametrize("dist", ["uniform", "zipf"])
@pytest.mark.parametrize("w", [1 << 10, 1 << 16])
def test_c2_rbi_mul_full(w, dist):
    d = W.c2_rbi_mul(w=w, dist=dist)
    op = B.Op.of("mul")
    got = B.vjp_reduce_by_index(op, w, dev(d["is_"]), dev(d["vs"]), dev(d["hist_bar"])).cpu().numpy()
    ref, rz, rp = oracle.vjp_rbi_mul(w, d["is_"], d["vs"], d["hist_bar"])
    z, p = B.rbi_zero_prod(op, w, dev(d["is_"]), dev(d["vs"]))
    assert np.array_equal(z.cpu().numpy(), rz)                          # zero counts bit-exact
    assert nrel(got, ref) <= 1e-4
    # bins whose product neither under- nor overflows f32: relative error per bin
    p = p.cpu().numpy().astype(np.float64)
    ok = (np.abs(rp) > 1e-30) & (np.abs(rp) < 1e30)
    assert np.max(np.abs(p[ok] - rp[ok]) / np.abs(rp[ok]), initial=0.0) <= 1e-4


def test_c3_scan_add_full():
    d = W.c3_scan_add()
    got = B.vjp_scan(B.Op.of("add"), None, dev(d["ys_bar"])).cpu().numpy()
    assert nrel(got, oracle.vjp_scan("add", d["xs"], d["ys_bar"])) <= 1e-4


def test_c3_scan_mul_f64_full():
    d = W.c3_scan_mul()
    got = B.vjp_scan(B.Op.of("mul", torch.float64), dev(d["xs"]), dev(d["ys_bar"])).cpu().numpy()
    assert nrel(got, oracle.vjp_scan("mul", d["xs"], d["ys_bar"])) <= 1e-10


def test_c3_scan_linrec_full():
    d = W.c3_scan_linrec()
    got = B.vjp_scan(B.Op.of("linrec"), dev(d["xs"]), dev(d["ys_bar"])).cpu().numpy()
    assert nrel(got, oracle.vjp_scan("linrec", d["xs"], d["ys_bar"])) <= 1e-4


@pytest.mark.parametrize("q", [2, 3, 5])
def test_c4_scan_matmul_full(q):
    # q = 3 is not a BASELINE config (NEXT row f4): run at the 5x5 size, n = 2^22
    d = W.c4_scan_matmul(q, n=(1 << 22) if q == 3 else None)
    got = B.vjp_scan(B.Op.of("matmul%d" % q), dev(d["xs"]), dev(d["ys_bar"])).cpu().numpy()
    ref = oracle.vjp_scan("matmul", d["xs"], d["ys_bar"], q=q)
    e = nrel(got, ref)
    print("matmul %dx%d full size: normwise error %.3e" % (q, q, e))
    assert e <= 1e-4


def test_c5_rbi_satadd_full():
    d = W.c5_rbi_satadd()
    w = d["w"]
    ref = oracle.vjp_rbi_general("satadd", w, d["is_"], d["vs"], d["hist_bar"], S=d["S"])
    for route in (0, 2):  # the library's choice (sort-free walks at w = 4096) and Fig. 4 as written
        got = B.vjp_reduce_by_index(B.Op.of("satadd", S=d["S"], force_general=route), w, dev(d["is_"]), dev(d["vs"]),
                                    dev(d["hist_bar"]))
        assert np.array_equal(got.cpu().numpy().astype(np.float64), ref)
    sk, perm = B.rbi_sort_perm(w, dev(d["is_"]))
    rsk, rperm = oracle.rbi_sort_perm(w, d["is_"])
    assert np.array_equal(sk.cpu().numpy(), rsk) and np.array_equal(perm.cpu().numpy(), rperm)


@pytest.mark.parametrize("opname", ["min", "max"])
def test_f4_scan_minmax_full(opname):
    """NEXT row f4: scan with min / max at n = 2^26: the adjoint of a record-setting element is the sum of the
    ys_bar of the run it dominates; all other adjoints are exactly 0."""
    d = W.c3_scan_add()
    xs = np.round(d["xs"], 2)
    got = B.vjp_scan(B.Op.of(opname), dev(xs), dev(d["ys_bar"])).cpu().numpy()
    ref = oracle.vjp_scan(opname, xs, d["ys_bar"])
    assert np.array_equal(got != 0, ref != 0)
    assert nrel(got, ref) <= 1e-4
