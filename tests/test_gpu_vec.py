"""GPU parity of the vectorised-operator rules (NEXT row f3; sections 3.2.4 / 4.2.5, eq. 3) against the oracle."""
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


@pytest.mark.parametrize("n,w", [(1, 1), (5, 3), (4097, 7), (50021, 1024), (100003, 20000)])
@pytest.mark.parametrize("d", [1, 3, 8])
@pytest.mark.parametrize("opname", ["add", "min", "max", "mul"])
def test_rbi_vec_vjp_matches_oracle(opname, d, n, w):
    data = W.f3_rbi_vec(opname, n=n, d=d, w=w, zero_rate=min(0.3, 0.7 * w / n))
    got = B.vjp_reduce_by_index_vec(B.Op.of(opname), w, dev(data["is_"]), dev(data["vss"]), dev(data["hist_bar"])).cpu().numpy()
    ref = oracle.vjp_rbi_vec(opname, w, data["is_"], data["vss"], data["hist_bar"])
    if opname == "mul":
        assert nrel(got, ref) <= 1e-4
    else:
        assert np.array_equal(got.astype(np.float64), ref)       # copies


def test_rbi_vec_satadd_and_accumulate():
    n, d, w = 30011, 3, 50
    data = W.f3_rbi_vec("satadd", n=n, d=d, w=w)
    ok = (data["is_"] >= 0) & (data["is_"] < w)
    S = 0.37 + 0.5 * n / w / 2
    for c in range(d):   # keep every bin total of every column off the kink (Q17)
        tot = np.bincount(data["is_"][ok], weights=data["vss"][ok, c].astype(np.float64), minlength=w)
        while np.any(np.abs(tot - S) < 2.0 ** -6):
            S += 2.0 ** -5
    S = float(np.float32(S))
    prior = np.random.default_rng(2).standard_normal((n, d)).astype(np.float32)
    out = dev(prior).view(-1)
    B.vjp_reduce_by_index_vec(B.Op.of("satadd", S=S, accumulate=True), w, dev(data["is_"]), dev(data["vss"]),
                              dev(data["hist_bar"]), out=out)
    ref = oracle.vjp_rbi_vec("satadd", w, data["is_"], data["vss"], data["hist_bar"], S=S)
    assert np.array_equal(out.cpu().numpy().reshape(n, d), (prior.astype(np.float64) + ref).astype(np.float32))


@pytest.mark.parametrize("n", [1, 777, 16385, 100003])
@pytest.mark.parametrize("d", [2, 5])
@pytest.mark.parametrize("opname", ["add", "mul", "min"])
def test_scan_vec_vjp_matches_oracle(opname, d, n):
    rng = np.random.default_rng([n, d])
    xss = (1.0 + 2e-3 * rng.standard_normal((n, d))).astype(np.float32) if opname == "mul" else np.round(rng.standard_normal((n, d)), 1).astype(np.float32)
    yb = rng.standard_normal((n, d)).astype(np.float32)
    got = B.vjp_scan_vec(B.Op.of(opname), dev(xss), dev(yb)).cpu().numpy()
    ref = oracle.vjp_scan_vec(opname, xss, yb)
    assert nrel(got, ref) <= 1e-4
    if opname == "min":
        assert np.array_equal(got != 0, ref != 0)


def test_vec_rejects_bad_arguments():
    is_ = torch.zeros(4, dtype=torch.int64, device="cuda")
    v = torch.ones(4, 2, device="cuda")
    hb = torch.ones(3, 2, device="cuda")
    with pytest.raises(B.VjpError):
        B.vjp_reduce_by_index_vec(B.Op.of("linrec"), 3, is_, v, hb)
    with pytest.raises(B.VjpError):
        B.vjp_scan_vec(B.Op.of("matmul2"), v, v)
    with pytest.raises(B.VjpError):
        B.vjp_reduce_by_index_vec(B.Op.of("mul"), 3, is_, torch.ones(4, 3, device="cuda"), hb)   # d mismatch


@pytest.mark.parametrize("opname", ["mul", "min"])
def test_f3_rbi_vec_full_size(opname):
    data = W.f3_rbi_vec(opname)      # n = 2^22 rows of d = 4: 2^24 scalars
    got = B.vjp_reduce_by_index_vec(B.Op.of(opname), data["w"], dev(data["is_"]), dev(data["vss"]), dev(data["hist_bar"])).cpu().numpy()
    ref = oracle.vjp_rbi_vec(opname, data["w"], data["is_"], data["vss"], data["hist_bar"])
    if opname == "mul":
        assert nrel(got, ref) <= 1e-4
    else:
        assert np.array_equal(got.astype(np.float64), ref)


# `map2 (*)` with d a power of two and 1024 < w * d <= 12288 runs FUSED: one scalar '*' problem on the flat [n * d] array
# with virtual keys (bin, column) -- no transposes (csrc: ms_hist_kernel<VEC>, rbi_mul_sweep_kernel<VEC>).  The shapes
# below sit on both sides of every condition (d = 6: not a power of two; w * d = 1024 and 12292: outside the range).
@pytest.mark.parametrize("n,d,w", [(1, 2, 600), (33, 4, 300), (50021, 4, 1024), (100003, 2, 513), (65537, 8, 1536),
                                   (40001, 16, 768), (70001, 4, 3072), (30011, 4, 256), (30011, 4, 3073), (30011, 6, 500)])
def test_rbi_vec_mul_fused_matches_oracle(n, d, w):
    data = W.f3_rbi_vec("mul", n=n, d=d, w=w, zero_rate=min(0.3, 0.7 * w / n))
    is_ = data["is_"].copy()
    is_[::41] = w + 5                       # out of range on the high side: the virtual key must not alias bin 0 ... d
    is_[::43] = -1
    ref = oracle.vjp_rbi_vec("mul", w, is_, data["vss"], data["hist_bar"])
    got = B.vjp_reduce_by_index_vec(B.Op.of("mul"), w, dev(is_), dev(data["vss"]), dev(data["hist_bar"])).cpu().numpy()
    assert nrel(got, ref) <= 1e-4
    oob = (is_ < 0) | (is_ >= w)
    assert not got.reshape(n, d)[oob].any()
    # the three branches of Fig. 3 per (bin, column): compare per column against the scalar entry point as well
    for c in (0, d - 1):
        col = B.vjp_reduce_by_index(B.Op.of("mul"), w, dev(is_), dev(data["vss"][:, c]), dev(data["hist_bar"][:, c]))
        assert nrel(got.reshape(n, d)[:, c], col.cpu().numpy()) <= 1e-4
    # accumulate: out += contribution
    prior = np.random.default_rng(n).standard_normal((n, d)).astype(np.float32)
    out = dev(prior).view(-1)
    B.vjp_reduce_by_index_vec(B.Op.of("mul", accumulate=True), w, dev(is_), dev(data["vss"]), dev(data["hist_bar"]), out=out)
    assert nrel(out.cpu().numpy().reshape(n, d).astype(np.float64) - prior, ref) <= 1e-4


# Non-redundant block-diagonal sparsity: an operator that applies linrec / a q x q product to each of the
# d blocks of its element = d scans with the scaled-down operator (vjp_scan_vec with an operator of arity > 1).
@pytest.mark.parametrize("n", [1, 129, 4097, 30011])
@pytest.mark.parametrize("opname,q,d", [("linrec", 0, 3), ("matmul2", 2, 2), ("matmul3", 3, 2), ("matmul5", 5, 2), ("linrec", 0, 1)])
def test_scan_bds_vjp_matches_oracle(opname, q, d, n):
    rng = np.random.default_rng([n, d, q])
    a = 2 if opname == "linrec" else q * q
    if opname == "linrec":
        blocks = [np.stack([rng.uniform(0.9, 1.0, n), rng.standard_normal(n)], axis=1) for _ in range(d)]
    else:
        blocks = [W.c4_scan_matmul(q, n=n, seed=7 + c)["xs"].reshape(n, a) for c in range(d)]
    xss = np.concatenate(blocks, axis=1).astype(np.float32)
    ybar = rng.standard_normal((n, d * a)).astype(np.float32)
    got = B.vjp_scan_vec(B.Op.of(opname), dev(xss), dev(ybar)).cpu().numpy()
    ref = oracle.vjp_scan_vec("linrec" if opname == "linrec" else "matmul", xss, ybar, q=q)
    assert got.shape == (n, d * a) and nrel(got, ref) <= 1e-4
    for c in range(d):    # every block column equals the small operator's own VJP on that column
        one = B.vjp_scan(B.Op.of(opname), dev(np.ascontiguousarray(xss[:, c * a:(c + 1) * a])),
                         dev(np.ascontiguousarray(ybar[:, c * a:(c + 1) * a]))).cpu().numpy().reshape(n, a)
        assert nrel(got[:, c * a:(c + 1) * a], one) <= 1e-5
    prior = rng.standard_normal((n, d * a)).astype(np.float32)
    out = dev(prior).view(-1)
    B.vjp_scan_vec(B.Op.of(opname, accumulate=True), dev(xss), dev(ybar), out=out)
    assert nrel(out.cpu().numpy().reshape(n, d * a).astype(np.float64) - prior, ref) <= 1e-4
