"""GPU parity of the SORT-FREE route of the general reduce-by-index rule (eq. 5; csrc/rbi_multiscan.cu)
against the f64 CPU oracle of eq. 5, on the cases that route has of its own: chunk boundaries, rows whose lanes share
bins (the match.any path) and rows whose lanes do not (the claim path), ties of min / max across chunks (the lowest
index must win), keys out of range, the hand-over to the sort-based route above w = 12 288, accumulate.
Integer-valued results (copies of hist_bar or 0) are compared bit-exactly, products normwise at 1e-4."""
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


def run(opname, w, is_, vs, hb, route, S=0.0):
    return B.vjp_reduce_by_index(B.Op.of(opname, S=S, force_general=route), w, dev(is_), dev(vs), dev(hb))


# n: below one row, one ragged row, a few rows (fewer chunks than warps), many chunks with a ragged tail
@pytest.mark.parametrize("n", [1, 31, 33, 1000, 8 * 32 * 3 + 5, 300007])
@pytest.mark.parametrize("w", [1, 2, 13, 1024, 4096])
@pytest.mark.parametrize("opname", ["min", "max"])
def test_ties_of_min_max_go_to_the_lowest_index_across_rows_and_chunks(opname, w, n):
    rng = np.random.default_rng([n, w, 7])
    is_ = rng.integers(-1, w + 1, size=n, dtype=np.int64)          # both out-of-range sides occur
    vs = rng.integers(0, 3, size=n).astype(np.float32)             # three distinct values: ties everywhere
    hb = rng.standard_normal(w).astype(np.float32)
    ref = oracle.vjp_rbi_general(opname, w, is_, vs, hb)
    for route in (1, 2):
        got = run(opname, w, is_, vs, hb, route).cpu().numpy()
        assert np.array_equal(got.astype(np.float64), ref), "route %d" % route
    # exactly one element per non-empty bin takes the adjoint, and it is the first extremum of the bin
    inr = (is_ >= 0) & (is_ < w)
    got = run(opname, w, is_, vs, hb, 1).cpu().numpy()
    for k in np.unique(is_[inr])[:50]:
        idx = np.flatnonzero(is_ == k)
        ext = vs[idx].min() if opname == "min" else vs[idx].max()
        first = idx[np.flatnonzero(vs[idx] == ext)[0]]
        want = np.zeros(idx.size, dtype=np.float32)
        want[np.searchsorted(idx, first)] = hb[k]
        assert np.array_equal(got[idx], want)


@pytest.mark.parametrize("dist", ["uniform", "zipf", "one_bin", "runs"])
@pytest.mark.parametrize("opname", ["add", "mul", "satadd"])
def test_key_distributions(opname, dist):
    n, w = 200003, 4096
    rng = np.random.default_rng([11, {"uniform": 0, "zipf": 1, "one_bin": 2, "runs": 3}[dist]])
    if dist == "uniform":
        is_ = rng.integers(0, w, size=n, dtype=np.int64)
    elif dist == "zipf":
        is_ = W.c2_rbi_min(n=n, w=w, dist="zipf")["is_"]
    elif dist == "one_bin":
        is_ = np.full(n, 77, dtype=np.int64)                       # every row takes the match.any path, 32 lanes deep
    else:
        is_ = np.repeat(rng.integers(0, w, size=n // 5 + 1, dtype=np.int64), 5)[:n]   # runs of 5 equal keys
    is_[::97] = -3
    hb = rng.standard_normal(w).astype(np.float32)
    if opname == "mul":
        vs = rng.uniform(0.99, 1.01, n).astype(np.float32)
        vs[rng.random(n) < 1e-4] = 0.0
    else:
        vs = rng.random(n, dtype=np.float32)
    S = 0.0
    if opname == "satadd":                                         # keep every bin total away from the kink (Q17)
        tot = np.bincount(is_[is_ >= 0], weights=vs[is_ >= 0].astype(np.float64), minlength=w)
        S = float(np.float32(np.median(tot[tot > 0]) * 1.001 + 0.37))
        while np.any(np.abs(tot - S) < 2.0 ** -4 + 2e-4 * S):      # f32 sums of a bin's ~S / 0.5 values
            S = float(np.float32(S * 1.0005 + 2.0 ** -3))
    ref = oracle.vjp_rbi_general(opname, w, is_, vs, hb, S=S)
    for route in (1, 2):
        got = run(opname, w, is_, vs, hb, route, S=S).cpu().numpy()
        if opname == "mul":
            assert nrel(got, ref) <= 1e-4
        else:
            assert np.array_equal(got.astype(np.float64), ref)
        assert not got[is_ < 0].any()


def test_all_keys_out_of_range_and_empty_bins():
    n, w = 70001, 300
    rng = np.random.default_rng(3)
    vs, hb = rng.random(n, dtype=np.float32), rng.standard_normal(w).astype(np.float32)
    is_ = np.where(rng.random(n) < 0.5, -1 - rng.integers(0, 5, n), w + rng.integers(0, 5, n)).astype(np.int64)
    for opname in ("add", "min", "mul", "satadd"):
        assert not run(opname, w, is_, vs, hb, 1, S=5.0).cpu().numpy().any()
    is_ = np.full(n, 5, dtype=np.int64)                            # one bin in use, all others empty
    got = run("add", w, is_, vs, hb, 1).cpu().numpy()
    assert np.array_equal(got, np.full(n, hb[5], dtype=np.float32))


@pytest.mark.parametrize("w", [4097, 8192, 12288, 12289, 20000])   # 6, 3 warps per SM; then the sort-based route
def test_handover_to_the_sort_based_route_above_12288_bins(w):
    n = 150001
    d = W.c2_rbi_min(n=n, w=w)
    ref = oracle.vjp_rbi_general("min", w, d["is_"], d["vs"], d["hist_bar"])
    for route in (1, 2):
        got = run("min", w, d["is_"], d["vs"], d["hist_bar"], route).cpu().numpy()
        assert np.array_equal(got.astype(np.float64), ref)


def test_accumulate_and_workspace_query():
    n, w = 90001, 777
    d = W.c5_rbi_satadd(n=n, w=w)
    ref = oracle.vjp_rbi_general("satadd", w, d["is_"], d["vs"], d["hist_bar"], S=d["S"])
    prior = np.random.default_rng(5).standard_normal(n).astype(np.float32)
    out = dev(prior)
    op = B.Op.of("satadd", S=d["S"], accumulate=True)
    B.vjp_reduce_by_index(op, w, dev(d["is_"]), dev(d["vs"]), dev(d["hist_bar"]), out=out)
    assert np.array_equal(out.cpu().numpy(), prior + ref.astype(np.float32))
    # one workspace query serves both routes; a workspace one byte short is refused, nothing is launched
    need = B.vjp_reduce_by_index_workspace_bytes(B.Op.of("satadd", S=d["S"]), n, w)
    assert need == B.vjp_reduce_by_index_workspace_bytes(B.Op.of("satadd", S=d["S"], force_general=2), n, w)
    small = torch.empty(need - 1, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.VjpError):
        B.vjp_reduce_by_index(B.Op.of("satadd", S=d["S"]), w, dev(d["is_"]), dev(d["vs"]), dev(d["hist_bar"]), ws=small)


def test_full_size_c5_routes_agree_bit_for_bit():
    d = W.c5_rbi_satadd()
    w = d["w"]
    is_, vs, hb = dev(d["is_"]), dev(d["vs"]), dev(d["hist_bar"])
    a = B.vjp_reduce_by_index(B.Op.of("satadd", S=d["S"], force_general=1), w, is_, vs, hb)
    b = B.vjp_reduce_by_index(B.Op.of("satadd", S=d["S"], force_general=2), w, is_, vs, hb)
    assert torch.equal(a, b)


def test_routes_agree_on_random_shapes():
    """Differential check of the two routes of eq. 5 on 40 random (n, w, operator, key distribution) draws: the
    sort-free walks must reproduce the sort-based route bit for bit wherever the result is a copy of hist_bar or 0,
    and within rounding for '*' (chunk boundaries, ragged rows and the warps-per-CTA choice all move with n and w)."""
    rng = np.random.default_rng(20231003)
    for trial in range(40):
        n = int(rng.integers(1, 1 << int(rng.integers(1, 20))))
        w = int(rng.integers(1, 1 << int(rng.integers(1, 14))))   # up to 8191: both sides of 4096, below 12 288
        opname = ["add", "min", "max", "mul", "satadd"][trial % 5]
        hot = rng.random() < 0.5
        is_ = (rng.zipf(1.3, n) % (w + 2) - 1 if hot else rng.integers(-1, w + 1, n)).astype(np.int64)
        vs = (rng.integers(0, 4, n).astype(np.float32) if opname in ("min", "max")
              else rng.uniform(0.99, 1.01, n).astype(np.float32) if opname == "mul"    # products of a bin stay in range
              else rng.uniform(0.5, 1.5, n).astype(np.float32))
        hb = rng.standard_normal(w).astype(np.float32)
        S = 0.0
        if opname == "satadd":
            inr = (is_ >= 0) & (is_ < w)
            tot = np.bincount(is_[inr], weights=vs[inr].astype(np.float64), minlength=w)
            S = float(np.float32(np.median(tot) + 0.31))
            while np.any(np.abs(tot - S) < 2.0 ** -4 + 2e-4 * S):
                S = float(np.float32(S * 1.0005 + 2.0 ** -3))
        a = run(opname, w, is_, vs, hb, 1, S=S).cpu().numpy()
        b = run(opname, w, is_, vs, hb, 2, S=S).cpu().numpy()
        if opname == "mul":
            assert nrel(a, b) <= 1e-4, (trial, n, w)
        else:
            assert np.array_equal(a, b), (trial, opname, n, w, hot)
