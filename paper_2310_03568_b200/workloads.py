"""Seeded synthetic inputs shaped like the paper's workloads ("randomly generated arrays").

This module serves BOTH the CUDA path and the CPU oracle (tests, bench.py) and holds none of
the method's arithmetic: it only draws numbers.  Every stream comes from
``numpy.random.default_rng([seed, config_id, field_id])`` (PCG64).  The recipes are the five
configurations of BASELINE.json (they stand in for the paper's D1/D2/D_{i,j} datasets)
and are restated in DESIGN.md.  Sizes are parameters so that the parity tests can run the same
distributions at sizes the oracle finishes in seconds.
"""
from __future__ import annotations

import numpy as np

FULL = {
    "c1": dict(n=1 << 20, w=1024),
    "c2": dict(n=1 << 24, ws=(1 << 10, 1 << 16)),
    "c3": dict(n=1 << 26),
    "c4": dict(n2=1 << 24, n5=1 << 22),
    "c5": dict(n=1 << 24, w=4096, S=2048.0),
}


def _rng(seed, config_id, field_id):
    return np.random.default_rng([int(seed), int(config_id), int(field_id)])


def _normal_f32(rng, shape):
    return rng.standard_normal(shape, dtype=np.float32)


def zipf_keys(rng, n, w, s=1.1):
    """Truncated Zipf(s) over ranks 1..w by inverse CDF; bin = rank-1 (hot bins adjacent)."""
    p = np.arange(1, w + 1, dtype=np.float64) ** (-s)
    cdf = np.cumsum(p)
    cdf /= cdf[-1]
    u = rng.random(n)
    k = np.searchsorted(cdf, u, side="left")
    return np.minimum(k, w - 1).astype(np.int64)


def c1_rbi_add(n=FULL["c1"]["n"], w=FULL["c1"]["w"], seed=0):
    """Config 1: reduce-by-index '+', keys uniform in [-16, w+16) so ~3 % fall outside [0,w)."""
    return dict(
        n=n, w=w,
        vs=_normal_f32(_rng(seed, 1, 0), n),
        is_=_rng(seed, 1, 1).integers(-16, w + 16, size=n, dtype=np.int64),
        hist_bar=_normal_f32(_rng(seed, 1, 2), w),
    )


def _keys(dist, rng, n, w):
    if dist == "uniform":
        return rng.integers(0, w, size=n, dtype=np.int64)
    if dist == "zipf":
        return zipf_keys(rng, n, w, 1.1)
    raise ValueError(dist)


def c2_rbi_min(n=FULL["c2"]["n"], w=1 << 10, dist="uniform", seed=0):
    """Config 2, min: N(0,1) values; 1 % of the positions become copies of another element of
    the SAME bin (ties anywhere in the bin), and every fourth bin gets the same 'floor' value
    planted on up to three of its members so that the bin minimum itself is tied (lowest index
    must win).  No minimum is computed here -- the floor lies below every N(0,1) draw."""
    cell = {"uniform": 0, "zipf": 1}[dist] + 2 * int(np.log2(w))
    is_ = _keys(dist, _rng(seed, 2, 10 + cell), n, w)
    vs = _normal_f32(_rng(seed, 2, 40 + cell), n)
    rng = _rng(seed, 2, 70 + cell)
    if n >= 2:
        order = np.argsort(is_, kind="stable")
        sk = is_[order]
        same = np.flatnonzero(sk[1:] == sk[:-1]) + 1          # sorted positions with a same-bin left neighbour
        if same.size:
            pick = same[rng.random(same.size) < 0.01]
            vs[order[pick]] = vs[order[pick - 1]]
            # floor values: first, middle and last member of every fourth multi-member bin
            starts = np.flatnonzero(np.r_[True, sk[1:] != sk[:-1]])
            ends = np.r_[starts[1:], sk.size]
            multi = (ends - starts) >= 2
            chosen = multi & (sk[starts] % 4 == 1)
            s, e = starts[chosen], ends[chosen]
            floor = (-8.0 - (sk[s] % 7) * 0.25).astype(np.float32)
            for pos in (s, (s + e) // 2, e - 1):
                vs[order[pos]] = floor
    return dict(n=n, w=w, is_=is_, vs=vs, hist_bar=_normal_f32(_rng(seed, 2, 100 + cell), w))


def c2_rbi_mul(n=FULL["c2"]["n"], w=1 << 10, dist="uniform", seed=0, zero_rate=1e-3):
    """Config 2, '*': U[0.9,1.1] values with exact zeros at rate zero_rate."""
    cell = {"uniform": 0, "zipf": 1}[dist] + 2 * int(np.log2(w))
    is_ = _keys(dist, _rng(seed, 2, 130 + cell), n, w)
    rng = _rng(seed, 2, 160 + cell)
    vs = (0.9 + 0.2 * rng.random(n)).astype(np.float32)
    vs[rng.random(n) < zero_rate] = 0.0
    return dict(n=n, w=w, is_=is_, vs=vs, hist_bar=_normal_f32(_rng(seed, 2, 190 + cell), w))


def c3_scan_add(n=FULL["c3"]["n"], seed=0, dtype=np.float32):
    xs = _rng(seed, 3, 0).standard_normal(n, dtype=dtype)
    ys_bar = _rng(seed, 3, 1).standard_normal(n, dtype=dtype)
    return dict(n=n, xs=xs, ys_bar=ys_bar)


def c3_scan_mul(n=FULL["c3"]["n"], seed=0, dtype=np.float64, zero_rate=1e-4, lo=0.99, hi=1.01):
    rng = _rng(seed, 3, 2)
    xs = (lo + (hi - lo) * rng.random(n)).astype(dtype)
    if zero_rate > 0:
        xs[rng.random(n) < zero_rate] = 0.0
    ys_bar = _rng(seed, 3, 3).standard_normal(n).astype(dtype)
    return dict(n=n, xs=xs, ys_bar=ys_bar)


def c3_scan_linrec(n=FULL["c3"]["n"], seed=0, dtype=np.float32):
    rng = _rng(seed, 3, 4)
    xs = np.empty((n, 2), dtype=dtype)
    xs[:, 0] = (0.9 + 0.1 * rng.random(n)).astype(dtype)
    xs[:, 1] = rng.standard_normal(n).astype(dtype)
    ys_bar = _rng(seed, 3, 5).standard_normal((n, 2)).astype(dtype)
    return dict(n=n, xs=xs, ys_bar=ys_bar)


def random_orthogonal(rng, n, q, chunk=1 << 20):
    """n random orthogonal q-by-q matrices: Q of the QR factorisation of an N(0,1) matrix with the
    signs fixed so that diag(R) > 0 -- which is what Gram-Schmidt on the columns yields directly.
    Computed in f64, returned f32 [n, q*q] row-major."""
    out = np.empty((n, q * q), dtype=np.float32)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        m = rng.standard_normal((b - a, q, q))
        for j in range(q):
            v = m[:, :, j]
            for i in range(j):
                u = m[:, :, i]
                v -= np.sum(u * v, axis=1, keepdims=True) * u
            for i in range(j):  # second orthogonalisation pass (numerical hygiene)
                u = m[:, :, i]
                v -= np.sum(u * v, axis=1, keepdims=True) * u
            v /= np.linalg.norm(v, axis=1, keepdims=True)
        out[a:b] = m.reshape(b - a, q * q)
    return out


def c4_scan_matmul(q, n=None, seed=0):
    if n is None:
        n = FULL["c4"]["n2"] if q == 2 else FULL["c4"]["n5"]
    xs = random_orthogonal(_rng(seed, 4, 10 * q), n, q)
    ys_bar = _normal_f32(_rng(seed, 4, 10 * q + 1), (n, q * q))
    return dict(n=n, q=q, xs=xs, ys_bar=ys_bar)


def c5_rbi_satadd(n=FULL["c5"]["n"], w=FULL["c5"]["w"], S=None, seed=0, margin=2.0 ** -6):
    """Config 5: saturated add min(a+b,S), U[0,1) values, uniform keys; S defaults to n/(2w) (the
    mean bin total, 2048 at full size) so that about half of the bins saturate.  A bin whose total
    lies within `margin` of S would make the (discontinuous) derivative depend on f32 rounding, so
    one member of such a bin is nudged by 4*margin (reading Q17); the totals are only
    looked at to keep the input away from the kink."""
    if S is None:
        S = n / (2.0 * w)
    is_ = _rng(seed, 5, 0).integers(0, w, size=n, dtype=np.int64)
    vs = _rng(seed, 5, 1).random(n, dtype=np.float32)
    for _ in range(4):
        tot = np.bincount(is_, weights=vs.astype(np.float64), minlength=w)
        bad = np.flatnonzero(np.abs(tot - S) < margin)
        if bad.size == 0:
            break
        first = np.full(w, -1, dtype=np.int64)
        idx = np.flatnonzero(np.isin(is_, bad))
        first[is_[idx[::-1]]] = idx[::-1]
        for k in bad:
            i = first[k]
            vs[i] = np.float32(vs[i] + 4 * margin) if vs[i] < 0.5 else np.float32(vs[i] - 4 * margin)
    return dict(n=n, w=w, S=float(S), is_=is_, vs=vs, hist_bar=_normal_f32(_rng(seed, 5, 2), w))


def f2_reduce(op, n=1 << 24, seed=0):
    """NEXT row f2 (reduce VJP, section 3): one array per operator, shaped like config 2's values.  '+', min, max:
    N(0,1) with 1 % duplicated values (ties); '*': U[1-2e-3, 1+2e-3] (the product of 2^24 of them stays inside f32)
    with exact zeros at rate `1/n` scale chosen by the caller; satadd: U[0,1) with S = n/2 +- a margin."""
    rng = _rng(seed, 6, {"add": 0, "min": 1, "max": 2, "mul": 3, "satadd": 4}[op])
    if op == "mul":
        xs = (1.0 + 2e-3 * (2.0 * rng.random(n) - 1.0)).astype(np.float32)
    elif op == "satadd":
        xs = rng.random(n, dtype=np.float32)
    else:
        xs = _normal_f32(rng, n)
        if n >= 2 and op in ("min", "max"):
            dup = rng.random(n) < 0.01
            dup[0] = False
            idx = np.flatnonzero(dup)
            xs[idx] = xs[idx - 1]
            ext = np.float32(-9.0 if op == "min" else 9.0)       # the extremum itself is tied (lowest index must win)
            for pos in (n // 3, n // 2, n - 1):
                xs[pos] = ext
    y_bar = np.asarray(_rng(seed, 6, 9).standard_normal(1), dtype=np.float32)
    return dict(n=n, xs=xs, y_bar=y_bar)


def f1_rbi_sumofprod(n=1 << 24, w=1 << 10, dist="uniform", seed=0):
    """NEXT row f1 (invertible operator sumOfProd, sections 3.3 / 4.2.4): pairs (p, s) ~ N(0,1)^2 as [n, 2] f32, keys as
    in config 2 (uniform or Zipf(1.1)) with 3 % out of range on both sides, bin adjoints (Pbar, Sbar) ~ N(0,1)^2."""
    cell = {"uniform": 0, "zipf": 1}[dist] + 2 * int(np.log2(w))
    is_ = _keys(dist, _rng(seed, 7, 10 + cell), n, w)
    oob = _rng(seed, 7, 40 + cell).random(n) < 0.03
    is_[oob] = np.where(np.arange(n)[oob] % 2 == 0, -1 - (is_[oob] % 5), w + (is_[oob] % 7))
    vs = _normal_f32(_rng(seed, 7, 70 + cell), (n, 2))
    return dict(n=n, w=w, is_=is_, vs=vs, hist_bar=_normal_f32(_rng(seed, 7, 100 + cell), (w, 2)))


def f3_rbi_vec(op, n=1 << 22, d=4, w=1 << 10, seed=0, zero_rate=1e-3):
    """NEXT row f3 (vectorised operators map2 (.), sections 3.2.4 / 4.2.5): rows of d scalars, uniform keys with 3 % out of
    range, values per column as in config 2 ('*': U[0.9,1.1] with exact zeros; min/max/+: N(0,1) rounded to 2 decimals for
    ties; satadd: U[0,1))."""
    rng = _rng(seed, 8, d)
    is_ = rng.integers(-w // 64 - 1, w + w // 64 + 1, size=n, dtype=np.int64)
    if op == "mul":
        vss = (0.9 + 0.2 * rng.random((n, d))).astype(np.float32)
        vss[rng.random((n, d)) < zero_rate] = 0.0
    elif op == "satadd":
        vss = rng.random((n, d), dtype=np.float32)
    else:
        vss = np.round(_normal_f32(rng, (n, d)), 2)
    return dict(n=n, d=d, w=w, is_=is_, vss=vss, hist_bar=_normal_f32(_rng(seed, 8, 100 + d), (w, d)))
