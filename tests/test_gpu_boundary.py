"""GPU tests of the boundary (include/vjp_b200.h): accumulate ("+="), the
in-place '+' scan, argument checks (sizes, alignment), the *_host entry points against the ORACLE, and a
stress test of the decoupled look-back."""
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


# ------------------------------------------------------------------ accumulate ------------

SCAN_CASES = [("add", torch.float32, 0), ("add", torch.float64, 0), ("mul", torch.float64, 0), ("linrec", torch.float32, 0),
              ("matmul2", torch.float32, 2), ("matmul3", torch.float32, 3), ("matmul5", torch.float32, 5)]


def scan_data(name, n):
    if name == "add":
        return W.c3_scan_add(n=n)
    if name == "mul":
        return W.c3_scan_mul(n=n, zero_rate=1e-3)
    if name == "linrec":
        return W.c3_scan_linrec(n=n)
    return W.c4_scan_matmul(int(name[-1]), n=n)


@pytest.mark.parametrize("n", [1, 777, 16385, 100003])
@pytest.mark.parametrize("name,dtype,q", SCAN_CASES)
def test_scan_vjp_accumulate_adds_to_prior(name, dtype, q, n):
    d = scan_data(name, n)
    npdt = np.float64 if dtype == torch.float64 else np.float32
    xs, yb = d["xs"].astype(npdt), d["ys_bar"].astype(npdt)
    prior = np.random.default_rng([n, q]).standard_normal(xs.shape).astype(npdt)
    out = dev(prior)
    B.vjp_scan(B.Op.of(name, dtype, accumulate=True), dev(xs), dev(yb), out=out)
    oname = "matmul" if q else name
    ref = prior.astype(np.float64) + oracle.vjp_scan(oname, xs, yb, q=q)
    assert nrel(out.cpu().numpy(), ref) <= (1e-10 if dtype == torch.float64 else 1e-4)


@pytest.mark.parametrize("n,w", [(5, 3), (4097, 7), (100003, 1024), (100003, 20000), (1 << 18, 70000)])
@pytest.mark.parametrize("opname", ["add", "min", "max", "mul", "satadd"])
def test_rbi_vjp_accumulate_adds_to_prior(opname, n, w):
    rng = np.random.default_rng([n, w, 9])
    if opname == "mul":
        d = W.c2_rbi_mul(n=n, w=w, zero_rate=min(0.3, 0.7 * w / n))
    elif opname == "satadd":
        d = W.c5_rbi_satadd(n=n, w=w)
    else:
        d = W.c2_rbi_min(n=n, w=w)
    is_ = d["is_"].copy()
    is_[::61] = -2
    vs, hb = d["vs"], d["hist_bar"]
    S = float(d.get("S", 0.0))
    if opname == "satadd":  # keep the bin totals off the kink after the keys changed (Q17)
        tot = np.bincount(is_[is_ >= 0], weights=vs[is_ >= 0].astype(np.float64), minlength=w)
        while np.any(np.abs(tot - S) < 2.0 ** -6):
            S += 2.0 ** -5
        S = float(np.float32(S))
    prior = rng.standard_normal(n).astype(np.float32)
    out = dev(prior)
    B.vjp_reduce_by_index(B.Op.of(opname, S=S, accumulate=True), w, dev(is_), dev(vs), dev(hb), out=out)
    if opname == "add":
        con = oracle.vjp_rbi_add(w, is_, hb)
    elif opname in ("min", "max"):
        con = oracle.vjp_rbi_minmax(opname, w, is_, vs, hb)[0]
    elif opname == "mul":
        con = oracle.vjp_rbi_mul(w, is_, vs, hb)[0]
    else:
        con = oracle.vjp_rbi_general("satadd", w, is_, vs, hb, S=S)
    got = out.cpu().numpy()
    if opname == "mul":
        assert nrel(got.astype(np.float64) - prior, con) <= 1e-4
    else:  # the contribution is a copy or 0: prior + copy, rounded once in f32
        assert np.array_equal(got, (prior.astype(np.float64) + con).astype(np.float32))


def test_accumulate_needs_an_output_tensor():
    x = torch.ones(8, device="cuda")
    with pytest.raises(B.VjpError):
        B.vjp_scan(B.Op.of("add", accumulate=True), None, x)


# ------------------------------------------------------------------ aliasing, alignment, sizes --

@pytest.mark.parametrize("n", [5, 16384, 100003, 1 << 22])
def test_scan_add_vjp_runs_in_place(n):
    d = W.c3_scan_add(n=n)
    buf = dev(d["ys_bar"])
    B.vjp_scan(B.Op.of("add"), None, buf, out=buf)
    assert nrel(buf.cpu().numpy(), oracle.vjp_scan("add", d["xs"], d["ys_bar"])) <= 1e-4


def test_in_place_is_rejected_for_other_operators_and_for_accumulate():
    x = torch.rand(64, device="cuda")
    y = torch.rand(64, device="cuda")
    with pytest.raises(B.VjpError):
        B.vjp_scan(B.Op.of("mul"), x, y, out=y)
    with pytest.raises(B.VjpError):
        B.vjp_scan(B.Op.of("add", accumulate=True), None, y, out=y)


def test_misaligned_views_and_wrong_sizes_are_rejected_before_any_launch():
    n, w = 1000, 16
    is_ = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
    vs = torch.ones(n + 1, device="cuda")
    hb = torch.ones(w, device="cuda")
    l0 = B.launch_count()
    with pytest.raises(B.VjpError):   # vs[1:] is 4-byte aligned only
        B.vjp_reduce_by_index(B.Op.of("mul"), w, is_[:n], vs[1:], hb)
    with pytest.raises(B.VjpError):   # is[1:] is 8-byte aligned only
        B.vjp_reduce_by_index(B.Op.of("add"), w, is_[1:], None, hb)
    with pytest.raises(B.VjpError):   # hist_bar of the wrong size
        B.vjp_reduce_by_index(B.Op.of("add"), w + 1, is_[:n], None, hb)
    with pytest.raises(B.VjpError):   # vs of the wrong size
        B.vjp_reduce_by_index(B.Op.of("mul"), w, is_[:n], vs, hb)
    with pytest.raises(B.VjpError):   # out of the wrong dtype
        B.vjp_reduce_by_index(B.Op.of("add"), w, is_[:n], None, hb, out=torch.empty(n, dtype=torch.float64, device="cuda"))
    with pytest.raises(B.VjpError):
        B.vjp_scan(B.Op.of("add"), None, vs[1:])
    # the C side checks too (a caller that bypasses the Python checks): misaligned pointer -> INVALID_ARG
    import ctypes
    lib, o = B.load(), B.Op.of("add").c()
    ws = torch.empty(1 << 16, dtype=torch.uint8, device="cuda")
    out = torch.empty(n, device="cuda")
    rc = lib.vjp_reduce_by_index(ctypes.byref(o), n, w, ctypes.c_void_p(is_.data_ptr() + 8), None,
                                 ctypes.c_void_p(hb.data_ptr()), ctypes.c_void_p(out.data_ptr()),
                                 ctypes.c_void_p(ws.data_ptr()), ws.numel(), None)
    assert rc == B.ERR_INVALID_ARG
    assert B.launch_count() == l0    # nothing was enqueued by any of the rejected calls
    torch.cuda.synchronize()


# ------------------------------------------------------------------ host entry points vs the oracle --

@pytest.mark.parametrize("name,dtype,q", SCAN_CASES)
def test_vjp_scan_host_matches_the_oracle(name, dtype, q):
    n = 50021
    d = scan_data(name, n)
    npdt = np.float64 if dtype == torch.float64 else np.float32
    xs, yb = np.ascontiguousarray(d["xs"].astype(npdt)), np.ascontiguousarray(d["ys_bar"].astype(npdt))
    op = B.Op.of(name, dtype)
    hx, hy = torch.from_numpy(xs).pin_memory(), torch.from_numpy(yb).pin_memory()
    out = torch.empty(hy.shape, dtype=dtype).pin_memory()
    scratch = torch.empty(B.vjp_scan_host_scratch_bytes(op, n), dtype=torch.uint8, device="cuda")
    B.vjp_scan_host(op, None if name == "add" else hx, hy, out, scratch)
    ref = oracle.vjp_scan("matmul" if q else name, xs, yb, q=q)
    assert nrel(out.numpy(), ref) <= (1e-10 if dtype == torch.float64 else 1e-4)
    # accumulate through the host entry point: the prior travels host -> device with the inputs
    prior = np.random.default_rng(3).standard_normal(xs.shape).astype(npdt)
    out2 = torch.from_numpy(prior.copy()).pin_memory()
    B.vjp_scan_host(B.Op.of(name, dtype, accumulate=True), None if name == "add" else hx, hy, out2, scratch)
    assert nrel(out2.numpy(), prior.astype(np.float64) + ref) <= (1e-10 if dtype == torch.float64 else 1e-4)


@pytest.mark.parametrize("opname", ["add", "min", "mul", "satadd"])
def test_rbi_host_entry_points_match_the_oracle(opname):
    n, w = 100003, 3000
    rng = np.random.default_rng(11)
    is_ = rng.integers(-100, w + 100, size=n, dtype=np.int64)
    vs = rng.uniform(0.5, 1.5, n).astype(np.float32)
    hb = rng.standard_normal(w).astype(np.float32)
    S = 20.123
    tot = np.bincount(is_[(is_ >= 0) & (is_ < w)], weights=vs[(is_ >= 0) & (is_ < w)].astype(np.float64), minlength=w)
    while np.any(np.abs(tot - S) < 2.0 ** -6):
        S += 2.0 ** -5
    S = float(np.float32(S))
    op = B.Op.of(opname, S=S)
    if opname == "add":
        ref = oracle.vjp_rbi_add(w, is_, hb)
    elif opname == "min":
        ref = oracle.vjp_rbi_minmax("min", w, is_, vs, hb)[0]
    elif opname == "mul":
        ref = oracle.vjp_rbi_mul(w, is_, vs, hb)[0]
    else:
        ref = oracle.vjp_rbi_general("satadd", w, is_, vs, hb, S=S)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hi, hv, hh = pin(is_), pin(vs), pin(hb)
    nbytes = B.vjp_reduce_by_index_host_scratch_bytes(op, n, w)
    same = (lambda a: np.array_equal(a.astype(np.float64), ref)) if opname != "mul" else (lambda a: nrel(a, ref) <= 1e-4)
    out = torch.empty(n, dtype=torch.float32).pin_memory()
    scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    B.vjp_reduce_by_index_host(op, w, hi, hv, hh, out, scratch)
    assert same(out.numpy())
    # two problems in flight on two streams through the asynchronous variant
    streams, outs, keep = [torch.cuda.Stream(), torch.cuda.Stream()], [], []
    for s in streams:
        o = torch.empty(n, dtype=torch.float32).pin_memory()
        sc = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        keep.append(sc)
        B.vjp_reduce_by_index_host_async(op, w, hi, hv, hh, o, sc, stream=s)
        outs.append(o)
    for s in streams:
        s.synchronize()
    assert all(same(o.numpy()) for o in outs)


# ------------------------------------------------------------------ look-back stress ----------

@pytest.mark.parametrize("name", ["add", "linrec", "matmul5"])
@pytest.mark.parametrize("tiles", [2, 33, 1025])
def test_lookback_stress_200_repetitions(name, tiles):
    """200 back-to-back calls at 2, 33 and 1025 tiles (tile order comes from an atomic ticket and changes
    from call to call): every result within the tolerance, '+' results of f32 inputs in a fixed range."""
    tile = {"add": 16384, "linrec": 8192, "matmul5": 768}[name]
    n = (tiles - 1) * tile + tile // 3 + 1
    d = scan_data(name, n)
    op = B.Op.of(name)
    xs, yb = dev(d["xs"]), dev(d["ys_bar"])
    ref = torch.from_numpy(oracle.vjp_scan("matmul" if name == "matmul5" else name, d["xs"], d["ys_bar"],
                                           q=5 if name == "matmul5" else 0)).cuda().reshape(yb.shape)
    den = ref.abs().max().item()
    ws = torch.empty(B.vjp_scan_workspace_bytes(op, n), dtype=torch.uint8, device="cuda")
    out = torch.empty_like(yb)
    worst = 0.0
    for _ in range(200):
        out.fill_(float("nan"))
        B.vjp_scan(op, xs, yb, out=out, ws=ws)
        err = (out.double() - ref).abs().max().item()
        assert err == err, "NaN left in the output"
        worst = max(worst, err / den)
    assert worst <= 1e-4


# ------------------------------------------------------------------ canary guards ------------
# compute-sanitizer is closed on this GPU pool (profiles/r2_sanitizer.md), so out-of-bounds WRITES are looked
# for directly: every output and workspace sits between two guard bands filled with a canary pattern, at the
# exact size the library asked for, and the bands must come back untouched.

GUARD = 4096  # bytes on either side


def guarded(nbytes, fill=0xA5):
    """(payload view, check()) -- a 16-byte aligned payload of nbytes between two canary bands."""
    pad = (-nbytes) % 16
    buf = torch.full((GUARD + nbytes + pad + GUARD,), fill, dtype=torch.uint8, device="cuda")
    payload = buf[GUARD:GUARD + nbytes]

    def check():
        torch.cuda.synchronize()
        assert bool((buf[:GUARD] == fill).all()) and bool((buf[GUARD + nbytes:] == fill).all()), "guard band overwritten"
    return payload, check


@pytest.mark.parametrize("n", [1, 4097, 16385, 100003])
def test_no_write_outside_outputs_and_workspaces(n):
    rng = np.random.default_rng(n)
    checks = []

    def out_ws(nbytes_out, nbytes_ws, dtype):
        o, c1 = guarded(nbytes_out)
        w, c2 = guarded(max(256, nbytes_ws))
        checks.extend([c1, c2])
        return o.view(dtype), w

    # scans
    for name, dtype, q in SCAN_CASES:
        d = scan_data(name, n)
        npdt = np.float64 if dtype == torch.float64 else np.float32
        op = B.Op.of(name, dtype)
        xs, yb = dev(d["xs"].astype(npdt)), dev(d["ys_bar"].astype(npdt))
        out, ws = out_ws(yb.numel() * yb.element_size(), B.vjp_scan_workspace_bytes(op, n), dtype)
        B.vjp_scan(op, xs, yb, out=out.view(yb.shape), ws=ws)
        out2, ws2 = out_ws(yb.numel() * yb.element_size(), B.vjp_scan_workspace_bytes(op, n), dtype)
        B.scan_forward(op, xs, out=out2.view(xs.shape), ws=ws2)
    # reduce-by-index, narrow and wide histograms
    for w in (7, 1024, 20000, 70000):
        is_ = dev(rng.integers(-3, w + 3, size=n, dtype=np.int64))
        vs = dev(rng.uniform(0.5, 1.5, n).astype(np.float32))
        hb = dev(rng.standard_normal(w).astype(np.float32))
        for opname in ("add", "min", "max", "mul", "satadd"):
            op = B.Op.of(opname, S=0.6 * n / w + 0.37)
            out, ws = out_ws(n * 4, B.vjp_reduce_by_index_workspace_bytes(op, n, w), torch.float32)
            B.vjp_reduce_by_index(op, w, is_, vs, hb, out=out, ws=ws)
            hist, ws2 = out_ws(w * 4, B.vjp_reduce_by_index_workspace_bytes(op, n, w), torch.float32)
            B.reduce_by_index_forward(op, w, is_, vs, out=hist, ws=ws2)
    # reduce
    xs = dev(rng.uniform(0.5, 1.5, n).astype(np.float32))
    yb1 = torch.ones(1, device="cuda")
    for opname in ("add", "min", "mul", "satadd"):
        op = B.Op.of(opname, S=0.3 * n)
        out, ws = out_ws(n * 4, B.vjp_reduce_workspace_bytes(op, n), torch.float32)
        B.vjp_reduce(op, xs, yb1, out=out, ws=ws)
    for c in checks:
        c()


# ------------------------------------------------------------------ CUDA graph capture ------------

def test_calls_can_be_captured_in_a_cuda_graph_and_replayed():
    """The library only enqueues on the caller's stream (no allocation, no synchronisation: include/vjp_b200.h), so a
    sequence of calls can be captured into a CUDA graph -- bench.py times its step that way.  Every replay must give
    the oracle's result again (outputs are poisoned in between; workspaces are re-initialised by the calls)."""
    n, w = 100003, 20000
    dm, dx = W.c2_rbi_min(n=n, w=w, dist="zipf"), W.c2_rbi_mul(n=n, w=w, dist="uniform", zero_rate=1e-3)
    ds = W.c3_scan_linrec(n=n)
    op_min, op_mul, op_lin = B.Op.of("min"), B.Op.of("mul"), B.Op.of("linrec")
    g_min = [dev(dm["is_"]), dev(dm["vs"]), dev(dm["hist_bar"])]
    g_mul = [dev(dx["is_"]), dev(dx["vs"]), dev(dx["hist_bar"])]
    xs, yb = dev(ds["xs"]), dev(ds["ys_bar"])
    o_min, o_mul, o_lin = torch.empty(n, device="cuda"), torch.empty(n, device="cuda"), torch.empty_like(yb)
    ws_rbi = torch.empty(max(B.vjp_reduce_by_index_workspace_bytes(op_min, n, w),
                             B.vjp_reduce_by_index_workspace_bytes(op_mul, n, w)), dtype=torch.uint8, device="cuda")
    ws_scan = torch.empty(B.vjp_scan_workspace_bytes(op_lin, n), dtype=torch.uint8, device="cuda")

    def calls():
        B.vjp_reduce_by_index(op_min, w, *g_min, out=o_min, ws=ws_rbi)
        B.vjp_reduce_by_index(op_mul, w, *g_mul, out=o_mul, ws=ws_rbi)
        B.vjp_scan(op_lin, xs, yb, out=o_lin, ws=ws_scan)

    calls()  # first call outside the capture (function attributes are set lazily)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side, capture_error_mode="thread_local"):
        calls()
    ref_min = oracle.vjp_rbi_minmax("min", w, dm["is_"], dm["vs"], dm["hist_bar"])[0]
    ref_mul = oracle.vjp_rbi_mul(w, dx["is_"], dx["vs"], dx["hist_bar"])[0]
    ref_lin = oracle.vjp_scan("linrec", ds["xs"], ds["ys_bar"])
    for _ in range(3):
        for o in (o_min, o_mul, o_lin):
            o.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        assert np.array_equal(o_min.cpu().numpy().astype(np.float64), np.asarray(ref_min, dtype=np.float64))  # a copy: bit-identical
        assert nrel(o_mul.cpu().numpy(), ref_mul) <= 1e-4
        assert nrel(o_lin.cpu().numpy(), ref_lin) <= 1e-4
