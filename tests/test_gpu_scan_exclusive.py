"""GPU parity of the exclusive-scan variants (NEXT row f4; scan^exc of Fig. 2) against the f64 CPU oracle:
scan_exclusive_forward and vjp_scan_exclusive for every scan operator, at sizes around the tile boundaries; tolerances
are those of the inclusive tests (1e-4 normwise f32, 1e-10 f64)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2310_03568_b200 import binding as B
from test_gpu_parity import SCAN_OPS, TOL, dev, nrel, scan_inputs

pytestmark = pytest.mark.gpu

SIZES = [1, 2, 33, 4095, 4096, 4097, 16385, 100003]


@pytest.mark.parametrize("n", SIZES)
@pytest.mark.parametrize("name", SCAN_OPS)
def test_vjp_scan_exclusive_matches_oracle(name, n):
    op, oname, q, xs, ys_bar = scan_inputs(name, n)
    got = B.vjp_scan_exclusive(op, dev(xs), dev(ys_bar)).cpu().numpy()
    ref = oracle.vjp_scan_exclusive(oname, xs, ys_bar, q=q)
    if name in ("min_f32", "max_f32"):
        assert np.array_equal(got != 0, ref != 0)
    assert nrel(got, ref) <= TOL[op.torch_dtype]
    d = got.size // n
    assert not got.reshape(n, d)[-1].any()          # x_{n-1} enters no output: exactly 0


@pytest.mark.parametrize("n", [1, 129, 4097, 100003])
@pytest.mark.parametrize("name", SCAN_OPS)
def test_scan_exclusive_forward_matches_oracle(name, n):
    op, oname, q, xs, _ = scan_inputs(name, n)
    got = B.scan_exclusive_forward(op, dev(xs)).cpu().numpy()
    ref = oracle.scan_exclusive_forward(oname, xs, q=q)
    d = got.size // n
    assert np.array_equal(got.reshape(n, d)[0].astype(np.float64), oracle.scan_neutral(oname, q))   # ys_0 = e, bit-exact
    if n > 1:
        g, r = got.reshape(n, d)[1:], ref.reshape(n, d)[1:]
        if oname == "linrec":  # the A component underflows: compare the B component (as in the inclusive test)
            g, r = g[:, 1], r[:, 1]
        assert nrel(g, r) <= TOL[op.torch_dtype]
        # output i of the exclusive scan IS output i - 1 of the inclusive one: same kernel, moved
        inc = B.scan_forward(op, dev(xs)).cpu().numpy().reshape(n, d)
        if name not in ("add_f32", "add_f64", "mul_f32", "mul_f64", "mul_f64_nozero", "linrec", "matmul2", "matmul3", "matmul5"):
            assert np.array_equal(got.reshape(n, d)[1:], inc[:-1])     # min / max: no rounding, bit-exact
        else:
            assert nrel(got.reshape(n, d)[1:] if oname != "linrec" else got.reshape(n, d)[1:, 1],
                        inc[:-1] if oname != "linrec" else inc[:-1, 1]) <= TOL[op.torch_dtype]


def test_accumulate_add_without_xs_and_errors():
    n = 50021
    yb = np.random.default_rng(1).standard_normal(n).astype(np.float32)
    ref = oracle.vjp_scan_exclusive("add", np.zeros(n), yb)
    got = B.vjp_scan_exclusive(B.Op.of("add"), None, dev(yb)).cpu().numpy()        # '+' needs no xs
    assert nrel(got, ref) <= 1e-4
    prior = np.random.default_rng(2).standard_normal(n).astype(np.float32)
    out = dev(prior)
    B.vjp_scan_exclusive(B.Op.of("add", accumulate=True), None, dev(yb), out=out)
    assert nrel(out.cpu().numpy().astype(np.float64) - prior, ref) <= 1e-4
    with pytest.raises(B.VjpError):                                                   # satadd is not a scan operator
        B.vjp_scan_exclusive(B.Op.of("satadd", S=1.0), dev(yb), dev(yb))
    need = B.vjp_scan_exclusive_workspace_bytes(B.Op.of("add"), n)
    assert need > B.vjp_scan_workspace_bytes(B.Op.of("add"), n)
    with pytest.raises(B.VjpError):
        B.vjp_scan_exclusive(B.Op.of("add"), None, dev(yb), ws=torch.empty(need - 1, dtype=torch.uint8, device="cuda"))
    e = torch.zeros(0, device="cuda")
    assert B.vjp_scan_exclusive(B.Op.of("add"), None, e).numel() == 0
