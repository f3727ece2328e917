"""vjp_scan_add_f32_noalloc: the '+' scan VJP whose scratch is a static __device__ array of the library (no workspace,
no cudaMalloc) against the existing path vjp_scan(VJP_OP_ADD, f32), which takes a caller-owned workspace.  Two calls in
a row share the scratch (it keeps the first call's status words: the second call must clear them).  Tolerance: the
f32 normwise 1e-4 of the other GPU tests (the look-back folds the same tile aggregates, but which predecessor already
holds a full prefix depends on timing, so the two runs may round differently).

This file sorts after every other test file on purpose: the suite runs with `pytest -x`."""
import numpy as np
import pytest
import torch

from paper_2310_03568_b200 import binding as B

pytestmark = pytest.mark.gpu


def nrel(got, ref):
    got, ref = got.double(), ref.double()
    assert torch.isfinite(got).all()
    den = ref.abs().max().item()
    err = (got - ref).abs().max().item()
    return (0.0 if err == 0.0 else float("inf")) if den == 0.0 else err / den


def existing_path(ys_bar):
    return B.vjp_scan(B.Op.of("add"), None, ys_bar)


@pytest.mark.parametrize("n", [1, 5, 16384, 16385, (1 << 22) + 77, 1 << 24])
def test_two_calls_in_a_row_match_the_existing_path(n):
    assert n <= B.vjp_scan_add_f32_noalloc_max_n()
    g = torch.Generator(device="cuda").manual_seed(n)
    out = torch.empty(n, device="cuda")
    for call in range(2):  # the second call finds the first call's tickets and prefixes in the scratch
        ys_bar = torch.randn(n, device="cuda", generator=g)
        ref = existing_path(ys_bar)
        got = B.vjp_scan_add_f32_noalloc(ys_bar, out)
        assert got.data_ptr() == out.data_ptr()
        assert nrel(got, ref) <= 1e-4, "call %d" % call
        # closed form on the last tile: xs_bar[n-1] = ys_bar[n-1] exactly
        assert got[-1].item() == ys_bar[-1].item()


def test_large_then_small_then_accumulate_and_in_place():
    n_big, n_small = (1 << 23) + 3, 40001
    big = torch.randn(n_big, device="cuda")
    B.vjp_scan_add_f32_noalloc(big, torch.empty_like(big))           # leaves 513 used slots behind
    ys_bar = torch.randn(n_small, device="cuda")
    ref = existing_path(ys_bar)
    prior = torch.randn(n_small, device="cuda")
    out = prior.clone()
    B.vjp_scan_add_f32_noalloc(ys_bar, out, accumulate=True)
    assert nrel(out - prior, ref) <= 1e-4
    inplace = ys_bar.clone()
    B.vjp_scan_add_f32_noalloc(inplace, inplace)                      # xs_bar == ys_bar is allowed for '+'
    assert nrel(inplace, ref) <= 1e-4


def test_rejects_sizes_beyond_the_static_scratch_and_bad_arguments():
    nmax = B.vjp_scan_add_f32_noalloc_max_n()
    assert nmax == 1 << 24
    before = B.launch_count()
    too_big = torch.empty(nmax + 1, device="cuda")
    with pytest.raises(B.VjpError, match="VJP_ERR_UNSUPPORTED"):
        B.vjp_scan_add_f32_noalloc(too_big, torch.empty_like(too_big))
    with pytest.raises(B.VjpError):
        B.vjp_scan_add_f32_noalloc(torch.empty(8, device="cuda"), None)          # the wrapper allocates nothing either
    x = torch.empty(9, device="cuda")
    with pytest.raises(B.VjpError):
        B.vjp_scan_add_f32_noalloc(x[1:], torch.empty(8, device="cuda"))         # misaligned view
    assert B.launch_count() == before                                            # nothing was enqueued
    e = torch.empty(0, device="cuda")
    assert B.vjp_scan_add_f32_noalloc(e, torch.empty(0, device="cuda")).numel() == 0


def test_no_device_memory_is_allocated_by_the_call():
    n = 1 << 20
    ys_bar, out = torch.randn(n, device="cuda"), torch.empty(n, device="cuda")
    B.vjp_scan_add_f32_noalloc(ys_bar, out)                                      # set-up (symbol address) done
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    stats0 = torch.cuda.memory_stats().get("allocation.all.allocated", 0)
    for _ in range(3):
        B.vjp_scan_add_f32_noalloc(ys_bar, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_stats().get("allocation.all.allocated", 0) == stats0   # no torch allocation in the wrapper
    assert free1 == free0                                                             # no cudaMalloc underneath
