"""Thin Python binding of the C ABI in ``include/vjp_b200.h`` (same entry-point names).

Argument marshalling only: every step of the path runs in the CUDA kernels of
``libvjp_b200.so``.  PyTorch is used for device memory (``torch.empty``, ``data_ptr``) and for the
current stream, nothing else.  There is no CPU fallback: if the library is missing and cannot be
built, or a call returns a negative status, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

from . import build as _build

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE, ERR_CUDA = 0, -1, -2, -3, -4
_STATUS = {-1: "VJP_ERR_INVALID_ARG", -2: "VJP_ERR_UNSUPPORTED", -3: "VJP_ERR_WORKSPACE", -4: "VJP_ERR_CUDA"}

OP_ADD, OP_MIN, OP_MAX, OP_MUL, OP_LINREC, OP_MATMUL2, OP_MATMUL5, OP_SATADD, OP_MATMUL3 = range(9)
OPCODES = {"add": OP_ADD, "min": OP_MIN, "max": OP_MAX, "mul": OP_MUL, "linrec": OP_LINREC,
           "matmul2": OP_MATMUL2, "matmul3": OP_MATMUL3, "matmul5": OP_MATMUL5, "satadd": OP_SATADD}
F32, F64 = 0, 1

EXPORTS = [
    "vjp_scan_arity", "vjp_version", "vjp_scan_workspace_bytes", "scan_forward", "vjp_scan",
    "vjp_scan_host_scratch_bytes", "vjp_scan_host", "vjp_scan_add_f32_noalloc_max_n", "vjp_scan_add_f32_noalloc",
    "vjp_scan_exclusive_workspace_bytes", "scan_exclusive_forward", "vjp_scan_exclusive",
    "vjp_reduce_by_index_workspace_bytes",
    "reduce_by_index_forward", "vjp_reduce_by_index", "vjp_reduce_by_index_host_scratch_bytes",
    "vjp_reduce_by_index_host", "vjp_reduce_by_index_host_async", "rbi_argext", "rbi_zero_prod", "rbi_sort_perm",
    "vjp_reduce_workspace_bytes", "reduce_forward", "vjp_reduce", "reduce_lifted",
    "rbi_sumofprod_workspace_bytes", "rbi_sumofprod_forward", "vjp_rbi_sumofprod",
    "vjp_reduce_by_index_vec_workspace_bytes", "vjp_reduce_by_index_vec", "vjp_scan_vec_workspace_bytes", "vjp_scan_vec",
    "vjp_kernel_count", "vjp_kernel_name", "vjp_launch_count", "vjp_profile_enable", "vjp_profile_read",
]


class VjpError(RuntimeError):
    pass


class _OpStruct(ctypes.Structure):
    _fields_ = [("code", ctypes.c_int32), ("dtype", ctypes.c_int32), ("param", ctypes.c_double),
                ("force_general", ctypes.c_int32), ("accumulate", ctypes.c_int32)]


_OP_STRUCTS = {}


@dataclass(frozen=True)
class Op:
    """Operator descriptor (vjp_op_t)."""
    code: int
    dtype: int = F32
    param: float = 0.0
    force_general: int = 0     # 1: the general rule (eq. 5), route chosen by the library; 2: its sort-based form (Fig. 4)
    accumulate: bool = False   # VJP calls: out += contribution (the paper's "+=") instead of out = contribution

    @staticmethod
    def of(name: str, dtype=torch.float32, S: float = 0.0, force_general: int = 0,
           accumulate: bool = False) -> "Op":
        return Op(OPCODES[name], F64 if dtype in (torch.float64, F64) else F32, float(S), int(force_general),
                  bool(accumulate))

    def c(self) -> _OpStruct:
        o = _OP_STRUCTS.get(self)  # the library only reads the descriptor: one struct per distinct Op
        if o is None:
            o = _OP_STRUCTS[self] = _OpStruct(self.code, self.dtype, self.param, int(self.force_general), int(self.accumulate))
        return o

    @property
    def torch_dtype(self):
        return torch.float64 if self.dtype == F64 else torch.float32


_lib = None


def library_path() -> str:
    return _build.LIB


def load() -> ctypes.CDLL:
    """Loads (building first if needed) libvjp_b200.so.  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    # build() is an mtime check when the library is up to date; a stale binary is never loaded
    path = _build.build(force=bool(os.environ.get("VJP_B200_REBUILD")))
    lib = ctypes.CDLL(path)
    vp, i64, sz, opp = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t, ctypes.POINTER(_OpStruct)
    sig = {
        "vjp_scan_arity": (ctypes.c_int, [opp]),
        "vjp_version": (ctypes.c_char_p, []),
        "vjp_scan_workspace_bytes": (sz, [opp, i64]),
        "scan_forward": (ctypes.c_int, [opp, i64, vp, vp, vp, sz, vp]),
        "vjp_scan": (ctypes.c_int, [opp, i64, vp, vp, vp, vp, sz, vp]),
        "vjp_scan_host_scratch_bytes": (sz, [opp, i64]),
        "vjp_scan_host": (ctypes.c_int, [opp, i64, vp, vp, vp, vp, sz, vp]),
        "vjp_scan_exclusive_workspace_bytes": (sz, [opp, i64]),
        "scan_exclusive_forward": (ctypes.c_int, [opp, i64, vp, vp, vp, sz, vp]),
        "vjp_scan_exclusive": (ctypes.c_int, [opp, i64, vp, vp, vp, vp, sz, vp]),
        "vjp_scan_add_f32_noalloc_max_n": (i64, []),
        "vjp_scan_add_f32_noalloc": (ctypes.c_int, [i64, vp, vp, ctypes.c_int, vp]),
        "vjp_reduce_by_index_workspace_bytes": (sz, [opp, i64, i64]),
        "reduce_by_index_forward": (ctypes.c_int, [opp, i64, i64, vp, vp, vp, vp, sz, vp]),
        "vjp_reduce_by_index": (ctypes.c_int, [opp, i64, i64, vp, vp, vp, vp, vp, sz, vp]),
        "vjp_reduce_by_index_host_scratch_bytes": (sz, [opp, i64, i64]),
        "vjp_reduce_by_index_host": (ctypes.c_int, [opp, i64, i64, vp, vp, vp, vp, vp, sz, vp]),
        "vjp_reduce_by_index_host_async": (ctypes.c_int, [opp, i64, i64, vp, vp, vp, vp, vp, sz, vp]),
        "rbi_argext": (ctypes.c_int, [opp, i64, i64, vp, vp, vp, vp, vp, sz, vp]),
        "rbi_zero_prod": (ctypes.c_int, [opp, i64, i64, vp, vp, vp, vp, vp, sz, vp]),
        "rbi_sort_perm": (ctypes.c_int, [i64, i64, vp, vp, vp, vp, sz, vp]),
        "vjp_reduce_by_index_vec_workspace_bytes": (sz, [opp, i64, i64, i64]),
        "vjp_reduce_by_index_vec": (ctypes.c_int, [opp, i64, i64, i64, vp, vp, vp, vp, vp, sz, vp]),
        "vjp_scan_vec_workspace_bytes": (sz, [opp, i64, i64]),
        "vjp_scan_vec": (ctypes.c_int, [opp, i64, i64, vp, vp, vp, vp, sz, vp]),
        "rbi_sumofprod_workspace_bytes": (sz, [i64, i64, ctypes.c_int]),
        "rbi_sumofprod_forward": (ctypes.c_int, [i64, i64, vp, vp, vp, vp, sz, vp]),
        "vjp_rbi_sumofprod": (ctypes.c_int, [i64, i64, vp, vp, vp, vp, ctypes.c_int, ctypes.c_int, vp, sz, vp]),
        "vjp_reduce_workspace_bytes": (sz, [opp, i64]),
        "reduce_forward": (ctypes.c_int, [opp, i64, vp, vp, vp, sz, vp]),
        "vjp_reduce": (ctypes.c_int, [opp, i64, vp, vp, vp, vp, sz, vp]),
        "reduce_lifted": (ctypes.c_int, [opp, i64, vp, vp, vp, vp, sz, vp]),
        "vjp_kernel_count": (ctypes.c_int, []),
        "vjp_kernel_name": (ctypes.c_char_p, [ctypes.c_int]),
        "vjp_launch_count": (i64, [ctypes.c_int]),
        "vjp_profile_enable": (None, [ctypes.c_int]),
        "vjp_profile_read": (ctypes.c_int, [ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                            ctypes.POINTER(ctypes.c_int64)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)  # AttributeError if the library does not export it
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _check(rc: int, what: str) -> None:
    if rc != OK:
        raise VjpError("%s failed: %s (%d)" % (what, _STATUS.get(rc, "?"), rc))


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _dev(t: torch.Tensor, dtype, numel=None, what="tensor") -> torch.Tensor:
    """An input: CUDA, right dtype and size, made contiguous, 16-byte aligned (the kernels use 128-bit
    accesses: a view such as x[1:] is rejected here instead of faulting on the device)."""
    if not t.is_cuda:
        raise VjpError("%s: expected a CUDA tensor (there is no CPU path)" % what)
    if t.dtype != dtype:
        raise VjpError("%s: expected dtype %s, got %s" % (what, dtype, t.dtype))
    if numel is not None and t.numel() != numel:
        raise VjpError("%s: expected %d elements, got %d" % (what, numel, t.numel()))
    t = t.contiguous()
    if t.numel() and t.data_ptr() % 16:
        raise VjpError("%s: data pointer is not 16-byte aligned" % what)
    return t


def _out(t, dtype, numel, device, what="out") -> torch.Tensor:
    """A caller-supplied output (or None: allocate): must be usable in place."""
    if t is None:
        return torch.empty(numel, dtype=dtype, device=device)
    if not t.is_cuda or t.device != device or t.dtype != dtype or t.numel() != numel or not t.is_contiguous():
        raise VjpError("%s: expected a contiguous %s CUDA tensor of %d elements on %s" % (what, dtype, numel, device))
    if t.numel() and t.data_ptr() % 16:
        raise VjpError("%s: data pointer is not 16-byte aligned" % what)
    return t


def _workspace(nbytes: int, device, ws=None) -> torch.Tensor:
    if ws is None:
        return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)
    if not ws.is_cuda or ws.dtype != torch.uint8 or not ws.is_contiguous() or ws.data_ptr() % 16:
        raise VjpError("ws: expected a contiguous, 16-byte aligned uint8 CUDA tensor")
    return ws


def scan_arity(op: Op) -> int:
    o = op.c()
    return load().vjp_scan_arity(ctypes.byref(o))


def version() -> str:
    return load().vjp_version().decode()


def _scan_n(op: Op, xs: torch.Tensor) -> int:
    d = scan_arity(op)
    if d < 0:
        raise VjpError("not a scan operator")
    if xs.numel() % d:
        raise VjpError("tensor size is not a multiple of the operator arity %d" % d)
    return xs.numel() // d


def vjp_scan_workspace_bytes(op: Op, n: int) -> int:
    o = op.c()
    return load().vjp_scan_workspace_bytes(ctypes.byref(o), n)


def scan_forward(op: Op, xs: torch.Tensor, out=None, ws=None, stream=None) -> torch.Tensor:
    """Primal inclusive scan."""
    xs = _dev(xs, op.torch_dtype, what="xs")
    n = _scan_n(op, xs)
    ys = torch.empty_like(xs) if out is None else _out(out, op.torch_dtype, xs.numel(), xs.device)
    ws = _workspace(vjp_scan_workspace_bytes(op, n) if ws is None else 0, xs.device, ws)
    o = op.c()
    _check(load().scan_forward(ctypes.byref(o), n, _ptr(xs), _ptr(ys), _ptr(ws), ws.numel(), _stream(stream)),
           "scan_forward")
    return ys


def vjp_scan(op: Op, xs, ys_bar: torch.Tensor, out=None, ws=None, stream=None) -> torch.Tensor:
    """xs_bar = J^T ys_bar of the inclusive scan (Fig. 7).  xs may be None for '+'."""
    ys_bar = _dev(ys_bar, op.torch_dtype, what="ys_bar")
    if xs is not None:
        xs = _dev(xs, op.torch_dtype, what="xs")
        if xs.shape != ys_bar.shape:
            raise VjpError("xs and ys_bar differ in shape")
    n = _scan_n(op, ys_bar)
    if out is None and op.accumulate:
        raise VjpError("accumulate needs the tensor to add to (out=)")
    xs_bar = torch.empty_like(ys_bar) if out is None else _out(out, op.torch_dtype, ys_bar.numel(), ys_bar.device)
    ws = _workspace(vjp_scan_workspace_bytes(op, n) if ws is None else 0, ys_bar.device, ws)
    o = op.c()
    _check(load().vjp_scan(ctypes.byref(o), n, _ptr(xs), _ptr(ys_bar), _ptr(xs_bar), _ptr(ws), ws.numel(),
                           _stream(stream)), "vjp_scan")
    return xs_bar


def vjp_scan_exclusive_workspace_bytes(op: Op, n: int) -> int:
    o = op.c()
    return load().vjp_scan_exclusive_workspace_bytes(ctypes.byref(o), n)


def scan_exclusive_forward(op: Op, xs: torch.Tensor, out=None, ws=None, stream=None) -> torch.Tensor:
    """ys_0 = e, ys_i = x_0 (.) ... (.) x_{i-1} (scan^exc)."""
    xs = _dev(xs, op.torch_dtype, what="xs")
    n = _scan_n(op, xs)
    ys = torch.empty_like(xs) if out is None else _out(out, op.torch_dtype, xs.numel(), xs.device)
    ws = _workspace(vjp_scan_exclusive_workspace_bytes(op, n) if ws is None else 0, xs.device, ws)
    o = op.c()
    _check(load().scan_exclusive_forward(ctypes.byref(o), n, _ptr(xs), _ptr(ys), _ptr(ws), ws.numel(), _stream(stream)),
           "scan_exclusive_forward")
    return ys


def vjp_scan_exclusive(op: Op, xs, ys_bar: torch.Tensor, out=None, ws=None, stream=None) -> torch.Tensor:
    """xs_bar = J^T ys_bar of the exclusive scan.  xs may be None for '+'."""
    ys_bar = _dev(ys_bar, op.torch_dtype, what="ys_bar")
    if xs is not None:
        xs = _dev(xs, op.torch_dtype, what="xs")
        if xs.shape != ys_bar.shape:
            raise VjpError("xs and ys_bar differ in shape")
    n = _scan_n(op, ys_bar)
    if out is None and op.accumulate:
        raise VjpError("accumulate needs the tensor to add to (out=)")
    xs_bar = torch.empty_like(ys_bar) if out is None else _out(out, op.torch_dtype, ys_bar.numel(), ys_bar.device)
    ws = _workspace(vjp_scan_exclusive_workspace_bytes(op, n) if ws is None else 0, ys_bar.device, ws)
    o = op.c()
    _check(load().vjp_scan_exclusive(ctypes.byref(o), n, _ptr(xs), _ptr(ys_bar), _ptr(xs_bar), _ptr(ws), ws.numel(),
                                     _stream(stream)), "vjp_scan_exclusive")
    return xs_bar


def vjp_scan_add_f32_noalloc_max_n() -> int:
    return load().vjp_scan_add_f32_noalloc_max_n()


def vjp_scan_add_f32_noalloc(ys_bar: torch.Tensor, out: torch.Tensor, accumulate: bool = False, stream=None) -> torch.Tensor:
    """The '+' scan VJP (f32) with the scratch in a static device array of the library: no workspace, no allocation
    -- `out` must be given (this wrapper allocates nothing either).  n <= vjp_scan_add_f32_noalloc_max_n(); calls
    that overlap on the GPU race on the shared scratch (include/vjp_b200.h)."""
    if out is None:
        raise VjpError("vjp_scan_add_f32_noalloc allocates nothing: pass out=")
    ys_bar = _dev(ys_bar, torch.float32, what="ys_bar")
    n = ys_bar.numel()
    xs_bar = _out(out, torch.float32, n, ys_bar.device, "xs_bar")
    _check(load().vjp_scan_add_f32_noalloc(n, _ptr(ys_bar), _ptr(xs_bar), int(accumulate), _stream(stream)),
           "vjp_scan_add_f32_noalloc")
    return xs_bar


def vjp_scan_host_scratch_bytes(op: Op, n: int) -> int:
    o = op.c()
    return load().vjp_scan_host_scratch_bytes(ctypes.byref(o), n)


def _host(t, dtype, numel, what):
    if t is None:
        return None
    if t.is_cuda or t.dtype != dtype or t.numel() != numel or not t.is_contiguous():
        raise VjpError("%s: expected a contiguous %s HOST tensor of %d elements" % (what, dtype, numel))
    return t


def vjp_scan_host(op: Op, xs, ys_bar: torch.Tensor, out: torch.Tensor, scratch: torch.Tensor, stream=None):
    """HOST tensors in and out (pinned for speed); `scratch` is a device uint8 tensor."""
    n = _scan_n(op, ys_bar)
    _host(ys_bar, op.torch_dtype, ys_bar.numel(), "ys_bar")
    _host(xs, op.torch_dtype, ys_bar.numel(), "xs")
    _host(out, op.torch_dtype, ys_bar.numel(), "out")
    scratch = _workspace(0, None, scratch)
    o = op.c()
    _check(load().vjp_scan_host(ctypes.byref(o), n, _ptr(xs), _ptr(ys_bar), _ptr(out), _ptr(scratch),
                                scratch.numel(), _stream(stream)), "vjp_scan_host")
    return out


def vjp_reduce_by_index_workspace_bytes(op: Op, n: int, num_bins: int) -> int:
    o = op.c()
    return load().vjp_reduce_by_index_workspace_bytes(ctypes.byref(o), n, num_bins)


def reduce_by_index_forward(op: Op, num_bins: int, is_: torch.Tensor, vs: torch.Tensor, out=None, ws=None,
                            stream=None) -> torch.Tensor:
    """Primal reduce_by_index over a neutral-initialised histogram."""
    is_ = _dev(is_, torch.int64, what="is")
    n = is_.numel()
    vs = _dev(vs, op.torch_dtype, n, "vs")
    hist = _out(out, op.torch_dtype, num_bins, is_.device, "hist")
    ws = _workspace(vjp_reduce_by_index_workspace_bytes(op, n, num_bins) if ws is None else 0, is_.device, ws)
    o = op.c()
    _check(load().reduce_by_index_forward(ctypes.byref(o), n, num_bins, _ptr(is_), _ptr(vs), _ptr(hist),
                                          _ptr(ws), ws.numel(), _stream(stream)), "reduce_by_index_forward")
    return hist


def vjp_reduce_by_index(op: Op, num_bins: int, is_: torch.Tensor, vs, hist_bar: torch.Tensor, out=None,
                        ws=None, stream=None) -> torch.Tensor:
    """vs_bar of reduce_by_index given hist_bar (Fig. 4 for the general rule)."""
    is_ = _dev(is_, torch.int64, what="is")
    n = is_.numel()
    hist_bar = _dev(hist_bar, op.torch_dtype, num_bins, "hist_bar")
    if vs is not None:
        vs = _dev(vs, op.torch_dtype, n, "vs")
    if out is None and op.accumulate:
        raise VjpError("accumulate needs the tensor to add to (out=)")
    vs_bar = _out(out, op.torch_dtype, n, is_.device, "vs_bar")
    ws = _workspace(vjp_reduce_by_index_workspace_bytes(op, n, num_bins) if ws is None else 0, is_.device, ws)
    o = op.c()
    _check(load().vjp_reduce_by_index(ctypes.byref(o), n, num_bins, _ptr(is_), _ptr(vs), _ptr(hist_bar),
                                      _ptr(vs_bar), _ptr(ws), ws.numel(), _stream(stream)),
           "vjp_reduce_by_index")
    return vs_bar


def vjp_reduce_by_index_host_scratch_bytes(op: Op, n: int, num_bins: int) -> int:
    o = op.c()
    return load().vjp_reduce_by_index_host_scratch_bytes(ctypes.byref(o), n, num_bins)


def vjp_reduce_by_index_host(op: Op, num_bins: int, is_, vs, hist_bar, out, scratch, stream=None):
    """HOST tensors in and out (pinned for speed); `scratch` is a device uint8 tensor."""
    n = is_.numel()
    _host(is_, torch.int64, n, "is"), _host(vs, op.torch_dtype, n, "vs")
    _host(hist_bar, op.torch_dtype, num_bins, "hist_bar"), _host(out, op.torch_dtype, n, "out")
    scratch = _workspace(0, None, scratch)
    o = op.c()
    _check(load().vjp_reduce_by_index_host(ctypes.byref(o), n, num_bins, _ptr(is_), _ptr(vs), _ptr(hist_bar),
                                           _ptr(out), _ptr(scratch), scratch.numel(), _stream(stream)),
           "vjp_reduce_by_index_host")
    return out


def vjp_reduce_by_index_host_async(op: Op, num_bins: int, is_, vs, hist_bar, out, scratch, stream=None):
    """As vjp_reduce_by_index_host, but only enqueued on `stream`: synchronise it before reading `out`."""
    n = is_.numel()
    _host(is_, torch.int64, n, "is"), _host(vs, op.torch_dtype, n, "vs")
    _host(hist_bar, op.torch_dtype, num_bins, "hist_bar"), _host(out, op.torch_dtype, n, "out")
    scratch = _workspace(0, None, scratch)
    o = op.c()
    _check(load().vjp_reduce_by_index_host_async(ctypes.byref(o), n, num_bins, _ptr(is_), _ptr(vs),
                                                 _ptr(hist_bar), _ptr(out), _ptr(scratch), scratch.numel(),
                                                 _stream(stream)), "vjp_reduce_by_index_host_async")
    return out


def rbi_argext(op: Op, num_bins: int, is_: torch.Tensor, vs: torch.Tensor, ws=None, stream=None):
    """(arg[w] int64 with n for an empty bin, ext[w]) of the lifted min/max primal (Fig. 5)."""
    is_ = _dev(is_, torch.int64, what="is")
    n = is_.numel()
    vs = _dev(vs, torch.float32, n, "vs")
    arg = torch.empty(num_bins, dtype=torch.int64, device=is_.device)
    ext = torch.empty(num_bins, dtype=torch.float32, device=is_.device)
    ws = _workspace(vjp_reduce_by_index_workspace_bytes(op, n, num_bins) if ws is None else 0, is_.device, ws)
    o = op.c()
    _check(load().rbi_argext(ctypes.byref(o), n, num_bins, _ptr(is_), _ptr(vs), _ptr(arg), _ptr(ext), _ptr(ws),
                             ws.numel(), _stream(stream)), "rbi_argext")
    return arg, ext


def rbi_zero_prod(op: Op, num_bins: int, is_: torch.Tensor, vs: torch.Tensor, ws=None, stream=None):
    """(zeros[w] int64, prod_nz[w]) of the lifted '*' primal."""
    is_ = _dev(is_, torch.int64, what="is")
    n = is_.numel()
    vs = _dev(vs, torch.float32, n, "vs")
    zeros = torch.empty(num_bins, dtype=torch.int64, device=is_.device)
    prod = torch.empty(num_bins, dtype=torch.float32, device=is_.device)
    ws = _workspace(vjp_reduce_by_index_workspace_bytes(op, n, num_bins) if ws is None else 0, is_.device, ws)
    o = op.c()
    _check(load().rbi_zero_prod(ctypes.byref(o), n, num_bins, _ptr(is_), _ptr(vs), _ptr(zeros), _ptr(prod),
                                _ptr(ws), ws.numel(), _stream(stream)), "rbi_zero_prod")
    return zeros, prod


def rbi_sort_perm(num_bins: int, is_: torch.Tensor, ws=None, stream=None):
    """(sorted_keys, perm) of the stable sort by clamped key (Fig. 4)."""
    is_ = _dev(is_, torch.int64, what="is")
    n = is_.numel()
    sk = torch.empty(n, dtype=torch.int64, device=is_.device)
    perm = torch.empty(n, dtype=torch.int64, device=is_.device)
    ws = _workspace(vjp_reduce_by_index_workspace_bytes(Op(OP_SATADD), n, num_bins) if ws is None else 0, is_.device, ws)
    _check(load().rbi_sort_perm(n, num_bins, _ptr(is_), _ptr(sk), _ptr(perm), _ptr(ws), ws.numel(),
                                _stream(stream)), "rbi_sort_perm")
    return sk, perm


# ------------------------------------------------------------------ vectorised operators --

def vjp_reduce_by_index_vec(op: Op, num_bins: int, is_: torch.Tensor, vss, hist_bar: torch.Tensor, out=None, ws=None,
                            stream=None) -> torch.Tensor:
    """vss_bar [n, d] of reduce_by_index with map2 (.) on rows of d scalars (eq. 3); hist_bar is [w, d]."""
    is_ = _dev(is_, torch.int64, what="is")
    n, d = is_.numel(), hist_bar.shape[-1]
    hist_bar = _dev(hist_bar, torch.float32, num_bins * d, "hist_bar")
    if vss is not None:
        vss = _dev(vss, torch.float32, n * d, "vss")
    if out is None and op.accumulate:
        raise VjpError("accumulate needs the tensor to add to (out=)")
    vss_bar = _out(out, torch.float32, n * d, is_.device, "vss_bar")
    o = op.c()
    need = load().vjp_reduce_by_index_vec_workspace_bytes(ctypes.byref(o), n, d, num_bins)
    ws = _workspace(need, is_.device, ws)
    _check(load().vjp_reduce_by_index_vec(ctypes.byref(o), n, d, num_bins, _ptr(is_), _ptr(vss), _ptr(hist_bar),
                                          _ptr(vss_bar), _ptr(ws), ws.numel(), _stream(stream)), "vjp_reduce_by_index_vec")
    return vss_bar.view(n, d)


def vjp_scan_vec(op: Op, xss, yss_bar: torch.Tensor, out=None, ws=None, stream=None) -> torch.Tensor:
    """xss_bar [n, d * a] of the inclusive scan whose operator applies `op` (arity a) to each of the d blocks of a row:
    a = 1 is map2 (.) on rows of d scalars (ISWIM); a > 1 (linrec, matmul) is a block-diagonal operator of
    d different blocks (non-redundant BDS)."""
    if yss_bar.dim() != 2:
        raise VjpError("yss_bar must be [n, d * arity]")
    a = scan_arity(op)
    if a < 1 or yss_bar.shape[1] % a:
        raise VjpError("row length is not a multiple of the operator's arity")
    n, da = yss_bar.shape
    d = da // a
    yss_bar = _dev(yss_bar, torch.float32, n * da, "yss_bar")
    if xss is not None:
        xss = _dev(xss, torch.float32, n * da, "xss")
    if out is None and op.accumulate:
        raise VjpError("accumulate needs the tensor to add to (out=)")
    xss_bar = _out(out, torch.float32, n * da, yss_bar.device, "xss_bar")
    o = op.c()
    ws = _workspace(load().vjp_scan_vec_workspace_bytes(ctypes.byref(o), n, d) if ws is None else 0, yss_bar.device, ws)
    _check(load().vjp_scan_vec(ctypes.byref(o), n, d, _ptr(xss), _ptr(yss_bar), _ptr(xss_bar), _ptr(ws), ws.numel(),
                               _stream(stream)), "vjp_scan_vec")
    return xss_bar.view(n, da)


# ------------------------------------------------------------------ sumOfProd ------------

def rbi_sumofprod_workspace_bytes(n: int, num_bins: int, general: bool = False) -> int:
    return load().rbi_sumofprod_workspace_bytes(n, num_bins, int(general))


def rbi_sumofprod_forward(num_bins: int, is_: torch.Tensor, vs: torch.Tensor, out=None, ws=None, stream=None):
    """reduce_by_index with sumOfProd: vs [n, 2] = (p, s) -> hist [num_bins, 2]."""
    is_ = _dev(is_, torch.int64, what="is")
    n = is_.numel()
    vs = _dev(vs, torch.float32, 2 * n, "vs")
    hist = _out(out, torch.float32, 2 * num_bins, is_.device, "hist")
    ws = _workspace(rbi_sumofprod_workspace_bytes(n, num_bins) if ws is None else 0, is_.device, ws)
    _check(load().rbi_sumofprod_forward(n, num_bins, _ptr(is_), _ptr(vs), _ptr(hist), _ptr(ws), ws.numel(),
                                        _stream(stream)), "rbi_sumofprod_forward")
    return hist.view(num_bins, 2)


def vjp_rbi_sumofprod(num_bins: int, is_: torch.Tensor, vs: torch.Tensor, hist_bar: torch.Tensor, general: int = 0,
                      accumulate: bool = False, out=None, ws=None, stream=None):
    """vs_bar [n, 2] by the invertible-operator rule (Fig. 6) or by the general rule (eq. 5): general=1 lets the
    library choose the route (sort-free when the bin table fits a warp's shared memory), general=2 is Fig. 4 as
    written (sort + segmented scans)."""
    is_ = _dev(is_, torch.int64, what="is")
    n = is_.numel()
    vs = _dev(vs, torch.float32, 2 * n, "vs")
    hist_bar = _dev(hist_bar, torch.float32, 2 * num_bins, "hist_bar")
    if out is None and accumulate:
        raise VjpError("accumulate needs the tensor to add to (out=)")
    vs_bar = _out(out, torch.float32, 2 * n, is_.device, "vs_bar")
    ws = _workspace(rbi_sumofprod_workspace_bytes(n, num_bins, general) if ws is None else 0, is_.device, ws)
    _check(load().vjp_rbi_sumofprod(n, num_bins, _ptr(is_), _ptr(vs), _ptr(hist_bar), _ptr(vs_bar), int(general),
                                    int(accumulate), _ptr(ws), ws.numel(), _stream(stream)), "vjp_rbi_sumofprod")
    return vs_bar.view(n, 2)


# ------------------------------------------------------------------ reduce ---------------

def vjp_reduce_workspace_bytes(op: Op, n: int) -> int:
    o = op.c()
    return load().vjp_reduce_workspace_bytes(ctypes.byref(o), n)


def reduce_forward(op: Op, xs: torch.Tensor, ws=None, stream=None) -> torch.Tensor:
    """y = reduce (.) e xs as a 1-element device tensor."""
    xs = _dev(xs, op.torch_dtype, what="xs")
    n = xs.numel()
    y = torch.empty(1, dtype=op.torch_dtype, device=xs.device)
    ws = _workspace(vjp_reduce_workspace_bytes(op, n) if ws is None else 0, xs.device, ws)
    o = op.c()
    _check(load().reduce_forward(ctypes.byref(o), n, _ptr(xs), _ptr(y), _ptr(ws), ws.numel(), _stream(stream)),
           "reduce_forward")
    return y


def vjp_reduce(op: Op, xs, y_bar: torch.Tensor, n=None, out=None, ws=None, stream=None) -> torch.Tensor:
    """xs_bar of reduce given the 1-element device tensor y_bar (section 3).  xs may be None for '+' (pass n)."""
    y_bar = _dev(y_bar, op.torch_dtype, 1, "y_bar")
    if xs is not None:
        xs = _dev(xs, op.torch_dtype, what="xs")
        n = xs.numel()
    if n is None:
        raise VjpError("n is required when xs is None")
    if out is None and op.accumulate:
        raise VjpError("accumulate needs the tensor to add to (out=)")
    xs_bar = _out(out, op.torch_dtype, n, y_bar.device, "xs_bar")
    ws = _workspace(vjp_reduce_workspace_bytes(op, n) if ws is None else 0, y_bar.device, ws)
    o = op.c()
    _check(load().vjp_reduce(ctypes.byref(o), n, _ptr(xs), _ptr(y_bar), _ptr(xs_bar), _ptr(ws), ws.numel(),
                             _stream(stream)), "vjp_reduce")
    return xs_bar


def reduce_lifted(op: Op, xs: torch.Tensor, ws=None, stream=None):
    """(aux_i, aux_v) of the lifted primal: (k, extremum) for min/max, (zeros, product of non-zeros) for '*'."""
    xs = _dev(xs, torch.float32, what="xs")
    n = xs.numel()
    ai = torch.empty(1, dtype=torch.int64, device=xs.device)
    av = torch.empty(1, dtype=torch.float32, device=xs.device)
    ws = _workspace(vjp_reduce_workspace_bytes(op, n) if ws is None else 0, xs.device, ws)
    o = op.c()
    _check(load().reduce_lifted(ctypes.byref(o), n, _ptr(xs), _ptr(ai), _ptr(av), _ptr(ws), ws.numel(),
                                _stream(stream)), "reduce_lifted")
    return ai, av


# ------------------------------------------------------------------ instrumentation ------

def kernel_names():
    lib = load()
    return [lib.vjp_kernel_name(i).decode() for i in range(lib.vjp_kernel_count())]


def launch_count(kid: int = -1) -> int:
    """Launches of kernel `kid` (all kernels if negative) since the library was loaded."""
    return int(load().vjp_launch_count(kid))


def profile_enable(on: bool) -> None:
    load().vjp_profile_enable(1 if on else 0)


def profile_read():
    """{kernel name: (total ms, recorded launches)} for the kernels recorded since profile_enable(True)."""
    lib = load()
    out = {}
    for i, name in enumerate(kernel_names()):
        ms, cnt = ctypes.c_double(0.0), ctypes.c_int64(0)
        _check(lib.vjp_profile_read(i, ctypes.byref(ms), ctypes.byref(cnt)), "vjp_profile_read")
        if cnt.value:
            out[name] = (ms.value, cnt.value)
    return out
