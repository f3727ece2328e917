"""TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front end of the f64 single-threaded CPU oracle in ``vjp_oracle.c`` (see that file's
header for what it computes and which passage of arxiv/paper_2310_03568 each function
follows).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; it imports nothing from the CUDA package
``paper_2310_03568_b200`` and the product never imports it.

All inputs are converted to float64 / int64 numpy arrays (f32 -> f64 is exact, so comparisons,
zero tests, argmins and sort order are the same in both precisions); all outputs are float64 /
int64 numpy arrays.  Scan arrays are ``[n]`` or ``[n, d]`` (row-major, a q-by-q matrix element
is stored row-major).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vjp_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

ADD, MIN, MAX, MUL, LINREC, MATMUL, SATADD = range(7)
OPS = {"add": ADD, "min": MIN, "max": MAX, "mul": MUL, "linrec": LINREC,
       "matmul": MATMUL, "satadd": SATADD}


def build(force: bool = False) -> str:
    """Compile vjp_oracle.c with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    return _lib


def _f64(a):
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def _i64(a):
    return np.ascontiguousarray(np.asarray(a), dtype=np.int64)


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _check(rc, what):
    if rc != 0:
        raise RuntimeError("oracle %s failed with status %d" % (what, rc))


def _opcode(op):
    return OPS[op] if isinstance(op, str) else int(op)


def _scan_shape(op, q, xs):
    d = _load().orc_scan_arity(op, q)
    if d < 0:
        raise ValueError("not a scan operator")
    n = xs.size // d
    if xs.size != n * d:
        raise ValueError("xs size is not a multiple of the operator arity %d" % d)
    return n, d


def scan_forward(op, xs, q: int = 0):
    """Inclusive scan."""
    op = _opcode(op)
    xs = _f64(xs)
    n, _ = _scan_shape(op, q, xs)
    ys = np.empty_like(xs)
    _check(_load().orc_scan_forward(op, q, ctypes.c_int64(n), _p(xs), _p(ys)), "scan_forward")
    return ys


def vjp_scan(op, xs, ys_bar, q: int = 0):
    """Input adjoints of the inclusive scan (return sweep P:L553-558)."""
    op = _opcode(op)
    xs, ys_bar = _f64(xs), _f64(ys_bar)
    if xs.shape != ys_bar.shape:
        raise ValueError("xs and ys_bar differ in shape")
    n, _ = _scan_shape(op, q, xs)
    xs_bar = np.zeros_like(xs)
    _check(_load().orc_scan_vjp(op, q, ctypes.c_int64(n), _p(xs), _p(ys_bar), _p(xs_bar)), "scan_vjp")
    return xs_bar


def reduce_by_index_forward(op, num_bins, is_, vs, S: float = 0.0):
    """reduce_by_index over a neutral-initialised histogram."""
    op = _opcode(op)
    is_, vs = _i64(is_), _f64(vs)
    hist = np.empty(num_bins, dtype=np.float64)
    _check(_load().orc_rbi_forward(op, ctypes.c_double(S), ctypes.c_int64(is_.size),
                                   ctypes.c_int64(num_bins), _p(is_), _p(vs), _p(hist)), "rbi_forward")
    return hist


def vjp_rbi_add(num_bins, is_, hist_bar):
    is_, hist_bar = _i64(is_), _f64(hist_bar)
    vs_bar = np.empty(is_.size, dtype=np.float64)
    _check(_load().orc_rbi_vjp_add(ctypes.c_int64(is_.size), ctypes.c_int64(num_bins), _p(is_),
                                   _p(hist_bar), _p(vs_bar)), "rbi_vjp_add")
    return vs_bar


def vjp_rbi_minmax(op, num_bins, is_, vs, hist_bar):
    """Returns (vs_bar, arg[w] int64 with n for an empty bin, ext[w])."""
    op = _opcode(op)
    is_, vs, hist_bar = _i64(is_), _f64(vs), _f64(hist_bar)
    vs_bar = np.empty(is_.size, dtype=np.float64)
    arg = np.empty(num_bins, dtype=np.int64)
    ext = np.empty(num_bins, dtype=np.float64)
    _check(_load().orc_rbi_vjp_minmax(op, ctypes.c_int64(is_.size), ctypes.c_int64(num_bins), _p(is_),
                                      _p(vs), _p(hist_bar), _p(arg), _p(ext), _p(vs_bar)), "rbi_vjp_minmax")
    return vs_bar, arg, ext


def vjp_rbi_mul(num_bins, is_, vs, hist_bar):
    """Returns (vs_bar, zeros[w] int64, prod_nz[w])."""
    is_, vs, hist_bar = _i64(is_), _f64(vs), _f64(hist_bar)
    vs_bar = np.empty(is_.size, dtype=np.float64)
    zeros = np.empty(num_bins, dtype=np.int64)
    prod = np.empty(num_bins, dtype=np.float64)
    _check(_load().orc_rbi_vjp_mul(ctypes.c_int64(is_.size), ctypes.c_int64(num_bins), _p(is_), _p(vs),
                                   _p(hist_bar), _p(zeros), _p(prod), _p(vs_bar)), "rbi_vjp_mul")
    return vs_bar, zeros, prod


def vjp_rbi_general(op, num_bins, is_, vs, hist_bar, S: float = 0.0, with_lr: bool = False):
    """General-case rule, eq. 5.  Returns vs_bar, or (vs_bar, ls, rs)."""
    op = _opcode(op)
    is_, vs, hist_bar = _i64(is_), _f64(vs), _f64(hist_bar)
    n = is_.size
    vs_bar = np.empty(n, dtype=np.float64)
    ls = np.empty(n, dtype=np.float64) if with_lr else None
    rs = np.empty(n, dtype=np.float64) if with_lr else None
    _check(_load().orc_rbi_vjp_general(op, ctypes.c_double(S), ctypes.c_int64(n), ctypes.c_int64(num_bins),
                                       _p(is_), _p(vs), _p(hist_bar), _p(vs_bar), _p(ls), _p(rs)),
           "rbi_vjp_general")
    return (vs_bar, ls, rs) if with_lr else vs_bar


def rbi_sort_perm(num_bins, is_):
    """Stable sort by clamped key (Fig. 4).  Returns (sorted_keys, perm)."""
    is_ = _i64(is_)
    sk = np.empty(is_.size, dtype=np.int64)
    perm = np.empty(is_.size, dtype=np.int64)
    _check(_load().orc_rbi_sort_perm(ctypes.c_int64(is_.size), ctypes.c_int64(num_bins), _p(is_), _p(sk),
                                     _p(perm)), "rbi_sort_perm")
    return sk, perm


# ------------------------------------------------------------------ reduce (section 3) ----

def reduce_forward(op, xs, S: float = 0.0):
    """y = reduce (.) e xs; the neutral element for an empty array."""
    op = _opcode(op)
    xs = _f64(xs)
    y = ctypes.c_double(0.0)
    _check(_load().orc_reduce_forward(op, ctypes.c_double(S), ctypes.c_int64(xs.size), _p(xs), ctypes.byref(y)),
           "reduce_forward")
    return y.value


def vjp_reduce_general(op, xs, y_bar, S: float = 0.0, with_lr: bool = False):
    """General rule, eq. 2 with the two exclusive scans of Fig. 2.  Returns xs_bar or (xs_bar, ls, rs)."""
    op = _opcode(op)
    xs = _f64(xs)
    n = xs.size
    xs_bar = np.empty(n, dtype=np.float64)
    ls = np.empty(n, dtype=np.float64) if with_lr else None
    rs = np.empty(n, dtype=np.float64) if with_lr else None
    _check(_load().orc_reduce_vjp_general(op, ctypes.c_double(S), ctypes.c_int64(n), _p(xs),
                                          ctypes.c_double(float(y_bar)), _p(xs_bar), _p(ls), _p(rs)),
           "reduce_vjp_general")
    return (xs_bar, ls, rs) if with_lr else xs_bar


def vjp_reduce(op, xs, y_bar):
    """Specialised rules of section 3.2 ('+', min, max, '*').  Returns (xs_bar, aux_i, aux_v): aux = (k, extremum)
    for min/max, (number of zeros, product of the non-zeros) for '*', (0, 0.0) for '+'."""
    op = _opcode(op)
    xs = _f64(xs)
    n = xs.size
    xs_bar = np.empty(n, dtype=np.float64)
    ai, av = ctypes.c_int64(0), ctypes.c_double(0.0)
    _check(_load().orc_reduce_vjp(op, ctypes.c_int64(n), _p(xs), ctypes.c_double(float(y_bar)), _p(xs_bar),
                                  ctypes.byref(ai), ctypes.byref(av)), "reduce_vjp")
    return xs_bar, ai.value, av.value


# ------------------------------------------------------------------ sumOfProd (sections 3.3, 4.2.4) ----

def sop_apply(a, b):
    """(p1,s1) sumOfProd (p2,s2)."""
    a, b, out = _f64(a), _f64(b), np.empty(2)
    _check(_load().orc_sop_apply(_p(a), _p(b), _p(out)), "sop_apply")
    return out


def sop_inv(z, b):
    """(p,s) sumOfProd_inv (p2,s2)."""
    z, b, out = _f64(z), _f64(b), np.empty(2)
    _check(_load().orc_sop_inv(_p(z), _p(b), _p(out)), "sop_inv")
    return out


def rbi_sop_forward(num_bins, is_, vs):
    """reduce_by_index with sumOfProd; vs is [n, 2] = (p, s), the result [w, 2]."""
    is_, vs = _i64(is_), _f64(vs)
    hist = np.empty((num_bins, 2), dtype=np.float64)
    _check(_load().orc_rbi_sop_forward(ctypes.c_int64(is_.size), ctypes.c_int64(num_bins), _p(is_), _p(vs), _p(hist)),
           "rbi_sop_forward")
    return hist


def vjp_rbi_sop(num_bins, is_, vs, hist_bar, general: bool = False):
    """vs_bar [n, 2] by the invertible-operator rule (Fig. 6) or, general=True, by eq. 5 with pair folds."""
    is_, vs, hist_bar = _i64(is_), _f64(vs), _f64(hist_bar)
    vs_bar = np.empty((is_.size, 2), dtype=np.float64)
    fn = _load().orc_rbi_sop_vjp_general if general else _load().orc_rbi_sop_vjp_inv
    _check(fn(ctypes.c_int64(is_.size), ctypes.c_int64(num_bins), _p(is_), _p(vs), _p(hist_bar), _p(vs_bar)),
           "rbi_sop_vjp")
    return vs_bar


# ------------------------------------------------------------------ vectorised operators (3.2.4, 4.2.5) ----
# reduce_by_index / scan with the operator `map2 (.)` on rows of d scalars.  By IRWIM / ISWIM (eq. 3 P:L252-263,
# P:L464-466) the combinator moves inside the map: column c of the result depends on column c of the
# input only, so the plain definition is the scalar definition applied to every column.

def rbi_forward_vec(op, num_bins, is_, vss, S: float = 0.0):
    """hist[k, :] = fold over i with is[i] = k of vss[i, :] under map2 (.); vss is [n, d]."""
    vss = _f64(vss)
    return np.stack([reduce_by_index_forward(op, num_bins, is_, vss[:, c], S=S) for c in range(vss.shape[1])], axis=1)


def vjp_rbi_vec(op, num_bins, is_, vss, hist_bar, S: float = 0.0):
    """vss_bar [n, d] of the vectorised reduce_by_index given hist_bar [w, d]: the scalar rule per column."""
    vss, hist_bar = _f64(vss), _f64(hist_bar)
    name = op if isinstance(op, str) else {v: k for k, v in OPS.items()}[op]
    cols = []
    for c in range(vss.shape[1]):
        if name == "add":
            cols.append(vjp_rbi_add(num_bins, is_, hist_bar[:, c]))
        elif name in ("min", "max"):
            cols.append(vjp_rbi_minmax(name, num_bins, is_, vss[:, c], hist_bar[:, c])[0])
        elif name == "mul":
            cols.append(vjp_rbi_mul(num_bins, is_, vss[:, c], hist_bar[:, c])[0])
        else:
            cols.append(vjp_rbi_general(name, num_bins, is_, vss[:, c], hist_bar[:, c], S=S))
    return np.stack(cols, axis=1)


def vjp_scan_vec(op, xss, yss_bar, q: int = 0):
    """xss_bar [n, d * a] of the inclusive scan whose operator applies (.) (arity a) to each of the d blocks of a row:
    a = 1 is map2 (.) on rows of d scalars (ISWIM); a > 1 is an operator with a block-diagonal Jacobian of
    d DIFFERENT blocks (non-redundant BDS: "the computation of rs_bar is performed with k different scans").
    Either way: the rule of the small operator per block column."""
    xss, yss_bar = _f64(xss), _f64(yss_bar)
    a = _load().orc_scan_arity(_opcode(op), q)
    d = xss.shape[1] // a
    cols = [vjp_scan(op, np.ascontiguousarray(xss[:, c * a:(c + 1) * a]), np.ascontiguousarray(yss_bar[:, c * a:(c + 1) * a]), q)
            .reshape(xss.shape[0], a) for c in range(d)]
    return np.concatenate(cols, axis=1)


# ------------------------------------------------------------------ exclusive scan (NEXT row f4) -------------
#
# scan^exc (used by the paper in Fig. 2):  ys_0 = e,  ys_i = x_0 (.) ... (.) x_{i-1}.  Output i of the
# exclusive scan IS output i-1 of the inclusive scan of P:L515-529 (and output 0 is the constant e), so with the shift
# matrix S (S y)_i = y_{i-1}:  d ys^exc / d xs = S . d ys^inc / d xs,  and  xs_bar = (d ys^inc / d xs)^T (S^T ys_bar):
# the inclusive return sweep applied to ys_bar moved down by one element, with a zero in the last place.
# x_{n-1} enters no output: its adjoint is 0.

def scan_neutral(op, q: int = 0):
    """The neutral element e of a scan operator as a row of its arity."""
    op = _opcode(op)
    if op == ADD:
        return np.array([0.0])
    if op == MUL:
        return np.array([1.0])
    if op == MIN:
        return np.array([np.inf])
    if op == MAX:
        return np.array([-np.inf])
    if op == LINREC:
        return np.array([1.0, 0.0])          # (a, b) = (1, 0): the identity map x -> 1 x + 0
    if op == MATMUL:
        return np.eye(q).ravel()
    raise ValueError("not a scan operator")


def scan_exclusive_forward(op, xs, q: int = 0):
    """Exclusive scan: ys_0 = e, ys_i = x_0 (.) ... (.) x_{i-1}."""
    xs = _f64(xs)
    e = scan_neutral(op, q)
    n = xs.size // e.size
    ys = np.empty((n, e.size))
    if n:
        ys[0] = e
        ys[1:] = scan_forward(op, xs, q).reshape(n, e.size)[:-1]
    return ys.reshape(xs.shape)


def vjp_scan_exclusive(op, xs, ys_bar, q: int = 0):
    """Input adjoints of the exclusive scan: the inclusive return sweep on S^T ys_bar (see above)."""
    xs, ys_bar = _f64(xs), _f64(ys_bar)
    if xs.shape != ys_bar.shape:
        raise ValueError("xs and ys_bar differ in shape")
    d = scan_neutral(op, q).size
    n = xs.size // d
    moved = np.zeros((n, d))
    if n:
        moved[:-1] = ys_bar.reshape(n, d)[1:]
    return vjp_scan(op, xs, moved.reshape(xs.shape), q)
