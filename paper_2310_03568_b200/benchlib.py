"""Measurement helpers for bench.py: CUDA-event timing, clock sampling, the algorithmic byte
counts of SURVEY.md section 8(d) / DESIGN.md, and the per-config measurements (VJP time, primal
time, AD overhead, achieved GB/s).  No arithmetic of the method and no oracle import here."""
from __future__ import annotations

import json
import os
import statistics
import subprocess
import threading

import numpy as np
import torch

from . import binding as B
from . import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NORTH_STAR_PEAK_GBS = 8000.0   # "~8 TB/s" of BASELINE.json:north_star, reported beside the measured peak
FALLBACK_PEAK_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peak():
    """(GB/s, 'measured' | 'fallback') from MEASURED_PEAKS.json (driver-written)."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return FALLBACK_PEAK_GBS, "fallback"


# Algorithmic bytes per element of each kernel (what the method itself must move once; look-back
# words, w-sized tables and L2-resident histograms excluded).  Keyed by the library's kernel name.
def kernel_bytes_per_elem(name: str, elem_bytes: int = 4) -> float:
    table = {
        "rbi_vjp_add_kernel": 8 + elem_bytes,        # is + write vs_bar
        "rbi_minmax_lifted_kernel": 8 + 4 + 4,       # is + vs + zero-fill of vs_bar
        "rbi_cached_small_kernel": 8 + 4,            # is + vs
        "rbi_cached_big_kernel": 8 + 4,
        "rbi_mul_sweep_kernel": 8 + 4 + 4,           # is + vs + write vs_bar
        "rbi_forward_kernel": 8 + elem_bytes,
        "scan_lookback_kernel<MODE_SCAN>": 2 * elem_bytes,
        "scan_lookback_kernel<MODE_TILEAGG>": elem_bytes,
        "tile_agg_tma_kernel": elem_bytes,
        "scan_vjp_reverse_kernel": 3 * elem_bytes,
        "sort_hist_kernel": 8,                       # first pass reads int64 keys (4 on later passes)
        "sort_scatter_kernel": 24,                   # read 12, write 12
        "seg_forward_kernel": 12 + 4,
        "seg_reverse_vjp_kernel": 16 + 4,
        "ms_forward_kernel": 8 + 4 + 4,              # is + vs, l written
        "ms_backward_kernel": 8 + 4 + 4 + 4,         # is + vs + l, vs_bar written
        "ms_hist_kernel": 8 + 4,                     # is + vs
    }
    return float(table.get(name, 0.0))


def event_time_ms(fn, reps: int, warmup: int = 3, inner: int = 4):
    """Per-call device times (ms) of fn() on the current stream, CUDA events, after warm-up.  Each sample
    brackets `inner` back-to-back calls (divided out): with one call per event pair the host-side cost of a
    call (ctypes + argument checks, ~20 us) would be measured instead of a kernel that takes 12 us."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    out = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(inner):
            fn()
        b.record()
        b.synchronize()
        out.append(a.elapsed_time(b) / inner)
    return out


def graph_time_ms(fn, reps: int, inner: int = 8):
    """Per-call device times (ms) of fn() replayed from a CUDA graph: `inner` calls are captured once (the library
    only enqueues on the given stream and never allocates or synchronises, so its calls can be captured) and every
    sample replays the graph between two CUDA events -- no host work per call, so a 5 us kernel is timed as such.
    Returns None if the capture fails (the eager timing of event_time_ms then stands alone)."""
    side = torch.cuda.Stream()
    try:
        g = torch.cuda.CUDAGraph()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            fn()  # first call on this stream outside the capture (lazy function attributes, static set-up)
            side.synchronize()
            with torch.cuda.graph(g, stream=side, capture_error_mode="thread_local"):
                for _ in range(inner):
                    fn()
        torch.cuda.synchronize()
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize()
        out = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            g.replay()
            b.record()
            b.synchronize()
            out.append(a.elapsed_time(b) / inner)
        return out
    except Exception:  # noqa: BLE001 -- a capture that fails must not take the bench down
        torch.cuda.synchronize()
        return None


class ClockSampler:
    """Samples SM clocks and throttle reasons while a timed region runs: NVML in a thread (a few ms
    per sample: the timed region of the default run is well under a second), nvidia-smi as fallback."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index: int = 0, period_ms: float = 5.0):
        self.sm, self.mask, self.power = [], 0, []
        self.max_mhz = None
        self._stop = threading.Event()
        self.thread = None
        self.source = "none"
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.period = period_ms / 1e3
            self.source = "nvml"
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.nv = None

    def _sample(self):
        nv = self.nv
        self.sm.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
        try:
            self.mask |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
        except Exception:
            self.mask |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        try:
            self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1e3)
        except Exception:
            pass

    def _pump(self):
        while not self._stop.is_set():
            try:
                self._sample()
            except Exception:
                break
            self._stop.wait(self.period)

    def stop(self):
        if self.thread is not None:
            self._stop.set()
            self.thread.join(timeout=2)
        if not self.sm:  # NVML unavailable: one nvidia-smi query
            try:
                out = subprocess.run(["nvidia-smi", "--query-gpu=clocks.sm,clocks.max.sm", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=20).stdout.split("\n")[0].split(",")
                self.sm, self.max_mhz, self.source = [float(out[0])], float(out[1]), "nvidia-smi (after the region)"
            except Exception:
                pass
        reasons = sorted(name for bit, name in self.REASONS.items() if self.mask & bit)
        return {"sm_mhz": statistics.median(self.sm) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples": len(self.sm), "source": self.source,
                "power_w_max": max(self.power) if self.power else None}


def max_over_ranks(ms: float, device="cpu") -> float:
    """The slowest rank's time (the only cross-rank step of the bench: the path itself shards by
    independent problems and has no collective).  No-op without an initialised process group."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_throughput(elems_per_rank: int, world: int, ms_max: float) -> float:
    """Gelem/s of the whole job: every rank's elements over the slowest rank's time (weak scaling)."""
    return world * elems_per_rank / (ms_max * 1e-3) / 1e9


def to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def to_pinned(a):
    t = torch.from_numpy(np.ascontiguousarray(a))
    return t.pin_memory()


# ------------------------------------------------------------------ workloads ------------

C2_CELLS = [(op, w, dist) for op in ("min", "mul") for w in (1 << 10, 1 << 16) for dist in ("uniform", "zipf")]
VJP_BYTES_PER_ELEM = {  # algorithmic bytes of the whole VJP call per element (roofline table)
    "c1_rbi_add": 12, "c2_rbi_min": 16, "c2_rbi_mul": 28, "c3_scan_add_f32": 8, "c3_scan_mul_f64": 32,
    "c3_scan_linrec_f32": 32, "c4_scan_matmul2": 64, "c4_scan_matmul5": 400,
    # general rule: sort-free walks = forward (is 8 + vs 4 read, l 4 written) + backward (is 8 + vs 4 + l 4 read, 4 written);
    # sort-based (Fig. 4 as written) = the budget of SURVEY.md 8(d)
    "c5_rbi_satadd": 36, "c5_rbi_satadd_sorted": 88,
    "f2_reduce_add": 4, "f2_reduce_min": 8, "f2_reduce_mul": 12,   # fill / read + zero-fill / read, read, write
    "f4_scan_matmul3": 144, "f4_scan_min": 16,
    "f4_scan_exc_linrec": 32 + 16,   # the inclusive rule + the move of ys_bar by one element (read 8, write 8)
    "f3_rbi_vec_mul": (8 + 16) + (8 + 16 + 16),   # per ROW of d = 4, fused: lifted primal (key + row) + sweep (key + row read, row written)
    "f1_sop_inv": 40, "f1_sop_general": 40, "f1_sop_general_sorted": 40,   # primal pass (8 + 8 read) + sweep (8 + 8 read, 8 write): the invertible rule's bytes, used for both rules
}
PRIMAL_BYTES_PER_ELEM = {
    "c1_rbi_add": 12, "c2_rbi_min": 12, "c2_rbi_mul": 12, "c3_scan_add_f32": 8, "c3_scan_mul_f64": 16,
    "c3_scan_linrec_f32": 16, "c4_scan_matmul2": 32, "c4_scan_matmul5": 200, "c5_rbi_satadd": 12, "c5_rbi_satadd_sorted": 12,
    "f2_reduce_add": 4, "f2_reduce_min": 4, "f2_reduce_mul": 4, "f4_scan_matmul3": 72, "f4_scan_min": 8, "f4_scan_exc_linrec": 16 + 16, "f1_sop_inv": 16, "f1_sop_general": 16, "f1_sop_general_sorted": 16, "f3_rbi_vec_mul": 8 + 4 * 4,
}


def gen_c2_cell(op, w, dist, n, seed=0):
    d = (W.c2_rbi_min if op == "min" else W.c2_rbi_mul)(n=n, w=w, dist=dist, seed=seed)
    d["op"], d["dist"] = op, dist
    return d


class RbiCase:
    """One reduce-by-index VJP problem resident on the device, with preallocated output/workspace."""

    def __init__(self, op: B.Op, d, with_host: bool = False):
        self.op, self.n, self.w = op, int(d["n"]), int(d["w"])
        self.is_, self.vs, self.hb = to_dev(d["is_"]), to_dev(d["vs"]), to_dev(d["hist_bar"])
        self.out = torch.empty(self.n, dtype=op.torch_dtype, device="cuda")
        self.hist = torch.empty(self.w, dtype=op.torch_dtype, device="cuda")
        self.ws = torch.empty(max(256, B.vjp_reduce_by_index_workspace_bytes(op, self.n, self.w)),
                              dtype=torch.uint8, device="cuda")
        self.host = None
        if with_host:
            self.host = dict(is_=to_pinned(d["is_"]), vs=to_pinned(d["vs"]), hb=to_pinned(d["hist_bar"]),
                             out=torch.empty(self.n, dtype=op.torch_dtype).pin_memory())
            self.scratch = torch.empty(B.vjp_reduce_by_index_host_scratch_bytes(op, self.n, self.w),
                                       dtype=torch.uint8, device="cuda")

    def vjp(self):
        return B.vjp_reduce_by_index(self.op, self.w, self.is_, self.vs, self.hb, out=self.out, ws=self.ws)

    def primal(self):
        return B.reduce_by_index_forward(self.op, self.w, self.is_, self.vs, out=self.hist, ws=self.ws)

    def vjp_host(self):
        h = self.host
        return B.vjp_reduce_by_index_host(self.op, self.w, h["is_"], h["vs"], h["hb"], h["out"], self.scratch)

    def vjp_host_async(self, stream):
        h = self.host
        return B.vjp_reduce_by_index_host_async(self.op, self.w, h["is_"], h["vs"], h["hb"], h["out"],
                                                self.scratch, stream=stream)

    def h2d_bytes(self):
        h = self.host
        return h["is_"].numel() * 8 + h["vs"].numel() * h["vs"].element_size() + h["hb"].numel() * h["hb"].element_size()

    def d2h_bytes(self):
        return self.host["out"].numel() * self.host["out"].element_size()


class ScanCase:
    def __init__(self, op: B.Op, d, exclusive: bool = False):
        self.op, self.n, self.exclusive = op, int(d["n"]), exclusive
        self.xs, self.yb = to_dev(d["xs"]), to_dev(d["ys_bar"])
        self.out = torch.empty_like(self.yb)
        need = B.vjp_scan_exclusive_workspace_bytes(op, self.n) if exclusive else B.vjp_scan_workspace_bytes(op, self.n)
        self.ws = torch.empty(max(256, need), dtype=torch.uint8, device="cuda")

    def vjp(self):
        if self.exclusive:
            return B.vjp_scan_exclusive(self.op, self.xs, self.yb, out=self.out, ws=self.ws)
        return B.vjp_scan(self.op, self.xs, self.yb, out=self.out, ws=self.ws)

    def primal(self):
        if self.exclusive:
            return B.scan_exclusive_forward(self.op, self.xs, out=self.out, ws=self.ws)
        return B.scan_forward(self.op, self.xs, out=self.out, ws=self.ws)


class SopCase:
    """NEXT row f1: reduce-by-index with sumOfProd, by the invertible-operator rule or the general rule."""

    def __init__(self, d, general):
        self.n, self.w, self.general = int(d["n"]), int(d["w"]), general
        self.is_, self.vs, self.hb = to_dev(d["is_"]), to_dev(d["vs"]), to_dev(d["hist_bar"])
        self.out = torch.empty(2 * self.n, dtype=torch.float32, device="cuda")
        self.hist = torch.empty(2 * self.w, dtype=torch.float32, device="cuda")
        self.ws = torch.empty(max(256, B.rbi_sumofprod_workspace_bytes(self.n, self.w, True)), dtype=torch.uint8, device="cuda")

    def vjp(self):
        return B.vjp_rbi_sumofprod(self.w, self.is_, self.vs, self.hb, general=self.general, out=self.out, ws=self.ws)

    def primal(self):
        return B.rbi_sumofprod_forward(self.w, self.is_, self.vs, out=self.hist, ws=self.ws)


class VecCase:
    """NEXT row f3: reduce-by-index with map2 (*) on rows of d scalars; the primal column = d scalar primal calls."""

    def __init__(self, d):
        self.n, self.d, self.w = int(d["n"]), int(d["d"]), int(d["w"])
        self.op = B.Op.of("mul")
        self.is_, self.vss, self.hb = to_dev(d["is_"]), to_dev(d["vss"]), to_dev(d["hist_bar"])
        self.cols = self.vss.t().contiguous()
        self.out = torch.empty(self.n * self.d, dtype=torch.float32, device="cuda")
        self.hist = torch.empty(self.w, dtype=torch.float32, device="cuda")
        o = self.op.c()
        import ctypes
        self.ws = torch.empty(B.load().vjp_reduce_by_index_vec_workspace_bytes(ctypes.byref(o), self.n, self.d, self.w),
                              dtype=torch.uint8, device="cuda")

    def vjp(self):
        return B.vjp_reduce_by_index_vec(self.op, self.w, self.is_, self.vss, self.hb, out=self.out, ws=self.ws)

    def primal(self):  # the interchanged primal: d scalar histograms on the columns (transposed once, outside the timing)
        for c in range(self.d):
            B.reduce_by_index_forward(self.op, self.w, self.is_, self.cols[c], out=self.hist, ws=self.ws)


class ReduceCase:
    """NEXT row f2: one reduce VJP problem (section 3 of the paper) resident on the device."""

    def __init__(self, op: B.Op, d):
        self.op, self.n = op, int(d["n"])
        self.xs, self.yb = to_dev(d["xs"]), to_dev(d["y_bar"])
        self.out = torch.empty(self.n, dtype=op.torch_dtype, device="cuda")
        self.ws = torch.empty(max(256, B.vjp_reduce_workspace_bytes(op, self.n)), dtype=torch.uint8, device="cuda")

    def vjp(self):
        return B.vjp_reduce(self.op, self.xs, self.yb, out=self.out, ws=self.ws)

    def primal(self):
        return B.reduce_forward(self.op, self.xs, ws=self.ws)


def measure_case(key, label, case, reps, peak_gbs, graph=True):
    """VJP and primal timings of one case (median over reps, CUDA events)."""
    tv = statistics.median(event_time_ms(case.vjp, reps))
    tp = statistics.median(event_time_ms(case.primal, reps))
    n = case.n
    vb, pb = VJP_BYTES_PER_ELEM[key] * n, PRIMAL_BYTES_PER_ELEM[key] * n
    gbs = vb / (tv * 1e-3) / 1e9
    extra = {}
    if graph:  # the same calls replayed from a CUDA graph: what a C caller in a tight loop sees (no Python per call)
        gv, gp = graph_time_ms(case.vjp, reps), graph_time_ms(case.primal, reps)
        if gv is not None and gp is not None:
            gv, gp = statistics.median(gv), statistics.median(gp)
            extra = {"vjp_ms_graph": round(gv, 4), "primal_ms_graph": round(gp, 4),
                     "frac_graph": round(vb / (gv * 1e-3) / 1e9 / peak_gbs, 3)}
    return {
        "case": label, "n": n, "vjp_ms": round(tv, 4), "primal_ms": round(tp, 4),
        "vjp_gelem_s": round(n / (tv * 1e-3) / 1e9, 3),
        "ad_overhead": round((tp + tv) / tp, 3),            # BASELINE.json: (primal + VJP) / primal
        "vjp_over_primal": round(tv / tp, 3),               # the VJP call alone (it re-executes the forward part)
        "vjp_alg_gbs": round(gbs, 1), "frac_of_measured_peak": round(gbs / peak_gbs, 3),
        "frac_of_8tbs": round(gbs / NORTH_STAR_PEAK_GBS, 3),
        "primal_alg_gbs": round(pb / (tp * 1e-3) / 1e9, 1),
        **extra,
    }


def case_table(scale=1.0):
    """(key, label, factory) of every measured case: the five BASELINE configs at full size
    (scale < 1 shrinks n, for quick checks) plus the config-1 bandwidth twin."""
    def sz(n):
        return max(1024, int(n * scale))

    def rbi(opname, gen, **kw):
        def make():
            d = gen()
            return RbiCase(B.Op.of(opname, **({"S": d["S"]} if opname == "satadd" else {}), **kw), d)
        return make

    def scan(opname, gen, dtype=None):
        def make():
            return ScanCase(B.Op.of(opname, dtype) if dtype is not None else B.Op.of(opname), gen())
        return make

    t = [
        ("c1_rbi_add", "c1 rbi + f32 w=1024 (L2-resident, latency-bound)",
         rbi("add", lambda: W.c1_rbi_add(n=sz(W.FULL["c1"]["n"])))),
        ("c1_rbi_add", "c1 twin rbi + f32 w=1024 n=2^26 (bandwidth)",
         rbi("add", lambda: W.c1_rbi_add(n=sz(1 << 26)))),
    ]
    for op, w, dist in C2_CELLS:
        t.append(("c2_rbi_" + op, "c2 rbi %s f32 w=%d %s" % (op, w, dist),
                  rbi(op, lambda op=op, w=w, dist=dist: gen_c2_cell(op, w, dist, sz(W.FULL["c2"]["n"])))))
    n3 = sz(W.FULL["c3"]["n"])
    t += [
        ("c3_scan_add_f32", "c3 scan + f32", scan("add", lambda: W.c3_scan_add(n=n3))),
        ("c3_scan_mul_f64", "c3 scan * f64", scan("mul", lambda: W.c3_scan_mul(n=n3), torch.float64)),
        ("c3_scan_linrec_f32", "c3 scan linrec f32x2", scan("linrec", lambda: W.c3_scan_linrec(n=n3))),
        ("c4_scan_matmul2", "c4 scan matmul 2x2 f32",
         scan("matmul2", lambda: W.c4_scan_matmul(2, n=sz(W.FULL["c4"]["n2"])))),
        ("c4_scan_matmul5", "c4 scan matmul 5x5 f32",
         scan("matmul5", lambda: W.c4_scan_matmul(5, n=sz(W.FULL["c4"]["n5"])))),
        ("c5_rbi_satadd", "c5 rbi satadd (general rule, sort-free walks) f32 w=4096",
         rbi("satadd", lambda: W.c5_rbi_satadd(n=sz(W.FULL["c5"]["n"])))),
        ("c5_rbi_satadd_sorted", "c5 rbi satadd (general rule as Fig. 4: sort + segmented scans) f32 w=4096",
         rbi("satadd", lambda: W.c5_rbi_satadd(n=sz(W.FULL["c5"]["n"])), force_general=2)),
    ]
    t.append(("f3_rbi_vec_mul", "f3 rbi map2(*) d=4 n=2^22 rows w=1024 (NEXT row)", lambda: VecCase(W.f3_rbi_vec("mul", n=sz(1 << 22)))))
    for general in (0, 1, 2):  # NEXT row f1: the same data through both rules
        t.append((("f1_sop_inv", "f1_sop_general", "f1_sop_general_sorted")[general],
                  "f1 rbi sumOfProd w=1024 uniform, %s (NEXT row)" % (
                      "invertible rule", "general rule, sort-free walks", "general rule as Fig. 4 (sort)")[general],
                  lambda general=general: SopCase(W.f1_rbi_sumofprod(n=sz(1 << 24)), general)))
    t.append(("f4_scan_matmul3", "f4 scan matmul 3x3 f32 n=2^22 (NEXT row)",
              scan("matmul3", lambda: W.c4_scan_matmul(3, n=sz(1 << 22)))))
    t.append(("f4_scan_min", "f4 scan min f32 n=2^26 (NEXT row)", scan("min", lambda: W.c3_scan_add(n=n3))))
    t.append(("f4_scan_exc_linrec", "f4 scan^exc (exclusive) linrec f32x2 n=2^26 (NEXT row)",
              lambda: ScanCase(B.Op.of("linrec"), W.c3_scan_linrec(n=n3), exclusive=True)))
    for opname in ("add", "min", "mul"):  # NEXT row f2 (not a BASELINE config): reduce VJP, n = 2^24
        t.append(("f2_reduce_" + opname, "f2 reduce %s f32 n=2^24 (NEXT row)" % opname,
                  lambda opname=opname: ReduceCase(B.Op.of(opname), W.f2_reduce(opname, n=sz(1 << 24)))))
    return t


def measure_all_configs(reps, peak_gbs, scale=1.0, log=None, only=None, kernels=False):
    """Every case of case_table(), one at a time; `only` = substrings of the labels to keep."""
    rows = []
    for key, label, make in case_table(scale):
        if only and not any(s in label for s in only):
            continue
        if log:
            log(label)
        case = make()
        row = measure_case(key, label, case, reps, peak_gbs)
        if kernels:  # per-kernel CUDA-event times of the VJP call (library instrumentation)
            B.profile_enable(True)
            for _ in range(3):
                case.vjp()
            torch.cuda.synchronize()
            prof = B.profile_read()
            B.profile_enable(False)
            row["vjp_kernels_ms"] = {k: round(ms / cnt, 4) for k, (ms, cnt) in prof.items()}
            row["vjp_kernel_launches"] = {k: cnt // 3 for k, (ms, cnt) in prof.items()}
        rows.append(row)
        del case
        torch.cuda.empty_cache()
    return rows


def main(argv=None):
    """python -m paper_2310_03568_b200.benchlib --cases 'scan +,matmul' [--reps R] [--scale S]
    times the named cases only (one JSON row per line): the command the ncu captures under
    profiles/ were taken with."""
    import argparse
    ap = argparse.ArgumentParser()
    ap.add_argument("--cases", default="")
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--kernels", action="store_true", help="add the per-kernel times of the VJP call")
    a = ap.parse_args(argv)
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device: there is no CPU path")
    B.load()
    peak, _ = measured_peak()
    only = [s for s in a.cases.split(",") if s] or None
    for row in measure_all_configs(a.reps, peak, a.scale, only=only, kernels=a.kernels):
        print(json.dumps(row), flush=True)


if __name__ == "__main__":
    main()
