"""The C ABI of include/vjp_b200.h, the binding's EXPORTS list and the dynamic symbol table of the built
library agree (no GPU needed: nvcc cross-compiles, nothing is launched)."""
import ctypes
import os
import re
import subprocess

from paper_2310_03568_b200 import binding as B
from paper_2310_03568_b200 import build as cuda_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_prototypes():
    """Names of the functions include/vjp_b200.h declares."""
    src = open(os.path.join(ROOT, "include", "vjp_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)                     # comments
    src = re.sub(r"typedef\s+(enum|struct)\s*\{.*?\}\s*\w+\s*;", "", src, flags=re.S)
    names = re.findall(r"\b([A-Za-z_]\w*)\s*\([^;{}]*\)\s*;", src)
    return sorted(set(names))


def test_header_binding_and_library_export_the_same_entry_points():
    lib = cuda_build.build()
    out = subprocess.run(["nm", "-D", "--defined-only", lib], capture_output=True, text=True, check=True).stdout
    exported = {line.split()[-1] for line in out.splitlines() if " T " in line}
    declared = header_prototypes()
    assert declared, "no prototypes parsed from the header"
    assert sorted(B.EXPORTS) == declared
    missing = [n for n in declared if n not in exported]
    assert not missing, "declared in the header but not exported: %s" % missing
    # nothing but the declared C entry points is exported without C++ mangling
    extra = sorted(n for n in exported if not n.startswith("_Z") and n not in declared
                   and not n.startswith("__") and n not in ("_init", "_fini"))
    assert not extra, "exported but not declared in the header: %s" % extra


def test_library_loads_and_answers_host_only_queries():
    lib = B.load()
    assert lib.vjp_version().decode().startswith("vjp_b200")
    assert B.scan_arity(B.Op.of("matmul5")) == 25 and B.scan_arity(B.Op.of("matmul3")) == 9
    assert B.scan_arity(B.Op.of("min")) == 1 and B.scan_arity(B.Op.of("satadd")) == -1
    assert B.vjp_scan_workspace_bytes(B.Op.of("linrec"), 1 << 20) > 0
    assert B.vjp_reduce_by_index_workspace_bytes(B.Op.of("mul"), 1 << 20, 1 << 16) > 0
    assert len(B.kernel_names()) == lib.vjp_kernel_count() and all(B.kernel_names())
    assert B.launch_count() == 0  # nothing was launched by the queries


def test_op_struct_layout_matches_the_header():
    # {int32 code, int32 dtype, double param, int32 force_general, int32 accumulate}
    o = B.Op.of("satadd", S=3.5, force_general=True, accumulate=True).c()
    assert ctypes.sizeof(o) == 24
    assert (o.code, o.dtype, o.param, o.force_general, o.accumulate) == (B.OP_SATADD, B.F32, 3.5, 1, 1)
