"""CPU-side checks of the boundary: libqhap.so loads, exports every symbol include/qhap.h declares, the ctypes mirrors
have the C layout, the size-query protocol works without a GPU, and compute calls fail loudly (no CPU fallback)."""
from __future__ import annotations

import ctypes as C
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "qhap.h"


@pytest.fixture(scope="module")
def lib():
    from paper_2603_25762_b200 import build
    return C.CDLL(str(build.build()))


def declared_symbols():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(qhap_[a-z_0-9]+)\s*\(", text)))


def test_exports_match_header(lib):
    syms = declared_symbols()
    assert {"qhap_build_read_graph", "qhap_build_snp_graph", "qhap_bsb_solve", "qhap_cut_eval"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in qhap.h but not exported"
    from paper_2603_25762_b200 import binding
    assert sorted(binding.EXPORTS) == syms


def test_struct_layouts_match_c(tmp_path):
    """sizeof/offsetof of the ctypes mirrors equal what the C compiler sees for include/qhap.h."""
    from paper_2603_25762_b200 import binding as B
    src = tmp_path / "layout.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "qhap.h"\nint main(void){'
                   'printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n", sizeof(qhap_frags), offsetof(qhap_frags, frag_ptr), offsetof(qhap_frags, h1),'
                   'sizeof(qhap_csr), offsetof(qhap_csr, w), sizeof(qhap_bsb_params), offsetof(qhap_bsb_params, seed),'
                   'offsetof(qhap_bsb_params, finalize), offsetof(qhap_bsb_params, eval_every), offsetof(qhap_bsb_params, trace_cut),'
                   'offsetof(qhap_bsb_params, tuning), sizeof(qhap_bsb_tuning), offsetof(qhap_bsb_tuning, state16), offsetof(qhap_bsb_tuning, reserved));'
                   ' return 0;}')
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", str(ROOT / "include"), str(src), "-o", str(exe)])
    got = [int(v) for v in subprocess.check_output([str(exe)]).split()]
    exp = [C.sizeof(B._Frags), B._Frags.frag_ptr.offset, B._Frags.h1.offset, C.sizeof(B._Csr), B._Csr.w.offset,
           C.sizeof(B._BsbParams), B._BsbParams.seed.offset, B._BsbParams.finalize.offset, B._BsbParams.eval_every.offset,
           B._BsbParams.trace_cut.offset, B._BsbParams.tuning.offset, C.sizeof(B._BsbTuning), B._BsbTuning.state16.offset,
           B._BsbTuning.reserved.offset]
    assert got == exp


def test_size_query_and_loud_failure_without_gpu(lib):
    import torch
    from paper_2603_25762_b200 import binding as B
    lib.qhap_last_error.restype = C.c_char_p
    fr = B._Frags(10, 20, 100, None, None, None, None, None, None)
    g = B._Csr(10, 0, None, None, None, None, None, None)
    ws = C.c_size_t(0)
    assert lib.qhap_build_read_graph(C.byref(fr), 0, C.byref(g), None, 0, 0, None, C.byref(ws), None) == B.QHAP_OK
    assert ws.value > 0
    ws2 = C.c_size_t(0)
    assert lib.qhap_build_snp_graph(C.byref(fr), C.c_int32(10), C.c_double(0.1), None, C.byref(g), None, C.byref(ws2), None) == B.QHAP_OK
    assert ws2.value > ws.value
    assert lib.qhap_build_snp_graph(C.byref(fr), C.c_int32(11), C.c_double(0.1), None, C.byref(g), None, C.byref(ws2), None) == B.QHAP_ERR_INVALID_ARG
    assert b"linkage_tenths" in lib.qhap_last_error()
    p = B._BsbParams(64, 100, 0, 100, 1.25, 1.0, 0.0, 1, 0, 0, 2, 0, 1, 1, 0)
    ws3 = C.c_size_t(0)
    g.nnz = 50
    assert lib.qhap_bsb_solve(C.byref(g), 1, None, None, 0, 0, C.byref(p), None, None, None, None, None, None, None, C.byref(ws3), None) == B.QHAP_OK
    assert ws3.value >= 10 * 64 * 4
    # the size query of every step path, and the optional tuning block: reserved fields must be 0
    sizes = {}
    for path in (1, 2, 4):
        p.path = path
        w = C.c_size_t(0)
        dj = C.c_void_p(256) if path == 1 else None
        assert lib.qhap_bsb_solve(C.byref(g), 1, None, dj, 16, B.QHAP_DENSE_FP16, C.byref(p), None, None, None, None, None, None, None, C.byref(w), None) == B.QHAP_OK
        sizes[path] = w.value
    assert sizes[1] > sizes[2] and sizes[4] > sizes[2]
    t = B._BsbTuning()
    t.reserved[3] = 1
    p.tuning = C.pointer(t)
    assert lib.qhap_bsb_solve(C.byref(g), 1, None, None, 0, 0, C.byref(p), None, None, None, None, None, None, None, C.byref(ws3), None) == B.QHAP_ERR_INVALID_ARG
    assert b"reserved" in lib.qhap_last_error()
    p.tuning = None
    p.force_mode = 2
    assert lib.qhap_bsb_solve(C.byref(g), 1, None, None, 0, 0, C.byref(p), None, None, None, None, None, None, None, C.byref(ws3), None) == B.QHAP_ERR_INVALID_ARG
    if not torch.cuda.is_available():
        # a compute call without a device must fail loudly, not fall back
        buf = (C.c_char * (ws.value + 512))()
        addr = (C.addressof(buf) + 255) & ~255
        ws = C.c_size_t(ws.value)
        st = lib.qhap_build_read_graph(C.byref(fr), 0, C.byref(g), None, 0, 0, C.c_void_p(addr), C.byref(ws), None)
        assert st == B.QHAP_ERR_CUDA and b"no CPU fallback" in lib.qhap_last_error()


def test_no_oracle_in_product_path():
    """The package never imports oracle/ (the oracle is test infrastructure)."""
    for f in (ROOT / "paper_2603_25762_b200").rglob("*.py"):
        assert "oracle" not in re.sub(r"#.*|\"\"\".*?\"\"\"", "", f.read_text(), flags=re.S).replace("the oracle", ""), f
    for f in (ROOT / "paper_2603_25762_b200" / "csrc").glob("*.cu*"):
        assert "orc_" not in f.read_text() and "oracle/" not in f.read_text().replace("used by oracle/", ""), f
