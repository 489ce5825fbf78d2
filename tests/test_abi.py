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


def test_pair_tile_plan_covers_every_box_once_and_balances(lib):
    """qhap_plan_pair_tiles (host only): rebuilding the slot list from the documented numbering, every box appears in exactly one
    slot, the reported per-CTA maxima / minima are those of slot % grid, pairs never raise the most loaded CTA above
    ceil(boxes / grid), and fused plans leave every CTA at least two boxes.  cfg1's shape gives the plan DESIGN.md 4.4g quotes."""
    from paper_2603_25762_b200 import binding as B
    assert B.qhap_plan_pair_tiles(125, 8, 148, 2) == (55, 7, 5)
    for n_boxes, m, grid, min_boxes in [(125, 8, 148, 2), (63, 16, 148, 2), (38, 8, 148, 2), (36, 16, 148, 2), (36, 16, 148, 0), (13, 3, 39, 0),
                                        (2, 1, 2, 0), (2, 1, 1, 2), (3672, 2, 148, 0), (9, 5, 22, 2), (40, 1, 7, 2), (41, 4, 148, 2), (1, 1, 1, 0)]:
        P, mx, mn = B.qhap_plan_pair_tiles(n_boxes, m, grid, min_boxes)
        assert 0 <= P <= n_boxes // 2
        slots = [(2 * q, 2, t) for q in range(P) for t in range(m)] + [(b, 1, t) for b in range(2 * P, n_boxes) for t in range(m)]
        seen = set()
        load = [0] * grid
        for s, (b0, w, t) in enumerate(slots):
            for b in range(b0, b0 + w):
                assert (b, t) not in seen
                seen.add((b, t))
            load[s % grid] += w
        assert len(seen) == n_boxes * m
        assert (max(load), min(load)) == (mx, mn), (n_boxes, m, grid, P)
        if P > 0:
            assert mx <= -(-n_boxes * m // grid) and mn >= min_boxes
    with pytest.raises(B.QhapError):
        B.qhap_plan_pair_tiles(4, 1, 5, 0)                     # more CTAs than boxes
