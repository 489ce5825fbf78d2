"""Thin ctypes binding of libqhap.so (include/qhap.h): same names, argument marshalling only.

Device memory and the stream come from PyTorch; every step of the path runs in the library's CUDA kernels.
Importing this module loads the library and fails loudly if it is missing -- there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from pathlib import Path
from typing import Optional

import numpy as np
import torch

_LIB_PATH = Path(__file__).resolve().parent / "libqhap.so"
if not _LIB_PATH.exists():
    raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2603_25762_b200.build` "
                      "(libqhap has no CPU fallback)")
_lib = C.CDLL(str(_LIB_PATH))

QHAP_OK, QHAP_ERR_INVALID_ARG, QHAP_ERR_RANGE, QHAP_ERR_WORKSPACE, QHAP_ERR_CUDA = range(5)
QHAP_WEIGHT_D, QHAP_WEIGHT_D_MINUS_C, QHAP_WEIGHT_FX = 0, 1, 2
QHAP_DENSE_NONE, QHAP_DENSE_FP16, QHAP_DENSE_BF16 = 0, 1, 2

EXPORTS = ["qhap_build_read_graph", "qhap_build_snp_graph", "qhap_build_snp_graph_fill", "qhap_bsb_solve", "qhap_cut_eval", "qhap_cut_eval_static",
           "qhap_phase_readout_reads", "qhap_phase_readout_snps", "qhap_block_split", "qhap_block_stitch",
           "qhap_gauge_transform", "qhap_flip_count_update", "qhap_refine_readout", "qhap_snp_refine",
           "qhap_component_split", "qhap_component_merge", "qhap_plan_pair_tiles",
           "qhap_last_error", "qhap_launch_count", "qhap_version"]


class _Frags(C.Structure):
    _fields_ = [("n_frag", C.c_int32), ("n_snp", C.c_int32), ("nnz", C.c_int64), ("frag_ptr", C.c_void_p),
                ("snp_idx", C.c_void_p), ("allele", C.c_void_p), ("qual", C.c_void_p), ("frag_flags", C.c_void_p),
                ("h1", C.c_void_p)]


class _Csr(C.Structure):
    _fields_ = [("n", C.c_int32), ("nnz", C.c_int64), ("row_ptr", C.c_void_p), ("col", C.c_void_p), ("d", C.c_void_p),
                ("c", C.c_void_p), ("w_fx", C.c_void_p), ("w", C.c_void_p)]


class _BsbTuning(C.Structure):
    _fields_ = [("dense_bn", C.c_int32), ("step_launch", C.c_int32), ("l2_hints", C.c_int32), ("dense_stg_bufs", C.c_int32),
                ("dense_epi_sync", C.c_int32), ("l2_keep_16ths", C.c_int32), ("state16", C.c_int32), ("split_acc", C.c_int32), ("y_ring", C.c_int32), ("pair_tiles", C.c_int32), ("reserved", C.c_int32 * 6)]


class _BsbParams(C.Structure):
    _fields_ = [("replicas", C.c_int32), ("steps_total", C.c_int32), ("step_begin", C.c_int32), ("steps_run", C.c_int32),
                ("dt", C.c_double), ("a0", C.c_double), ("c0", C.c_double), ("seed", C.c_uint64),
                ("replica_begin", C.c_int32), ("weight_mode", C.c_int32), ("path", C.c_int32), ("tile_skip", C.c_int32), ("init_state", C.c_int32),
                ("finalize", C.c_int32), ("force_mode", C.c_int32), ("eval_every", C.c_int32),
                ("trace_cut", C.c_void_p), ("trace_best_cut", C.c_void_p), ("tuning", C.POINTER(_BsbTuning))]


TUNING_KEYS = ("dense_bn", "step_launch", "l2_hints", "dense_stg_bufs", "dense_epi_sync", "l2_keep_16ths", "state16", "split_acc", "y_ring", "pair_tiles")


def _tuning(kw: dict):
    """qhap_bsb_tuning from keyword arguments (None when every knob is automatic)."""
    if not any(kw.get(k) for k in TUNING_KEYS):
        return None
    t = _BsbTuning()
    for k in TUNING_KEYS:
        setattr(t, k, int(kw.get(k) or 0))
    return t


for _name in EXPORTS[:-3]:           # every entry point but the last three returns a qhap_status
    getattr(_lib, _name).restype = C.c_int
_lib.qhap_last_error.restype = C.c_char_p
_lib.qhap_version.restype = C.c_char_p
_lib.qhap_launch_count.restype = C.c_uint64


class QhapError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: status {status}: {_lib.qhap_last_error().decode()}")


def qhap_version() -> str:
    return _lib.qhap_version().decode()


def qhap_launch_count() -> int:
    return int(_lib.qhap_launch_count())


def qhap_last_error() -> str:
    return _lib.qhap_last_error().decode()


def _check(status: int, where: str):
    if status != QHAP_OK:
        raise QhapError(status, where)


def _ptr(t: Optional[torch.Tensor]):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device pointers must come from contiguous CUDA tensors"
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev():
    if not torch.cuda.is_available():
        raise RuntimeError("libqhap needs a CUDA device (sm_100); there is no CPU fallback")
    return torch.device("cuda", torch.cuda.current_device())


def _workspace(nbytes: int) -> torch.Tensor:
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=_dev())


@dataclass
class Frags:
    """Device copy of a fragment matrix (qhap_frags)."""
    n_frag: int
    n_snp: int
    nnz: int
    frag_ptr: torch.Tensor
    snp_idx: torch.Tensor
    allele: torch.Tensor
    qual: Optional[torch.Tensor]
    frag_flags: Optional[torch.Tensor]
    h1: Optional[torch.Tensor]

    def c_struct(self) -> _Frags:
        return _Frags(self.n_frag, self.n_snp, self.nnz, _ptr(self.frag_ptr), _ptr(self.snp_idx), _ptr(self.allele),
                      _ptr(self.qual), _ptr(self.frag_flags), _ptr(self.h1))


def upload_frags(fr, non_blocking: bool = False) -> Frags:
    """Host (numpy, synth.Fragments-like) -> device."""
    dev = _dev()

    def up(a, dt):
        if a is None:
            return None
        return torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).to(dev, non_blocking=non_blocking)
    return Frags(int(fr.n_frag), int(fr.n_snp), int(fr.frag_ptr[-1]) if fr.n_frag > 0 else 0, up(fr.frag_ptr, np.int64),
                 up(fr.snp_idx, np.int32), up(fr.allele, np.uint8), up(fr.qual, np.uint8), up(fr.frag_flags, np.uint8),
                 up(fr.h1, np.uint8))


@dataclass
class Csr:
    """Device CSR graph (qhap_csr)."""
    n: int
    nnz: int
    row_ptr: torch.Tensor
    col: Optional[torch.Tensor] = None
    d: Optional[torch.Tensor] = None
    c: Optional[torch.Tensor] = None
    w_fx: Optional[torch.Tensor] = None
    w: Optional[torch.Tensor] = None
    inst_ptr: Optional[np.ndarray] = None      # host int32 [n_inst+1] for block-diagonal graphs

    def c_struct(self, capacity: Optional[int] = None) -> _Csr:
        return _Csr(self.n, self.nnz if capacity is None else capacity, _ptr(self.row_ptr), _ptr(self.col), _ptr(self.d),
                    _ptr(self.c), _ptr(self.w_fx), _ptr(self.w))

    def to_host(self) -> dict:
        out = dict(n=self.n, nnz=self.nnz)
        for k in ("row_ptr", "col", "d", "c", "w_fx", "w"):
            v = getattr(self, k)
            if v is not None:
                out[k] = v.cpu().numpy()
        if self.inst_ptr is not None:
            out["inst_ptr"] = self.inst_ptr
        return out


def upload_csr(g: dict) -> Csr:
    dev = _dev()

    def up(k, dt):
        return torch.from_numpy(np.ascontiguousarray(g[k], dtype=dt)).to(dev) if g.get(k) is not None else None
    return Csr(int(g["n"]), int(g["nnz"]), up("row_ptr", np.int32), up("col", np.int32), up("d", np.int32), up("c", np.int32),
               up("w_fx", np.int64), up("w", np.float32), g.get("inst_ptr"))


def _two_phase(fn_name, call, alloc):
    """Workspace query -> count call -> allocate -> fill call (qhap.h capacity protocol)."""
    ws_bytes = C.c_size_t(0)
    _check(call(None, C.byref(ws_bytes), None), fn_name + " (size query)")
    ws = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(ws.numel())
    _check(call(_ptr(ws), C.byref(ws_bytes), None), fn_name + " (count)")
    cstruct = alloc()
    ws_bytes = C.c_size_t(ws.numel())
    _check(call(_ptr(ws), C.byref(ws_bytes), cstruct), fn_name + " (fill)")


def qhap_build_read_graph(frags: Frags, weight_mode: int = QHAP_WEIGHT_D, dense_dtype: int = QHAP_DENSE_NONE,
                          dense_ld: Optional[int] = None, capacity_hint: int = 0):
    """(1) read-graph build -> (Csr with d, c; dense J tensor or None).  PAPER.md:L235-L246.
    capacity_hint > 0 (e.g. the nnz of a previous region of the same kind): the edge arrays are allocated up front with that
    capacity and ONE call counts, scans and fills (qhap.h capacity protocol); if the hint is too small the call reports the
    required nnz and the normal count -> allocate -> fill sequence runs."""
    dev = _dev()
    if capacity_hint > 0:
        g = Csr(frags.n_frag, 0, torch.empty(frags.n_frag + 1, dtype=torch.int32, device=dev))
        g.col, g.d, g.c = (torch.empty(capacity_hint, dtype=torch.int32, device=dev) for _ in range(3))
        if dense_dtype != QHAP_DENSE_NONE and dense_ld is None:
            dense_ld = (frags.n_frag + 127) // 128 * 128
        J = None
        if dense_dtype != QHAP_DENSE_NONE:
            J = torch.empty((dense_ld, dense_ld), dtype=torch.float16 if dense_dtype == QHAP_DENSE_FP16 else torch.bfloat16, device=dev)
        fs, cs = frags.c_struct(), g.c_struct(capacity=capacity_hint)

        def once(ws, ws_bytes):
            return _lib.qhap_build_read_graph(C.byref(fs), C.c_int32(weight_mode), C.byref(cs), _ptr(J), C.c_int32(dense_ld or 0),
                                              C.c_int32(dense_dtype), ws, ws_bytes, _stream())
        nb = C.c_size_t(0)
        _check(once(None, C.byref(nb)), "qhap_build_read_graph (size query)")
        ws = _workspace(nb.value)
        nb = C.c_size_t(ws.numel())
        st = once(_ptr(ws), C.byref(nb))
        if st == QHAP_OK:
            g.nnz = int(cs.nnz)
            g.col, g.d, g.c = g.col[:g.nnz], g.d[:g.nnz], g.c[:g.nnz]
            return g, J
        if st != QHAP_ERR_WORKSPACE:
            _check(st, "qhap_build_read_graph")
        # hint too small: fall through to the two-phase protocol
    g = Csr(frags.n_frag, 0, torch.empty(frags.n_frag + 1, dtype=torch.int32, device=dev))
    fs = frags.c_struct()
    state = {"cs": g.c_struct(), "J": None}
    if dense_dtype != QHAP_DENSE_NONE and dense_ld is None:
        dense_ld = (frags.n_frag + 127) // 128 * 128

    def call(ws, ws_bytes, cs):
        cs = cs if cs is not None else state["cs"]
        state["cs"] = cs
        J = state["J"]
        return _lib.qhap_build_read_graph(C.byref(fs), C.c_int32(weight_mode), C.byref(cs), _ptr(J),
                                          C.c_int32(dense_ld or 0), C.c_int32(dense_dtype if J is not None else 0), ws,
                                          ws_bytes, _stream())

    def alloc():
        nnz = state["cs"].nnz
        g.nnz = nnz
        g.col, g.d, g.c = (torch.empty(max(nnz, 1), dtype=torch.int32, device=dev) for _ in range(3))
        if dense_dtype != QHAP_DENSE_NONE:
            state["J"] = torch.empty((dense_ld, dense_ld), dtype=torch.float16 if dense_dtype == QHAP_DENSE_FP16 else torch.bfloat16,
                                     device=dev)
        return g.c_struct(capacity=max(nnz, 1))
    _two_phase("qhap_build_read_graph", call, alloc)
    g.nnz = int(state["cs"].nnz)
    g.col, g.d, g.c = g.col[:g.nnz], g.d[:g.nnz], g.c[:g.nnz]
    return g, state["J"]


def qhap_build_snp_graph(frags: Frags, linkage_tenths: int = 10, alpha: float = 0.1,
                         llr_table: Optional[np.ndarray] = None, resume: bool = True) -> Csr:
    """(2) SNP-graph build -> Csr with w_fx (int64, 2^-32) and w (fp32).  PAPER.md:L287-L319, L85, L350.
    Count call, allocation, then qhap_build_snp_graph_fill on the same workspace (`resume=False`: the fill call is
    qhap_build_snp_graph again, which repeats the count pass)."""
    dev = _dev()
    g = Csr(frags.n_snp, 0, torch.empty(frags.n_snp + 1, dtype=torch.int32, device=dev))
    fs = frags.c_struct()
    tab = None
    if llr_table is not None:
        tab = np.ascontiguousarray(llr_table, dtype=np.float64)
        assert tab.size == 94 * 94
    tab_p = tab.ctypes.data_as(C.c_void_p) if tab is not None else None
    args = (C.byref(fs), C.c_int32(linkage_tenths), C.c_double(alpha))

    ws_bytes = C.c_size_t(0)
    cs = g.c_struct()
    _check(_lib.qhap_build_snp_graph(*args, tab_p, C.byref(cs), None, C.byref(ws_bytes), _stream()), "qhap_build_snp_graph (size query)")
    ws = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(ws.numel())
    _check(_lib.qhap_build_snp_graph(*args, tab_p, C.byref(cs), _ptr(ws), C.byref(ws_bytes), _stream()), "qhap_build_snp_graph (count)")
    nnz = int(cs.nnz)
    g.col = torch.empty(max(nnz, 1), dtype=torch.int32, device=dev)
    g.w_fx = torch.empty(max(nnz, 1), dtype=torch.int64, device=dev)
    g.w = torch.empty(max(nnz, 1), dtype=torch.float32, device=dev)
    cs = g.c_struct(capacity=max(nnz, 1))
    ws_bytes = C.c_size_t(ws.numel())
    if resume:
        _check(_lib.qhap_build_snp_graph_fill(*args, C.byref(cs), _ptr(ws), C.byref(ws_bytes), _stream()), "qhap_build_snp_graph_fill")
    else:
        _check(_lib.qhap_build_snp_graph(*args, tab_p, C.byref(cs), _ptr(ws), C.byref(ws_bytes), _stream()), "qhap_build_snp_graph (fill)")
    g.nnz = int(cs.nnz)
    g.col, g.w_fx, g.w = g.col[:g.nnz], g.w_fx[:g.nnz], g.w[:g.nnz]
    return g


def qhap_block_split(graph: Csr, windows: np.ndarray) -> Csr:
    """(7) induced sub-graphs of the SNP windows as one block-diagonal Csr (inst_ptr set)."""
    dev = _dev()
    win = np.ascontiguousarray(windows, dtype=np.int64).reshape(-1, 2)
    nb = len(win)
    inst_ptr = np.concatenate([[0], np.cumsum(win[:, 1] - win[:, 0])]).astype(np.int32)
    out = Csr(int(inst_ptr[-1]), 0, torch.empty(int(inst_ptr[-1]) + 1, dtype=torch.int32, device=dev), inst_ptr=inst_ptr)
    gs = graph.c_struct()
    state = {"cs": out.c_struct()}

    def call(ws, ws_bytes, cs):
        cs = cs if cs is not None else state["cs"]
        state["cs"] = cs
        return _lib.qhap_block_split(C.byref(gs), C.c_int32(nb), win.ctypes.data_as(C.c_void_p), C.byref(cs), ws, ws_bytes,
                                     _stream())

    def alloc():
        nnz = state["cs"].nnz
        out.col = torch.empty(max(nnz, 1), dtype=torch.int32, device=dev)
        out.w_fx = torch.empty(max(nnz, 1), dtype=torch.int64, device=dev) if graph.w_fx is not None else None
        out.w = torch.empty(max(nnz, 1), dtype=torch.float32, device=dev) if graph.w is not None else None
        return out.c_struct(capacity=max(nnz, 1))
    _two_phase("qhap_block_split", call, alloc)
    out.nnz = int(state["cs"].nnz)
    out.col = out.col[:out.nnz]
    out.w_fx = out.w_fx[:out.nnz] if out.w_fx is not None else None
    out.w = out.w[:out.nnz] if out.w is not None else None
    return out


def qhap_bsb_solve(graph: Csr, *, replicas: int, steps_total: int, step_begin: int = 0, steps_run: Optional[int] = None,
                   dt: float = 1.25, a0: float = 1.0, c0: float = 0.0, seed: int = 0, weight_mode: int = QHAP_WEIGHT_D,
                   path: int = 0, tile_skip: int = 0, force_mode: int = 0, eval_every: int = 0, trace_cuts: bool = False, replica_begin: int = 0,
                   x: Optional[torch.Tensor] = None, y: Optional[torch.Tensor] = None,
                   dense_J: Optional[torch.Tensor] = None, finalize: bool = True, cut_per_replica: bool = True,
                   workspace: Optional[torch.Tensor] = None, workspace_bytes: Optional[int] = None, **tuning) -> dict:
    """(3)(4)(5) bSB solve.  x, y: [n][R] fp32 CUDA tensors updated in place; None -> seeded on the device.
    Keyword arguments named like the fields of qhap_bsb_tuning (dense_bn, step_launch, l2_hints, ..., state16) fill that
    optional block; eval_every = k > 0 returns `trace_best_cut` [steps_run // k][n_inst] (and `trace_cut` [..][n_inst][R]
    with trace_cuts=True)."""
    dev = _dev()
    unknown = set(tuning) - set(TUNING_KEYS)
    assert not unknown, f"unknown arguments {sorted(unknown)}"
    n, R = graph.n, int(replicas)
    init = x is None
    if init:
        assert y is None and step_begin == 0
        x = torch.empty((n, R), dtype=torch.float32, device=dev)
        y = torch.empty((n, R), dtype=torch.float32, device=dev)
    assert x.shape == (n, R) and y.shape == (n, R) and x.dtype == torch.float32 and y.dtype == torch.float32
    steps_run = steps_total - step_begin if steps_run is None else steps_run
    inst_ptr = graph.inst_ptr
    n_inst = 1 if inst_ptr is None else len(inst_ptr) - 1
    ip = np.ascontiguousarray(inst_ptr, dtype=np.int32) if inst_ptr is not None else None
    n_eval = steps_run // eval_every if eval_every > 0 else 0
    tr_best = torch.empty((n_eval, n_inst), dtype=torch.int64, device=dev) if n_eval else None
    tr_cut = torch.empty((n_eval, n_inst, R), dtype=torch.int64, device=dev) if (n_eval and trace_cuts) else None
    tun = _tuning(tuning)
    p = _BsbParams(R, steps_total, step_begin, steps_run, dt, a0, c0, seed, int(replica_begin), weight_mode, path, tile_skip, int(init),
                   int(finalize), int(force_mode), int(eval_every), tr_cut.data_ptr() if tr_cut is not None else None,
                   tr_best.data_ptr() if tr_best is not None else None, C.pointer(tun) if tun is not None else None)
    gs = graph.c_struct()
    dd = QHAP_DENSE_NONE
    ld = 0
    if dense_J is not None:
        dd = QHAP_DENSE_FP16 if dense_J.dtype == torch.float16 else QHAP_DENSE_BF16
        ld = dense_J.shape[1]
    best_spins = torch.empty(max(n, 1), dtype=torch.int8, device=dev) if finalize else None
    best_cut = torch.empty(n_inst, dtype=torch.int64, device=dev) if finalize else None
    best_rep = torch.empty(n_inst, dtype=torch.int32, device=dev) if finalize else None
    cuts = torch.empty((n_inst, R), dtype=torch.int64, device=dev) if (finalize and cut_per_replica) else None

    def call(ws, ws_bytes):
        return _lib.qhap_bsb_solve(C.byref(gs), C.c_int32(n_inst), ip.ctypes.data_as(C.c_void_p) if ip is not None else None,
                                   _ptr(dense_J), C.c_int32(ld), C.c_int32(dd), C.byref(p), _ptr(x), _ptr(y), _ptr(best_spins),
                                   _ptr(best_cut), _ptr(best_rep), _ptr(cuts), ws, ws_bytes, _stream())
    ws_bytes = C.c_size_t(0)
    _check(call(None, C.byref(ws_bytes)), "qhap_bsb_solve (size query)")
    if workspace is None or workspace.numel() < ws_bytes.value:
        workspace = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(workspace.numel() if workspace_bytes is None else int(workspace_bytes))   # the size the library is told
    _check(call(_ptr(workspace), C.byref(ws_bytes)), "qhap_bsb_solve")
    return dict(x=x, y=y, best_spins=best_spins[:n] if finalize else None, best_cut=best_cut, best_replica=best_rep,
                cut=cuts, workspace=workspace, trace_best_cut=tr_best, trace_cut=tr_cut, workspace_bytes=int(ws_bytes.value))


def qhap_cut_eval(graph: Csr, weight_mode: int, spins: torch.Tensor, want_energy: bool = True):
    """(5) cut[R], energy[R] (int64) of int8 spins [n][R]."""
    dev = _dev()
    if spins.dim() == 1:
        spins = spins[:, None].contiguous()
    n, R = spins.shape
    assert n == graph.n and spins.dtype == torch.int8
    cut = torch.empty(R, dtype=torch.int64, device=dev)
    energy = torch.empty(R, dtype=torch.int64, device=dev) if want_energy else None
    gs = graph.c_struct()

    def call(ws, ws_bytes):
        return _lib.qhap_cut_eval(C.byref(gs), C.c_int32(weight_mode), _ptr(spins), C.c_int32(R), _ptr(cut), _ptr(energy), ws,
                                  ws_bytes, _stream())
    ws_bytes = C.c_size_t(0)
    _check(call(None, C.byref(ws_bytes)), "qhap_cut_eval (size query)")
    ws = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(ws.numel())
    _check(call(_ptr(ws), C.byref(ws_bytes)), "qhap_cut_eval")
    return cut, energy


QHAP_CUT_STATIC_BYTES = 4 << 20


def qhap_cut_eval_static(graph: Csr, weight_mode: int, spins: torch.Tensor, cut: Optional[torch.Tensor] = None,
                         energy: Optional[torch.Tensor] = None, want_energy: bool = True):
    """(5') qhap_cut_eval without a workspace: the scratch is a static device array inside the library
    (QHAP_CUT_STATIC_BYTES; larger problems are rejected).  `cut` / `energy` may be passed in (int64 [R], device), in which
    case this call allocates nothing at all.  Calls that overlap on the GPU share the scratch and race."""
    dev = _dev()
    if spins.dim() == 1:
        spins = spins[:, None].contiguous()
    n, R = spins.shape
    assert n == graph.n and spins.dtype == torch.int8
    if cut is None:
        cut = torch.empty(R, dtype=torch.int64, device=dev)
    if energy is None and want_energy:
        energy = torch.empty(R, dtype=torch.int64, device=dev)
    assert cut.dtype == torch.int64 and cut.numel() == R and (energy is None or (energy.dtype == torch.int64 and energy.numel() == R))
    gs = graph.c_struct()
    _check(_lib.qhap_cut_eval_static(C.byref(gs), C.c_int32(weight_mode), _ptr(spins), C.c_int32(R), _ptr(cut), _ptr(energy), _stream()),
           "qhap_cut_eval_static")
    return cut, energy


def qhap_plan_pair_tiles(n_boxes: int, n_replica_tiles: int, grid: int, min_boxes: int = 2):
    """Host-only: (pairs per replica tile, max boxes per CTA, min boxes per CTA) of the paired-tile plan."""
    out = [C.c_int32(0) for _ in range(3)]
    _check(_lib.qhap_plan_pair_tiles(C.c_int32(n_boxes), C.c_int32(n_replica_tiles), C.c_int32(grid), C.c_int32(min_boxes),
                                     *[C.byref(o) for o in out]), "qhap_plan_pair_tiles")
    return tuple(int(o.value) for o in out)


def qhap_phase_readout_reads(frags: Frags, spins: torch.Tensor) -> torch.Tensor:
    """(6) read-based vote -> hap1 [n_snp] int8 in {0, 1, -1 unphased}."""
    hap = torch.empty(max(frags.n_snp, 1), dtype=torch.int8, device=_dev())
    fs = frags.c_struct()

    def call(ws, ws_bytes):
        return _lib.qhap_phase_readout_reads(C.byref(fs), _ptr(spins), _ptr(hap), ws, ws_bytes, _stream())
    ws_bytes = C.c_size_t(0)
    _check(call(None, C.byref(ws_bytes)), "qhap_phase_readout_reads (size query)")
    ws = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(ws.numel())
    _check(call(_ptr(ws), C.byref(ws_bytes)), "qhap_phase_readout_reads")
    return hap[:frags.n_snp]


def qhap_phase_readout_snps(h1: Optional[torch.Tensor], spins: torch.Tensor) -> torch.Tensor:
    n = spins.numel()
    hap = torch.empty(max(n, 1), dtype=torch.int8, device=_dev())
    _check(_lib.qhap_phase_readout_snps(C.c_int32(n), _ptr(h1), _ptr(spins), _ptr(hap), _stream()), "qhap_phase_readout_snps")
    return hap[:n]


def qhap_block_stitch(n: int, windows: np.ndarray, block_spins: torch.Tensor) -> torch.Tensor:
    win = np.ascontiguousarray(windows, dtype=np.int64).reshape(-1, 2)
    out = torch.empty(max(n, 1), dtype=torch.int8, device=_dev())

    def call(ws, ws_bytes):
        return _lib.qhap_block_stitch(C.c_int32(n), C.c_int32(len(win)), win.ctypes.data_as(C.c_void_p), _ptr(block_spins),
                                      _ptr(out), ws, ws_bytes, _stream())
    ws_bytes = C.c_size_t(0)
    _check(call(None, C.byref(ws_bytes)), "qhap_block_stitch (size query)")
    ws = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(ws.numel())
    _check(call(_ptr(ws), C.byref(ws_bytes)), "qhap_block_stitch")
    return out[:n]


# ------------------------------------------------------------------ (f1) SNP-based iterative refinement, Eq. 15-17
def qhap_gauge_transform(graph: Csr, spins: torch.Tensor) -> None:
    """Eq. 15 in place on graph.w_fx / graph.w."""
    gs = graph.c_struct()
    _check(_lib.qhap_gauge_transform(C.byref(gs), _ptr(spins), _stream()), "qhap_gauge_transform")


def qhap_flip_count_update(spins: torch.Tensor, flip_count: torch.Tensor) -> None:
    """Eq. 16: flip_count += 1 on the smaller subset of spins."""
    n = spins.numel()

    def call(ws, ws_bytes):
        return _lib.qhap_flip_count_update(C.c_int32(n), _ptr(spins), _ptr(flip_count), ws, ws_bytes, _stream())
    ws_bytes = C.c_size_t(0)
    _check(call(None, C.byref(ws_bytes)), "qhap_flip_count_update (size query)")
    ws = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(ws.numel())
    _check(call(_ptr(ws), C.byref(ws_bytes)), "qhap_flip_count_update")


def qhap_refine_readout(h1: Optional[torch.Tensor], flip_count: torch.Tensor) -> torch.Tensor:
    """Eq. 17 -> hap1 [n] int8."""
    n = flip_count.numel()
    hap = torch.empty(max(n, 1), dtype=torch.int8, device=_dev())
    _check(_lib.qhap_refine_readout(C.c_int32(n), _ptr(h1), _ptr(flip_count), _ptr(hap), _stream()), "qhap_refine_readout")
    return hap[:n]


def qhap_snp_refine(graph: Csr, *, replicas: int, steps_total: int, max_iter: int, dt: float = 1.25, a0: float = 1.0,
                    c0: float = 0.0, seed: int = 0, path: int = 0, workspace: Optional[torch.Tensor] = None) -> dict:
    """The refinement loop on one instance; graph.w_fx / graph.w are updated in place."""
    dev = _dev()
    n, R = graph.n, int(replicas)
    x = torch.empty((n, R), dtype=torch.float32, device=dev)
    y = torch.empty((n, R), dtype=torch.float32, device=dev)
    flip = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    p = _BsbParams(R, steps_total, 0, steps_total, dt, a0, c0, seed, 0, QHAP_WEIGHT_FX, path, 0, 1, 1, 0, 0, None, None, None)
    gs = graph.c_struct()
    iters = C.c_int32(0)
    cuts = (C.c_int64 * max_iter)()

    def call(ws, ws_bytes):
        return _lib.qhap_snp_refine(C.byref(gs), C.byref(p), C.c_int32(max_iter), _ptr(x), _ptr(y), _ptr(flip), C.byref(iters), cuts,
                                    ws, ws_bytes, _stream())
    ws_bytes = C.c_size_t(0)
    _check(call(None, C.byref(ws_bytes)), "qhap_snp_refine (size query)")
    if workspace is None or workspace.numel() < ws_bytes.value:
        workspace = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(workspace.numel())
    _check(call(_ptr(workspace), C.byref(ws_bytes)), "qhap_snp_refine")
    return dict(flip_count=flip[:n], iterations=int(iters.value), cuts=[int(c) for c in cuts[:iters.value]], workspace=workspace)


# ------------------------------------------------------------------ (f2) connected components, per-component batching
def qhap_component_split(graph: Csr, min_size: int = 2):
    """-> (block-diagonal Csr of the kept components with inst_ptr set, perm tensor [n_kept] int32)."""
    dev = _dev()
    n, nnz = graph.n, graph.nnz

    def like(t, dt):
        return torch.empty(max(nnz, 1), dtype=dt, device=dev) if t is not None else None
    out = Csr(0, 0, torch.empty(n + 1, dtype=torch.int32, device=dev), torch.empty(max(nnz, 1), dtype=torch.int32, device=dev),
              like(graph.d, torch.int32), like(graph.c, torch.int32), like(graph.w_fx, torch.int64), like(graph.w, torch.float32))
    perm = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
    inst_ptr = np.zeros(n + 1, np.int32)
    n_comp = C.c_int32(0)
    gs, os_ = graph.c_struct(), out.c_struct()

    def call(ws, ws_bytes):
        return _lib.qhap_component_split(C.byref(gs), C.c_int32(min_size), C.byref(os_), _ptr(perm), inst_ptr.ctypes.data_as(C.c_void_p),
                                         C.byref(n_comp), ws, ws_bytes, _stream())
    ws_bytes = C.c_size_t(0)
    _check(call(None, C.byref(ws_bytes)), "qhap_component_split (size query)")
    ws = _workspace(ws_bytes.value)
    ws_bytes = C.c_size_t(ws.numel())
    _check(call(_ptr(ws), C.byref(ws_bytes)), "qhap_component_split")
    m, mnnz = int(os_.n), int(os_.nnz)
    res = Csr(m, mnnz, out.row_ptr[:m + 1], out.col[:mnnz], *(t[:mnnz] if t is not None else None for t in (out.d, out.c, out.w_fx, out.w)),
              inst_ptr=inst_ptr[:n_comp.value + 1].copy())
    return res, perm[:m]


def qhap_component_merge(n: int, perm: torch.Tensor, comp_spins: torch.Tensor) -> torch.Tensor:
    out = torch.empty(max(n, 1), dtype=torch.int8, device=_dev())
    _check(_lib.qhap_component_merge(C.c_int32(n), C.c_int32(perm.numel()), _ptr(perm), _ptr(comp_spins), _ptr(out), _stream()),
           "qhap_component_merge")
    return out[:n]
