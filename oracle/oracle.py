"""ctypes front end of the QHap CPU oracle (oracle/qhap_oracle.cpp) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / ``--impl reference`` legs may import
this module.  It imports nothing from the CUDA package.  The arithmetic of O1-O5 lives in the C++ file, which this
module compiles with g++ (once, into oracle/_build/) and calls with numpy arrays; O6 (iterative refinement, Eq. 15-17)
and O7 (connected components; scipy's connected_components is the library step) are plain numpy below.
Pins: tests/test_oracle_pins.py (O6: gauge identity + planted recovery; O7: hand-made graph + plain BFS).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "qhap_oracle.cpp"
_LIB = _HERE / "_build" / "libqhap_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (no CUDA, no FMA contraction) if the .so is missing or stale."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        _LIB.parent.mkdir(exist_ok=True)
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-pthread",
                               str(_SRC), "-o", str(tmp)])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.orc_read_graph.restype = C.c_int64
        _lib.orc_snp_graph.restype = C.c_int64
        _lib.orc_bsb_c0.restype = C.c_double
        _lib.orc_best_replica.restype = C.c_int32
        _lib.orc_block_split.restype = C.c_int64
        _lib.orc_hardware_threads.restype = C.c_int32
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dt):
    return None if a is None else np.ascontiguousarray(a, dtype=dt)


def hardware_threads() -> int:
    return int(lib().orc_hardware_threads())


# ---------------------------------------------------------------------------------------------- O1
def read_graph(fr) -> dict:
    """Symmetric CSR of the read graph with discordant (d) and concordant (c) counts."""
    L = lib()
    fp, si, al, h1 = _c(fr.frag_ptr, np.int64), _c(fr.snp_idx, np.int32), _c(fr.allele, np.uint8), _c(fr.h1, np.uint8)
    args = (C.c_int32(fr.n_frag), C.c_int32(fr.n_snp), _p(fp), _p(si), _p(al), _p(h1))
    nnz = L.orc_read_graph(*args, None, None, None, None, C.c_int64(0))
    row_ptr = np.zeros(fr.n_frag + 1, np.int32)
    col, d, c = (np.zeros(nnz, np.int32) for _ in range(3))
    L.orc_read_graph(*args, _p(row_ptr), _p(col), _p(d), _p(c), C.c_int64(nnz))
    return dict(n=fr.n_frag, nnz=int(nnz), row_ptr=row_ptr, col=col, d=d, c=c)


# ---------------------------------------------------------------------------------------------- O2
def llr_table() -> np.ndarray:
    T = np.zeros((94, 94), np.float64)
    lib().orc_llr_table(_p(T))
    return T


def snp_graph(fr, linkage_tenths: int = 10, alpha: float = 0.1) -> dict:
    """Symmetric CSR of the SNP graph: w_fx (int64, scale 2^-32) and derived fp32 w."""
    L = lib()
    fp, si, al = _c(fr.frag_ptr, np.int64), _c(fr.snp_idx, np.int32), _c(fr.allele, np.uint8)
    qu, fl, h1 = _c(fr.qual, np.uint8), _c(fr.frag_flags, np.uint8), _c(fr.h1, np.uint8)
    args = (C.c_int32(fr.n_frag), C.c_int32(fr.n_snp), _p(fp), _p(si), _p(al), _p(qu), _p(fl), _p(h1),
            C.c_int32(linkage_tenths), C.c_double(alpha))
    nnz = L.orc_snp_graph(*args, None, None, None, None, C.c_int64(0))
    row_ptr = np.zeros(fr.n_snp + 1, np.int32)
    col, w_fx, w = np.zeros(nnz, np.int32), np.zeros(nnz, np.int64), np.zeros(nnz, np.float32)
    L.orc_snp_graph(*args, _p(row_ptr), _p(col), _p(w_fx), _p(w), C.c_int64(nnz))
    return dict(n=fr.n_snp, nnz=int(nnz), row_ptr=row_ptr, col=col, w_fx=w_fx, w=w)


# ---------------------------------------------------------------------------------------------- O3
def bsb_c0(row_ptr, jval) -> float:
    rp, jv = _c(row_ptr, np.int32), _c(jval, np.float32)
    return float(lib().orc_bsb_c0(C.c_int32(len(rp) - 1), _p(rp), _p(jv)))


def bsb_run(row_ptr, col, jval, x, y, *, steps_total, step_begin=0, steps_run=None, dt=1.25, a0=1.0, c0=None,
            n_threads=1, xpre=None, force_mode=0):
    """Advance fp64 state x, y ([n][R]) in place by ``steps_run`` bSB steps; returns (x, y, c0).

    ``xpre`` (optional fp64 [n][R] array) receives x of the last step before the wall rule.
    ``force_mode`` 1 = dSB (F = J sgn(x)), 0 = bSB (L265)."""
    rp, cl, jv = _c(row_ptr, np.int32), _c(col, np.int32), _c(jval, np.float32)
    n = len(rp) - 1
    x = np.ascontiguousarray(x, np.float64); y = np.ascontiguousarray(y, np.float64)
    assert x.shape == y.shape and x.shape[0] == n
    R = x.shape[1]
    if c0 is None or c0 <= 0:
        c0 = bsb_c0(rp, jv)
    if steps_run is None:
        steps_run = steps_total - step_begin
    lib().orc_bsb_run(C.c_int32(n), _p(rp), _p(cl), _p(jv), C.c_int32(R), C.c_int32(steps_total),
                      C.c_int32(step_begin), C.c_int32(steps_run), C.c_double(dt), C.c_double(a0), C.c_double(c0),
                      _p(x), _p(y), _p(xpre), C.c_int32(n_threads), C.c_int32(force_mode))
    return x, y, c0


def bsb_run_dense(J, x, y, *, steps_total, step_begin=0, steps_run=None, dt=1.25, a0=1.0, c0=1.0):
    J = np.ascontiguousarray(J, np.float64)
    n = J.shape[0]
    x = np.ascontiguousarray(x, np.float64); y = np.ascontiguousarray(y, np.float64)
    if steps_run is None:
        steps_run = steps_total - step_begin
    lib().orc_bsb_run_dense(C.c_int32(n), _p(J), C.c_int32(x.shape[1]), C.c_int32(steps_total), C.c_int32(step_begin),
                            C.c_int32(steps_run), C.c_double(dt), C.c_double(a0), C.c_double(c0), _p(x), _p(y))
    return x, y


# ---------------------------------------------------------------------------------------------- O4
def cut_eval(row_ptr, col, w_int, spins):
    """cut[R], energy[R] (int64) of spins [n][R] (or [n]) on canonical integer weights."""
    rp, cl, w = _c(row_ptr, np.int32), _c(col, np.int32), _c(w_int, np.int64)
    s = _c(spins, np.int8)
    if s.ndim == 1:
        s = s[:, None].copy()
    n, R = s.shape
    assert n == len(rp) - 1
    cut, en = np.zeros(R, np.int64), np.zeros(R, np.int64)
    lib().orc_cut_eval(C.c_int32(n), _p(rp), _p(cl), _p(w), _p(s), C.c_int32(R), _p(cut), _p(en))
    return cut, en


def sign_spins(x) -> np.ndarray:
    x = np.ascontiguousarray(x, np.float64)
    s = np.zeros(x.shape, np.int8)
    lib().orc_sign_spins(C.c_int64(x.size), _p(x), _p(s))
    return s


def best_replica(cut) -> int:
    cut = _c(cut, np.int64)
    return int(lib().orc_best_replica(C.c_int32(len(cut)), _p(cut)))


# ---------------------------------------------------------------------------------------------- O5
def read_vote(fr, spins) -> np.ndarray:
    fp, si, al, h1 = _c(fr.frag_ptr, np.int64), _c(fr.snp_idx, np.int32), _c(fr.allele, np.uint8), _c(fr.h1, np.uint8)
    s = _c(spins, np.int8)
    hap = np.zeros(fr.n_snp, np.int8)
    lib().orc_read_vote(C.c_int32(fr.n_frag), C.c_int32(fr.n_snp), _p(fp), _p(si), _p(al), _p(h1), _p(s), _p(hap))
    return hap


def snp_readout(h1, spins) -> np.ndarray:
    h1, s = _c(h1, np.uint8), _c(spins, np.int8)
    hap = np.zeros(len(s), np.int8)
    lib().orc_snp_readout(C.c_int32(len(s)), _p(h1), _p(s), _p(hap))
    return hap


def block_stitch(n, windows, block_spins) -> np.ndarray:
    win = _c(windows, np.int64)
    bs = _c(np.concatenate([np.asarray(b, np.int8) for b in block_spins]), np.int8)
    out = np.zeros(n, np.int8)
    lib().orc_block_stitch(C.c_int32(n), C.c_int32(len(win)), _p(win), _p(bs), _p(out))
    return out


def block_split(g, windows) -> dict:
    """Block-diagonal CSR of the sub-graphs induced by the index windows (SNP graph g with w_fx / w)."""
    rp, cl = _c(g["row_ptr"], np.int32), _c(g["col"], np.int32)
    wfx, w = _c(g.get("w_fx"), np.int64), _c(g.get("w"), np.float32)
    win = _c(windows, np.int64)
    nb = len(win)
    args = (C.c_int32(len(rp) - 1), _p(rp), _p(cl), _p(wfx), _p(w), C.c_int32(nb), _p(win))
    nnz = lib().orc_block_split(*args, None, None, None, None, C.c_int64(0))
    ntot = int((win[:, 1] - win[:, 0]).sum())
    orp, ocl = np.zeros(ntot + 1, np.int32), np.zeros(nnz, np.int32)
    owfx = np.zeros(nnz, np.int64) if wfx is not None else None
    ow = np.zeros(nnz, np.float32) if w is not None else None
    lib().orc_block_split(*args, _p(orp), _p(ocl), _p(owfx), _p(ow), C.c_int64(nnz))
    inst_ptr = np.concatenate([[0], np.cumsum(win[:, 1] - win[:, 0])]).astype(np.int32)
    return dict(n=ntot, nnz=int(nnz), row_ptr=orp, col=ocl, w_fx=owfx, w=ow, inst_ptr=inst_ptr)


def switch_hamming(hap1, truth) -> dict:
    """SE = switches/(n_phased-1); HE_raw = mismatches/n_phased in the given orientation
    (PAPER.md:L382); HE = min over the two orientations (reading R12)."""
    h, t = _c(hap1, np.int8), _c(truth, np.uint8)
    out = np.zeros(3, np.int64)
    lib().orc_switch_hamming(C.c_int32(len(h)), _p(h), _p(t), _p(out))
    sw, npz, mm = (int(v) for v in out)
    se = sw / (npz - 1) if npz > 1 else 0.0
    he_raw = mm / npz if npz > 0 else 0.0
    return dict(switches=sw, n_phased=npz, mismatches=mm, se=se, he_raw=he_raw, he=min(he_raw, 1.0 - he_raw))


# ------------------------------------------------------------------------------------------ helpers
def read_weights(g, weight_mode: int) -> np.ndarray:
    """Canonical integer read-graph weight: mode 0 w = D (paper Eq. 3), mode 1 w = D - C (BASELINE.json)."""
    return (g["d"].astype(np.int64) if weight_mode == 0 else g["d"].astype(np.int64) - g["c"].astype(np.int64))


def solve(row_ptr, col, w_int, jval, x0, y0, *, steps_total, dt=1.25, a0=1.0, c0=None, n_threads=1, force_mode=0,
          eval_every=0):
    """Full single-instance solve: bSB from fp32 x0,y0 -> spins, cuts, best replica.

    ``eval_every`` = k > 0 additionally returns ``trace``: the per-replica cuts of sign(x) after steps k, 2k, ... (what
    Fig. 3 plots as the minimum energy over the samples at every time step): int64 [n_evals][R], plus
    ``trace_steps`` (the number of steps completed at each evaluation).  The state is simply advanced k steps at a time."""
    x, y = x0.astype(np.float64), y0.astype(np.float64)
    trace, trace_steps = [], []
    if eval_every and eval_every > 0:
        k = 0
        while k + eval_every <= steps_total:
            x, y, c0 = bsb_run(row_ptr, col, jval, x, y, steps_total=steps_total, step_begin=k, steps_run=eval_every, dt=dt, a0=a0,
                               c0=c0, n_threads=n_threads, force_mode=force_mode)
            k += eval_every
            trace.append(cut_eval(row_ptr, col, w_int, sign_spins(x))[0]); trace_steps.append(k)
        if k < steps_total:
            x, y, c0 = bsb_run(row_ptr, col, jval, x, y, steps_total=steps_total, step_begin=k, dt=dt, a0=a0, c0=c0,
                               n_threads=n_threads, force_mode=force_mode)
    else:
        x, y, c0 = bsb_run(row_ptr, col, jval, x, y, steps_total=steps_total, dt=dt, a0=a0, c0=c0, n_threads=n_threads,
                           force_mode=force_mode)
    s = sign_spins(x)
    cut, en = cut_eval(row_ptr, col, w_int, s)
    r = best_replica(cut)
    out = dict(x=x, y=y, c0=c0, spins=s, cut=cut, energy=en, best_replica=r, best_cut=int(cut[r]),
               best_spins=s[:, r].copy())
    if trace:
        out["trace"] = np.stack(trace); out["trace_steps"] = np.array(trace_steps, np.int32)
    return out


# ---------------------------------------------------------------------------------------------- O6
# SNP-based iterative refinement, PAPER.md:L325-L338 [Eq. 15-17].  Plain numpy, in the paper's
# order.  Readings (R16): the termination test (cut <= 0, or one side empty) is made right after the solve and
# BEFORE the counter / weight update of that iteration; the smaller subset on a tie is the -1 side; every iteration
# starts bSB from a fresh seeded state handed in by the caller (the oracle draws no numbers).
def gauge_transform(row_ptr, col, w_fx, w, spins):
    """Eq. 15: w'_uv = -w_uv if s_u != s_v else w_uv, on the fixed-point and the fp32 weights alike (exact sign flips)."""
    rp, cl = _c(row_ptr, np.int32), _c(col, np.int32)
    s = _c(spins, np.int8).astype(np.int64)
    rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
    sg = s[rows] * s[cl]
    return (np.asarray(w_fx, np.int64) * sg).astype(np.int64), (np.asarray(w, np.float32) * sg.astype(np.float32)).astype(np.float32)


def smaller_subset(spins) -> np.ndarray:
    """Boolean mask of S_min (Eq. 16): the side with fewer vertices; the -1 side on a tie."""
    s = _c(spins, np.int8)
    n_pos, n_neg = int((s > 0).sum()), int((s < 0).sum())
    return (s > 0) if n_pos < n_neg else (s < 0)


def refine_snp(row_ptr, col, w_fx, w, init_states, *, steps_total, max_iter, dt=1.25, a0=1.0, n_threads=1):
    """Iterative refinement.  init_states(t) -> (x0, y0) fp32 [n][R] for iteration t = 0, 1, ...
    Returns dict(flip_count [n] int32, iterations (solves run), cuts (best cut of every solve), w_fx, w (final weights))."""
    rp, cl = _c(row_ptr, np.int32), _c(col, np.int32)
    wfx, wf = np.asarray(w_fx, np.int64).copy(), np.asarray(w, np.float32).copy()
    n = len(rp) - 1
    count = np.zeros(n, np.int32)
    cuts = []
    for t in range(max_iter):
        x0, y0 = init_states(t)
        res = solve(rp, cl, wfx, (-wf).astype(np.float32), x0, y0, steps_total=steps_total, dt=dt, a0=a0, n_threads=n_threads)
        s = res["best_spins"]
        cuts.append(int(res["best_cut"]))
        if res["best_cut"] <= 0 or abs(int(s.astype(np.int64).sum())) == n:      # L333: non-positive cut or a single subset
            break
        count[smaller_subset(s)] += 1                                          # Eq. 16
        wfx, wf = gauge_transform(rp, cl, wfx, wf, s)                          # Eq. 15
    return dict(flip_count=count, iterations=len(cuts), cuts=cuts, w_fx=wfx, w=wf)


def refine_readout(h1, flip_count) -> np.ndarray:
    """Eq. 17: H1'[u] = H1[u] if C(p_u) is even else H2[u] = 1 - H1[u]."""
    h = np.zeros(len(flip_count), np.uint8) if h1 is None else _c(h1, np.uint8)
    return np.where(np.asarray(flip_count) % 2 == 0, h, 1 - h).astype(np.int8)


# ---------------------------------------------------------------------------------------------- O7
# Connected components and per-component batching, PAPER.md:L248 ("each connected component ... independently"), L319
# (SURVEY.md 8(f) f2).  Canonical form (R14): components are numbered by their smallest vertex, vertices keep
# their ascending order inside a component, components with fewer than `min_size` vertices are dropped (singletons carry
# no phase information).  The library step is scipy's connected_components; the rest is index arithmetic.
def component_split(g: dict, min_size: int = 2) -> dict:
    """Block-diagonal CSR of the kept components + perm (new index -> old vertex) + inst_ptr."""
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import connected_components
    n = int(g["n"])
    rp, cl = _c(g["row_ptr"], np.int32), _c(g["col"], np.int32)
    A = csr_matrix((np.ones(len(cl), np.int8), cl, rp), shape=(n, n))
    _, lab = connected_components(A, directed=False)
    first = np.full(lab.max() + 1 if n else 0, n, np.int64)
    np.minimum.at(first, lab, np.arange(n))
    root = first[lab]                                   # canonical label = smallest vertex of the component
    size = np.bincount(root, minlength=n)[root] if n else np.zeros(0, np.int64)
    keep = size >= min_size
    order = np.lexsort((np.arange(n), root))            # by component (smallest vertex), then by vertex
    perm = order[keep[order]].astype(np.int32)
    inv = np.full(n, -1, np.int64)
    inv[perm] = np.arange(len(perm))
    roots_kept = root[perm]
    starts = np.flatnonzero(np.r_[True, roots_kept[1:] != roots_kept[:-1]]) if len(perm) else np.zeros(0, np.int64)
    inst_ptr = np.r_[starts, len(perm)].astype(np.int32)
    deg = (rp[1:] - rp[:-1])[perm]
    new_rp = np.r_[0, np.cumsum(deg)].astype(np.int32)
    idx = np.concatenate([np.arange(rp[v], rp[v + 1]) for v in perm]) if len(perm) else np.zeros(0, np.int64)
    out = dict(n=len(perm), nnz=int(new_rp[-1]), row_ptr=new_rp, col=inv[cl[idx]].astype(np.int32), perm=perm, inst_ptr=inst_ptr)
    for k in ("d", "c", "w_fx", "w"):
        if g.get(k) is not None:
            out[k] = np.asarray(g[k])[idx]
    return out


def component_merge(n: int, perm, comp_spins) -> np.ndarray:
    """Spins of the kept components back to the original vertices; dropped vertices get 0 (unphased)."""
    s = np.zeros(n, np.int8)
    s[np.asarray(perm)] = np.asarray(comp_spins, np.int8)
    return s
