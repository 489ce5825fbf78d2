"""GPU tests added in round 2: the workspace contract (exact sizes, guard bands), the dSB force mode (SURVEY 8(f) f4,
PAPER.md:L71-L77) and the eval_every trace on every step path, against the CPU oracle."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2603_25762_b200 import synth

pytestmark = pytest.mark.gpu

GUARD = 1 << 16          # bytes of canary behind every workspace
CANARY = 0xA5


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests selected (-m gpu) but no CUDA device is visible"
    from paper_2603_25762_b200 import binding
    return binding


@pytest.fixture()
def guarded(B, monkeypatch):
    """Every workspace the binding allocates gets EXACTLY the size the library asked for, followed by a canary band that
    must come back untouched (a carve that walks past the size the query reported)."""
    import torch
    made = []

    def alloc(nbytes):
        n = max(int(nbytes), 256)
        n_al = (n + 255) // 256 * 256
        buf = torch.full((n_al + GUARD,), CANARY, dtype=torch.uint8, device="cuda")
        made.append((buf, n_al))
        return buf[:n]
    monkeypatch.setattr(B, "_workspace", alloc)

    def check():
        torch.cuda.synchronize()
        assert made, "no workspace was allocated"
        for buf, n in made:
            tail = buf[n:]
            assert bool((tail == CANARY).all()), f"workspace of {n} bytes: the guard band behind it was written"
        return len(made)
    return check


def test_workspace_guard_bands_every_entry_point(B, oracle, guarded):
    """Graph builds, block split, component split / merge, refinement pieces, read-out, cut evaluation and the bSB solve on
    paths 1-4 (fused and per-step, with and without a remainder CSR) run inside workspaces of exactly the queried size."""
    import torch
    fr, p = synth.make_config(1, scale=0.1)
    dfr = B.upload_frags(fr)
    g, J = B.qhap_build_read_graph(dfr, weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
    for path, kw in ((1, dict(tile_skip=1)), (1, dict(tile_skip=0)), (1, dict(tile_skip=1, step_launch=1)), (2, {}), (4, {}), (4, dict(step_launch=1)),
                     (4, dict(state16=2))):
        res = B.qhap_bsb_solve(g, replicas=256, steps_total=p["T"], steps_run=12, seed=3, weight_mode=1, path=path, dense_J=J if path == 1 else None, **kw)
        assert int(res["best_cut"].cpu()[0]) > 0
    fr0, p0 = synth.make_config(0)
    g0, _ = B.qhap_build_read_graph(B.upload_frags(fr0), weight_mode=1)
    B.qhap_bsb_solve(g0, replicas=64, steps_total=50, seed=1, weight_mode=1, path=3)
    hap = B.qhap_phase_readout_reads(B.upload_frags(fr0), torch.ones(fr0.n_frag, dtype=torch.int8, device="cuda"))
    assert hap.numel() == fr0.n_snp
    B.qhap_cut_eval(g0, 1, torch.ones((fr0.n_frag, 8), dtype=torch.int8, device="cuda"))
    B.qhap_component_split(g0, 2)
    # SNP graph, blocks, hybrid path with a remainder CSR (Pore-C long-range edges)
    fr3, p3 = synth.make_config(3, scale=0.01)
    d3 = B.upload_frags(fr3)
    for tenths in (3, 10):
        g3 = B.qhap_build_snp_graph(d3, tenths, 0.1)
    win = synth.block_windows(fr3.n_snp, 500, 450)
    bs = B.qhap_block_split(g3, win)
    res = B.qhap_bsb_solve(bs, replicas=64, steps_total=100, seed=5, weight_mode=2, path=4)
    B.qhap_block_stitch(fr3.n_snp, win, res["best_spins"])
    B.qhap_bsb_solve(bs, replicas=64, steps_total=100, seed=5, weight_mode=2, path=2)
    fr4, p4 = synth.make_config(4, scale=0.02)
    g4 = B.qhap_build_snp_graph(B.upload_frags(fr4), 3, 0.1)
    B.qhap_bsb_solve(g4, replicas=128, steps_total=60, seed=5, weight_mode=2, path=4)
    B.qhap_snp_refine(g4, replicas=32, steps_total=60, max_iter=2, seed=5, path=4)
    B.qhap_flip_count_update(torch.ones(g4.n, dtype=torch.int8, device="cuda"), torch.zeros(g4.n, dtype=torch.int32, device="cuda"))
    B.qhap_component_split(g4, 2)
    assert guarded() >= 20


def test_workspace_one_byte_short_is_refused(B, oracle):
    """Every path reports the size it needs and refuses a workspace one byte short with QHAP_ERR_WORKSPACE (no partial run)."""
    import ctypes as C
    import torch
    fr, p = synth.make_config(1, scale=0.1)
    g, J = B.qhap_build_read_graph(B.upload_frags(fr), weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
    for path in (1, 2, 4):
        res = B.qhap_bsb_solve(g, replicas=128, steps_total=50, steps_run=2, seed=1, weight_mode=1, path=path, dense_J=J if path == 1 else None, tile_skip=1)
        need = res["workspace"].numel()
        with pytest.raises(B.QhapError) as ei:
            B.qhap_bsb_solve(g, replicas=128, steps_total=50, steps_run=2, seed=1, weight_mode=1, path=path, dense_J=J if path == 1 else None, tile_skip=1,
                             workspace=res["workspace"], workspace_bytes=need - 1)
        assert ei.value.status == B.QHAP_ERR_WORKSPACE


# ------------------------------------------------------------------------------------------------ dSB (force_mode 1)
def _dsb_case(B, oracle, name):
    if name == "cfg0":
        fr, p = synth.make_config(0)
        g = oracle.read_graph(fr); w = oracle.read_weights(g, 1); mode = 1
        dg, J = B.qhap_build_read_graph(B.upload_frags(fr), weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
        return g, w, (-w).astype(np.float32), mode, dg, J, fr.n_frag, p, None
    if name == "cfg1-scaled":
        fr, p = synth.make_config(1, scale=0.1)
        g = oracle.read_graph(fr); w = oracle.read_weights(g, 1); mode = 1
        dg, J = B.qhap_build_read_graph(B.upload_frags(fr), weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
        return g, w, (-w).astype(np.float32), mode, dg, J, fr.n_frag, p, None
    fr, p = synth.make_config(3, scale=0.01)
    g0 = oracle.snp_graph(fr, 3, 0.1)
    g = oracle.block_split(g0, synth.block_windows(fr.n_snp, 500, 450))
    return g, g["w_fx"], (-g["w"]).astype(np.float32), 2, B.upload_csr(g), None, g["n"], p, g["inst_ptr"]


@pytest.mark.parametrize("name,R", [("cfg0", 48), ("cfg1-scaled", 136), ("cfg3-scaled", 256)])
def test_dsb_one_step_from_identical_states_every_path(B, oracle, name, R):
    """dSB, F = J sgn(x): from the SAME fp32 state the force of every path is an exactly representable integer combination
    (read graphs: exact on the tensor cores, so the step must agree with the fp64 oracle to fp32 rounding, 1e-6; SNP graphs:
    fp32 weights, 1e-5 as VERDICT r1 asks), at several points of a trajectory that has walls and sign changes."""
    import torch
    g, w_int, jval, mode, dg, J, n, p, inst_ptr = _dsb_case(B, oracle, name)
    T = p["T"]
    x0, y0 = synth.bsb_init_state(11, n, R)
    bounds = [(0, n)] if inst_ptr is None else [(int(inst_ptr[b]), int(inst_ptr[b + 1])) for b in range(len(inst_ptr) - 1)]

    def orc(x, y, k, steps):
        x, y = x.copy(), y.copy()
        for lo, hi in bounds:
            rp = (g["row_ptr"][lo:hi + 1] - g["row_ptr"][lo]).astype(np.int32)
            e = slice(int(g["row_ptr"][lo]), int(g["row_ptr"][hi]))
            xs, ys = x[lo:hi].copy(), y[lo:hi].copy()
            oracle.bsb_run(rp, (g["col"][e] - lo).astype(np.int32), jval[e], xs, ys, steps_total=T, step_begin=k, steps_run=steps, n_threads=8, force_mode=1)
            x[lo:hi], y[lo:hi] = xs, ys
        return x, y
    xo, yo = x0.astype(np.float64), y0.astype(np.float64)
    tol = 1e-6 if mode == 1 else 1e-5
    paths = [(2, {}), (4, {}), (4, {"step_launch": 1})] + ([(1, {"tile_skip": 1}), (1, {"tile_skip": 0})] if J is not None else []) + \
        ([(3, {})] if n * R <= 65536 else [])
    k = 0
    for seg in (1, 7, 12, 30):                       # compare ONE step at k = 0, 1, 8, 20, 50 (free-running oracle in between)
        x32, y32 = xo.astype(np.float32), yo.astype(np.float32)
        xr, yr = orc(x32.astype(np.float64), y32.astype(np.float64), k, 1)
        for path, kw in paths:
            xg, yg = torch.from_numpy(x32.copy()).cuda(), torch.from_numpy(y32.copy()).cuda()
            B.qhap_bsb_solve(dg, replicas=R, steps_total=T, step_begin=k, steps_run=1, weight_mode=mode, path=path, dense_J=J if path == 1 else None,
                             force_mode=1, x=xg, y=yg, finalize=False, **kw)
            dx = np.abs(xg.cpu().numpy() - xr).max(); dy = np.abs(yg.cpu().numpy() - yr).max()
            assert dx <= tol and dy <= tol, (name, path, kw, k, dx, dy)
        xo, yo = orc(xo, yo, k, seg)
        k += seg
    assert np.any(np.abs(xo) == 1.0)                 # walls were reached
    # dSB differs from bSB on the same state (the flag reaches the kernels)
    xg, yg = torch.from_numpy(x32.copy()).cuda(), torch.from_numpy(y32.copy()).cuda()
    B.qhap_bsb_solve(dg, replicas=R, steps_total=T, step_begin=k - seg, steps_run=1, weight_mode=mode, path=2, force_mode=0, x=xg, y=yg, finalize=False)
    assert np.abs(yg.cpu().numpy() - yr).max() > 1e-3


def test_dsb_multi_step_paths_agree_and_solve_quality(B, oracle):
    """Integer read graph: the dSB force is exact on every path, so 25 steps in one call give the SAME bits on the CSR,
    resident, dense (fused and per-step) and block paths; and a full dSB solve reaches the oracle's dSB cut - 0.5 %."""
    import torch
    g, w, jval, mode, dg, J, n, p, _ = _dsb_case(B, oracle, "cfg0")
    R, T = p["R"], p["T"]
    outs = []
    for path, kw in ((2, {}), (3, {}), (1, {"tile_skip": 1}), (1, {"tile_skip": 1, "step_launch": 1}), (4, {})):
        res = B.qhap_bsb_solve(dg, replicas=R, steps_total=T, steps_run=25, seed=p["seed"], weight_mode=1, path=path, dense_J=J if path == 1 else None,
                               force_mode=1, finalize=False, **kw)
        outs.append((res["x"].cpu().numpy(), res["y"].cpu().numpy()))
    for o in outs[1:]:
        # same fp32 operations up to the order of an exact integer sum: identical
        assert np.array_equal(o[0], outs[0][0]) and np.array_equal(o[1], outs[0][1])
    x0, y0 = synth.bsb_init_state(p["seed"], n, R)
    ores = oracle.solve(g["row_ptr"], g["col"], w, jval, x0, y0, steps_total=T, n_threads=8, force_mode=1)
    for path in (2, 1, 4):
        res = B.qhap_bsb_solve(dg, replicas=R, steps_total=T, seed=p["seed"], weight_mode=1, path=path, dense_J=J if path == 1 else None, tile_skip=1, force_mode=1)
        gcut = int(res["best_cut"].cpu()[0])
        assert gcut >= ores["best_cut"] - 0.005 * abs(ores["best_cut"]), (path, gcut, ores["best_cut"])
        ccut, _ = oracle.cut_eval(g["row_ptr"], g["col"], w, res["best_spins"].cpu().numpy())
        assert ccut[0] == gcut


# ------------------------------------------------------------------------------------------------------- eval_every
@pytest.mark.parametrize("path", [2, 3, 1, 4])
def test_eval_every_trace(B, oracle, path):
    """eval_every = k: row j of the trace is the cut of sgn(x) after (j + 1) k steps -- bit-exact against the oracle's cut
    evaluation of the GPU state taken at those steps by separate resumed calls, and the run with a trace ends in the same
    state and cuts as the run without one (Fig. 3: best sample per time step)."""
    import torch
    g, w, jval, mode, dg, J, n, p, _ = _dsb_case(B, oracle, "cfg0")
    R, T, k = 48, 200, 30
    kw = dict(replicas=R, steps_total=T, weight_mode=1, path=path, dense_J=J if path == 1 else None, tile_skip=1)
    res = B.qhap_bsb_solve(dg, seed=4, steps_run=100, eval_every=k, trace_cuts=True, **kw)
    ref = B.qhap_bsb_solve(dg, seed=4, steps_run=100, **kw)
    assert torch.equal(res["x"], ref["x"]) and torch.equal(res["y"], ref["y"]) and torch.equal(res["cut"], ref["cut"])
    assert res["trace_cut"].shape == (3, 1, R) and res["trace_best_cut"].shape == (3, 1)
    x0, y0 = synth.bsb_init_state(4, n, R)
    xg, yg = torch.from_numpy(x0.copy()).cuda(), torch.from_numpy(y0.copy()).cuda()
    for j in range(3):
        B.qhap_bsb_solve(dg, step_begin=j * k, steps_run=k, x=xg, y=yg, finalize=False, **kw)
        s = np.where(xg.cpu().numpy() >= 0, 1, -1).astype(np.int8)
        ecut, _ = oracle.cut_eval(g["row_ptr"], g["col"], w, s)
        assert np.array_equal(res["trace_cut"][j, 0].cpu().numpy(), ecut)
        assert int(res["trace_best_cut"][j, 0].cpu()) == int(ecut.max())
    # against the oracle's own trace: the best cut per evaluation within 0.5 % (same seeds, same replica count)
    ores = oracle.solve(g["row_ptr"], g["col"], w, jval, x0, y0, steps_total=T, n_threads=4, eval_every=k)
    for j in range(3):
        ob = int(ores["trace"][j].max())
        assert int(res["trace_best_cut"][j, 0].cpu()) >= ob - 0.005 * abs(ob) - 1


def test_read_graph_single_call_with_capacity_hint(B, oracle):
    """qhap.h capacity protocol: with edge arrays of sufficient capacity ONE call counts, scans and fills; a hint that is too
    small falls back to count -> allocate -> fill.  Same graph and dense J, bit for bit."""
    import torch
    fr, _ = synth.make_config(1, scale=0.1)
    dfr = B.upload_frags(fr)
    exp = oracle.read_graph(fr)
    ref, Jref = B.qhap_build_read_graph(dfr, weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
    for hint in (exp["nnz"] + 1000, exp["nnz"], 17):
        g, J = B.qhap_build_read_graph(dfr, weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16, capacity_hint=hint)
        h = g.to_host()
        assert h["nnz"] == exp["nnz"]
        for k in ("row_ptr", "col", "d", "c"):
            assert np.array_equal(h[k], exp[k]), (hint, k)
        assert torch.equal(J, Jref)


# ---------------------------------------------------------- block path with exactly as many tiles as the tile arrays hold
@pytest.mark.parametrize("extra_tile", [0, 1])
def test_block_path_at_exact_tile_capacity(B, oracle, guarded, extra_tile):
    """The block path's tile arrays hold 16 nnz / 4096 + ceil(n / 64) + 1 tiles of 64 x 64.  A graph whose non-empty tiles number
    EXACTLY that capacity (extra_tile = 0) keeps every tile; one tile more (extra_tile = 1) no longer fits, the threshold rises
    and every entry goes to the remainder CSR.  Both run inside a guarded workspace of exactly the queried size and follow the
    fp64 oracle over 10 steps; cuts of the final signs are exact."""
    import torch
    T_rows, n = 6, 6 * 64
    edges = []

    def inside(tr, tc, k):                       # k edges from tile row tr into tile column tc (distinct rows and columns)
        for i in range(k):
            a, b = tr * 64 + 3 + 5 * i, tc * 64 + 40 + 4 * i
            edges.append((min(a, b), max(a, b)))
    for t in range(4):
        inside(t, t, 3)                          # four diagonal tiles
    inside(4, 5, 3)                              # tiles (4, 5) and (5, 4)
    inside(4, 4, 2)                              # seventh tile
    if extra_tile:
        inside(5, 5, 2)                          # eighth tile: one more than the capacity
    edges = sorted(set(edges))
    rng = np.random.default_rng(5)
    wd = rng.integers(1, 9, len(edges)); wc = rng.integers(0, 5, len(edges))
    rows = np.array([e[0] for e in edges] + [e[1] for e in edges]); cols = np.array([e[1] for e in edges] + [e[0] for e in edges])
    d2 = np.concatenate([wd, wd]).astype(np.int32); c2 = np.concatenate([wc, wc]).astype(np.int32)
    order = np.lexsort((cols, rows))
    rows, cols, d2, c2 = rows[order], cols[order].astype(np.int32), d2[order], c2[order]
    row_ptr = np.zeros(n + 1, np.int64); np.add.at(row_ptr, rows + 1, 1); row_ptr = np.cumsum(row_ptr).astype(np.int32)
    nnz = len(cols)
    tiles = {(int(a) // 64, int(b) // 64) for a, b in zip(rows, cols)}
    n_tiles = len(tiles) + sum(1 for t in range(T_rows) if not any(tt[0] == t for tt in tiles))      # + a forced tile per empty tile row
    cap = 16 * nnz // 4096 + T_rows + 1
    assert n_tiles == cap + extra_tile, (n_tiles, cap)
    g = B.Csr(n, nnz, torch.from_numpy(row_ptr).cuda(), torch.from_numpy(cols).cuda(), torch.from_numpy(d2).cuda(), torch.from_numpy(c2).cuda())
    w = (d2 - c2).astype(np.int64)
    R, T = 64, 200
    x0, y0 = synth.bsb_init_state(9, n, R)
    outs = {}
    for path in (4, 2):
        xg, yg = torch.from_numpy(x0.copy()).cuda(), torch.from_numpy(y0.copy()).cuda()
        res = B.qhap_bsb_solve(g, replicas=R, steps_total=T, steps_run=10, weight_mode=1, path=path, x=xg, y=yg)
        outs[path] = (xg.cpu().numpy(), yg.cpu().numpy(), res)
    xo, yo = x0.astype(np.float64), y0.astype(np.float64)
    oracle.bsb_run(row_ptr, cols, (-w).astype(np.float32), xo, yo, steps_total=T, step_begin=0, steps_run=10, n_threads=4)
    for path in (4, 2):
        dx = np.abs(outs[path][0] - xo).max(); dy = np.abs(outs[path][1] - yo).max()
        assert dx <= 1e-3 and dy <= 1e-3, (path, extra_tile, dx, dy)
        res = outs[path][2]
        ccut, _ = oracle.cut_eval(row_ptr, cols, w, res["best_spins"].cpu().numpy())
        assert int(ccut[0]) == int(res["best_cut"].cpu()[0])
    assert guarded() >= 2


# ------------------------------------------------------------------------------ paired tiles: same bits
@pytest.mark.parametrize("shape", ["all-pairs-ragged", "pairs-and-singles", "three-boxes-per-cta"])
def test_paired_tiles_are_bit_identical_to_single_boxes(B, oracle, shape):
    """pair_tiles = 1 (two neighbouring 64-spin boxes share one N = 128 accumulator where that keeps the CTAs balanced) against
    pair_tiles = 2 (every box on its own): a k-block that only one box of a pair lists contributes exact zeros to the other, so
    every bit must agree -- fused launch and one launch per step, y through the ring and by plain loads, odd step counts, resume.
    Shapes (148 CTAs): 36 boxes x 16 replica tiles -> every box is in a pair and the ragged last box (10 spins) is the RIGHT
    half of one; 38 boxes x 8 replica tiles -> 18 pairs + 2 single boxes per replica tile; 38 boxes x 16 replica tiles -> every CTA
    has at least three boxes per step, so the fused launch reloads its staging buffers early.  Against the CSR
    path within 1e-3."""
    import torch
    scale, R = {"all-pairs-ragged": (0.28125, 2048), "pairs-and-singles": (0.3, 1024), "three-boxes-per-cta": (0.3, 2048)}[shape]
    fr, pp = synth.make_config(1, scale=scale)
    g, J = B.qhap_build_read_graph(B.upload_frags(fr), weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
    n, T = g.n, pp["T"]
    boxes = (n + 63) // 64
    assert (boxes, n % 64 != 0) == ((36, True) if shape == "all-pairs-ragged" else (38, True)), (n, boxes)
    plan = B.qhap_plan_pair_tiles(boxes, (R + 127) // 128, 148, 2)
    assert plan[0] > 0 and (plan[2] >= 3) == (shape == "three-boxes-per-cta"), plan
    x0, y0 = synth.bsb_init_state(17, n, R)

    def run(path=1, **knobs):
        xg, yg = torch.from_numpy(x0.copy()).cuda(), torch.from_numpy(y0.copy()).cuda()
        kw = dict(replicas=R, steps_total=T, weight_mode=1, path=path, dense_J=J if path == 1 else None, tile_skip=1 if path == 1 else 0,
                  finalize=False, x=xg, y=yg, **knobs)
        B.qhap_bsb_solve(g, step_begin=0, steps_run=9, **kw)
        first = (xg.cpu().numpy(), yg.cpu().numpy())
        B.qhap_bsb_solve(g, step_begin=9, steps_run=6, **kw)
        return first, (xg.cpu().numpy(), yg.cpu().numpy())

    ref = run(pair_tiles=2, step_launch=1)
    for knobs in (dict(pair_tiles=1), dict(pair_tiles=1, step_launch=1), dict(pair_tiles=1, y_ring=1), dict(pair_tiles=1, y_ring=1, step_launch=1),
                  dict(pair_tiles=2), dict(),
                  # the block path on the same read graph (tiles built from the CSR; pairs carry per-box tiles and a zero tile)
                  dict(path=4), dict(path=4, step_launch=1), dict(path=4, pair_tiles=2), dict(path=4, y_ring=1)):
        got = run(**knobs)
        for a, b in zip(ref, got):
            assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]), (shape, knobs)
    # against the CSR path after the first 9 steps (all replicas), against the fp64 oracle after all 15 on sampled replicas (walls
    # are hit from step 3 on here, so single marginal wall decisions separate fp32 trajectories of different kernels later on)
    csr = run(path=2)
    dx = np.abs(ref[0][0] - csr[0][0]).max(); dy = np.abs(ref[0][1] - csr[0][1]).max()
    og = oracle.read_graph(fr)
    sample = np.array([0, 5, R // 3, R - 1])
    xo, yo = np.ascontiguousarray(x0[:, sample], np.float64), np.ascontiguousarray(y0[:, sample], np.float64)
    oracle.bsb_run(og["row_ptr"].astype(np.int32), og["col"].astype(np.int32), (-oracle.read_weights(og, 1)).astype(np.float32), xo, yo,
                   steps_total=T, step_begin=0, steps_run=15, n_threads=8)
    ox = np.abs(ref[1][0][:, sample] - xo).max(); oy = np.abs(ref[1][1][:, sample] - yo).max()
    print(f"paired tiles {shape}: n {n} R {R}: 9 steps against the CSR path max|dx| {dx:.2e} max|dy| {dy:.2e}; 15 steps against the oracle "
          f"(4 replicas) {ox:.2e} {oy:.2e}")
    assert dx <= 1e-3 and dy <= 1e-3 and ox <= 1e-3 and oy <= 1e-3


# ----------------------------------------------- whole solves at full size: same bits whatever the launch mode, run after run
@pytest.mark.parametrize("cfg", [1, 2])
def test_full_size_solves_bit_identical_across_launch_modes(B, cfg):
    """BASELINE configs 1 and 2 at full size, all 2,000 / 3,000 steps: the automatic setting (one fused cooperative launch, paired
    tiles, y by plain loads, early staging reload) three times in a row, then one launch per step, single boxes, and single boxes
    with the y ring -- final x, y, best cut and best replica agree bit for bit (a race in the tile-level step boundary of the
    fused launch would show up here as a run-to-run difference)."""
    import hashlib
    import torch
    fr, p = synth.make_config(cfg)
    g, J = B.qhap_build_read_graph(B.upload_frags(fr), weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
    seen = []
    for kw in (dict(), dict(), dict(), dict(step_launch=1), dict(pair_tiles=2), dict(pair_tiles=2, y_ring=1)):
        r = B.qhap_bsb_solve(g, replicas=p["R"], steps_total=p["T"], seed=p["seed"], weight_mode=1, path=1, dense_J=J, tile_skip=1, **kw)
        torch.cuda.synchronize()
        h = hashlib.sha1(r["x"].cpu().numpy().tobytes() + r["y"].cpu().numpy().tobytes()).hexdigest()
        seen.append((h, int(r["best_cut"][0]), int(r["best_replica"][0])))
    assert len(set(seen)) == 1, seen


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_snp_solves_repeat_bit_identically(B, cfg):
    """BASELINE configs 3 (47 SNP blocks, block path) and 4 (Pore-C SNP graph, hybrid path with state16 next to the remainder
    CSR) at full size, 300 steps: repeated runs agree bit for bit, and on config 3 so does the y ring against plain loads."""
    import hashlib
    import torch
    fr, p = synth.make_config(cfg)
    g = B.qhap_build_snp_graph(B.upload_frags(fr), p.get("linkage_tenths", 10), p.get("alpha", 0.1))
    if "block" in p:
        g = B.qhap_block_split(g, synth.block_windows(fr.n_snp, p["block"], p["stride"]))
    seen = []
    for kw in (dict(), dict()) + ((dict(y_ring=1),) if cfg == 3 else ()):
        r = B.qhap_bsb_solve(g, replicas=p["R"], steps_total=p["T"], steps_run=300, seed=p["seed"], weight_mode=2, path=4, **kw)
        torch.cuda.synchronize()
        seen.append((hashlib.sha1(r["x"].cpu().numpy().tobytes() + r["y"].cpu().numpy().tobytes()).hexdigest(),
                     tuple(r["best_cut"].cpu().tolist())))
    assert len(set(seen)) == 1, [s[0] for s in seen]
