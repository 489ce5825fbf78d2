"""`python -m paper_2603_25762_b200.selfcheck` -- one small invocation of every entry point and every bSB step path.

Meant to be run under `compute-sanitizer --tool memcheck | racecheck | synccheck` (see profiles/r2_sanitizer.md) and as a
quick installation check: small seeded inputs, a few steps each, no comparison against anything (the parity tests do that).
"""
from __future__ import annotations

import sys

import torch

from . import binding as B, synth


def main(steps: int = 6) -> int:
    assert torch.cuda.is_available(), "selfcheck needs a CUDA device (no CPU fallback)"
    done = []

    def ok(name):
        torch.cuda.synchronize()
        done.append(name)

    # read graph, tiny (cfg0): resident path, CSR path, dense full GEMM, tile_skip, block path
    fr, p = synth.make_config(0)
    dfr = B.upload_frags(fr)
    g, J = B.qhap_build_read_graph(dfr, weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
    ok("build_read_graph")
    for path, kw in ((3, {}), (2, {}), (1, dict(tile_skip=0)), (1, dict(tile_skip=1)), (4, {}), (2, dict(force_mode=1)), (1, dict(tile_skip=1, force_mode=1))):
        res = B.qhap_bsb_solve(g, replicas=p["R"], steps_total=p["T"], steps_run=steps, seed=1, weight_mode=1, path=path, dense_J=J if path == 1 else None, **kw)
        ok(f"solve cfg0 path {path} {kw}")
    B.qhap_phase_readout_reads(dfr, res["best_spins"]); ok("readout_reads")
    B.qhap_cut_eval(g, 1, torch.ones((fr.n_frag, 5), dtype=torch.int8, device="cuda")); ok("cut_eval")
    B.qhap_component_split(g, 2); ok("component_split")
    # read graph with several tiles per CTA: fused launch (two waves), per-step launches, state16 off, eval_every
    fr, p = synth.make_config(1, scale=0.05)
    g, J = B.qhap_build_read_graph(B.upload_frags(fr), weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
    for path, kw in ((1, dict(tile_skip=1)), (1, dict(tile_skip=1, step_launch=1)), (4, {}), (4, dict(state16=2)), (1, dict(tile_skip=1, eval_every=3))):
        B.qhap_bsb_solve(g, replicas=264, steps_total=p["T"], steps_run=steps, seed=2, weight_mode=1, path=path, dense_J=J if path == 1 else None, **kw)
        ok(f"solve cfg1-scaled path {path} {kw}")
    # paired tiles (two boxes per N = 128 accumulator): active from two boxes per CTA on -- 38 boxes x 8 replica tiles
    fr, p = synth.make_config(1, scale=0.3)
    g, J = B.qhap_build_read_graph(B.upload_frags(fr), weight_mode=1, dense_dtype=B.QHAP_DENSE_FP16)
    for kw in (dict(), dict(step_launch=1), dict(pair_tiles=2), dict(y_ring=1)):
        B.qhap_bsb_solve(g, replicas=1024, steps_total=p["T"], steps_run=steps, seed=2, weight_mode=1, path=1, tile_skip=1, dense_J=J, **kw)
        ok(f"solve cfg1-scaled paired tiles {kw}")
    B.qhap_cut_eval_static(g, 1, torch.ones((g.n, 300), dtype=torch.int8, device="cuda")); ok("cut_eval_static")
    # SNP graph: build (both depths), block split, batched block path and CSR path, stitch, SNP readout
    fr, p = synth.make_config(3, scale=0.005)
    d3 = B.upload_frags(fr)
    g3 = B.qhap_build_snp_graph(d3, 10, 0.1)
    g3 = B.qhap_build_snp_graph(d3, 3, 0.1); ok("build_snp_graph")
    win = synth.block_windows(fr.n_snp, 300, 250)
    bs = B.qhap_block_split(g3, win); ok("block_split")
    for path in (4, 2):
        res = B.qhap_bsb_solve(bs, replicas=64, steps_total=200, steps_run=steps, seed=3, weight_mode=2, path=path)
        ok(f"solve cfg3-scaled batched path {path}")
    st = B.qhap_block_stitch(fr.n_snp, win, res["best_spins"]); ok("block_stitch")
    B.qhap_phase_readout_snps(d3.h1, st); ok("readout_snps")
    # Pore-C graph: hybrid block path (tiles + remainder CSR), refinement loop
    fr, p = synth.make_config(4, scale=0.01)
    g4 = B.qhap_build_snp_graph(B.upload_frags(fr), 3, 0.1)
    B.qhap_bsb_solve(g4, replicas=128, steps_total=200, steps_run=steps, seed=4, weight_mode=2, path=4); ok("solve cfg4-scaled hybrid")
    B.qhap_snp_refine(g4, replicas=32, steps_total=steps, max_iter=2, seed=4, path=2); ok("snp_refine")
    print(f"selfcheck: {len(done)} invocations OK ({B.qhap_version()})")
    return 0


if __name__ == "__main__":
    sys.exit(main(int(sys.argv[1]) if len(sys.argv) > 1 else 6))
