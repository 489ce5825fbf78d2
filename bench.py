#!/usr/bin/env python
"""bench.py -- QHap hot path on B200: bSB spin-updates/s and phasing wall-time per region (BASELINE.json `metric`).

A "step" is one pass of the whole hot path over one synthetic region:
  qhap_build_read_graph -> qhap_bsb_solve (T bSB steps x R replicas, cut evaluation, best replica) -> qhap_phase_readout_reads
on BASELINE.json config 1 (read-based MHC-like region: ~8,000 HiFi-like reads, R = 1,024, T = 2,000) by default.
`value` = n * R * T * n_gpus / seconds per step with the fragments already resident in HBM; `e2e` is the same call
sequence fed from pinned HOST buffers (H2D of the fragment matrix and D2H of the haplotype + best cut inside the timed
region).  N > 1 (torchrun, or `--gpus N` from a plain shell, which re-executes itself under torchrun): every rank runs its
own R replicas of the same region (weak scaling; `--scaling strong` splits ONE seed's R replicas instead), no per-step
exchange, then 8 bytes per rank are all-gathered to pick the global best replica (paper_2603_25762_b200/parallel.py).

`--config 3` / `--config 4` (not the default; extra measurements of the sparse CSR step) run the SNP-based path instead:
  qhap_build_snp_graph -> [qhap_block_split] -> qhap_bsb_solve (CSR) -> [qhap_block_stitch] -> qhap_phase_readout_snps.

`--impl reference` times the fp64 CPU oracle (oracle/, test infrastructure) on the box's host cores on a bounded sample
of the same workload -- a reported baseline, not the target.

Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "bsb_spin_updates_per_s"
UNIT = "spin-updates/s"
L2_FLUSH_BYTES = 512 << 20


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (1 = the config the metric is quoted on)")
    ap.add_argument("--path", default="auto", choices=["auto", "dense", "dense-full", "sparse", "block"],
                    help="bSB step kernel: dense = tcgen05 tiles over the non-zero k-blocks of J (tile_skip, bit-identical to "
                         "dense-full = the whole N x N GEMM); sparse = CSR; auto = dense")
    ap.add_argument("--step-launch", type=int, default=0, choices=[0, 1],
                    help="tcgen05 paths: 0 = one launch runs all T steps where the tiles allow (tile-level dependencies between "
                         "steps), 1 = one launch per step; same bits")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU seconds of the oracle sample")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1 on single-instance configs: weak = every rank runs R replicas from its own seed; strong = ONE seed's R "
                         "replicas are split into contiguous slices (SURVEY 8(e)); config 3 always shards its blocks (strong)")
    ap.add_argument("--linkage-tenths", type=int, default=0,
                    help="SNP configs: linkage depth k/10 of the graph build (0 = the config's own, 3; 10 = the paper's exhaustive setting, PAPER.md:L114)")
    ap.add_argument("--porec-edges", type=int, default=0,
                    help="read configs: add Pore-C multi-contact fragments until this many long-range SNP pairs exist (non-banded read graph, SURVEY 8(f) f3)")
    ap.add_argument("--refine-iters", type=int, default=0,
                    help="SNP configs with one instance (config 4): also time qhap_snp_refine (Eq. 15-17) with at most this many solves")
    return ap.parse_args()


def workload_name(cfg, fr, p):
    return (f"BASELINE.json configs[{cfg}] {p['name']}: {fr.n_frag} fragments x {fr.n_snp} het SNPs, "
            f"{p['graph']} graph, R={p['R']}, T={p['T']}, dt={p['dt']}, a0={p['a0']}")


# ---------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_id: str):
        self.proc = None
        self.gpu_id = gpu_id

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", self.gpu_id, f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        d = json.loads(f.read_text())
        return dict(hbm=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]), bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    which="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, which="fallback (B200_PROFILING.md)")


# ------------------------------------------------------------------------------------------ reference arm
def oracle_sample(fr, p, cores, cpu_seconds, R_o=None):
    """One pass of the path in the fp64 oracle on a bounded sample: full graph build + R_o replicas x T_o steps + cut +
    vote.  Returns timings; T_o is sized from a 2-step probe so that the bSB part takes about `cpu_seconds`."""
    from oracle import oracle as O
    mode = 1
    t0 = time.perf_counter()
    if p["graph"] == "read":
        g = O.read_graph(fr)
        w_int = O.read_weights(g, mode)
        jval = (-w_int).astype(np.float32)
    else:
        g = O.snp_graph(fr, p.get("linkage_tenths", 10), p.get("alpha", 0.1))
        w_int = g["w_fx"]
        jval = (-g["w"]).astype(np.float32)
    t_build = time.perf_counter() - t0
    n = g["n"]
    R_o = R_o or min(p["R"], 16 * cores)
    from paper_2603_25762_b200 import synth
    x0, y0 = synth.bsb_init_state(p["seed"], n, R_o)
    x, y = x0.astype(np.float64), y0.astype(np.float64)
    t0 = time.perf_counter()
    O.bsb_run(g["row_ptr"], g["col"], jval, x, y, steps_total=p["T"], step_begin=0, steps_run=2, n_threads=cores)
    probe = (time.perf_counter() - t0) / 2
    T_o = int(max(4, min(p["T"] - 2, cpu_seconds / max(probe, 1e-6))))
    t0 = time.perf_counter()
    x, y, _ = O.bsb_run(g["row_ptr"], g["col"], jval, x, y, steps_total=p["T"], step_begin=2, steps_run=T_o, n_threads=cores)
    t_bsb = time.perf_counter() - t0
    t0 = time.perf_counter()
    s = O.sign_spins(x)
    cut, _ = O.cut_eval(g["row_ptr"], g["col"], w_int, s)
    r = O.best_replica(cut)
    if p["graph"] == "read":
        O.read_vote(fr, s[:, r].copy())
    else:
        O.snp_readout(fr.h1, s[:, r].copy())
    t_read = time.perf_counter() - t0
    return dict(n=n, R_o=R_o, T_o=T_o, t_build=t_build, t_bsb=t_bsb, t_read=t_read, edges=int(g["nnz"]) // 2)


def sample_value(s):
    """spin-updates/s of the bounded sample itself: its n x R_o x T_o spin-updates over its whole wall time (graph build +
    bSB steps + cut + readout).  No extrapolation: `value` and the time it is divided by describe the same run."""
    t = s["t_build"] + s["t_bsb"] + s["t_read"]
    return s["n"] * s["R_o"] * s["T_o"] / t, t


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2603_25762_b200 import synth
    from oracle import oracle as O
    O.build()
    cores = O.hardware_threads()
    fr, p = synth.make_config(args.config, porec_edges=args.porec_edges)
    per_step = max(2.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
    times, samples = [], []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        s = oracle_sample(fr, p, cores, per_step)
        dt = time.perf_counter() - t0
        if it >= args.warmup:
            times.append(dt); samples.append(s)
    vals = [sample_value(s) for s in samples]
    value = float(np.mean([v[0] for v in vals]))
    s = samples[-1]
    sample = (f"per step: full graph build + {s['R_o']} of {p['R']} replicas x {s['T_o']} of {p['T']} bSB steps + cut + readout of that sample; "
              f"value = n R_o T_o / (t_build + t_bsb + t_readout) of the sample itself (no extrapolation)")
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean([v[1] for v in vals])), "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(args.config, fr, p), "sampled": sample},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "bsb_only_value": float(np.mean([x["n"] * x["R_o"] * x["T_o"] / x["t_bsb"] for x in samples])), "gpu_launches": 0}
    print(json.dumps(out), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2603_25762_b200 import binding as B, parallel, synth

    rank, world, local = parallel.init_from_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    fr, p = synth.make_config(args.config, porec_edges=args.porec_edges)
    snp = p["graph"] == "snp"
    mode = B.QHAP_WEIGHT_FX if snp else B.QHAP_WEIGHT_D_MINUS_C     # BASELINE.json: "discordant minus concordant"
    T = p["T"]
    n = fr.n_snp if snp else fr.n_frag
    blocks_cfg = "block" in p
    plan = parallel.plan_rank(p["R"], p["seed"], rank, world, "weak" if blocks_cfg else args.scaling)
    if blocks_cfg:                       # config 3 shards its independent blocks; every rank runs all R replicas of its blocks
        plan = dict(replicas=p["R"], replica_begin=0, seed=p["seed"], replicas_total=p["R"])
    R, seed, r_begin = plan["replicas"], plan["seed"], plan["replica_begin"]
    tenths = args.linkage_tenths or p.get("linkage_tenths", 10)
    if snp:
        assert args.path in ("auto", "sparse", "block"), "the SNP graphs (configs 3, 4) have no dense J"
        # auto: tcgen05 step on the block-compressed J (config 4: tiles for the banded part + remainder CSR for the long-range edges)
        path = {"auto": 4, "sparse": 2, "block": 4}[args.path]
        tile_skip = 0
    else:
        path = {"auto": 1, "sparse": 2, "dense": 1, "dense-full": 1, "block": 4}[args.path]
        if args.path == "auto" and n * R <= 65536:
            path = 3                                  # config 0: the whole solve in one shared-memory-resident launch
        tile_skip = 0 if args.path == "dense-full" else 1
    dense_dtype = B.QHAP_DENSE_FP16 if path == 1 else B.QHAP_DENSE_NONE
    win = synth.block_windows(fr.n_snp, p["block"], p["stride"]) if "block" in p else None
    if win is not None and world > 1:
        win_mine = win[parallel.block_shard(len(win), rank, world)]   # strong scaling over independent blocks (no exchange)
    else:
        win_mine = win

    dfr = B.upload_frags(fr)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    state = {}

    def one_pass(frags):
        if snp:
            g0 = B.qhap_build_snp_graph(frags, tenths, p.get("alpha", 0.1))
            g = B.qhap_block_split(g0, win_mine) if win is not None else g0
            res = B.qhap_bsb_solve(g, replicas=R, steps_total=T, seed=seed, replica_begin=r_begin, weight_mode=mode, path=path, cut_per_replica=False,
                                   step_launch=args.step_launch, workspace=state.get("ws"))
            state["ws"] = res["workspace"]
            cut, spins = res["best_cut"], res["best_spins"]
            if win is not None:
                spins = B.qhap_block_stitch(fr.n_snp, win_mine, spins) if world == 1 else spins
            elif world > 1:
                cut, spins, _ = parallel.select_best_across_ranks(cut, spins)
            hap = B.qhap_phase_readout_snps(frags.h1, spins) if (win is None or world == 1) else spins
            state["g"] = g
            return cut, hap
        # the edge capacity of the previous pass is the hint for this one (one build call instead of count -> allocate -> fill)
        g, J = B.qhap_build_read_graph(frags, weight_mode=mode, dense_dtype=dense_dtype, capacity_hint=state.get("nnz_hint", 0))
        state["nnz_hint"] = g.nnz + 1024
        res = B.qhap_bsb_solve(g, replicas=R, steps_total=T, seed=seed, replica_begin=r_begin, weight_mode=mode, path=path, dense_J=J, tile_skip=tile_skip,
                               step_launch=args.step_launch, cut_per_replica=False, workspace=state.get("ws"))
        state["ws"] = res["workspace"]
        cut, spins = res["best_cut"], res["best_spins"]
        if world > 1:
            cut, spins, _ = parallel.select_best_across_ranks(cut, spins)
        hap = B.qhap_phase_readout_reads(frags, spins)
        state["g"] = g
        return cut, hap

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, warmup, steps):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        launches0 = 0
        barrier()
        for it in range(warmup + steps):
            flush.zero_()                                   # L2 flush between iterations (outside the event pairs)
            if it == warmup:
                barrier()
                launches0 = B.qhap_launch_count()
            if it >= warmup:
                ev[it - warmup][0].record()
            fn()
            if it >= warmup:
                ev[it - warmup][1].record()
        barrier()
        launches = B.qhap_launch_count() - launches0
        ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms, launches

    props = torch.cuda.get_device_properties(local)
    gpu_id = str(local)
    try:
        u = str(props.uuid)
        gpu_id = u if u.startswith("GPU-") else "GPU-" + u
    except Exception:
        pass
    sampler = ClockSampler(gpu_id)
    sampler.start()
    ms, launches = timed(lambda: one_pass(dfr), args.warmup, args.steps)
    clocks = sampler.stop()
    g = state["g"]
    # spins solved per pass: the read/SNP graph's vertices; config 3 solves overlapping blocks (sum of the window lengths),
    # sharded over ranks (strong scaling); every other config runs R replicas of the whole instance per rank (weak scaling)
    blocks = win is not None
    n_solved = int((win[:, 1] - win[:, 0]).sum()) if blocks else n
    work = n_solved * plan["replicas_total"] * T           # whole job: weak = R per rank x world, strong / blocks = R
    value = work / (ms * 1e-3)
    edges = g.nnz // 2

    # ---- e2e: the same pass fed from pinned host buffers, result read back to the host
    host = {k: torch.from_numpy(np.ascontiguousarray(getattr(fr, k), dtype=dt)).pin_memory()
            for k, dt in (("frag_ptr", np.int64), ("snp_idx", np.int32), ("allele", np.uint8), ("qual", np.uint8)) + ((("frag_flags", np.uint8),) if snp else ())}
    dbuf = {k: torch.empty_like(v, device=dev) for k, v in host.items()}
    hap_host = torch.empty(fr.n_snp, dtype=torch.int8).pin_memory()
    cut_host = torch.empty(len(win_mine) if blocks else 1, dtype=torch.int64).pin_memory()
    h2d = sum(v.numel() * v.element_size() for v in host.values())
    d2h = hap_host.numel() + 8 * cut_host.numel()

    def e2e_pass():
        for k in host:
            dbuf[k].copy_(host[k], non_blocking=True)
        frags = B.Frags(fr.n_frag, fr.n_snp, fr.nnz, dbuf["frag_ptr"], dbuf["snp_idx"], dbuf["allele"], dbuf["qual"],
                        dbuf.get("frag_flags"), None)
        cut, hap = one_pass(frags)
        hap_host[:hap.numel()].copy_(hap, non_blocking=True)
        cut_host.copy_(cut, non_blocking=True)

    e2e_ms, _ = timed(e2e_pass, args.warmup, args.steps)
    e2e_value = work / (e2e_ms * 1e-3)

    # ---- phases of one pass (CUDA events around each C-ABI call; one extra untimed-by-the-headline pass)
    def phase_times():
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        flush.zero_()
        torch.cuda.synchronize()
        ev[0].record()
        if snp:
            g0 = B.qhap_build_snp_graph(dfr, tenths, p.get("alpha", 0.1))
            gg = B.qhap_block_split(g0, win_mine) if win is not None else g0
            JJ = None
        else:
            gg, JJ = B.qhap_build_read_graph(dfr, weight_mode=mode, dense_dtype=dense_dtype)
            g0 = gg
        ev[1].record()
        res = B.qhap_bsb_solve(gg, replicas=R, steps_total=T, seed=seed, weight_mode=mode, path=path, dense_J=JJ, tile_skip=tile_skip, step_launch=args.step_launch,
                               cut_per_replica=False, workspace=state.get("ws"))
        ev[2].record()
        sp = res["best_spins"]
        if snp:
            if win is not None and world == 1:
                sp = B.qhap_block_stitch(fr.n_snp, win_mine, sp)
            B.qhap_phase_readout_snps(dfr.h1, sp[:fr.n_snp] if sp.numel() >= fr.n_snp else sp)
        else:
            B.qhap_phase_readout_reads(dfr, sp)
        ev[3].record()
        torch.cuda.synchronize()
        t = [ev[i].elapsed_time(ev[i + 1]) for i in range(3)]
        # algorithmic bytes of the build (DESIGN.md 4.1 / 4.2): fragment entries in, directed edges out (+ dense J)
        if snp:
            b_bytes = 6.0 * fr.nnz + 20.0 * g0.nnz
        else:
            b_bytes = 5.0 * fr.nnz + 16.0 * g0.nnz + (2.0 * JJ.numel() if JJ is not None else 0.0)
        return {"graph_build_ms": t[0], "bsb_solve_ms": t[1], "readout_ms": t[2], "graph_build_algorithmic_bytes": b_bytes,
                "graph_build_GBps": b_bytes / (t[0] * 1e-3) / 1e9, "graph_build_frac_of_hbm_peak": b_bytes / (t[0] * 1e-3) / 1e9 / measured_peaks()["hbm"],
                "directed_edges": int(g0.nnz)}

    phases = phase_times()

    # ---- the widened rows of SURVEY 8(f), timed once each (not part of the headline pass)
    def timed_once(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        r = fn()
        e1.record()
        torch.cuda.synchronize()
        return r, e0.elapsed_time(e1)

    g_full = B.qhap_build_snp_graph(dfr, tenths, p.get("alpha", 0.1)) if snp else \
        B.qhap_build_read_graph(dfr, weight_mode=mode)[0]
    B.qhap_component_split(g_full, 2)                                      # warm-up
    (cs, _perm), cs_ms = timed_once(lambda: B.qhap_component_split(g_full, 2))
    phases["component_split_ms"] = cs_ms
    phases["components_kept"] = int(len(cs.inst_ptr) - 1)
    if snp and win is None and args.refine_iters > 0:
        rr, rf_ms = timed_once(lambda: B.qhap_snp_refine(g_full, replicas=R, steps_total=T, max_iter=args.refine_iters, seed=seed, path=path))
        phases["refine"] = {"ms": rf_ms, "iterations": rr["iterations"], "cuts": rr["cuts"], "max_iter": args.refine_iters}

    # ---- roofline of the dominant kernel (the bSB step): launches timed with CUDA events on the launching stream
    J = None
    if path == 1:
        _, J = B.qhap_build_read_graph(dfr, weight_mode=mode, dense_dtype=dense_dtype)
    peaks = measured_peaks()

    def time_steps(path_, skip_, steps_):
        res0 = B.qhap_bsb_solve(g, replicas=R, steps_total=T, steps_run=0, seed=seed, weight_mode=mode, path=2, finalize=False)
        x, y = res0["x"], res0["y"]
        kw = dict(replicas=R, steps_total=T, weight_mode=mode, path=path_, x=x, y=y, dense_J=J if path_ == 1 else None, finalize=False,
                  tile_skip=skip_, step_launch=args.step_launch)
        r = B.qhap_bsb_solve(g, step_begin=0, steps_run=min(20, steps_), **kw)          # warm-up (also sizes the workspace)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        l0 = B.qhap_launch_count()
        e0.record()
        B.qhap_bsb_solve(g, step_begin=0, steps_run=steps_, workspace=r["workspace"], **kw)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps_, B.qhap_launch_count() - l0

    step_ms, step_launches = time_steps(path, tile_skip, T)
    n_pad = (n + 127) // 128 * 128

    def tensor_roofline(ms_):
        # flops the full GEMM performs per launch: 2 n^2 R per split term, 2 terms (x_hi, x_lo)
        alg_flops = 2.0 * n * n * R * 2
        return {"kernel": "dense_step_kernel (full N x N GEMM)", "bound": "tensor", "achieved": alg_flops / (ms_ * 1e-3) / 1e12,
                "peak": peaks["bf16_sustained"], "unit": "TFLOP/s", "traffic": None, "flops_per_launch": alg_flops, "launch_ms": ms_,
                "frac": alg_flops / (ms_ * 1e-3) / 1e12 / peaks["bf16_sustained"],
                "peak_source": peaks["which"] + ": sustained bf16 (fp16 inputs run at the same kind::f16 rate)"}

    extra = {}
    if path in (2, 3):
        # algorithmic bytes per launch: 16 B of fp32 state per spin-update (read x, read y, write y, write x')
        # + the CSR once per launch (int32 col + fp32 val per directed entry, int32 row_ptr per row)
        # + SURVEY 8(d): 4 B per replica for every non-zero whose column lies far outside the swept band (|col - row| > 4096:
        # config 4's long-range Pore-C entries), whose x rows cannot come from the cached neighbourhood
        hg = g.to_host()                              # bookkeeping for the byte count only
        rows = np.repeat(np.arange(g.n, dtype=np.int64), np.diff(hg["row_ptr"]))
        long_range = int((np.abs(hg["col"].astype(np.int64) - rows) > 4096).sum())   # x rows far outside the swept band
        alg_bytes = 16.0 * g.n * R + 8.0 * g.nnz + 4.0 * (g.n + 1) + 4.0 * R * long_range
        extra["long_range_nnz"] = long_range
        roofline = {"kernel": "sparse_step_kernel" if path == 2 else "bsb_resident_kernel (latency-bound: one launch runs all T steps; per-step figures)", "bound": "hbm", "achieved": alg_bytes / (step_ms * 1e-3) / 1e9, "peak": peaks["hbm"],
                    "unit": "GB/s", "traffic": None, "bytes_per_launch": alg_bytes, "launch_ms": step_ms, "peak_source": peaks["which"]}
        roofline["frac"] = roofline["achieved"] / roofline["peak"]
    elif tile_skip or path == 4:
        # algorithmic bytes per launch: fp32 state 16 B + fp16 split copies written once (4 B) and read at
        # least once (4 B) per spin-update + the non-zero 64 x 64 fp16 blocks of J once
        hg = g.to_host()                              # bookkeeping for the byte count only
        rows = np.repeat(np.arange(g.n, dtype=np.int64), np.diff(hg["row_ptr"]))
        tile_id = (rows // 64) * (1 << 32) + hg["col"].astype(np.int64) // 64
        tiles, inv, cnt = np.unique(tile_id, return_inverse=True, return_counts=True)
        j_terms = 2 if (path == 4 and snp) else 1     # fp32 SNP weights are stored as J_hi + J_lo
        thr = 1
        tile_cost = 8192.0 * j_terms + 32768.0 * ((R + 127) // 128)      # the library's first threshold (tile_threshold)
        thr0 = 16
        while thr0 < 4096 and thr0 * 1.4142 < tile_cost / (1.2 * (8.0 + 4.0 * R)):
            thr0 *= 2
        if path == 4:                                 # the library's rule: keep all tiles if they fit the
            cap = 16 * g.nnz // 4096 + (g.n + 63) // 64 + 1      # capacity, else only tiles with >= thr0, 2 thr0, ... entries
            while int((cnt >= thr).sum()) > cap:
                thr = thr0 if thr == 1 else thr * 2
        nz_blocks = int((cnt >= thr).sum())
        rem = cnt[inv] < thr                          # entries that go through the remainder CSR gather
        rem_rows = int(np.unique(rows[rem]).size)
        # per spin-update: state16 (the 64-wide tiles' default when R % 4 == 0) carries x as
        # the fp16 pair -- read the pair 4 B, write it 4 B, read y 4 B, write y 4 B = 16 B; the fp32-x kernel adds x read and
        # written in fp32 = 24 B.  Plus the kept tiles of J once, and for a remainder: (col, val) once, one x row gathered per
        # entry, y read-modify-written for the rows that have one
        # next to a remainder CSR state16 also writes the fp32 x for the gather (write only): 20 B
        state16 = (R % 4 == 0)
        state_bytes = (20.0 if int(rem.sum()) > 0 else 16.0) if state16 else 24.0
        alg_bytes = state_bytes * g.n * R + nz_blocks * 64 * 64 * 2.0 * j_terms + int(rem.sum()) * (8.0 + 4.0 * R) + rem_rows * 8.0 * R
        extra["state_bytes_per_spin_update"] = state_bytes
        extra["remainder_nnz"] = int(rem.sum())
        extra["tile_threshold"] = thr
        if int(rem.sum()) > 0:
            extra["roofline_note"] = ("the remainder gathers (4 B x R per far non-zero, SURVEY 8(d)) are counted as algorithmic HBM bytes, but "
                                      "x (%.0f MB) largely stays in the 126 MB L2, so most of them are L2 hits: frac can exceed 1; "
                                      "state + tiles alone = %.0f MB per launch" % (4e-6 * g.n * R, (state_bytes * g.n * R + nz_blocks * 8192.0 * j_terms) / 1e6))
        roofline = {"kernel": "dense_step_kernel (tile_skip)" if path == 1 else "dense_step_kernel (block-compressed J)", "bound": "hbm", "achieved": alg_bytes / (step_ms * 1e-3) / 1e9,
                    "peak": peaks["hbm"], "unit": "GB/s", "traffic": None, "bytes_per_launch": alg_bytes, "launch_ms": step_ms,
                    "peak_source": peaks["which"], "nonzero_64x64_blocks_of_J": nz_blocks}
        roofline["frac"] = roofline["achieved"] / roofline["peak"]
        if path == 1:
            full_ms, _ = time_steps(1, 0, 200)        # the same kernel over ALL k-blocks (north_star's dense GEMM), 200 launches
            extra["roofline_dense_full"] = tensor_roofline(full_ms)
            extra["roofline_dense_full"]["spin_updates_per_s"] = n * R / (full_ms * 1e-3)
    else:
        roofline = tensor_roofline(step_ms)
    # fused launch: one launch ran all T steps; the per-launch figures are T x the per-step ones
    spl = T if (path in (1, 4) and step_launches < T) else 1
    roofline["steps_per_launch"] = spl
    roofline["step_ms"] = step_ms
    if spl > 1:
        for kb_ in ("bytes_per_launch", "flops_per_launch"):
            if kb_ in roofline:
                roofline[kb_.replace("launch", "step")] = roofline[kb_]
                roofline[kb_] = roofline[kb_] * spl
        roofline["launch_ms"] = step_ms * spl
    prof = ROOT / "profiles" / "roofline_traffic.csv"      # dram bytes per launch from the committed ncu captures (kernel, config)
    if prof.exists():
        for line in prof.read_text().splitlines()[1:]:
            f = line.split(",")
            if len(f) >= 3 and f[1] == str(args.config):
                for rl in [roofline] + [v for k, v in extra.items() if k.startswith("roofline") and isinstance(v, dict)]:
                    if rl["kernel"] == f[0]:
                        rl["traffic"] = float(f[2]) * rl.get("steps_per_launch", 1)      # the CSV holds bytes per bSB step

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms, "higher_is_better": True, "scaling": "strong" if (blocks or (args.scaling == "strong" and world > 1)) else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": workload_name(args.config, fr, p),
                      "path": {1: "dense-tcgen05" + (" tile_skip (non-zero k-blocks only; bit-identical to the full GEMM; state16, paired tiles, one fused cooperative launch per solve)" if tile_skip else " full GEMM"),
                               2: "sparse-csr", 3: "shared-memory resident (one launch for all steps)", 4: "tcgen05 step on the block-compressed J (64 x 64 tiles built from the CSR)"}[path],
                      "weight_mode": "fixed-point Eq. 14" if snp else "D-C", "replicas_per_gpu": R, "spins_solved": n_solved, "l2": f"flushed between iterations ({L2_FLUSH_BYTES >> 20} MiB write)",
                      "parallelism": f"blocks x{world} (strong)" if blocks else f"replicas x{world} ({args.scaling if world > 1 else 'weak'})",
                      "linkage_tenths": tenths if snp else None},
           "region_ms": ms, "edges_replicas_per_s": edges * plan["replicas_total"] * T / (ms * 1e-3), "undirected_edges": edges,
           "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
           "gpu_launches": int(launches), "bsb_step_launches_per_solve": int(step_launches),
           "clocks": clocks, "roofline": roofline, "phases": phases, "library": B.qhap_version()}
    out.update(extra)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        O.build()
        cores = O.hardware_threads()
        s = oracle_sample(fr, p, cores, args.cpu_seconds)
        v, t_sample = sample_value(s)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": (f"full graph build ({s['t_build']:.2f} s) + {s['R_o']} of {R} replicas x {s['T_o']} of {T} bSB steps "
                                          f"({s['t_bsb']:.2f} s) + cut + readout ({s['t_read']:.2f} s); value = the sample's own n R_o T_o / its wall time"),
                               "bsb_only_value": s["n"] * s["R_o"] * s["T_o"] / s["t_bsb"], "sample_s": t_sample}
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        # started as a plain process: become N ranks, one per GPU (the driver's torchrun launch sets WORLD_SIZE itself)
        from paper_2603_25762_b200 import parallel
        parallel.spawn_under_torchrun(args.gpus, str(Path(__file__).resolve()), sys.argv[1:])
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
