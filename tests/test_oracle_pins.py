"""Pins of the CPU oracle (oracle/) against what the paper and the mathematics fix -- CPU only.

Every pin names the SURVEY.md 8(c) pin id (P1..P11) and the PAPER.md passage.  None of them re-types the
oracle's own loop: they use integer matmuls, closed forms, hand values (tests/golden/), brute force over all
partitions, explicit linear-map products and exact symmetries.
"""
from __future__ import annotations

import itertools
from pathlib import Path

import numpy as np
import pytest

from paper_2603_25762_b200 import synth

GOLDEN = Path(__file__).resolve().parent / "golden"


# ------------------------------------------------------------------------------------------ helpers
def tiny_fragments(seed, n_snp=40, n_reads=30, flip=0.1, missing=0.1, L=40_000):
    return synth.make_fragments(seed=seed, L=L, n_snp=n_snp, n_reads=n_reads, len_law=("uniform", 4_000, 15_000),
                                flip=flip, missing=missing, qual=("normal", 20, 8, 1, 60))


def ternary_matrix(fr, h1=None):
    """Dense M of Eq. 1 built directly from the fragment list."""
    h1 = fr.h1 if h1 is None else h1
    M = np.zeros((fr.n_frag, fr.n_snp), np.int64)
    for i in range(fr.n_frag):
        for e in range(int(fr.frag_ptr[i]), int(fr.frag_ptr[i + 1])):
            if fr.allele[e] <= 1:
                M[i, fr.snp_idx[e]] = 1 if fr.allele[e] == h1[fr.snp_idx[e]] else -1
    return M


def csr_to_dense(g, vals):
    n = g["n"]
    A = np.zeros((n, n), dtype=np.asarray(vals).dtype)
    for a in range(n):
        for e in range(g["row_ptr"][a], g["row_ptr"][a + 1]):
            A[a, g["col"][e]] = vals[e]
    return A


def one_fragment(snps, alleles, quals, n_snp, flag=0):
    k = len(snps)
    return synth.Fragments(
        n_frag=1, n_snp=n_snp, frag_ptr=np.array([0, k], np.int64), snp_idx=np.array(snps, np.int32),
        allele=np.array(alleles, np.uint8), qual=np.array(quals, np.uint8), frag_flags=np.array([flag], np.uint8),
        h1=np.zeros(n_snp, np.uint8), hap_a=np.zeros(n_snp, np.uint8), frag_hap=np.zeros(1, np.uint8),
        snp_pos=np.arange(n_snp, dtype=np.int64))


# ------------------------------------------------------------------------------------- O1 read graph
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_P1_read_graph_is_integer_matmul(oracle, seed):
    """P1: C - D = M M^T and C + D = |M| |M|^T off the diagonal (Eq. 1-3)."""
    fr = tiny_fragments(seed)
    rng = np.random.default_rng(seed)
    fr.h1 = rng.integers(0, 2, fr.n_snp).astype(np.uint8)          # random gauge
    g = oracle.read_graph(fr)
    M = ternary_matrix(fr)
    S, A = M @ M.T, np.abs(M) @ np.abs(M).T
    np.fill_diagonal(S, 0); np.fill_diagonal(A, 0)
    D, Cc = csr_to_dense(g, g["d"]), csr_to_dense(g, g["c"])
    assert np.array_equal(Cc - D, S)
    assert np.array_equal(Cc + D, A)
    # edge set = pairs sharing >= 1 covered SNP, kept even if the weight is 0
    present = csr_to_dense(g, np.ones(g["nnz"], np.int64))
    assert np.array_equal(present, (A > 0).astype(np.int64))
    # columns strictly ascending inside each row
    for a in range(g["n"]):
        cols = g["col"][g["row_ptr"][a]:g["row_ptr"][a + 1]]
        assert np.all(np.diff(cols) > 0)


def test_P1_cfg0_matmul(oracle):
    fr, _ = synth.make_config(0)
    g = oracle.read_graph(fr)
    M = ternary_matrix(fr)
    S, A = M @ M.T, np.abs(M) @ np.abs(M).T
    np.fill_diagonal(S, 0); np.fill_diagonal(A, 0)
    assert np.array_equal(csr_to_dense(g, g["c"]) - csr_to_dense(g, g["d"]), S)
    assert np.array_equal(csr_to_dense(g, g["c"]) + csr_to_dense(g, g["d"]), A)
    assert 1000 < g["nnz"] // 2 < 2000            # ~1.4k edges at cfg0


def test_P2_interval_closed_form_and_gauge(oracle):
    """P2: without missing sites C + D = size of the intersection of the two index intervals; symmetric; zero
    diagonal.  P6 (read part): D and C do not depend on the gauge h1."""
    fr = tiny_fragments(7, missing=0.0)
    g = oracle.read_graph(fr)
    lo = fr.snp_idx[fr.frag_ptr[:-1]].astype(np.int64)
    hi = fr.snp_idx[fr.frag_ptr[1:] - 1].astype(np.int64)
    T = csr_to_dense(g, g["d"] + g["c"])
    for a in range(fr.n_frag):
        assert T[a, a] == 0
        for b in range(fr.n_frag):
            if a != b:
                assert T[a, b] == max(0, min(hi[a], hi[b]) - max(lo[a], lo[b]) + 1)
    assert np.array_equal(T, T.T)
    fr2 = tiny_fragments(7, missing=0.0)
    fr2.h1 = np.random.default_rng(0).integers(0, 2, fr.n_snp).astype(np.uint8)
    g2 = oracle.read_graph(fr2)
    for k in ("row_ptr", "col", "d", "c"):
        assert np.array_equal(g[k], g2[k])


def test_P3_error_free_reads_bipartite(oracle):
    """P3 / PAPER.md:L246: error-free reads give w = 0 inside a haplotype and w = #shared across."""
    fr = tiny_fragments(11, n_snp=60, n_reads=40, flip=0.0, missing=0.0)
    g = oracle.read_graph(fr)
    for a in range(fr.n_frag):
        for e in range(g["row_ptr"][a], g["row_ptr"][a + 1]):
            b = g["col"][e]
            if fr.frag_hap[a] == fr.frag_hap[b]:
                assert g["d"][e] == 0 and g["c"][e] > 0
            else:
                assert g["c"][e] == 0 and g["d"][e] > 0
    # planted partition cuts every positive-weight edge: cut = total weight (mode 0), and energy = -W_tot
    s = np.where(fr.frag_hap == 0, 1, -1).astype(np.int8)
    w0 = oracle.read_weights(g, 0)
    cut, en = oracle.cut_eval(g["row_ptr"], g["col"], w0, s)
    assert cut[0] == w0.sum() // 2 and en[0] == -(w0.sum() // 2)


# -------------------------------------------------------------------------------------- O2 SNP graph
def test_P4_hand_values(oracle):
    """P4: hand-evaluated contributions of Eq. 9-14 and the alpha scaling of PAPER.md:L350."""
    rows = [ln.split() for ln in (GOLDEN / "snp_edge_hand_values.txt").read_text().splitlines()
            if ln.strip() and not ln.startswith("#")]
    assert len(rows) >= 9
    for qu, qv, k, same, pc, alpha, expect in rows:
        qu, qv, k, same, pc = int(qu), int(qv), int(k), int(same), int(pc)
        snps = list(range(k))
        alleles = [0] * k
        if not same:
            alleles[1] = 1
        quals = [qu, qv] + [qu] * (k - 2)
        g = oracle.snp_graph(one_fragment(snps, alleles, quals, n_snp=k, flag=pc), 10, float(alpha))
        W = csr_to_dense(g, g["w_fx"])
        got = W[0, 1] / 2.0 ** 32
        assert abs(got - float(expect)) <= 2.0 ** -32, (qu, qv, k, same, pc, got, expect)      # one fixed-point ulp
        assert W[0, 1] == W[1, 0]
        assert np.array_equal(g["w"], (g["w_fx"].astype(np.float64) * 2.0 ** -32).astype(np.float32))


def test_P5_snp_graph_invariants(oracle):
    """P5: table symmetric, q = 0.5 gives zero, symmetry, exact independence of fragment order, depth monotone."""
    T = oracle.llr_table()
    assert np.array_equal(T[1:, 1:], T[1:, 1:].T)
    assert np.all(T[1:, 1:][np.ix_(np.arange(3, 93), np.arange(3, 93))] > 0)      # Q >= 4 -> q > 0.5 -> cis favoured
    # q = 0.5 exactly is Q = 10 log10(2) (not an integer): check the sign change around it instead
    assert T[3, 40] < 0 < T[4, 40]
    fr = tiny_fragments(5, n_snp=50, n_reads=40)
    g = oracle.snp_graph(fr, 10, 0.1)
    W = csr_to_dense(g, g["w_fx"])
    assert np.array_equal(W, W.T) and np.all(np.diag(W) == 0)
    # fragment order: reverse the fragment list (still a valid CSR; the oracle does not require sortedness)
    order = np.arange(fr.n_frag)[::-1]
    cnt = np.diff(fr.frag_ptr)[order]
    ptr = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int64)
    src = np.concatenate([np.arange(fr.frag_ptr[i], fr.frag_ptr[i + 1]) for i in order])
    fr_rev = synth.Fragments(fr.n_frag, fr.n_snp, ptr, fr.snp_idx[src], fr.allele[src], fr.qual[src],
                             fr.frag_flags[order], fr.h1, fr.hap_a, fr.frag_hap[order], fr.snp_pos)
    g_rev = oracle.snp_graph(fr_rev, 10, 0.1)
    for k in ("row_ptr", "col", "w_fx", "w"):
        assert np.array_equal(g[k], g_rev[k])
    # depth k edge set is a subset of depth 10; depth 10 = every covered pair inside a fragment
    prev = None
    for tenths in (1, 3, 6, 10):
        gk = oracle.snp_graph(fr, tenths, 0.1)
        E = csr_to_dense(gk, np.ones(gk["nnz"], np.int64))
        if prev is not None:
            assert np.all(prev <= E)
        prev = E
    M = ternary_matrix(fr)
    cov = (np.abs(M).T @ np.abs(M)) > 0
    np.fill_diagonal(cov, False)
    assert np.array_equal(prev.astype(bool), cov)


def test_P5_linkage_depth_reach(oracle):
    """depth k/10 links each SNP to its nearest floor(k (N-1) / 10) downstream SNPs of the read."""
    k = 11
    fr = one_fragment(list(range(k)), [0] * k, [20] * k, n_snp=k)
    for tenths in range(1, 11):
        g = oracle.snp_graph(fr, tenths, 0.1)
        E = csr_to_dense(g, np.ones(g["nnz"], np.int64))
        reach = (tenths * (k - 1)) // 10
        for u in range(k):
            for v in range(u + 1, k):
                assert E[u, v] == (1 if v - u <= reach else 0)


def test_P6_gauge_invariance_snp(oracle):
    """P6: flipping h1[u] negates every w_u. exactly; E(s) is invariant when s_u is flipped too."""
    fr = tiny_fragments(9, n_snp=30, n_reads=40)
    g = oracle.snp_graph(fr, 10, 0.1)
    W = csr_to_dense(g, g["w_fx"])
    u = 7
    fr.h1 = fr.h1.copy(); fr.h1[u] = 1
    g2 = oracle.snp_graph(fr, 10, 0.1)
    W2 = csr_to_dense(g2, g2["w_fx"])
    sgn = np.ones(fr.n_snp, np.int64); sgn[u] = -1
    assert np.array_equal(W2, W * sgn[:, None] * sgn[None, :])
    s = synth.random_spins(3, fr.n_snp, 5)
    s2 = s.copy(); s2[u] *= -1
    _, e1 = oracle.cut_eval(g["row_ptr"], g["col"], g["w_fx"], s)
    _, e2 = oracle.cut_eval(g2["row_ptr"], g2["col"], g2["w_fx"], s2)
    assert np.array_equal(e1, e2)


# --------------------------------------------------------------------------------- O4 cut and energy
def random_graph(seed, n, p=0.4, lo=-9, hi=9):
    """Small random symmetric integer graph as CSR (test input only)."""
    rng = np.random.default_rng(seed)
    A = np.triu((rng.uniform(size=(n, n)) < p) * rng.integers(lo, hi + 1, size=(n, n)), 1)
    P = np.triu(rng.uniform(size=(n, n)) < p, 1)          # structural pattern (zero-weight edges allowed)
    A = A * P
    A = A + A.T; P = P | P.T
    row_ptr = np.zeros(n + 1, np.int32); col = []; w = []
    for a in range(n):
        for b in range(n):
            if P[a, b]:
                col.append(b); w.append(A[a, b])
        row_ptr[a + 1] = len(col)
    return A.astype(np.int64), row_ptr, np.array(col, np.int32), np.array(w, np.int64)


def test_P7_P8_cut_brute_force_and_identities(oracle):
    """P7: cut equals the direct crossing-edge sum for every partition of a small graph.
    P8: E = W_tot - 2 cut = -1/2 s^T J s with J = -A (Eq. 4-6); cut(s) = cut(-s); cut(+1) = 0."""
    n = 10
    A, rp, cl, w = random_graph(4, n)
    parts = np.array(list(itertools.product([-1, 1], repeat=n)), np.int8).T.copy()       # [n][2^n]
    cut, en = oracle.cut_eval(rp, cl, w, parts)
    S = parts.astype(np.int64)
    quad = np.einsum("ar,ab,br->r", S, A, S)                     # s^T A s
    wtot = A.sum() // 2
    assert np.array_equal(cut, (2 * wtot - quad) // 4 * 1) and np.all((2 * wtot - quad) % 4 == 0)   # Eq. 6
    assert np.array_equal(en, quad // 2)                         # Eq. 5 with J = -A:  -1/2 s^T J s = +1/2 s^T A s
    assert np.array_equal(en, wtot - 2 * cut)
    assert np.array_equal(cut, cut[::-1])                        # column r and its complement 2^n-1-r
    assert cut[-1] == 0 and cut[0] == 0
    # direct definition on a few columns
    for r in (1, 37, 500, 1023):
        direct = sum(A[a, b] for a in range(n) for b in range(a + 1, n) if parts[a, r] != parts[b, r])
        assert cut[r] == direct
    assert oracle.best_replica(cut) == int(np.flatnonzero(cut == cut.max())[0])


# ------------------------------------------------------------------------------------------- O3 bSB
def csr_from_dense(J):
    n = J.shape[0]
    rp = np.zeros(n + 1, np.int32); cl = []; v = []
    for a in range(n):
        for b in range(n):
            if J[a, b] != 0:
                cl.append(b); v.append(J[a, b])
        rp[a + 1] = len(cl)
    return rp, np.array(cl, np.int32), np.array(v, np.float32)


def test_P9_linear_regime_matrix_product(oracle):
    """P9: before any wall hit one step is the linear map (y first from the old x, then x from the new y):
        y' = y + dt(-(a0 - a_k) x + c0 J x);  x' = x + dt a0 y'.   Compared with an explicit product of 2N x 2N matrices."""
    n, R, T, dt, a0, c0 = 6, 3, 40, 0.25, 1.0, 0.05
    rng = np.random.default_rng(0)
    J = rng.integers(-3, 4, size=(n, n)).astype(np.float64); J = np.triu(J, 1); J = J + J.T
    rp, cl, jv = csr_from_dense(J)
    x0 = rng.uniform(-1e-3, 1e-3, size=(n, R)); y0 = rng.uniform(-1e-3, 1e-3, size=(n, R))
    steps = 12
    x, y, _ = oracle.bsb_run(rp, cl, jv, x0.copy(), y0.copy(), steps_total=T, steps_run=steps, dt=dt, a0=a0, c0=c0)
    z = np.vstack([x0, y0])
    I = np.eye(n)
    for k in range(steps):
        a_k = a0 * k / (T - 1)
        B = dt * (-(a0 - a_k) * I + c0 * J)                      # y' = y + B x
        Mk = np.block([[I + dt * a0 * B, dt * a0 * I], [B, I]])  # x' = x + dt a0 (y + B x)
        z = Mk @ z
    assert np.max(np.abs(x)) < 1.0
    np.testing.assert_allclose(np.vstack([x, y]), z, rtol=1e-11, atol=1e-15)
    # the dense loop of the oracle is the same recurrence
    xd, yd = oracle.bsb_run_dense(J, x0.copy(), y0.copy(), steps_total=T, steps_run=steps, dt=dt, a0=a0, c0=c0)
    np.testing.assert_allclose(xd, x, rtol=1e-12, atol=1e-18); np.testing.assert_allclose(yd, y, rtol=1e-12, atol=1e-18)


def test_P9_scalar_recurrence_ramp_and_wall(oracle):
    """P9 (J = 0): each spin follows y <- y - dt (a0 - a_k) x, x <- x + dt a0 y with a_k = a0 k/(T-1)
    (BASELINE.json "a(t) linear 0->1": a = 0 at the first step, a0 at the last); strict |x| > 1 wall: x = sign(x), y = 0."""
    rp = np.zeros(2, np.int32); cl = np.zeros(0, np.int32); jv = np.zeros(0, np.float32)
    T, dt, a0 = 5, 0.5, 2.0
    x, y, _ = oracle.bsb_run(rp, cl, jv, np.array([[0.25]]), np.array([[0.5]]), steps_total=T, steps_run=1, dt=dt, a0=a0, c0=1.0)
    assert y[0, 0] == 0.5 - 0.5 * 2.0 * 0.25 and x[0, 0] == 0.25 + 0.5 * 2.0 * y[0, 0]        # k = 0 -> a_k = 0
    x, y, _ = oracle.bsb_run(rp, cl, jv, np.array([[0.25]]), np.array([[0.5]]), steps_total=T, step_begin=T - 1, steps_run=1,
                             dt=dt, a0=a0, c0=1.0)
    assert y[0, 0] == 0.5 and x[0, 0] == 0.75                                                  # k = T-1 -> a_k = a0
    # wall: exactly 1.0 is not clamped; beyond it x = sign(x), y = 0
    x, y, _ = oracle.bsb_run(rp, cl, jv, np.array([[0.5, 0.5, -0.5]]), np.array([[0.5, 0.75, -2.0]]), steps_total=T,
                             step_begin=T - 1, steps_run=1, dt=dt, a0=a0, c0=1.0)
    assert x.tolist() == [[1.0, 1.0, -1.0]] and y.tolist() == [[0.5, 0.0, 0.0]]
    # xpre reports x before the wall rule
    xp = np.zeros((1, 3))
    oracle.bsb_run(rp, cl, jv, np.array([[0.5, 0.5, -0.5]]), np.array([[0.5, 0.75, -2.0]]), steps_total=T,
                   step_begin=T - 1, steps_run=1, dt=dt, a0=a0, c0=1.0, xpre=xp)
    assert xp.tolist() == [[1.0, 1.25, -2.5]]


def test_P10_exact_symmetries_and_resume(oracle):
    """P10: negating (x0, y0) negates the trajectory bit for bit; permuting replicas permutes outputs;
    running k steps then T-k steps equals running T steps (steps_run / step_begin, SURVEY section 5 'resume')."""
    fr = tiny_fragments(21, n_snp=60, n_reads=40)
    g = oracle.read_graph(fr)
    jv = (-oracle.read_weights(g, 1)).astype(np.float32)
    n, R, T = fr.n_frag, 6, 60
    x0, y0 = synth.bsb_init_state(5, n, R)
    x0 = x0.astype(np.float64); y0 = y0.astype(np.float64)
    xa, ya, c0 = oracle.bsb_run(g["row_ptr"], g["col"], jv, x0.copy(), y0.copy(), steps_total=T)
    assert np.any(np.abs(xa) == 1.0)                                   # walls were reached: the nonlinear part is exercised
    xb, yb, _ = oracle.bsb_run(g["row_ptr"], g["col"], jv, -x0, -y0, steps_total=T)
    assert np.array_equal(xb, -xa) and np.array_equal(yb, -ya)
    perm = np.array([3, 0, 5, 1, 2, 4])
    xc, yc, _ = oracle.bsb_run(g["row_ptr"], g["col"], jv, x0[:, perm].copy(), y0[:, perm].copy(), steps_total=T)
    assert np.array_equal(xc, xa[:, perm]) and np.array_equal(yc, ya[:, perm])
    xd, yd, _ = oracle.bsb_run(g["row_ptr"], g["col"], jv, x0.copy(), y0.copy(), steps_total=T, steps_run=17)
    xd, yd, _ = oracle.bsb_run(g["row_ptr"], g["col"], jv, xd, yd, steps_total=T, step_begin=17, steps_run=T - 17)
    assert np.array_equal(xd, xa) and np.array_equal(yd, ya)
    xe, ye, _ = oracle.bsb_run(g["row_ptr"], g["col"], jv, x0.copy(), y0.copy(), steps_total=T, n_threads=3)
    assert np.array_equal(xe, xa) and np.array_equal(ye, ya)           # threads only slice replicas
    # c0 = 0.5 sqrt(N-1) / ||J||_F over all ordered entries (reading R10c)
    Jd = csr_to_dense(g, jv.astype(np.float64))
    assert abs(c0 - 0.5 * np.sqrt(n - 1) / np.linalg.norm(Jd)) <= 1e-15 * c0 * 8


def test_P7_bsb_quality_vs_brute_force(oracle):
    """P7: on small graphs the bSB best cut never exceeds the optimum and reaches it on planted instances."""
    fr = synth.make_fragments(seed=31, L=30_000, n_snp=40, n_reads=16, len_law=("uniform", 8_000, 16_000), flip=0.03,
                              missing=0.0, qual=("const", 30))
    g = oracle.read_graph(fr)
    n = fr.n_frag
    assert n <= 20
    for mode in (0, 1):
        w = oracle.read_weights(g, mode)
        parts = np.array(list(itertools.product([-1, 1], repeat=n - 1)), np.int8)
        parts = np.hstack([np.ones((len(parts), 1), np.int8), parts]).T.copy()
        cut, _ = oracle.cut_eval(g["row_ptr"], g["col"], w, parts)
        opt = int(cut.max())
        x0, y0 = synth.bsb_init_state(1, n, 32)
        res = oracle.solve(g["row_ptr"], g["col"], w, (-w).astype(np.float32), x0, y0, steps_total=300)
        assert np.all(res["cut"] <= opt)
        assert res["best_cut"] == opt, (mode, res["best_cut"], opt)
        assert res["best_replica"] == int(np.flatnonzero(res["cut"] == res["cut"].max())[0])
        assert np.array_equal(res["best_spins"], res["spins"][:, res["best_replica"]])


def test_P3_planted_recovery_end_to_end(oracle):
    """P3 (north_star's third oracle check): error-free reads with connected coverage -> the optimum is the planted
    partition (unique up to a global flip) -> exact haplotype recovery, SE = HE = 0."""
    fr = synth.make_fragments(seed=41, L=100_000, n_snp=120, n_reads=80, len_law=("uniform", 10_000, 25_000), flip=0.0,
                              missing=0.0, qual=("const", 30))
    g = oracle.read_graph(fr)
    planted = np.where(fr.frag_hap == 0, 1, -1).astype(np.int8)
    for mode in (0, 1):
        w = oracle.read_weights(g, mode)
        x0, y0 = synth.bsb_init_state(2, fr.n_frag, 16)
        res = oracle.solve(g["row_ptr"], g["col"], w, (-w).astype(np.float32), x0, y0, steps_total=400)
        pcut, _ = oracle.cut_eval(g["row_ptr"], g["col"], w, planted)
        assert res["best_cut"] == pcut[0] == w[w > 0].sum() // 2
        s = res["best_spins"]
        assert np.array_equal(s, planted) or np.array_equal(s, -planted)
        hap = oracle.read_vote(fr, s)
        covered = np.bincount(fr.snp_idx, minlength=fr.n_snp) > 0
        m = oracle.switch_hamming(hap, fr.hap_a)
        assert m["se"] == 0.0 and m["he"] == 0.0 and m["n_phased"] == int(covered.sum())
    # SNP-graph route on the same reads: sign pattern of the planted haplotype is the optimum
    gs = oracle.snp_graph(fr, 10, 0.1)
    x0, y0 = synth.bsb_init_state(3, fr.n_snp, 16)
    res = oracle.solve(gs["row_ptr"], gs["col"], gs["w_fx"], (-gs["w"]).astype(np.float32), x0, y0, steps_total=400)
    hap = oracle.snp_readout(fr.h1, res["best_spins"])
    m = oracle.switch_hamming(hap[covered], fr.hap_a[covered])
    assert m["se"] == 0.0 and m["he"] == 0.0


# ----------------------------------------------------------------------------- O5 readouts and metrics
def test_P11_paper_worked_example(oracle):
    """P11: PAPER.md:L380-L382 -- "01110" vs "00000": 2 switches -> SE = 2/(5-1) = 50 %; 3 mismatches -> HE = 60 %."""
    rows = [ln.split() for ln in (GOLDEN / "se_he_example.txt").read_text().splitlines() if ln.strip() and not ln.startswith("#")]
    for inferred, ref, sw, n, se, mm, he in rows:
        h = np.array([int(ch) for ch in inferred], np.int8); t = np.array([int(ch) for ch in ref], np.uint8)
        m = oracle.switch_hamming(h, t)
        assert m["switches"] == int(sw) and m["n_phased"] == int(n) and m["mismatches"] == int(mm)
        assert m["se"] == float(se) and m["he_raw"] == float(he)
    # unphased sites (-1) are skipped, not counted as switches
    m = oracle.switch_hamming(np.array([0, -1, 1, 1, -1, 0], np.int8), np.zeros(6, np.uint8))
    assert (m["switches"], m["n_phased"], m["mismatches"]) == (2, 4, 2)


def test_read_vote_rule(oracle):
    """PAPER.md:L271-L281 (Eq. 7-8 and the rule, reading R13): hap(S1) = sign(d1 - d2), d_l = c_l(+) - c_l(-)."""
    # 4 fragments over 5 SNPs, h1 = all-ref: allele 0 -> M=+1, allele 1 -> M=-1
    ptr = np.array([0, 5, 10, 15, 20], np.int64)
    idx = np.tile(np.arange(5, dtype=np.int32), 4)
    #            snp: 0  1  2  3  4
    al = np.array([0, 0, 1, 2, 0,      # f0 in S1
                   0, 1, 1, 2, 1,      # f1 in S1
                   1, 1, 0, 2, 0,      # f2 in S2
                   1, 0, 0, 2, 1], np.uint8)
    fr = synth.Fragments(4, 5, ptr, idx, al, np.full(20, 30, np.uint8), np.zeros(4, np.uint8), np.zeros(5, np.uint8),
                         np.zeros(5, np.uint8), np.zeros(4, np.uint8), np.arange(5, dtype=np.int64))
    s = np.array([1, 1, -1, -1], np.int8)
    # snp0: d1=+2,d2=-2 -> + -> H1 allele (0);  snp1: d1=0,d2=0 -> unphased;  snp2: d1=-2,d2=+2 -> other allele (1)
    # snp3: no coverage -> unphased;  snp4: d1=0 (one each), d2=0 -> unphased
    assert oracle.read_vote(fr, s).tolist() == [0, -1, 1, -1, -1]
    assert oracle.read_vote(fr, -s).tolist() == [1, -1, 0, -1, -1]
    assert oracle.snp_readout(np.array([0, 1, 0], np.uint8), np.array([1, 1, -1], np.int8)).tolist() == [0, 1, 1]


def test_block_split_and_stitch(oracle):
    """Reading R17: windows of `block` SNPs every `stride`; an edge is in a block iff both ends are; stitching flips a
    block when the overlap with the previous (already oriented) block disagrees, and each block owns up to the overlap midpoint."""
    win = synth.block_windows(23, 10, 7)
    assert win.tolist() == [[0, 10], [7, 17], [14, 23]]
    truth = np.where(np.random.default_rng(0).integers(0, 2, 23) == 1, 1, -1).astype(np.int8)
    blocks = [truth[0:10].copy(), -truth[7:17], truth[14:23].copy()]            # middle block globally flipped
    out = oracle.block_stitch(23, win, blocks)
    assert np.array_equal(out, truth)
    blocks[2] = -blocks[2]
    assert np.array_equal(oracle.block_stitch(23, win, blocks), truth)
    # split: induced sub-graphs, block-diagonal numbering
    fr = tiny_fragments(13, n_snp=23, n_reads=30)
    g = oracle.snp_graph(fr, 10, 0.1)
    W = csr_to_dense(g, g["w_fx"])
    P = csr_to_dense(g, np.ones(g["nnz"], np.int64))
    bs = oracle.block_split(g, win)
    assert bs["inst_ptr"].tolist() == [0, 10, 20, 29] and bs["n"] == 29
    Wb = csr_to_dense(bs, bs["w_fx"]); Pb = csr_to_dense(bs, np.ones(bs["nnz"], np.int64))
    expectW = np.zeros((29, 29), np.int64); expectP = np.zeros((29, 29), np.int64)
    for b, (lo, hi) in enumerate(win.tolist()):
        o = int(bs["inst_ptr"][b])
        expectW[o:o + hi - lo, o:o + hi - lo] = W[lo:hi, lo:hi]
        expectP[o:o + hi - lo, o:o + hi - lo] = P[lo:hi, lo:hi]
    assert np.array_equal(Wb, expectW) and np.array_equal(Pb, expectP)


def test_init_state_is_uniform_and_fp32(oracle):
    """Reading R11: x0, y0 ~ U(-0.1, 0.1) from a counter hash; fp32; different for x and y, replicas and seeds."""
    x, y = synth.bsb_init_state(123, 500, 64)
    assert x.dtype == np.float32 and x.shape == (500, 64)
    for a in (x, y):
        assert np.all(np.abs(a) < 0.1) and abs(a.mean()) < 1e-3 and abs(a.std() - 0.2 / np.sqrt(12)) < 1e-3
    assert not np.array_equal(x, y) and not np.array_equal(x[:, 0], x[:, 1])
    x2, _ = synth.bsb_init_state(124, 500, 64)
    assert not np.array_equal(x, x2)


# ------------------------------------------------------------------------------------ O6 iterative refinement (f1)
def test_refine_gauge_identity_and_planted_recovery(oracle):
    """Eq. 15 is a gauge transform: E_{w'}(t) = E_w(s o t) for every t (exact, int64), so E_{w'}(all +1) = E_w(s).
    Error-free reads: the first solve is optimal, the transformed graph's best cut is <= 0 -> the loop stops after two
    solves with C = indicator of the smaller side, and Eq. 17 returns the planted haplotype (SE = HE = 0)."""
    fr = synth.make_fragments(seed=11, L=60_000, n_snp=80, n_reads=60, len_law=("uniform", 6_000, 15_000), flip=0.0,
                              missing=0.0, qual=("const", 30))
    g = oracle.snp_graph(fr, 10, 0.1)
    rng = np.random.default_rng(0)
    s = rng.choice(np.array([-1, 1], np.int8), size=g["n"])
    wfx2, w2 = oracle.gauge_transform(g["row_ptr"], g["col"], g["w_fx"], g["w"], s)
    assert np.array_equal(np.abs(wfx2), np.abs(g["w_fx"])) and np.array_equal(np.abs(w2), np.abs(g["w"]))
    for _ in range(5):
        t = rng.choice(np.array([-1, 1], np.int8), size=g["n"])
        _, e2 = oracle.cut_eval(g["row_ptr"], g["col"], wfx2, t)
        _, e1 = oracle.cut_eval(g["row_ptr"], g["col"], g["w_fx"], (s * t).astype(np.int8))
        assert e1[0] == e2[0]
    ones = np.ones(g["n"], np.int8)
    assert np.array_equal(oracle.gauge_transform(g["row_ptr"], g["col"], g["w_fx"], g["w"], ones)[0], g["w_fx"])
    m = oracle.smaller_subset(np.array([1, -1, -1, 1, 1], np.int8))
    assert m.tolist() == [False, True, True, False, False]
    assert oracle.smaller_subset(np.array([1, -1], np.int8)).tolist() == [False, True]          # tie -> the -1 side
    R, T = 16, 300
    res = oracle.refine_snp(g["row_ptr"], g["col"], g["w_fx"], g["w"], lambda t: synth.bsb_init_state(100 + t, g["n"], R),
                            steps_total=T, max_iter=6, n_threads=4)
    assert res["iterations"] == 2 and res["cuts"][0] > 0 and res["cuts"][1] <= 0, res["cuts"]
    hap = oracle.refine_readout(fr.h1, res["flip_count"])
    covered = np.bincount(fr.snp_idx[fr.allele <= 1], minlength=fr.n_snp) > 0
    mm = oracle.switch_hamming(hap[covered], fr.hap_a[covered])
    assert mm["se"] == 0.0 and mm["he"] == 0.0
    assert set(np.unique(res["flip_count"])) <= {0, 1}


# ------------------------------------------------------------------------------- O7 connected components (f2)
def test_component_split_known_graph_and_bfs(oracle):
    """A hand-made graph with known components, and random graphs against a plain BFS."""
    # components: {0, 3, 4}, {1}, {2, 5}, {6, 7, 8} (path), 9 isolated
    edges = [(0, 3), (3, 4), (2, 5), (6, 7), (7, 8)]
    n = 10
    rows = [[] for _ in range(n)]
    for a, b in edges:
        rows[a].append(b); rows[b].append(a)
    rp = np.r_[0, np.cumsum([len(r) for r in rows])].astype(np.int32)
    cl = np.array([c for r in rows for c in sorted(r)], np.int32)
    g = dict(n=n, nnz=len(cl), row_ptr=rp, col=cl, w_fx=np.arange(1, len(cl) + 1, dtype=np.int64))
    cs = oracle.component_split(g, 2)
    assert cs["perm"].tolist() == [0, 3, 4, 2, 5, 6, 7, 8] and cs["inst_ptr"].tolist() == [0, 3, 5, 8]
    assert cs["row_ptr"].tolist() == [0, 1, 3, 4, 5, 6, 7, 9, 10]
    assert cs["col"].tolist() == [1, 0, 2, 1, 4, 3, 6, 5, 7, 6]
    # weights travel with their entries: entry (0,3) had w 1; (3,0) 4; (3,4) 5 ...
    assert cs["w_fx"][0] == 1 and cs["w_fx"][1] == g["w_fx"][rp[3]]
    assert oracle.component_split(g, 1)["inst_ptr"].tolist() == [0, 3, 4, 6, 9, 10]
    assert oracle.component_merge(n, cs["perm"], np.ones(8, np.int8)).tolist() == [1, 0, 1, 1, 1, 1, 1, 1, 1, 0]
    rng = np.random.default_rng(3)
    for _ in range(5):
        n = 60
        m = rng.random((n, n)) < 0.02
        m = np.triu(m, 1); m = m | m.T
        rp = np.r_[0, np.cumsum(m.sum(1))].astype(np.int32)
        cl = np.concatenate([np.flatnonzero(m[i]) for i in range(n)]).astype(np.int32)
        cs = oracle.component_split(dict(n=n, nnz=len(cl), row_ptr=rp, col=cl), 2)
        seen, comps = np.zeros(n, bool), []
        for v in range(n):                                # plain BFS in vertex order
            if seen[v]:
                continue
            comp, todo = [], [v]
            seen[v] = True
            while todo:
                u = todo.pop()
                comp.append(u)
                for wv in np.flatnonzero(m[u]):
                    if not seen[wv]:
                        seen[wv] = True; todo.append(int(wv))
            if len(comp) >= 2:
                comps.append(sorted(comp))
        assert cs["perm"].tolist() == [v for c in comps for v in c]
        assert np.diff(cs["inst_ptr"]).tolist() == [len(c) for c in comps]


# ------------------------------------------------- round 2: the four behaviours VERDICT r1 listed as "parity unpinned"
def test_R10e_sign_of_zero_is_plus_one(oracle):
    """Reading R10e ("s = sgn(x)"; Eq. 6 needs s in {-1, +1}, so sgn(0) must pick a side): x = +0.0 and
    x = -0.0 both read out as +1; the smallest negative number as -1.  A spin vector therefore never contains 0 and every
    vertex is on exactly one side of the cut."""
    x = np.array([[0.0, -0.0, 5e-324, -5e-324, 1.0, -1.0]])
    assert oracle.sign_spins(x).tolist() == [[1, 1, 1, -1, 1, -1]]
    # consequence for the solver: a spin that sits exactly at 0 (isolated vertex, x0 = y0 = 0) is reported as +1
    rp = np.zeros(3, np.int32); cl = np.zeros(0, np.int32)
    res = oracle.solve(rp, cl, np.zeros(0, np.int64), np.zeros(0, np.float32), np.zeros((2, 1), np.float32), np.zeros((2, 1), np.float32),
                       steps_total=5)
    assert res["best_spins"].tolist() == [1, 1] and np.all(res["x"] == 0.0)


def _golden_depth_rows():
    edges, clamps = {}, []
    for ln in (GOLDEN / "snp_edge_depth_porec_clamp.txt").read_text().splitlines():
        f = ln.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] == "edge":
            edges.setdefault((int(f[1]), int(f[2]), float(f[3])), {})[(int(f[4]), int(f[5]))] = float(f[6])
        elif f[0] == "clamp":
            clamps.append((int(f[1]), int(f[2]), float(f[3])))
    return edges, clamps


def test_R8_porec_fragments_keep_every_pair_and_scale_by_alpha(oracle):
    """PAPER.md:L85 (depth), L344-L350 (Pore-C, alpha), reading R8: a k = 5 fragment at depth 3/10 emits only its 4 adjacent
    pairs; the SAME fragment flagged Pore-C emits all 10 pairs (reach = k - 1 whatever the depth) and every weight is
    alpha x the unflagged exhaustive one.  Expected edge lists and 20-digit weights: tests/golden/ (mpmath script beside it);
    a build that applied the depth limit to Pore-C fragments, forgot alpha, or used alpha on ordinary reads fails here."""
    edges, _ = _golden_depth_rows()
    Q = [12, 25, 7, 33, 18]
    assert len(edges) == 4
    for (tenths, flag, alpha), exp in edges.items():
        g = oracle.snp_graph(one_fragment(list(range(5)), [0] * 5, Q, n_snp=5, flag=flag), tenths, alpha)
        W = csr_to_dense(g, g["w_fx"]).astype(np.float64) / 2.0 ** 32
        got = {(u, v) for u in range(5) for v in range(u + 1, 5) if csr_to_dense(g, np.ones(g["nnz"], np.int64))[u, v]}
        assert got == set(exp), (tenths, flag, sorted(got))
        for (u, v), w in exp.items():
            assert abs(W[u, v] - w) <= 2.0 ** -32 and W[v, u] == W[u, v], (tenths, flag, u, v, W[u, v], w)
    assert len(edges[(3, 0, 0.1)]) == 4 and len(edges[(3, 1, 0.1)]) == 10
    # a Pore-C fragment next to an ordinary read through the same SNP pair: the two contributions add (alpha only on one)
    fr2 = synth.Fragments(2, 5, np.array([0, 5, 10], np.int64), np.tile(np.arange(5, dtype=np.int32), 2), np.zeros(10, np.uint8),
                          np.array(Q * 2, np.uint8), np.array([0, 1], np.uint8), np.zeros(5, np.uint8), np.zeros(5, np.uint8),
                          np.zeros(2, np.uint8), np.arange(5, dtype=np.int64))
    g2 = oracle.snp_graph(fr2, 3, 0.1)
    W2 = csr_to_dense(g2, g2["w_fx"]).astype(np.float64) / 2.0 ** 32
    for (u, v), w in edges[(3, 1, 0.1)].items():
        expect = w + edges[(3, 0, 0.1)].get((u, v), 0.0)
        assert abs(W2[u, v] - expect) <= 2 * 2.0 ** -32


def test_R5_phred_clamp(oracle):
    """Reading R5: integer Phred is clamped to [1, 93] before Eq. 9 (Q = 0 would make q = 0 and, for two such sites,
    P_trans = P_cis; Q > 93 has no table entry).  Q = 0 weighs exactly like Q = 1 and Q = 200 like Q = 93; the values are the
    mpmath evaluation of Eq. 9-14 at the CLAMPED qualities (tests/golden/snp_edge_depth_porec_clamp.txt)."""
    _, clamps = _golden_depth_rows()
    assert len(clamps) >= 6
    for qu, qv, w in clamps:
        g = oracle.snp_graph(one_fragment([0, 1], [0, 0], [min(qu, 255), min(qv, 255)], n_snp=2), 10, 0.1)
        got = csr_to_dense(g, g["w_fx"])[0, 1] / 2.0 ** 32
        # fp64 conditioning of Eq. 11-12 as printed: 1 - q = 10^(-Q/10) is formed by subtraction from 1, so P_trans carries a
        # relative error of about eps / (1 - q); beyond Q ~ 60 that exceeds one fixed-point ulp (Q = 93: 2e-7 relative)
        qmax = min(93, max(1, max(qu, qv)))
        tol = max(2.0 ** -32, 4 * 2.0 ** -53 * 10.0 ** (qmax / 10.0) / np.log(10.0))
        assert abs(got - w) <= tol, (qu, qv, got, w, tol)
    same = lambda a, b: np.array_equal(oracle.snp_graph(one_fragment([0, 1], [0, 1], list(a), n_snp=2), 10, 0.1)["w_fx"],
                                       oracle.snp_graph(one_fragment([0, 1], [0, 1], list(b), n_snp=2), 10, 0.1)["w_fx"])
    assert same((0, 20), (1, 20)) and same((200, 20), (93, 20)) and same((94, 0), (93, 1)) and not same((2, 20), (1, 20)) \
        and not same((92, 20), (93, 20))


def test_R17_stitch_tie_keeps_orientation(oracle):
    """Reading R17: a block is flipped only when the overlap DISAGREES with the (already oriented) previous block, i.e. when
    the agreement sum is negative; a tie (sum = 0) keeps the block as solved.  Two blocks, overlap of two SNPs, one agreeing
    and one disagreeing -> no flip; make both disagree -> flip; the tie rule also chains through an already flipped block."""
    win = np.array([[0, 4], [2, 6]], np.int64)
    b0 = np.array([1, 1, 1, -1], np.int8)
    b1 = np.array([1, 1, -1, 1], np.int8)            # overlap SNPs 2, 3: b0 = (1, -1), b1 = (1, 1) -> +1 - 1 = 0: tie
    out = oracle.block_stitch(6, win, [b0, b1])
    assert out.tolist() == [1, 1, 1, 1, -1, 1]       # block 0 owns [0, 3), block 1 owns [3, 6), unflipped
    b1f = np.array([-1, 1, -1, 1], np.int8)          # overlap (−1, 1) vs (1, −1): both disagree -> flipped
    assert oracle.block_stitch(6, win, [b0, b1f]).tolist() == [1, 1, 1, -1, 1, -1]
    win3 = np.array([[0, 4], [2, 6], [4, 8]], np.int64)
    b2 = np.array([1, -1, 1, 1], np.int8)            # vs oriented block 1 (flipped b1f = (1,-1,1,-1)) on SNPs 4, 5: (1,-1) vs (1,-1): agree
    assert oracle.block_stitch(8, win3, [b0, b1f, b2]).tolist() == [1, 1, 1, -1, 1, -1, 1, 1]
    b2t = np.array([1, 1, 1, 1], np.int8)            # (1,-1) vs (1,1): tie -> kept
    assert oracle.block_stitch(8, win3, [b0, b1f, b2t]).tolist() == [1, 1, 1, -1, 1, 1, 1, 1]


# ------------------------------------------------------------------------------------- O3 dSB variant
def test_dsb_force_uses_signs_only(oracle):
    """PAPER.md:L71-L77 (dSB in the bake-off): the force is J sgn(x).  (i) J = 0: identical to bSB.  (ii) The increment of y
    beyond the spin's own -dt (a0 - a_k) x term depends only on the SIGNS of the other spins: rescaling every |x_j| by an
    arbitrary positive factor leaves it unchanged bit for bit (it would not under bSB).  (iii) hand values on two coupled
    spins, including sgn(0) = +1.  (iv) while no sign changes, the step is an affine map: explicit matrix product."""
    rp0 = np.zeros(4, np.int32); e = np.zeros(0, np.int32)
    x0 = np.array([[0.3, -0.2], [0.05, 0.0], [-0.6, 0.4]]); y0 = np.array([[0.1, 0.2], [-0.3, 0.0], [0.2, -0.1]])
    a = oracle.bsb_run(rp0, e, np.zeros(0, np.float32), x0.copy(), y0.copy(), steps_total=9, steps_run=4, c0=0.3, force_mode=1)
    b = oracle.bsb_run(rp0, e, np.zeros(0, np.float32), x0.copy(), y0.copy(), steps_total=9, steps_run=4, c0=0.3, force_mode=0)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    rng = np.random.default_rng(2)
    n, R, T, dt, a0, c0 = 7, 5, 30, 0.5, 1.0, 0.125
    J = rng.integers(-3, 4, size=(n, n)).astype(np.float64); J = np.triu(J, 1); J = J + J.T
    rp, cl, jv = csr_from_dense(J)
    x = rng.uniform(-0.5, 0.5, size=(n, R)); y = rng.uniform(-0.1, 0.1, size=(n, R))
    scale = 2.0 ** rng.integers(-3, 1, size=(n, R)).astype(np.float64)           # exact rescaling, signs kept
    k = 11
    a_k = a0 * k / (T - 1)
    incs = []
    for xs in (x, x * scale):
        _, y1, _ = oracle.bsb_run(rp, cl, jv, xs.copy(), y.copy(), steps_total=T, step_begin=k, steps_run=1, dt=dt, a0=a0, c0=c0, force_mode=1)
        incs.append(y1 - (y + dt * (-(a0 - a_k) * xs)))
    clamped = np.abs(oracle.bsb_run(rp, cl, jv, x.copy(), y.copy(), steps_total=T, step_begin=k, steps_run=1, dt=dt, a0=a0, c0=c0, force_mode=1)[0]) == 1.0
    assert not clamped.any()
    np.testing.assert_allclose(incs[0], incs[1], rtol=0, atol=1e-15)
    np.testing.assert_allclose(incs[0], dt * c0 * (J @ np.where(x >= 0, 1.0, -1.0)), rtol=0, atol=1e-15)       # = dt c0 J sgn(x): library matmul
    _, yb, _ = oracle.bsb_run(rp, cl, jv, (x * scale).copy(), y.copy(), steps_total=T, step_begin=k, steps_run=1, dt=dt, a0=a0, c0=c0, force_mode=0)
    assert np.abs((yb - (y + dt * (-(a0 - a_k) * x * scale))) - incs[0]).max() > 1e-3                          # bSB does depend on |x|
    # (iii) two spins, J01 = -2 (w = 2), x = (0, 0.5): sgn = (+1, +1) -> F = (-2, -2); T = 1 -> a_k = 0
    rp2 = np.array([0, 1, 2], np.int32); cl2 = np.array([1, 0], np.int32); jv2 = np.array([-2, -2], np.float32)
    x2, y2, _ = oracle.bsb_run(rp2, cl2, jv2, np.array([[0.0], [0.5]]), np.array([[0.0], [0.0]]), steps_total=1, dt=0.5, a0=1.0, c0=0.25, force_mode=1)
    assert y2.tolist() == [[0.5 * 0.25 * -2.0], [0.5 * (-0.5 + 0.25 * -2.0)]] and x2.tolist() == [[0.5 * y2[0, 0]], [0.5 + 0.5 * y2[1, 0]]]
    # (iv) antiferromagnetic pair pushed apart: signs (+, -) never change -> affine map z' = M z + b per step
    x0 = np.array([[0.01], [-0.02]]); y0 = np.array([[0.0], [0.0]])
    steps, T = 6, 50
    xa, ya, _ = oracle.bsb_run(rp2, cl2, jv2, x0.copy(), y0.copy(), steps_total=T, steps_run=steps, dt=0.25, a0=1.0, c0=0.1, force_mode=1)
    z = np.vstack([x0, y0, [[1.0]]])
    Fc = 0.25 * 0.1 * (np.array([[0.0, -2.0], [-2.0, 0.0]]) @ np.array([[1.0], [-1.0]]))                     # dt c0 J s, constant
    I = np.eye(2)
    for k in range(steps):
        B = -0.25 * (1.0 - k / (T - 1)) * I
        Mk = np.block([[I + 0.25 * B, 0.25 * I, 0.25 * Fc], [B, I, Fc], [np.zeros((1, 4)), np.ones((1, 1))]])
        z = Mk @ z
    assert np.all(np.abs(xa) < 1.0) and xa[0, 0] > 0 > xa[1, 0]
    np.testing.assert_allclose(np.vstack([xa, ya]), z[:4], rtol=1e-12, atol=1e-18)


def test_eval_every_trace_is_the_cut_at_those_steps(oracle):
    """PAPER.md:L118 (Fig. 3: energy of the best sample at every time step): the trace rows equal a fresh cut evaluation of
    sign(x) after exactly that many steps (resume property P10), and the run with a trace ends in the same state."""
    fr = tiny_fragments(21, n_snp=60, n_reads=40)
    g = oracle.read_graph(fr)
    w = oracle.read_weights(g, 1); jv = (-w).astype(np.float32)
    x0, y0 = synth.bsb_init_state(5, fr.n_frag, 6)
    T = 60
    res = oracle.solve(g["row_ptr"], g["col"], w, jv, x0, y0, steps_total=T, eval_every=25)
    ref = oracle.solve(g["row_ptr"], g["col"], w, jv, x0, y0, steps_total=T)
    assert np.array_equal(res["x"], ref["x"]) and np.array_equal(res["cut"], ref["cut"])
    assert res["trace_steps"].tolist() == [25, 50] and res["trace"].shape == (2, 6)
    for row, k in zip(res["trace"], res["trace_steps"]):
        xk, _, _ = oracle.bsb_run(g["row_ptr"], g["col"], jv, x0.astype(np.float64), y0.astype(np.float64), steps_total=T, steps_run=int(k))
        assert np.array_equal(row, oracle.cut_eval(g["row_ptr"], g["col"], w, np.where(xk >= 0, 1, -1).astype(np.int8))[0])
