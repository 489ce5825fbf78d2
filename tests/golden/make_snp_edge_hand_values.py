#!/usr/bin/env python
"""Writes tests/golden/snp_edge_hand_values.txt and tests/golden/snp_edge_depth_porec_clamp.txt.

A 50-digit evaluation (mpmath) of the formulas PAPER.md prints for ONE fragment's contribution to an SNP-graph edge:
  q = 1 - 10^(-Q/10)                                   (Eq. 9,  PAPER.md:L289-L295)
  P_cis = q_u q_v + (1 - q_u)(1 - q_v)                 (Eq. 11)
  P_trans = q_u (1 - q_v) + (1 - q_u) q_v              (Eq. 12)
  l = sgn(W_iu W_iv) log10(P_cis / P_trans)            (Eq. 13)
  w_uv = - alpha_i l / (|S_i| - 1)                     (Eq. 14; alpha: L350)
and of the linkage-depth rule "nearest floor(k (N-1) / 10) downstream SNPs" (L85).
It imports nothing from oracle/ or from the CUDA package: the expected values are independent of both.
Run:  python tests/golden/make_snp_edge_hand_values.py      (rewrites the two .txt files in place)
"""
from pathlib import Path

import mpmath as mp

mp.mp.dps = 50
HERE = Path(__file__).resolve().parent


def llr(qu, qv):
    a = 1 - mp.mpf(10) ** (-mp.mpf(qu) / 10)
    b = 1 - mp.mpf(10) ** (-mp.mpf(qv) / 10)
    return mp.log10((a * b + (1 - a) * (1 - b)) / (a * (1 - b) + (1 - a) * b))


def term(qu, qv, k, same, alpha_i):
    return -(mp.mpf(alpha_i) * (1 if same else -1) * llr(qu, qv)) / (k - 1)


def fmt(v):
    return mp.nstr(v, 20)


def hand_values():
    out = ["# Closed-form values of one fragment's contribution to w_uv, PAPER.md:L287-L319 (Eq. 9, 11, 12, 13, 14) and L350 (alpha).",
           "# One fragment covering k SNPs, pair (u,v) with Phred Qu,Qv, equal (same=1) or opposite (same=0) alleles w.r.t. h1 = all-ref,",
           "# Pore-C flag pc.  Worked by hand: Q=10 -> q=0.9, P_cis=0.82, P_trans=0.18, w = -log10(0.82/0.18) = -0.658541...;",
           "# digits below from a 50-digit evaluation (mpmath) of the printed formulas, independent of oracle/:",
           "# written by tests/golden/make_snp_edge_hand_values.py.",
           "# Qu Qv k same pc alpha  w_uv"]
    rows = [(10, 10, 2, 1, 0), (20, 20, 2, 1, 0), (30, 30, 2, 1, 0), (10, 30, 2, 1, 0), (3, 3, 2, 1, 0), (3, 40, 2, 1, 0),
            (20, 20, 3, 1, 0), (20, 20, 2, 1, 1), (20, 20, 2, 0, 0)]
    for qu, qv, k, same, pc in rows:
        v = term(qu, qv, k, same, "0.1" if pc else 1)
        out.append(f"{qu:<2d} {qv:<2d} {k} {same} {pc} 0.1 {fmt(v)}")
    (HERE / "snp_edge_hand_values.txt").write_text("\n".join(out) + "\n")


def depth_porec_clamp():
    """One fragment of k = 5 SNPs (indices 0..4, all alleles = h1, Phred Q_j below); the edge list that the linkage depth
    and the Pore-C flag must produce, with every weight.  Rows: tenths flag alpha u v w_uv.
    flag 0, depth 3/10: reach = floor(3 * 4 / 10) = 1 -> the 4 adjacent pairs only (L85).
    flag 1, depth 3/10: Pore-C fragments keep ALL 10 pairs (R8: their contacts are far apart by construction,
                        a depth limit would delete exactly the long-range links L344-L350 add them for) and every term is
                        scaled by alpha (L350).
    Phred clamp (R5): Q = 0 would give q = 0 and Q > 93 is outside the table; both are clamped to [1, 93], so a
    fragment with Q = (0, 20) weighs like Q = (1, 20) and Q = (200, 20) like Q = (93, 20).  Rows: 'clamp' Qu_in Qv_in w_uv."""
    Q = [12, 25, 7, 33, 18]
    k = len(Q)
    out = ["# Linkage depth (PAPER.md:L85), Pore-C exhaustive depth + alpha scaling (L344-L350, DESIGN.md R8) and the Phred clamp",
           "# (DESIGN.md R5) on hand-made fragments; 50-digit mpmath evaluation of Eq. 9-14, independent of oracle/:",
           "# written by tests/golden/make_snp_edge_hand_values.py.",
           f"# fragment: SNPs 0..{k - 1}, alleles all equal to h1, Phred {' '.join(map(str, Q))}",
           "# edge tenths flag alpha u v  w_uv      (every edge the build must emit for that (tenths, flag); nothing else)"]
    for tenths, flag, alpha in ((3, 0, "0.1"), (3, 1, "0.1"), (10, 0, "0.1"), (6, 1, "0.25")):
        reach = (k - 1) if flag else (tenths * (k - 1)) // 10
        for u in range(k):
            for v in range(u + 1, min(k - 1, u + reach) + 1):
                out.append(f"edge {tenths} {flag} {alpha} {u} {v} {fmt(term(Q[u], Q[v], k, 1, alpha if flag else 1))}")
    out.append("# clamp Qu_in Qv_in  w_uv          (k = 2, equal alleles, flag 0)")
    for qu_in, qv_in in ((0, 20), (1, 20), (200, 20), (93, 20), (94, 94), (0, 0)):
        cl = lambda q: min(93, max(1, q))
        out.append(f"clamp {qu_in} {qv_in} {fmt(term(cl(qu_in), cl(qv_in), 2, 1, 1))}")
    (HERE / "snp_edge_depth_porec_clamp.txt").write_text("\n".join(out) + "\n")


if __name__ == "__main__":
    hand_values()
    depth_porec_clamp()
    print("wrote", HERE / "snp_edge_hand_values.txt", "and", HERE / "snp_edge_depth_porec_clamp.txt")
