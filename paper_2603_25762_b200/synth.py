"""Seeded synthetic inputs for the QHap hot path (fragment matrices and bSB start states).

This module holds NO arithmetic of the method: it only draws inputs.  It is the one module
that both the CPU oracle's tests and the CUDA path's tests/bench import (numpy only; importing
it never loads the CUDA library).

The recipes restate BASELINE.json's five configs; SURVEY.md section 8(d) "Common generator
rules" fills in what BASELINE.json leaves open.  The paper's own workloads are GIAB HG002 reads
on the MHC region / chr22; these seeded inputs take their shapes and stand
in for them.

Fragment matrix layout = the C ABI's ``qhap_frags`` (include/qhap.h): CSR by fragment, fragments
sorted by first SNP index, ``snp_idx`` strictly ascending inside a fragment, ``allele`` in
{0 ref, 1 alt, 2 missing}, integer Phred ``qual``, ``frag_flags`` bit0 = Pore-C derived.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = [
    "Fragments", "CONFIGS", "make_config", "make_fragments", "make_porec_fragments",
    "merge_fragments", "bsb_init_state", "block_windows", "random_spins",
]


@dataclass
class Fragments:
    """Fragment x het-SNP observations (PAPER.md:L216 last sentence) plus the planted truth."""
    n_frag: int
    n_snp: int
    frag_ptr: np.ndarray      # int64 [n_frag+1]
    snp_idx: np.ndarray       # int32 [nnz]
    allele: np.ndarray        # uint8 [nnz]  0 ref / 1 alt / 2 missing
    qual: np.ndarray          # uint8 [nnz]  integer Phred
    frag_flags: np.ndarray    # uint8 [n_frag]  bit0: Pore-C derived
    h1: np.ndarray            # uint8 [n_snp]  allele carried by initial H1 (gauge)
    # planted truth (never seen by the library)
    hap_a: np.ndarray         # uint8 [n_snp]  truth haplotype A; B is its complement
    frag_hap: np.ndarray      # uint8 [n_frag] 0: read drawn from A, 1: from B
    snp_pos: np.ndarray       # int64 [n_snp]  sorted positions
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.frag_ptr[-1])


# ------------------------------------------------------------------------------------------------
# Config table (BASELINE.json "configs").  "scale" shrinks the region length,
# SNP count and read count together, keeping density, coverage and read-length law.
# ------------------------------------------------------------------------------------------------
CONFIGS = {
    0: dict(name="read-tiny", L=300_000, n_snp=300, n_reads=150, len_law=("uniform", 10_000, 30_000),
            flip=0.02, missing=0.0, qual=("const", 30), graph="read", R=64, T=1000),
    1: dict(name="read-mhc-hifi", L=4_000_000, n_snp=16_000, n_reads=8_000,
            len_law=("lognormal", 15_000, 5_000), flip=0.01, missing=0.0,
            qual=("normal", 30, 5, 5, 60), graph="read", R=1024, T=2000),
    2: dict(name="read-mhc-ont", L=4_000_000, n_snp=16_000, n_reads=4_000,
            len_law=("lognormal", 40_000, 25_000), flip=0.06, missing=0.03,
            qual=("normal", 15, 4, 3, 40), graph="read", R=2048, T=3000),
    3: dict(name="snp-chrom-blocks", L=250_000_000, n_snp=210_000, n_reads=250_000,
            len_law=("lognormal", 30_000, 10_000), flip=0.05, missing=0.0,
            qual=("normal", 18, 5, 3, 40), graph="snp", R=256, T=2000,
            linkage_tenths=3, block=5000, stride=4500),
    4: dict(name="snp-chrom-porec", L=250_000_000, n_snp=210_000, n_reads=250_000,
            len_law=("lognormal", 30_000, 10_000), flip=0.05, missing=0.0,
            qual=("normal", 18, 5, 3, 40), graph="snp", R=128, T=5000,
            linkage_tenths=3, porec_edges=500_000, alpha=0.1),
}
BSB_DT = 1.25
BSB_A0 = 1.0


def _seed_for(cfg: int) -> int:
    return 20260000 + cfg


def _draw_lengths(rng, law, n, L):
    kind = law[0]
    if kind == "uniform":
        ln = rng.uniform(law[1], law[2], size=n)
    elif kind == "lognormal":
        m, s = float(law[1]), float(law[2])
        sigma2 = np.log(1.0 + (s / m) ** 2)
        mu = np.log(m) - sigma2 / 2.0
        ln = rng.lognormal(mu, np.sqrt(sigma2), size=n)
    else:
        raise ValueError(kind)
    return np.clip(ln, 1000.0, float(L)).astype(np.int64)


def _draw_quals(rng, law, n):
    if law[0] == "const":
        return np.full(n, law[1], dtype=np.uint8)
    _, mean, sd, lo, hi = law
    q = np.rint(rng.normal(mean, sd, size=n))
    return np.clip(q, lo, hi).astype(np.uint8)


def _csr_from_ranges(lo, cnt):
    """Concatenate integer ranges [lo_i, lo_i+cnt_i) -> (ptr, values)."""
    ptr = np.zeros(len(cnt) + 1, dtype=np.int64)
    np.cumsum(cnt, out=ptr[1:])
    total = int(ptr[-1])
    owner = np.repeat(np.arange(len(cnt), dtype=np.int64), cnt)
    within = np.arange(total, dtype=np.int64) - ptr[owner]
    return ptr, (lo[owner] + within), owner


def _finish(n_snp, ptr, idx, allele, qual, flags, hap_a, frag_hap, pos, meta):
    """Drop fragments with < 2 non-missing entries, sort fragments by first SNP index."""
    n_frag = len(ptr) - 1
    cnt = np.diff(ptr)
    owner = np.repeat(np.arange(n_frag, dtype=np.int64), cnt)
    informative = np.bincount(owner, weights=(allele != 2).astype(np.float64), minlength=n_frag)
    first = np.full(n_frag, n_snp, dtype=np.int64)
    nz = cnt > 0
    first[nz] = idx[ptr[:-1][nz]]
    keep = informative >= 2
    order = np.argsort(first, kind="stable")
    order = order[keep[order]]
    new_cnt = cnt[order]
    new_ptr, src, _ = _csr_from_ranges(ptr[:-1][order], new_cnt)
    return Fragments(
        n_frag=len(order), n_snp=int(n_snp), frag_ptr=new_ptr,
        snp_idx=idx[src].astype(np.int32), allele=allele[src].astype(np.uint8),
        qual=qual[src].astype(np.uint8), frag_flags=flags[order].astype(np.uint8),
        h1=np.zeros(n_snp, dtype=np.uint8), hap_a=hap_a.astype(np.uint8),
        frag_hap=frag_hap[order].astype(np.uint8), snp_pos=pos.astype(np.int64), meta=meta)


def make_fragments(*, seed, L, n_snp, n_reads, len_law, flip, missing, qual, hap_a=None, snp_pos=None,
                   **_ignored) -> Fragments:
    """Contiguous long reads over a planted diploid genome (SURVEY.md 8(d) common rules)."""
    rng = np.random.default_rng(seed)
    if snp_pos is None:
        snp_pos = np.sort(rng.choice(L, size=n_snp, replace=False)).astype(np.int64)
    if hap_a is None:
        hap_a = rng.integers(0, 2, size=n_snp, dtype=np.uint8)
    frag_hap = rng.integers(0, 2, size=n_reads, dtype=np.uint8)
    ln = _draw_lengths(rng, len_law, n_reads, L)
    start = np.floor(rng.uniform(0.0, 1.0, size=n_reads) * (L - ln + 1)).astype(np.int64)
    lo = np.searchsorted(snp_pos, start, side="left")
    hi = np.searchsorted(snp_pos, start + ln, side="left")
    cnt = (hi - lo).astype(np.int64)
    ptr, idx, owner = _csr_from_ranges(lo.astype(np.int64), cnt)
    nnz = int(ptr[-1])
    true_allele = hap_a[idx] ^ frag_hap[owner]
    flips = rng.uniform(size=nnz) < flip
    allele = (true_allele ^ flips.astype(np.uint8)).astype(np.uint8)
    if missing > 0:
        allele[rng.uniform(size=nnz) < missing] = 2
    q = _draw_quals(rng, qual, nnz)
    flags = np.zeros(n_reads, dtype=np.uint8)
    meta = dict(seed=seed, L=L, kind="long-read")
    return _finish(n_snp, ptr, idx, allele, q, flags, hap_a, frag_hap, snp_pos, meta)


def make_porec_fragments(*, seed, base: Fragments, L, flip, qual, target_edges,
                         batch=4096, d_min=1e4, d_max=1e8, **_ignored) -> Fragments:
    """Pore-C multi-contact fragments (BASELINE.json config 4).

    contacts ~ U{2..6}; first contact uniform in [0,L); each next contact at distance
    d = d_min * (d_max/d_min)^U from the previous one (P(d) ~ 1/d), random side, redrawn if
    outside; each contact covers U{1,2,3} consecutive SNPs starting at the nearest one.
    Fragments are drawn until ``target_edges`` distinct SNP pairs that join two different
    contacts exist.
    """
    rng = np.random.default_rng(seed)
    pos, n_snp, hap_a = base.snp_pos, base.n_snp, base.hap_a
    ptrs, idxs, als, qs, haps = [np.zeros(1, dtype=np.int64)], [], [], [], []
    seen = np.zeros(0, dtype=np.int64)
    n_frag_total = 0
    while len(seen) < target_edges:
        ncont = rng.integers(2, 7, size=batch)
        hap = rng.integers(0, 2, size=batch, dtype=np.uint8)
        cur = rng.uniform(0.0, L, size=batch)
        rows = []       # (frag, contact_id, snp)
        for c in range(6):
            active = ncont > c
            if c > 0:
                nxt = cur.copy()
                todo = active.copy()
                for _ in range(64):
                    if not todo.any():
                        break
                    k = int(todo.sum())
                    d = d_min * (d_max / d_min) ** rng.uniform(size=k)
                    sgn = np.where(rng.uniform(size=k) < 0.5, -1.0, 1.0)
                    cand = cur[todo] + sgn * d
                    ok = (cand >= 0) & (cand < L)
                    t_idx = np.flatnonzero(todo)
                    nxt[t_idx[ok]] = cand[ok]
                    todo[t_idx[ok]] = False
                active &= ~todo          # could not place within 64 tries: contact skipped
                cur = np.where(active, nxt, cur)
            near = np.clip(np.searchsorted(pos, cur.astype(np.int64), side="left"), 0, n_snp - 1)
            width = rng.integers(1, 4, size=batch)
            for w in range(3):
                sel = active & (width > w) & (near + w < n_snp)
                f = np.flatnonzero(sel)
                rows.append(np.stack([f, np.full(len(f), c), near[sel] + w], axis=1))
        rows = np.concatenate(rows, axis=0).astype(np.int64)
        # strictly ascending snp_idx inside a fragment: sort by (frag, snp), drop duplicates
        key = rows[:, 0] * n_snp + rows[:, 2]
        _, first = np.unique(key, return_index=True)
        rows = rows[first]
        frag, cont, snp = rows[:, 0], rows[:, 1], rows[:, 2]
        cnt = np.bincount(frag, minlength=batch).astype(np.int64)
        # long-range pairs of this batch: all pairs inside a fragment whose contacts differ
        fptr = np.zeros(batch + 1, dtype=np.int64)
        np.cumsum(cnt, out=fptr[1:])
        new_keys = []
        maxc = int(cnt.max()) if len(cnt) else 0
        within = np.arange(len(frag)) - fptr[frag]
        for sh in range(1, maxc):
            ok = within + sh < cnt[frag]
            i0 = np.flatnonzero(ok)
            i1 = i0 + sh
            diff = cont[i0] != cont[i1]
            new_keys.append(snp[i0][diff] * n_snp + snp[i1][diff])
        if new_keys:
            seen = np.union1d(seen, np.concatenate(new_keys))
        nn = len(frag)
        true_allele = hap_a[snp] ^ hap[frag]
        allele = (true_allele ^ (rng.uniform(size=nn) < flip).astype(np.uint8)).astype(np.uint8)
        ptrs.append(fptr[1:] + ptrs[-1][-1])
        idxs.append(snp); als.append(allele); qs.append(_draw_quals(rng, qual, nn)); haps.append(hap)
        n_frag_total += batch
    ptr = np.concatenate(ptrs)
    flags = np.ones(n_frag_total, dtype=np.uint8)
    meta = dict(seed=seed, L=L, kind="pore-c", long_range_edges=int(len(seen)), drawn_fragments=n_frag_total)
    return _finish(n_snp, ptr, np.concatenate(idxs), np.concatenate(als), np.concatenate(qs), flags,
                   hap_a, np.concatenate(haps), pos, meta)


def merge_fragments(a: Fragments, b: Fragments) -> Fragments:
    """Union of two fragment sets over the same SNPs, re-sorted by first SNP index."""
    assert a.n_snp == b.n_snp
    ptr = np.concatenate([a.frag_ptr, b.frag_ptr[1:] + a.frag_ptr[-1]])
    meta = dict(a.meta); meta.update({"merged_" + k: v for k, v in b.meta.items()})
    return _finish(a.n_snp, ptr, np.concatenate([a.snp_idx, b.snp_idx]).astype(np.int64),
                   np.concatenate([a.allele, b.allele]), np.concatenate([a.qual, b.qual]),
                   np.concatenate([a.frag_flags, b.frag_flags]), a.hap_a,
                   np.concatenate([a.frag_hap, b.frag_hap]), a.snp_pos, meta)


def make_config(cfg: int, scale: float = 1.0, seed: int | None = None, porec_edges: int = 0) -> tuple[Fragments, dict]:
    """Fragments + solver parameters of BASELINE.json config ``cfg`` (optionally shrunk by ``scale``).

    ``porec_edges`` > 0 on a read-based config adds Pore-C multi-contact fragments (contact distances 10 kb .. L) until that
    many long-range SNP pairs exist: the reads of such a region no longer form a banded read graph (SURVEY.md
    8(f) f3)."""
    p = dict(CONFIGS[cfg])
    seed = _seed_for(cfg) if seed is None else seed
    if scale != 1.0:
        p["L"] = max(int(p["L"] * scale), 50_000)
        p["n_snp"] = max(int(p["n_snp"] * scale), 16)
        p["n_reads"] = max(int(p["n_reads"] * scale), 8)
        if "porec_edges" in p:
            p["porec_edges"] = max(int(p["porec_edges"] * scale), 16)
    # configs 3 and 4 share the same long reads (BASELINE.json: "config 3's ... graph")
    base_seed = _seed_for(3) if cfg == 4 and seed == _seed_for(4) else seed
    fr = make_fragments(seed=base_seed, **p)
    if cfg == 4:
        pc = make_porec_fragments(seed=seed + 7919, base=fr, L=p["L"], flip=p["flip"], qual=p["qual"],
                                  target_edges=p["porec_edges"])
        fr = merge_fragments(fr, pc)
    if porec_edges > 0 and cfg != 4:
        pc = make_porec_fragments(seed=seed + 7919, base=fr, L=p["L"], flip=p["flip"], qual=p["qual"],
                                  target_edges=int(porec_edges), batch=256, d_min=1e4, d_max=float(p["L"]))
        fr = merge_fragments(fr, pc)
        p["name"] += f"+porec{int(porec_edges)}"
    p["dt"], p["a0"], p["seed"] = BSB_DT, BSB_A0, seed
    return fr, p


# ------------------------------------------------------------------------------------------------
# bSB start state: x0, y0 ~ U(-0.1, 0.1) "from seed" (BASELINE.json config 0).  Counter-based so that
# the library's on-device initialiser (x == NULL) can reproduce it bit for bit (reading R11).
#   idx  = (r * n + i) * 2 + (0 for x, 1 for y)          r = replica, i = spin (global row)
#   z    = splitmix64_finalise(seed + GOLDEN * (idx + 1))
#   u    = z >> 40                                        24 bits
#   val  = fp32( fp64(2u + 1 - 2^24) * fp64(0.1 * 2^-24) )    one fp64 multiply, one rounding to fp32
# ------------------------------------------------------------------------------------------------
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    z = z.copy()
    z ^= z >> np.uint64(30); z *= np.uint64(0xBF58476D1CE4E5B9)
    z ^= z >> np.uint64(27); z *= np.uint64(0x94D049BB133111EB)
    z ^= z >> np.uint64(31)
    return z


def bsb_init_state(seed: int, n: int, replicas: int) -> tuple[np.ndarray, np.ndarray]:
    """x0, y0 as fp32 arrays of shape [n, replicas] (replica index contiguous)."""
    with np.errstate(over="ignore"):
        i = np.arange(n, dtype=np.uint64)[:, None]
        r = np.arange(replicas, dtype=np.uint64)[None, :]
        base = (r * np.uint64(n) + i) * np.uint64(2)
        out = []
        for which in (0, 1):
            idx = base + np.uint64(which)
            z = _splitmix64(np.uint64(seed) + _GOLDEN * (idx + np.uint64(1)))
            u = (z >> np.uint64(40)).astype(np.int64)
            v = (2 * u + 1 - (1 << 24)).astype(np.float64) * (0.1 / float(1 << 24))
            out.append(v.astype(np.float32))
    return out[0], out[1]


def random_spins(seed: int, n: int, replicas: int) -> np.ndarray:
    """int8 spins in {-1,+1}, shape [n, replicas]; for cut-evaluation parity tests."""
    rng = np.random.default_rng(seed)
    return (rng.integers(0, 2, size=(n, replicas), dtype=np.int8) * 2 - 1).astype(np.int8)


def block_windows(n: int, block: int, stride: int) -> np.ndarray:
    """Overlapping index windows [start, end) covering 0..n: int64 [nb, 2]."""
    starts = [0]
    while starts[-1] + block < n:
        starts.append(starts[-1] + stride)
    return np.array([[s, min(s + block, n)] for s in starts], dtype=np.int64)
