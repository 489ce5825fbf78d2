// QHap CPU oracle -- TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct restatement of what the QHap hot path computes
// (arxiv/paper_2603_25762; citations are /root/reference/PAPER.md line numbers).  Integers and fp64.
// It shares no code with the CUDA path (paper_2603_25762_b200/csrc) and neither includes the other.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
//
// Pins (tests/test_oracle_pins.py) and what stays "parity unpinned":
//   O1 read graph, O2 SNP graph, O4 cut/energy, O5 readouts+metrics: pinned (library matmul special
//   case, closed forms, hand values, brute force, the paper's SE/HE worked example); the readings sgn(0) = +1
//   (R10e), Pore-C fragments' exhaustive reach and alpha (R8), the Phred clamp [1, 93] (R5) and the stitch tie
//   rule (R17) each have a hand-made pin (tests/golden/snp_edge_depth_porec_clamp.txt for R5 / R8).
//   O3 bSB: its ARITHMETIC and update order are pinned (explicit linear-map product, scalar
//   recurrence, exact symmetries; dSB: sign-only force, hand values, affine-map product), its solution quality by
//   brute force and planted recovery; the
//   CONSTANTS c0, the ramp end points and the wall rule are "parity unpinned" against the paper,
//   which prints no bSB equation (PAPER.md:L265 is prose) -- see DESIGN.md readings R10a-f.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC -pthread (oracle/oracle.py does it).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <map>
#include <thread>
#include <utility>
#include <vector>

namespace {

struct DC { int32_t d = 0, c = 0; };

inline uint64_t pair_key(int32_t a, int32_t b) { return (uint64_t(uint32_t(a)) << 32) | uint32_t(b); }

// Emit a symmetric CSR (both (a,b) and (b,a), columns ascending) from a map keyed by (a<b).
template <class V, class Emit>
int64_t emit_symmetric(int32_t n, const std::map<uint64_t, V>& edges, int32_t* row_ptr, int64_t capacity, Emit emit) {
  std::vector<std::vector<std::pair<int32_t, const V*>>> rows(n);
  for (auto& kv : edges) {
    int32_t a = int32_t(kv.first >> 32), b = int32_t(kv.first & 0xffffffffu);
    rows[a].push_back({b, &kv.second});
    rows[b].push_back({a, &kv.second});
  }
  int64_t nnz = 2 * int64_t(edges.size());
  if (row_ptr == nullptr || capacity < nnz) return nnz;
  int64_t e = 0;
  for (int32_t a = 0; a < n; ++a) {
    row_ptr[a] = int32_t(e);
    std::sort(rows[a].begin(), rows[a].end(), [](auto& x, auto& y) { return x.first < y.first; });
    for (auto& pr : rows[a]) emit(e++, pr.first, *pr.second);
  }
  row_ptr[n] = int32_t(e);
  return nnz;
}

}  // namespace

extern "C" {

// ------------------------------------------------------------------------------------------------
// O1  Read graph.  PAPER.md:L226-L246: ternary matrix M (Eq. 1), column span per SNP (L237), conflict
// indicator delta = 1[M_aj * M_bj = -1] (Eq. 2), w_ab = sum_j delta (Eq. 3).  We also count the
// complement C_ab = #shared positions with M_aj * M_bj = +1, because BASELINE.json config 0 defines the
// weight as "discordant minus concordant" (reading R1).  Edge set = pairs with D + C >= 1.
// Returns the directed nnz; fills the arrays only if row_ptr != NULL and capacity >= nnz.
// ------------------------------------------------------------------------------------------------
int64_t orc_read_graph(int32_t n_frag, int32_t n_snp, const int64_t* frag_ptr, const int32_t* snp_idx,
                       const uint8_t* allele, const uint8_t* h1, int32_t* row_ptr, int32_t* col, int32_t* d,
                       int32_t* c, int64_t capacity) {
  // column lists L_j = fragments with a non-missing observation at SNP j, with their M value
  std::vector<std::vector<std::pair<int32_t, int>>> L(n_snp);
  for (int32_t i = 0; i < n_frag; ++i)
    for (int64_t e = frag_ptr[i]; e < frag_ptr[i + 1]; ++e) {
      if (allele[e] > 1) continue;                                  // "0 otherwise" (Eq. 1): missing
      int32_t j = snp_idx[e];
      int m = (allele[e] == (h1 ? h1[j] : 0)) ? +1 : -1;            // Eq. 1
      L[j].push_back({i, m});
    }
  std::map<uint64_t, DC> edges;
  for (int32_t j = 0; j < n_snp; ++j)
    for (size_t p = 0; p < L[j].size(); ++p)
      for (size_t q = p + 1; q < L[j].size(); ++q) {
        int32_t a = L[j][p].first, b = L[j][q].first;
        if (a == b) continue;
        DC& e = edges[pair_key(std::min(a, b), std::max(a, b))];
        if (L[j][p].second * L[j][q].second == -1) e.d += 1;        // Eq. 2
        else e.c += 1;
      }
  return emit_symmetric(n_frag, edges, row_ptr, capacity, [&](int64_t e, int32_t b, const DC& v) {
    col[e] = b; d[e] = v.d; c[e] = v.c;
  });
}

// ------------------------------------------------------------------------------------------------
// O2  SNP graph.  PAPER.md:L287-L319.  q = 1 - 10^(-Q/10) (Eq. 9); P_cis, P_trans (Eq. 11-12);
// l = sgn(W_iu W_iv) log10(P_cis/P_trans) (Eq. 13); w_uv = - sum_i l / (|S_i| - 1) (Eq. 14).
// Linkage depth k/10: each SNP linked to its nearest floor(k (N-1) / 10) downstream SNPs of the read
// (L85).  Pore-C fragments: contribution scaled by alpha (L350) and always exhaustive depth (R8).
// Sum is canonical: every term rounded to int64 at scale 2^32, then integer-added (R6).
// ------------------------------------------------------------------------------------------------
void orc_llr_table(double* T /* [94*94], index Qu*94+Qv, Q in 0..93 (rows/cols 0 unused) */) {
  for (int qu = 0; qu < 94; ++qu)
    for (int qv = 0; qv < 94; ++qv) {
      double a = 1.0 - std::pow(10.0, -double(qu) / 10.0);          // Eq. 9
      double b = 1.0 - std::pow(10.0, -double(qv) / 10.0);
      double pc = a * b + (1.0 - a) * (1.0 - b);                    // Eq. 11
      double pt = a * (1.0 - b) + (1.0 - a) * b;                    // Eq. 12
      T[qu * 94 + qv] = (qu == 0 || qv == 0) ? 0.0 : std::log10(pc / pt);
    }
}

int64_t orc_snp_graph(int32_t n_frag, int32_t n_snp, const int64_t* frag_ptr, const int32_t* snp_idx,
                      const uint8_t* allele, const uint8_t* qual, const uint8_t* frag_flags, const uint8_t* h1,
                      int32_t linkage_tenths, double alpha, int32_t* row_ptr, int32_t* col, int64_t* w_fx,
                      float* w, int64_t capacity) {
  std::vector<double> T(94 * 94);
  orc_llr_table(T.data());
  std::map<uint64_t, int64_t> edges;
  for (int32_t i = 0; i < n_frag; ++i) {
    std::vector<int64_t> S;                                         // non-missing entries, ascending snp
    for (int64_t e = frag_ptr[i]; e < frag_ptr[i + 1]; ++e)
      if (allele[e] <= 1) S.push_back(e);
    int64_t k = int64_t(S.size());
    if (k < 2) continue;
    bool porec = frag_flags && (frag_flags[i] & 1);
    int64_t reach = porec ? (k - 1) : (int64_t(linkage_tenths) * (k - 1)) / 10;   // floor, L85
    double alpha_i = porec ? alpha : 1.0;                           // L350
    for (int64_t p = 0; p < k; ++p)
      for (int64_t t = p + 1; t <= std::min(k - 1, p + reach); ++t) {
        int64_t eu = S[p], ev = S[t];
        int32_t u = snp_idx[eu], v = snp_idx[ev];
        bool mu = allele[eu] == (h1 ? h1[u] : 0), mv = allele[ev] == (h1 ? h1[v] : 0);
        double sg = (mu == mv) ? 1.0 : -1.0;                        // sgn(W_iu W_iv), Eq. 13
        int qu = std::min(93, std::max(1, int(qual[eu]))), qv = std::min(93, std::max(1, int(qual[ev])));
        double term = -(alpha_i * sg * T[qu * 94 + qv]) / double(k - 1);          // Eq. 14
        edges[pair_key(u, v)] += std::llrint(term * 4294967296.0);
      }
  }
  return emit_symmetric(n_snp, edges, row_ptr, capacity, [&](int64_t e, int32_t b, const int64_t& v) {
    col[e] = b; w_fx[e] = v; w[e] = float(double(v) * (1.0 / 4294967296.0));
  });
}

// ------------------------------------------------------------------------------------------------
// O3  bSB.  PAPER.md:L252-L265 (J = -A, Eq. 4; "continuous spin and momentum variables", "adiabatic
// schedule", "boundary constraints and momentum resets", many samples, s = sgn(x)); constants from
// BASELINE.json (dt, a0, linear ramp 0 -> a0, |x| > 1 -> x = sign(x), y = 0); readings R10a-f.
//   a_k = a0 k / (T-1);  F = J x (x of the previous step for every row);
//   y += dt (-(a0 - a_k) x + c0 F);  x += dt a0 y;  |x| > 1: x = sign(x), y = 0.
// State layout [n][R], replica index contiguous.  jval[e] = J entry = -w (fp32 value, promoted).
// force_mode 1 = dSB, the discrete variant the paper's bake-off contrasts with bSB (Fig. 2-3;
// SURVEY.md 8(f) f4): the force is evaluated on the discretised positions, F = J sgn(x), with sgn(0) = +1 (R10e);
// everything else is unchanged.  force_mode 0 = bSB (the paper's solver, L265).
// ------------------------------------------------------------------------------------------------
double orc_bsb_c0(int32_t n, const int32_t* row_ptr, const float* jval) {
  double ss = 0.0;
  for (int64_t e = 0; e < row_ptr[n]; ++e) ss += double(jval[e]) * double(jval[e]);   // all ordered entries
  if (ss == 0.0 || n < 2) return 1.0;
  return 0.5 * std::sqrt(double(n - 1)) / std::sqrt(ss);
}

static void bsb_slice(int32_t n, const int32_t* row_ptr, const int32_t* col, const float* jval, int32_t R,
                      int32_t steps_total, int32_t step_begin, int32_t steps_run, double dt, double a0, double c0,
                      double* x, double* y, double* xpre, int32_t r0, int32_t r1, int32_t force_mode) {
  std::vector<double> F(size_t(n) * size_t(r1 - r0));
  for (int32_t k = step_begin; k < step_begin + steps_run; ++k) {
    double a_k = (steps_total > 1) ? a0 * double(k) / double(steps_total - 1) : 0.0;
    for (int32_t i = 0; i < n; ++i)
      for (int32_t r = r0; r < r1; ++r) {
        double f = 0.0;
        for (int32_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
          double xj = x[size_t(col[e]) * R + r];
          if (force_mode == 1) xj = (xj >= 0.0) ? 1.0 : -1.0;          // dSB: F = J sgn(x), sgn(0) = +1
          f += double(jval[e]) * xj;
        }
        F[size_t(i) * (r1 - r0) + (r - r0)] = f;
      }
    for (int32_t i = 0; i < n; ++i)
      for (int32_t r = r0; r < r1; ++r) {
        size_t p = size_t(i) * R + r;
        y[p] = y[p] + dt * (-(a0 - a_k) * x[p] + c0 * F[size_t(i) * (r1 - r0) + (r - r0)]);
        x[p] = x[p] + dt * a0 * y[p];
        if (xpre) xpre[p] = x[p];                                   // x before the wall rule (test diagnostics)
        if (std::fabs(x[p]) > 1.0) { x[p] = (x[p] > 0.0) ? 1.0 : -1.0; y[p] = 0.0; }
      }
  }
}

void orc_bsb_run(int32_t n, const int32_t* row_ptr, const int32_t* col, const float* jval, int32_t R,
                 int32_t steps_total, int32_t step_begin, int32_t steps_run, double dt, double a0, double c0,
                 double* x, double* y, double* xpre /* optional [n][R]: x of the last step before the wall rule */,
                 int32_t n_threads, int32_t force_mode /* 0 bSB, 1 dSB */) {
  if (n_threads <= 1) { bsb_slice(n, row_ptr, col, jval, R, steps_total, step_begin, steps_run, dt, a0, c0, x, y, xpre, 0, R, force_mode); return; }
  std::vector<std::thread> th;                                      // replicas are independent (L265)
  for (int32_t t = 0; t < n_threads; ++t) {
    int32_t r0 = int32_t(int64_t(R) * t / n_threads), r1 = int32_t(int64_t(R) * (t + 1) / n_threads);
    if (r1 > r0) th.emplace_back(bsb_slice, n, row_ptr, col, jval, R, steps_total, step_begin, steps_run, dt, a0, c0, x, y, xpre, r0, r1, force_mode);
  }
  for (auto& t : th) t.join();
}

// Same recurrence with J as a dense row-major n x n fp64 matrix (small n; cross-check of the CSR loop).
void orc_bsb_run_dense(int32_t n, const double* J, int32_t R, int32_t steps_total, int32_t step_begin,
                       int32_t steps_run, double dt, double a0, double c0, double* x, double* y) {
  std::vector<double> F(size_t(n) * R);
  for (int32_t k = step_begin; k < step_begin + steps_run; ++k) {
    double a_k = (steps_total > 1) ? a0 * double(k) / double(steps_total - 1) : 0.0;
    for (int32_t i = 0; i < n; ++i)
      for (int32_t r = 0; r < R; ++r) {
        double f = 0.0;
        for (int32_t j = 0; j < n; ++j) f += J[size_t(i) * n + j] * x[size_t(j) * R + r];
        F[size_t(i) * R + r] = f;
      }
    for (size_t p = 0; p < size_t(n) * R; ++p) {
      y[p] = y[p] + dt * (-(a0 - a_k) * x[p] + c0 * F[p]);
      x[p] = x[p] + dt * a0 * y[p];
      if (std::fabs(x[p]) > 1.0) { x[p] = (x[p] > 0.0) ? 1.0 : -1.0; y[p] = 0.0; }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// O4  Cut and Ising energy.  PAPER.md:L254-L263: E(s) = -1/2 s^T J s with J = -A (Eq. 4-5);
// cut(s) = 1/4 sum_{a,b} A_ab (1 - s_a s_b) (Eq. 6) = sum over undirected edges with s_a != s_b.
// In the same integer units E(s) = W_tot - 2 cut(s), W_tot = sum_{a<b} w_ab.  w = canonical integer
// weights per directed CSR entry (D, D-C, or the 2^-32 fixed-point SNP weight).  spins [n][R] in {-1,+1}.
// ------------------------------------------------------------------------------------------------
void orc_cut_eval(int32_t n, const int32_t* row_ptr, const int32_t* col, const int64_t* w, const int8_t* spins,
                  int32_t R, int64_t* cut, int64_t* energy) {
  for (int32_t r = 0; r < R; ++r) {
    int64_t cs = 0, wtot = 0;
    for (int32_t a = 0; a < n; ++a)
      for (int32_t e = row_ptr[a]; e < row_ptr[a + 1]; ++e) {
        int32_t b = col[e];
        if (b <= a) continue;                                       // each undirected edge once
        wtot += w[e];
        if (spins[size_t(a) * R + r] != spins[size_t(b) * R + r]) cs += w[e];
      }
    cut[r] = cs;
    if (energy) energy[r] = wtot - 2 * cs;
  }
}

// s = sgn(x) with sgn(0) = +1 (R10e); best replica = lowest index with maximal cut.
void orc_sign_spins(int64_t count, const double* x, int8_t* s) {
  for (int64_t p = 0; p < count; ++p) s[p] = (x[p] >= 0.0) ? 1 : -1;
}
int32_t orc_best_replica(int32_t R, const int64_t* cut) {
  int32_t best = 0;
  for (int32_t r = 1; r < R; ++r) if (cut[r] > cut[best]) best = r;
  return best;
}

// ------------------------------------------------------------------------------------------------
// O5  Readouts and metrics.
// Read-based vote, PAPER.md:L271-L281 (Eq. 7-8; the rule at L279 is partly garbled, reading R13):
//   v_j = sum_i s_i M_ij = (c1+ - c1-) - (c2+ - c2-);  H1'[j] = H1 allele if v_j > 0, the other allele
//   if v_j < 0, unphased (-1) if v_j == 0 (covers zero coverage and equal support, L281).
// SNP-based: hap1[u] = h1[u] if s_u > 0 else 1 - h1[u] (L336-L338 with a single solve).
// ------------------------------------------------------------------------------------------------
void orc_read_vote(int32_t n_frag, int32_t n_snp, const int64_t* frag_ptr, const int32_t* snp_idx, const uint8_t* allele,
                   const uint8_t* h1, const int8_t* spins, int8_t* hap1) {
  std::vector<int64_t> v(n_snp, 0);
  for (int32_t i = 0; i < n_frag; ++i)
    for (int64_t e = frag_ptr[i]; e < frag_ptr[i + 1]; ++e) {
      if (allele[e] > 1) continue;
      int32_t j = snp_idx[e];
      int m = (allele[e] == (h1 ? h1[j] : 0)) ? +1 : -1;
      v[j] += int64_t(spins[i]) * m;
    }
  for (int32_t j = 0; j < n_snp; ++j) {
    uint8_t hj = h1 ? h1[j] : 0;
    hap1[j] = v[j] > 0 ? int8_t(hj) : (v[j] < 0 ? int8_t(1 - hj) : int8_t(-1));
  }
}

void orc_snp_readout(int32_t n_snp, const uint8_t* h1, const int8_t* spins, int8_t* hap1) {
  for (int32_t u = 0; u < n_snp; ++u) {
    uint8_t hu = h1 ? h1[u] : 0;
    hap1[u] = spins[u] > 0 ? int8_t(hu) : int8_t(1 - hu);
  }
}

// Block stitch (reading R17): blocks b with windows [win[2b], win[2b+1]); block_spins concatenated.
// o_0 = +1; o_b = +1 if sum_{i in overlap(b-1,b)} (o_{b-1} s^{b-1}_i) s^b_i >= 0 else -1;
// block b owns [m_b, m_{b+1}), m_0 = 0, m_b = floor((start_b + end_{b-1}) / 2), m_nb = n.
void orc_block_stitch(int32_t n, int32_t nb, const int64_t* win, const int8_t* block_spins, int8_t* out) {
  std::vector<int64_t> off(nb + 1, 0);
  for (int32_t b = 0; b < nb; ++b) off[b + 1] = off[b] + (win[2 * b + 1] - win[2 * b]);
  std::vector<int> o(nb, 1);
  for (int32_t b = 1; b < nb; ++b) {
    int64_t agree = 0;
    for (int64_t i = win[2 * b]; i < win[2 * (b - 1) + 1]; ++i)
      agree += int64_t(o[b - 1]) * block_spins[off[b - 1] + (i - win[2 * (b - 1)])] * block_spins[off[b] + (i - win[2 * b])];
    o[b] = agree >= 0 ? 1 : -1;
  }
  for (int32_t b = 0; b < nb; ++b) {
    int64_t lo = b == 0 ? 0 : (win[2 * b] + win[2 * (b - 1) + 1]) / 2;
    int64_t hi = b == nb - 1 ? n : (win[2 * (b + 1)] + win[2 * b + 1]) / 2;
    for (int64_t i = lo; i < hi; ++i) out[i] = int8_t(o[b] * block_spins[off[b] + (i - win[2 * b])]);
  }
}

// Block split (reading R17; BASELINE.json config 3 "independent 5k-SNP overlapping blocks"): block b is the
// sub-graph induced by the SNP window [win[2b], win[2b+1]) -- an edge belongs to the block iff both ends are
// inside.  Output: block-diagonal CSR over the concatenated blocks (row/col = offset_b + (g - start_b)).
// Returns the directed nnz; fills only if out_row_ptr != NULL and capacity >= nnz.
int64_t orc_block_split(int32_t n, const int32_t* row_ptr, const int32_t* col, const int64_t* w_fx, const float* w,
                        int32_t nb, const int64_t* win, int32_t* out_row_ptr, int32_t* out_col, int64_t* out_w_fx,
                        float* out_w, int64_t capacity) {
  (void)n;
  int64_t nnz = 0;
  for (int32_t b = 0; b < nb; ++b)
    for (int64_t g = win[2 * b]; g < win[2 * b + 1]; ++g)
      for (int32_t e = row_ptr[g]; e < row_ptr[g + 1]; ++e)
        if (col[e] >= win[2 * b] && col[e] < win[2 * b + 1]) ++nnz;
  if (out_row_ptr == nullptr || capacity < nnz) return nnz;
  int64_t off = 0, o = 0;
  for (int32_t b = 0; b < nb; ++b) {
    for (int64_t g = win[2 * b]; g < win[2 * b + 1]; ++g) {
      out_row_ptr[off + (g - win[2 * b])] = int32_t(o);
      for (int32_t e = row_ptr[g]; e < row_ptr[g + 1]; ++e)
        if (col[e] >= win[2 * b] && col[e] < win[2 * b + 1]) {
          out_col[o] = int32_t(off + (col[e] - win[2 * b]));
          if (out_w_fx) out_w_fx[o] = w_fx[e];
          if (out_w) out_w[o] = w[e];
          ++o;
        }
    }
    off += win[2 * b + 1] - win[2 * b];
  }
  out_row_ptr[off] = int32_t(o);
  return nnz;
}

// Switch / Hamming errors.  hap1[j] in {0,1} or -1 (unphased); truth in {0,1}.
// out[0] = switches between consecutive phased SNPs, out[1] = number of phased SNPs,
// out[2] = mismatches against `truth` in the given orientation (the paper's example takes one orientation).
void orc_switch_hamming(int32_t n, const int8_t* hap1, const uint8_t* truth, int64_t* out) {
  int64_t sw = 0, np = 0, mm = 0;
  int prev = -1;
  for (int32_t j = 0; j < n; ++j) {
    if (hap1[j] < 0) continue;
    int diff = (int(hap1[j]) != int(truth[j])) ? 1 : 0;
    if (prev >= 0 && diff != prev) sw += 1;
    prev = diff; np += 1; mm += diff;
  }
  out[0] = sw; out[1] = np; out[2] = mm;
}

int32_t orc_hardware_threads() { return int32_t(std::thread::hardware_concurrency()); }

}  // extern "C"
