// bg_engine.cuh — ordered-current engine for g g -> t tbar + (n-2) g, n = 2..5 gluons.
//
// What it evaluates: the n! colour-flow amplitudes
//     M = sum_sigma J_sigma (T^{a_s1} ... T^{a_sn})_{ij}
// for every helicity configuration, the colour form J^dagger C J, the helicity sum, for BOTH
// parameter sets, and eq. 3.  J_sigma is the colour-ordered amplitude, built from
// colour-ordered currents (the colour-string bookkeeping of SURVEY C5 resolved analytically):
//   gluon current of an ordered tuple t (|t| = m >= 2):
//     J(t) = 1/K_t^2 { -g3 sum_k L3(J(t_1..k), J(t_k+1..m)) + g4 sum_{j<k} V4(J(t_1..j), J(t_j+1..k), J(t_k+1..m)) }
//     J(t reversed) = (-1)^{m+1} J(t)   -> only tuples with t_1 < t_m are stored
//   right quark current (antiquark end)  R(t) = -gq (q-slash+m)/(q^2-m^2) sum_k Jslash(t_1..k) R(t_k+1..m),  q = K_t - p_tbar, R() = v
//   left  quark current (quark end)      L(t) = -gq sum_k L(t_1..m-k) Jslash(t_m-k+1..m) (q'-slash+m)/(q'^2-m^2), q' = p_t - K_t, L() = ubar
//   J_sigma = sum_{i < c <= j} L(s_1..i) Jslash(s_i+1..j) R(s_j+1..n)          (c = split position; common factor i gq dropped)
// Every diagram of SURVEY C6 is contained exactly once (each composition of sigma has one block covering position c).
//
// B200 mapping: one persistent CTA per SM works on E event slots at a time; all currents of a slot live in
// shared memory as SoA planes [component][entry] (conflict-free for consecutive helicity variants); a thread
// owns one (current, helicity-variant) task per phase; phases are separated by __syncthreads.  Each current is
// computed once per helicity assignment of the gluons it contains (2^m variants, not 2^n).  The schedule
// (task descriptors) is built on the host at rwgt_create and read through the read-only path.
#pragma once
#include <cuda_runtime.h>
#include <algorithm>
#include <cstdint>
#include <map>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <string>
#include <type_traits>
#include <vector>

#include "../../include/rwgt.h"
#include "rwgt_math.cuh"

constexpr int RWGT_NBUF_N3 = 2;

namespace rwgt {

// ------------------------------------------------------------------------------------------------ host: colour matrix
// C_{ss'} = sum_a Tr(T^{a_s1}..T^{a_sn} T^{a_s'n}..T^{a_s'1}) by repeated use of the SU(N) Fierz identity
//   T^a_ij T^a_kl = 1/2 (d_il d_jk - 1/N d_ij d_kl), exact integers over (2N)^n.  (Independent of the oracle's
// explicit Gell-Mann sum.)
static long long fierz_reduce(std::vector<std::vector<int>> words) {
  const long long N = 3;
  // find a label to contract
  for (size_t w = 0; w < words.size(); w++) {
    if (words[w].empty()) continue;
    int a = words[w][0];
    // same word?
    for (size_t j = 1; j < words[w].size(); j++) if (words[w][j] == a) {
      std::vector<int> Y(words[w].begin() + 1, words[w].begin() + j), Z(words[w].begin() + j + 1, words[w].end());
      // Tr(T^a Y T^a Z) = 1/2 [Tr(Y) Tr(Z) - 1/N Tr(Y Z)]   -> numerators over 2N: N * (..) - (..)
      std::vector<std::vector<int>> w1 = words, w2 = words;
      w1[w] = Y; w1.push_back(Z);
      std::vector<int> YZ = Y; YZ.insert(YZ.end(), Z.begin(), Z.end()); w2[w] = YZ;
      return N * fierz_reduce(w1) - fierz_reduce(w2);
    }
    // other word: Tr(T^a A) Tr(T^a B) = 1/2 [Tr(A B) - 1/N Tr(A) Tr(B)]
    for (size_t u = 0; u < words.size(); u++) if (u != w) for (size_t j = 0; j < words[u].size(); j++) if (words[u][j] == a) {
      std::vector<int> A(words[w].begin() + 1, words[w].end());
      std::vector<int> B(words[u].begin() + j + 1, words[u].end()); B.insert(B.end(), words[u].begin(), words[u].begin() + j);
      std::vector<std::vector<int>> w1, w2;
      for (size_t x = 0; x < words.size(); x++) if (x != w && x != u) { w1.push_back(words[x]); w2.push_back(words[x]); }
      std::vector<int> AB = A; AB.insert(AB.end(), B.begin(), B.end());
      w1.push_back(AB); w2.push_back(A); w2.push_back(B);
      return N * fierz_reduce(w1) - fierz_reduce(w2);
    }
  }
  long long r = 1; for (size_t w = 0; w < words.size(); w++) r *= N;   // Tr(1) = N per remaining empty trace
  return r;
}
static std::vector<double> colour_matrix_fierz(int n) {
  std::vector<std::vector<int>> perms; std::vector<int> p(n); for (int i = 0; i < n; i++) p[i] = i;
  do perms.push_back(p); while (std::next_permutation(p.begin(), p.end()));
  int np = (int)perms.size(); double den = 1; for (int i = 0; i < n; i++) den *= 6.0;
  std::vector<double> C((size_t)np * np);
  // C_{ss'} depends only on s^-1 s': compute row 0 and relabel
  std::map<std::vector<int>, int> rank; for (int i = 0; i < np; i++) rank[perms[i]] = i;
  std::vector<double> row0(np);
  for (int u = 0; u < np; u++) {
    std::vector<int> word = perms[0]; for (int i = n - 1; i >= 0; i--) word.push_back(perms[u][i]);
    row0[u] = (double)fierz_reduce({word}) / den;
  }
  for (int s = 0; s < np; s++) {
    std::vector<int> inv(n); for (int i = 0; i < n; i++) inv[perms[s][i]] = i;
    for (int u = 0; u < np; u++) { std::vector<int> rel(n); for (int i = 0; i < n; i++) rel[i] = inv[perms[u][i]]; C[(size_t)s * np + u] = row0[rank[rel]]; }
  }
  return C;
}

// ------------------------------------------------------------------------------------------------ schedule
// Storage conventions of the current tables (chosen so that the device never needs a run-time sign flip):
//   * entry = base(tuple) + helicity-variant bits of the tuple's gluons in the tuple's own position order
//     (+ the quark helicity bit on top for R/L);
//   * gluon tuples of length 1: one entry set per gluon; length 2: BOTH orientations are stored (J(b,a) = -J(a,b));
//     length 3: the orientation with t_1 < t_3 (J(rev) = +J, only the variant bits are reversed: REF_REV);
//     length 4 (n = 5 only): the orientation that runs along the "forward" direction of the 5-necklace
//     (t_1..t_4, missing label) -- every block of a forward permutation is then stored as used, every block of
//     its reversal is stored reversed (static sign (-1)^{m+1} and static bit reversal on the device);
//   * gluon 0 only has helicity + (parity, reading R5): variants with its bit set are neither computed nor read.
enum : uint32_t { REF_REV = 0x8000u };

struct BgSched {
  int n, c, lmax, rmax, nperm, npair;
  int nG, nR, nL;                    // table entries per slot
  int offD[3][6];                    // descriptor offsets  [0:G,1:R,2:L][level]
  int offT[6], ntask[3][6];          // per phase M: task-list offset, number of G / R / L tasks
  int offF, strideF;                 // finals: one descriptor per permutation pair
  std::vector<uint32_t> words;
  std::vector<double> lfrag;         // Cholesky factor L^T of the colour matrix in mma-fragment order
  double fp_ops[8];                  // operation counts per event and parameter set: L3, V4, slash, lightcone, prop, rowcol, gstore, gstore2
  double fp_final[8];                // the part of fp_ops that belongs to the amplitude phase (the rest: current levels)
};

static int mask_of(const std::vector<int>& t) { int m = 0; for (int x : t) m |= 1 << x; return m; }
static bool has0(const std::vector<int>& t) { for (int x : t) if (x == 0) return true; return false; }
static int pos0(const std::vector<int>& t) { for (size_t i = 0; i < t.size(); i++) if (t[i] == 0) return (int)i; return -1; }
static std::vector<int> reversed(std::vector<int> t) { std::reverse(t.begin(), t.end()); return t; }
// forward direction of a cyclic arrangement: the rotations of the lexicographically smallest of its 2n dihedral images
static bool necklace_forward(const std::vector<int>& s) {
  int n = (int)s.size(); std::vector<int> best; bool best_fwd = true;
  for (int dir = 0; dir < 2; dir++) { std::vector<int> t = dir ? reversed(s) : s;
    for (int r = 0; r < n; r++) { std::vector<int> u(n); for (int i = 0; i < n; i++) u[i] = t[(i + r) % n];
      if (best.empty() || u < best) { best = u; best_fwd = (dir == 0); } } }
  return best_fwd;
}
// is this ordered gluon tuple the stored orientation?
static bool is_stored(int n, const std::vector<int>& t) {
  int m = (int)t.size();
  if (m <= 2) return true;
  if (m == 4 && n == 5) { std::vector<int> s = t; for (int e = 0; e < 5; e++) if (!(mask_of(t) >> e & 1)) s.push_back(e); return necklace_forward(s); }
  return t.front() < t.back();
}
static void all_tuples(int n, int m, std::vector<std::vector<int>>& out) {
  out.clear(); std::vector<int> cur; std::vector<bool> usedl(n, false);
  struct Rec { static void go(int n, int m, std::vector<int>& cur, std::vector<bool>& u, std::vector<std::vector<int>>& out) {
    if ((int)cur.size() == m) { out.push_back(cur); return; }
    for (int i = 0; i < n; i++) if (!u[i]) { u[i] = true; cur.push_back(i); go(n, m, cur, u, out); cur.pop_back(); u[i] = false; } } };
  Rec::go(n, m, cur, usedl, out);
}

// compile-time geometry of the schedule for N gluons (mirrored by build_schedule and checked in bg_create)
__host__ __device__ constexpr int cfact(int n) { return n <= 1 ? 1 : n * cfact(n - 1); }
__host__ __device__ constexpr int ctuples(int n, int m) { return m > n ? 0 : cfact(n) / cfact(n - m); }     // ordered m-tuples of n labels
// table entries per slot after the hole-sharing allocation of build_schedule (checked against the builder in bg_create)
__host__ __device__ constexpr int c_nG(int n) { return n == 2 ? 4 : n == 3 ? 22 : n == 4 ? 112 : 818; }
__host__ __device__ constexpr int c_nR(int n) { return n == 2 ? 10 : n == 3 ? 14 : n == 4 ? 98 : 150; }
__host__ __device__ constexpr int c_nL(int n) { return n == 2 ? 2 : n == 3 ? 14 : n == 4 ? 18 : 150; }
// tasks of one level after parity pruning (gluon 0 at helicity + only)
__host__ __device__ constexpr int c_ntaskG(int n, int m) { int can = ctuples(n, m) / 2, c0 = m * ctuples(n - 1, m - 1) / 2; return ((can - c0) << m) + (c0 << (m - 1)); }
__host__ __device__ constexpr int c_ntaskQ(int n, int m) { int all = ctuples(n, m), c0 = m * ctuples(n - 1, m - 1); return ((all - c0) << (m + 1)) + (c0 << m); }
__host__ __device__ constexpr int pad4(int x) { return (x + 3) / 4 * 4; }
template <int N> struct Geo {
  static constexpr int C = (N + 1) / 2, LMAX = C - 1, RMAX = N - C, NJ = N - C + 1;            // N=2: C=1; 3: 2; 4: 2; 5: 3
  static constexpr int NPERM = cfact(N), NPAIR = NPERM / 2, NPERM_P = (NPERM + 7) / 8 * 8;
  // helicity batches: gluon 0 has helicity + only (parity); NB more gluon helicities are fixed per batch so that a
  // batch is 16 amplitude columns (4 free gluon configurations x 4 quark helicities) for N >= 3
  static constexpr int NB = (N == 5) ? 2 : (N == 4) ? 1 : 0, NBATCH = 1 << NB;
  static constexpr int NFREE = 1 << (N - 1 - NB), NCOL = NFREE * 4;
  // row stride (elements) of the amplitude buffer, bank-conflict-free for the mma B-fragment loads: rows r = lane & 3 must land
  // 8 32-bit banks apart: 64-bit elements: stride = 4 mod 16 elements, 32-bit elements: stride = 8 mod 32
  template <typename TA> __host__ __device__ static constexpr int astr() { return 2 * NCOL + (sizeof(TA) == 8 ? 4 : 8); }
  template <typename TA> __host__ __device__ static constexpr size_t abuf() { return (size_t)(2 * NHK) * astr<TA>(); }   // elements per slot per buffer: rows [u of all pairs | v of all pairs]
  // colour form split by the reflection symmetry C[s][s'] = C[rev s][rev s']: with u = J_s + J_rev(s), v = J_s - J_rev(s) per pair,
  // J^dagger C J = 1/2 u^dagger C+ u + 1/2 v^dagger C- v, C+- = C[s_p][s_q] +- C[s_p][rev s_q]: two NPAIR x NPAIR forms, half the flops
  static constexpr int NHK = pad4(NPAIR);                                // amplitude rows per half (K dimension of the mma, padded to 4)
  static constexpr int MTH = (NPAIR + 7) / 8, KTH = NHK / 4, UH = (MTH + 1) / 2, U = 2 * UH;
  static constexpr int KSH = MTH * KTH - MTH * (MTH - 1);                // k-steps of one half (upper-triangular tiles)
  static constexpr int NT = 2 * NCOL / 8;                                // mma n-tiles per batch
  static constexpr int NMASK = 1 << N;
  // amplitude buffers: two (the colour warps work on one batch while the workers fill the next).  (Round 2, before the fused n = 3 pass:
  // ONE buffer for n = 3 FP64 put its space into event slots, 21 -> 32, 4.65 -> 4.22 ms with 12 worker warps.  The fused pass writes the
  // rows of two parameter sets back to back, a single buffer stalls it on the colour form (12 % of the workers' time): two buffers, 8 worker
  // warps at 224 registers and 21 slots: 3.64 -> 3.32 ms.)
  template <typename TA> __host__ __device__ static constexpr int nbuf() { return (N == 3 && sizeof(TA) == 8 && RWGT_NBUF_N3 == 1) ? 1 : 2; }
  static constexpr int NPHASE = (N - 1 > (RMAX > LMAX ? RMAX : LMAX) + 1) ? N - 1 : (RMAX > LMAX ? RMAX : LMAX) + 1;
  static constexpr int NL3 = N - 1, NV4 = (N - 1) * (N - 2) / 2;
  static constexpr int JW = pad4(2 * NL3 + 3 * NV4);                     // words of the n-gluon current's references
  static constexpr int QH = C + NJ + NJ * C, QW = pad4((QH + 1) / 2);    // halfwords / words of one quark-line reference block
  static constexpr int STRIDEF = 4 + JW + 2 * QW;
  static constexpr int NG = c_nG(N), NR = c_nR(N), NL = c_nL(N);   // entries of the current tables (checked against the schedule)
};
__host__ __device__ constexpr int gdesc_words(int m) { return pad4(2 + 2 * (m - 1) + 3 * (m - 1) * (m - 2) / 2); }
__host__ __device__ constexpr int qdesc_words(int m) { return pad4(1 + m); }

struct TupleTables {
  std::map<std::vector<int>, int> gbase, rbase, lbase;
};
// 16-bit reference to the gluon current of the ordered tuple `used`; `exact` reports whether it is stored as used
static uint32_t gref16(int n, const TupleTables& T, const std::vector<int>& used, bool* exact = nullptr) {
  bool st = is_stored(n, used);
  if (exact) *exact = st;
  int base = T.gbase.at(st ? used : reversed(used));
  return (uint32_t)base | ((!st && used.size() == 3) ? REF_REV : 0u);      // length 4: reversal and sign are static on the device
}
static std::vector<int> sub(const std::vector<int>& s, int lo, int hi) { return std::vector<int>(s.begin() + lo, s.begin() + hi); }

static BgSched build_schedule(int n, std::string& err) {
  BgSched S; S.n = n;
  for (int k = 0; k < 3; k++) for (int m = 0; m < 6; m++) { S.offD[k][m] = 0; S.ntask[k][m] = 0; }
  for (int m = 0; m < 6; m++) S.offT[m] = 0;
  for (int k = 0; k < 8; k++) { S.fp_ops[k] = 0; S.fp_final[k] = 0; }
  S.c = (n + 1) / 2; S.lmax = S.c - 1; S.rmax = n - S.c;
  TupleTables T; std::vector<std::vector<int>> tl;
  int nG = 0, nR = 0, nL = 0;
  // Table allocation.  A tuple with gluon 0 at position q only ever uses the variants with bit q clear (parity: gluon 0 at
  // helicity +), so two such tuples of the same length and the same q share one block: the second one's base is offset by 1 << q
  // and its entries fall exactly into the holes of the first (the device still computes entry = base + variant bits).
  auto allocate = [&](std::map<std::vector<int>, int>& base, int& count, const std::vector<std::vector<int>>& tuples, int m, int block) {
    int open_base[6] = {-1, -1, -1, -1, -1, -1};                      // first half of an open pair, per position of gluon 0
    for (auto& t : tuples) {
      int q = pos0(t);
      if (q < 0 || m == 1) { base[t] = count; count += block; continue; }
      if (open_base[q] < 0) { base[t] = count; open_base[q] = count; count += block; }
      else { base[t] = open_base[q] + (1 << q); open_base[q] = -1; }
    }
  };
  for (int m = 1; m <= n - 1; m++) { all_tuples(n, m, tl); std::vector<std::vector<int>> st; for (auto& t : tl) if (is_stored(n, t)) st.push_back(t); allocate(T.gbase, nG, st, m, 1 << m); }
  T.rbase[{}] = nR; nR += 2; T.lbase[{}] = nL; nL += 2;
  for (int m = 1; m <= S.rmax; m++) { all_tuples(n, m, tl); allocate(T.rbase, nR, tl, m, 2 << m); }
  for (int m = 1; m <= S.lmax; m++) { all_tuples(n, m, tl); allocate(T.lbase, nL, tl, m, 2 << m); }
  S.nG = nG; S.nR = nR; S.nL = nL;
  auto pad = [&]() { while (S.words.size() % 4) S.words.push_back(0u); };
  auto gref32 = [&](const std::vector<int>& t, int lo, int hi) {          // reference inside a gluon recursion: must be stored as used (or length 3)
    std::vector<int> u = sub(t, lo, hi); bool ex; uint32_t r = gref16(n, T, u, &ex);
    if (!ex && u.size() != 3) err = "internal: gluon block not stored in the orientation it is used in";
    return r | ((uint32_t)(mask_of(u) * 4) << 16);                        // high half: element offset of the block's momentum sum
  };
  auto gluon_refs = [&](const std::vector<int>& t) {
    int m = (int)t.size();
    for (int k = 1; k < m; k++) { S.words.push_back(gref32(t, 0, k)); S.words.push_back(gref32(t, k, m)); }
    for (int j = 1; j < m; j++) for (int k = j + 1; k < m; k++) { S.words.push_back(gref32(t, 0, j)); S.words.push_back(gref32(t, j, k)); S.words.push_back(gref32(t, k, m)); }
  };
  std::vector<std::vector<uint32_t>> tasks(6);
  // descriptors + task lists of the gluon levels
  std::vector<std::vector<uint32_t>> tG(6), tR(6), tL(6);
  for (int m = 2; m <= n - 1; m++) {
    all_tuples(n, m, tl); pad(); S.offD[0][m] = (int)S.words.size(); int idx = 0;
    for (auto& t : tl) {
      if (m == 2 ? !(t[0] < t[1]) : !is_stored(n, t)) continue;          // length 2: one task fills both orientations
      size_t d0 = S.words.size();
      S.words.push_back((uint32_t)T.gbase[t] | ((uint32_t)(m == 2 ? T.gbase[reversed(t)] : 0) << 16)); S.words.push_back((uint32_t)mask_of(t));
      gluon_refs(t); pad();
      if ((int)(S.words.size() - d0) != gdesc_words(m)) err = "internal: gluon descriptor size";
      int p0 = pos0(t);
      for (uint32_t v = 0; v < (1u << m); v++) if (p0 < 0 || !(v >> p0 & 1)) tG[m].push_back((uint32_t)idx | (v << 16));
      idx++;
      S.fp_ops[0] += (double)(m - 1) * ((p0 < 0) ? (1 << m) : (1 << (m - 1))); S.fp_ops[1] += (double)((m - 1) * (m - 2) / 2) * ((p0 < 0) ? (1 << m) : (1 << (m - 1)));
      S.fp_ops[m > 2 ? 6 : 7] += (p0 < 0) ? (1 << m) : (1 << (m - 1));
    }
  }
  for (int side = 0; side < 2; side++) {
    int mmax = side == 0 ? S.rmax : S.lmax; auto& base = side == 0 ? T.rbase : T.lbase;
    for (int m = 1; m <= mmax; m++) {
      all_tuples(n, m, tl); pad(); S.offD[1 + side][m] = (int)S.words.size(); int idx = 0;
      for (auto& t : tl) {
        size_t d0 = S.words.size();
        S.words.push_back((uint32_t)base[t] | ((uint32_t)mask_of(t) << 16));
        for (int k = 1; k <= m; k++) {
          // right: Jslash(t_1..k) R(t_k+1..m);  left: L(t_1..m-k) Jslash(t_m-k+1..m)
          std::vector<int> gj = side == 0 ? sub(t, 0, k) : sub(t, m - k, m), q = side == 0 ? sub(t, k, m) : sub(t, 0, m - k);
          bool ex; uint32_t rj = gref16(n, T, gj, &ex); if (!ex && gj.size() != 3) err = "internal: quark-current gluon block orientation";
          S.words.push_back(rj | ((uint32_t)base.at(q) << 16));
        }
        pad();
        if ((int)(S.words.size() - d0) != qdesc_words(m)) err = "internal: quark descriptor size";
        int p0 = pos0(t);
        for (uint32_t v = 0; v < (2u << m); v++) if (p0 < 0 || !(v >> p0 & 1)) (side == 0 ? tR : tL)[m + 1].push_back((uint32_t)idx | (v << 16));
        idx++;
        double cnt = (p0 < 0) ? (2 << m) : (1 << m);
        S.fp_ops[2] += m * cnt; S.fp_ops[3] += m * cnt; S.fp_ops[4] += cnt;
      }
    }
  }
  for (int M = 2; M < 6; M++) {
    pad(); S.offT[M] = (int)S.words.size();
    S.ntask[0][M] = (int)tG[M].size(); S.ntask[1][M] = (int)tR[M].size(); S.ntask[2][M] = (int)tL[M].size();
    for (auto w : tG[M]) S.words.push_back(w); for (auto w : tR[M]) S.words.push_back(w); for (auto w : tL[M]) S.words.push_back(w);
  }
  // finals: one descriptor per pair (sigma, sigma reversed); "which = 0" is the forward permutation (n = 5: along the necklace)
  std::vector<std::vector<int>> perms; { std::vector<int> p(n); for (int i = 0; i < n; i++) p[i] = i; do perms.push_back(p); while (std::next_permutation(p.begin(), p.end())); }
  S.nperm = (int)perms.size(); std::map<std::vector<int>, int> rank; for (int i = 0; i < S.nperm; i++) rank[perms[i]] = i;
  const int C = S.c, NJ = n - C + 1;
  const int JW = pad4(2 * (n - 1) + 3 * (n - 1) * (n - 2) / 2), QH = C + NJ + NJ * C, QW = pad4((QH + 1) / 2);
  pad(); S.offF = (int)S.words.size(); S.strideF = 4 + JW + 2 * QW; S.npair = 0;
  std::vector<int> pair_rank, pair_rank_rev;
  for (auto& s0 : perms) {
    bool fwd = (n == 5) ? necklace_forward(s0) : (s0.front() < s0.back());
    if (!fwd) continue;
    S.npair++; pair_rank.push_back(rank[s0]); pair_rank_rev.push_back(rank[reversed(s0)]);
    size_t d0 = S.words.size();
    std::vector<int> sr = reversed(s0);
    uint32_t packed = 0; for (int j = 0; j < n; j++) packed |= (uint32_t)s0[j] << (3 * j);
    // word 0: pair index p = row of u (v is at row NHK + p); word 1: the permutation, 3 bits per position
    S.words.push_back((uint32_t)(S.npair - 1)); S.words.push_back(packed); S.words.push_back(0u); S.words.push_back(0u);
    gluon_refs(s0); pad();
    for (int which = 0; which < 2; which++) {
      const std::vector<int>& s = which ? sr : s0;
      std::vector<uint32_t> hw;
      for (int i = 0; i < C; i++) hw.push_back((uint32_t)T.lbase.at(sub(s, 0, i)));
      for (int j = C; j <= n; j++) hw.push_back((uint32_t)T.rbase.at(sub(s, j, n)));
      for (int j = C; j <= n; j++) for (int i = 0; i < C; i++) {
        if (i == 0 && j == n) { hw.push_back(0u); continue; }
        std::vector<int> u = sub(s, i, j); bool ex; uint32_t r = gref16(n, T, u, &ex);
        // static rule of the device code: blocks of length 4 are stored as used for which = 0 and reversed for which = 1
        if (u.size() == 4 && ex != (which == 0)) err = "internal: length-4 block orientation does not follow the necklace rule";
        if (u.size() != 3 && u.size() != 4 && !ex) err = "internal: block orientation";
        hw.push_back(r);
      }
      while ((int)hw.size() < 2 * QW) hw.push_back(0u);
      for (int k = 0; k < QW; k++) S.words.push_back(hw[2 * k] | (hw[2 * k + 1] << 16));
    }
    if ((int)(S.words.size() - d0) != S.strideF) err = "internal: final descriptor size";
  }
  {
    double nf = (double)S.npair * (double)(1 << (n - 1));
    S.fp_final[0] = nf * (n - 1); S.fp_final[1] = nf * ((n - 1) * (n - 2) / 2); S.fp_final[n > 2 ? 6 : 7] = nf;
    S.fp_final[3] = nf * (1 + 2 * (NJ * C - 1)); S.fp_final[2] = nf * 2 * 2 * NJ * C; S.fp_final[5] = nf * 2 * NJ * 4;
    for (int k = 0; k < 8; k++) S.fp_ops[k] += S.fp_final[k];
  }
  // Colour form.  C commutes with the reversal s -> rev(s) (a trace and its transpose), so in the basis u_p = J_{s_p} + J_{rev s_p},
  // v_p = J_{s_p} - J_{rev s_p} it is block diagonal: J^dagger C J = u^dagger (C+/2) u + v^dagger (C-/2) v with
  // C+-[p][q] = C[s_p][s_q] +- C[s_p][rev s_q].  Each block is positive definite (C is): Cholesky C+-/2 = L L^T and
  // the form is |L+^T u|^2 + |L-^T v|^2.  L^T in mma.m8n8k4 A-fragment order: for half h, m-tile mt, k-steps kt = 2 mt .. KTH-1
  // (upper triangle), element (lane>>2, lane&3) of the 8x4 tile; rows/columns beyond npair are zero.
  {
    int np = S.nperm, nh = S.npair, nhk = (nh + 3) / 4 * 4, MTH = (nh + 7) / 8, KTH = nhk / 4;
    std::vector<double> Cm = colour_matrix_fierz(n);
    for (int h = 0; h < 2; h++) {
      std::vector<double> Ch((size_t)nh * nh), L((size_t)nh * nh, 0.0);
      for (int p = 0; p < nh; p++) for (int q = 0; q < nh; q++)
        Ch[(size_t)p * nh + q] = 0.5 * (Cm[(size_t)pair_rank[p] * np + pair_rank[q]] + (h ? -1.0 : 1.0) * Cm[(size_t)pair_rank[p] * np + pair_rank_rev[q]]);
      for (int j = 0; j < nh; j++) {
        double d = Ch[(size_t)j * nh + j]; for (int k = 0; k < j; k++) d -= L[(size_t)j * nh + k] * L[(size_t)j * nh + k];
        if (!(d > 0)) { err = "internal: colour block not positive definite"; return S; }
        d = std::sqrt(d); L[(size_t)j * nh + j] = d;
        for (int i = j + 1; i < nh; i++) { double x = Ch[(size_t)i * nh + j]; for (int k = 0; k < j; k++) x -= L[(size_t)i * nh + k] * L[(size_t)j * nh + k]; L[(size_t)i * nh + j] = x / d; }
      }
      for (int mt = 0; mt < MTH; mt++) for (int kt = 2 * mt; kt < KTH; kt++) for (int lane = 0; lane < 32; lane++) {
        int row = 8 * mt + (lane >> 2), col = 4 * kt + (lane & 3);
        S.lfrag.push_back((row < nh && col < nh && col >= row) ? L[(size_t)col * nh + row] : 0.0);      // L^T[row][col] = L[col][row]
      }
    }
  }
  return S;
}

// ------------------------------------------------------------------------------------------------ device side
struct BgSet { double gq, g3, g4, mt, fac; };        // fac = 2 gq^2 / D  (|i gq|^2, parity factor 2, averaging)
constexpr int BG_NSMAX = 1 + RWGT_MAX_SETS;      // the old set plus up to RWGT_MAX_SETS new ones
constexpr int BG_RMAX = 6;                       // most node sets of the polynomial mode (n = 4 needs at most 6, n = 5 five on the diagonal ggg = gggg)
struct BgDev {
  int nwords, nslot, shared_ext, nsets;
  int fuse;              // n = 3, parameter sets of equal top mass: ONE pass over the currents serves all sets, the amplitude phase two sets at a time (QuarkLine3F)
  int offD[3][6], offT[6], offF;
  const uint32_t* words; const double* lfrag;
  BgSet set[BG_NSMAX];
  // polynomial mode (coupling-only parameter sets, see bg_plan_poly): the currents are evaluated at nnode node sets only; every
  // parameter set k is the exact linear combination J(k) = sum_j cw[k][j] J(node j) of them
  int poly, nnode; BgSet node[BG_RMAX]; double cw[BG_NSMAX][BG_RMAX];
  double* poly_scratch; long long poly_stride;   // Z = L^T (u | v) of every node set of one event group, per CTA (global memory, mostly L2 resident)
  const int* idx;        // multiprocess handles: event i of this launch is event idx[i] of the buffers (null: identity)
};

struct BgProcess {
  double* d_poly;        // polynomial mode: Z of the node sets, one slice per CTA
  BgSched S; BgDev D; uint32_t* d_words; double* d_lfrag; int sm_count; size_t smem64, smem32; int nslot64, nslot32;
};

template <typename T> struct pair_of;
template <> struct pair_of<double> { typedef double2 type; };
template <> struct pair_of<float> { typedef float2 type; };
template <typename T> __device__ __forceinline__ cx<T> ldc(const cx<T>* p) { typename pair_of<T>::type t = *reinterpret_cast<const typename pair_of<T>::type*>(p); return mk<T>(t.x, t.y); }
template <typename T> __device__ __forceinline__ void stc(cx<T>* p, cx<T> v) { typename pair_of<T>::type t; t.x = v.re; t.y = v.im; *reinterpret_cast<typename pair_of<T>::type*>(p) = t; }

constexpr int RWGT_STAGE_MIN_N = 4;
template <typename T> struct Smem {
  uint32_t* W;    // schedule words (whole CTA)
  double* LF;     // Cholesky factors L+^T, L-^T of the colour blocks in mma-fragment order (whole CTA)
  double* pm;     // [nslot][n_ext][4] momenta (always double)
  double* acc;    // [nslot][BG_NSMAX]   helicity-summed colour forms per parameter set (owned by the colour warps)
  double* red;    // [nslot][8]   per-warp partial sums of the colour form
  double* pred;   // [16][BG_RMAX (BG_RMAX + 1) / 2]   polynomial mode: per-warp partial cross forms
  cx<T>* G; cx<T>* R; cx<T>* L;   // [nslot][4][nX]   component planes of (re,im) pairs: one vector load per component,
                                  //                  conflict-free for consecutive helicity variants
  T* K;           // [nslot][NMASK][4] momentum sums of gluon subsets
  T* iK2;         // [nslot][NMASK]
  T* dR; T* dL;   // [nslot][NMASK] 1/(q^2-m^2)
  // staging copy of everything step a1/a2 produces for the NEXT event group (written by the colour warps while the workers run the
  // current group): momenta, external wavefunctions (table entries 0..2N-1 of G, 0..1 of R and L), momentum sums, denominators
  double* pmS; cx<T>* GS; cx<T>* RS; cx<T>* LS; T* KS; T* iK2S; T* dRS; T* dLS;
  T* A;           // [2][nslot][2 NHK][astr] double-buffered rows u = J_s + J_rev(s), v = J_s - J_rev(s) (re,im interleaved), formed in double,
                  // stored in T (the colour form itself always runs in double)
};
template <int N, typename T> __host__ __device__ inline size_t carve(Smem<T>& s, unsigned char* base, int ns, int nwords) {
  typedef Geo<N> Ge; size_t off = 0; constexpr int nG = Ge::NG, nR = Ge::NR, nL = Ge::NL;
  auto al = [&]() { off = (off + 15) / 16 * 16; };
  s.A = (T*)(base + off); off += sizeof(T) * Ge::template nbuf<T>() * (size_t)ns * Ge::template abuf<T>(); al();
  s.LF = (double*)(base + off); off += sizeof(double) * 2 * Ge::KSH * 32; al();
  s.pm = (double*)(base + off); off += sizeof(double) * ns * (N + 2) * 4; al();
  s.acc = (double*)(base + off); off += sizeof(double) * ns * BG_NSMAX; al();
  s.red = (double*)(base + off); off += sizeof(double) * ns * 8; al();
  s.pred = (double*)(base + off); off += sizeof(double) * 16 * (BG_RMAX * (BG_RMAX + 1) / 2); al();
  s.G = (cx<T>*)(base + off); off += sizeof(T) * (size_t)ns * 8 * nG; al();
  s.R = (cx<T>*)(base + off); off += sizeof(T) * (size_t)ns * 8 * nR; al();
  s.L = (cx<T>*)(base + off); off += sizeof(T) * (size_t)ns * 8 * nL; al();
  s.K = (T*)(base + off); off += sizeof(T) * ns * Ge::NMASK * 4; al();
  s.iK2 = (T*)(base + off); off += sizeof(T) * ns * Ge::NMASK; al();
  s.dR = (T*)(base + off); off += sizeof(T) * ns * Ge::NMASK; al();
  s.dL = (T*)(base + off); off += sizeof(T) * ns * Ge::NMASK; al();
  const int nst = (N >= RWGT_STAGE_MIN_N) ? ns : 0;                         // staging exists only where the colour warps prefetch (bg_kernel: STAGE)
  s.pmS = (double*)(base + off); off += sizeof(double) * nst * (N + 2) * 4; al();
  s.GS = (cx<T>*)(base + off); off += sizeof(T) * (size_t)nst * 8 * (2 * N); al();
  s.RS = (cx<T>*)(base + off); off += sizeof(T) * (size_t)nst * 8 * 2; al();
  s.LS = (cx<T>*)(base + off); off += sizeof(T) * (size_t)nst * 8 * 2; al();
  s.KS = (T*)(base + off); off += sizeof(T) * nst * Ge::NMASK * 4; al();
  s.iK2S = (T*)(base + off); off += sizeof(T) * nst * Ge::NMASK; al();
  s.dRS = (T*)(base + off); off += sizeof(T) * nst * Ge::NMASK; al();
  s.dLS = (T*)(base + off); off += sizeof(T) * nst * Ge::NMASK; al();
  s.W = (uint32_t*)(base + off); off += sizeof(uint32_t) * nwords; al();
  return off;
}

template <typename T> __device__ __forceinline__ vec4<T> ld4(const cx<T>* tab, int stride, int e) {
  vec4<T> r;
#pragma unroll
  for (int c = 0; c < 4; c++) r.c[c] = ldc(tab + c * stride + e);
  return r;
}
template <typename T> __device__ __forceinline__ spn<T> lds4(const cx<T>* tab, int stride, int e) {
  spn<T> r;
#pragma unroll
  for (int c = 0; c < 4; c++) r.c[c] = ldc(tab + c * stride + e);
  return r;
}
template <typename T, typename V> __device__ __forceinline__ void st4(cx<T>* tab, int stride, int e, const V& v) {
#pragma unroll
  for (int c = 0; c < 4; c++) stc(tab + c * stride + e, v.c[c]);
}
// the 4 momentum components of a gluon subset as vector loads
__device__ __forceinline__ void ldk(double* k, const double* p) { double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 2); k[0] = a.x; k[1] = a.y; k[2] = b.x; k[3] = b.y; }
__device__ __forceinline__ void ldk(float* k, const float* p) { float4 a = *reinterpret_cast<const float4*>(p); k[0] = a.x; k[1] = a.y; k[2] = a.z; k[3] = a.w; }
// NW words of a descriptor (16-byte aligned, NW a multiple of 4) into registers
template <int NW> __device__ __forceinline__ void ldw(uint32_t* d, const uint32_t* s) {
#pragma unroll
  for (int i = 0; i < NW / 4; i++) { uint4 t = *reinterpret_cast<const uint4*>(s + 4 * i); d[4 * i] = t.x; d[4 * i + 1] = t.y; d[4 * i + 2] = t.z; d[4 * i + 3] = t.w; }
}
// helicity-variant bits [SH, SH+M) of the task's variant word; all shifts and widths are compile-time
template <int M, int SH> __device__ __forceinline__ uint32_t fieldv(uint32_t v) { return M == 0 ? 0u : (v >> SH) & ((1u << M) - 1u); }
template <int M> __device__ __forceinline__ uint32_t brevm(uint32_t f) { return __brev(f) >> (32 - M); }
// entry of the gluon current referenced by the low 16 bits of r, for a block of static length M at static position SH
template <int M, int SH> __device__ __forceinline__ int gentry(uint32_t r, uint32_t v) {
  uint32_t f = fieldv<M, SH>(v);
  if (M == 3) { if (r & REF_REV) f = brevm<3>(f); }
  return (int)((r & 0x7fffu) + f);
}
__device__ __forceinline__ uint32_t halfw(const uint32_t* w, int k) { return (k & 1) ? (w[k >> 1] >> 16) : (w[k >> 1] & 0xffffu); }

// named barriers (ids 1..6; id 0 is __syncthreads): workers among themselves, colour warps among themselves,
// and the full/empty handshake of the two amplitude buffers
enum { BAR_WORK = 1, BAR_FULL0 = 2, BAR_EMPTY0 = 4, BAR_COLOUR = 6, BAR_STAGE_FULL = 7, BAR_STAGE_EMPTY = 8, BAR_ZFULL = 9 };
// the barrier id is an immediate (a register id makes ptxas reserve all 16 barriers, which limits the CTAs per SM)
__device__ __forceinline__ void bar_sync(int id, int count) {
  switch (id) {
    case 1: asm volatile("bar.sync 1, %0;" ::"r"(count) : "memory"); break; case 2: asm volatile("bar.sync 2, %0;" ::"r"(count) : "memory"); break;
    case 3: asm volatile("bar.sync 3, %0;" ::"r"(count) : "memory"); break; case 4: asm volatile("bar.sync 4, %0;" ::"r"(count) : "memory"); break;
    case 5: asm volatile("bar.sync 5, %0;" ::"r"(count) : "memory"); break; case 6: asm volatile("bar.sync 6, %0;" ::"r"(count) : "memory"); break;
    case 7: asm volatile("bar.sync 7, %0;" ::"r"(count) : "memory"); break; case 8: asm volatile("bar.sync 8, %0;" ::"r"(count) : "memory"); break;
    default: asm volatile("bar.sync 9, %0;" ::"r"(count) : "memory");
  }
}
__device__ __forceinline__ void bar_arrive(int id, int count) {
  switch (id) {
    case 2: asm volatile("bar.arrive 2, %0;" ::"r"(count) : "memory"); break; case 3: asm volatile("bar.arrive 3, %0;" ::"r"(count) : "memory"); break;
    case 4: asm volatile("bar.arrive 4, %0;" ::"r"(count) : "memory"); break; case 5: asm volatile("bar.arrive 5, %0;" ::"r"(count) : "memory"); break;
    case 7: asm volatile("bar.arrive 7, %0;" ::"r"(count) : "memory"); break; case 8: asm volatile("bar.arrive 8, %0;" ::"r"(count) : "memory"); break;
    default: asm volatile("bar.arrive 9, %0;" ::"r"(count) : "memory");
  }
}

// gluon current of one ordered M-tuple / helicity variant from shorter currents (unscaled by the propagator).
// w: the 2(M-1) + 3(M-1)(M-2)/2 reference words of the tuple, in registers.  No signs: every block is stored as used.
template <int M, int nG, typename T> struct GluonSum {
  template <int K> static __device__ __forceinline__ void l3(vec4<T>& a3, const uint32_t* w, uint32_t v, const cx<T>* G, const T* Kt) {
    if constexpr (K < M) {
      uint32_t ra = w[2 * (K - 1)], rb = w[2 * (K - 1) + 1];
      vec4<T> A = ld4(G, nG, gentry<K, 0>(ra, v)), B = ld4(G, nG, gentry<M - K, K>(rb, v));
      T ka[4], kb[4]; ldk(ka, Kt + (ra >> 16)); ldk(kb, Kt + (rb >> 16));
      L3_acc(a3, A, ka, B, kb);
      l3<K + 1>(a3, w, v, G, Kt);
    }
  }
  // V4 terms over the compositions (J, K) with 1 <= J < K < M, enumerated in the builder's order
  template <int J, int K, int IDX> static __device__ __forceinline__ void v4(vec4<T>& a4, const uint32_t* w4, uint32_t v, const cx<T>* G) {
    if constexpr (J < M - 1) {
      if constexpr (K < M) {
        uint32_t rx = w4[3 * IDX], ry = w4[3 * IDX + 1], rz = w4[3 * IDX + 2];
        vec4<T> X = ld4(G, nG, gentry<J, 0>(rx, v)), Y = ld4(G, nG, gentry<K - J, J>(ry, v)), Z = ld4(G, nG, gentry<M - K, K>(rz, v));
        V4_acc(a4, X, Y, Z);
        v4<J, K + 1, IDX + 1>(a4, w4, v, G);
      } else v4<J + 1, J + 2, IDX>(a4, w4, v, G);
    }
  }
  // the two coupling structures apart: a3 = sum of the L3 terms, a4 = sum of the V4 terms (no coupling applied)
  static __device__ __forceinline__ void run_split(vec4<T>& a3, vec4<T>& a4, const uint32_t* w, uint32_t v, const cx<T>* G, const T* Kt) {
#pragma unroll
    for (int i = 0; i < 4; i++) { a3.c[i] = mk<T>(0, 0); a4.c[i] = mk<T>(0, 0); }
    l3<1>(a3, w, v, G, Kt);
    v4<1, 2, 0>(a4, w + 2 * (M - 1), v, G);
  }
  static __device__ __forceinline__ vec4<T> run(const uint32_t* w, uint32_t v, const cx<T>* G, const T* Kt, T g3, T g4) {
    vec4<T> a3, a4;
#pragma unroll
    for (int i = 0; i < 4; i++) { a3.c[i] = mk<T>(0, 0); a4.c[i] = mk<T>(0, 0); }
    l3<1>(a3, w, v, G, Kt);
    v4<1, 2, 0>(a4, w + 2 * (M - 1), v, G);
    vec4<T> r;
#pragma unroll
    for (int i = 0; i < 4; i++) { r.c[i] = (-g3) * a3.c[i]; if (M > 2) rfma(r.c[i], g4, a4.c[i]); }
    return r;
  }
};

template <typename T> struct Ctx {
  Smem<T> s; int tid, ns; T g3, g4, gq, mt; const BgDev* D;
};

// quark-current terms  acc += Jslash(block) R(rest)  resp.  acc += L(rest) Jslash(block), block lengths K = 1..MM
template <int MM, int K, int nG, int nQ, bool RIGHT, typename T>
__device__ __forceinline__ void quark_terms(spn<T>& acc, const uint32_t* w, uint32_t v, int hb, const cx<T>* G, const cx<T>* Q) {
  if constexpr (K <= MM) {
    uint32_t r = w[K];
    // right: gluon block [0,K), quark rest [K,MM);  left: quark rest [0,MM-K), gluon block [MM-K,MM)
    int eg = RIGHT ? gentry<K, 0>(r, v) : gentry<K, MM - K>(r, v);
    int eq = (int)(r >> 16) + (int)(RIGHT ? fieldv<MM - K, K>(v) : fieldv<MM - K, 0>(v)) + (hb << (MM - K));
    lcv<T> J = lightcone(ld4(G, nG, eg));
    if (RIGHT) slash_acc(acc, J, lds4(Q, nQ, eq)); else row_slash_acc(acc, lds4(Q, nQ, eq), J);
    quark_terms<MM, K + 1, nG, nQ, RIGHT, T>(acc, w, v, hb, G, Q);
  }
}

// phase M (worker warps): gluon currents of length M, right/left quark currents of length M-1, all helicity variants with
// gluon 0 at helicity +.  Tasks are ordered [G of all slots][R of all slots][L of all slots]: a warp diverges at most at the two seams.
template <int N, int M, typename T, int NWT> __device__ __forceinline__ void level_phase(const Ctx<T>& c) {
  typedef Geo<N> Ge;
  constexpr bool HASG = (M <= N - 1), HASR = (M - 1 >= 1 && M - 1 <= Ge::RMAX), HASL = (M - 1 >= 1 && M - 1 <= Ge::LMAX);
  constexpr int MM = M - 1;
  constexpr int tg = HASG ? c_ntaskG(N, M) : 0, tr = HASR ? c_ntaskQ(N, MM) : 0, tl = HASL ? c_ntaskQ(N, MM) : 0;
  const Smem<T>& s = c.s; constexpr int nG = Ge::NG, nR = Ge::NR, nL = Ge::NL, next = N + 2;
  const int ns = c.ns, nGt = ns * tg, nRt = ns * tr, nLt = ns * tl;
  const uint32_t* TL = s.W + c.D->offT[M];
  for (int t = c.tid; t < nGt + nRt + nLt; t += NWT) {
    if (HASG && t < nGt) {
     if constexpr (HASG) {
      int sl = t / tg, o = t - sl * tg; uint32_t tw = TL[o]; uint32_t v = tw >> 16;
      cx<T>* G = s.G + (size_t)sl * 4 * nG; const T* K = s.K + (size_t)sl * Ge::NMASK * 4;
      constexpr int DW = gdesc_words(M);
      uint32_t w[DW]; ldw<DW>(w, s.W + c.D->offD[0][M] + (tw & 0xffffu) * DW);
      vec4<T> r = GluonSum<M, nG, T>::run(w + 2, v, G, K, c.g3, c.g4);
      T sc = s.iK2[sl * Ge::NMASK + w[1]];
#pragma unroll
      for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
      st4(G, nG, (int)(w[0] & 0xffffu) + (int)v, r);
      if (M == 2) {                                       // the other orientation: J(b,a) = -J(a,b), variant bits swapped
#pragma unroll
        for (int i = 0; i < 4; i++) r.c[i] = -r.c[i];
        st4(G, nG, (int)(w[0] >> 16) + (int)(((v & 1u) << 1) | (v >> 1)), r);
      }
     }
    } else if (HASR && t < nGt + nRt) {
     if constexpr (HASR) {
      int tt = t - nGt, sl = tt / tr, o = tt - sl * tr; uint32_t tw = TL[tg + o]; uint32_t vv = tw >> 16, v = vv & ((1u << MM) - 1u); int hb = (int)(vv >> MM);
      const cx<T>* G = s.G + (size_t)sl * 4 * nG; cx<T>* R = s.R + (size_t)sl * 4 * nR; const T* K = s.K + (size_t)sl * Ge::NMASK * 4;
      constexpr int DW = qdesc_words(MM);
      uint32_t w[DW]; ldw<DW>(w, s.W + c.D->offD[1][MM] + (tw & 0xffffu) * DW);
      int ob = (int)(w[0] & 0xffffu), mask = (int)(w[0] >> 16);
      spn<T> acc;
#pragma unroll
      for (int i = 0; i < 4; i++) acc.c[i] = mk<T>(0, 0);
      quark_terms<MM, 1, nG, nR, true, T>(acc, w, v, hb, G, R);
      T q[4], k[4]; ldk(k, K + 4 * mask);
#pragma unroll
      for (int mu = 0; mu < 4; mu++) q[mu] = k[mu] - (T)s.pm[sl * next * 4 + 12 + mu];
      spn<T> r = slash_r_plus_m(q, c.mt, acc); T sc = -c.gq * s.dR[sl * Ge::NMASK + mask];
#pragma unroll
      for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
      st4(R, nR, ob + (int)vv, r);
     }
    } else if constexpr (HASL) {
      int tt = t - nGt - nRt, sl = tt / tl, o = tt - sl * tl; uint32_t tw = TL[tg + tr + o]; uint32_t vv = tw >> 16, v = vv & ((1u << MM) - 1u); int hb = (int)(vv >> MM);
      const cx<T>* G = s.G + (size_t)sl * 4 * nG; cx<T>* L = s.L + (size_t)sl * 4 * nL; const T* K = s.K + (size_t)sl * Ge::NMASK * 4;
      constexpr int DW = qdesc_words(MM);
      uint32_t w[DW]; ldw<DW>(w, s.W + c.D->offD[2][MM] + (tw & 0xffffu) * DW);
      int ob = (int)(w[0] & 0xffffu), mask = (int)(w[0] >> 16);
      spn<T> acc;
#pragma unroll
      for (int i = 0; i < 4; i++) acc.c[i] = mk<T>(0, 0);
      quark_terms<MM, 1, nG, nL, false, T>(acc, w, v, hb, G, L);
      T q[4], k[4]; ldk(k, K + 4 * mask);
#pragma unroll
      for (int mu = 0; mu < 4; mu++) q[mu] = (T)s.pm[sl * next * 4 + 8 + mu] - k[mu];
      spn<T> r = row_slash_r_plus_m(acc, q, c.mt); T sc = -c.gq * s.dL[sl * Ge::NMASK + mask];
#pragma unroll
      for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
      st4(L, nL, ob + (int)vv, r);
    }
  }
  bar_sync(BAR_WORK, NWT);
}

// The ordering and its reversal share the term ubar Jn-slash v of the full gluon current (up to the sign (-1)^(n+1)): formed once per
// pair it saves two row-slash products of 2 x 2 x NJ C.  Measured on B200: gg->ttggg FP64 40.85 -> 39.71 ms, FP32 19.43 -> 19.19,
// gg->ttgg FP32 5.43 -> 5.30; gg->ttgg FP64 gets slower (10.84 -> 10.91).  Used wherever it is faster: events/s is the metric, and that the
// saved flops lower the FP32 roofline fraction a little (0.505 -> 0.500) is not a reason to run the slower kernel (round 3).
template <int N, typename T> __host__ __device__ constexpr bool share_full_term() { return N == 5 || (N == 4 && sizeof(T) == 4); }
// a4: the quark line of one colour ordering (WHICH = 0: the pair's forward permutation, 1: its reversal) around the split position C:
//   Acc[ht][hb] += sum_{i < C <= j} L(s_1..i; ht) Jslash(s_i+1..j) R(s_j+1..n; hb)
// wq: the block's 16-bit references (L bases, R bases, gluon blocks), v: helicity bits by position in THIS ordering.
template <int N, int WHICH, typename T> struct QuarkLine {
  typedef Geo<N> Ge;
  static constexpr int C = Ge::C, NJ = Ge::NJ, nG = Ge::NG, nR = Ge::NR, nL = Ge::NL;
  template <int JJ, int I> static __device__ __forceinline__ void iterm(spn<T>& X0, spn<T>& X1, const uint32_t* wq, uint32_t v, const vec4<T>& Jn,
                                                                        const cx<T>* G, const cx<T>* L) {
    if constexpr (I < C) {
      constexpr int J = C + JJ, M = J - I;                     // gluon block [I, J) of length M
      lcv<T> Jl;
      if constexpr (I == 0 && J == N) {
        Jl = (WHICH == 1 && N % 2 == 0) ? lightcone_neg(Jn) : lightcone(Jn);          // J(reversed) = (-1)^{n+1} J
      } else {
        uint32_t r = halfw(wq, C + NJ + JJ * C + I);
        uint32_t f = fieldv<M, I>(v);
        if constexpr (M == 3) { if (r & REF_REV) f = brevm<3>(f); }
        if constexpr (M == 4 && WHICH == 1) f = brevm<4>(f);                           // stored reversed (necklace rule)
        vec4<T> Jv = ld4(G, nG, (int)((r & 0x7fffu) + f));
        Jl = (M == 4 && WHICH == 1) ? lightcone_neg(Jv) : lightcone(Jv);
      }
      int el = (int)halfw(wq, I) + (int)fieldv<I, 0>(v);
      row_slash_acc(X0, lds4(L, nL, el), Jl); row_slash_acc(X1, lds4(L, nL, el + (1 << I)), Jl);
      iterm<JJ, I + 1>(X0, X1, wq, v, Jn, G, L);
    }
  }
  // XT: ubar(ht) Jn-slash for the two top helicities, formed once per pair by the caller: the ordering and its reversal share the term
  // of the full gluon current up to the sign (-1)^(n+1)
  template <int JJ> static __device__ __forceinline__ void jterm(cx<T> (&Acc)[2][2], const uint32_t* wq, uint32_t v, const vec4<T>& Jn, const spn<T> (&XT)[2],
                                                                 const cx<T>* G, const cx<T>* R, const cx<T>* L) {
    if constexpr (JJ < NJ) {
      constexpr int J = C + JJ;
      spn<T> X0, X1;
      if constexpr (J == N && share_full_term<N, T>()) {
        constexpr bool NEG = (WHICH == 1 && N % 2 == 0);
#pragma unroll
        for (int i = 0; i < 4; i++) { X0.c[i] = NEG ? -XT[0].c[i] : XT[0].c[i]; X1.c[i] = NEG ? -XT[1].c[i] : XT[1].c[i]; }
        iterm<JJ, 1>(X0, X1, wq, v, Jn, G, L);
      } else {
#pragma unroll
        for (int i = 0; i < 4; i++) { X0.c[i] = mk<T>(0, 0); X1.c[i] = mk<T>(0, 0); }
        iterm<JJ, 0>(X0, X1, wq, v, Jn, G, L);
      }
      int er = (int)halfw(wq, C + JJ) + (int)fieldv<N - J, J>(v);
#pragma unroll
      for (int hb = 0; hb < 2; hb++) {
        spn<T> Rr = lds4(R, nR, er + (hb << (N - J)));
        rowcol_acc(Acc[0][hb], X0, Rr); rowcol_acc(Acc[1][hb], X1, Rr);
      }
      jterm<JJ + 1>(Acc, wq, v, Jn, XT, G, R, L);
    }
  }
  static __device__ __forceinline__ void run(cx<T> (&Acc)[2][2], const uint32_t* wq, uint32_t v, const vec4<T>& Jn, const spn<T> (&XT)[2], const cx<T>* G, const cx<T>* R, const cx<T>* L) {
#pragma unroll
    for (int a = 0; a < 2; a++)
#pragma unroll
      for (int b = 0; b < 2; b++) Acc[a][b] = mk<T>(0, 0);
    jterm<0>(Acc, wq, v, Jn, XT, G, R, L);
  }
};

// n = 3, two parameter sets in ONE pass (the amplitude-level form of SURVEY C6's polynomial structure; PAPER.md:87 steps 3-6 for
// both sets at the price of one).  With the currents of the level phase evaluated at UNIT couplings (gq = g3 = 1) every colour-ordered
// amplitude of g g -> t tbar g is
//     J_sigma = gq^2 c0 + gq g3 c1 + g3^2 c2 + g4 c3,
//     c0 = L(s1) eps-slash(s2) R(s3),   c1 = ubar J-slash(s1 s2) R(s3) + L(s1) J-slash(s2 s3) v,
//     c2 = -ubar A3-slash v / K^2,      c3 = ubar A4-slash v / K^2      (A3 / A4: the L3 / V4 sums of the three-gluon current),
// so the four coefficient amplitudes are formed once and each parameter set costs four real-times-complex multiply-adds per amplitude.
// Acc[s][ht][hb] += sum_m wt[s][m] c_m[ht][hb] for the two sets s; J2 = -A3 / K^2 and J3 = A4 / K^2 are passed in.
// Reference layout of wq (16-bit): [L(), L(s1), R(s3), R(), block(s1 s2), block(s2), -, block(s2 s3)], as built by build_schedule.
template <typename T> struct QuarkLine3F {
  typedef Geo<3> Ge;
  static constexpr int nG = Ge::NG, nR = Ge::NR, nL = Ge::NL;
  // Acc[s][ht][.] += wt[s][m] * (X . R_hb) for one top helicity ht
  static __device__ __forceinline__ void fold(cx<T> (&Acc)[2][2][2], int m, int ht, const spn<T>& X, const spn<T>& Ra, const spn<T>& Rb, const T (&wt)[2][4]) {
    const cx<T> da = rowcol(X, Ra), db = rowcol(X, Rb);
#pragma unroll
    for (int s2 = 0; s2 < 2; s2++) { rfma(Acc[s2][ht][0], wt[s2][m], da); rfma(Acc[s2][ht][1], wt[s2][m], db); }
  }
  // X = W a-slash for both top helicities, one after the other (one row spinor live at a time), folded with coefficient m
  static __device__ __forceinline__ void term(cx<T> (&Acc)[2][2][2], int m, const cx<T>* L, int el, int dl, const lcv<T>& Jl, const spn<T>& Ra, const spn<T>& Rb, const T (&wt)[2][4]) {
#pragma unroll
    for (int ht = 0; ht < 2; ht++) {
      spn<T> X;
#pragma unroll
      for (int i = 0; i < 4; i++) X.c[i] = mk<T>(0, 0);
      row_slash_acc(X, lds4(L, nL, el + ht * dl), Jl);
      fold(Acc, m, ht, X, Ra, Rb, wt);
    }
  }
  // the term both colour orderings of a pair share: c2, c3 = ubar (three-gluon current) v, J(reversed) = +J for three gluons
  static __device__ __forceinline__ void common(cx<T> (&Acc)[2][2][2], const uint32_t* wq, const vec4<T>& J2, const vec4<T>& J3, const cx<T>* R, const cx<T>* L, const T (&wt)[2][4]) {
#pragma unroll
    for (int s2 = 0; s2 < 2; s2++)
#pragma unroll
      for (int a = 0; a < 2; a++)
#pragma unroll
        for (int b = 0; b < 2; b++) Acc[s2][a][b] = mk<T>(0, 0);
    const int el0 = (int)halfw(wq, 0), er3 = (int)halfw(wq, 3);
    const spn<T> R3a = lds4(R, nR, er3), R3b = lds4(R, nR, er3 + 1);
    term(Acc, 2, L, el0, 1, lightcone(J2), R3a, R3b, wt);
    term(Acc, 3, L, el0, 1, lightcone(J3), R3a, R3b, wt);
  }
  // c0 and c1 of one colour ordering, added to Acc (which the caller initialises with the common term)
  static __device__ __forceinline__ void run(cx<T> (&Acc)[2][2][2], const uint32_t* wq, uint32_t v, const cx<T>* G, const cx<T>* R, const cx<T>* L, const T (&wt)[2][4]) {
    const int el0 = (int)halfw(wq, 0), el1 = (int)halfw(wq, 1) + (int)fieldv<1, 0>(v);
    {
      const int er2 = (int)halfw(wq, 2) + (int)fieldv<1, 2>(v);
      const spn<T> R2a = lds4(R, nR, er2), R2b = lds4(R, nR, er2 + 2);
      // c0: L(s1) eps-slash(s2) . R(s3)
      term(Acc, 0, L, el1, 2, lightcone(ld4(G, nG, (int)((halfw(wq, 5) & 0x7fffu) + fieldv<1, 1>(v)))), R2a, R2b, wt);
      // c1, first part: ubar J-slash(s1 s2) . R(s3)
      term(Acc, 1, L, el0, 1, lightcone(ld4(G, nG, (int)((halfw(wq, 4) & 0x7fffu) + fieldv<2, 0>(v)))), R2a, R2b, wt);
    }
    {   // c1, second part: L(s1) J-slash(s2 s3) . v
      const int er3 = (int)halfw(wq, 3);
      const spn<T> R3a = lds4(R, nR, er3), R3b = lds4(R, nR, er3 + 1);
      term(Acc, 1, L, el1, 2, lightcone(ld4(G, nG, (int)((halfw(wq, 7) & 0x7fffu) + fieldv<2, 1>(v)))), R3a, R3b, wt);
    }
  }
};

// Steps a1 + a2 for one event group, by `nth` threads (index t0): momenta (coalesced over the events of the group) into pm, then
// external wavefunctions (gluon i, helicity bit hb -> entry 2 i + hb of G; v(p_tbar) -> entries 0,1 of R; ubar(p_t) -> 0,1 of L),
// momentum sums of the gluon subsets and the inverse propagator denominators.  sG / sR / sL: entries per component plane of the
// destination tables.  SYNC(): a barrier over the calling threads between the two steps.
template <typename T, typename TE, typename V> __device__ __forceinline__ void st4cvt(cx<T>* tab, int stride, int e, const V& v) {
#pragma unroll
  for (int c = 0; c < 4; c++) stc(tab + c * stride + e, mk<T>((T)v.c[c].re, (T)v.c[c].im));
}
template <int N, typename T, typename TK, typename TE, typename SYNC>
__device__ __forceinline__ void group_externals(int t0, int nth, int ns, long long ev0, long long nev, long long stride, const double* __restrict__ mom, const int* __restrict__ idx,
                                                double mtd, double* pmD, cx<T>* Gd, int sG, cx<T>* Rd, int sR, cx<T>* Ld, int sL, T* Kd, T* iK2d, T* dRd, T* dLd,
                                                bool load, SYNC sync) {
  typedef Geo<N> Ge; constexpr int next = N + 2;
  if (load) {
    for (int t = t0; t < ns * next * 4; t += nth) {
      int sl = t % ns, comp = t / ns; long long ev = ev0 + sl; if (ev >= nev) ev = nev - 1;
      if (idx) ev = idx[ev];
      pmD[(sl * next * 4) + comp] = __ldg(mom + (size_t)comp * stride + ev);
    }
    sync();
  }
  // objects per slot: N gluons (both helicities each), v (both helicities), ubar (both helicities), the NMASK - 1 non-empty gluon
  // subsets: n = 3: 12 objects, i.e. ONE round of equally long tasks for 32 slots x 384 threads (round 1: 18 objects, 1.5 rounds, and
  // the rsqrt chains of a leg done once per helicity)
  constexpr int nobj = N + 2 + (Ge::NMASK - 1);
  for (int t = t0; t < ns * nobj; t += nth) {
    int o = t / ns, sl = t - o * ns; const double* pm = pmD + sl * next * 4;      // object-major: the lanes of a warp run the same branch
    if (o < N) {                             // gluon i, both helicities (bit 0: +1, 1: -1); entries 2 i, 2 i + 1
      int i = o, leg = i < 2 ? i : i + 2; const double* p = pm + 4 * leg;
      vec4<TE> ep, em; polvec_pair<TE>((TE)p[1], (TE)p[2], (TE)p[3], ep, em);
      if (i >= 2) { ep = conj4(ep); em = conj4(em); }              // outgoing gluon carries eps*
      st4cvt<T, TE>(Gd + (size_t)sl * 4 * sG, sG, 2 * i, ep); st4cvt<T, TE>(Gd + (size_t)sl * 4 * sG, sG, 2 * i + 1, em);
    } else if (o == N) {                     // v(p_tbar, +-), R() entries 0,1
      const double* p = pm + 12;
      chi_pair<TE> x = make_chi<TE>((TE)p[1], (TE)p[2], (TE)p[3]); const shell<TE> sh = make_shell<TE>((TE)p[0], (TE)mtd);
      st4cvt<T, TE>(Rd + (size_t)sl * 4 * sR, sR, 0, spinor_v<TE>(x, sh, +1)); st4cvt<T, TE>(Rd + (size_t)sl * 4 * sR, sR, 1, spinor_v<TE>(x, sh, -1));
    } else if (o == N + 1) {                 // ubar(p_t, +-), L() entries 0,1
      const double* p = pm + 8;
      chi_pair<TE> x = make_chi<TE>((TE)p[1], (TE)p[2], (TE)p[3]); const shell<TE> sh = make_shell<TE>((TE)p[0], (TE)mtd);
      st4cvt<T, TE>(Ld + (size_t)sl * 4 * sL, sL, 0, bar(spinor_u<TE>(x, sh, +1))); st4cvt<T, TE>(Ld + (size_t)sl * 4 * sL, sL, 1, bar(spinor_u<TE>(x, sh, -1)));
    } else {                                 // gluon subset `mask` (the empty subset is never referenced: its entries are zeroed by the last task)
      int mask = o - (N + 2) + 1;
      if (mask == Ge::NMASK - 1) { T* K0 = Kd + (size_t)sl * Ge::NMASK * 4; for (int mu = 0; mu < 4; mu++) K0[mu] = T(0);
        iK2d[sl * Ge::NMASK] = T(0); dRd[sl * Ge::NMASK] = T(0); dLd[sl * Ge::NMASK] = T(0); }
      TK k[4] = {0, 0, 0, 0};
#pragma unroll
      for (int i = 0; i < N; i++) if (mask >> i & 1) { int leg = i < 2 ? i : i + 2; TK sg = i < 2 ? TK(1) : TK(-1);
        for (int mu = 0; mu < 4; mu++) k[mu] += sg * (TK)pm[4 * leg + mu]; }
      TK k2 = mdot_rr<TK>(k, k);
      TK qr[4], ql[4]; for (int mu = 0; mu < 4; mu++) { qr[mu] = k[mu] - (TK)pm[12 + mu]; ql[mu] = (TK)pm[8 + mu] - k[mu]; }
      TK m2 = (TK)mtd * (TK)mtd;
      T* K = Kd + ((size_t)sl * Ge::NMASK + mask) * 4; for (int mu = 0; mu < 4; mu++) K[mu] = (T)k[mu];
      // only the denominators some current uses (warp-uniform conditions): gluon propagators of >= 2 gluons, quark propagators
      // behind 1..RMAX (right) resp. 1..LMAX (left) gluons
      const int pc = __popc(mask);
      iK2d[sl * Ge::NMASK + mask] = (pc >= 2) ? (T)(TK(1) / k2) : T(0);
      dRd[sl * Ge::NMASK + mask] = (pc >= 1 && pc <= Ge::RMAX) ? (T)(TK(1) / (mdot_rr<TK>(qr, qr) - m2)) : T(0);
      dLd[sl * Ge::NMASK + mask] = (pc >= 1 && pc <= Ge::LMAX) ? (T)(TK(1) / (mdot_rr<TK>(ql, ql) - m2)) : T(0);
    }
  }
}

// B-fragment operands of one k-step for all NT n-tiles of a lane.  The colour form is a sum of squares over all columns, so the
// assignment of amplitude columns to (n-tile, lane) is free: FP32 amplitude buffers give lane group n = lane >> 2 the NT = 4 ADJACENT
// columns 4 n .. 4 n + 3 (one LDS.128, conflict-free with the row stride of astr()); FP64 buffers keep columns n + 8 nt (four
// conflict-free LDS.64; two LDS.128 would conflict two ways).  bfrag_off() is the lane's column offset, ldB() the loads.
template <typename T, int NT> __device__ __forceinline__ constexpr bool bfrag_vec() { return sizeof(T) == 4 && NT == 4; }
template <typename T, int NT> __device__ __forceinline__ int bfrag_off(int lane) { return bfrag_vec<T, NT>() ? (lane >> 2) * NT : (lane >> 2); }
template <typename T, int NT> __device__ __forceinline__ void ldB(T* b, const T* p) {
  if constexpr (bfrag_vec<T, NT>()) { const float4 v = *reinterpret_cast<const float4*>(p); b[0] = v.x; b[1] = v.y; b[2] = v.z; b[3] = v.w; }
  else {
#pragma unroll
    for (int nt = 0; nt < NT; nt++) b[nt] = p[8 * nt];
  }
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// One persistent CTA per SM.  Warps 0..NW-1 ("workers") build the currents and the colour-flow amplitudes of one helicity
// batch after the other on the FP64 pipe; the last NCW warps ("colour") turn finished batches into |L^T J|^2 on the FP64
// tensor pipe (a separate pipe, so the two overlap) and write the outputs.  The two amplitude buffers are handed over with
// named barriers.  MX (T = float only): 1 = momentum sums / propagator denominators are formed in double before rounding to T (the
// FP32 mode: with float denominators gg -> ttggg misses the 1e-4 / 1e-6 tolerances on 8,192 events, profiles/r2_parity.md);
// 2 = the external wavefunctions too (the mixed mode).  Everything downstream of the amplitudes (u, v rows, colour form,
// helicity sum, eq. 3) runs in double in every mode.
template <int N, typename T, int MX, int NW, int NCW, int CTAS, bool POLY = false>
__global__ void __launch_bounds__((NW + NCW) * 32, CTAS) bg_kernel(const double* __restrict__ mom, const double* __restrict__ wgt,
                                                               double* __restrict__ me_old, double* __restrict__ me_new,
                                                               double* __restrict__ w_new, long long nev, long long stride, long long ostride, BgDev D) {
  typedef Geo<N> Ge;
  constexpr int NTH = (NW + NCW) * 32, NWT = NW * 32, NCT = NCW * 32;
  // register hand-over between the warpgroups: the colour warps need few registers, the workers get the rest
  // (setmaxnreg is a warpgroup instruction: both groups must be whole warpgroups of 4 warps)
  // a1/a2 of the next group on the colour warps: pays when the colour warps are mostly idle and the per-group fixed work is small
  // next to the currents (n >= 4); for n = 3 four colour warps are slower at it than the workers (measured: 5.4 -> 5.9 ms, and 4.58 -> 4.76 ms
  // after the externals became object-major)
  constexpr bool STAGE = (N >= RWGT_STAGE_MIN_N);
  constexpr bool HANDOVER = NW % 4 == 0 && NCW % 4 == 0;
  // the CTA's pool is what it was launched with: (registers per thread under the launch bounds) x warps; an inc beyond it never returns
  constexpr int REG_LAUNCH = (65536 / CTAS / NTH) / 8 * 8 > 255 ? 248 : (65536 / CTAS / NTH) / 8 * 8, REG_POOL = REG_LAUNCH * (NW + NCW);
  constexpr int REG_COL = 56, REG_WORK = ((REG_POOL - NCW * REG_COL) / NW) / 8 * 8 > 232 ? 232 : ((REG_POOL - NCW * REG_COL) / NW) / 8 * 8;
  static_assert(NW * REG_WORK + NCW * REG_COL <= REG_POOL, "register hand-over exceeds the CTA's pool");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Ctx<T> c; c.D = &D; c.ns = D.nslot;
  carve<N, T>(c.s, smem_raw, D.nslot, D.nwords);
  const Smem<T>& s = c.s;
  typedef typename std::conditional<MX >= 1, double, T>::type TK;
  typedef typename std::conditional<MX >= 2, double, T>::type TE;
  constexpr int next = N + 2, nG = Ge::NG, nR = Ge::NR, nL = Ge::NL; const int ns = D.nslot;
  const long long ngroups = (nev + ns - 1) / ns;
  // once per CTA: zero both amplitude buffers (their padding rows are never written again)
  constexpr int ASTR = Ge::template astr<T>(), NBUF = Ge::template nbuf<T>(); constexpr size_t ABUF = Ge::template abuf<T>();
  for (int t = threadIdx.x; t < NBUF * ns * (int)ABUF; t += NTH) s.A[t] = T(0);
  for (int t = threadIdx.x; t < 2 * Ge::KSH * 32; t += NTH) s.LF[t] = __ldg(D.lfrag + t);
  __syncthreads();
  if (threadIdx.x < NWT) {
    // =========================================================================================== worker warps
    if constexpr (HANDOVER) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REG_WORK));
    const int tid = threadIdx.x; c.tid = tid;
    for (int t = tid; t < D.nwords; t += NWT) s.W[t] = __ldg(D.words + t);
    unsigned step = 0;
    // !STAGE (n <= 3): a1 is software-pipelined by the workers themselves: the momenta of the next group travel from HBM into
    // registers while this group's levels and amplitudes run (the load latency was 6 % of the workers' time at n = 3)
    constexpr int MAXSLOT = (N == 2) ? 64 : NWT / (Ge::NPAIR * 4);           // bg_create: pick
    constexpr int NPRE = STAGE ? 1 : (MAXSLOT * next * 4 + NWT - 1) / NWT;
    double pre[NPRE];
    auto fetch = [&](long long g) {
#pragma unroll
      for (int j = 0; j < NPRE; j++) {
        const int t = tid + j * NWT;
        if (t < ns * next * 4) { int sl = t % ns, comp = t / ns; long long ev = g * ns + sl; if (ev >= nev) ev = nev - 1;
          if (D.idx) ev = D.idx[ev];
          pre[j] = __ldg(mom + (size_t)comp * stride + ev); }
      }
    };
    if constexpr (!STAGE) { if ((long long)blockIdx.x < ngroups) fetch(blockIdx.x); }
    for (long long grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
      const long long ev0 = grp * ns;
      if constexpr (!STAGE) {
        // ---- a1/a2 by the workers themselves ----
        bar_sync(BAR_WORK, NWT);
#pragma unroll
        for (int j = 0; j < NPRE; j++) {
          const int t = tid + j * NWT;
          if (t < ns * next * 4) { int sl = t % ns, comp = t / ns; s.pm[(sl * next * 4) + comp] = pre[j]; }
        }
        bar_sync(BAR_WORK, NWT);
        if (grp + gridDim.x < ngroups) fetch(grp + gridDim.x);
        group_externals<N, T, TK, TE>(tid, NWT, ns, ev0, nev, stride, mom, D.idx, D.set[0].mt, s.pm, s.G, nG, s.R, nR, s.L, nL, s.K, s.iK2, s.dR, s.dL, false,
                                  [] { bar_sync(BAR_WORK, NWT); });
      } else {
      // ---- a1/a2 were done for this group by the colour warps (staging buffers): copy them into the tables ----
      bar_sync(BAR_STAGE_FULL, NTH);
      {
        constexpr int n2 = 2 * N;
        for (int t = tid; t < ns * next * 4; t += NWT) s.pm[t] = s.pmS[t];
        for (int t = tid; t < ns * 4 * n2; t += NWT) { int sl = t / (4 * n2), r = t - sl * 4 * n2, cc = r / n2, e = r - cc * n2; s.G[(size_t)sl * 4 * nG + cc * nG + e] = s.GS[t]; }
        for (int t = tid; t < ns * 8; t += NWT) { int sl = t >> 3, r = t & 7, cc = r >> 1, e = r & 1;
          s.R[(size_t)sl * 4 * nR + cc * nR + e] = s.RS[t]; s.L[(size_t)sl * 4 * nL + cc * nL + e] = s.LS[t]; }
        for (int t = tid; t < ns * Ge::NMASK * 4; t += NWT) s.K[t] = s.KS[t];
        for (int t = tid; t < ns * Ge::NMASK; t += NWT) { s.iK2[t] = s.iK2S[t]; s.dR[t] = s.dRS[t]; s.dL[t] = s.dLS[t]; }
      }
      __threadfence_block();
      bar_arrive(BAR_STAGE_EMPTY, NTH);                        // the colour warps may stage the next group
      }
      bar_sync(BAR_WORK, NWT);
      bool fused = false;
      if constexpr (N == 3 && !POLY) if (D.fuse) {
        // ---- n = 3, two sets of equal mass: one pass at unit couplings, four coefficient amplitudes, both sets folded from them ----
        fused = true;
        c.g3 = T(1); c.g4 = T(0); c.gq = T(1); c.mt = (T)D.set[0].mt;
        level_phase<N, 2, T, NWT>(c);
        constexpr int per = Ge::NPAIR * Ge::NFREE;             // one helicity batch for n = 3; at most one task per thread (bg_create: ns * per <= NWT)
        const bool live = tid < ns * per;
        const int sl = live ? tid / per : 0, o = live ? tid - sl * per : 0, pair = o / Ge::NFREE, f = o % Ge::NFREE;
        const cx<T>* G = s.G + (size_t)sl * 4 * nG; const cx<T>* R = s.R + (size_t)sl * 4 * nR; const cx<T>* L = s.L + (size_t)sl * 4 * nL;
        const uint32_t* w = s.W + D.offF + pair * Ge::STRIDEF;
        const uint32_t w0 = w[0], packed = w[1];
        uint32_t v = 0;
#pragma unroll
        for (int j = 0; j < N; j++) v |= ((((uint32_t)f << 1) >> ((packed >> (3 * j)) & 7u)) & 1u) << j;   // helicity bits by position; gluon 0: + (parity)
        // the parameter sets two at a time: the coefficient amplitudes of a chunk are formed once and folded with the chunk's weights
        // (the split three-gluon current is re-formed per chunk: it is dead after the common term, which keeps 32 registers free)
#pragma unroll 1
        for (int k0 = 0; k0 < D.nsets; k0 += 2) {
          const int nk = (k0 + 1 < D.nsets) ? 2 : 1;
          T wt[2][4];
#pragma unroll
          for (int s2 = 0; s2 < 2; s2++) { const BgSet& P = D.set[k0 + (s2 < nk ? s2 : 0)]; wt[s2][0] = (T)(P.gq * P.gq); wt[s2][1] = (T)(P.gq * P.g3); wt[s2][2] = (T)(P.g3 * P.g3); wt[s2][3] = (T)P.g4; }
          cx<T> A0[2][2][2], A1[2][2][2];
          if (live) {
            {
              vec4<T> J2, J3;
              {
                uint32_t jw[Ge::JW]; ldw<Ge::JW>(jw, w + 4);
                GluonSum<N, nG, T>::run_split(J2, J3, jw, v, G, s.K + (size_t)sl * Ge::NMASK * 4);
                const T sc = s.iK2[sl * Ge::NMASK + Ge::NMASK - 1];
#pragma unroll
                for (int i = 0; i < 4; i++) { J2.c[i] = (-sc) * J2.c[i]; J3.c[i] = sc * J3.c[i]; }
              }
              uint32_t wq[Ge::QW]; ldw<Ge::QW>(wq, w + 4 + Ge::JW);
              QuarkLine3F<T>::common(A0, wq, J2, J3, R, L, wt);  // the same for the ordering and its reversal
#pragma unroll
              for (int s2 = 0; s2 < 2; s2++)
#pragma unroll
                for (int a = 0; a < 2; a++)
#pragma unroll
                  for (int b = 0; b < 2; b++) A1[s2][a][b] = A0[s2][a][b];
              QuarkLine3F<T>::run(A0, wq, v, G, R, L, wt);
            }
            {
              uint32_t wq[Ge::QW]; ldw<Ge::QW>(wq, w + 4 + Ge::JW + Ge::QW);
              QuarkLine3F<T>::run(A1, wq, brevm<N>(v), G, R, L, wt);
            }
          }
#pragma unroll
          for (int s2 = 0; s2 < 2; s2++) {
            if (s2 < nk) {
              const int buf = step % NBUF;
              if (step >= NBUF) bar_sync(BAR_EMPTY0 + buf, NTH);    // colour warps have finished reading this buffer
              if (live) {
                T* Au = s.A + (size_t)buf * ns * ABUF + (size_t)sl * ABUF + (size_t)w0 * ASTR; T* Av = Au + (size_t)Ge::NHK * ASTR;
#pragma unroll
                for (int ht = 0; ht < 2; ht++)
#pragma unroll
                  for (int hb = 0; hb < 2; hb++) {
                    const int col = f * 4 + ht * 2 + hb;
                    const double ar = (double)A0[s2][ht][hb].re, ai = (double)A0[s2][ht][hb].im, br = (double)A1[s2][ht][hb].re, bi = (double)A1[s2][ht][hb].im;
                    stc(reinterpret_cast<cx<T>*>(Au + 2 * col), mk<T>((T)(ar + br), (T)(ai + bi)));
                    stc(reinterpret_cast<cx<T>*>(Av + 2 * col), mk<T>((T)(ar - br), (T)(ai - bi)));
                  }
              }
              __threadfence_block();
              bar_arrive(BAR_FULL0 + buf, NTH);                  // hand this set's amplitudes to the colour warps
              step++;
            }
          }
        }
        bar_sync(BAR_WORK, NWT);                               // the current tables are rewritten for the next group
      }
      const int neval = fused ? 0 : (POLY ? D.nnode : D.nsets);   // polynomial mode: one evaluation per node set, not per parameter set
#pragma unroll 1
      for (int iset = 0; iset < neval; iset++) {
        const BgSet& P = POLY ? D.node[iset] : D.set[iset];
        c.g3 = (T)P.g3; c.g4 = (T)P.g4; c.gq = (T)P.gq; c.mt = (T)P.mt;
        if (!POLY && iset > 0 && !D.shared_ext) {
          // a set with another top mass: external spinors and denominators are redone for it (reading R12)
          group_externals<N, T, TK, TE>(tid, NWT, ns, ev0, nev, stride, mom, D.idx, P.mt, s.pm, s.G, nG, s.R, nR, s.L, nL, s.K, s.iK2, s.dR, s.dL, false, [] {});
          bar_sync(BAR_WORK, NWT);
        }
        // ---- a3: current levels ----
        level_phase<N, 2, T, NWT>(c);
        if constexpr (Ge::NPHASE >= 3) level_phase<N, 3, T, NWT>(c);
        if constexpr (Ge::NPHASE >= 4) level_phase<N, 4, T, NWT>(c);
        // ---- a3/a4: colour-flow amplitudes, one helicity batch per buffer hand-over ----
#pragma unroll 1
        for (int batch = 0; batch < Ge::NBATCH; batch++, step++) {
          const int buf = step % NBUF;
          if (step >= NBUF) bar_sync(BAR_EMPTY0 + buf, NTH);      // colour warps have finished reading this buffer
          T* Abuf = s.A + (size_t)buf * ns * ABUF;
          constexpr int per = Ge::NPAIR * Ge::NFREE;
          for (int t = tid; t < ns * per; t += NWT) {
            int sl = t / per, o = t - sl * per; int pair = o / Ge::NFREE, f = o % Ge::NFREE;
            const cx<T>* G = s.G + (size_t)sl * 4 * nG; const cx<T>* R = s.R + (size_t)sl * 4 * nR; const cx<T>* L = s.L + (size_t)sl * 4 * nL;
            const T* K = s.K + (size_t)sl * Ge::NMASK * 4;
            const uint32_t* w = s.W + D.offF + pair * Ge::STRIDEF;
            uint32_t w0 = w[0], packed = w[1];
            uint32_t g = ((uint32_t)batch << 1) | ((uint32_t)f << (1 + Ge::NB));   // helicity bits by gluon label; gluon 0: + (parity)
            uint32_t v = 0;
#pragma unroll
            for (int j = 0; j < N; j++) v |= ((g >> ((packed >> (3 * j)) & 7u)) & 1u) << j;   // by position in sigma
            vec4<T> Jn;
            {
              uint32_t jw[Ge::JW]; ldw<Ge::JW>(jw, w + 4);
              Jn = GluonSum<N, nG, T>::run(jw, v, G, K, c.g3, c.g4);
            }
            T sc = s.iK2[sl * Ge::NMASK + Ge::NMASK - 1];
#pragma unroll
            for (int i = 0; i < 4; i++) Jn.c[i] = sc * Jn.c[i];
            cx<T> A0[2][2], A1[2][2];
            {
              uint32_t wq[Ge::QW]; ldw<Ge::QW>(wq, w + 4 + Ge::JW);
              spn<T> XT[2];                                        // ubar Jn-slash, shared by the ordering and its reversal
              if constexpr (share_full_term<N, T>()) {
                const lcv<T> Jl = lightcone(Jn); const int el0 = (int)halfw(wq, 0);
#pragma unroll
                for (int ht = 0; ht < 2; ht++) {
#pragma unroll
                  for (int i = 0; i < 4; i++) XT[ht].c[i] = mk<T>(0, 0);
                  row_slash_acc(XT[ht], lds4(L, nL, el0 + ht), Jl);
                }
              }
              QuarkLine<N, 0, T>::run(A0, wq, v, Jn, XT, G, R, L);
              uint32_t wr[Ge::QW]; ldw<Ge::QW>(wr, w + 4 + Ge::JW + Ge::QW);
              QuarkLine<N, 1, T>::run(A1, wr, brevm<N>(v), Jn, XT, G, R, L);
            }
            // rows u = J_s + J_rev(s) and v = J_s - J_rev(s) of the pair (formed in double)
            T* Au = Abuf + (size_t)sl * ABUF + (size_t)w0 * ASTR; T* Av = Au + (size_t)Ge::NHK * ASTR;
#pragma unroll
            for (int ht = 0; ht < 2; ht++)
#pragma unroll
              for (int hb = 0; hb < 2; hb++) {
                const int col = f * 4 + ht * 2 + hb;
                const double ar = (double)A0[ht][hb].re, ai = (double)A0[ht][hb].im, br = (double)A1[ht][hb].re, bi = (double)A1[ht][hb].im;
                stc(reinterpret_cast<cx<T>*>(Au + 2 * col), mk<T>((T)(ar + br), (T)(ai + bi)));
                stc(reinterpret_cast<cx<T>*>(Av + 2 * col), mk<T>((T)(ar - br), (T)(ai - bi)));
              }
          }
          __threadfence_block();
          bar_arrive(BAR_FULL0 + buf, NTH);                    // hand the batch to the colour warps
        }
        bar_sync(BAR_WORK, NWT);                               // the current tables are rewritten for the next parameter set / group
      }
      if constexpr (POLY) {
        // ---- a5/a6 in polynomial mode: the colour warps have written Z_j = L^T (u_j | v_j) of every node set j and helicity batch to the
        // CTA's global scratch (all nodes in one element order).  The colour form is quadratic in J and J(set k) = sum_j cw_kj J_j, so
        // what an event needs are the cross forms Q_jj' = sum_elements Z_j Z_j': a streaming pass, fixed reduction order.
        constexpr int NP = BG_RMAX * (BG_RMAX + 1) / 2, ZEL = Ge::NBATCH * Ge::U * 2 * Ge::NT * 64;   // doubles of one (node, slot)
        static_assert(Ge::MTH % 2 == 0, "polynomial mode: every (unit, half) of the triangular mma must exist");
        const double* Zc = D.poly_scratch + (size_t)blockIdx.x * D.poly_stride;
        double* red = s.pred;                                  // [NW][NP], one slot at a time
        const int warp = tid >> 5, lane = tid & 31, nnode = D.nnode;
        bar_sync(BAR_ZFULL, NTH);                              // all Z of this group are in the scratch
#pragma unroll 1
        for (int sl = 0; sl < ns; sl++) {
          double q[NP];
#pragma unroll
          for (int pi = 0; pi < NP; pi++) q[pi] = 0.0;
          for (int e2 = tid; e2 < ZEL / 2; e2 += NWT) {
            double2 z[BG_RMAX];
#pragma unroll
            for (int j = 0; j < BG_RMAX; j++) z[j] = (j < nnode) ? __ldcg(reinterpret_cast<const double2*>(Zc + ((size_t)j * ns + sl) * ZEL) + e2) : make_double2(0.0, 0.0);
            int pi = 0;
#pragma unroll
            for (int j = 0; j < BG_RMAX; j++)
#pragma unroll
              for (int j2 = j; j2 < BG_RMAX; j2++, pi++) { q[pi] = fma(z[j].x, z[j2].x, q[pi]); q[pi] = fma(z[j].y, z[j2].y, q[pi]); }
          }
#pragma unroll
          for (int d = 16; d >= 1; d >>= 1)
#pragma unroll
            for (int pi = 0; pi < NP; pi++) q[pi] += __shfl_xor_sync(0xffffffffu, q[pi], d);
          if (lane == 0) {
#pragma unroll
            for (int pi = 0; pi < NP; pi++) red[warp * NP + pi] = q[pi];
          }
          bar_sync(BAR_WORK, NWT);
          // ---- a6/a7: one thread: the warps' partial sums in fixed order, every parameter set, eq. 3, stores ----
          if (tid == 0) {
            long long ev = ev0 + sl;
            if (ev < nev) {
              if (D.idx) ev = D.idx[ev];
              double Q[NP];
#pragma unroll
              for (int pi = 0; pi < NP; pi++) { double a = 0.0; for (int wv = 0; wv < NW; wv++) a += red[wv * NP + pi]; Q[pi] = a; }
              const double W = __ldg(wgt + ev); double a0 = 0.0;
              for (int k = 0; k < D.nsets; k++) {
                double me = 0.0; int pi = 0;
#pragma unroll
                for (int j = 0; j < BG_RMAX; j++)
#pragma unroll
                  for (int j2 = j; j2 < BG_RMAX; j2++, pi++) me = fma((j == j2 ? 1.0 : 2.0) * D.cw[k][j] * D.cw[k][j2], Q[pi], me);
                me *= D.set[k].fac;
                if (k == 0) { a0 = me; me_old[ev] = me; }
                else { me_new[(size_t)(k - 1) * ostride + ev] = me; w_new[(size_t)(k - 1) * ostride + ev] = W * (me / a0); }
              }
            }
          }
          bar_sync(BAR_WORK, NWT);                             // red is reused by the next slot
        }
      }
    }
  } else {
    // =========================================================================================== colour warps
    if constexpr (HANDOVER) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REG_COL));
    const int ctid = threadIdx.x - NWT, cwarp = ctid >> 5, lane = ctid & 31;
    unsigned step = 0;
    // a1 + a2 of an event group into the staging buffers (parameter set 0; masses of the other sets: see the workers)
    auto stage = [&](long long g) {
      group_externals<N, T, TK, TE>(ctid, NCT, ns, g * ns, nev, stride, mom, D.idx, D.set[0].mt, s.pmS, s.GS, 2 * N, s.RS, 2, s.LS, 2, s.KS, s.iK2S, s.dRS, s.dLS, true,
                                [] { bar_sync(BAR_COLOUR, NCT); });
      __threadfence_block();
      bar_arrive(BAR_STAGE_FULL, NTH);
    };
    if (STAGE && (long long)blockIdx.x < ngroups) stage(blockIdx.x);
    for (long long grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
      const long long ev0 = grp * ns;
      for (int t = ctid; t < ns * BG_NSMAX; t += NCT) s.acc[t] = 0.0;
      if constexpr (STAGE) {
        bar_sync(BAR_STAGE_EMPTY, NTH);                        // the workers have taken this group's staged data
        if (grp + gridDim.x < ngroups) stage(grp + gridDim.x); // the next group's fixed work overlaps the workers' currents and amplitudes
      }
      bar_sync(BAR_COLOUR, NCT);
      const int neval = POLY ? D.nnode : D.nsets;
      double* const Zc = POLY ? D.poly_scratch + (size_t)blockIdx.x * D.poly_stride : nullptr;
#pragma unroll 1
      for (int iset = 0; iset < neval; iset++) {
#pragma unroll 1
        for (int batch = 0; batch < Ge::NBATCH; batch++, step++) {
          const int buf = step % NBUF;
          bar_sync(BAR_FULL0 + buf, NTH);                      // the workers have filled this buffer
          const T* Abuf = s.A + (size_t)buf * ns * ABUF;
          // a5: Z = L^T A with FP64 tensor-core mma over the upper-triangular tiles, colour form = sum of squares of Z
          if constexpr (Ge::MTH == 1 && Ge::KTH == 1) {
            // n <= 3: one 8x4 tile per half, so a unit is four mma and a shuffle tree, i.e. pure latency.  Four units (slot x half) are
            // written out side by side so that their chains overlap; each unit's arithmetic and order are the same as in the general path.
            constexpr int UB = 4;
            for (int u0 = cwarp * UB; u0 < ns * 2; u0 += NCW * UB) {
              double part[UB];
#pragma unroll
              for (int j = 0; j < UB; j++) {
                const int u = (u0 + j < ns * 2) ? u0 + j : ns * 2 - 1, sl = u >> 1, h = u & 1;
                const T* A = Abuf + (size_t)sl * ABUF + (size_t)(h * Ge::NHK + (lane & 3)) * ASTR + bfrag_off<T, Ge::NT>(lane);
                const double a = s.LF[h * 32 + lane];
                double acc[Ge::NT][2]; T bb[Ge::NT]; ldB<T, Ge::NT>(bb, A);
#pragma unroll
                for (int nt = 0; nt < Ge::NT; nt++) { acc[nt][0] = 0.0; acc[nt][1] = 0.0; dmma884(acc[nt][0], acc[nt][1], a, (double)bb[nt]); }
                double pj = 0.0;
#pragma unroll
                for (int nt = 0; nt < Ge::NT; nt++) { pj = fma(acc[nt][0], acc[nt][0], pj); pj = fma(acc[nt][1], acc[nt][1], pj); }
                part[j] = pj;
              }
#pragma unroll
              for (int d = 16; d >= 1; d >>= 1)
#pragma unroll
                for (int j = 0; j < UB; j++) part[j] += __shfl_xor_sync(0xffffffffu, part[j], d);
#pragma unroll
              for (int j = 0; j < UB; j++) if (lane == 0 && u0 + j < ns * 2) s.red[((u0 + j) >> 1) * 8 + ((u0 + j) & 1)] = part[j];
            }
          } else
          for (int u = cwarp; u < ns * Ge::U; u += NCW) {
            int sl = u / Ge::U, unit = u % Ge::U; const int h = unit / Ge::UH, uu = unit % Ge::UH;     // h: 0 = u rows / L+, 1 = v rows / L-
            const T* A = Abuf + (size_t)sl * ABUF + (size_t)(h * Ge::NHK + (lane & 3)) * ASTR + bfrag_off<T, Ge::NT>(lane);
            double part = 0.0;
#pragma unroll 1
            for (int half = 0; half < 2; half++) {
              int mt = half ? Ge::MTH - 1 - uu : uu;
              if (half && mt == uu) break;
              double acc[Ge::NT][2];
#pragma unroll
              for (int nt = 0; nt < Ge::NT; nt++) { acc[nt][0] = 0.0; acc[nt][1] = 0.0; }
              const double* F = s.LF + (h * Ge::KSH + mt * Ge::KTH - mt * (mt - 1)) * 32 + lane;
              const int nk = Ge::KTH - 2 * mt;
              const T* Br = A + (size_t)(8 * mt) * ASTR;
              // operands of k-step kk + 1 are fetched from shared memory while the mma of k-step kk issue
              double a_cur = F[0]; T b_cur[Ge::NT];
              ldB<T, Ge::NT>(b_cur, Br);
#pragma unroll 2
              for (int kk = 0; kk < nk; kk++) {
                const int kn = (kk + 1 < nk) ? kk + 1 : kk;
                const double a_nxt = F[kn * 32]; T b_nxt[Ge::NT];
                ldB<T, Ge::NT>(b_nxt, Br + (size_t)(4 * kn) * ASTR);
#pragma unroll
                for (int nt = 0; nt < Ge::NT; nt++) dmma884(acc[nt][0], acc[nt][1], a_cur, (double)b_cur[nt]);
                a_cur = a_nxt;
#pragma unroll
                for (int nt = 0; nt < Ge::NT; nt++) b_cur[nt] = b_nxt[nt];
              }
              if constexpr (POLY) {
                // polynomial mode: keep Z itself (global scratch, [node][slot][batch][unit][half][n-tile][lane][2]); the workers form the cross terms
                double* z = Zc + ((((size_t)(iset * ns + sl) * Ge::NBATCH + batch) * Ge::U + unit) * 2 + half) * (Ge::NT * 64) + lane * 2;
#pragma unroll
                for (int nt = 0; nt < Ge::NT; nt++) __stcg(reinterpret_cast<double2*>(z + nt * 64), make_double2(acc[nt][0], acc[nt][1]));
              } else {
#pragma unroll
              for (int nt = 0; nt < Ge::NT; nt++) { part = fma(acc[nt][0], acc[nt][0], part); part = fma(acc[nt][1], acc[nt][1], part); }
              }
            }
            if constexpr (!POLY) {
            // a6: deterministic reduction (same order for both parameter sets => old == new gives a ratio of exactly 1)
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
            if (lane == 0) s.red[sl * 8 + unit] = part;
            }
          }
          if constexpr (POLY) {
            __threadfence_block();
            bar_arrive(BAR_EMPTY0 + buf, NTH);                 // buffer may be refilled
          } else {
          bar_sync(BAR_COLOUR, NCT);
          bar_arrive(BAR_EMPTY0 + buf, NTH);                   // buffer may be refilled
          for (int sl = ctid; sl < ns; sl += NCT) { double a = 0.0; for (int j = 0; j < Ge::U; j++) a += s.red[sl * 8 + j]; s.acc[sl * BG_NSMAX + iset] += a; }
          bar_sync(BAR_COLOUR, NCT);
          }
        }
      }
      if constexpr (POLY) {
        __threadfence_block();
        bar_arrive(BAR_ZFULL, NTH);                            // every Z of this group is written: the workers form the cross terms and the outputs
      }
      // ---- a7: eq. 3 and stores ----
      if constexpr (!POLY)
      for (int sl = ctid; sl < ns; sl += NCT) {
        long long ev = ev0 + sl;
        if (ev < nev) {
          if (D.idx) ev = D.idx[ev];
          const double a = s.acc[sl * BG_NSMAX] * D.set[0].fac, W = __ldg(wgt + ev);
          me_old[ev] = a;
          for (int k = 1; k < D.nsets; k++) {
            const double b = s.acc[sl * BG_NSMAX + k] * D.set[k].fac;
            me_new[(size_t)(k - 1) * ostride + ev] = b; w_new[(size_t)(k - 1) * ostride + ev] = W * (b / a);
          }
        }
      }
      bar_sync(BAR_COLOUR, NCT);
    }
  }
}

// ------------------------------------------------------------------------------------------------ polynomial mode (host)
// PAPER.md:87 step 7 / PAPER.md:117 (run time against the number of parameter sets); "each extra coupling-only set
// costs one more J accumulation + one quadratic form, no new wavefunctions".  With summed currents the route to that is exact
// interpolation: for fixed g_s and m_t every J_sigma is a polynomial in (x, y) = (ggg_scale, gggg_scale) with the monomials
// x^a y^b, a + 2 b <= n - 1 (a three-gluon vertices, b four-gluon vertices of a diagram), and alpha_s is an overall
// factor g_s^(n-1).  Let P[k][m] be the monomials at the requested sets.  Its rank r is the number of sets that have to be evaluated:
// r rows ("node sets", chosen among the requested ones by complete pivoting) span the row space, every other set is an exact linear
// combination P[k] = sum_j cw[k][j] P[node_j], hence J(set k) = (g_k/g_0)^(n-1) sum_j cw[k][j] J(node_j) for every sigma and helicity.
// The colour form is quadratic in J, so the kernel keeps the r (r + 1) / 2 cross forms Q_jj' = sum_h Re(J_j^+ C J_j') of an event and
// every parameter set costs r (r + 1) / 2 multiply-adds.  Used when all sets share m_t, n >= 4, and r <= BG_RMAX is smaller than
// the number of sets.  A set equal to the old one has the same weights and factor as the old one: W' = W bitwise.
static bool bg_plan_poly(int n, const rwgt_params* sets, int nsets, BgDev& D) {
  D.poly = 0; D.nnode = 0;
  if (n < 4 || nsets < 3) return false;
  for (int k = 1; k < nsets; k++) if (sets[k].mt != sets[0].mt) return false;
  std::vector<std::pair<int, int>> mono;
  for (int b = 0; 2 * b <= n - 1; b++) for (int a = 0; a + 2 * b <= n - 1; a++) mono.push_back({a, b});
  const int M = (int)mono.size();
  std::vector<std::vector<long double>> P(nsets, std::vector<long double>(M));
  for (int k = 0; k < nsets; k++) for (int m = 0; m < M; m++) P[k][m] = std::pow((long double)sets[k].ggg_scale, mono[m].first) * std::pow((long double)sets[k].gggg_scale, mono[m].second);
  // complete pivoting: rows = sets, columns = monomials
  std::vector<std::vector<long double>> Wk = P; std::vector<int> rows, cols; std::vector<bool> rused(nsets, false), cused(M, false);
  long double scale = 0; for (auto& r : P) for (auto v : r) scale = std::max(scale, std::fabs(v));
  for (int step = 0; step < std::min(nsets, M); step++) {
    int br = -1, bc = -1; long double best = 0;
    for (int k = 0; k < nsets; k++) if (!rused[k]) for (int m = 0; m < M; m++) if (!cused[m] && std::fabs(Wk[k][m]) > best) { best = std::fabs(Wk[k][m]); br = k; bc = m; }
    if (br < 0 || best < 1e-9L * scale) break;
    rused[br] = true; cused[bc] = true; rows.push_back(br); cols.push_back(bc);
    for (int k = 0; k < nsets; k++) if (!rused[k]) { long double f = Wk[k][bc] / Wk[br][bc]; for (int m = 0; m < M; m++) Wk[k][m] -= f * Wk[br][m]; }
  }
  const int r = (int)rows.size();
  if (r > BG_RMAX || r >= nsets) return false;
  std::sort(rows.begin(), rows.end());
  // weights: cw[k] B = P[k][cols], B[j][s] = P[node_j][col_s]  (transposed system, Gaussian elimination with partial pivoting)
  for (int k = 0; k < nsets; k++) {
    long double A[BG_RMAX][BG_RMAX + 1];
    for (int s2 = 0; s2 < r; s2++) { for (int j = 0; j < r; j++) A[s2][j] = P[rows[j]][cols[s2]]; A[s2][r] = P[k][cols[s2]]; }
    for (int c0 = 0; c0 < r; c0++) {
      int pv = c0; for (int i = c0 + 1; i < r; i++) if (std::fabs(A[i][c0]) > std::fabs(A[pv][c0])) pv = i;
      if (A[pv][c0] == 0) return false;
      if (pv != c0) for (int j = 0; j <= r; j++) std::swap(A[pv][j], A[c0][j]);
      for (int i = 0; i < r; i++) if (i != c0) { long double f = A[i][c0] / A[c0][c0]; for (int j = c0; j <= r; j++) A[i][j] -= f * A[c0][j]; }
    }
    long double wsum = 0;
    for (int j = 0; j < BG_RMAX; j++) { D.cw[k][j] = j < r ? (double)(A[j][r] / A[j][j]) : 0.0; wsum += std::fabs((long double)D.cw[k][j]); }
    // exactness on EVERY monomial (the rank argument), and no blow-up of rounding errors
    for (int m = 0; m < M; m++) { long double v = 0; for (int j = 0; j < r; j++) v += (long double)D.cw[k][j] * P[rows[j]][m]; if (std::fabs(v - P[k][m]) > 1e-13L * scale * (1 + wsum)) return false; }
    if (wsum > 50) return false;
  }
  const double gs0 = std::sqrt(4.0 * 3.14159265358979323846 * sets[0].alpha_s);
  for (int j = 0; j < r; j++) { D.node[j].gq = gs0; D.node[j].g3 = gs0 * sets[rows[j]].ggg_scale; D.node[j].g4 = gs0 * gs0 * sets[rows[j]].gggg_scale; D.node[j].mt = sets[0].mt; D.node[j].fac = 0; }
  D.poly = 1; D.nnode = r;
  return true;
}

// ------------------------------------------------------------------------------------------------ host API of the engine
template <int N> static size_t smem_need(const BgSched& S, int nslot, bool dbl) {
  if (dbl) { Smem<double> s; return carve<N, double>(s, nullptr, nslot, (int)S.words.size()); }
  Smem<float> s; return carve<N, float>(s, nullptr, nslot, (int)S.words.size());
}
static size_t smem_need_n(int n, const BgSched& S, int nslot, bool dbl) {
  switch (n) { case 2: return smem_need<2>(S, nslot, dbl); case 3: return smem_need<3>(S, nslot, dbl); case 4: return smem_need<4>(S, nslot, dbl); default: return smem_need<5>(S, nslot, dbl); }
}
// Warp split: one CTA per SM, 8 worker warps (FP64 / FP32 pipe) + 4 colour warps (DMMA) = 3 warps x 168 registers per SM
// sub-partition.  Measured on B200 against 10+2, 6+2, 12+4 and (n = 3) two CTAs of 4+2 warps per SM: best or within 4 % of best
// for every process.  (The kernel is parametrised on the split and on the CTAs per SM.)  FP32/mixed n = 4: 12 worker warps with 152
// registers (hand-over from the colour warps) and 8 event slots: 6.35 -> 5.70 ms (16 workers at 104 registers: 6.47).  n = 5 stays at 8:
// one event slot gives 240 amplitude tasks per batch, a second slot does not fit beside the FP64 amplitude buffers.  FP32/mixed n = 3:
// 12 workers 3.79 -> 3.16 ms.  FP64 with 12 workers at 152 registers is slower (n = 4: 10.9 -> 11.9 ms, n = 3: 5.39 -> 5.50 ms).
// Round 2: n = 5 FP32 has two event slots (float amplitude buffers).  n = 3 FP64: 12 workers with one amplitude buffer and 32 slots
// (4.65 -> 4.22 ms) until the one-pass form, whose amplitude threads hold two sets' amplitudes: 8 workers at 224 registers, 21 slots
// and two buffers 3.32 ms against 3.60 (12 workers, spills to a 28 KB L1) and 3.64 (8 workers, one buffer: the second set's rows wait
// for the colour form of the first).
constexpr int RWGT_NW32_N4 = 12;
constexpr int RWGT_NW64_N4 = 8;
constexpr int RWGT_NW32_N3 = 12;
constexpr int RWGT_NW64_N3 = 8;
constexpr int RWGT_NW32_N5 = 8;
// CTAs per SM at n = 3 (the phases of independent CTAs drift apart and could overlap one CTA's per-group fixed work with another's
// amplitude phase): measured after the one-pass form, 2 CTAs of 4 + 4 warps 3.93 ms FP64 / 2.18 ms FP32 (8 + 4: 1.99 FP32), 3 CTAs 4.92 / 2.11,
// against 3.36 / 1.67 for one CTA: the colour warpgroups of the extra CTAs cost more registers and shared memory than the overlap returns
constexpr int RWGT_CTAS64_N3 = 1;
constexpr int RWGT_CTAS32_N3 = 1;
constexpr int RWGT_SLOTS32_N5 = 2;
template <int N, typename T> struct BgCfg { static constexpr int NW = (N == 4) ? (sizeof(T) == 4 ? RWGT_NW32_N4 : RWGT_NW64_N4) : (N == 3) ? (sizeof(T) == 4 ? RWGT_NW32_N3 : RWGT_NW64_N3) : (N == 5 && sizeof(T) == 4) ? RWGT_NW32_N5 : 8, NCW = 4,
                                                        CTAS = (N == 3) ? (sizeof(T) == 4 ? RWGT_CTAS32_N3 : RWGT_CTAS64_N3) : 1; };
static int bg_nw(int n, bool dbl) { return n == 4 ? (dbl ? BgCfg<4, double>::NW : BgCfg<4, float>::NW) : n == 3 ? (dbl ? BgCfg<3, double>::NW : BgCfg<3, float>::NW) : n == 5 ? (dbl ? BgCfg<5, double>::NW : BgCfg<5, float>::NW) : 8; }
static int bg_ctas(int n, bool dbl) { return n == 3 ? (dbl ? BgCfg<3, double>::CTAS : BgCfg<3, float>::CTAS) : 1; }

template <int N> static cudaError_t bg_set_attr(size_t s64, size_t s32) {
  typedef BgCfg<N, double> Cd; typedef BgCfg<N, float> Cf;
  cudaError_t e = cudaFuncSetAttribute(bg_kernel<N, double, 0, Cd::NW, Cd::NCW, Cd::CTAS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s64);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<N, float, 1, Cf::NW, Cf::NCW, Cf::CTAS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s32);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<N, float, 2, Cf::NW, Cf::NCW, Cf::CTAS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s32);
  if constexpr (N >= 4) {
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<N, double, 0, Cd::NW, Cd::NCW, Cd::CTAS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s64);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<N, float, 1, Cf::NW, Cf::NCW, Cf::CTAS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s32);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<N, float, 2, Cf::NW, Cf::NCW, Cf::CTAS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s32);
  }
  return e;
}
template <int N> static void bg_launch(int precision, int grid, size_t s64, size_t s32, cudaStream_t st, const double* mom, const double* w,
                                       double* a, double* b, double* o, long long nev, long long stride, long long ostride, const BgDev& D) {
  typedef BgCfg<N, double> Cd; typedef BgCfg<N, float> Cf;
  if constexpr (N >= 4) if (D.poly) {
    if (precision == RWGT_FP64) bg_kernel<N, double, 0, Cd::NW, Cd::NCW, Cd::CTAS, true><<<grid, (Cd::NW + Cd::NCW) * 32, s64, st>>>(mom, w, a, b, o, nev, stride, ostride, D);
    else if (precision == RWGT_FP32) bg_kernel<N, float, 1, Cf::NW, Cf::NCW, Cf::CTAS, true><<<grid, (Cf::NW + Cf::NCW) * 32, s32, st>>>(mom, w, a, b, o, nev, stride, ostride, D);
    else bg_kernel<N, float, 2, Cf::NW, Cf::NCW, Cf::CTAS, true><<<grid, (Cf::NW + Cf::NCW) * 32, s32, st>>>(mom, w, a, b, o, nev, stride, ostride, D);
    return;
  }
  if (precision == RWGT_FP64) bg_kernel<N, double, 0, Cd::NW, Cd::NCW, Cd::CTAS><<<grid, (Cd::NW + Cd::NCW) * 32, s64, st>>>(mom, w, a, b, o, nev, stride, ostride, D);
  else if (precision == RWGT_FP32) bg_kernel<N, float, 1, Cf::NW, Cf::NCW, Cf::CTAS><<<grid, (Cf::NW + Cf::NCW) * 32, s32, st>>>(mom, w, a, b, o, nev, stride, ostride, D);
  else bg_kernel<N, float, 2, Cf::NW, Cf::NCW, Cf::CTAS><<<grid, (Cf::NW + Cf::NCW) * 32, s32, st>>>(mom, w, a, b, o, nev, stride, ostride, D);
}

static size_t bg_zel(int n) { return n == 5 ? (size_t)Geo<5>::NBATCH * Geo<5>::U * 2 * Geo<5>::NT * 64 : (size_t)Geo<4>::NBATCH * Geo<4>::U * 2 * Geo<4>::NT * 64; }
static BgProcess* bg_create(int n, const rwgt_params* sets, int nsets, std::string& err) {
  BgProcess* B = new BgProcess();
  B->d_words = nullptr; B->d_lfrag = nullptr; B->d_poly = nullptr;
  B->S = build_schedule(n, err);
  if (!err.empty()) { delete B; return nullptr; }
  const BgSched& S = B->S;
  BgDev& D = B->D;
  D.nwords = (int)S.words.size(); D.offF = S.offF; D.idx = nullptr;
  bool ok = (S.nG == c_nG(n) && S.nR == c_nR(n) && S.nL == c_nL(n) && S.npair == S.nperm / 2);
  for (int m = 2; m <= n - 1; m++) ok = ok && S.ntask[0][m] == c_ntaskG(n, m);
  for (int m = 1; m <= S.rmax; m++) ok = ok && S.ntask[1][m + 1] == c_ntaskQ(n, m);
  for (int m = 1; m <= S.lmax; m++) ok = ok && S.ntask[2][m + 1] == c_ntaskQ(n, m);
  switch (n) { case 2: ok = ok && S.strideF == Geo<2>::STRIDEF; break; case 3: ok = ok && S.strideF == Geo<3>::STRIDEF; break;
               case 4: ok = ok && S.strideF == Geo<4>::STRIDEF; break; default: ok = ok && S.strideF == Geo<5>::STRIDEF; }
  if (!ok) { err = "internal: schedule/geometry mismatch"; delete B; return nullptr; }
  for (int k = 0; k < 3; k++) for (int m = 0; m < 6; m++) D.offD[k][m] = S.offD[k][m];
  for (int m = 0; m < 6; m++) D.offT[m] = S.offT[m];
  double fact = 1; for (int i = 2; i <= n - 2; i++) fact *= i;
  D.nsets = nsets; D.shared_ext = 1;
  for (int k = 0; k < nsets; k++) {
    double gs = std::sqrt(4.0 * 3.14159265358979323846 * sets[k].alpha_s);
    D.set[k].gq = gs; D.set[k].g3 = gs * sets[k].ggg_scale; D.set[k].g4 = gs * gs * sets[k].gggg_scale; D.set[k].mt = sets[k].mt;
    D.set[k].fac = 2.0 * gs * gs / (256.0 * fact);
    if (sets[k].mt != sets[0].mt) D.shared_ext = 0;     // externals, momentum sums and denominators are then redone per set
  }
  D.poly_scratch = nullptr; D.poly_stride = 0;
  D.fuse = (n == 3 && D.shared_ext) ? 1 : 0;
  if (bg_plan_poly(n, sets, nsets, D)) {
    // node currents carry the OLD set's g_s; a set's own alpha_s is the overall factor (g_k / g_0)^(2 (n - 1)) of its colour form
    const double gs0 = D.node[0].gq;
    for (int k = 0; k < nsets; k++) D.set[k].fac *= std::pow(D.set[k].gq / gs0, 2.0 * (n - 1));
  }
  int dev = 0; cudaGetDevice(&dev); cudaDeviceProp prop; cudaGetDeviceProperties(&prop, dev);
  B->sm_count = prop.multiProcessorCount; size_t maxsm = prop.sharedMemPerBlockOptin;
  // event slots per CTA: as many as make the amplitude phase fill the 256 worker threads (npair * 4 tasks per slot and batch)
  auto pick = [&](bool dbl, int& nslot, size_t& bytes) {
    int cap = std::max(1, std::min(64, (bg_nw(n, dbl) * 32) / (S.npair * (n == 2 ? 2 : 4)))); nslot = 0;
    if (n == 5 && !dbl) cap = RWGT_SLOTS32_N5;       // float amplitude buffers: a second event slot fits (two rounds of amplitude tasks per batch)
    // with k CTAs per SM each gets 1/k of the SM's shared memory (1 KB per CTA is reserved by the system)
    size_t budget = std::min(maxsm, prop.sharedMemPerMultiprocessor / bg_ctas(n, dbl) - 1024);
    for (int e = cap; e >= 1; e--) if (smem_need_n(n, S, e, dbl) <= budget) { nslot = e; break; }
    bytes = nslot ? smem_need_n(n, S, nslot, dbl) : 0;
  };
  pick(true, B->nslot64, B->smem64); pick(false, B->nslot32, B->smem32);
  if (!B->nslot64 || !B->nslot32) { err = "not enough shared memory per block on this device"; delete B; return nullptr; }
  cudaError_t e = cudaMalloc((void**)&B->d_words, S.words.size() * sizeof(uint32_t));
  if (e == cudaSuccess) e = cudaMalloc((void**)&B->d_lfrag, S.lfrag.size() * sizeof(double));
  if (e == cudaSuccess) e = cudaMemcpy(B->d_words, S.words.data(), S.words.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(B->d_lfrag, S.lfrag.data(), S.lfrag.size() * sizeof(double), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) switch (n) { case 2: e = bg_set_attr<2>(B->smem64, B->smem32); break; case 3: e = bg_set_attr<3>(B->smem64, B->smem32); break;
                                     case 4: e = bg_set_attr<4>(B->smem64, B->smem32); break; default: e = bg_set_attr<5>(B->smem64, B->smem32); }
  if (e == cudaSuccess && D.poly) {
    // scratch of the polynomial mode: per CTA nnode x slots x (NBATCH x U x 2 x NT x 64) doubles
    auto elems = [&](bool dbl) { return (size_t)D.nnode * (dbl ? B->nslot64 : B->nslot32) * bg_zel(n); };
    e = cudaMalloc((void**)&B->d_poly, sizeof(double) * std::max(elems(true), elems(false)) * (size_t)B->sm_count * std::max(bg_ctas(n, true), bg_ctas(n, false)));
    D.poly_scratch = B->d_poly;
  }
  if (e != cudaSuccess) { err = std::string("CUDA: ") + cudaGetErrorString(e); cudaFree(B->d_words); cudaFree(B->d_lfrag); cudaFree(B->d_poly); delete B; return nullptr; }
  D.words = B->d_words; D.lfrag = B->d_lfrag;
  return B;
}
static void bg_destroy(BgProcess* B) { if (!B) return; cudaFree(B->d_words); cudaFree(B->d_lfrag); cudaFree(B->d_poly); delete B; }

// Algorithmic flop count of the schedule on the FP64 (or FP32) FMA pipe, all parameter sets of the handle, per event: FMA = 2 flop,
// MUL = ADD = 1 flop, per operation of rwgt_math.cuh (L3 74 FMA + 6 MUL + 4 ADD, V4 90 + 6 + 2, slash-accumulate 32 FMA,
// light-cone 8 ADD, propagator 24 FMA + 17 MUL + 6 ADD, row.col 16 FMA, current store 8 FMA + 16 MUL), times the number of
// such operations the schedule executes (helicity variants with gluon 0 at helicity - are not evaluated and not counted).
static double bg_flops_per_event(const BgProcess* B, int precision) {
  const int n = B->S.n; const double fl[8] = {158, 188, 64, 8, 71, 32, 32, 16};
  double fp = 0; for (int k = 0; k < 8; k++) fp += B->S.fp_ops[k] * fl[k];
  const double ext = n * 2 * 30.0 + 4 * 40.0 + (1 << n) * 40.0;
  if (B->D.fuse) {
    // n = 3 fused pass: the current levels once; per amplitude thread (pair x gluon helicities) the split three-gluon current
    // (2 L3 + V4 + two scalings), the term the two orderings of a pair share (2 light-cone forms, 4 row-slash products, 8 row.col products of
    // 30 flops, 2 folds of 4 amplitudes into 2 sets at 4 flops), per colour ordering 3 / 6 / 12 / 3 of the same, and the u / v rows of both sets
    double lev = 0; for (int k = 0; k < 8; k++) lev += (B->S.fp_ops[k] - B->S.fp_final[k]) * fl[k];
    const double nf = (double)B->S.npair * (double)(1 << (n - 1));
    const double per_thread = 2 * fl[0] + fl[1] + 16.0 + (2 * fl[3] + 4 * fl[2] + 8 * 30.0 + 2 * 2 * 4 * 4.0) + 2.0 * (3 * fl[3] + 6 * fl[2] + 12 * 30.0 + 3 * 2 * 4 * 4.0) + 2 * 4 * 4.0;
    return lev + ((B->D.nsets + 1) / 2) * nf * per_thread + ext;
  }
  const int neval = B->D.poly ? B->D.nnode : B->D.nsets;      // polynomial mode: the currents are evaluated at the node sets only
  // the row-slash products of the full current once per pair instead of once per ordering (share_full_term: n = 5, and n = 4 in FP32 / mixed)
  if (n == 5 || (n == 4 && precision != RWGT_FP64)) fp -= (double)B->S.npair * (double)(1 << (n - 1)) * 2 * fl[2];
  return neval * fp + (B->D.shared_ext ? 1 : B->D.nsets) * ext;
}
// Algorithmic flops of the colour form |L+^T u|^2 + |L-^T v|^2 (a5), all parameter sets: per evaluated helicity (2^(n+1) after
// parity) each of the two reflection blocks (size nh = n!/2) costs nh (nh + 1) / 2 FMAs for the real and for the imaginary part,
// plus 2 nh FMAs for the sum of squares.  They run as mma.m8n8k4 (DMMA) on the FP64 pipe, which DFMA and DMMA share on B200 (include/rwgt_microbench.h, kind 7).
static double bg_tensor_flops_per_event(const BgProcess* B) {
  const int n = B->S.n; const double nh = B->S.npair, nhel = (double)(1 << (n + 1));
  if (B->D.poly) {       // Z = L^T J per node set, then r (r + 1) / 2 cross products instead of r squares
    const double r = B->D.nnode;
    return nhel * 2.0 * (r * 2.0 * (nh * (nh + 1) / 2) + r * (r + 1) / 2 * 2.0 * nh) * 2.0;
  }
  return B->D.nsets * nhel * 2.0 * (2.0 * (nh * (nh + 1) / 2) + 2.0 * nh) * 2.0;     // two reflection blocks of size n!/2
}

static int bg_run(BgProcess* B, int precision, const double* mom, const double* w, const int* idx, double* a, double* b, double* o, long long nev, long long stride, long long ostride, cudaStream_t st) {
  BgDev D = B->D; D.idx = idx; const bool dbl = (precision == RWGT_FP64);
  D.nslot = dbl ? B->nslot64 : B->nslot32;
  if (D.poly) D.poly_stride = (long long)D.nnode * D.nslot * bg_zel(B->S.n);
  long long ngroups = (nev + D.nslot - 1) / D.nslot; int grid = (int)std::min<long long>(ngroups, (long long)B->sm_count * bg_ctas(B->S.n, dbl));
  switch (B->S.n) {
    case 2: bg_launch<2>(precision, grid, B->smem64, B->smem32, st, mom, w, a, b, o, nev, stride, ostride, D); break;
    case 3: bg_launch<3>(precision, grid, B->smem64, B->smem32, st, mom, w, a, b, o, nev, stride, ostride, D); break;
    case 4: bg_launch<4>(precision, grid, B->smem64, B->smem32, st, mom, w, a, b, o, nev, stride, ostride, D); break;
    default: bg_launch<5>(precision, grid, B->smem64, B->smem32, st, mom, w, a, b, o, nev, stride, ostride, D);
  }
  return 0;
}

}  // namespace rwgt
