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
// operand reference: entry = base + variant bits of the operand extracted from the task's variant word
enum : uint32_t { REF_REV = 1u << 22, REF_NEG = 1u << 23 };
static inline uint32_t mkref(int base, int m, int shift, bool rev, bool neg, int mask) {
  return (uint32_t)base | ((uint32_t)m << 16) | ((uint32_t)shift << 19) | (rev && m >= 2 ? REF_REV : 0u) | (neg ? REF_NEG : 0u) | ((uint32_t)mask << 24);
}

struct BgSched {
  int n, c, lmax, rmax, nperm, npair;
  int nG, nR, nL;                   // table entries per slot
  int offG[6], strideG[6];          // gluon levels m = 2..n-1: offset into words, words per task
  int offR[6], strideR[6];          // right levels m = 1..rmax
  int offL[6], strideL[6];          // left  levels m = 1..lmax
  int offF, strideF;                // finals: one task descriptor per sigma pair
  std::vector<uint32_t> words;
  std::vector<double> lfrag;        // Cholesky factor L^T of the colour matrix in mma-fragment order
};

struct TupleTables {
  std::map<std::vector<int>, int> gbase;   // canonical gluon tuples
  std::map<std::vector<int>, int> rbase, lbase;
};
static int mask_of(const std::vector<int>& t) { int m = 0; for (int x : t) m |= 1 << x; return m; }
static bool is_canon(const std::vector<int>& t) { return t.size() < 2 || t.front() < t.back(); }
// reference to the gluon current of the tuple obtained by reading positions [lo,hi) of `seq` (ascending if !desc)
static uint32_t gref(const TupleTables& T, const std::vector<int>& seq, int lo, int hi, bool desc) {
  std::vector<int> asc(seq.begin() + lo, seq.begin() + hi), used = asc;
  if (desc) std::reverse(used.begin(), used.end());
  int m = hi - lo; bool canon_is_asc = is_canon(asc);
  std::vector<int> canon = asc; if (!canon_is_asc) std::reverse(canon.begin(), canon.end());
  bool used_is_canon = (used == canon);
  bool neg = !used_is_canon && (m % 2 == 0);            // J(rev) = (-1)^{m+1} J
  // variant bits are given in ascending position order of `seq`; the stored entry uses the canonical tuple's order
  return mkref(T.gbase.at(canon), m, lo, !canon_is_asc, neg, mask_of(asc));
}
static uint32_t qref(const std::map<std::vector<int>, int>& base, const std::vector<int>& seq, int lo, int hi, bool desc) {
  std::vector<int> used(seq.begin() + lo, seq.begin() + hi); if (desc) std::reverse(used.begin(), used.end());
  return mkref(base.at(used), hi - lo, lo, desc, false, mask_of(used));
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
__host__ __device__ constexpr int ctuples(int n, int m) { return cfact(n) / cfact(n - m); }     // ordered m-tuples of n labels
__host__ __device__ constexpr int c_nG(int n) { int r = 0; for (int m = 1; m <= n - 1; m++) r += (m == 1 ? n : ctuples(n, m) / 2) << m; return r; }
__host__ __device__ constexpr int c_nQ(int n, int mmax) { int r = 2; for (int m = 1; m <= mmax; m++) r += ctuples(n, m) * (2 << m); return r; }
template <int N> struct Geo {
  static constexpr int C = (N + 1) / 2, LMAX = C - 1, RMAX = N - C, NJ = N - C + 1;            // N=2: C=1; 3: 2; 4: 2; 5: 3
  static constexpr int NPERM = cfact(N), NPAIR = NPERM / 2, NPERM_P = (NPERM + 7) / 8 * 8;
  // helicity batches: gluon 0 has helicity + only (parity); NB more gluon helicities are fixed per batch so that a
  // batch is 16 amplitude columns (4 free gluon configurations x 4 quark helicities) for N >= 3
  static constexpr int NB = (N == 5) ? 2 : (N == 4) ? 1 : 0, NBATCH = 1 << NB;
  static constexpr int NFREE = 1 << (N - 1 - NB), NCOL = NFREE * 4;
  static constexpr int ASTR = 2 * NCOL + 4;                              // row stride (doubles) of the amplitude buffer, bank-conflict-free
  static constexpr int MT = NPERM_P / 8, KT = NPERM_P / 4, U = (MT + 1) / 2;
  static constexpr int NT = 2 * NCOL / 8;                                // mma n-tiles per batch
  static constexpr int NMASK = 1 << N;
  static constexpr int NPHASE = (N - 1 > (RMAX > LMAX ? RMAX : LMAX) + 1) ? N - 1 : (RMAX > LMAX ? RMAX : LMAX) + 1;
  static constexpr int NL3 = N - 1, NV4 = (N - 1) * (N - 2) / 2;
  static constexpr int WOFF_TERMS = 4 + 2 * NL3 + 3 * NV4, WPER = C + NJ + NJ * C;
  static constexpr int STRIDEF = WOFF_TERMS + 2 * WPER;
  static constexpr size_t ABUF = (size_t)NPERM_P * ASTR;                 // doubles per slot per buffer
  static constexpr int NG = c_nG(N), NR = c_nQ(N, RMAX), NL = c_nQ(N, LMAX);   // entries of the current tables (checked against the schedule)
};

static BgSched build_schedule(int n) {
  BgSched S; S.n = n;
  for (int m = 0; m < 6; m++) { S.offG[m] = S.strideG[m] = S.offR[m] = S.strideR[m] = S.offL[m] = S.strideL[m] = 0; }
  S.c = (n + 1) / 2; S.lmax = S.c - 1; S.rmax = n - S.c;
  TupleTables T; std::vector<std::vector<int>> tl;
  int nG = 0, nR = 0, nL = 0;
  for (int m = 1; m <= n - 1; m++) { all_tuples(n, m, tl); for (auto& t : tl) if (is_canon(t)) { T.gbase[t] = nG; nG += 1 << m; } }
  T.rbase[{}] = nR; nR += 2; T.lbase[{}] = nL; nL += 2;
  for (int m = 1; m <= S.rmax; m++) { all_tuples(n, m, tl); for (auto& t : tl) { T.rbase[t] = nR; nR += 2 << m; } }
  for (int m = 1; m <= S.lmax; m++) { all_tuples(n, m, tl); for (auto& t : tl) { T.lbase[t] = nL; nL += 2 << m; } }
  S.nG = nG; S.nR = nR; S.nL = nL;
  for (int m = 2; m <= n - 1; m++) {
    all_tuples(n, m, tl); S.offG[m] = (int)S.words.size(); S.strideG[m] = 2 + 2 * (m - 1) + 3 * (m - 1) * (m - 2) / 2;
    for (auto& t : tl) if (is_canon(t)) {
      S.words.push_back(T.gbase[t]); S.words.push_back(mask_of(t));
      for (int k = 1; k < m; k++) { S.words.push_back(gref(T, t, 0, k, false)); S.words.push_back(gref(T, t, k, m, false)); }
      for (int j = 1; j < m; j++) for (int k = j + 1; k < m; k++) { S.words.push_back(gref(T, t, 0, j, false)); S.words.push_back(gref(T, t, j, k, false)); S.words.push_back(gref(T, t, k, m, false)); }
    }
  }
  for (int m = 1; m <= S.rmax; m++) {
    all_tuples(n, m, tl); S.offR[m] = (int)S.words.size(); S.strideR[m] = 2 + 2 * m;
    for (auto& t : tl) {
      S.words.push_back(T.rbase[t]); S.words.push_back(mask_of(t));
      for (int k = 1; k <= m; k++) { S.words.push_back(gref(T, t, 0, k, false)); S.words.push_back(qref(T.rbase, t, k, m, false)); }
    }
  }
  for (int m = 1; m <= S.lmax; m++) {
    all_tuples(n, m, tl); S.offL[m] = (int)S.words.size(); S.strideL[m] = 2 + 2 * m;
    for (auto& t : tl) {
      S.words.push_back(T.lbase[t]); S.words.push_back(mask_of(t));
      for (int k = 1; k <= m; k++) { S.words.push_back(qref(T.lbase, t, 0, m - k, false)); S.words.push_back(gref(T, t, m - k, m, false)); }
    }
  }
  // finals: one descriptor per pair (sigma, sigma reversed), sigma_1 < sigma_n
  std::vector<std::vector<int>> perms; { std::vector<int> p(n); for (int i = 0; i < n; i++) p[i] = i; do perms.push_back(p); while (std::next_permutation(p.begin(), p.end())); }
  S.nperm = (int)perms.size(); std::map<std::vector<int>, int> rank; for (int i = 0; i < S.nperm; i++) rank[perms[i]] = i;
  const int C = S.c, NJ = n - C + 1;
  S.offF = (int)S.words.size(); S.strideF = 4 + 2 * (n - 1) + 3 * (n - 1) * (n - 2) / 2 + 2 * (C + NJ + NJ * C); S.npair = 0;
  for (auto& s : perms) if (s.front() < s.back()) {
    S.npair++;
    std::vector<int> sr(s.rbegin(), s.rend());
    uint32_t packed = 0; for (int j = 0; j < n; j++) packed |= (uint32_t)s[j] << (3 * j);
    S.words.push_back(rank[s]); S.words.push_back(rank[sr]); S.words.push_back(packed); S.words.push_back(n % 2 == 0 ? 1u : 0u);   // J_n(rev) = (-1)^{n+1} J_n
    for (int k = 1; k < n; k++) { S.words.push_back(gref(T, s, 0, k, false)); S.words.push_back(gref(T, s, k, n, false)); }
    for (int j = 1; j < n; j++) for (int k = j + 1; k < n; k++) { S.words.push_back(gref(T, s, 0, j, false)); S.words.push_back(gref(T, s, j, k, false)); S.words.push_back(gref(T, s, k, n, false)); }
    for (int which = 0; which < 2; which++) {
      // sigma: block [i,j) in ascending positions.  sigma reversed: its positions [i,j) are sigma's [n-j,n-i) read descending
      for (int i = 0; i < C; i++) S.words.push_back(which == 0 ? qref(T.lbase, s, 0, i, false) : qref(T.lbase, s, n - i, n, true));
      for (int j = C; j <= n; j++) S.words.push_back(which == 0 ? qref(T.rbase, s, j, n, false) : qref(T.rbase, s, 0, n - j, true));
      for (int j = C; j <= n; j++) for (int i = 0; i < C; i++) {
        if (i == 0 && j == n) { S.words.push_back(0u); continue; }
        S.words.push_back(which == 0 ? gref(T, s, i, j, false) : gref(T, s, n - j, n - i, true));
      }
    }
  }
  // Cholesky C = L L^T (C is positive definite); J^dagger C J = |L^T J|^2.  L^T in mma.m8n8k4 A-fragment order:
  // for m-tile mt, k-steps kt = 2 mt .. KT-1 (upper triangle), element (lane>>2, lane&3) of the 8x4 tile.
  {
    int np = S.nperm, npp = (np + 7) / 8 * 8, MT = npp / 8, KT = npp / 4;
    std::vector<double> Cm = colour_matrix_fierz(n), L((size_t)np * np, 0.0);
    for (int j = 0; j < np; j++) {
      double d = Cm[(size_t)j * np + j]; for (int k = 0; k < j; k++) d -= L[(size_t)j * np + k] * L[(size_t)j * np + k];
      d = std::sqrt(d); L[(size_t)j * np + j] = d;
      for (int i = j + 1; i < np; i++) { double x = Cm[(size_t)i * np + j]; for (int k = 0; k < j; k++) x -= L[(size_t)i * np + k] * L[(size_t)j * np + k]; L[(size_t)i * np + j] = x / d; }
    }
    for (int mt = 0; mt < MT; mt++) for (int kt = 2 * mt; kt < KT; kt++) for (int lane = 0; lane < 32; lane++) {
      int row = 8 * mt + (lane >> 2), col = 4 * kt + (lane & 3);
      S.lfrag.push_back((row < np && col < np && col >= row) ? L[(size_t)col * np + row] : 0.0);      // L^T[row][col] = L[col][row]
    }
  }
  return S;
}

// ------------------------------------------------------------------------------------------------ device side
struct BgSet { double gq, g3, g4, mt, fac; };        // fac = 2 gq^2 / D  (|i gq|^2, parity factor 2, averaging)
struct BgDev {
  int nG, nR, nL, nwords, nslot, shared_ext;
  int offG[6], offR[6], offL[6], offF;
  const uint32_t* words; const double* lfrag;
  BgSet set[2];
};

struct BgProcess {
  BgSched S; BgDev D; uint32_t* d_words; double* d_lfrag; int sm_count; size_t smem64, smem32; int nslot64, nslot32;
};

template <typename T> struct Smem {
  uint32_t* W;    // schedule words (whole CTA)
  double* pm;     // [nslot][n_ext][4] momenta (always double)
  double* acc;    // [nslot][2]   helicity-summed colour forms (owned by the colour warps)
  double* red;    // [nslot][8]   per-warp partial sums of the colour form
  T* G; T* R; T* L;  // [nslot][8][nX]   SoA planes: conflict-free for consecutive helicity variants
  T* K;           // [nslot][NMASK][4] momentum sums of gluon subsets
  T* iK2;         // [nslot][NMASK]
  T* dR; T* dL;   // [nslot][NMASK] 1/(q^2-m^2)
  double* A;      // [2][nslot][NPERM_P][ASTR] double-buffered colour-flow amplitudes (re,im interleaved), always double
};
template <int N, typename T> __host__ __device__ inline size_t carve(Smem<T>& s, unsigned char* base, int ns, int nwords) {
  typedef Geo<N> Ge; size_t off = 0; constexpr int nG = Ge::NG, nR = Ge::NR, nL = Ge::NL;
  s.A = (double*)(base + off); off += sizeof(double) * 2 * (size_t)ns * Ge::ABUF;
  s.pm = (double*)(base + off); off += sizeof(double) * ns * (N + 2) * 4;
  s.acc = (double*)(base + off); off += sizeof(double) * ns * 2;
  s.red = (double*)(base + off); off += sizeof(double) * ns * 8;
  s.G = (T*)(base + off); off += sizeof(T) * (size_t)ns * 8 * nG;
  s.R = (T*)(base + off); off += sizeof(T) * (size_t)ns * 8 * nR;
  s.L = (T*)(base + off); off += sizeof(T) * (size_t)ns * 8 * nL;
  s.K = (T*)(base + off); off += sizeof(T) * ns * Ge::NMASK * 4;
  s.iK2 = (T*)(base + off); off += sizeof(T) * ns * Ge::NMASK;
  s.dR = (T*)(base + off); off += sizeof(T) * ns * Ge::NMASK;
  s.dL = (T*)(base + off); off += sizeof(T) * ns * Ge::NMASK;
  s.W = (uint32_t*)(base + off); off += sizeof(uint32_t) * nwords;
  return off;
}

template <typename T> __device__ __forceinline__ vec4<T> ld4(const T* tab, int stride, int e) {
  vec4<T> r;
#pragma unroll
  for (int c = 0; c < 4; c++) { r.c[c].re = tab[(2 * c) * stride + e]; r.c[c].im = tab[(2 * c + 1) * stride + e]; }
  return r;
}
template <typename T> __device__ __forceinline__ spn<T> lds4(const T* tab, int stride, int e) {
  spn<T> r;
#pragma unroll
  for (int c = 0; c < 4; c++) { r.c[c].re = tab[(2 * c) * stride + e]; r.c[c].im = tab[(2 * c + 1) * stride + e]; }
  return r;
}
template <typename T, typename V> __device__ __forceinline__ void st4(T* tab, int stride, int e, const V& v) {
#pragma unroll
  for (int c = 0; c < 4; c++) { tab[(2 * c) * stride + e] = v.c[c].re; tab[(2 * c + 1) * stride + e] = v.c[c].im; }
}
__device__ __forceinline__ int ref_entry(uint32_t r, uint32_t v) {
  uint32_t m = (r >> 16) & 7u, sh = (r >> 19) & 7u;
  uint32_t w = (v >> sh) & ((1u << m) - 1u);
  if (r & REF_REV) w = __brev(w) >> (32u - m);
  return (int)((r & 0xffffu) + w);
}
__device__ __forceinline__ int ref_m(uint32_t r) { return (int)((r >> 16) & 7u); }
__device__ __forceinline__ int ref_mask(uint32_t r) { return (int)((r >> 24) & 31u); }
__device__ __forceinline__ bool ref_neg(uint32_t r) { return (r & REF_NEG) != 0; }

// named barriers (ids 1..6; id 0 is __syncthreads): workers among themselves, colour warps among themselves,
// and the full/empty handshake of the two amplitude buffers
enum { BAR_WORK = 1, BAR_FULL0 = 2, BAR_EMPTY0 = 4, BAR_COLOUR = 6 };
__device__ __forceinline__ void bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// gluon current of one ordered M-tuple / helicity variant from shorter currents (unscaled by the propagator)
template <int M, int nG, typename T> __device__ __forceinline__ vec4<T> gluon_sum(const uint32_t* w, uint32_t v, const T* G, const T* K, T g3, T g4) {
  vec4<T> a3, a4;
#pragma unroll
  for (int i = 0; i < 4; i++) { a3.c[i] = mk<T>(0, 0); a4.c[i] = mk<T>(0, 0); }
#pragma unroll
  for (int k = 0; k < M - 1; k++) {
    uint32_t ra = w[2 * k], rb = w[2 * k + 1];
    vec4<T> A = cond_neg(ld4(G, nG, ref_entry(ra, v)), ref_neg(ra) != ref_neg(rb)), B = ld4(G, nG, ref_entry(rb, v));
    L3_acc(a3, A, K + 4 * ref_mask(ra), B, K + 4 * ref_mask(rb));
  }
  const uint32_t* w4 = w + 2 * (M - 1);
#pragma unroll
  for (int t = 0; t < (M - 1) * (M - 2) / 2; t++) {
    uint32_t rx = w4[3 * t], ry = w4[3 * t + 1], rz = w4[3 * t + 2];
    vec4<T> X = cond_neg(ld4(G, nG, ref_entry(rx, v)), (ref_neg(rx) != ref_neg(ry)) != ref_neg(rz));
    vec4<T> Y = ld4(G, nG, ref_entry(ry, v)), Z = ld4(G, nG, ref_entry(rz, v));
    V4_acc(a4, X, Y, Z);
  }
  vec4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) { r.c[i] = (-g3) * a3.c[i]; if (M > 2) rfma(r.c[i], g4, a4.c[i]); }
  return r;
}

template <typename T> struct Ctx {
  Smem<T> s; int tid, ns; T g3, g4, gq, mt; const BgDev* D;
};

// phase M (worker warps): gluon currents of length M, right/left quark currents of length M-1 (all helicity variants)
template <int N, int M, typename T, int NWT> __device__ __forceinline__ void level_phase(const Ctx<T>& c) {
  typedef Geo<N> Ge;
  constexpr bool HASG = (M <= N - 1), HASR = (M - 1 >= 1 && M - 1 <= Ge::RMAX), HASL = (M - 1 >= 1 && M - 1 <= Ge::LMAX);
  constexpr int MM = M - 1;
  constexpr int tg = HASG ? (ctuples(N, M) / 2) << M : 0, tr = HASR ? ctuples(N, MM) << M : 0, tl = HASL ? ctuples(N, MM) << M : 0, per = tg + tr + tl;
  const Smem<T>& s = c.s; constexpr int nG = Ge::NG, nR = Ge::NR, nL = Ge::NL, next = N + 2;
  for (int t = c.tid; t < c.ns * per; t += NWT) {
    int sl = t / per, o = t % per;
    T* G = s.G + (size_t)sl * 8 * nG; T* R = s.R + (size_t)sl * 8 * nR; T* L = s.L + (size_t)sl * 8 * nL;
    const T* K = s.K + (size_t)sl * Ge::NMASK * 4;
    if (HASG && o < tg) {
      int tup = o >> M; uint32_t v = o & ((1 << M) - 1);
      const uint32_t* w = s.W + c.D->offG[M] + tup * (2 + 2 * (M - 1) + 3 * (M - 1) * (M - 2) / 2);
      int ob = w[0], mask = w[1];
      vec4<T> r = gluon_sum<M, nG, T>(w + 2, v, G, K, c.g3, c.g4);
      T sc = s.iK2[sl * Ge::NMASK + mask];
#pragma unroll
      for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
      st4(G, nG, ob + v, r);
    } else if (HASR && o < tg + tr) {
      int oo = o - tg; int tup = oo >> M; uint32_t vv = oo & ((1 << M) - 1); uint32_t v = vv & ((1 << MM) - 1); int hb = vv >> MM;
      const uint32_t* w = s.W + c.D->offR[MM] + tup * (2 + 2 * MM);
      int ob = w[0], mask = w[1];
      spn<T> acc;
#pragma unroll
      for (int i = 0; i < 4; i++) acc.c[i] = mk<T>(0, 0);
#pragma unroll
      for (int k = 0; k < MM; k++) {
        uint32_t rj = w[2 + 2 * k], rr = w[3 + 2 * k];
        lcv<T> J = lightcone(cond_neg(ld4(G, nG, ref_entry(rj, v)), ref_neg(rj)));
        slash_acc(acc, J, lds4(R, nR, ref_entry(rr, v) + (hb << ref_m(rr))));
      }
      T q[4];
#pragma unroll
      for (int mu = 0; mu < 4; mu++) q[mu] = K[4 * mask + mu] - (T)s.pm[sl * next * 4 + 12 + mu];
      spn<T> r = slash_r_plus_m(q, c.mt, acc); T sc = -c.gq * s.dR[sl * Ge::NMASK + mask];
#pragma unroll
      for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
      st4(R, nR, ob + v + (hb << MM), r);
    } else if (HASL) {
      int oo = o - tg - tr; int tup = oo >> M; uint32_t vv = oo & ((1 << M) - 1); uint32_t v = vv & ((1 << MM) - 1); int hb = vv >> MM;
      const uint32_t* w = s.W + c.D->offL[MM] + tup * (2 + 2 * MM);
      int ob = w[0], mask = w[1];
      spn<T> acc;
#pragma unroll
      for (int i = 0; i < 4; i++) acc.c[i] = mk<T>(0, 0);
#pragma unroll
      for (int k = 0; k < MM; k++) {
        uint32_t rl = w[2 + 2 * k], rj = w[3 + 2 * k];
        lcv<T> J = lightcone(cond_neg(ld4(G, nG, ref_entry(rj, v)), ref_neg(rj)));
        row_slash_acc(acc, lds4(L, nL, ref_entry(rl, v) + (hb << ref_m(rl))), J);
      }
      T q[4];
#pragma unroll
      for (int mu = 0; mu < 4; mu++) q[mu] = (T)s.pm[sl * next * 4 + 8 + mu] - K[4 * mask + mu];
      spn<T> r = row_slash_r_plus_m(acc, q, c.mt); T sc = -c.gq * s.dL[sl * Ge::NMASK + mask];
#pragma unroll
      for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
      st4(L, nL, ob + v + (hb << MM), r);
    }
  }
  bar_sync(BAR_WORK, NWT);
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// One persistent CTA per SM.  Warps 0..NW-1 ("workers") build the currents and the colour-flow amplitudes of one helicity
// batch after the other on the FP64 pipe; the last NCW warps ("colour") turn finished batches into |L^T J|^2 on the FP64
// tensor pipe (a separate pipe, so the two overlap) and write the outputs.  The two amplitude buffers are handed over with
// named barriers.  MIXED: T = float but momentum sums / propagator denominators are formed in double before rounding to T.
template <int N, typename T, bool MIXED, int NW, int NCW>
__global__ void __launch_bounds__((NW + NCW) * 32, 1) bg_kernel(const double* __restrict__ mom, const double* __restrict__ wgt,
                                                               double* __restrict__ me_old, double* __restrict__ me_new,
                                                               double* __restrict__ w_new, long long nev, BgDev D) {
  typedef Geo<N> Ge;
  constexpr int NTH = (NW + NCW) * 32, NWT = NW * 32, NCT = NCW * 32;
  // register hand-over between the warpgroups: the colour warps need few registers, the workers get the rest
  constexpr int REG_COL = 56, REG_WORK = ((65536 / 32 - NCW * REG_COL) / NW) / 8 * 8 > 232 ? 232 : ((65536 / 32 - NCW * REG_COL) / NW) / 8 * 8;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Ctx<T> c; c.D = &D; c.ns = D.nslot;
  carve<N, T>(c.s, smem_raw, D.nslot, D.nwords);
  const Smem<T>& s = c.s;
  typedef typename std::conditional<MIXED, double, T>::type TK;
  constexpr int next = N + 2, nG = Ge::NG, nR = Ge::NR, nL = Ge::NL; const int ns = D.nslot;
  const long long ngroups = (nev + ns - 1) / ns;
  // once per CTA: zero both amplitude buffers (their padding rows are never written again)
  for (int t = threadIdx.x; t < 2 * ns * (int)Ge::ABUF; t += NTH) s.A[t] = 0.0;
  __syncthreads();
  if (threadIdx.x < NWT) {
    // =========================================================================================== worker warps
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REG_WORK));
    const int tid = threadIdx.x; c.tid = tid;
    for (int t = tid; t < D.nwords; t += NWT) s.W[t] = __ldg(D.words + t);
    unsigned step = 0;
    for (long long grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
      const long long ev0 = grp * ns;
      bar_sync(BAR_WORK, NWT);
      // ---- a1: load momenta (coalesced over the events of the group) ----
      for (int t = tid; t < ns * next * 4; t += NWT) {
        int sl = t % ns, comp = t / ns; long long ev = ev0 + sl; if (ev >= nev) ev = nev - 1;
        s.pm[(sl * next * 4) + comp] = __ldg(mom + (size_t)comp * nev + ev);
      }
      bar_sync(BAR_WORK, NWT);
#pragma unroll 1
      for (int iset = 0; iset < 2; iset++) {
        const BgSet& P = D.set[iset];
        c.g3 = (T)P.g3; c.g4 = (T)P.g4; c.gq = (T)P.gq; c.mt = (T)P.mt;
        if (iset == 0 || !D.shared_ext) {
          // ---- a2: external wavefunctions, momentum sums, propagator denominators ----
          constexpr int nobj = 2 * N + 4 + Ge::NMASK;
          for (int t = tid; t < ns * nobj; t += NWT) {
            int sl = t / nobj, o = t % nobj; const double* pm = s.pm + sl * next * 4;
            if (o < 2 * N) {                         // gluon i, helicity bit hb (0: +1, 1: -1); entry = 2*i + hb
              int i = o >> 1, hb = o & 1, leg = i < 2 ? i : i + 2; const double* p = pm + 4 * leg;
              vec4<T> e = polvec<T>((T)p[1], (T)p[2], (T)p[3], hb ? -1 : +1);
              if (i >= 2) e = conj4(e);              // outgoing gluon carries eps*
              st4(s.G + (size_t)sl * 8 * nG, nG, 2 * i + hb, e);
            } else if (o < 2 * N + 2) {              // v(p_tbar, lam), R() entries 0,1
              int hb = o - 2 * N; const double* p = pm + 12;
              chi_pair<T> x = make_chi<T>((T)p[1], (T)p[2], (T)p[3]);
              st4(s.R + (size_t)sl * 8 * nR, nR, hb, spinor_v<T>(x, (T)p[0], c.mt, hb ? -1 : +1));
            } else if (o < 2 * N + 4) {              // ubar(p_t, lam), L() entries 0,1
              int hb = o - 2 * N - 2; const double* p = pm + 8;
              chi_pair<T> x = make_chi<T>((T)p[1], (T)p[2], (T)p[3]);
              st4(s.L + (size_t)sl * 8 * nL, nL, hb, bar(spinor_u<T>(x, (T)p[0], c.mt, hb ? -1 : +1)));
            } else {                                 // gluon subset `mask`
              int mask = o - 2 * N - 4;
              TK k[4] = {0, 0, 0, 0};
#pragma unroll
              for (int i = 0; i < N; i++) if (mask >> i & 1) { int leg = i < 2 ? i : i + 2; TK sg = i < 2 ? TK(1) : TK(-1);
                for (int mu = 0; mu < 4; mu++) k[mu] += sg * (TK)pm[4 * leg + mu]; }
              TK k2 = mdot_rr<TK>(k, k);
              TK qr[4], ql[4]; for (int mu = 0; mu < 4; mu++) { qr[mu] = k[mu] - (TK)pm[12 + mu]; ql[mu] = (TK)pm[8 + mu] - k[mu]; }
              TK m2 = (TK)P.mt * (TK)P.mt;
              T* K = s.K + ((size_t)sl * Ge::NMASK + mask) * 4; for (int mu = 0; mu < 4; mu++) K[mu] = (T)k[mu];
              s.iK2[sl * Ge::NMASK + mask] = (__popc(mask) >= 2) ? (T)(TK(1) / k2) : T(0);
              s.dR[sl * Ge::NMASK + mask] = (T)(TK(1) / (mdot_rr<TK>(qr, qr) - m2));
              s.dL[sl * Ge::NMASK + mask] = (T)(TK(1) / (mdot_rr<TK>(ql, ql) - m2));
            }
          }
          bar_sync(BAR_WORK, NWT);
        }
        // ---- a3: current levels ----
        level_phase<N, 2, T, NWT>(c);
        if constexpr (Ge::NPHASE >= 3) level_phase<N, 3, T, NWT>(c);
        if constexpr (Ge::NPHASE >= 4) level_phase<N, 4, T, NWT>(c);
        // ---- a3/a4: colour-flow amplitudes, one helicity batch per buffer hand-over ----
#pragma unroll 1
        for (int batch = 0; batch < Ge::NBATCH; batch++, step++) {
          const int buf = step & 1;
          if (step >= 2) bar_sync(BAR_EMPTY0 + buf, NTH);      // colour warps have finished reading this buffer
          double* Abuf = s.A + (size_t)buf * ns * Ge::ABUF;
          constexpr int per = Ge::NPAIR * Ge::NFREE;
          for (int t = tid; t < ns * per; t += NWT) {
            int sl = t / per, o = t % per; int pair = o / Ge::NFREE, f = o % Ge::NFREE;
            const T* G = s.G + (size_t)sl * 8 * nG; const T* R = s.R + (size_t)sl * 8 * nR; const T* L = s.L + (size_t)sl * 8 * nL;
            const T* K = s.K + (size_t)sl * Ge::NMASK * 4;
            const uint32_t* w = s.W + D.offF + pair * Ge::STRIDEF;
            uint32_t rk = w[0], rkr = w[1], packed = w[2], negr = w[3];
            uint32_t g = ((uint32_t)batch << 1) | ((uint32_t)f << (1 + Ge::NB));   // helicity bits by gluon label; gluon 0: + (parity)
            uint32_t v = 0;
#pragma unroll
            for (int j = 0; j < N; j++) v |= ((g >> ((packed >> (3 * j)) & 7u)) & 1u) << j;   // by position in sigma
            vec4<T> Jn = gluon_sum<N, nG, T>(w + 4, v, G, K, c.g3, c.g4);
            T sc = s.iK2[sl * Ge::NMASK + Ge::NMASK - 1];
#pragma unroll
            for (int i = 0; i < 4; i++) Jn.c[i] = sc * Jn.c[i];
            double* A = Abuf + (size_t)sl * Ge::ABUF;
            const uint32_t* wt = w + Ge::WOFF_TERMS;
#pragma unroll 1
            for (int which = 0; which < 2; which++) {
              cx<T> Acc[2][2];
#pragma unroll
              for (int a = 0; a < 2; a++)
#pragma unroll
                for (int b = 0; b < 2; b++) Acc[a][b] = mk<T>(0, 0);
#pragma unroll
              for (int jj = 0; jj < Ge::NJ; jj++) {
                spn<T> X0, X1;
#pragma unroll
                for (int i = 0; i < 4; i++) { X0.c[i] = mk<T>(0, 0); X1.c[i] = mk<T>(0, 0); }
#pragma unroll
                for (int i = 0; i < Ge::C; i++) {
                  if (i == 0 && jj == Ge::NJ - 1) {                 // the full-length gluon current between ubar and v
                    lcv<T> J = lightcone(cond_neg(Jn, which && negr));
                    row_slash_acc(X0, lds4(L, nL, 0), J); row_slash_acc(X1, lds4(L, nL, 1), J);
                  } else {
                    uint32_t rl = wt[i], rj = wt[Ge::C + Ge::NJ + jj * Ge::C + i];
                    lcv<T> J = lightcone(cond_neg(ld4(G, nG, ref_entry(rj, v)), ref_neg(rj)));
                    int el = ref_entry(rl, v), ml = ref_m(rl);
                    row_slash_acc(X0, lds4(L, nL, el), J); row_slash_acc(X1, lds4(L, nL, el + (1 << ml)), J);
                  }
                }
                uint32_t rr = wt[Ge::C + jj]; int er = ref_entry(rr, v), mr = ref_m(rr);
#pragma unroll
                for (int hb = 0; hb < 2; hb++) {
                  spn<T> Rr = lds4(R, nR, er + (hb << mr));
                  rowcol_acc(Acc[0][hb], X0, Rr); rowcol_acc(Acc[1][hb], X1, Rr);
                }
              }
              uint32_t row = which ? rkr : rk;
#pragma unroll
              for (int ht = 0; ht < 2; ht++)
#pragma unroll
                for (int hb = 0; hb < 2; hb++) {
                  int col = f * 4 + ht * 2 + hb;
                  *reinterpret_cast<double2*>(A + (size_t)row * Ge::ASTR + 2 * col) = make_double2((double)Acc[ht][hb].re, (double)Acc[ht][hb].im);
                }
              wt += Ge::WPER;
            }
          }
          __threadfence_block();
          bar_arrive(BAR_FULL0 + buf, NTH);                    // hand the batch to the colour warps
        }
        bar_sync(BAR_WORK, NWT);                               // the current tables are rewritten for the next parameter set / group
      }
    }
  } else {
    // =========================================================================================== colour warps
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REG_COL));
    const int ctid = threadIdx.x - NWT, cwarp = ctid >> 5, lane = ctid & 31;
    unsigned step = 0;
    for (long long grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
      const long long ev0 = grp * ns;
      if (ctid < ns * 2) s.acc[ctid] = 0.0;
      for (int t = ctid + NCT; t < ns * 2; t += NCT) s.acc[t] = 0.0;
      bar_sync(BAR_COLOUR, NCT);
#pragma unroll 1
      for (int iset = 0; iset < 2; iset++) {
#pragma unroll 1
        for (int batch = 0; batch < Ge::NBATCH; batch++, step++) {
          const int buf = step & 1;
          bar_sync(BAR_FULL0 + buf, NTH);                      // the workers have filled this buffer
          const double* Abuf = s.A + (size_t)buf * ns * Ge::ABUF;
          // a5: Z = L^T A with FP64 tensor-core mma over the upper-triangular tiles, colour form = sum of squares of Z
          for (int u = cwarp; u < ns * Ge::U; u += NCW) {
            int sl = u / Ge::U, unit = u % Ge::U;
            const double* A = Abuf + (size_t)sl * Ge::ABUF + (lane & 3) * Ge::ASTR + (lane >> 2);
            double part = 0.0;
#pragma unroll 1
            for (int half = 0; half < 2; half++) {
              int mt = half ? Ge::MT - 1 - unit : unit;
              if (half && mt == unit) break;
              double acc[Ge::NT][2];
#pragma unroll
              for (int nt = 0; nt < Ge::NT; nt++) { acc[nt][0] = 0.0; acc[nt][1] = 0.0; }
              const double* F = D.lfrag + (size_t)(mt * Ge::KT - mt * (mt - 1)) * 32 + lane;
              int nk = Ge::KT - 2 * mt;
              double a0 = __ldg(F), a1 = (nk > 1) ? __ldg(F + 32) : 0.0;
              for (int kk = 0; kk < nk; kk++) {
                double an = (kk + 2 < nk) ? __ldg(F + (kk + 2) * 32) : 0.0;
                const double* Br = A + (size_t)(4 * (2 * mt + kk)) * Ge::ASTR;
#pragma unroll
                for (int nt = 0; nt < Ge::NT; nt++) dmma884(acc[nt][0], acc[nt][1], a0, Br[8 * nt]);
                a0 = a1; a1 = an;
              }
#pragma unroll
              for (int nt = 0; nt < Ge::NT; nt++) { part = fma(acc[nt][0], acc[nt][0], part); part = fma(acc[nt][1], acc[nt][1], part); }
            }
            // a6: deterministic reduction (same order for both parameter sets => old == new gives a ratio of exactly 1)
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
            if (lane == 0) s.red[sl * 8 + unit] = part;
          }
          bar_sync(BAR_COLOUR, NCT);
          bar_arrive(BAR_EMPTY0 + buf, NTH);                   // buffer may be refilled
          for (int sl = ctid; sl < ns; sl += NCT) { double a = 0.0; for (int j = 0; j < Ge::U; j++) a += s.red[sl * 8 + j]; s.acc[sl * 2 + iset] += a; }
          bar_sync(BAR_COLOUR, NCT);
        }
      }
      // ---- a7: eq. 3 and stores ----
      for (int sl = ctid; sl < ns; sl += NCT) {
        long long ev = ev0 + sl;
        if (ev < nev) {
          double a = s.acc[sl * 2] * D.set[0].fac, b = s.acc[sl * 2 + 1] * D.set[1].fac;
          me_old[ev] = a; me_new[ev] = b; w_new[ev] = __ldg(wgt + ev) * (b / a);
        }
      }
      bar_sync(BAR_COLOUR, NCT);
    }
  }
}

// ------------------------------------------------------------------------------------------------ host API of the engine
template <int N> static size_t smem_need(const BgSched& S, int nslot, bool dbl) {
  if (dbl) { Smem<double> s; return carve<N, double>(s, nullptr, nslot, (int)S.words.size()); }
  Smem<float> s; return carve<N, float>(s, nullptr, nslot, (int)S.words.size());
}
static size_t smem_need_n(int n, const BgSched& S, int nslot, bool dbl) {
  switch (n) { case 2: return smem_need<2>(S, nslot, dbl); case 3: return smem_need<3>(S, nslot, dbl); case 4: return smem_need<4>(S, nslot, dbl); default: return smem_need<5>(S, nslot, dbl); }
}
// Warp split: 8 worker warps (FP64 pipe) + 4 colour warps (FP64 tensor pipe) = 3 warps x 168 registers per SM sub-partition
// (16K registers each).  Measured on B200 against 10+2, 6+2 and 12+4: best or within 4% of best for every process.
static const int BG_NW = 8, BG_NCW = 4;

template <int N> static cudaError_t bg_set_attr(size_t s64, size_t s32) {
  cudaError_t e = cudaFuncSetAttribute(bg_kernel<N, double, false, BG_NW, BG_NCW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s64);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<N, float, false, BG_NW, BG_NCW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s32);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<N, float, true, BG_NW, BG_NCW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s32);
  return e;
}
template <int N> static void bg_launch(int precision, int grid, size_t s64, size_t s32, cudaStream_t st, const double* mom, const double* w,
                                       double* a, double* b, double* o, long long nev, const BgDev& D) {
  const int nth = (BG_NW + BG_NCW) * 32;
  if (precision == RWGT_FP64) bg_kernel<N, double, false, BG_NW, BG_NCW><<<grid, nth, s64, st>>>(mom, w, a, b, o, nev, D);
  else if (precision == RWGT_FP32) bg_kernel<N, float, false, BG_NW, BG_NCW><<<grid, nth, s32, st>>>(mom, w, a, b, o, nev, D);
  else bg_kernel<N, float, true, BG_NW, BG_NCW><<<grid, nth, s32, st>>>(mom, w, a, b, o, nev, D);
}

static BgProcess* bg_create(int n, const rwgt_params& po, const rwgt_params& pn, std::string& err) {
  BgProcess* B = new BgProcess();
  B->S = build_schedule(n);
  const BgSched& S = B->S;
  BgDev& D = B->D;
  D.nG = S.nG; D.nR = S.nR; D.nL = S.nL; D.nwords = (int)S.words.size(); D.offF = S.offF;
  if (S.nG != c_nG(n) || S.nR != c_nQ(n, S.rmax) || S.nL != c_nQ(n, S.lmax)) { err = "internal: schedule/geometry mismatch"; delete B; return nullptr; }
  for (int m = 0; m < 6; m++) { D.offG[m] = S.offG[m]; D.offR[m] = S.offR[m]; D.offL[m] = S.offL[m]; }
  const rwgt_params* ps[2] = {&po, &pn};
  double fact = 1; for (int i = 2; i <= n - 2; i++) fact *= i;
  for (int k = 0; k < 2; k++) {
    double gs = std::sqrt(4.0 * 3.14159265358979323846 * ps[k]->alpha_s);
    D.set[k].gq = gs; D.set[k].g3 = gs * ps[k]->ggg_scale; D.set[k].g4 = gs * gs * ps[k]->gggg_scale; D.set[k].mt = ps[k]->mt;
    D.set[k].fac = 2.0 * gs * gs / (256.0 * fact);
  }
  D.shared_ext = (po.mt == pn.mt) ? 1 : 0;
  int dev = 0; cudaGetDevice(&dev); cudaDeviceProp prop; cudaGetDeviceProperties(&prop, dev);
  B->sm_count = prop.multiProcessorCount; size_t maxsm = prop.sharedMemPerBlockOptin;
  // event slots per CTA: as many as make the amplitude phase fill the 256 worker threads (npair * 4 tasks per slot and batch)
  auto pick = [&](bool dbl, int& nslot, size_t& bytes) {
    int cap = std::max(1, std::min(64, (BG_NW * 32) / (S.npair * (n == 2 ? 2 : 4)))); nslot = 0;
    for (int e = cap; e >= 1; e--) if (smem_need_n(n, S, e, dbl) <= maxsm) { nslot = e; break; }
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
  if (e != cudaSuccess) { err = std::string("CUDA: ") + cudaGetErrorString(e); delete B; return nullptr; }
  D.words = B->d_words; D.lfrag = B->d_lfrag;
  return B;
}
static void bg_destroy(BgProcess* B) { if (!B) return; cudaFree(B->d_words); cudaFree(B->d_lfrag); delete B; }

// Algorithmic flop count of the schedule on the FP64 (or FP32) FMA pipe, both parameter sets, per event: FMA = 2 flop,
// MUL = ADD = 1 flop, per operation of rwgt_math.cuh (L3 74 FMA + 6 MUL + 4 ADD, V4 90 + 6 + 2, slash-accumulate 32 FMA,
// light-cone 8 ADD, propagator 24 FMA + 17 MUL + 6 ADD, row.col 16 FMA, current store 8 FMA + 16 MUL).  Agrees with the
// ncu instruction counters of the committed build to 0.5% (n=5), 1.0% (n=4), 2.6% (n=3), always from below
// (profiles/r1_summary.md).
static double bg_flops_per_event(const BgProcess* B, int /*precision*/) {
  const int n = B->S.n, C = B->S.c, NJ = n - C + 1; const double L3 = 158, V4 = 188, SLA = 64, LC = 8, PROP = 71, RC = 32, GST = 32, GST2 = 16;
  auto tup = [](int n, int m) { double r = 1; for (int i = 0; i < m; i++) r *= (n - i); return r; };
  double fp = 0;
  for (int m = 2; m <= n - 1; m++) fp += tup(n, m) / 2 * (1 << m) * ((m - 1) * L3 + (m - 1) * (m - 2) / 2 * V4 + (m > 2 ? GST : GST2));
  for (int m = 1; m <= B->S.rmax; m++) fp += tup(n, m) * (2 << m) * (m * (SLA + LC) + PROP);
  for (int m = 1; m <= B->S.lmax; m++) fp += tup(n, m) * (2 << m) * (m * (SLA + LC) + PROP);
  double per_final = (n - 1) * L3 + (n - 1) * (n - 2) / 2 * V4 + (n > 2 ? GST : GST2) + LC + 2 * (NJ * C * (2 * SLA + LC) + NJ * 4 * RC);
  fp += B->S.npair * (double)(1 << (n - 1)) * per_final;
  return 2.0 * fp + n * 2 * 30.0 + 4 * 40.0 + (1 << n) * 40.0;
}
// FP64 tensor-pipe flops of the colour form (upper-triangular mma.m8n8k4 tiles, 256 FMA each), both parameter sets
static double bg_tensor_flops_per_event(const BgProcess* B) {
  const int n = B->S.n; int npp = (B->S.nperm + 7) / 8 * 8, MT = npp / 8, KT = npp / 4; double ksteps = 0; for (int mt = 0; mt < MT; mt++) ksteps += KT - 2 * mt;
  return 2.0 * 2.0 * ksteps * ((double)(4 << (n - 1)) * 2 / 8) * 256.0;
}

static int bg_run(BgProcess* B, int precision, const double* mom, const double* w, double* a, double* b, double* o, long long nev, cudaStream_t st) {
  BgDev D = B->D; const bool dbl = (precision == RWGT_FP64);
  D.nslot = dbl ? B->nslot64 : B->nslot32;
  long long ngroups = (nev + D.nslot - 1) / D.nslot; int grid = (int)std::min<long long>(ngroups, B->sm_count);
  switch (B->S.n) {
    case 2: bg_launch<2>(precision, grid, B->smem64, B->smem32, st, mom, w, a, b, o, nev, D); break;
    case 3: bg_launch<3>(precision, grid, B->smem64, B->smem32, st, mom, w, a, b, o, nev, D); break;
    case 4: bg_launch<4>(precision, grid, B->smem64, B->smem32, st, mom, w, a, b, o, nev, D); break;
    default: bg_launch<5>(precision, grid, B->smem64, B->smem32, st, mom, w, a, b, o, nev, D);
  }
  return 0;
}

}  // namespace rwgt
