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
  int fixbits;                      // number of gluon labels (0..fixbits-1) whose helicity is fixed per batch
  int nbatch, nfree, ncol;          // batches, free gluon configs per batch, columns of the amplitude buffer
  int ntG[6], offG[6], strideG[6];  // gluon levels m = 2..n-1: tuples, offset into words, words per task
  int ntR[6], offR[6], strideR[6];  // right levels m = 1..rmax
  int ntL[6], offL[6], strideL[6];  // left  levels m = 1..lmax
  int offF, strideF, ntermF;        // finals: one task descriptor per sigma pair
  std::vector<uint32_t> words;
  // instruction counts (FP-pipe instructions per event, one parameter set, all helicities)
  double fp_per_set, fp_shared;
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
  std::vector<int> idx(m); out.clear();
  // ordered tuples of distinct labels, lexicographic
  std::vector<int> cur; std::vector<bool> usedl(n, false);
  struct Rec { static void go(int n, int m, std::vector<int>& cur, std::vector<bool>& u, std::vector<std::vector<int>>& out) {
    if ((int)cur.size() == m) { out.push_back(cur); return; }
    for (int i = 0; i < n; i++) if (!u[i]) { u[i] = true; cur.push_back(i); go(n, m, cur, u, out); cur.pop_back(); u[i] = false; } } };
  Rec::go(n, m, cur, usedl, out);
}

// per-operation FP-pipe instruction counts of rwgt_math.cuh (FMA, MUL, ADD each 1); see DESIGN.md "Flop counts"
static const double OP_L3 = 90, OP_V4 = 102, OP_SLASH = 40, OP_PROP = 43, OP_ROWCOL = 16, OP_GSTORE = 24;

static BgSched build_schedule(int n) {
  BgSched S; S.n = n;
  for (int m = 0; m < 6; m++) { S.ntG[m] = S.offG[m] = S.strideG[m] = S.ntR[m] = S.offR[m] = S.strideR[m] = S.ntL[m] = S.offL[m] = S.strideL[m] = 0; }
  S.c = (n + 1) / 2; S.lmax = S.c - 1; S.rmax = n - S.c;          // n=2: c=1; 3: 2; 4: 2; 5: 3
  S.fixbits = (n == 5) ? 2 : 0;
  S.nbatch = 1 << S.fixbits; S.nfree = 1 << (n - S.fixbits); S.ncol = S.nfree * 4;
  TupleTables T; std::vector<std::vector<int>> tl;
  int nG = 0, nR = 0, nL = 0;
  for (int m = 1; m <= n - 1; m++) { all_tuples(n, m, tl); for (auto& t : tl) if (is_canon(t)) { T.gbase[t] = nG; nG += 1 << m; } }
  T.rbase[{}] = nR; nR += 2; T.lbase[{}] = nL; nL += 2;
  for (int m = 1; m <= S.rmax; m++) { all_tuples(n, m, tl); for (auto& t : tl) { T.rbase[t] = nR; nR += 2 << m; } }
  for (int m = 1; m <= S.lmax; m++) { all_tuples(n, m, tl); for (auto& t : tl) { T.lbase[t] = nL; nL += 2 << m; } }
  S.nG = nG; S.nR = nR; S.nL = nL;
  double fp = 0;
  // gluon levels
  for (int m = 2; m <= n - 1; m++) {
    all_tuples(n, m, tl); S.offG[m] = (int)S.words.size(); S.strideG[m] = 2 + 2 * (m - 1) + 3 * (m - 1) * (m - 2) / 2; int cnt = 0;
    for (auto& t : tl) if (is_canon(t)) {
      cnt++; S.words.push_back(T.gbase[t]); S.words.push_back(mask_of(t));
      for (int k = 1; k < m; k++) { S.words.push_back(gref(T, t, 0, k, false)); S.words.push_back(gref(T, t, k, m, false)); }
      for (int j = 1; j < m; j++) for (int k = j + 1; k < m; k++) { S.words.push_back(gref(T, t, 0, j, false)); S.words.push_back(gref(T, t, j, k, false)); S.words.push_back(gref(T, t, k, m, false)); }
    }
    S.ntG[m] = cnt;
    fp += (double)cnt * (1 << m) * ((m - 1) * OP_L3 + (m - 1) * (m - 2) / 2 * OP_V4 + OP_GSTORE);
  }
  for (int m = 1; m <= S.rmax; m++) {
    all_tuples(n, m, tl); S.offR[m] = (int)S.words.size(); S.strideR[m] = 2 + 2 * m; S.ntR[m] = (int)tl.size();
    for (auto& t : tl) {
      S.words.push_back(T.rbase[t]); S.words.push_back(mask_of(t));
      for (int k = 1; k <= m; k++) { S.words.push_back(gref(T, t, 0, k, false)); S.words.push_back(qref(T.rbase, t, k, m, false)); }
    }
    fp += (double)tl.size() * (2 << m) * (m * (OP_SLASH + 8) + OP_PROP);
  }
  for (int m = 1; m <= S.lmax; m++) {
    all_tuples(n, m, tl); S.offL[m] = (int)S.words.size(); S.strideL[m] = 2 + 2 * m; S.ntL[m] = (int)tl.size();
    for (auto& t : tl) {
      S.words.push_back(T.lbase[t]); S.words.push_back(mask_of(t));
      for (int k = 1; k <= m; k++) { S.words.push_back(qref(T.lbase, t, 0, m - k, false)); S.words.push_back(gref(T, t, m - k, m, false)); }
    }
    fp += (double)tl.size() * (2 << m) * (m * (OP_SLASH + 8) + OP_PROP);
  }
  // finals: one descriptor per pair (sigma, sigma reversed), sigma_1 < sigma_n
  std::vector<std::vector<int>> perms; { std::vector<int> p(n); for (int i = 0; i < n; i++) p[i] = i; do perms.push_back(p); while (std::next_permutation(p.begin(), p.end())); }
  S.nperm = (int)perms.size(); std::map<std::vector<int>, int> rank; for (int i = 0; i < S.nperm; i++) rank[perms[i]] = i;
  S.ntermF = S.c * (n - S.c + 1) - 1;
  S.offF = (int)S.words.size(); S.strideF = 4 + 2 * (n - 1) + 3 * (n - 1) * (n - 2) / 2 + 2 * 3 * S.ntermF; S.npair = 0;
  for (auto& s : perms) if (n == 1 || s.front() < s.back()) {
    S.npair++;
    std::vector<int> sr(s.rbegin(), s.rend());
    uint32_t packed = 0; for (int j = 0; j < n; j++) packed |= (uint32_t)s[j] << (3 * j);
    S.words.push_back(rank[s]); S.words.push_back(rank[sr]); S.words.push_back(packed); S.words.push_back(n % 2 == 0 ? 1u : 0u);   // J_n(rev) = (-1)^{n+1} J_n
    for (int k = 1; k < n; k++) { S.words.push_back(gref(T, s, 0, k, false)); S.words.push_back(gref(T, s, k, n, false)); }
    for (int j = 1; j < n; j++) for (int k = j + 1; k < n; k++) { S.words.push_back(gref(T, s, 0, j, false)); S.words.push_back(gref(T, s, j, k, false)); S.words.push_back(gref(T, s, k, n, false)); }
    // terms of sigma: blocks [i,j) in sigma's ascending positions
    for (int i = 0; i < S.c; i++) for (int j = S.c; j <= n; j++) { if (i == 0 && j == n) continue;
      S.words.push_back(qref(T.lbase, s, 0, i, false)); S.words.push_back(gref(T, s, i, j, false)); S.words.push_back(qref(T.rbase, s, j, n, false)); }
    // terms of sigma reversed: its positions [i,j) are sigma positions [n-j, n-i) read descending
    for (int i = 0; i < S.c; i++) for (int j = S.c; j <= n; j++) { if (i == 0 && j == n) continue;
      S.words.push_back(qref(T.lbase, s, n - i, n, true)); S.words.push_back(gref(T, s, n - j, n - i, true)); S.words.push_back(qref(T.rbase, s, 0, n - j, true)); }
  }
  double per_final = (n - 1) * OP_L3 + (n - 1) * (n - 2) / 2 * OP_V4 + OP_GSTORE + 2 * OP_SLASH + 4 * OP_ROWCOL + 2 * S.ntermF * (2 * OP_SLASH + 4 * OP_ROWCOL);
  fp += (double)S.npair * (1 << n) * per_final;
  // colour form: per helicity column nperm^2 complex-by-real FMAs (2 each) + nperm * 2 for the row products
  fp += (double)(4 << n) * (2.0 * S.nperm * S.nperm + 2.0 * S.nperm);
  S.fp_per_set = fp;
  // externals: polarisation vectors, spinors, 2^n momentum sums and denominators (rough, small)
  S.fp_shared = n * 2 * 30.0 + 4 * 40.0 + (1 << n) * 40.0;
  return S;
}

// ------------------------------------------------------------------------------------------------ device side
struct BgSet { double gq, g3, g4, mt, fac; };        // fac = gq^2 / D  (common factor |i gq|^2 and averaging)
struct BgDev {
  int n, c, nperm, npair, nG, nR, nL, fixbits, nbatch, nfree, ncol, ntermF;
  int ntG[6], offG[6], strideG[6], ntR[6], offR[6], strideR[6], ntL[6], offL[6], strideL[6];
  int offF, strideF, lmax, rmax;
  int nslot, rows_per_chunk, nchunk;
  int shared_ext;                    // 1: both sets share masses -> externals computed once
  const uint32_t* words;
  const double* C64; const float* C32;
  BgSet set[2];
};

struct BgProcess {
  BgSched S; BgDev D; uint32_t* d_words; double* d_C64; float* d_C32; int sm_count; size_t smem64, smem32; int nslot64, nslot32;
};

template <typename T> struct Smem {
  // pointers into the dynamic shared memory of one CTA
  double* pm;     // [nslot][n_ext][4] momenta (always double)
  T* G; T* R; T* L;  // [nslot][8][nX]
  T* K;           // [nslot][32][4] momentum sums of gluon subsets
  T* iK2;         // [nslot][32]
  T* dR; T* dL;   // [nslot][32] 1/(q^2-m^2)
  T* A;           // [nslot][nperm][ncol][2]
  double* acc;    // [nslot][2]
  double* red;    // [nslot][8] per-warp partial sums of the colour form
};

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
template <typename T> __device__ __forceinline__ T ref_sign(uint32_t r) { return (r & REF_NEG) ? T(-1) : T(1); }

// gluon current of one ordered tuple/variant from lower currents; returns the unscaled sums
template <typename T> __device__ __forceinline__ vec4<T> gluon_sum(const uint32_t* __restrict__ w, int m, uint32_t v, const T* G, int nG,
                                                                  const T* K, T g3, T g4) {
  vec4<T> a3, a4;
#pragma unroll
  for (int i = 0; i < 4; i++) { a3.c[i] = mk<T>(0, 0); a4.c[i] = mk<T>(0, 0); }
  for (int k = 0; k < m - 1; k++) {
    uint32_t ra = __ldg(w + 2 * k), rb = __ldg(w + 2 * k + 1);
    vec4<T> A = ld4(G, nG, ref_entry(ra, v)), B = ld4(G, nG, ref_entry(rb, v));
    L3_acc(a3, ref_sign<T>(ra) * ref_sign<T>(rb), A, K + 4 * ref_mask(ra), B, K + 4 * ref_mask(rb));
  }
  const uint32_t* w4 = w + 2 * (m - 1);
  int n4 = (m - 1) * (m - 2) / 2;
  for (int t = 0; t < n4; t++) {
    uint32_t rx = __ldg(w4 + 3 * t), ry = __ldg(w4 + 3 * t + 1), rz = __ldg(w4 + 3 * t + 2);
    vec4<T> X = ld4(G, nG, ref_entry(rx, v)), Y = ld4(G, nG, ref_entry(ry, v)), Z = ld4(G, nG, ref_entry(rz, v));
    V4_acc(a4, ref_sign<T>(rx) * ref_sign<T>(ry) * ref_sign<T>(rz), X, Y, Z);
  }
  vec4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) { r.c[i] = (-g3) * a3.c[i]; rfma(r.c[i], g4, a4.c[i]); }
  return r;
}

template <typename T> __device__ __forceinline__ void carve(Smem<T>& s, unsigned char* base, const BgDev& D) {
  size_t off = 0; int ns = D.nslot;
  s.pm = (double*)(base + off); off += sizeof(double) * ns * (D.n + 2) * 4;
  s.acc = (double*)(base + off); off += sizeof(double) * ns * 2;
  s.red = (double*)(base + off); off += sizeof(double) * ns * 8;
  s.G = (T*)(base + off); off += sizeof(T) * ns * 8 * D.nG;
  s.R = (T*)(base + off); off += sizeof(T) * ns * 8 * D.nR;
  s.L = (T*)(base + off); off += sizeof(T) * ns * 8 * D.nL;
  s.K = (T*)(base + off); off += sizeof(T) * ns * 32 * 4;
  s.iK2 = (T*)(base + off); off += sizeof(T) * ns * 32;
  s.dR = (T*)(base + off); off += sizeof(T) * ns * 32;
  s.dL = (T*)(base + off); off += sizeof(T) * ns * 32;
  off = (off + 15) & ~(size_t)15;
  s.A = (T*)(base + off);
}
static size_t smem_bytes(const BgSched& S, int nslot, size_t sz) {
  size_t off = 0;
  off += sizeof(double) * nslot * (S.n + 2) * 4 + sizeof(double) * nslot * 10;
  off += sz * nslot * 8 * (size_t)(S.nG + S.nR + S.nL);
  off += sz * nslot * 32 * 7;
  off = (off + 15) & ~(size_t)15;
  off += sz * nslot * (size_t)S.nperm * S.ncol * 2;
  return off;
}

// MIXED: T = float but momentum sums / denominators are formed in double before rounding to T.
template <typename T, bool MIXED>
__global__ void __launch_bounds__(256, 1) bg_kernel(const double* __restrict__ mom, const double* __restrict__ wgt,
                                                    double* __restrict__ me_old, double* __restrict__ me_new,
                                                    double* __restrict__ w_new, long long nev, BgDev D) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<T> s; carve<T>(s, smem_raw, D);
  typedef typename std::conditional<MIXED, double, T>::type TK;      // type used to form momentum sums and denominators
  const int tid = threadIdx.x, nth = blockDim.x, n = D.n, next = n + 2, ns = D.nslot;
  const int nG = D.nG, nR = D.nR, nL = D.nL;
  const long long ngroups = (nev + ns - 1) / ns;
  for (long long grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
    const long long ev0 = grp * ns;
    __syncthreads();   // previous group's outputs were read
    // ---- a1: load momenta (coalesced over events within the group) ----
    for (int t = tid; t < ns * next * 4; t += nth) {
      int sl = t % ns, comp = t / ns; long long ev = ev0 + sl; if (ev >= nev) ev = nev - 1;
      s.pm[(sl * next * 4) + comp] = __ldg(mom + (size_t)comp * nev + ev);
    }
    if (tid < ns * 2) s.acc[tid] = 0.0;
    __syncthreads();
    for (int iset = 0; iset < 2; iset++) {
      const BgSet& P = D.set[iset];
      const T g3 = (T)P.g3, g4 = (T)P.g4, gq = (T)P.gq, mt = (T)P.mt;
      if (iset == 0 || !D.shared_ext) {
        // ---- a2: external wavefunctions, momentum sums, propagator denominators ----
        int nobj = 2 * n + 4 + 32;
        for (int t = tid; t < ns * nobj; t += nth) {
          int sl = t / nobj, o = t % nobj; const double* pm = s.pm + sl * next * 4;
          if (o < 2 * n) {                         // gluon i, helicity bit hb (0: +1, 1: -1); entry = 2*i + hb
            int i = o >> 1, hb = o & 1, leg = i < 2 ? i : i + 2; const double* p = pm + 4 * leg;
            vec4<T> e = polvec<T>((T)p[1], (T)p[2], (T)p[3], hb ? -1 : +1);
            if (i >= 2) e = conj4(e);              // outgoing gluon carries eps*
            st4(s.G + (size_t)sl * 8 * nG, nG, 2 * i + hb, e);
          } else if (o < 2 * n + 2) {              // v(p_tbar, lam), R() entries 0,1
            int hb = o - 2 * n; const double* p = pm + 12;
            chi_pair<T> x = make_chi<T>((T)p[1], (T)p[2], (T)p[3]);
            st4(s.R + (size_t)sl * 8 * nR, nR, hb, spinor_v<T>(x, (T)p[0], mt, hb ? -1 : +1));
          } else if (o < 2 * n + 4) {              // ubar(p_t, lam), L() entries 0,1
            int hb = o - 2 * n - 2; const double* p = pm + 8;
            chi_pair<T> x = make_chi<T>((T)p[1], (T)p[2], (T)p[3]);
            st4(s.L + (size_t)sl * 8 * nL, nL, hb, bar(spinor_u<T>(x, (T)p[0], mt, hb ? -1 : +1)));
          } else {                                 // subset mask
            int mask = o - 2 * n - 4;
            if (mask < (1 << n)) {
              TK k[4] = {0, 0, 0, 0};
              for (int i = 0; i < n; i++) if (mask >> i & 1) { int leg = i < 2 ? i : i + 2; TK sg = i < 2 ? TK(1) : TK(-1);
                for (int mu = 0; mu < 4; mu++) k[mu] += sg * (TK)pm[4 * leg + mu]; }
              TK k2 = mdot_rr<TK>(k, k);
              TK qr[4], ql[4]; for (int mu = 0; mu < 4; mu++) { qr[mu] = k[mu] - (TK)pm[12 + mu]; ql[mu] = (TK)pm[8 + mu] - k[mu]; }
              TK m2 = (TK)P.mt * (TK)P.mt;
              T* K = s.K + (size_t)sl * 128 + 4 * mask; for (int mu = 0; mu < 4; mu++) K[mu] = (T)k[mu];
              s.iK2[sl * 32 + mask] = (__popc(mask) >= 2) ? (T)(TK(1) / k2) : T(0);
              s.dR[sl * 32 + mask] = (T)(TK(1) / (mdot_rr<TK>(qr, qr) - m2));
              s.dL[sl * 32 + mask] = (T)(TK(1) / (mdot_rr<TK>(ql, ql) - m2));
            }
          }
        }
        __syncthreads();
      }
      // ---- a3: current levels.  phase m: gluon level m, right level m-1, left level m-1 ----
      int nphase = max(n - 1, max(D.rmax, D.lmax) + 1);
      for (int m = 2; m <= nphase; m++) {
        int tg = (m <= n - 1) ? (D.ntG[m] << m) : 0;
        int tr = (m - 1 >= 1 && m - 1 <= D.rmax) ? (D.ntR[m - 1] << m) : 0;      // 2^(m-1) variants x 2 quark helicities
        int tl = (m - 1 >= 1 && m - 1 <= D.lmax) ? (D.ntL[m - 1] << m) : 0;
        int per = tg + tr + tl;
        for (int t = tid; t < ns * per; t += nth) {
          int sl = t / per, o = t % per;
          T* G = s.G + (size_t)sl * 8 * nG; T* R = s.R + (size_t)sl * 8 * nR; T* L = s.L + (size_t)sl * 8 * nL;
          const T* K = s.K + (size_t)sl * 128;
          if (o < tg) {
            int tup = o >> m; uint32_t v = o & ((1 << m) - 1);
            const uint32_t* w = D.words + D.offG[m] + tup * D.strideG[m];
            int ob = __ldg(w), mask = __ldg(w + 1);
            vec4<T> r = gluon_sum<T>(w + 2, m, v, G, nG, K, g3, g4);
            T sc = s.iK2[sl * 32 + mask];
#pragma unroll
            for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
            st4(G, nG, ob + v, r);
          } else if (o < tg + tr) {
            int mm = m - 1, oo = o - tg; int tup = oo >> m; uint32_t vv = oo & ((1 << m) - 1); uint32_t v = vv & ((1 << mm) - 1); int hb = vv >> mm;
            const uint32_t* w = D.words + D.offR[mm] + tup * D.strideR[mm];
            int ob = __ldg(w), mask = __ldg(w + 1);
            spn<T> acc; for (int i = 0; i < 4; i++) acc.c[i] = mk<T>(0, 0);
            for (int k = 0; k < mm; k++) {
              uint32_t rj = __ldg(w + 2 + 2 * k), rr = __ldg(w + 3 + 2 * k);
              vec4<T> J = ld4(G, nG, ref_entry(rj, v));
              spn<T> Rr = lds4(R, nR, ref_entry(rr, v) + (hb << ref_m(rr)));
              spn<T> x = slash_c(J, Rr); T sg = ref_sign<T>(rj);
              for (int i = 0; i < 4; i++) rfma(acc.c[i], sg, x.c[i]);
            }
            T q[4]; for (int mu = 0; mu < 4; mu++) q[mu] = K[4 * mask + mu] - (T)s.pm[sl * next * 4 + 12 + mu];
            spn<T> r = slash_r_plus_m(q, mt, acc); T sc = -gq * s.dR[sl * 32 + mask];
            for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
            st4(R, nR, ob + v + (hb << mm), r);
          } else {
            int mm = m - 1, oo = o - tg - tr; int tup = oo >> m; uint32_t vv = oo & ((1 << m) - 1); uint32_t v = vv & ((1 << mm) - 1); int hb = vv >> mm;
            const uint32_t* w = D.words + D.offL[mm] + tup * D.strideL[mm];
            int ob = __ldg(w), mask = __ldg(w + 1);
            spn<T> acc; for (int i = 0; i < 4; i++) acc.c[i] = mk<T>(0, 0);
            for (int k = 0; k < mm; k++) {
              uint32_t rl = __ldg(w + 2 + 2 * k), rj = __ldg(w + 3 + 2 * k);
              spn<T> Ll = lds4(L, nL, ref_entry(rl, v) + (hb << ref_m(rl)));
              vec4<T> J = ld4(G, nG, ref_entry(rj, v));
              spn<T> x = row_slash_c(Ll, J); T sg = ref_sign<T>(rj);
              for (int i = 0; i < 4; i++) rfma(acc.c[i], sg, x.c[i]);
            }
            T q[4]; for (int mu = 0; mu < 4; mu++) q[mu] = (T)s.pm[sl * next * 4 + 8 + mu] - K[4 * mask + mu];
            spn<T> r = row_slash_r_plus_m(acc, q, mt); T sc = -gq * s.dL[sl * 32 + mask];
            for (int i = 0; i < 4; i++) r.c[i] = sc * r.c[i];
            st4(L, nL, ob + v + (hb << mm), r);
          }
        }
        __syncthreads();
      }
      // ---- a3/a4: colour-flow amplitudes per helicity batch; a5/a6: colour form and helicity sum ----
      const int ncol = D.ncol, nperm = D.nperm;
      for (int batch = 0; batch < D.nbatch; batch++) {
        int per = D.npair * D.nfree;
        for (int t = tid; t < ns * per; t += nth) {
          int sl = t / per, o = t % per; int pair = o / D.nfree, f = o % D.nfree;
          const T* G = s.G + (size_t)sl * 8 * nG; const T* R = s.R + (size_t)sl * 8 * nR; const T* L = s.L + (size_t)sl * 8 * nL;
          const T* K = s.K + (size_t)sl * 128;
          const uint32_t* w = D.words + D.offF + pair * D.strideF;
          uint32_t rk = __ldg(w), rkr = __ldg(w + 1), packed = __ldg(w + 2), negr = __ldg(w + 3);
          uint32_t g = (uint32_t)batch | ((uint32_t)f << D.fixbits);        // helicity bits by gluon label
          uint32_t v = 0; for (int j = 0; j < n; j++) v |= ((g >> ((packed >> (3 * j)) & 7u)) & 1u) << j;   // by position in sigma
          vec4<T> Jn = gluon_sum<T>(w + 4, n, v, G, nG, K, g3, g4);
          T sc = s.iK2[sl * 32 + ((1 << n) - 1)];
#pragma unroll
          for (int i = 0; i < 4; i++) Jn.c[i] = sc * Jn.c[i];
          cx<T> As[2][2], Ar[2][2];
          {
            spn<T> u0 = lds4(L, nL, 0), u1 = lds4(L, nL, 1);
#pragma unroll
            for (int hb = 0; hb < 2; hb++) {
              spn<T> x = slash_c(Jn, lds4(R, nR, hb));
              As[0][hb] = rowcol(u0, x); As[1][hb] = rowcol(u1, x);
            }
            T sr = negr ? T(-1) : T(1);
#pragma unroll
            for (int ht = 0; ht < 2; ht++)
#pragma unroll
              for (int hb = 0; hb < 2; hb++) Ar[ht][hb] = sr * As[ht][hb];
          }
          const uint32_t* wt = w + 4 + 2 * (n - 1) + 3 * (n - 1) * (n - 2) / 2;
          for (int which = 0; which < 2; which++) {
            cx<T>(*Acc)[2] = which ? Ar : As;
            for (int term = 0; term < D.ntermF; term++) {
              uint32_t rl = __ldg(wt + 3 * term), rj = __ldg(wt + 3 * term + 1), rr = __ldg(wt + 3 * term + 2);
              vec4<T> J = ld4(G, nG, ref_entry(rj, v)); T sg = ref_sign<T>(rj);
              int el = ref_entry(rl, v), er = ref_entry(rr, v), ml = ref_m(rl), mr = ref_m(rr);
              spn<T> l0 = lds4(L, nL, el), l1 = lds4(L, nL, el + (1 << ml));
#pragma unroll
              for (int hb = 0; hb < 2; hb++) {
                spn<T> x = slash_c(J, lds4(R, nR, er + (hb << mr)));
                cx<T> a0 = rowcol(l0, x), a1 = rowcol(l1, x);
                rfma(Acc[0][hb], sg, a0); rfma(Acc[1][hb], sg, a1);
              }
            }
            wt += 3 * D.ntermF;
          }
          T* A = s.A + (size_t)sl * nperm * ncol * 2;
#pragma unroll
          for (int ht = 0; ht < 2; ht++)
#pragma unroll
            for (int hb = 0; hb < 2; hb++) {
              int col = f * 4 + ht * 2 + hb;
              A[((size_t)rk * ncol + col) * 2] = As[ht][hb].re; A[((size_t)rk * ncol + col) * 2 + 1] = As[ht][hb].im;
              A[((size_t)rkr * ncol + col) * 2] = Ar[ht][hb].re; A[((size_t)rkr * ncol + col) * 2 + 1] = Ar[ht][hb].im;
            }
        }
        __syncthreads();
        // colour form: thread = (slot, chunk of rows, column)
        {
          const int RB = D.rows_per_chunk, nchunk = D.nchunk; int percf = ncol * nchunk;
          for (int t = tid; t < ns * percf; t += nth) {
            int sl = t / percf, o = t % percf; int chunk = o / ncol, col = o % ncol;
            const T* A = s.A + (size_t)sl * nperm * ncol * 2;
            int r0 = chunk * RB, nr = max(0, min(RB, nperm - r0));
            double part = 0.0;
            if (sizeof(T) == 8) {
              const double* C = D.C64;
              for (int rb = 0; rb < nr; rb += 5) {            // register block of 5 rows
                double yr[5] = {0, 0, 0, 0, 0}, yi[5] = {0, 0, 0, 0, 0}; int nb = min(5, nr - rb);
                for (int sp = 0; sp < nperm; sp++) {
                  double ar = (double)A[((size_t)sp * ncol + col) * 2], ai = (double)A[((size_t)sp * ncol + col) * 2 + 1];
                  const double* Cr = C + (size_t)sp * nperm + r0 + rb;       // C symmetric: column sp == row sp
#pragma unroll
                  for (int r = 0; r < 5; r++) if (r < nb) { double c = __ldg(Cr + r); yr[r] = fma(c, ar, yr[r]); yi[r] = fma(c, ai, yi[r]); }
                }
#pragma unroll
                for (int r = 0; r < 5; r++) if (r < nb) {
                  double ar = (double)A[((size_t)(r0 + rb + r) * ncol + col) * 2], ai = (double)A[((size_t)(r0 + rb + r) * ncol + col) * 2 + 1];
                  part = fma(ar, yr[r], part); part = fma(ai, yi[r], part);
                }
              }
            } else {
              const float* C = D.C32;
              for (int rb = 0; rb < nr; rb += 5) {
                float yr[5] = {0, 0, 0, 0, 0}, yi[5] = {0, 0, 0, 0, 0}; int nb = min(5, nr - rb);
                for (int sp = 0; sp < nperm; sp++) {
                  float ar = (float)A[((size_t)sp * ncol + col) * 2], ai = (float)A[((size_t)sp * ncol + col) * 2 + 1];
                  const float* Cr = C + (size_t)sp * nperm + r0 + rb;
#pragma unroll
                  for (int r = 0; r < 5; r++) if (r < nb) { float c = __ldg(Cr + r); yr[r] = fmaf(c, ar, yr[r]); yi[r] = fmaf(c, ai, yi[r]); }
                }
#pragma unroll
                for (int r = 0; r < 5; r++) if (r < nb) {
                  float ar = (float)A[((size_t)(r0 + rb + r) * ncol + col) * 2], ai = (float)A[((size_t)(r0 + rb + r) * ncol + col) * 2 + 1];
                  part += (double)(ar * yr[r] + ai * yi[r]);
                }
              }
            }
            // deterministic reduction (identical for both parameter sets, so old == new gives a ratio of exactly 1):
            // ncol*nchunk is a multiple of 32, hence a warp never straddles two slots
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
            if ((tid & 31) == 0) s.red[sl * 8 + (o >> 5)] = part;
          }
          __syncthreads();
          if (tid < ns) { double a = 0.0; for (int j = 0; j < percf / 32; j++) a += s.red[tid * 8 + j]; s.acc[tid * 2 + iset] += a; }
        }
        __syncthreads();
      }
    }
    // ---- a7: eq. 3 and stores ----
    if (tid < ns) {
      long long ev = ev0 + tid;
      if (ev < nev) {
        double a = s.acc[tid * 2] * D.set[0].fac, b = s.acc[tid * 2 + 1] * D.set[1].fac;
        me_old[ev] = a; me_new[ev] = b; w_new[ev] = __ldg(wgt + ev) * (b / a);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ host API of the engine
static BgProcess* bg_create(int n, const rwgt_params& po, const rwgt_params& pn, std::string& err) {
  BgProcess* B = new BgProcess();
  B->S = build_schedule(n);
  const BgSched& S = B->S;
  BgDev& D = B->D;
  D.n = n; D.c = S.c; D.nperm = S.nperm; D.npair = S.npair; D.nG = S.nG; D.nR = S.nR; D.nL = S.nL; D.fixbits = S.fixbits; D.nbatch = S.nbatch;
  D.nfree = S.nfree; D.ncol = S.ncol; D.ntermF = S.ntermF; D.offF = S.offF; D.strideF = S.strideF; D.lmax = S.lmax; D.rmax = S.rmax;
  for (int m = 0; m < 6; m++) { D.ntG[m] = S.ntG[m]; D.offG[m] = S.offG[m]; D.strideG[m] = S.strideG[m]; D.ntR[m] = S.ntR[m]; D.offR[m] = S.offR[m];
    D.strideR[m] = S.strideR[m]; D.ntL[m] = S.ntL[m]; D.offL[m] = S.offL[m]; D.strideL[m] = S.strideL[m]; }
  const rwgt_params* ps[2] = {&po, &pn};
  double fact = 1; for (int i = 2; i <= n - 2; i++) fact *= i;
  for (int k = 0; k < 2; k++) {
    double gs = std::sqrt(4.0 * 3.14159265358979323846 * ps[k]->alpha_s);
    D.set[k].gq = gs; D.set[k].g3 = gs * ps[k]->ggg_scale; D.set[k].g4 = gs * gs * ps[k]->gggg_scale; D.set[k].mt = ps[k]->mt;
    D.set[k].fac = gs * gs / (256.0 * fact);
  }
  D.shared_ext = (po.mt == pn.mt) ? 1 : 0;
  // rows per colour chunk: aim at ~256 colour tasks per slot-batch
  // colour tasks per slot and batch = ncol * nchunk: a multiple of 32 (warp-aligned reduction) and at most 256
  int nchunk = std::max(1, std::min(S.nperm, 256 / S.ncol)); if ((S.ncol * nchunk) % 32) nchunk &= ~1;
  D.rows_per_chunk = (S.nperm + nchunk - 1) / nchunk; D.nchunk = nchunk;
  int dev = 0; cudaGetDevice(&dev); cudaDeviceProp prop; cudaGetDeviceProperties(&prop, dev);
  B->sm_count = prop.multiProcessorCount; size_t maxsm = prop.sharedMemPerBlockOptin;
  auto pick = [&](size_t sz, int& nslot, size_t& bytes) {
    int cap = (n == 2) ? 64 : (n == 3) ? 32 : (n == 4) ? 8 : 1; nslot = 0;
    for (int e = cap; e >= 1; e--) if (smem_bytes(S, e, sz) <= maxsm) { nslot = e; break; }
    bytes = nslot ? smem_bytes(S, nslot, sz) : 0;
  };
  pick(8, B->nslot64, B->smem64); pick(4, B->nslot32, B->smem32);
  if (!B->nslot64 || !B->nslot32) { err = "not enough shared memory per block on this device"; delete B; return nullptr; }
  std::vector<double> C = colour_matrix_fierz(n); std::vector<float> Cf(C.begin(), C.end());
  cudaError_t e = cudaMalloc((void**)&B->d_words, S.words.size() * sizeof(uint32_t));
  if (e == cudaSuccess) e = cudaMalloc((void**)&B->d_C64, C.size() * sizeof(double));
  if (e == cudaSuccess) e = cudaMalloc((void**)&B->d_C32, Cf.size() * sizeof(float));
  if (e == cudaSuccess) e = cudaMemcpy(B->d_words, S.words.data(), S.words.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(B->d_C64, C.data(), C.size() * sizeof(double), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(B->d_C32, Cf.data(), Cf.size() * sizeof(float), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<double, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)B->smem64);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<float, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)B->smem32);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(bg_kernel<float, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)B->smem32);
  if (e != cudaSuccess) { err = std::string("CUDA: ") + cudaGetErrorString(e); delete B; return nullptr; }
  D.words = B->d_words; D.C64 = B->d_C64; D.C32 = B->d_C32;
  return B;
}
static void bg_destroy(BgProcess* B) { if (!B) return; cudaFree(B->d_words); cudaFree(B->d_C64); cudaFree(B->d_C32); delete B; }
static double bg_flops_per_event(const BgProcess* B, int /*precision*/) { return 2.0 * (2.0 * B->S.fp_per_set + B->S.fp_shared); }
static int bg_run(BgProcess* B, int precision, const double* mom, const double* w, double* a, double* b, double* o, long long nev, cudaStream_t st) {
  BgDev D = B->D;
  if (precision == RWGT_FP64) {
    D.nslot = B->nslot64; long long ngroups = (nev + D.nslot - 1) / D.nslot; int grid = (int)std::min<long long>(ngroups, B->sm_count);
    bg_kernel<double, false><<<grid, 256, B->smem64, st>>>(mom, w, a, b, o, nev, D);
  } else {
    D.nslot = B->nslot32; long long ngroups = (nev + D.nslot - 1) / D.nslot; int grid = (int)std::min<long long>(ngroups, B->sm_count);
    if (precision == RWGT_FP32) bg_kernel<float, false><<<grid, 256, B->smem32, st>>>(mom, w, a, b, o, nev, D);
    else bg_kernel<float, true><<<grid, 256, B->smem32, st>>>(mom, w, a, b, o, nev, D);
  }
  return 0;
}

}  // namespace rwgt
