// photon_kernel.cuh — e+(p1) e-(p2) -> NG photons, NG = 2..5, FP64 (NG = 5 is the process the paper itself measured:
// PAPER.md:72-77, Table 1).  Steps a1-a7 of SURVEY 8(a) in one launch.
//
// What it evaluates: the sum of the NG! diagrams in which the photons leave the massless electron line in every order
// (rules of SURVEY C3: vertex -i e Q gamma^mu, propagator i q-slash / q^2; outgoing photons carry eps*), squared, summed over
// helicities, averaged (1/4 for the initial helicities, 1/NG! for the identical photons; reading R3), for every parameter set, and
// eq. 3.  Only alpha_em enters, and only through the overall factor e^(2 NG): the currents are evaluated once with
// unit coupling and each set multiplies the helicity sum by its own factor ("setting the electroweak coupling
// constant to be a randomly determined non-zero value for each reweight iteration"; so |M'|^2/|M|^2 = (alpha'/alpha)^NG exactly).
//
// Algorithm (not the diagram sum): off-shell electron currents of photon SUBSETS with helicity recycling,
//     psi_S = 1/q_S^2  q_S-slash  sum_{i in S} eps-slash*_i psi_{S \ i},   q_S = p2 - sum_{i in S} k_i,   psi_{} = u(p2, +),
// one per subset S and helicity assignment of ITS photons (3^NG - 2^NG currents instead of NG! 2^NG diagram evaluations), then
//     M(h) = vbar(p1, -) sum_i eps-slash*_i psi_{all \ i}.
// Massless line in the chiral representation: u(p2,+) has lower components only, eps-slash maps lower -> upper with the 2x2 block
// (eps0 - sigma.eps), q-slash maps upper -> lower with (q0 + sigma.q): every current is a TWO-component spinor.  The other electron
// helicity follows from parity (|M_{-h}| = |M_h|, pinned on the oracle): x2.  Equal e+ and e- helicities give zero.
//
// B200 mapping: persistent CTAs; a CTA holds E events in shared memory (currents as two component planes of (re,im) pairs,
// consecutive helicity variants in consecutive 16-byte words), a thread owns one (event, subset, helicity variant) task per level,
// levels are separated by __syncthreads; the 2^NG final amplitudes of an event sit in consecutive lanes and are reduced by a fixed
// shuffle tree (deterministic: equal parameter sets give W' = W bitwise).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "../../include/rwgt.h"
#include "rwgt_math.cuh"
#include "kernels_small.cuh"
#include "bg_engine.cuh"      // ldc / stc (vector loads of (re,im) pairs)

namespace rwgt {

struct PhotonParams { double fac[SMALL_NSMAX]; int nsets; };      // fac = 2 e^(2 NG) / (4 NG!)  per parameter set

__host__ __device__ constexpr int ipow(int b, int e) { return e == 0 ? 1 : b * ipow(b, e - 1); }
__host__ __device__ constexpr int binom(int n, int k) { return k == 0 ? 1 : binom(n - 1, k - 1) * n / k; }

__host__ __device__ constexpr int ph_level_size(int ng, int k) { return binom(ng, k) << k; }        // currents of k photons, all helicities
// most entries of a level of the given parity (levels 1 .. ng-1 are stored; the full set is consumed by the amplitudes)
__host__ __device__ constexpr int ph_max_level(int ng, int parity) {
  int m = 0; for (int k = 1; k < ng; k++) if ((k & 1) == parity && ph_level_size(ng, k) > m) m = ph_level_size(ng, k); return m;
}
template <int NG> struct PhGeo {
  static constexpr int NSUB = 1 << NG;
  // Level K reads level K-1 only, so the currents live in two buffers: odd levels in A (entries [0, NA)), even levels in B
  // ([NA, NA + NB)); a level overwrites the level two below it.  n = 5: 160 entries instead of 3^5 - 2^5 = 211 for all levels,
  // which is what lets a fourth CTA of 8 events fit into the SM's shared memory.
  static constexpr int NA = ph_max_level(NG, 1), NB = ph_max_level(NG, 0), NENT = NA + NB;
  static constexpr int NEXTOBJ = 2 * NG + 2 + NSUB;                        // external tasks per event
  // doubles per event slot.  Q holds q_S / q_S^2 (the propagator folded into the momentum).  The momenta are dead once the externals
  // are formed; for n = 5 they lie on the tail of component plane 1 of buffer B, which nothing writes before level 4.
  static constexpr bool PM_OVERLAY = (NG == 5);
  static constexpr int NPM = (NG + 2) * 4;
  static constexpr int O_EPS = PM_OVERLAY ? 0 : NPM, O_Q = O_EPS + NG * 2 * 8, O_W = O_Q + NSUB * 4, O_PSI = O_W + 4, SLOT0 = O_PSI + 4 * NENT;
  static constexpr int O_PM = PM_OVERLAY ? SLOT0 - NPM : 0;
  static_assert(!PM_OVERLAY || (2 * (NB - ph_level_size(NG, NG - 3)) >= NPM && ((NG - 1) & 1) == 0), "momenta overlay");
  // slot stride: an odd number of 16-byte words, so that the same word of 8 consecutive event slots falls into 8 different
  // bank groups (an LDS.128 of a quarter-warp whose lanes are 8 events x one task is then one conflict-free wavefront)
  static constexpr int SLOT = (SLOT0 / 2) % 2 == 1 ? SLOT0 : SLOT0 + 2;
};

// barrier over the cooperating group: the whole CTA (CG == NTH) or one warp (CG == 32)
template <int CG, int NTH> __device__ __forceinline__ void gsync() { if constexpr (CG == NTH) __syncthreads(); else __syncwarp(); }

// bit helpers for helicity-variant words (all arguments but v are compile-time after unrolling)
__device__ __forceinline__ constexpr unsigned remove_bit(unsigned v, int r) { return (v & ((1u << r) - 1u)) | ((v >> (r + 1)) << r); }
__device__ __forceinline__ constexpr unsigned insert_bit(unsigned v, int b, unsigned h) { return (v & ((1u << b) - 1u)) | (h << b) | ((v >> b) << (b + 1)); }

// Accumulation of one task: subset S of K photons (members by rank r = 0..K-1, ascending label; helicity-variant bit r belongs to
// member r), the helicities of the first KF = K - VB members fixed by `vfix`, ALL 2^VB helicity assignments of the last VB members
// evaluated by this thread:  acc[u] = sum_r eps-slash*(member r, its helicity) psi_{S minus r}(the other helicities).
// A fixed member loads one block and 2^VB child spinors, a free member both blocks and 2^(VB-1) child spinors (each spinor is used
// with both blocks): 2.0-2.2 LDS.128 per block product at VB = 3 against 4.2 at VB = 1 -- the shared-memory data pipe is what
// bounds this kernel.
// s_child[S][r] = (first entry of S without its r-th member) << 8 | (2 * that member's label).
template <int NG, int K, int VB>
__device__ __forceinline__ void photon_accumulate(cx<double> (&acc)[1 << VB][2], const double* s, const unsigned* s_child, int S, unsigned vfix) {
  typedef PhGeo<NG> Ge;
  constexpr int NENT = Ge::NENT, KF = K - VB, NV = 1 << VB;
  const cx<double>* M = reinterpret_cast<const cx<double>*>(s + Ge::O_EPS);
  const cx<double>* T = reinterpret_cast<const cx<double>*>(s + Ge::O_PSI);
#pragma unroll
  for (int u = 0; u < NV; u++) { acc[u][0] = mk<double>(0, 0); acc[u][1] = mk<double>(0, 0); }
#pragma unroll
  for (int r = 0; r < K; r++) {
    const unsigned ch = s_child[S * NG + r];
    const int cbase = (int)(ch >> 8);
    if (r < KF) {                                  // fixed member: one block, 2^VB spinors
      const unsigned hb = (vfix >> r) & 1u; const int e0 = cbase + (int)remove_bit(vfix, r);
      const cx<double>* m = M + ((ch & 0xffu) + hb) * 4;
      const cx<double> m0 = ldc(m), m1 = ldc(m + 1), m2 = ldc(m + 2), m3 = ldc(m + 3);
#pragma unroll
      for (int u = 0; u < NV; u++) {
        const int e = e0 + (u << (KF > 0 ? KF - 1 : 0));
        const cx<double> x0 = ldc(T + e), x1 = ldc(T + NENT + e);
        cfma(acc[u][0], m0, x0); cfma(acc[u][0], m1, x1); cfma(acc[u][1], m2, x0); cfma(acc[u][1], m3, x1);
      }
    } else {                                       // free member (bit b of u): both blocks, 2^(VB-1) spinors
      const int b = r - KF;
      const cx<double>* m = M + (ch & 0xffu) * 4;
      const cx<double> p0 = ldc(m), p1 = ldc(m + 1), p2 = ldc(m + 2), p3 = ldc(m + 3);
      const cx<double> n0 = ldc(m + 4), n1 = ldc(m + 5), n2 = ldc(m + 6), n3 = ldc(m + 7);
#pragma unroll
      for (int uc = 0; uc < NV / 2; uc++) {
        const int e = cbase + (int)vfix + (uc << KF);
        const cx<double> x0 = ldc(T + e), x1 = ldc(T + NENT + e);
        const int up = (int)insert_bit((unsigned)uc, b, 0u), un = (int)insert_bit((unsigned)uc, b, 1u);
        cfma(acc[up][0], p0, x0); cfma(acc[up][0], p1, x1); cfma(acc[up][1], p2, x0); cfma(acc[up][1], p3, x1);
        cfma(acc[un][0], n0, x0); cfma(acc[un][0], n1, x1); cfma(acc[un][1], n2, x0); cfma(acc[un][1], n3, x1);
      }
    }
  }
}

// One level of the recursion: all currents of K photons (K compile-time: constant divisors, branch-free member loops).
// VBMAX = [100 * (variant bits per thread at levels >= 4)] + 10 * (variant bits at level 2) + (variant bits at level 3 and, without the
// hundreds digit, above): the levels differ in tasks per event, and fewer variants per thread keep more threads busy.
// Lanes run event-fastest (a quarter-warp = 8 events x one task): every table access is then the same word of 8 event slots,
// conflict-free by the odd slot stride, and the task decode is uniform over the quarter-warp.
template <int NG, int K, int VBMAX, int E, int CG, int NTH>
__device__ __forceinline__ void photon_level(double* sm, const unsigned char* s_sub, const unsigned short* s_off, const unsigned* s_child, int first_sub, int tid) {
  typedef PhGeo<NG> Ge;
  constexpr int NENT = Ge::NENT, VBL = (K == 2 ? (VBMAX / 10) % 10 : (K >= 4 && VBMAX >= 100) ? VBMAX / 100 : VBMAX % 10), VB = K < VBL ? K : VBL, KF = K - VB, NV = 1 << VB, per = binom(NG, K) << KF;
  for (int t = tid; t < E * per; t += CG) {
    const int sl = t % E, o = t / E; const int S = s_sub[first_sub + (o >> KF)]; const unsigned vfix = o & ((1u << KF) - 1u);
    double* s = sm + sl * Ge::SLOT;
    cx<double> acc[NV][2];
    photon_accumulate<NG, K, VB>(acc, s, s_child, S, vfix);
    cx<double>* T = reinterpret_cast<cx<double>*>(s + Ge::O_PSI);
    const double* q = s + Ge::O_Q + 4 * S;               // q_S / q_S^2
    const double qp = q[0] + q[3], qm = q[0] - q[3]; const cx<double> qr = mk<double>(q[1], -q[2]), ql = mk<double>(q[1], q[2]);
    const int eo = s_off[S] + (int)vfix;
#pragma unroll
    for (int u = 0; u < NV; u++) {                 // (q0 + sigma.q) = [[q+, qr], [ql, q-]]
      cx<double> o0 = qp * acc[u][0]; cfma(o0, qr, acc[u][1]);
      cx<double> o1 = qm * acc[u][1]; cfma(o1, ql, acc[u][0]);
      stc(T + eo + (u << KF), o0); stc(T + NENT + eo + (u << KF), o1);
    }
  }
  gsync<CG, NTH>();
}
template <int NG, int K, int VBMAX, int E, int CG, int NTH>
__device__ __forceinline__ void photon_levels(double* sm, const unsigned char* s_sub, const unsigned short* s_off, const unsigned* s_child, const unsigned char* s_lvl, int tid) {
  if constexpr (K < NG) {
    photon_level<NG, K, VBMAX, E, CG, NTH>(sm, s_sub, s_off, s_child, s_lvl[K], tid);
    photon_levels<NG, K + 1, VBMAX, E, CG, NTH>(sm, s_sub, s_off, s_child, s_lvl, tid);
  }
}

// E events per cooperating group of CG threads (CG == NTH: the CTA, levels separated by __syncthreads; CG == 32: each warp works on
// its own E events and only ever waits for itself)
template <int NG, int E, int CG, int NTH, int VBL, int VBF>
__global__ void __launch_bounds__(NTH) epem_photons_kernel(const double* __restrict__ mom, const double* __restrict__ wgt,
                                                           double* __restrict__ me_old, double* __restrict__ me_new,
                                                           double* __restrict__ w_new, long long nev, long long stride, long long ostride,
                                                           PhotonParams P) {
  typedef PhGeo<NG> Ge;
  constexpr int next = NG + 2, NSUB = Ge::NSUB, NENT = Ge::NENT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = (CG == NTH) ? (int)threadIdx.x : (int)(threadIdx.x & 31u);                        // index within the group
  double* sm = reinterpret_cast<double*>(smem_raw) + (CG == NTH ? 0 : (threadIdx.x >> 5) * E * Ge::SLOT);   // the group's event slots
  __shared__ unsigned short s_off[NSUB];            // first entry of subset S
  __shared__ unsigned char s_sub[NSUB];             // subsets ordered by (size, value)
  __shared__ unsigned char s_lvl[NG + 2];           // s_sub index of the first subset of each size
  __shared__ unsigned s_child[NSUB * NG];           // (first entry of S without its r-th member) << 8 | 2 * member label
  if (threadIdx.x == 0) {
    int cnt[NG + 1]; for (int k = 0; k <= NG; k++) cnt[k] = (k & 1) ? 0 : Ge::NA;          // odd levels: buffer A, even levels: buffer B
    for (int S = 0; S < NSUB; S++) { const int k = __popc(S); s_off[S] = (unsigned short)cnt[k]; cnt[k] += 1 << k; }
    int j = 0; for (int k = 0; k <= NG; k++) { s_lvl[k] = (unsigned char)j; for (int S = 0; S < NSUB; S++) if (__popc(S) == k) s_sub[j++] = (unsigned char)S; }
    s_lvl[NG + 1] = (unsigned char)j;
    for (int S = 0; S < NSUB; S++) { int r = 0; for (int i = 0; i < NG; i++) if (S >> i & 1) s_child[S * NG + r++] = ((unsigned)s_off[S ^ (1 << i)] << 8) | (unsigned)(2 * i); }
  }
  __syncthreads();
  const long long ngroups = (nev + E - 1) / E;
  constexpr int GPB = NTH / CG;                                      // groups per CTA
  // a1 is software-pipelined: the momenta of a group are fetched into registers while the previous group's levels run
  constexpr int NPRE = (E * next * 4 + CG - 1) / CG;
  double pre[NPRE];
  auto fetch = [&](long long g) {
#pragma unroll
    for (int j = 0; j < NPRE; j++) {
      const int t = tid + j * CG;
      if (t < E * next * 4) { int sl = t % E, comp = t / E; long long ev = g * E + sl; if (ev >= nev) ev = nev - 1;
        pre[j] = __ldg(mom + (size_t)comp * stride + ev); }
    }
  };
  const long long grp0 = (long long)blockIdx.x * GPB + (CG == NTH ? 0 : threadIdx.x >> 5), gstep = (long long)gridDim.x * GPB;
  if (grp0 < ngroups) fetch(grp0);
  for (long long grp = grp0; grp < ngroups; grp += gstep) {
    const long long ev0 = grp * E;
    // ---- a1: momenta (coalesced over the events of the group) ----
#pragma unroll
    for (int j = 0; j < NPRE; j++) {
      const int t = tid + j * CG;
      if (t < E * next * 4) { int sl = t % E, comp = t / E; sm[sl * Ge::SLOT + Ge::O_PM + comp] = pre[j]; }
    }
    gsync<CG, NTH>();
    if (grp + gstep < ngroups) fetch(grp + gstep);
    // ---- a2: external wavefunctions, momenta and inverse virtualities of the electron line; the one-photon currents (level 1)
    //          are formed by the thread that builds the photon's polarisation block ----
    for (int t = tid; t < E * Ge::NEXTOBJ; t += CG) {
      int o = t / E, sl = t - o * E; double* s = sm + sl * Ge::SLOT; const double* pm = s + Ge::O_PM;      // object-major: few branches per warp
      if (o < 2 * NG) {                            // photon i, helicity bit hb (0: +1, 1: -1): the block (eps0 - sigma.eps*) = [[m, -r], [-l, p]]
        int i = o >> 1, hb = o & 1; const double* k = pm + 4 * (i + 2);
        lcv<double> a = lightcone(conj4(polvec<double>(k[1], k[2], k[3], hb ? -1 : +1)));
        cx<double>* M = reinterpret_cast<cx<double>*>(s + Ge::O_EPS) + (i * 2 + hb) * 4;
        const cx<double> m0 = a.m, m1 = -a.r, m2 = -a.l, m3 = a.p;
        M[0] = m0; M[1] = m1; M[2] = m2; M[3] = m3;
        // psi_{i}(hb) = q-slash / q^2 eps-slash* psi_{},  psi_{} = lower components of u(p2, +),  q = p2 - k_i
        const double* p = pm + 4; chi_pair<double> x = make_chi<double>(p[1], p[2], p[3]);
        spn<double> u = spinor_u<double>(x, make_shell<double>(p[0], 0.0), +1);
        cx<double> a0 = m0 * u.c[2]; cfma(a0, m1, u.c[3]);
        cx<double> a1 = m2 * u.c[2]; cfma(a1, m3, u.c[3]);
        const double q[4] = {p[0] - k[0], p[1] - k[1], p[2] - k[2], p[3] - k[3]}; const double sc = 1.0 / mdot_rr(q, q);
        const double qp = (q[0] + q[3]) * sc, qm = (q[0] - q[3]) * sc; const cx<double> qr = mk<double>(q[1] * sc, -q[2] * sc), ql = mk<double>(q[1] * sc, q[2] * sc);
        cx<double> o0 = qp * a0; cfma(o0, qr, a1);
        cx<double> o1 = qm * a1; cfma(o1, ql, a0);
        cx<double>* T = reinterpret_cast<cx<double>*>(s + Ge::O_PSI); const int e = s_off[1 << i] + hb;
        T[e] = o0; T[NENT + e] = o1;
      } else if (o == 2 * NG) {                    // (slot of the empty current: nothing left to store)
      } else if (o == 2 * NG + 1) {                // row of vbar(p1, -) that meets upper components: (lower components of v)^*
        const double* p = pm; chi_pair<double> x = make_chi<double>(p[1], p[2], p[3]);
        spn<double> v = spinor_v<double>(x, make_shell<double>(p[0], 0.0), -1);
        cx<double>* W = reinterpret_cast<cx<double>*>(s + Ge::O_W); W[0] = conj(v.c[2]); W[1] = conj(v.c[3]);
      } else {                                     // q_S = p2 - K_S
        int S = o - 2 * NG - 2; double q[4] = {pm[4], pm[5], pm[6], pm[7]};
#pragma unroll
        for (int i = 0; i < NG; i++) if (S >> i & 1) { for (int mu = 0; mu < 4; mu++) q[mu] -= pm[4 * (i + 2) + mu]; }
        const double sc = (S != 0 && S != NSUB - 1) ? 1.0 / mdot_rr(q, q) : 0.0;
        double* Q = s + Ge::O_Q + 4 * S; Q[0] = q[0] * sc; Q[1] = q[1] * sc; Q[2] = q[2] * sc; Q[3] = q[3] * sc;
      }
    }
    gsync<CG, NTH>();
    // ---- a3: current levels k = 2 .. NG-1 ----
    photon_levels<NG, 2, VBL, E, CG, NTH>(sm, s_sub, s_off, s_child, s_lvl, tid);
    // ---- a4-a7: the 2^NG amplitudes of an event, 2^VF per thread (all helicities of the last VF photons) in 2^(NG-VF) consecutive
    //             lanes, helicity sum in a fixed order (thread, then a fixed shuffle tree), eq. 3 ----
    constexpr int VF = VBF < NG ? VBF : NG, NFX = 1 << (NG - VF), NFIN = E * NFX, NFIN_W = (NFIN + 31) / 32 * 32;   // whole warps take part in the shuffles
    for (int t0 = tid; t0 < NFIN_W; t0 += CG) {
      const bool live = t0 < NFIN; const int t = live ? t0 : 0;
      const int sl = t / NFX; const unsigned v = t & (NFX - 1);
      const double* s = sm + sl * Ge::SLOT;
      cx<double> acc[1 << VF][2];
      photon_accumulate<NG, NG, VF>(acc, s, s_child, NSUB - 1, v);
      const cx<double>* W = reinterpret_cast<const cx<double>*>(s + Ge::O_W);
      const cx<double> w0 = W[0], w1 = W[1];
      double part = 0.0;
#pragma unroll
      for (int u = 0; u < (1 << VF); u++) { cx<double> amp = w0 * acc[u][0]; cfma(amp, w1, acc[u][1]); part += norm2(amp); }
#pragma unroll
      for (int d = NFX / 2; d >= 1; d >>= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
      const long long ev = ev0 + sl;
      if (live && v == 0 && ev < nev) {
        const double a = part * P.fac[0], Wt = __ldg(wgt + ev);
        me_old[ev] = a;
        for (int k = 1; k < P.nsets; k++) {
          const double b = part * P.fac[k];
          me_new[(size_t)(k - 1) * ostride + ev] = b; w_new[(size_t)(k - 1) * ostride + ev] = Wt * (b / a);
        }
      }
    }
    gsync<CG, NTH>();
  }
}

// Algorithmic flops per event (FMA = 2, MUL = ADD = 1): a level-k task is k 2x2 complex blocks (16 FMA each), the (q0 + sigma.q)
// block with the propagator folded in (8 FMA + 4 MUL for the block, 6 MUL + 2 ADD for its scaled entries); a final amplitude is NG
// blocks, the row contraction (6 FMA + 2 MUL) and the square (1 FMA + 1 MUL); externals ~30 per polarisation block, ~25 per
// spinor, ~12 per subset momentum (n = 5: 33 078 against 33 075 counted by ncu).
static double photon_flops_per_event(int ng) {
  double f = 0;
  for (int k = 1; k < ng; k++) f += (double)binom(ng, k) * (1 << k) * (32.0 * k + 16 + 4 + 8);
  f += (double)(1 << ng) * (32.0 * ng + 14 + 3);
  f += 2.0 * ng * 30 + 2 * 25 + (1 << ng) * 12.0;
  return f;
}

// host side.  Round 1 (one or two variants per thread, slot-major lanes): every E / threads / cooperating-group variant landed at
// 0.36-0.40 ms for 131072 e+e- -> 5 gamma events, bound by the shared-memory data pipe (82 % of its wavefront peak, 26 % of the
// wavefronts bank conflicts; an LDS.128 costs four wavefronts, and a 2x2 block product read 4.2 of them for its 16 DFMAs).
// Round 2, measured on B200 (ms for the same events): odd slot stride + event-fastest lanes, no bank conflict left: 0.356 -> 0.320;
// 2^VB variants per thread (photon_accumulate): 0.312 at VB = 2 (VB = 3 leaves too few busy warps: 0.36-0.39); momenta prefetched
// into registers and level 1 formed with the externals (two phases and their barriers gone): 0.296; two-buffer current storage +
// propagator folded into q_S + momenta on the tail of buffer B (6.8 KB per event): 4 CTAs of 8 events x 160 threads 0.272 (128: 0.272,
// 96: 0.309, 192: 0.299, 256: 0.32, register-limited to 3 CTAs); 2 CTAs of 16 events x 320 threads 0.265 (288: 0.303, 352: 0.286, 384: 0.284);
// 4 events per CTA (a quarter-warp then holds two tasks, conflicts return): 0.33-0.41; warp-private groups of 8 events (no CTA barriers, four
// warps per SM fit): 0.37-0.43; three variant bits at level 4: 0.28-0.37.
constexpr int RWGT_PH_E = 16;
constexpr int RWGT_PH_NTH = 320;
constexpr int RWGT_PH_VB = 22;
constexpr int RWGT_PH_VBF = 1;
constexpr int PH_E = RWGT_PH_E, PH_NTH = RWGT_PH_NTH, PH_CG = RWGT_PH_NTH, PH_VB = RWGT_PH_VB, PH_VBF = RWGT_PH_VBF;
template <int NG> constexpr size_t photon_smem() { return sizeof(double) * (PH_NTH / PH_CG) * PH_E * PhGeo<NG>::SLOT; }
// once per handle at rwgt_create, on the handle's device (the attribute belongs to the device's copy of the function)
static cudaError_t photon_prepare(int ng) {
  switch (ng) {
    case 2: return cudaFuncSetAttribute(epem_photons_kernel<2, PH_E, PH_CG, PH_NTH, PH_VB, PH_VBF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)photon_smem<2>());
    case 3: return cudaFuncSetAttribute(epem_photons_kernel<3, PH_E, PH_CG, PH_NTH, PH_VB, PH_VBF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)photon_smem<3>());
    case 4: return cudaFuncSetAttribute(epem_photons_kernel<4, PH_E, PH_CG, PH_NTH, PH_VB, PH_VBF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)photon_smem<4>());
    default: return cudaFuncSetAttribute(epem_photons_kernel<5, PH_E, PH_CG, PH_NTH, PH_VB, PH_VBF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)photon_smem<5>());
  }
}
template <int NG> static cudaError_t photon_launch_n(int sm_count, cudaStream_t st, const double* mom, const double* w, double* a, double* b, double* o,
                                                     long long nev, long long stride, long long ostride, const PhotonParams& P) {
  constexpr int GPB = PH_NTH / PH_CG;
  const size_t smem = photon_smem<NG>();
  const long long ngroups = (nev + PH_E - 1) / PH_E, nblocks = (ngroups + GPB - 1) / GPB;
  const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(2048 / PH_NTH, (size_t)(227 * 1024) / (smem + 2048)));
  const int grid = (int)std::min<long long>(nblocks, (long long)sm_count * per_sm);
  epem_photons_kernel<NG, PH_E, PH_CG, PH_NTH, PH_VB, PH_VBF><<<grid, PH_NTH, smem, st>>>(mom, w, a, b, o, nev, stride, ostride, P);
  return cudaSuccess;
}
static cudaError_t photon_launch(int ng, int sm_count, cudaStream_t st, const double* mom, const double* w, double* a, double* b, double* o,
                                 long long nev, long long stride, long long ostride, const PhotonParams& P) {
  switch (ng) {
    case 2: return photon_launch_n<2>(sm_count, st, mom, w, a, b, o, nev, stride, ostride, P);
    case 3: return photon_launch_n<3>(sm_count, st, mom, w, a, b, o, nev, stride, ostride, P);
    case 4: return photon_launch_n<4>(sm_count, st, mom, w, a, b, o, nev, stride, ostride, P);
    default: return photon_launch_n<5>(sm_count, st, mom, w, a, b, o, nev, stride, ostride, P);
  }
}

}  // namespace rwgt
