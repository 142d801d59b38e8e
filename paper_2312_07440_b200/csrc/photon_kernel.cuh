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

template <int NG> struct PhGeo {
  static constexpr int NSUB = 1 << NG, NENT = ipow(3, NG) - NSUB;          // stored currents: every subset but the full one
  static constexpr int NEXTOBJ = 2 * NG + 2 + NSUB;                        // external tasks per event
  // doubles per event slot
  static constexpr int O_PM = 0, O_EPS = O_PM + (NG + 2) * 4, O_Q = O_EPS + NG * 2 * 8, O_IQ2 = O_Q + NSUB * 4,
                       O_W = O_IQ2 + NSUB, O_PSI = O_W + 4, SLOT = O_PSI + 4 * NENT;
};

// barrier over the cooperating group: the whole CTA (CG == NTH) or one warp (CG == 32)
template <int CG, int NTH> __device__ __forceinline__ void gsync() { if constexpr (CG == NTH) __syncthreads(); else __syncwarp(); }

// y += B x for a 2x2 complex block B = (m[0] m[1]; m[2] m[3])
__device__ __forceinline__ void block_acc(cx<double>& y0, cx<double>& y1, const cx<double>* m, cx<double> x0, cx<double> x1) {
  cfma(y0, m[0], x0); cfma(y0, m[1], x1); cfma(y1, m[2], x0); cfma(y1, m[3], x1);
}
// One level of the recursion: all currents of K photons (K compile-time: constant divisors, branch-free member loop).
// A thread evaluates BOTH helicities of the subset's last member: for that member the spinor is shared and the block differs,
// for every other member the block is shared and the two spinors are neighbours (entry + 2^(K-2)); this halves the shared-memory
// wavefronts per block product, which is what bounds this kernel.
// s_child[S][r] = (first entry of S without its r-th member) << 8 | (2 * that member's label).
template <int NG, int K, int E, int CG, int NTH>
__device__ __forceinline__ void photon_level(double* sm, const unsigned char* s_sub, const unsigned short* s_off, const unsigned* s_child, int first_sub, int tid) {
  typedef PhGeo<NG> Ge;
  constexpr int NENT = Ge::NENT, KL = K - 1, per = binom(NG, K) << KL;
  for (int t = tid; t < E * per; t += CG) {
    const int sl = t / per, o = t - sl * per; const int S = s_sub[first_sub + (o >> KL)]; const unsigned v = o & ((1u << KL) - 1u);
    double* s = sm + sl * Ge::SLOT;
    const cx<double>* M = reinterpret_cast<const cx<double>*>(s + Ge::O_EPS);
    cx<double>* T = reinterpret_cast<cx<double>*>(s + Ge::O_PSI);
    cx<double> a0 = mk<double>(0, 0), a1 = mk<double>(0, 0), b0 = mk<double>(0, 0), b1 = mk<double>(0, 0);
    constexpr int HI = KL > 0 ? 1 << (KL > 0 ? KL - 1 : 0) : 0;      // entry distance of the two spinors
#pragma unroll
    for (int r = 0; r < KL; r++) {                 // members below the last one: one block, two spinors
      const unsigned ch = s_child[S * NG + r];
      const unsigned hb = (v >> r) & 1u, vp = (v & ((1u << r) - 1u)) | ((v >> (r + 1)) << r);
      const int e = (int)(ch >> 8) + (int)vp; const cx<double>* m = M + ((ch & 0xffu) + hb) * 4;
      const cx<double> m0 = ldc(m), m1 = ldc(m + 1), m2 = ldc(m + 2), m3 = ldc(m + 3);
      const cx<double> x0 = ldc(T + e), x1 = ldc(T + NENT + e), y0 = ldc(T + e + HI), y1 = ldc(T + NENT + e + HI);
      cfma(a0, m0, x0); cfma(a0, m1, x1); cfma(a1, m2, x0); cfma(a1, m3, x1);
      cfma(b0, m0, y0); cfma(b0, m1, y1); cfma(b1, m2, y0); cfma(b1, m3, y1);
    }
    {                                              // the last member: one spinor, two blocks
      const unsigned ch = s_child[S * NG + KL];
      const int e = (int)(ch >> 8) + (int)v; const cx<double>* m = M + (ch & 0xffu) * 4;
      const cx<double> x0 = ldc(T + e), x1 = ldc(T + NENT + e);
      block_acc(a0, a1, m, x0, x1); block_acc(b0, b1, m + 4, x0, x1);
    }
    const double* q = s + Ge::O_Q + 4 * S; const double sc = s[Ge::O_IQ2 + S];
    const double qp = (q[0] + q[3]) * sc, qm = (q[0] - q[3]) * sc; const cx<double> qr = mk<double>(q[1] * sc, -q[2] * sc), ql = mk<double>(q[1] * sc, q[2] * sc);
    cx<double> o0 = qp * a0; cfma(o0, qr, a1);           // (q0 + sigma.q) = [[q+, qr], [ql, q-]]
    cx<double> o1 = qm * a1; cfma(o1, ql, a0);
    cx<double> u0 = qp * b0; cfma(u0, qr, b1);
    cx<double> u1 = qm * b1; cfma(u1, ql, b0);
    const int eo = s_off[S] + (int)v;
    stc(T + eo, o0); stc(T + NENT + eo, o1); stc(T + eo + (1 << KL), u0); stc(T + NENT + eo + (1 << KL), u1);
  }
  gsync<CG, NTH>();
}
template <int NG, int K, int E, int CG, int NTH>
__device__ __forceinline__ void photon_levels(double* sm, const unsigned char* s_sub, const unsigned short* s_off, const unsigned* s_child, const unsigned char* s_lvl, int tid) {
  if constexpr (K < NG) {
    photon_level<NG, K, E, CG, NTH>(sm, s_sub, s_off, s_child, s_lvl[K], tid);
    photon_levels<NG, K + 1, E, CG, NTH>(sm, s_sub, s_off, s_child, s_lvl, tid);
  }
}

// E events per cooperating group of CG threads (CG == NTH: the CTA, levels separated by __syncthreads; CG == 32: each warp works on
// its own E events and only ever waits for itself)
template <int NG, int E, int CG, int NTH>
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
    int o = 0; for (int S = 0; S < NSUB; S++) { s_off[S] = (unsigned short)o; o += 1 << __popc(S); }
    int j = 0; for (int k = 0; k <= NG; k++) { s_lvl[k] = (unsigned char)j; for (int S = 0; S < NSUB; S++) if (__popc(S) == k) s_sub[j++] = (unsigned char)S; }
    s_lvl[NG + 1] = (unsigned char)j;
    for (int S = 0; S < NSUB; S++) { int r = 0; for (int i = 0; i < NG; i++) if (S >> i & 1) s_child[S * NG + r++] = ((unsigned)s_off[S ^ (1 << i)] << 8) | (unsigned)(2 * i); }
  }
  __syncthreads();
  const long long ngroups = (nev + E - 1) / E;
  constexpr int GPB = NTH / CG;                                      // groups per CTA
  for (long long grp = (long long)blockIdx.x * GPB + (CG == NTH ? 0 : threadIdx.x >> 5); grp < ngroups; grp += (long long)gridDim.x * GPB) {
    const long long ev0 = grp * E;
    // ---- a1: momenta (coalesced over the events of the group) ----
    for (int t = tid; t < E * next * 4; t += CG) {
      int sl = t % E, comp = t / E; long long ev = ev0 + sl; if (ev >= nev) ev = nev - 1;
      sm[sl * Ge::SLOT + Ge::O_PM + comp] = __ldg(mom + (size_t)comp * stride + ev);
    }
    gsync<CG, NTH>();
    // ---- a2: external wavefunctions, momenta and inverse virtualities of the electron line ----
    for (int t = tid; t < E * Ge::NEXTOBJ; t += CG) {
      int o = t / E, sl = t - o * E; double* s = sm + sl * Ge::SLOT; const double* pm = s + Ge::O_PM;      // object-major: few branches per warp
      if (o < 2 * NG) {                            // photon i, helicity bit hb (0: +1, 1: -1): the block (eps0 - sigma.eps*) = [[m, -r], [-l, p]]
        int i = o >> 1, hb = o & 1; const double* k = pm + 4 * (i + 2);
        lcv<double> a = lightcone(conj4(polvec<double>(k[1], k[2], k[3], hb ? -1 : +1)));
        cx<double>* M = reinterpret_cast<cx<double>*>(s + Ge::O_EPS) + (i * 2 + hb) * 4;
        M[0] = a.m; M[1] = -a.r; M[2] = -a.l; M[3] = a.p;
      } else if (o == 2 * NG) {                    // psi_{} = lower components of u(p2, +)
        const double* p = pm + 4; chi_pair<double> x = make_chi<double>(p[1], p[2], p[3]);
        spn<double> u = spinor_u<double>(x, make_shell<double>(p[0], 0.0), +1);
        cx<double>* T = reinterpret_cast<cx<double>*>(s + Ge::O_PSI); T[0] = u.c[2]; T[NENT] = u.c[3];
      } else if (o == 2 * NG + 1) {                // row of vbar(p1, -) that meets upper components: (lower components of v)^*
        const double* p = pm; chi_pair<double> x = make_chi<double>(p[1], p[2], p[3]);
        spn<double> v = spinor_v<double>(x, make_shell<double>(p[0], 0.0), -1);
        cx<double>* W = reinterpret_cast<cx<double>*>(s + Ge::O_W); W[0] = conj(v.c[2]); W[1] = conj(v.c[3]);
      } else {                                     // q_S = p2 - K_S
        int S = o - 2 * NG - 2; double q[4] = {pm[4], pm[5], pm[6], pm[7]};
#pragma unroll
        for (int i = 0; i < NG; i++) if (S >> i & 1) { for (int mu = 0; mu < 4; mu++) q[mu] -= pm[4 * (i + 2) + mu]; }
        double* Q = s + Ge::O_Q + 4 * S; Q[0] = q[0]; Q[1] = q[1]; Q[2] = q[2]; Q[3] = q[3];
        s[Ge::O_IQ2 + S] = (S != 0 && S != NSUB - 1) ? 1.0 / mdot_rr(q, q) : 0.0;
      }
    }
    gsync<CG, NTH>();
    // ---- a3: current levels k = 1 .. NG-1 ----
    photon_levels<NG, 1, E, CG, NTH>(sm, s_sub, s_off, s_child, s_lvl, tid);
    // ---- a4-a7: the 2^NG amplitudes of an event, two per thread (both helicities of the last photon) in 2^(NG-1) consecutive lanes,
    //             helicity sum by a fixed shuffle tree, eq. 3 ----
    constexpr int NFIN = E << (NG - 1), NFIN_W = (NFIN + 31) / 32 * 32;       // whole warps take part in the shuffles
    for (int t0 = tid; t0 < NFIN_W; t0 += CG) {
      const bool live = t0 < NFIN; const int t = live ? t0 : 0;
      const int sl = t >> (NG - 1); const unsigned v = t & (NSUB / 2 - 1);
      const double* s = sm + sl * Ge::SLOT;
      const cx<double>* M = reinterpret_cast<const cx<double>*>(s + Ge::O_EPS);
      const cx<double>* T = reinterpret_cast<const cx<double>*>(s + Ge::O_PSI);
      cx<double> a0 = mk<double>(0, 0), a1 = mk<double>(0, 0), b0 = mk<double>(0, 0), b1 = mk<double>(0, 0);
#pragma unroll
      for (int i = 0; i < NG - 1; i++) {
        const unsigned hb = (v >> i) & 1u, vp = (v & ((1u << i) - 1u)) | ((v >> (i + 1)) << i);
        const int e = (int)(s_child[(NSUB - 1) * NG + i] >> 8) + (int)vp; const cx<double>* m = M + (i * 2 + hb) * 4;
        const cx<double> m0 = ldc(m), m1 = ldc(m + 1), m2 = ldc(m + 2), m3 = ldc(m + 3);
        const cx<double> x0 = ldc(T + e), x1 = ldc(T + NENT + e), y0 = ldc(T + e + (1 << (NG - 2))), y1 = ldc(T + NENT + e + (1 << (NG - 2)));
        cfma(a0, m0, x0); cfma(a0, m1, x1); cfma(a1, m2, x0); cfma(a1, m3, x1);
        cfma(b0, m0, y0); cfma(b0, m1, y1); cfma(b1, m2, y0); cfma(b1, m3, y1);
      }
      {
        const int e = (int)(s_child[(NSUB - 1) * NG + NG - 1] >> 8) + (int)v; const cx<double>* m = M + (NG - 1) * 2 * 4;
        const cx<double> x0 = ldc(T + e), x1 = ldc(T + NENT + e);
        block_acc(a0, a1, m, x0, x1); block_acc(b0, b1, m + 4, x0, x1);
      }
      const cx<double>* W = reinterpret_cast<const cx<double>*>(s + Ge::O_W);
      cx<double> amp0 = W[0] * a0; cfma(amp0, W[1], a1);
      cx<double> amp1 = W[0] * b0; cfma(amp1, W[1], b1);
      double part = norm2(amp0) + norm2(amp1);
#pragma unroll
      for (int d = NSUB / 4; d >= 1; d >>= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
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

// host side: E = 8 events per CTA, 256 threads (the 8 x 32 final amplitudes of n = 5 are one task per thread), 3 CTAs per SM.
// Measured on B200 (n = 5, 131072 events), one variant per thread: E/threads 16/512 0.503 ms, 12/384 0.449, 8/256 0.410, 6/192 0.405,
// 4/128 0.408; two variants per thread: 8/256 0.398, 6/128 0.401, 12/256 0.421, 8/128 0.428, 16/256 0.565; warp-cooperative groups
// (CG = 32, no CTA barriers) with E events per warp / threads per CTA: 2/128 0.414, 2/64 0.415, 1/128 0.474, 4/64 0.608.  Every variant
// lands at ~0.40 ms: the shared-memory data pipe (72-75 % of its wavefront peak; an LDS.128 costs four wavefronts whether or not lanes
// share addresses, and every 2x2 block product reads 6 of them for 16 DFMAs) is the bound, not barriers or occupancy.
#ifndef RWGT_PH_E
#define RWGT_PH_E 8
#define RWGT_PH_CG 256
#define RWGT_PH_NTH 256
#endif
constexpr int PH_E = RWGT_PH_E, PH_CG = RWGT_PH_CG, PH_NTH = RWGT_PH_NTH;
template <int NG> constexpr size_t photon_smem() { return sizeof(double) * (PH_NTH / PH_CG) * PH_E * PhGeo<NG>::SLOT; }
// once per handle at rwgt_create, on the handle's device (the attribute belongs to the device's copy of the function)
static cudaError_t photon_prepare(int ng) {
  switch (ng) {
    case 2: return cudaFuncSetAttribute(epem_photons_kernel<2, PH_E, PH_CG, PH_NTH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)photon_smem<2>());
    case 3: return cudaFuncSetAttribute(epem_photons_kernel<3, PH_E, PH_CG, PH_NTH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)photon_smem<3>());
    case 4: return cudaFuncSetAttribute(epem_photons_kernel<4, PH_E, PH_CG, PH_NTH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)photon_smem<4>());
    default: return cudaFuncSetAttribute(epem_photons_kernel<5, PH_E, PH_CG, PH_NTH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)photon_smem<5>());
  }
}
template <int NG> static cudaError_t photon_launch_n(int sm_count, cudaStream_t st, const double* mom, const double* w, double* a, double* b, double* o,
                                                     long long nev, long long stride, long long ostride, const PhotonParams& P) {
  constexpr int GPB = PH_NTH / PH_CG;
  const size_t smem = photon_smem<NG>();
  const long long ngroups = (nev + PH_E - 1) / PH_E, nblocks = (ngroups + GPB - 1) / GPB;
  const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(2048 / PH_NTH, (size_t)(227 * 1024) / (smem + 2048)));
  const int grid = (int)std::min<long long>(nblocks, (long long)sm_count * per_sm);
  epem_photons_kernel<NG, PH_E, PH_CG, PH_NTH><<<grid, PH_NTH, smem, st>>>(mom, w, a, b, o, nev, stride, ostride, P);
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
