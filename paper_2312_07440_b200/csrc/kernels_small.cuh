// kernels_small.cuh — one-event-per-thread FP64 kernels for the two 2->2 processes.
//   cfg 1  e+ e- -> gamma/Z -> mu+ mu-   (2 diagrams, ncol = 1)
//   cfg 2  g g -> t tbar                 (SURVEY §8(c) C5/C6 with n = 2; 3 diagrams, ncol = 2)
// Steps a1-a7 of SURVEY §8(a) in one launch: coalesced SoA loads, external wavefunctions,
// vertices, colour form, helicity sum, eq. 3, three coalesced stores.
#pragma once
#include "../../include/rwgt.h"
#include "rwgt_math.cuh"

namespace rwgt {

// ------------------------------------------------------------------------------------- cfg 1
struct EpemSet {          // per parameter set, prepared on the host
  double e2;              // e^2 = 4 pi alpha
  double gz2;             // g_Z^2 = e^2 / (sW^2 cW^2)
  double gL, gR;          // -1/2 + sW^2, sW^2
  double mZ2, mZGZ;       // mZ^2, mZ*GammaZ
};
constexpr int SMALL_NSMAX = 1 + RWGT_MAX_SETS;     // the old set plus up to RWGT_MAX_SETS new ones
struct EpemParams { EpemSet set[SMALL_NSMAX]; int nsets; };

// Massless leptons: only the 4 helicity combinations with opposite helicities on each fermion line
// are non-zero (tests check the oracle's full 16-term sum against this, reading Q5).
constexpr int RWGT_EPEM_BS = 128;
constexpr int RWGT_EPEM_MINB = 6;
__global__ void __launch_bounds__(RWGT_EPEM_BS, RWGT_EPEM_MINB) epem_mupmum_kernel(const double* __restrict__ mom, const double* __restrict__ wgt,
                                                          double* __restrict__ me_old, double* __restrict__ me_new,
                                                          double* __restrict__ w_new, long long n, long long stride, long long ostride, EpemParams P) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double p[4][4];
#pragma unroll
  for (int ip = 0; ip < 4; ip++)
#pragma unroll
    for (int mu = 0; mu < 4; mu++) p[ip][mu] = __ldg(mom + (size_t)(ip * 4 + mu) * stride + i);
  double W = __ldg(wgt + i);
  double q[4] = {p[0][0] + p[1][0], p[0][1] + p[1][1], p[0][2] + p[1][2], p[0][3] + p[1][3]};
  double s = mdot_rr(q, q);
  // unnormalised two-spinors (|chi|^2 = n2): each of the four enters every |amplitude|^2 exactly once, so the four normalisations are
  // one division at the end instead of four reciprocal square roots
  chi_pair<double> x1 = make_chi_raw(p[0][1], p[0][2], p[0][3]), x2 = make_chi_raw(p[1][1], p[1][2], p[1][3]);
  chi_pair<double> x3 = make_chi_raw(p[2][1], p[2][2], p[2][3]), x4 = make_chi_raw(p[3][1], p[3][2], p[3][3]);
  // massless legs: spinor normalisation sqrt(2E), energy from the input and mass parameter 0 (reading Q8 / DESIGN.md R8); the four
  // normalisations enter every |amplitude|^2 as the product of the four 2E: no square root
  const double nrm = 16.0 * ((p[0][0] * p[1][0]) * (p[2][0] * p[3][0])) / ((x1.n2 * x2.n2) * (x3.n2 * x4.n2));
  // electron line vbar(p1) gamma^mu u(p2): L = (lam1,lam2) = (+,-), R = (-,+); muon line ubar(p4) gamma^mu v(p3) likewise.  The four
  // current contractions J_e . J_mu are done by the Fierz identities of the Pauli matrices (sigma^mu = (1, sigma), sigmabar^mu = (1, -sigma)):
  //   (a^+ sigmabar^mu b)(c^+ sigmabar_mu d) = (a^+ sigma^mu b)(c^+ sigma_mu d) = 2 conj(a ^ c) (b ^ d),   x ^ y = x_1 y_2 - x_2 y_1,
  //   (a^+ sigmabar^mu b)(c^+ sigma_mu d) = 2 (a^+ d)(c^+ b),
  // i.e. every helicity amplitude is a product of two two-spinor products.
  auto wedge = [](const cx<double>* x, const cx<double>* y) { cx<double> r = x[0] * y[1]; cfms(r, x[1], y[0]); return norm2(r); };
  auto inner = [](const cx<double>* x, const cx<double>* y) { cx<double> r = conj(x[0]) * y[0]; cfma(r, conj(x[1]), y[1]); return norm2(r); };
  const double c2 = 4.0 * nrm;
  double dLL = wedge(x1.m, x4.m) * wedge(x2.m, x3.m) * c2, dRR = wedge(x1.p, x4.p) * wedge(x2.p, x3.p) * c2;
  double dLR = inner(x1.m, x3.p) * inner(x4.p, x2.m) * c2, dRL = inner(x1.p, x3.m) * inner(x4.m, x2.p) * c2;
  double me0 = 0;
#pragma unroll 1
  for (int k = 0; k < P.nsets; k++) {
    const EpemSet& S = P.set[k];
    // photon e^2/s (Q_e Q_mu = +1) plus Z g_Z^2 g_a g_b / (s - mZ^2 + i mZ GammaZ)
    double dr = s - S.mZ2, di = S.mZGZ, inv = 1.0 / (dr * dr + di * di);
    double zr = S.gz2 * dr * inv, zi = -S.gz2 * di * inv, ph = S.e2 / s;
    double fLL = norm2(mk<double>(ph + S.gL * S.gL * zr, S.gL * S.gL * zi));
    double fLR = norm2(mk<double>(ph + S.gL * S.gR * zr, S.gL * S.gR * zi));
    double fRR = norm2(mk<double>(ph + S.gR * S.gR * zr, S.gR * S.gR * zi));
    const double me = 0.25 * (fLL * dLL + fLR * (dLR + dRL) + fRR * dRR);
    if (k == 0) { me0 = me; me_old[i] = me; }
    else { me_new[(size_t)(k - 1) * ostride + i] = me; w_new[(size_t)(k - 1) * ostride + i] = W * (me / me0); }
  }
}

// ------------------------------------------------------------------------------------- cfg 2
struct GGttxParams {
  double mt[SMALL_NSMAX];   // top mass per set
  double fac[SMALL_NSMAX];  // g_s^4 / 256 per set (averaging denominator D = 4*64)
  double s3[SMALL_NSMAX];   // ggg_scale per set
  int nsets;                // 1 + number of new sets
  int two_pass;             // masses differ: evaluate each set with its own mass
};

// Helicity-summed colour forms for ONE mass and two values of the ggg scale.
//   M = i g_s^2 [ (T^a T^b)(X12 + s3 Y) + (T^b T^a)(X21 - s3 Y) ]
//   X12 = ubar e1-slash Psi(2), Psi(i) = -(q_i-slash + m) e_i-slash v / (q_i^2 - m^2), q_i = k_i - p_tbar
//   Y   = -(1/s) ubar L3-slash(e1,k1;e2,k2) v
// Parity (|M_{-h}|^2 = |M_h|^2, tests/test_oracle_pins.py) halves the helicity loop: lam1 = +1 only, x2.
__device__ __forceinline__ void ggttx_sums(const double (*p)[4], double m, double sa, double sb, double& sum_a, double& sum_b) {
  const double* k1 = p[0]; const double* k2 = p[1];
  double q1[4], q2[4], kk[4];
#pragma unroll
  for (int mu = 0; mu < 4; mu++) { q1[mu] = k1[mu] - p[3][mu]; q2[mu] = k2[mu] - p[3][mu]; kk[mu] = k1[mu] + k2[mu]; }
  double m2 = m * m;
  double d1 = -1.0 / (mdot_rr(q1, q1) - m2), d2 = -1.0 / (mdot_rr(q2, q2) - m2), ds = -1.0 / mdot_rr(kk, kk);
  chi_pair<double> xt = make_chi_raw(p[2][1], p[2][2], p[2][3]), xb = make_chi_raw(p[3][1], p[3][2], p[3][3]);
  const shell<double> nt = make_shell(p[2][0], m, xt.n2), nb = make_shell(p[3][0], m, xb.n2);
  sum_a = 0; sum_b = 0;
  const int l1 = +1;
  vec4<double> e1 = polvec(k1[1], k1[2], k1[3], l1);
#pragma unroll
  for (int i2 = 0; i2 < 2; i2++) {
    int l2 = i2 ? -1 : +1;
    vec4<double> e2 = polvec(k2[1], k2[2], k2[3], l2);
    vec4<double> l3; for (int mu = 0; mu < 4; mu++) l3.c[mu] = mk<double>(0, 0);
    L3_acc(l3, e1, k1, e2, k2);
    for (int mu = 0; mu < 4; mu++) l3.c[mu] = ds * l3.c[mu];
#pragma unroll
    for (int ib = 0; ib < 2; ib++) {
      spn<double> v = spinor_v(xb, nb, ib ? -1 : +1);
      spn<double> psi1 = slash_r_plus_m(q1, m, slash_c(e1, v)), psi2 = slash_r_plus_m(q2, m, slash_c(e2, v));
      spn<double> c12 = slash_c(e1, psi2), c21 = slash_c(e2, psi1), cy = slash_c(l3, v);
#pragma unroll
      for (int it = 0; it < 2; it++) {
        spn<double> ub = bar(spinor_u(xt, nt, it ? -1 : +1));
        cx<double> X12 = d2 * rowcol(ub, c12), X21 = d1 * rowcol(ub, c21), Y = rowcol(ub, cy);
        cx<double> A1 = X12, A2 = X21; rfma(A1, sa, Y); rfma(A2, -sa, Y);
        sum_a += 16.0 * (norm2(A1) + norm2(A2)) - 4.0 * (A1.re * A2.re + A1.im * A2.im);
        cx<double> B1 = X12, B2 = X21; rfma(B1, sb, Y); rfma(B2, -sb, Y);
        sum_b += 16.0 * (norm2(B1) + norm2(B2)) - 4.0 * (B1.re * B2.re + B1.im * B2.im);
      }
    }
  }
  // colour matrix (16,-2;-2,16)/3, parity factor 2
  sum_a *= 2.0 / 3.0; sum_b *= 2.0 / 3.0;
}

// 168 registers with ~1.3 KB of spills at 12 warps per SM beats 254 registers without spills at 8 warps (0.171 -> 0.150 ms for 2^20 events):
// the kernel is bound by dependent-issue latency (sqrt / division chains), not by the L1-resident spill traffic
constexpr int RWGT_GGTTX_BS = 128;
constexpr int RWGT_GGTTX_MINB = 3;
constexpr int GGTTX_BS = RWGT_GGTTX_BS;
__global__ void __launch_bounds__(RWGT_GGTTX_BS, RWGT_GGTTX_MINB) gg_ttx_kernel(const double* __restrict__ mom, const double* __restrict__ wgt, const int* __restrict__ idx,
                                                     double* __restrict__ me_old, double* __restrict__ me_new,
                                                     double* __restrict__ w_new, long long n, long long stride, long long /*ostride*/, GGttxParams P) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (idx) i = idx[i];                      // multiprocess handles: the events of this process inside a mixed list
  double p[4][4];
#pragma unroll
  for (int ip = 0; ip < 4; ip++)
#pragma unroll
    for (int mu = 0; mu < 4; mu++) p[ip][mu] = __ldg(mom + (size_t)(ip * 4 + mu) * stride + i);
  double W = __ldg(wgt + i);
  double a, b;
  if (!P.two_pass) ggttx_sums(p, P.mt[0], P.s3[0], P.s3[1], a, b);
  else { double t; ggttx_sums(p, P.mt[0], P.s3[0], P.s3[0], a, t); ggttx_sums(p, P.mt[1], P.s3[1], P.s3[1], t, b); }
  a *= P.fac[0]; b *= P.fac[1];
  me_old[i] = a; me_new[i] = b; w_new[i] = W * (b / a);
}

// K > 1 new sets of equal top mass: the 8 x 3 helicity amplitudes X12, X21, Y are formed once by the same fully unrolled code as
// in ggttx_sums and kept (registers / L1-resident local memory); every set is then one more pair of real FMAs and one more colour form
// per helicity (PAPER.md:87 step 7).  sums[k] for k < nsets.
__device__ __forceinline__ void ggttx_sums_multi(const double (*p)[4], double m, const double* s3, int nsets, double* sums) {
  const double* k1 = p[0]; const double* k2 = p[1];
  double q1[4], q2[4], kk[4];
#pragma unroll
  for (int mu = 0; mu < 4; mu++) { q1[mu] = k1[mu] - p[3][mu]; q2[mu] = k2[mu] - p[3][mu]; kk[mu] = k1[mu] + k2[mu]; }
  double m2 = m * m;
  double d1 = -1.0 / (mdot_rr(q1, q1) - m2), d2 = -1.0 / (mdot_rr(q2, q2) - m2), ds = -1.0 / mdot_rr(kk, kk);
  chi_pair<double> xt = make_chi_raw(p[2][1], p[2][2], p[2][3]), xb = make_chi_raw(p[3][1], p[3][2], p[3][3]);
  const shell<double> nt = make_shell(p[2][0], m, xt.n2), nb = make_shell(p[3][0], m, xb.n2);
  cx<double> aX12[8], aX21[8], aY[8];
  vec4<double> e1 = polvec(k1[1], k1[2], k1[3], +1);
#pragma unroll
  for (int i2 = 0; i2 < 2; i2++) {
    vec4<double> e2 = polvec(k2[1], k2[2], k2[3], i2 ? -1 : +1);
    vec4<double> l3; for (int mu = 0; mu < 4; mu++) l3.c[mu] = mk<double>(0, 0);
    L3_acc(l3, e1, k1, e2, k2);
    for (int mu = 0; mu < 4; mu++) l3.c[mu] = ds * l3.c[mu];
#pragma unroll
    for (int ib = 0; ib < 2; ib++) {
      spn<double> v = spinor_v(xb, nb, ib ? -1 : +1);
      spn<double> psi1 = slash_r_plus_m(q1, m, slash_c(e1, v)), psi2 = slash_r_plus_m(q2, m, slash_c(e2, v));
      spn<double> c12 = slash_c(e1, psi2), c21 = slash_c(e2, psi1), cy = slash_c(l3, v);
#pragma unroll
      for (int it = 0; it < 2; it++) {
        spn<double> ub = bar(spinor_u(xt, nt, it ? -1 : +1));
        const int h = (i2 * 2 + ib) * 2 + it;
        aX12[h] = d2 * rowcol(ub, c12); aX21[h] = d1 * rowcol(ub, c21); aY[h] = rowcol(ub, cy);
      }
    }
  }
#pragma unroll 1
  for (int k = 0; k < nsets; k++) {
    const double sk = s3[k]; double acc = 0;
#pragma unroll
    for (int h = 0; h < 8; h++) {
      cx<double> A1 = aX12[h], A2 = aX21[h]; rfma(A1, sk, aY[h]); rfma(A2, -sk, aY[h]);
      acc += 16.0 * (norm2(A1) + norm2(A2)) - 4.0 * (A1.re * A2.re + A1.im * A2.im);
    }
    sums[k] = acc * (2.0 / 3.0);
  }
}

__global__ void __launch_bounds__(128) gg_ttx_multi_kernel(const double* __restrict__ mom, const double* __restrict__ wgt, const int* __restrict__ idx,
                                                           double* __restrict__ me_old, double* __restrict__ me_new,
                                                           double* __restrict__ w_new, long long n, long long stride, long long ostride, GGttxParams P) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (idx) i = idx[i];
  double p[4][4];
#pragma unroll
  for (int ip = 0; ip < 4; ip++)
#pragma unroll
    for (int mu = 0; mu < 4; mu++) p[ip][mu] = __ldg(mom + (size_t)(ip * 4 + mu) * stride + i);
  const double W = __ldg(wgt + i);
  if (!P.two_pass) {
    double sums[SMALL_NSMAX];
    ggttx_sums_multi(p, P.mt[0], P.s3, P.nsets, sums);
    const double a = sums[0] * P.fac[0];
    me_old[i] = a;
#pragma unroll
    for (int k = 1; k < SMALL_NSMAX; k++) if (k < P.nsets) {
      const double b = sums[k] * P.fac[k];
      me_new[(size_t)(k - 1) * ostride + i] = b; w_new[(size_t)(k - 1) * ostride + i] = W * (b / a);
    }
  } else {                               // masses differ: one full evaluation per set
    double a = 0;
#pragma unroll 1
    for (int k = 0; k < P.nsets; k++) {
      double x, t; ggttx_sums(p, P.mt[k], P.s3[k], P.s3[k], x, t); x *= P.fac[k];
      if (k == 0) { a = x; me_old[i] = x; }
      else { me_new[(size_t)(k - 1) * ostride + i] = x; w_new[(size_t)(k - 1) * ostride + i] = W * (x / a); }
    }
  }
}

}  // namespace rwgt
