// qq_kernels.cuh — q(p1) qbar(p2) -> t(p3) tbar(p4) [+ g(p5)], FP64, one event per thread.
//
// A structurally different amplitude for the final states of cfgs 2 / 3 (last sentence: "reweighting between
// structurally different amplitude routines"; real emissions "can be treated as LO multiprocesses").  Massless
// light quark, rules of SURVEY C3.  Steps a1-a7 of SURVEY 8(a) in one launch.
//
// What is evaluated (couplings and the common factor -i stripped; e = eps*(p5), K_A = p1 + p2 = Q_A, K_g = -p5, Q_B = Q_A - p5):
//   j_A^mu = vbar(p2) gamma^mu u(p1)                        the light line as a gluon source
//   b_1^mu = vbar(p2) gamma^mu q1-slash e-slash u(p1) / q1^2,   q1 = p1 - p5          (gluon off the quark,     colour T^c T^a)
//   b_2^mu = vbar(p2) e-slash q2-slash gamma^mu u(p1) / q2^2,   q2 = p5 - p2          (gluon off the antiquark, colour T^a T^c)
//   l^mu   = L3^mu(j_A, K_A; e, K_g)                                                  (gluon off the virtual gluon)
//   a_1 = ubar(p3) (b_2-slash + r l-slash / Q_A^2) v(p4) / Q_B^2      coefficient of C_1 = (T^a T^c)_ji T^c_kl,   r = ggg_scale
//   a_2 = ubar(p3) (b_1-slash - r l-slash / Q_A^2) v(p4) / Q_B^2      coefficient of C_2 = (T^c T^a)_ji T^c_kl
//   a_3 = ubar(p3) e-slash (qt-slash + m) j_A-slash v(p4) / (Q_A^2 (qt^2 - m^2)),   qt = p3 + p5      C_3 = T^c_ji (T^a T^c)_kl
//   a_4 = ubar(p3) j_A-slash (qb-slash + m) e-slash v(p4) / (Q_A^2 (qb^2 - m^2)),   qb = -p4 - p5     C_4 = T^c_ji (T^c T^a)_kl
//   |M_h|^2 = g^6 sum_ab a_a G_ab conj(a_b),  G_ab = sum_colours C_a conj(C_b)  (host, exact SU(3) Fierz reduction)
// without the gluon: |M_h|^2 = 2 g^4 |ubar(p3) j_A-slash v(p4)|^2 / Q_A^4.
// Helicities: the massless line needs opposite q / qbar labels (the others vanish identically; pinned on the oracle), parity gives the
// configurations with lambda_q = - from those with + (x2).  Average 1/36.
#pragma once
#include "../../include/rwgt.h"
#include "rwgt_math.cuh"
#include "kernels_small.cuh"

namespace rwgt {

struct QQParams {
  double mt[SMALL_NSMAX];     // top mass per set
  double fac[SMALL_NSMAX];    // 2 g^(4 + 2 NG) / 36 (parity factor 2, averaging) per set; NG = 0 also carries the colour factor 2
  double r[SMALL_NSMAX];      // ggg_scale per set
  double G[16];               // colour matrix of the four structures (NG = 1)
  int nsets, two_pass;        // two_pass: the masses differ, every set is evaluated on its own
};

// contravariant w gamma^mu s in the chiral representation
__device__ __forceinline__ vec4<double> bilinear(const spn<double>& w, const spn<double>& s) {
  vec4<double> j;
  cx<double> t02 = w.c[0] * s.c[2], t13 = w.c[1] * s.c[3], t20 = w.c[2] * s.c[0], t31 = w.c[3] * s.c[1];
  cx<double> t03 = w.c[0] * s.c[3], t12 = w.c[1] * s.c[2], t21 = w.c[2] * s.c[1], t30 = w.c[3] * s.c[0];
  j.c[0] = (t02 + t13) + (t20 + t31);
  j.c[3] = (t02 - t13) - (t20 - t31);
  j.c[1] = (t03 + t12) - (t21 + t30);
  cx<double> y = (t12 - t03) + (t21 - t30);                 // gamma^2: i (t12 - t03 + t21 - t30)
  j.c[2] = mk<double>(-y.im, y.re);
  return j;
}

// helicity sums of the colour forms for sets k0 .. k0 + nk - 1, all evaluated with top mass m (unit couplings)
template <int NG>
__device__ __forceinline__ void qq_sums(const double (*p)[4], double m, const QQParams& P, int k0, int nk, double* sums) {
  for (int k = 0; k < nk; k++) sums[k] = 0.0;
  double KA[4], Kg[4], q1[4], q2[4], qt[4], qb[4], QB[4];
#pragma unroll
  for (int mu = 0; mu < 4; mu++) {
    const double k5 = NG ? p[4][mu] : 0.0;
    KA[mu] = p[0][mu] + p[1][mu]; Kg[mu] = -k5; QB[mu] = KA[mu] - k5;
    q1[mu] = p[0][mu] - k5; q2[mu] = k5 - p[1][mu]; qt[mu] = p[2][mu] + k5; qb[mu] = -p[3][mu] - k5;
  }
  const double iQA = 1.0 / mdot_rr(KA, KA);
  chi_pair<double> x1 = make_chi_raw(p[0][1], p[0][2], p[0][3]), x2 = make_chi_raw(p[1][1], p[1][2], p[1][3]);
  chi_pair<double> xt = make_chi_raw(p[2][1], p[2][2], p[2][3]), xb = make_chi_raw(p[3][1], p[3][2], p[3][3]);
  const shell<double> n1 = make_shell(p[0][0], 0.0, x1.n2), n2 = make_shell(p[1][0], 0.0, x2.n2);
  const shell<double> nt = make_shell(p[2][0], m, xt.n2), nb = make_shell(p[3][0], m, xb.n2);
  const spn<double> u1 = spinor_u(x1, n1, +1), vb2 = bar(spinor_v(x2, n2, -1));
  const vec4<double> jA = bilinear(vb2, u1);
  if constexpr (NG == 0) {
#pragma unroll
    for (int ib = 0; ib < 2; ib++) {
      const spn<double> c = slash_c(jA, spinor_v(xb, nb, ib ? -1 : +1));
#pragma unroll
      for (int it = 0; it < 2; it++) {
        const double a = norm2(rowcol(bar(spinor_u(xt, nt, it ? -1 : +1)), c)) * (iQA * iQA);
        for (int k = 0; k < nk; k++) sums[k] += a;
      }
    }
  } else {
    const double iq1 = 1.0 / mdot_rr(q1, q1), iq2 = 1.0 / mdot_rr(q2, q2), iQB = 1.0 / mdot_rr(QB, QB);
    const double m2 = m * m, dt = iQA / (mdot_rr(qt, qt) - m2), db = iQA / (mdot_rr(qb, qb) - m2);
#pragma unroll 1
    for (int ig = 0; ig < 2; ig++) {
      const vec4<double> e = conj4(polvec<double>(p[4][1], p[4][2], p[4][3], ig ? -1 : +1));
      const lcv<double> el = lightcone(e);
      // b_1, b_2, l
      spn<double> psi = slash_r_plus_m(q1, 0.0, slash_c(e, u1));
      spn<double> om; for (int i = 0; i < 4; i++) om.c[i] = mk<double>(0, 0);
      row_slash_acc(om, vb2, el);
      om = row_slash_r_plus_m(om, q2, 0.0);
      vec4<double> b1 = bilinear(vb2, psi), b2 = bilinear(om, u1), l;
#pragma unroll
      for (int mu = 0; mu < 4; mu++) { b1.c[mu] = (iq1 * iQB) * b1.c[mu]; b2.c[mu] = (iq2 * iQB) * b2.c[mu]; l.c[mu] = mk<double>(0, 0); }
      L3_acc(l, jA, KA, e, Kg);
#pragma unroll
      for (int mu = 0; mu < 4; mu++) l.c[mu] = (iQA * iQB) * l.c[mu];
#pragma unroll 1
      for (int ib = 0; ib < 2; ib++) {
        const spn<double> v = spinor_v(xb, nb, ib ? -1 : +1);
        const spn<double> c1 = slash_c(b2, v), c2 = slash_c(b1, v), cy = slash_c(l, v);
        const spn<double> c3 = slash_c(e, slash_r_plus_m(qt, m, slash_c(jA, v)));
        const spn<double> c4 = slash_c(jA, slash_r_plus_m(qb, m, slash_c(e, v)));
#pragma unroll
        for (int it = 0; it < 2; it++) {
          const spn<double> ub = bar(spinor_u(xt, nt, it ? -1 : +1));
          const cx<double> X1 = rowcol(ub, c1), X2 = rowcol(ub, c2), Y = rowcol(ub, cy);
          cx<double> a[4]; a[2] = dt * rowcol(ub, c3); a[3] = db * rowcol(ub, c4);
#pragma unroll 1
          for (int k = 0; k < nk; k++) {
            const double r = P.r[k0 + k];
            a[0] = X1; rfma(a[0], r, Y); a[1] = X2; rfma(a[1], -r, Y);
            double s = 0.0;
#pragma unroll
            for (int x = 0; x < 4; x++) {
              cx<double> t = mk<double>(0, 0);
#pragma unroll
              for (int y = 0; y < 4; y++) rfma(t, P.G[4 * x + y], a[y]);
              s += a[x].re * t.re + a[x].im * t.im;
            }
            sums[k] += s;
          }
        }
      }
    }
  }
}

// CTAs of 128 per SM: without the gluon 6 (80 registers, small spills) 0.062 ms for 2^20 events against 0.074 at 140 registers / 3 CTAs
// (4: 0.064, 8: 0.073); with the gluon the unconstrained 255 registers win (0.339; 168 registers 0.378, 128: 0.472, 96: 0.727)
constexpr int RWGT_QQ0_MINB = 6;
constexpr int RWGT_QQ1_MINB = 1;
template <int NG>
__global__ void __launch_bounds__(128, NG ? RWGT_QQ1_MINB : RWGT_QQ0_MINB) qqx_ttx_kernel(const double* __restrict__ mom, const double* __restrict__ wgt, const int* __restrict__ idx,
                                                      double* __restrict__ me_old, double* __restrict__ me_new, double* __restrict__ w_new,
                                                      long long n, long long stride, long long ostride, QQParams P) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (idx) i = idx[i];                      // multiprocess handles: the events of this process inside a mixed list
  double p[4 + NG][4];
#pragma unroll
  for (int ip = 0; ip < 4 + NG; ip++)
#pragma unroll
    for (int mu = 0; mu < 4; mu++) p[ip][mu] = __ldg(mom + (size_t)(ip * 4 + mu) * stride + i);
  const double W = __ldg(wgt + i);
  double sums[SMALL_NSMAX];
  if (!P.two_pass) qq_sums<NG>(p, P.mt[0], P, 0, P.nsets, sums);
  else
#pragma unroll 1
    for (int k = 0; k < P.nsets; k++) qq_sums<NG>(p, P.mt[k], P, k, 1, sums + k);
  const double a = sums[0] * P.fac[0];
  me_old[i] = a;
  for (int k = 1; k < P.nsets; k++) {
    const double b = sums[k] * P.fac[k];
    me_new[(size_t)(k - 1) * ostride + i] = b; w_new[(size_t)(k - 1) * ostride + i] = W * (b / a);
  }
}

}  // namespace rwgt
