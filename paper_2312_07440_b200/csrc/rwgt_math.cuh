// rwgt_math.cuh — device arithmetic of the helicity-amplitude evaluation (§3.1),
// hand-specialised for the CHIRAL representation with two-component blocks.
// Conventions: DESIGN.md "Readings".  Metric (+,-,-,-).
//   gamma^0 = [[0,1],[1,0]], gamma^i = [[0,s^i],[-s^i,0]];  spinor = (psi0,psi1 | psi2,psi3)
//   a-slash = [[0, a0 - s.a],[a0 + s.a, 0]]
// Shares nothing with oracle/ (which uses generic 4x4 Dirac-representation matrices).
#pragma once
#include <cuda_runtime.h>

namespace rwgt {

template <typename T> struct cx { T re, im; };
template <typename T> __device__ __forceinline__ cx<T> mk(T a, T b) { cx<T> r; r.re = a; r.im = b; return r; }
template <typename T> __device__ __forceinline__ cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <typename T> __device__ __forceinline__ cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <typename T> __device__ __forceinline__ cx<T> operator-(cx<T> a) { return mk<T>(-a.re, -a.im); }
template <typename T> __device__ __forceinline__ cx<T> operator*(cx<T> a, cx<T> b) { return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
template <typename T> __device__ __forceinline__ cx<T> operator*(T s, cx<T> a) { return mk<T>(s * a.re, s * a.im); }
template <typename T> __device__ __forceinline__ cx<T> conj(cx<T> a) { return mk<T>(a.re, -a.im); }
template <typename T> __device__ __forceinline__ T norm2(cx<T> a) { return a.re * a.re + a.im * a.im; }
// acc += a*b  (4 FMA)
template <typename T> __device__ __forceinline__ void cfma(cx<T>& acc, cx<T> a, cx<T> b) {
  acc.re = fma(a.re, b.re, acc.re); acc.re = fma(-a.im, b.im, acc.re);
  acc.im = fma(a.re, b.im, acc.im); acc.im = fma(a.im, b.re, acc.im);
}
// acc += s*a  (2 FMA), s real
template <typename T> __device__ __forceinline__ void rfma(cx<T>& acc, T s, cx<T> a) { acc.re = fma(s, a.re, acc.re); acc.im = fma(s, a.im, acc.im); }
// acc -= a*b,  acc -= s*a   (the same instruction sequences as cfma(acc, -a, b), rfma(acc, -s, a))
template <typename T> __device__ __forceinline__ void cfms(cx<T>& acc, cx<T> a, cx<T> b) { cfma(acc, -a, b); }
template <typename T> __device__ __forceinline__ void rfms(cx<T>& acc, T s, cx<T> a) { rfma(acc, -s, a); }

// ---- FP32: packed two-lane arithmetic (PTX fma/mul/add.rn.f32x2 = SASS FFMA2/FMUL2/FADD2 on sm_100a) -------------------
// A complex float is an aligned (re, im) register pair.  A complex multiply-add is TWO FFMA2:
//     acc += b * a.re ;  acc += (-b.im, b.re) * a.im
// ptxas folds the lane swap, the per-lane negation and the scalar broadcast into operand modifiers of FFMA2
// (R.F32x2.LO_HI.NP, R.F32) when the swapped/negated pair is the FIRST source and the broadcast the second, so no
// packing instruction is issued (checked with cuobjdump -sass).  Measured on B200 with three distinct register sources:
// FFMA 42 TFLOP/s, FFMA2 50-67 TFLOP/s, and half the issue slots.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ cx<float> upk2(f32x2 v) { cx<float> r; asm("mov.b64 {%0,%1}, %2;" : "=f"(r.re), "=f"(r.im) : "l"(v)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ void cfma(cx<float>& acc, cx<float> a, cx<float> b) {
  f32x2 A = pk2(acc.re, acc.im);
  A = fma2(pk2(b.re, b.im), pk2(a.re, a.re), A); A = fma2(pk2(-b.im, b.re), pk2(a.im, a.im), A);
  acc = upk2(A);
}
__device__ __forceinline__ void cfms(cx<float>& acc, cx<float> a, cx<float> b) {
  f32x2 A = pk2(acc.re, acc.im);
  A = fma2(pk2(-b.re, -b.im), pk2(a.re, a.re), A); A = fma2(pk2(b.im, -b.re), pk2(a.im, a.im), A);
  acc = upk2(A);
}
__device__ __forceinline__ void rfma(cx<float>& acc, float s, cx<float> a) { acc = upk2(fma2(pk2(a.re, a.im), pk2(s, s), pk2(acc.re, acc.im))); }
__device__ __forceinline__ void rfms(cx<float>& acc, float s, cx<float> a) { acc = upk2(fma2(pk2(-a.re, -a.im), pk2(s, s), pk2(acc.re, acc.im))); }
__device__ __forceinline__ cx<float> operator*(cx<float> a, cx<float> b) {
  f32x2 A = mul2(pk2(b.re, b.im), pk2(a.re, a.re)); return upk2(fma2(pk2(-b.im, b.re), pk2(a.im, a.im), A));
}
__device__ __forceinline__ cx<float> operator*(float s, cx<float> a) { return upk2(mul2(pk2(a.re, a.im), pk2(s, s))); }
__device__ __forceinline__ cx<float> operator+(cx<float> a, cx<float> b) { return upk2(add2(pk2(a.re, a.im), pk2(b.re, b.im))); }
__device__ __forceinline__ cx<float> operator-(cx<float> a, cx<float> b) { return upk2(add2(pk2(a.re, a.im), pk2(-b.re, -b.im))); }

template <typename T> struct vec4 { cx<T> c[4]; };   // complex Lorentz vector, contravariant (t,x,y,z)
template <typename T> struct spn { cx<T> c[4]; };    // Dirac spinor, chiral representation

template <typename T> __device__ __forceinline__ T mdot_rr(const T* a, const T* b) { return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]; }
template <typename T> __device__ __forceinline__ cx<T> mdot_rc(const T* a, const vec4<T>& b) {
  cx<T> r = a[0] * b.c[0]; rfms(r, a[1], b.c[1]); rfms(r, a[2], b.c[2]); rfms(r, a[3], b.c[3]); return r;
}
template <typename T> __device__ __forceinline__ cx<T> mdot_cc(const vec4<T>& a, const vec4<T>& b) {
  cx<T> r = a.c[0] * b.c[0]; cfms(r, a.c[1], b.c[1]); cfms(r, a.c[2], b.c[2]); cfms(r, a.c[3], b.c[3]); return r;
}

// a-slash * psi, a complex
template <typename T> __device__ __forceinline__ spn<T> slash_c(const vec4<T>& a, const spn<T>& s) {
  cx<T> ap = a.c[0] + a.c[3], am = a.c[0] - a.c[3];
  cx<T> ar = mk<T>(a.c[1].re + a.c[2].im, a.c[1].im - a.c[2].re);   // a1 - i a2
  cx<T> al = mk<T>(a.c[1].re - a.c[2].im, a.c[1].im + a.c[2].re);   // a1 + i a2
  spn<T> r;
  r.c[0] = am * s.c[2]; cfms(r.c[0], ar, s.c[3]);
  r.c[1] = ap * s.c[3]; cfms(r.c[1], al, s.c[2]);
  r.c[2] = ap * s.c[0]; cfma(r.c[2], ar, s.c[1]);
  r.c[3] = am * s.c[1]; cfma(r.c[3], al, s.c[0]);
  return r;
}
// (q-slash + m) * psi, q real
template <typename T> __device__ __forceinline__ spn<T> slash_r_plus_m(const T* q, T m, const spn<T>& s) {
  T qp = q[0] + q[3], qm = q[0] - q[3];
  cx<T> qr = mk<T>(q[1], -q[2]), ql = mk<T>(q[1], q[2]);
  spn<T> r;
  r.c[0] = m * s.c[0]; rfma(r.c[0], qm, s.c[2]); cfms(r.c[0], qr, s.c[3]);
  r.c[1] = m * s.c[1]; rfma(r.c[1], qp, s.c[3]); cfms(r.c[1], ql, s.c[2]);
  r.c[2] = m * s.c[2]; rfma(r.c[2], qp, s.c[0]); cfma(r.c[2], qr, s.c[1]);
  r.c[3] = m * s.c[3]; rfma(r.c[3], qm, s.c[1]); cfma(r.c[3], ql, s.c[0]);
  return r;
}
// row * (q-slash + m), q real
template <typename T> __device__ __forceinline__ spn<T> row_slash_r_plus_m(const spn<T>& w, const T* q, T m) {
  T qp = q[0] + q[3], qm = q[0] - q[3];
  cx<T> qr = mk<T>(q[1], -q[2]), ql = mk<T>(q[1], q[2]);
  spn<T> r;
  r.c[0] = m * w.c[0]; rfma(r.c[0], qp, w.c[2]); cfma(r.c[0], w.c[3], ql);
  r.c[1] = m * w.c[1]; rfma(r.c[1], qm, w.c[3]); cfma(r.c[1], w.c[2], qr);
  r.c[2] = m * w.c[2]; rfma(r.c[2], qm, w.c[0]); cfms(r.c[2], w.c[1], ql);
  r.c[3] = m * w.c[3]; rfma(r.c[3], qp, w.c[1]); cfms(r.c[3], w.c[0], qr);
  return r;
}
template <typename T> __device__ __forceinline__ cx<T> rowcol(const spn<T>& w, const spn<T>& s) {
  cx<T> r = w.c[0] * s.c[0]; cfma(r, w.c[1], s.c[1]); cfma(r, w.c[2], s.c[2]); cfma(r, w.c[3], s.c[3]); return r;
}

// ---- external wavefunctions -------------------------------------------------------
// two-component helicity eigenspinors chi_+, chi_- of direction p_vec; exact on the beam axis.
template <typename T> struct chi_pair { cx<T> p[2], m[2]; T pabs, n2; };      // |chi_+-|^2 = n2 (1 once normalised)
// unnormalised: chi_+ = (|p|+pz, px + i py), chi_- = (-px + i py, |p|+pz), n2 = 2 |p| (|p|+pz); the caller folds 1/sqrt(n2) into
// the spinor normalisation (make_shell), which saves one reciprocal square root per leg
template <typename T> __device__ __forceinline__ chi_pair<T> make_chi_raw(T px, T py, T pz) {
  chi_pair<T> r; T pt2 = px * px + py * py; T pabs = sqrt(pt2 + pz * pz); r.pabs = pabs; r.n2 = T(1);
  if (pabs == T(0)) { r.p[0] = mk<T>(1, 0); r.p[1] = mk<T>(0, 0); r.m[0] = mk<T>(0, 0); r.m[1] = mk<T>(1, 0); return r; }
  if (pt2 == T(0) && pz < T(0)) { r.p[0] = mk<T>(0, 0); r.p[1] = mk<T>(1, 0); r.m[0] = mk<T>(-1, 0); r.m[1] = mk<T>(0, 0); return r; }
  T ppz = (pz >= T(0)) ? pabs + pz : pt2 / (pabs - pz);     // |p|+pz, cancellation-free
  r.n2 = T(2) * pabs * ppz;
  r.p[0] = mk<T>(ppz, 0); r.p[1] = mk<T>(px, py);
  r.m[0] = mk<T>(-px, py); r.m[1] = mk<T>(ppz, 0);
  return r;
}
template <typename T> __device__ __forceinline__ chi_pair<T> make_chi(T px, T py, T pz) {
  chi_pair<T> r = make_chi_raw(px, py, pz);
  if (r.n2 != T(1)) {
    const T N = rsqrt(r.n2); r.n2 = T(1);
#pragma unroll
    for (int i = 0; i < 2; i++) { r.p[i] = N * r.p[i]; r.m[i] = N * r.m[i]; }
  }
  return r;
}
// Spinor normalisation (reading Q8 / DESIGN.md R8): the energy comes from the input, the mass from the PARAMETER SET, and
// the magnitude of the 3-momentum in the normalisation is the one that follows from these two, P = sqrt((E-m)(E+m));
// only the direction chi(p_hat) comes from the input 3-momentum.  On the mass shell P = |p|; for a set whose mass differs from
// the one the events were generated with this is what "the parameter masses in spinors and propagators, E from the input"
// means, and it equals the oracle's Dirac-representation form (sqrt(E+m) chi, lam sqrt(E-m) chi) exactly:
// ((sqrt(E+m) -+ lam sqrt(E-m)) / sqrt2)^2 = E -+ lam P.
// If a set's mass exceeds the input energy (E < m: a slow top of the event's own, lighter mass shell) the oracle clamps
// sqrt(E-m) to 0, i.e. both chiral normalisations are sqrt((E+m)/2); the same here.
template <typename T> struct shell { T sp, sm; };       // sqrt(E+P) / sqrt(n2), sqrt(E-P) / sqrt(n2)
// n2: squared norm of the chi the spinor is built from (make_chi_raw), 1 for a normalised chi
template <typename T> __device__ __forceinline__ shell<T> make_shell(T E, T m, T n2 = T(1)) {
  const bool on = (E >= m);
  const T P = (m == T(0)) ? E : sqrt(fmax((E - m) * (E + m), T(0)));
  const T ep = on ? E + P : T(0.5) * (E + m), ir = rsqrt(ep * n2);
  shell<T> r; r.sp = ep * ir;       // sqrt(E+P) / sqrt(n2)
  r.sm = (on ? m : ep) * ir;        // sqrt(E-P) = m / sqrt(E+P): no cancellation, no division
  return r;
}
// u(p,lam) = ( sqrt(E-lam P) chi_lam , sqrt(E+lam P) chi_lam )
template <typename T> __device__ __forceinline__ spn<T> spinor_u(const chi_pair<T>& x, const shell<T>& n, int lam) {
  const T sp = n.sp, sm = n.sm;
  const cx<T>* c = lam > 0 ? x.p : x.m; T a = lam > 0 ? sm : sp, b = lam > 0 ? sp : sm;
  spn<T> r; r.c[0] = a * c[0]; r.c[1] = a * c[1]; r.c[2] = b * c[0]; r.c[3] = b * c[1]; return r;
}
// v(p,lam) = ( -lam sqrt(E+lam P) chi_{-lam} , lam sqrt(E-lam P) chi_{-lam} )
template <typename T> __device__ __forceinline__ spn<T> spinor_v(const chi_pair<T>& x, const shell<T>& n, int lam) {
  const T sp = n.sp, sm = n.sm;
  const cx<T>* c = lam > 0 ? x.m : x.p; T a = lam > 0 ? -sp : sm, b = lam > 0 ? sm : -sp;
  spn<T> r; r.c[0] = a * c[0]; r.c[1] = a * c[1]; r.c[2] = b * c[0]; r.c[3] = b * c[1]; return r;
}
// psibar = psi^dagger gamma^0 as a row
template <typename T> __device__ __forceinline__ spn<T> bar(const spn<T>& s) {
  spn<T> r; r.c[0] = conj(s.c[2]); r.c[1] = conj(s.c[3]); r.c[2] = conj(s.c[0]); r.c[3] = conj(s.c[1]); return r;
}
// eps(p,lam) = (0, (-lam e1 - i e2)/sqrt2), spatial-transverse in the given frame (binding, reading Q1)
template <typename T> __device__ __forceinline__ vec4<T> polvec(T px, T py, T pz, int lam) {
  T pt2 = px * px + py * py;
  T e1x, e1y, e1z, e2x, e2y;
  if (pt2 == T(0)) { e1x = pz >= T(0) ? T(1) : T(-1); e1y = 0; e1z = 0; e2x = 0; e2y = 1; }
  else { T ip = rsqrt(pt2), inv = ip * rsqrt(pt2 + pz * pz); e1x = px * pz * inv; e1y = py * pz * inv; e1z = -pt2 * inv; e2x = -py * ip; e2y = px * ip; }   // 1/pT, 1/(|p| pT)
  const T s = T(0.70710678118654752440); T l = T(lam);
  vec4<T> r; r.c[0] = mk<T>(0, 0); r.c[1] = mk<T>(-l * s * e1x, -s * e2x); r.c[2] = mk<T>(-l * s * e1y, -s * e2y); r.c[3] = mk<T>(-l * s * e1z, 0);
  return r;
}
// both helicities at once: eps(p,-1) differs from eps(p,+1) in the sign of the e1 part only (the rsqrt chain is shared)
template <typename T> __device__ __forceinline__ void polvec_pair(T px, T py, T pz, vec4<T>& ep, vec4<T>& em) {
  ep = polvec<T>(px, py, pz, +1);
  em.c[0] = mk<T>(0, 0);
#pragma unroll
  for (int i = 1; i < 4; i++) em.c[i] = mk<T>(-ep.c[i].re, ep.c[i].im);
}
template <typename T> __device__ __forceinline__ vec4<T> conj4(const vec4<T>& a) { vec4<T> r; for (int i = 0; i < 4; i++) r.c[i] = conj(a.c[i]); return r; }

// ---- gluon self-interaction Lorentz structures --------------------------------------
// acc += L3(A,B),  L3(A,B) = (JA.JB)(KA-KB) + JB ((KA+2KB).JA) - JA ((2KA+KB).JB).  Bilinear: a sign is applied by negating JA.
template <typename T> __device__ __forceinline__ void L3_acc(vec4<T>& acc, const vec4<T>& JA, const T* KA, const vec4<T>& JB, const T* KB) {
  T d[4], u[4], w[4];
#pragma unroll
  for (int i = 0; i < 4; i++) { d[i] = KA[i] - KB[i]; u[i] = fma(T(2), KB[i], KA[i]); w[i] = -fma(T(2), KA[i], KB[i]); }
  cx<T> ab = mdot_cc(JA, JB), c1 = mdot_rc(u, JA), c2 = mdot_rc(w, JB);
#pragma unroll
  for (int i = 0; i < 4; i++) { rfma(acc.c[i], d[i], ab); cfma(acc.c[i], c1, JB.c[i]); cfma(acc.c[i], c2, JA.c[i]); }
}
// FP32: the three real momentum combinations as packed pairs (2 FADD2 + 4 FFMA2 instead of 4 FADD + 8 FFMA)
__device__ __forceinline__ void L3_acc(vec4<float>& acc, const vec4<float>& JA, const float* KA, const vec4<float>& JB, const float* KB) {
  const f32x2 two = pk2(2.0f, 2.0f), mtwo = pk2(-2.0f, -2.0f);
  float d[4], u[4], w[4];
#pragma unroll
  for (int h = 0; h < 2; h++) {
    const f32x2 ka = pk2(KA[2 * h], KA[2 * h + 1]), kb = pk2(KB[2 * h], KB[2 * h + 1]), nkb = pk2(-KB[2 * h], -KB[2 * h + 1]);
    const cx<float> dd = upk2(add2(ka, nkb)), uu = upk2(fma2(two, kb, ka)), ww = upk2(fma2(mtwo, ka, nkb));
    d[2 * h] = dd.re; d[2 * h + 1] = dd.im; u[2 * h] = uu.re; u[2 * h + 1] = uu.im; w[2 * h] = ww.re; w[2 * h + 1] = ww.im;
  }
  cx<float> ab = mdot_cc(JA, JB), c1 = mdot_rc(u, JA), c2 = mdot_rc(w, JB);
#pragma unroll
  for (int i = 0; i < 4; i++) { rfma(acc.c[i], d[i], ab); cfma(acc.c[i], c1, JB.c[i]); cfma(acc.c[i], c2, JA.c[i]); }
}
// acc += V4(X,Y,Z), colour-ordered quartic structure V4 = 2 (X.Z) Y - (Y.Z) X - (X.Y) Z.  Trilinear: sign by negating X.
template <typename T> __device__ __forceinline__ void V4_acc(vec4<T>& acc, const vec4<T>& X, const vec4<T>& Y, const vec4<T>& Z) {
  cx<T> xz = mdot_cc(X, Z), yz = mdot_cc(Y, Z), xy = mdot_cc(X, Y);
  xz = mk<T>(xz.re + xz.re, xz.im + xz.im); yz = -yz; xy = -xy;
#pragma unroll
  for (int i = 0; i < 4; i++) { cfma(acc.c[i], xz, Y.c[i]); cfma(acc.c[i], yz, X.c[i]); cfma(acc.c[i], xy, Z.c[i]); }
}
// light-cone components of a complex vector: a+ = a0+a3, a- = a0-a3, ar = a1 - i a2, al = a1 + i a2 (what a-slash needs)
template <typename T> struct lcv { cx<T> p, m, r, l; };
template <typename T> __device__ __forceinline__ lcv<T> lightcone(const vec4<T>& a) {
  lcv<T> r; r.p = a.c[0] + a.c[3]; r.m = a.c[0] - a.c[3];
  r.r = mk<T>(a.c[1].re + a.c[2].im, a.c[1].im - a.c[2].re); r.l = mk<T>(a.c[1].re - a.c[2].im, a.c[1].im + a.c[2].re);
  return r;
}
// light-cone components of -a (the negation rides on the adds)
template <typename T> __device__ __forceinline__ lcv<T> lightcone_neg(const vec4<T>& a) {
  lcv<T> r; r.p = mk<T>(-a.c[0].re - a.c[3].re, -a.c[0].im - a.c[3].im); r.m = mk<T>(a.c[3].re - a.c[0].re, a.c[3].im - a.c[0].im);
  r.r = mk<T>(-a.c[1].re - a.c[2].im, a.c[2].re - a.c[1].im); r.l = mk<T>(a.c[2].im - a.c[1].re, -a.c[1].im - a.c[2].re);
  return r;
}
// packed FP32 forms: every component is one add.rn.f32x2 (the swap / negation of a2 rides on operand modifiers)
__device__ __forceinline__ lcv<float> lightcone(const vec4<float>& a) {
  lcv<float> r; const f32x2 a0 = pk2(a.c[0].re, a.c[0].im), a1 = pk2(a.c[1].re, a.c[1].im);
  r.p = upk2(add2(a0, pk2(a.c[3].re, a.c[3].im))); r.m = upk2(add2(a0, pk2(-a.c[3].re, -a.c[3].im)));
  r.r = upk2(add2(a1, pk2(a.c[2].im, -a.c[2].re))); r.l = upk2(add2(a1, pk2(-a.c[2].im, a.c[2].re)));
  return r;
}
__device__ __forceinline__ lcv<float> lightcone_neg(const vec4<float>& a) {
  lcv<float> r; const f32x2 n0 = pk2(-a.c[0].re, -a.c[0].im), n1 = pk2(-a.c[1].re, -a.c[1].im);
  r.p = upk2(add2(n0, pk2(-a.c[3].re, -a.c[3].im))); r.m = upk2(add2(n0, pk2(a.c[3].re, a.c[3].im)));
  r.r = upk2(add2(n1, pk2(-a.c[2].im, a.c[2].re))); r.l = upk2(add2(n1, pk2(a.c[2].im, -a.c[2].re)));
  return r;
}
// X += a-slash * s      (8 complex FMAs)
template <typename T> __device__ __forceinline__ void slash_acc(spn<T>& X, const lcv<T>& a, const spn<T>& s) {
  cfma(X.c[0], a.m, s.c[2]); cfms(X.c[0], a.r, s.c[3]);
  cfma(X.c[1], a.p, s.c[3]); cfms(X.c[1], a.l, s.c[2]);
  cfma(X.c[2], a.p, s.c[0]); cfma(X.c[2], a.r, s.c[1]);
  cfma(X.c[3], a.m, s.c[1]); cfma(X.c[3], a.l, s.c[0]);
}
// X += w * a-slash      (row vector, 8 complex FMAs)
template <typename T> __device__ __forceinline__ void row_slash_acc(spn<T>& X, const spn<T>& w, const lcv<T>& a) {
  cfma(X.c[0], w.c[2], a.p); cfma(X.c[0], w.c[3], a.l);
  cfma(X.c[1], w.c[2], a.r); cfma(X.c[1], w.c[3], a.m);
  cfma(X.c[2], w.c[0], a.m); cfms(X.c[2], w.c[1], a.l);
  cfma(X.c[3], w.c[1], a.p); cfms(X.c[3], w.c[0], a.r);
}
// acc += w . s
template <typename T> __device__ __forceinline__ void rowcol_acc(cx<T>& acc, const spn<T>& w, const spn<T>& s) {
  cfma(acc, w.c[0], s.c[0]); cfma(acc, w.c[1], s.c[1]); cfma(acc, w.c[2], s.c[2]); cfma(acc, w.c[3], s.c[3]);
}

}  // namespace rwgt
