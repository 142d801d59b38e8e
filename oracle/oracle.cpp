// oracle/oracle.cpp — CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, double-precision implementation of what the hot path computes:
//   W' = W * |M'|^2 / |M|^2            (§2.2 eq. 3; steps 3-6 of PAPER.md:87)
// with |M|^2 the tree-level squared matrix element evaluated as a sum of helicity
// amplitudes (§3.1: "helicity amplitudes", refs [14],[15]).  The paper
// prints no formula below eq. 3; every rule used here is the reading fixed in
// SURVEY.md §8(c) C1-C8 (restated in DESIGN.md "Readings") and is cited inline.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this.  It shares no code with paper_2312_07440_b200/csrc: generic 4x4
// gamma matrices in the DIRAC representation, matrix-valued currents with colour kept
// as formal strings of generator labels (route F) or as explicit SU(3) components
// (route E), colour matrix from explicit Gell-Mann matrices, every helicity combination
// evaluated from scratch, each parameter set evaluated independently.
//
// eq. 2 sigma ~ sum_k W_k: orc_cross_section, the plain sum, pinned against exactly rounded summation.
// Pins (tests/test_oracle_pins.py): Dirac equation + completeness for u,v; transversality,
// normalisation, helicity eigen-equation and completeness of eps; e+e- -> mu+mu- closed
// form and gg -> ttbar closed form; gauge invariance eps->k of
// every colour-flow amplitude at kappa=0 for n=2..5; Lorentz-boost invariance at kappa=0;
// rotation invariance for the new set; route F == route E (explicit 8^n colour sum, uses
// f^{abc} instead of colour strings) at n=2,3 (+ a few helicities at n=4); colour-matrix
// table SURVEY C7; polynomial degree 2(n-1) in kappa; worked values SURVEY C10.
// e+ e- -> n photons (n = 2..5; n = 5 is the paper's own measured process): pinned in
// tests/test_oracle_pins_photons.py by the textbook closed forms at n = 2, 3, the soft-photon theorem linking n + 1 to n up to
// n = 5, gauge invariance eps -> k of every helicity amplitude, boost/rotation invariance, helicity selection rules and the
// exact (alpha'/alpha)^n scaling.
// q qbar -> t tbar (+ g) (a structurally different amplitude): explicit colour on every leg; pinned in
// tests/test_oracle_pins_qq.py by the textbook closed form of q qbar -> Q Qbar, gauge invariance eps -> k, boost / rotation invariance,
// the soft-gluon (eikonal) limit with colour correlations, parity.
// PARITY UNPINNED (stated in DESIGN.md): absolute normalisation 1/(n-2)! of cfgs 4,5 and
// the explicit-colour check of all helicities at n=5 (too slow).
//
// Build: python oracle/build.py   (g++ -O2 -fopenmp -shared)

#include <complex>
#include <vector>
#include <map>
#include <array>
#include <cmath>
#include <cstring>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);

// ---------------------------------------------------------------- basic objects
struct V4 { cd c[4]; };   // contravariant Lorentz vector (t,x,y,z); complex for polarisations/currents
struct Sp { cd c[4]; };   // Dirac spinor
struct M4 { cd m[4][4]; };

static V4 v4zero() { V4 r; for (int i = 0; i < 4; i++) r.c[i] = 0; return r; }
static V4 operator+(const V4& a, const V4& b) { V4 r; for (int i = 0; i < 4; i++) r.c[i] = a.c[i] + b.c[i]; return r; }
static V4 operator-(const V4& a, const V4& b) { V4 r; for (int i = 0; i < 4; i++) r.c[i] = a.c[i] - b.c[i]; return r; }
static V4 operator*(cd s, const V4& a) { V4 r; for (int i = 0; i < 4; i++) r.c[i] = s * a.c[i]; return r; }
// metric (+,-,-,-), no complex conjugation
static cd dot(const V4& a, const V4& b) { return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3]; }
static Sp spzero() { Sp r; for (int i = 0; i < 4; i++) r.c[i] = 0; return r; }
static Sp operator+(const Sp& a, const Sp& b) { Sp r; for (int i = 0; i < 4; i++) r.c[i] = a.c[i] + b.c[i]; return r; }
static Sp operator*(cd s, const Sp& a) { Sp r; for (int i = 0; i < 4; i++) r.c[i] = s * a.c[i]; return r; }
static Sp operator*(const M4& A, const Sp& x) {
  Sp r; for (int i = 0; i < 4; i++) { cd s = 0; for (int j = 0; j < 4; j++) s += A.m[i][j] * x.c[j]; r.c[i] = s; } return r;
}
static M4 operator*(const M4& A, const M4& B) {
  M4 r; for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { cd s = 0; for (int k = 0; k < 4; k++) s += A.m[i][k] * B.m[k][j]; r.m[i][j] = s; } return r;
}
static M4 operator+(const M4& A, const M4& B) { M4 r; for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) r.m[i][j] = A.m[i][j] + B.m[i][j]; return r; }
static M4 operator*(cd s, const M4& A) { M4 r; for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) r.m[i][j] = s * A.m[i][j]; return r; }

// ---------------------------------------------------------------- gamma matrices, Dirac representation
// gamma^0 = diag(1,1,-1,-1), gamma^i = [[0,sigma^i],[-sigma^i,0]], gamma^5 = [[0,1],[1,0]].
// (Unitarily equivalent to the chiral representation quoted in SURVEY C2; helicity-summed
//  |M|^2 does not depend on the representation.)
struct Gammas {
  M4 g[4], g5, one, PL, PR;
  Gammas() {
    cd s[3][2][2] = {{{0, 1}, {1, 0}}, {{0, -I_}, {I_, 0}}, {{1, 0}, {0, -1}}};
    for (int mu = 0; mu < 4; mu++) for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) g[mu].m[i][j] = 0;
    for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { g5.m[i][j] = 0; one.m[i][j] = (i == j) ? 1.0 : 0.0; }
    g[0].m[0][0] = g[0].m[1][1] = 1; g[0].m[2][2] = g[0].m[3][3] = -1;
    for (int k = 0; k < 3; k++) for (int a = 0; a < 2; a++) for (int b = 0; b < 2; b++) {
      g[k + 1].m[a][2 + b] = s[k][a][b];
      g[k + 1].m[2 + a][b] = -s[k][a][b];
    }
    g5.m[0][2] = g5.m[1][3] = g5.m[2][0] = g5.m[3][1] = 1;
    PL = cd(0.5) * (one + cd(-1.0) * g5);
    PR = cd(0.5) * (one + g5);
  }
};
static const Gammas& GM() { static Gammas G; return G; }

// a-slash = gamma^mu a_mu = gamma^0 a^0 - gamma^i a^i
static M4 slash(const V4& a) {
  const Gammas& G = GM();
  return a.c[0] * G.g[0] + (-a.c[1]) * G.g[1] + (-a.c[2]) * G.g[2] + (-a.c[3]) * G.g[3];
}
// psibar = psi^dagger gamma^0 ; returned as a row stored in Sp
static Sp bar(const Sp& x) {
  Sp r; r.c[0] = std::conj(x.c[0]); r.c[1] = std::conj(x.c[1]); r.c[2] = -std::conj(x.c[2]); r.c[3] = -std::conj(x.c[3]); return r;
}
static cd rowcol(const Sp& row, const Sp& col) { cd s = 0; for (int i = 0; i < 4; i++) s += row.c[i] * col.c[i]; return s; }

// ---------------------------------------------------------------- external wavefunctions
// two-component helicity eigenspinor chi_lambda(p_vec), sigma.p_hat chi = lambda chi
static void chi2(const double p[4], int lam, cd out[2]) {
  double px = p[1], py = p[2], pz = p[3];
  double pabs = std::sqrt(px * px + py * py + pz * pz);
  double pt2 = px * px + py * py;
  if (pabs == 0.0) { pabs = 1.0; pz = 1.0; pt2 = 0.0; px = py = 0.0; }     // p_vec = 0: take p_hat = z_hat
  if (pt2 == 0.0 && pz < 0.0) {                                           // boundary p_T = 0, p_z < 0
    if (lam > 0) { out[0] = 0; out[1] = 1; } else { out[0] = -1; out[1] = 0; }
    return;
  }
  // |p|+p_z without cancellation for backward legs (SURVEY §7 "exact-axis legs": use the light-cone form)
  double ppz = (pz >= 0.0) ? pabs + pz : pt2 / (pabs - pz);
  double N = 1.0 / std::sqrt(2.0 * pabs * ppz);
  if (lam > 0) { out[0] = N * ppz; out[1] = N * cd(px, py); }
  else         { out[0] = N * cd(-px, py); out[1] = N * ppz; }
}
// u(p,lambda) in the Dirac representation: ( sqrt(E+m) chi_l , l sqrt(E-m) chi_l )
static Sp spinor_u(const double p[4], double m, int lam) {
  cd x[2]; chi2(p, lam, x);
  double a = std::sqrt(std::max(0.0, p[0] + m)), b = std::sqrt(std::max(0.0, p[0] - m));
  Sp r; r.c[0] = a * x[0]; r.c[1] = a * x[1]; r.c[2] = double(lam) * b * x[0]; r.c[3] = double(lam) * b * x[1]; return r;
}
// v(p,lambda) in the Dirac representation: ( -sqrt(E-m) chi_{-l} , l sqrt(E+m) chi_{-l} )
static Sp spinor_v(const double p[4], double m, int lam) {
  cd x[2]; chi2(p, -lam, x);
  double a = std::sqrt(std::max(0.0, p[0] + m)), b = std::sqrt(std::max(0.0, p[0] - m));
  Sp r; r.c[0] = -b * x[0]; r.c[1] = -b * x[1]; r.c[2] = double(lam) * a * x[0]; r.c[3] = double(lam) * a * x[1]; return r;
}
// polarisation vector of a massless vector, lambda = +-1 (binding convention Q1):
// eps = (0, (-lambda e1 - i e2)/sqrt2), purely spatial in the frame the momenta are given in.
static V4 polvec(const double p[4], int lam) {
  double px = p[1], py = p[2], pz = p[3];
  double pt = std::sqrt(px * px + py * py), pabs = std::sqrt(px * px + py * py + pz * pz);
  double e1[3], e2[3];
  if (pt == 0.0) { e1[0] = (pz >= 0 ? 1.0 : -1.0); e1[1] = 0; e1[2] = 0; e2[0] = 0; e2[1] = 1; e2[2] = 0; }
  else {
    e1[0] = px * pz / (pabs * pt); e1[1] = py * pz / (pabs * pt); e1[2] = -pt * pt / (pabs * pt);
    e2[0] = -py / pt; e2[1] = px / pt; e2[2] = 0;
  }
  V4 r; r.c[0] = 0; const double s = 1.0 / std::sqrt(2.0);
  for (int i = 0; i < 3; i++) r.c[i + 1] = s * cd(-double(lam) * e1[i], -e2[i]);
  return r;
}
static V4 conjv(const V4& a) { V4 r; for (int i = 0; i < 4; i++) r.c[i] = std::conj(a.c[i]); return r; }

// ---------------------------------------------------------------- parameters (order == struct rwgt_params)
struct Par { double alpha_em, alpha_s, mZ, GammaZ, sw2, mt, Gamma_t, ggg_scale, gggg_scale; };
static Par par_from(const double* x) { Par p; std::memcpy(&p, x, sizeof(Par)); return p; }
static const double PI = 3.14159265358979323846;

// ---------------------------------------------------------------- cfg 1: e+(p1) e-(p2) -> mu+(p3) mu-(p4)  (rules C3)
// iM = sum_V [vbar(p1) (-i g_V gamma^mu Gamma_V) u(p2)] (-i g_{mu nu}/D_V) [ubar(p4) (-i g_V gamma^nu Gamma_V) v(p3)]
static cd amp_epem(const Par& P, const double p[4][4], const int hel[4]) {
  const Gammas& G = GM();
  double e = std::sqrt(4.0 * PI * P.alpha_em), cw2 = 1.0 - P.sw2;
  double gZ = e / std::sqrt(P.sw2 * cw2), gL = -0.5 + P.sw2, gR = P.sw2, Q = -1.0;
  double s = 0; { double q[4]; for (int i = 0; i < 4; i++) q[i] = p[0][i] + p[1][i]; s = q[0] * q[0] - q[1] * q[1] - q[2] * q[2] - q[3] * q[3]; }
  Sp vb1 = bar(spinor_v(p[0], 0.0, hel[0])), u2 = spinor_u(p[1], 0.0, hel[1]);
  Sp v3 = spinor_v(p[2], 0.0, hel[2]), ub4 = bar(spinor_u(p[3], 0.0, hel[3]));
  cd tot = 0;
  for (int V = 0; V < 2; V++) {
    M4 Gam = (V == 0) ? G.one : (cd(gL) * G.PL + cd(gR) * G.PR);
    double gV = (V == 0) ? e * Q : gZ;
    cd D = (V == 0) ? cd(s, 0) : cd(s - P.mZ * P.mZ, P.mZ * P.GammaZ);
    V4 Je, Jm;
    for (int mu = 0; mu < 4; mu++) {
      M4 vert = (-I_ * gV) * (G.g[mu] * Gam);
      Je.c[mu] = rowcol(vb1, vert * u2);
      Jm.c[mu] = rowcol(ub4, vert * v3);
    }
    tot += dot(Je, Jm) * (-I_ / D);
  }
  return tot;     // = iM
}
static double me2_epem(const Par& P, const double p[4][4]) {
  double sum = 0; int hel[4];
  for (int h = 0; h < 16; h++) {                 // full helicity sum (Q5)
    for (int i = 0; i < 4; i++) hel[i] = ((h >> i) & 1) ? 1 : -1;
    sum += std::norm(amp_epem(P, p, hel));
  }
  return sum / 4.0;                               // average over 2x2 initial helicities (Q3)
}

// ---------------------------------------------------------------- SU(3): Gell-Mann matrices, f^{abc}
struct SU3 {
  cd T[8][3][3]; double f[8][8][8];
  SU3() {
    std::memset((void*)T, 0, sizeof(T));
    cd l[8][3][3]; for (int a = 0; a < 8; a++) for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) l[a][i][j] = 0;
    l[0][0][1] = l[0][1][0] = 1;
    l[1][0][1] = -I_; l[1][1][0] = I_;
    l[2][0][0] = 1; l[2][1][1] = -1;
    l[3][0][2] = l[3][2][0] = 1;
    l[4][0][2] = -I_; l[4][2][0] = I_;
    l[5][1][2] = l[5][2][1] = 1;
    l[6][1][2] = -I_; l[6][2][1] = I_;
    double r3 = 1.0 / std::sqrt(3.0); l[7][0][0] = r3; l[7][1][1] = r3; l[7][2][2] = -2.0 * r3;
    for (int a = 0; a < 8; a++) for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) T[a][i][j] = 0.5 * l[a][i][j];
    // [T^a,T^b] = i f^{abc} T^c, Tr T^a T^b = delta/2  =>  f^{abc} = -2i Tr([T^a,T^b] T^c)
    for (int a = 0; a < 8; a++) for (int b = 0; b < 8; b++) for (int c = 0; c < 8; c++) {
      cd tr = 0;
      for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) for (int k = 0; k < 3; k++)
        tr += (T[a][i][j] * T[b][j][k] - T[b][i][j] * T[a][j][k]) * T[c][k][i];
      f[a][b][c] = (-2.0 * I_ * tr).real();
    }
  }
};
static const SU3& SU() { static SU3 s; return s; }

// ---------------------------------------------------------------- n-gluon process g g -> t tbar + (n-2) g
typedef std::vector<int> Tup;                 // ordered tuple of distinct gluon labels = a colour string T^{a_t1}...T^{a_tm}
static Tup cat(const Tup& a, const Tup& b) { Tup r(a); r.insert(r.end(), b.begin(), b.end()); return r; }
static Tup cat3(const Tup& a, const Tup& b, const Tup& c) { return cat(cat(a, b), c); }

struct Kin {            // per event + helicity: the external objects in the notation of SURVEY C5
  int n;                // number of gluons
  double K[8][4];       // k_i = +p_i incoming, -p_i outgoing
  V4 e[8];              // e_i = eps(p_i,l_i) incoming, eps* outgoing
  double pt[4], ptb[4]; // top, antitop momenta
  Sp ubar, v;           // ubar(p_t,l_t), v(p_tbar,l_tbar)
  double mt, Gamma_t, gq, g3, g4;
};
// leg order [g,g,t,tbar,g,...]; gluon label i <-> leg (i<2 ? i : i+2)
static int gluon_leg(int i) { return i < 2 ? i : i + 2; }
static void make_kin(Kin& k, int n, const Par& P, const double* p /*[n+2][4]*/, const int* hel, const cd* eps_override /*[n][4] or null*/) {
  k.n = n; k.mt = P.mt; k.Gamma_t = P.Gamma_t;
  double gs = std::sqrt(4.0 * PI * P.alpha_s);
  k.gq = gs; k.g3 = gs * P.ggg_scale; k.g4 = gs * gs * P.gggg_scale;        // Q2: each coupling constant times its scale
  for (int i = 0; i < n; i++) {
    int leg = gluon_leg(i); const double* q = p + 4 * leg; bool inc = (i < 2);
    for (int mu = 0; mu < 4; mu++) k.K[i][mu] = inc ? q[mu] : -q[mu];
    V4 eps = polvec(q, hel[leg]);
    k.e[i] = inc ? eps : conjv(eps);
    if (eps_override) for (int mu = 0; mu < 4; mu++) k.e[i].c[mu] = eps_override[4 * i + mu];
  }
  for (int mu = 0; mu < 4; mu++) { k.pt[mu] = p[8 + mu]; k.ptb[mu] = p[12 + mu]; }
  k.ubar = bar(spinor_u(k.pt, P.mt, hel[2]));
  k.v = spinor_v(k.ptb, P.mt, hel[3]);
}
static V4 realv(const double a[4]) { V4 r; for (int i = 0; i < 4; i++) r.c[i] = a[i]; return r; }
static double mink2(const double a[4]) { return a[0] * a[0] - a[1] * a[1] - a[2] * a[2] - a[3] * a[3]; }

// Lorentz part of the three-gluon vertex:
// L3^s(A,B) = (JA.JB)(KA-KB)^s + JB^s ((KA+2KB).JA) - JA^s ((2KA+KB).JB)
static V4 L3(const V4& JA, const double KA[4], const V4& JB, const double KB[4]) {
  V4 ka = realv(KA), kb = realv(KB);
  cd ab = dot(JA, JB), c1 = dot(ka + cd(2.0) * kb, JA), c2 = dot(cd(2.0) * ka + kb, JB);
  return ab * (ka - kb) + c1 * JB - c2 * JA;
}

typedef std::map<Tup, V4> GCur;     // matrix-valued gluon current: colour string -> numeric 4-vector
typedef std::map<Tup, Sp> QCur;     // quark-line object: colour string -> numeric spinor
static void addv(GCur& m, const Tup& t, const V4& v) { auto it = m.find(t); if (it == m.end()) m[t] = v; else it->second = it->second + v; }
static void adds(QCur& m, const Tup& t, const Sp& v) { auto it = m.find(t); if (it == m.end()) m[t] = v; else it->second = it->second + v; }

// Route (F): colour as formal strings.  Returns the n! colour-flow amplitudes J_sigma
// (coefficients of (T^{a_s1}...T^{a_sn})_{ij}), permutations in lexicographic order.
static std::vector<cd> jamps_F(const Kin& k) {
  const int n = k.n, full = (1 << n) - 1;
  std::vector<std::array<double, 4>> KS(full + 1);
  for (int S = 0; S <= full; S++) { for (int mu = 0; mu < 4; mu++) { double s = 0; for (int i = 0; i < n; i++) if (S >> i & 1) s += k.K[i][mu]; KS[S][mu] = s; } }
  std::vector<GCur> J(full + 1);
  // subsets in order of increasing size
  std::vector<int> order; for (int sz = 1; sz <= n; sz++) for (int S = 1; S <= full; S++) if (__builtin_popcount(S) == sz) order.push_back(S);
  for (int S : order) {
    if (__builtin_popcount(S) == 1) { int i = __builtin_ctz(S); J[S][Tup{i}] = k.e[i]; continue; }
    GCur acc; int low = S & -S;
    // three-gluon vertex: unordered {A,B}, A contains the lowest label of S
    for (int A = (S - 1) & S; A > 0; A = (A - 1) & S) {
      if (!(A & low)) continue; int B = S ^ A;
      for (auto& ta : J[A]) for (auto& tb : J[B]) {
        V4 l = L3(ta.second, KS[A].data(), tb.second, KS[B].data());
        addv(acc, cat(ta.first, tb.first), cd(-k.g3) * l);          // -g3 ( [A,B] ordered AB ...
        addv(acc, cat(tb.first, ta.first), cd(+k.g3) * l);          //        - same numbers ordered BA )
      }
    }
    // four-gluon vertex: unordered {A,B,C}; A has the lowest label of S, B the lowest of S\A
    for (int A = (S - 1) & S; A > 0; A = (A - 1) & S) {
      if (!(A & low)) continue; int R = S ^ A; int lowR = R & -R;
      for (int B = (R - 1) & R; B > 0; B = (B - 1) & R) {
        if (!(B & lowR)) continue; int C = R ^ B;
        for (auto& ta : J[A]) for (auto& tb : J[B]) for (auto& tc : J[C]) {
          const V4 &a = ta.second, &b = tb.second, &c = tc.second;
          cd ab = dot(a, b), ac = dot(a, c), bc = dot(b, c);
          V4 l1 = ac * b - bc * a, l2 = ab * c - bc * a, l3 = ab * c - ac * b;
          const Tup &x = ta.first, &y = tb.first, &z = tc.first; cd g = k.g4;
          // + g4 [[A,B],C] l1 ; [[A,B],C] = ABC - BAC - CAB + CBA
          addv(acc, cat3(x, y, z), g * l1); addv(acc, cat3(y, x, z), -g * l1); addv(acc, cat3(z, x, y), -g * l1); addv(acc, cat3(z, y, x), g * l1);
          // + g4 [[A,C],B] l2 ; = ACB - CAB - BAC + BCA
          addv(acc, cat3(x, z, y), g * l2); addv(acc, cat3(z, x, y), -g * l2); addv(acc, cat3(y, x, z), -g * l2); addv(acc, cat3(y, z, x), g * l2);
          // - g4 [A,[B,C]] l3 ; [A,[B,C]] = ABC - ACB - BCA + CBA
          addv(acc, cat3(x, y, z), -g * l3); addv(acc, cat3(x, z, y), g * l3); addv(acc, cat3(y, z, x), g * l3); addv(acc, cat3(z, y, x), -g * l3);
        }
      }
    }
    double K2 = mink2(KS[S].data());
    for (auto& t : acc) J[S][t.first] = cd(1.0 / K2) * t.second;      // gluon propagator -i g/q^2 folded as in C5
  }
  // quark line: Psi_0 = v ; Psi_S = P_S sum_{B} i gq Jslash_B Psi_{S\B}, colour: B to the left of S\B
  std::vector<QCur> Psi(full + 1); Psi[0][Tup{}] = k.v;
  std::vector<int> qorder; for (int sz = 1; sz <= n; sz++) for (int S = 1; S <= full; S++) if (__builtin_popcount(S) == sz) qorder.push_back(S);
  std::vector<cd> out;
  for (int S : qorder) {
    QCur acc;
    for (int B = S; B > 0; B = (B - 1) & S) {
      int Rm = S ^ B;
      for (auto& tb : J[B]) { M4 js = slash(tb.second);
        for (auto& tr : Psi[Rm]) adds(acc, cat(tb.first, tr.first), (I_ * k.gq) * (js * tr.second)); }
    }
    if (S != full) {
      double q[4]; for (int mu = 0; mu < 4; mu++) q[mu] = -k.ptb[mu] + KS[S][mu];
      cd den = cd(mink2(q) - k.mt * k.mt, k.mt * k.Gamma_t);
      M4 prop = (I_ / den) * (slash(realv(q)) + cd(k.mt) * GM().one);
      for (auto& t : acc) Psi[S][t.first] = prop * t.second;
    } else {
      Tup perm(n); for (int i = 0; i < n; i++) perm[i] = i;
      do { auto it = acc.find(perm); out.push_back(it == acc.end() ? cd(0) : rowcol(k.ubar, it->second)); } while (std::next_permutation(perm.begin(), perm.end()));
    }
  }
  return out;
}

// Colour matrix C_{ss'} = sum_{a_1..a_n} Tr( T^{a_s1}..T^{a_sn} (T^{a_s'1}..T^{a_s'n})^dagger ), from explicit Gell-Mann matrices.
static const std::vector<double>& colour_matrix(int n) {
  static std::vector<double> cache[8];
  if (cache[n].empty()) {   // first call must come from serial code (orc_* entry points ensure it)
    const SU3& su = SU();
    std::vector<Tup> perms; Tup perm(n); for (int i = 0; i < n; i++) perm[i] = i;
    do perms.push_back(perm); while (std::next_permutation(perm.begin(), perm.end()));
    int np = (int)perms.size(); std::vector<cd> C(np * np, 0.0);
    long ncol = 1; for (int i = 0; i < n; i++) ncol *= 8;
    // plain sum over all 8^n colour assignments; threads only split the outer loop
#pragma omp parallel
    {
      std::vector<std::array<cd, 9>> prod(np);
      std::vector<cd> Cl(np * np, 0.0);
#pragma omp for schedule(static)
      for (long a = 0; a < ncol; a++) {
        int col[8]; long t = a; for (int i = 0; i < n; i++) { col[i] = t % 8; t /= 8; }
        for (int s = 0; s < np; s++) {
          cd m[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
          for (int pos = 0; pos < n; pos++) {
            const cd(*T)[3] = su.T[col[perms[s][pos]]]; cd r[3][3];
            for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) { cd x = 0; for (int l = 0; l < 3; l++) x += m[i][l] * T[l][j]; r[i][j] = x; }
            std::memcpy((void*)m, (void*)r, sizeof(m));
          }
          for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) prod[s][3 * i + j] = m[i][j];
        }
        for (int s = 0; s < np; s++) for (int u = 0; u < np; u++) { cd x = 0; for (int e = 0; e < 9; e++) x += prod[s][e] * std::conj(prod[u][e]); Cl[s * np + u] += x; }
      }
#pragma omp critical(colour_merge)
      for (int i = 0; i < np * np; i++) C[i] += Cl[i];
    }
    cache[n].resize(np * np); for (int i = 0; i < np * np; i++) cache[n][i] = C[i].real();
  }
  return cache[n];
}

static double quadform(const std::vector<cd>& J, const std::vector<double>& C) {
  int np = (int)J.size(); cd s = 0;
  for (int a = 0; a < np; a++) for (int b = 0; b < np; b++) s += std::conj(J[a]) * C[a * np + b] * J[b];
  return s.real();
}
static double denom_qcd(int n) { double f = 1; for (int i = 2; i <= n - 2; i++) f *= i; return 4.0 * 64.0 * f; }  // D = 4*64*(n-2)!

static double me2_qcd_F(int n, const Par& P, const double* p) {
  const std::vector<double>& C = colour_matrix(n);
  int next = n + 2, hel[9]; double sum = 0;
  for (int h = 0; h < (1 << next); h++) {
    for (int i = 0; i < next; i++) hel[i] = ((h >> i) & 1) ? 1 : -1;
    Kin k; make_kin(k, n, P, p, hel, nullptr);
    sum += quadform(jamps_F(k), C);
  }
  return sum / denom_qcd(n);
}

// Route (E): explicit colour.  Component currents J_S^{mu a} with the f^{abc} form of the rules,
// quark line as spinor x colour, loop over all 8^n external gluon colours and the antiquark colour j.
// Returns sum_{colours} sum_{ij} |M_ij|^2 for ONE helicity configuration.
struct GE { V4 c[8]; };
static double me2_hel_E(const Kin& k) {
  const SU3& su = SU(); const int n = k.n, full = (1 << n) - 1;
  std::vector<std::array<double, 4>> KS(full + 1);
  for (int S = 0; S <= full; S++) for (int mu = 0; mu < 4; mu++) { double s = 0; for (int i = 0; i < n; i++) if (S >> i & 1) s += k.K[i][mu]; KS[S][mu] = s; }
  std::vector<int> order; for (int sz = 1; sz <= n; sz++) for (int S = 1; S <= full; S++) if (__builtin_popcount(S) == sz) order.push_back(S);
  long ncol = 1; for (int i = 0; i < n; i++) ncol *= 8;
  double total = 0;
  for (long a = 0; a < ncol; a++) {
    int col[8]; long t = a; for (int i = 0; i < n; i++) { col[i] = t % 8; t /= 8; }
    std::vector<GE> J(full + 1);
    for (int S : order) {
      GE& out = J[S]; for (int d = 0; d < 8; d++) out.c[d] = v4zero();
      if (__builtin_popcount(S) == 1) { int i = __builtin_ctz(S); out.c[col[i]] = k.e[i]; continue; }
      int low = S & -S;
      for (int A = (S - 1) & S; A > 0; A = (A - 1) & S) {
        if (!(A & low)) continue; int B = S ^ A;
        // J^{rho c} += (-i/K^2) g3 f^{abc} L3^rho(J_A^a, J_B^b)
        for (int x = 0; x < 8; x++) for (int y = 0; y < 8; y++) {
          V4 l = L3(J[A].c[x], KS[A].data(), J[B].c[y], KS[B].data());
          for (int c = 0; c < 8; c++) if (su.f[x][y][c] != 0.0) out.c[c] = out.c[c] + (-I_ * k.g3 * su.f[x][y][c]) * l;
        }
      }
      for (int A = (S - 1) & S; A > 0; A = (A - 1) & S) {
        if (!(A & low)) continue; int R = S ^ A; int lowR = R & -R;
        for (int B = (R - 1) & R; B > 0; B = (B - 1) & R) {
          if (!(B & lowR)) continue; int Cc = R ^ B;
          // J^{s d} += (-i/K^2)(-i g4)[ f^{abe}f^{cde} l1 + f^{ace}f^{bde} l2 + f^{ade}f^{bce} l3 ]
          for (int x = 0; x < 8; x++) for (int y = 0; y < 8; y++) for (int z = 0; z < 8; z++) {
            const V4 &va = J[A].c[x], &vb = J[B].c[y], &vc = J[Cc].c[z];
            cd ab = dot(va, vb), ac = dot(va, vc), bc = dot(vb, vc);
            if (ab == 0.0 && ac == 0.0 && bc == 0.0) continue;
            V4 l1 = ac * vb - bc * va, l2 = ab * vc - bc * va, l3 = ab * vc - ac * vb;
            for (int d = 0; d < 8; d++) {
              double c1 = 0, c2 = 0, c3 = 0;
              for (int e = 0; e < 8; e++) { c1 += su.f[x][y][e] * su.f[z][d][e]; c2 += su.f[x][z][e] * su.f[y][d][e]; c3 += su.f[x][d][e] * su.f[y][z][e]; }
              if (c1 != 0.0) out.c[d] = out.c[d] + cd(-k.g4 * c1) * l1;
              if (c2 != 0.0) out.c[d] = out.c[d] + cd(-k.g4 * c2) * l2;
              if (c3 != 0.0) out.c[d] = out.c[d] + cd(-k.g4 * c3) * l3;
            }
          }
        }
      }
      double K2 = mink2(KS[S].data());
      // (-i g3 f) and (-i)(-i g4) = -g4 were applied above; what is left of both propagators is 1/K^2
      for (int d = 0; d < 8; d++) out.c[d] = cd(1.0 / K2) * out.c[d];
    }
    for (int j = 0; j < 3; j++) {          // antiquark colour
      // Psi_S[colour i] spinors
      std::vector<std::array<Sp, 3>> Psi(full + 1);
      for (int i = 0; i < 3; i++) Psi[0][i] = (i == j) ? k.v : spzero();
      cd Mi[3] = {0, 0, 0};
      for (int S : order) {
        std::array<Sp, 3> acc; for (int i = 0; i < 3; i++) acc[i] = spzero();
        for (int B = S; B > 0; B = (B - 1) & S) {
          int Rm = S ^ B;
          for (int c = 0; c < 8; c++) {
            M4 js = slash(J[B].c[c]);
            for (int i = 0; i < 3; i++) for (int l = 0; l < 3; l++) {
              if (su.T[c][i][l] == 0.0) continue;
              acc[i] = acc[i] + (I_ * k.gq * su.T[c][i][l]) * (js * Psi[Rm][l]);     // + i gq gamma^mu T^c
            }
          }
        }
        if (S != full) {
          double q[4]; for (int mu = 0; mu < 4; mu++) q[mu] = -k.ptb[mu] + KS[S][mu];
          cd den = cd(mink2(q) - k.mt * k.mt, k.mt * k.Gamma_t);
          M4 prop = (I_ / den) * (slash(realv(q)) + cd(k.mt) * GM().one);
          for (int i = 0; i < 3; i++) Psi[S][i] = prop * acc[i];
        } else for (int i = 0; i < 3; i++) Mi[i] = rowcol(k.ubar, acc[i]);
      }
      for (int i = 0; i < 3; i++) total += std::norm(Mi[i]);
    }
  }
  return total;
}


// ---------------------------------------------------------------- e+(p1) e-(p2) -> n photons  (Table 1: the paper's own
// measured process is e+ e- -> 5 gamma).  Plain definition: the sum of the n! Feynman diagrams, one per order in
// which the photons leave the electron line (SM, massless electron: no other tree diagram exists):
//   iM = sum_perm vbar(p1) (i e eps-slash*_{sn}) S(q_{n-1}) ... S(q_1) (i e eps-slash*_{s1}) u(p2),   q_j = p2 - k_{s1} - .. - k_{sj},
// with the rules of SURVEY C3: lepton-photon vertex -i e Q gamma^mu (Q = -1), massless propagator S(q) = i q-slash / q^2,
// outgoing photons carry eps* (SURVEY C2).  eps_override ([n][4] complex, used as given) serves the gauge test eps -> k.
static cd amp_epem_ng(const Par& P, int n, const double* p /*[n+2][4]*/, const int* hel /*[n+2]*/, const cd* eps_override) {
  const double e = std::sqrt(4.0 * PI * P.alpha_em), Q = -1.0;
  Sp vb1 = bar(spinor_v(p, 0.0, hel[0])), u2 = spinor_u(p + 4, 0.0, hel[1]);
  std::vector<M4> vert(n);
  for (int i = 0; i < n; i++) {
    V4 eps; if (eps_override) { for (int mu = 0; mu < 4; mu++) eps.c[mu] = eps_override[4 * i + mu]; } else eps = conjv(polvec(p + 4 * (i + 2), hel[i + 2]));
    vert[i] = (-I_ * e * Q) * slash(eps);
  }
  std::vector<int> perm(n); for (int i = 0; i < n; i++) perm[i] = i;
  cd tot = 0;
  do {
    Sp psi = u2; double q[4] = {p[4], p[5], p[6], p[7]};
    for (int j = 0; j < n; j++) {
      psi = vert[perm[j]] * psi;
      if (j + 1 < n) {
        const double* k = p + 4 * (perm[j] + 2); for (int mu = 0; mu < 4; mu++) q[mu] -= k[mu];
        psi = (I_ / mink2(q)) * (slash(realv(q)) * psi);
      }
    }
    tot += rowcol(vb1, psi);
  } while (std::next_permutation(perm.begin(), perm.end()));
  return tot;     // = iM
}
// averaged over the 2x2 initial helicities and divided by n! for the identical photons (reading Q3 applied to this process)
static double me2_epem_ng(const Par& P, int n, const double* p) {
  double sum = 0; int hel[8];
  for (int h = 0; h < (1 << (n + 2)); h++) {          // full helicity sum
    for (int i = 0; i < n + 2; i++) hel[i] = ((h >> i) & 1) ? 1 : -1;
    sum += std::norm(amp_epem_ng(P, n, p, hel, nullptr));
  }
  double fact = 1; for (int i = 2; i <= n; i++) fact *= i;
  return sum / (4.0 * fact);
}
static int process_n_photons(const char* proc) {
  if (!std::strcmp(proc, "epem_aa")) return 2;
  if (!std::strcmp(proc, "epem_aaa")) return 3;
  if (!std::strcmp(proc, "epem_aaaa")) return 4;
  if (!std::strcmp(proc, "epem_aaaaa")) return 5;
  return -1;
}

// ---------------------------------------------------------------- q(p1) qbar(p2) -> t(p3) tbar(p4) [+ g(p5)]
// A structurally different amplitude for the same final states as cfgs 2, 3 (PAPER.md:87 last sentence: "reweighting between structurally
// different amplitude routines"; real emissions "can be treated as LO multiprocesses").  Massless light quark, rules of
// SURVEY C3, explicit SU(3) colour on every leg (the plain definition: sum over all colours of |M|^2):
//   light line as a gluon source   J_A^{mu c} = (-i/Q^2) vbar(p2) (i g gamma^mu T^c) u(p1),  Q = p1 + p2          (incoming momentum K_A = Q)
//   with the gluon (colour a, wavefunction e = eps*(p5), K_g = -p5) radiated off the light line
//     J_B^{mu c} = (-i/Q_B^2) vbar(p2) [ (i g gamma^mu T^c) S0(p1-p5) (i g e-slash T^a) + (i g e-slash T^a) S0(-p2+p5) (i g gamma^mu T^c) ] u(p1)
//   or off the virtual gluon       J_C^{mu c} = (1/Q_B^2) (-i g3 f^{xac}) L3^mu(J_A^x, K_A; e, K_g),   Q_B = p1 + p2 - p5   (as in route E)
//   iM_kl = ubar(p3) [ i g (J_B + J_C)-slash^c T^c + (i g e-slash T^a) S(p3+p5) (i g J_A-slash^c T^c) + (i g J_A-slash^c T^c) S(-p4-p5) (i g e-slash T^a) ]_kl v(p4)
// S(q) = i (q-slash + m_t)/(q^2 - m_t^2), S0 the same with m = 0.  Without the gluon: iM_kl = ubar(p3) (i g J_A-slash^c T^c)_kl v(p4).
// Averaging: 1/(2*2*3*3) (initial helicities and colours); no identical final-state particles.
// eps_override: null or 4 complex numbers replacing e (gauge test).  Returns sum over colours of |M|^2 for ONE helicity configuration.
static double me2_hel_qq(int ng, const Par& P, const double* p, const int* hel, const cd* eps_override) {
  const SU3& su = SU(); const Gammas& G = GM();
  const double g = std::sqrt(4.0 * PI * P.alpha_s), g3 = g * P.ggg_scale, mt = P.mt;
  const double *p1 = p, *p2 = p + 4, *p3 = p + 8, *p4 = p + 12, *p5 = p + 16;
  Sp u1 = spinor_u(p1, 0.0, hel[0]), vb2 = bar(spinor_v(p2, 0.0, hel[1])), ub3 = bar(spinor_u(p3, mt, hel[2])), v4 = spinor_v(p4, mt, hel[3]);
  double KA[4], Kg[4] = {0, 0, 0, 0}, QB[4]; for (int mu = 0; mu < 4; mu++) { KA[mu] = p1[mu] + p2[mu]; QB[mu] = KA[mu]; }
  V4 e = v4zero();
  if (ng) {
    e = conjv(polvec(p5, hel[4])); if (eps_override) for (int mu = 0; mu < 4; mu++) e.c[mu] = eps_override[mu];
    for (int mu = 0; mu < 4; mu++) { Kg[mu] = -p5[mu]; QB[mu] = KA[mu] + Kg[mu]; }
  }
  auto prop = [&](const double q[4], double m) { return (I_ / cd(mink2(q) - m * m)) * (slash(realv(q)) + cd(m) * G.one); };
  const cd ig = I_ * g;
  // colour-stripped Lorentz pieces of the light line
  V4 jA, jB1, jB2;                 // vbar gamma^mu u ; vbar gamma^mu S0 e-slash u (colour T^c T^a) ; vbar e-slash S0 gamma^mu u (colour T^a T^c)
  double k5[4]; for (int mu = 0; mu < 4; mu++) k5[mu] = ng ? p5[mu] : 0.0;      // p5 lies outside the caller's buffer when there is no gluon: never read it then
  double q1[4], q2[4]; for (int mu = 0; mu < 4; mu++) { q1[mu] = p1[mu] - k5[mu]; q2[mu] = -p2[mu] + k5[mu]; }
  for (int mu = 0; mu < 4; mu++) {
    jA.c[mu] = rowcol(vb2, (ig * G.g[mu]) * u1);
    if (ng) {
      jB1.c[mu] = rowcol(vb2, (ig * G.g[mu]) * (prop(q1, 0.0) * ((ig * slash(e)) * u1)));
      jB2.c[mu] = rowcol(vb2, (ig * slash(e)) * (prop(q2, 0.0) * ((ig * G.g[mu]) * u1)));
    }
  }
  const double QA2 = mink2(KA), QB2 = mink2(QB);
  double qt[4], qtb[4]; for (int mu = 0; mu < 4; mu++) { qt[mu] = p3[mu] + k5[mu]; qtb[mu] = -p4[mu] - k5[mu]; }
  double total = 0;
  const int na = ng ? 8 : 1;
  for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) for (int a = 0; a < na; a++) {
    // currents entering the top line, colour component c
    V4 JA[8], JT[8];
    for (int c = 0; c < 8; c++) { JA[c] = ((-I_ / QA2) * su.T[c][j][i]) * jA; JT[c] = v4zero(); }
    if (ng) {
      for (int c = 0; c < 8; c++) {
        cd ca = 0, ac = 0; for (int l = 0; l < 3; l++) { ca += su.T[c][j][l] * su.T[a][l][i]; ac += su.T[a][j][l] * su.T[c][l][i]; }
        JT[c] = (-I_ / QB2) * (ca * jB1 + ac * jB2);
      }
      for (int x = 0; x < 8; x++) {
        V4 l = L3(JA[x], KA, e, Kg);
        for (int c = 0; c < 8; c++) if (su.f[x][a][c] != 0.0) JT[c] = JT[c] + (cd(1.0 / QB2) * (-I_ * g3 * su.f[x][a][c])) * l;
      }
    }
    for (int k = 0; k < 3; k++) for (int l = 0; l < 3; l++) {
      cd M = 0;
      for (int c = 0; c < 8; c++) {
        if (!ng) { if (su.T[c][k][l] != 0.0) M += su.T[c][k][l] * rowcol(ub3, (ig * slash(JA[c])) * v4); continue; }
        if (su.T[c][k][l] != 0.0) M += su.T[c][k][l] * rowcol(ub3, (ig * slash(JT[c])) * v4);
        cd ac = 0, ca = 0; for (int r = 0; r < 3; r++) { ac += su.T[a][k][r] * su.T[c][r][l]; ca += su.T[c][k][r] * su.T[a][r][l]; }
        if (ac != 0.0) M += ac * rowcol(ub3, (ig * slash(e)) * (prop(qt, mt) * ((ig * slash(JA[c])) * v4)));
        if (ca != 0.0) M += ca * rowcol(ub3, (ig * slash(JA[c])) * (prop(qtb, mt) * ((ig * slash(e)) * v4)));
      }
      total += std::norm(M);
    }
  }
  return total;
}
static int process_n_qq(const char* proc) {          // number of radiated gluons, -1 if not a q qbar process
  if (!std::strcmp(proc, "qqx_ttx")) return 0;
  if (!std::strcmp(proc, "qqx_ttxg")) return 1;
  return -1;
}
static double me2_qq(int ng, const Par& P, const double* p) {
  double sum = 0; int hel[5];
  for (int h = 0; h < (1 << (4 + ng)); h++) {          // full helicity sum
    for (int i = 0; i < 4 + ng; i++) hel[i] = ((h >> i) & 1) ? 1 : -1;
    sum += me2_hel_qq(ng, P, p, hel, nullptr);
  }
  return sum / 36.0;
}

// ---------------------------------------------------------------- process table
static int process_n_gluons(const char* proc) {
  if (!std::strcmp(proc, "gg_ttx")) return 2;
  if (!std::strcmp(proc, "gg_ttxg")) return 3;
  if (!std::strcmp(proc, "gg_ttxgg")) return 4;
  if (!std::strcmp(proc, "gg_ttxggg")) return 5;
  return -1;
}
static int process_n_ext(const char* proc) {
  if (!std::strcmp(proc, "epem_mupmum")) return 4;
  int na = process_n_photons(proc); if (na > 0) return na + 2;
  int nq = process_n_qq(proc); if (nq >= 0) return nq + 4;
  int n = process_n_gluons(proc); return n < 0 ? -1 : n + 2;
}
static double me2_any(const char* proc, const Par& P, const double* p) {
  if (!std::strcmp(proc, "epem_mupmum")) { double q[4][4]; std::memcpy(q, p, sizeof(q)); return me2_epem(P, q); }
  int na = process_n_photons(proc); if (na > 0) return me2_epem_ng(P, na, p);
  int nq = process_n_qq(proc); if (nq >= 0) return me2_qq(nq, P, p);
  return me2_qcd_F(process_n_gluons(proc), P, p);
}

extern "C" {

int orc_n_external(const char* proc) { return process_n_ext(proc); }

// |M|^2 of one event; p is AoS [n_ext][4] = (E,px,py,pz)
int orc_me2(const char* proc, const double* par, const double* p, double* out) {
  if (process_n_ext(proc) < 0) return -1; *out = me2_any(proc, par_from(par), p); return 0;
}

// The hot path on a whole event set (SoA momenta as in include/rwgt.h): eq. 3, both parameter sets
// evaluated independently.  nthreads <= 0: all cores.  Returns the number of threads used.
int orc_reweight(const char* proc, const double* par_old, const double* par_new, const double* momenta,
                 const double* weights, double* me_old, double* me_new, double* w_new, long n_events, int nthreads) {
  int next = process_n_ext(proc); if (next < 0) return -1;
  Par Po = par_from(par_old), Pn = par_from(par_new);
  int ng = process_n_gluons(proc); if (ng > 0) colour_matrix(ng);
  int used = 1;
#ifdef _OPENMP
  if (nthreads > 0) omp_set_num_threads(nthreads);
  used = (nthreads > 0) ? nthreads : omp_get_max_threads();
#endif
#pragma omp parallel for schedule(dynamic, 1)
  for (long ev = 0; ev < n_events; ev++) {
    double p[9 * 4];
    for (int ip = 0; ip < next; ip++) for (int mu = 0; mu < 4; mu++) p[4 * ip + mu] = momenta[(ip * 4 + mu) * n_events + ev];
    double a = me2_any(proc, Po, p), b = me2_any(proc, Pn, p);
    me_old[ev] = a; me_new[ev] = b; w_new[ev] = weights[ev] * (b / a);     // eq. 3; IEEE result if a == 0
  }
  return used;
}

// eq. 2 (§2.1): "the total cross section is the sum of all event weights", sigma ~ sum_k W_k.  The plain definition:
// a left-to-right sum in double.  Pin (tests/test_oracle_pins.py): against Python's exactly rounded math.fsum within the
// textbook bound (n-1) 2^-53 sum|W| of recursive summation.
double orc_cross_section(const double* w, long n) { double s = 0.0; for (long k = 0; k < n; k++) s += w[k]; return s; }

// ---- accessors used by the pins -------------------------------------------------------------
void orc_gamma(int mu, double* out32) {            // mu = 0..3, 5 ; 4x4 complex row-major (re,im)
  const M4& g = (mu == 5) ? GM().g5 : GM().g[mu];
  for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { out32[2 * (4 * i + j)] = g.m[i][j].real(); out32[2 * (4 * i + j) + 1] = g.m[i][j].imag(); }
}
void orc_spinor(int kind /*0=u,1=v*/, const double* p, double m, int lam, double* out8) {
  Sp s = kind == 0 ? spinor_u(p, m, lam) : spinor_v(p, m, lam);
  for (int i = 0; i < 4; i++) { out8[2 * i] = s.c[i].real(); out8[2 * i + 1] = s.c[i].imag(); }
}
void orc_polvec(const double* p, int lam, double* out8) {
  V4 e = polvec(p, lam); for (int i = 0; i < 4; i++) { out8[2 * i] = e.c[i].real(); out8[2 * i + 1] = e.c[i].imag(); }
}
int orc_colour_matrix(int n, double* out) { if (n < 1 || n > 5) return -1; const std::vector<double>& C = colour_matrix(n); std::memcpy(out, C.data(), C.size() * sizeof(double)); return 0; }
void orc_fabc(double* out512) { std::memcpy(out512, SU().f, sizeof(double) * 512); }

// colour-flow amplitudes of one helicity configuration; hel[n+2] in leg order, entries +-1;
// eps_override: null or [n][4] complex (re,im) replacing the gluon wavefunctions e_i (gauge test).
int orc_jamps(int n, const double* par, const double* p, const int* hel, const double* eps_override, double* out /*2*n!*/) {
  if (n < 1 || n > 5) return -1;
  Kin k; std::vector<cd> ov;
  if (eps_override) { ov.resize(4 * n); for (int i = 0; i < 4 * n; i++) ov[i] = cd(eps_override[2 * i], eps_override[2 * i + 1]); }
  make_kin(k, n, par_from(par), p, hel, eps_override ? ov.data() : nullptr);
  std::vector<cd> J = jamps_F(k);
  for (size_t i = 0; i < J.size(); i++) { out[2 * i] = J[i].real(); out[2 * i + 1] = J[i].imag(); }
  return (int)J.size();
}
// colour-summed |M_h|^2 of one helicity configuration (no averaging): route F and route E
int orc_me2_hel(int n, const double* par, const double* p, const int* hel, int route /*0=F,1=E*/, double* out) {
  if (n < 1 || n > 5) return -1;
  Kin k; make_kin(k, n, par_from(par), p, hel, nullptr);
  *out = route == 0 ? quadform(jamps_F(k), colour_matrix(n)) : me2_hel_E(k);
  return 0;
}
// helicity amplitude iM of cfg 1 for one helicity configuration
void orc_amp_epem(const double* par, const double* p, const int* hel, double* out2) {
  double q[4][4]; std::memcpy(q, p, sizeof(q)); cd a = amp_epem(par_from(par), q, hel); out2[0] = a.real(); out2[1] = a.imag();
}
double orc_denominator(int n) { return denom_qcd(n); }
// colour-summed |M_h|^2 of q qbar -> t tbar (+ g) for one helicity configuration; eps_override: null or 4 complex (re,im)
int orc_me2_hel_qq(int ng, const double* par, const double* p, const int* hel, const double* eps_override, double* out) {
  if (ng < 0 || ng > 1) return -1;
  cd ov[4]; if (eps_override) for (int i = 0; i < 4; i++) ov[i] = cd(eps_override[2 * i], eps_override[2 * i + 1]);
  *out = me2_hel_qq(ng, par_from(par), p, hel, eps_override ? ov : nullptr); return 0;
}
// helicity amplitude iM of e+ e- -> n photons for one helicity configuration; eps_override as in orc_jamps
void orc_amp_epem_ng(int n, const double* par, const double* p, const int* hel, const double* eps_override, double* out2) {
  std::vector<cd> ov;
  if (eps_override) { ov.resize(4 * n); for (int i = 0; i < 4 * n; i++) ov[i] = cd(eps_override[2 * i], eps_override[2 * i + 1]); }
  cd a = amp_epem_ng(par_from(par), n, p, hel, eps_override ? ov.data() : nullptr); out2[0] = a.real(); out2[1] = a.imag();
}

}  // extern "C"
