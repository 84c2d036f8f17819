// kho.cpp -- CPU ORACLE of one HARM/KHARMA ideal-GRMHD predictor-corrector step.
//
// TEST INFRASTRUCTURE, NOT THE PRODUCT (see kho.h).  Plain, slow, single-threaded, fp64,
// triple loops, no blocking / fusion / reordering beyond what the scheme states.  It shares
// no code with the CUDA path.  Compile with -O2 -ffp-contract=off (no FMA contraction).
// Optional -fopenmp only parallelises zone-independent outer loops (bit-identical results).
//
// Citations: "P:n" = /root/reference/PAPER.md line n.  "S#" = a point the paper leaves open
// (it gives the HARM scheme by citation only); the reading taken is listed in
// DESIGN.md "Readings" and SURVEY.md section 8(c).
//
// Parity pins (tests/test_oracle_*.py, all run with -m "not gpu"):
//   geometry: closed forms sqrt(-g)=Sigma sin(th), lapse, g*ginv=1, Gamma^mu_{mu nu}=d_nu ln sqrt(-g),
//             exact-vs-finite-difference connection, FMKS map end points / symmetry / paper's 2-8x
//   physics : u.u=-1, b.u=0, eq. 1.1 re-assembled from raised-index tensors, rest-frame U,
//             wave speeds vs relativistic velocity addition and the exact perpendicular fast speed
//   recon   : exactness on linear / quadratic data, mirror symmetry
//   LLF     : consistency, mirrored grids;  Flux-CT: d(divB)/dt = 0 for arbitrary fluxes
//   U->P    : P->U->P to 1e-12 in all three metrics; static unmagnetised limit
//   step    : uniform fixed point, linear-mode L1 slope in [-2.1,-1.9], Bondi steadiness
// PARITY UNPINNED (definitions of this build, pinned only by hand-built unit cases):
//   floors (S18), fix-up (S19), ghost fills (S20), dt rule (S22), flag codes and tolerances (S16).

#include "kho.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <vector>

namespace {

constexpr int NG = 3;   // ghost layers (WENO5 needs zones i-3..i+2 around a face)
constexpr int NP = 8;   // primitives: rho, u, ut1, ut2, ut3, B1, B2, B3   ("the eight")
enum { RHO = 0, UU = 1, U1 = 2, U2 = 3, U3 = 4, B1 = 5, B2 = 6, B3 = 7 };

enum { KHO_OK = 0, KHO_EINVAL = -1, KHO_ENOMEM = -2 };

// ---------------------------------------------------------------------------------------------
// Forward-mode dual numbers with two partials (d/dx1, d/dx2): exact derivatives of the metric
// for the connection (S6b: differentiate exactly rather than by a 1e-5 centred difference).
// ---------------------------------------------------------------------------------------------
struct Dual {
  double v, d1, d2;
  Dual() : v(0), d1(0), d2(0) {}
  Dual(double c) : v(c), d1(0), d2(0) {}
  Dual(double v_, double a, double b) : v(v_), d1(a), d2(b) {}
};
inline Dual operator+(Dual a, Dual b) { return Dual(a.v + b.v, a.d1 + b.d1, a.d2 + b.d2); }
inline Dual operator-(Dual a, Dual b) { return Dual(a.v - b.v, a.d1 - b.d1, a.d2 - b.d2); }
inline Dual operator-(Dual a) { return Dual(-a.v, -a.d1, -a.d2); }
inline Dual operator*(Dual a, Dual b) {
  return Dual(a.v * b.v, a.d1 * b.v + a.v * b.d1, a.d2 * b.v + a.v * b.d2);
}
inline Dual operator/(Dual a, Dual b) {
  double q = a.v / b.v;
  return Dual(q, (a.d1 - q * b.d1) / b.v, (a.d2 - q * b.d2) / b.v);
}
inline Dual sin(Dual a) { double c = std::cos(a.v); return Dual(std::sin(a.v), c * a.d1, c * a.d2); }
inline Dual cos(Dual a) { double s = -std::sin(a.v); return Dual(std::cos(a.v), s * a.d1, s * a.d2); }
inline Dual exp(Dual a) { double e = std::exp(a.v); return Dual(e, e * a.d1, e * a.d2); }
inline Dual powc(Dual a, double n) {   // a^n, constant exponent
  double dp = n * std::pow(a.v, n - 1.0);
  return Dual(std::pow(a.v, n), dp * a.d1, dp * a.d2);
}
inline double powc(double a, double n) { return std::pow(a, n); }
using std::sin; using std::cos; using std::exp;

// ---------------------------------------------------------------------------------------------
// C1. Geometry.  Native X = (t,x1,x2,x3); embedding (t,r,theta,phi) for KS / FMKS.
// ---------------------------------------------------------------------------------------------
// FMKS map (ref [61]; S5): r = e^{x1}, theta(x1,x2), phi = x3.  Returns r, theta and the
// Jacobian entries L^theta_1, L^theta_2 (L^r_1 = r, L^t_t = L^phi_3 = 1).
template <class T>
void fmks_map(const kho_params& p, T x1, T x2, T& r, T& th, T& dth1, T& dth2) {
  const double pi = M_PI;
  r = exp(x1);
  T y = 2.0 * x2 - 1.0;
  T thG = pi * x2 + 0.5 * (1.0 - p.hslope) * sin(2.0 * pi * x2);
  T dthG = pi * (T(1.0) + (1.0 - p.hslope) * cos(2.0 * pi * x2));
  double norm = 0.5 * pi / (1.0 + std::pow(p.poly_xt, -p.poly_alpha) / (p.poly_alpha + 1.0));
  T ya = powc(y / p.poly_xt, p.poly_alpha);
  T thJ = norm * y * (T(1.0) + ya / (p.poly_alpha + 1.0)) + 0.5 * pi;
  T dthJ = 2.0 * norm * (T(1.0) + ya);
  T e = exp(p.mks_smooth * (T(p.xmin[0]) - x1));
  th = thG + e * (thJ - thG);
  dth1 = -p.mks_smooth * e * (thJ - thG);
  dth2 = dthG + e * (dthJ - dthG);
}

// Kerr-Schild covariant metric in (t,r,theta,phi) (S4).
template <class T>
void gcov_ks(double a, T r, T th, T g[4][4]) {
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) g[m][n] = T(0.0);
  T s = sin(th), c = cos(th);
  T s2 = s * s;
  T Sig = r * r + a * a * c * c;
  T f = 2.0 * r / Sig;
  g[0][0] = -(T(1.0) - f);
  g[0][1] = g[1][0] = f;
  g[0][3] = g[3][0] = -a * f * s2;
  g[1][1] = T(1.0) + f;
  g[1][3] = g[3][1] = -a * s2 * (T(1.0) + f);
  g[2][2] = Sig;
  g[3][3] = s2 * (Sig + a * a * s2 * (T(1.0) + f));
}

// Covariant metric in native coordinates: g_native = L^T g_KS L.
template <class T>
void gcov_native(const kho_params& p, T x1, T x2, T g[4][4]) {
  if (p.coords == KHO_MINKOWSKI) {
    for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) g[m][n] = T(m == n ? (m == 0 ? -1.0 : 1.0) : 0.0);
    return;
  }
  T gks[4][4];
  if (p.coords == KHO_KS) { gcov_ks(p.a, x1, x2, g); return; }
  T r, th, dth1, dth2;
  fmks_map(p, x1, x2, r, th, dth1, dth2);
  gcov_ks(p.a, r, th, gks);
  T L[4][4];   // L[emb][native] = d X_emb / d X_native
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) L[m][n] = T(0.0);
  L[0][0] = T(1.0); L[1][1] = r; L[2][1] = dth1; L[2][2] = dth2; L[3][3] = T(1.0);
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) {
    T s(0.0);
    for (int al = 0; al < 4; al++) for (int be = 0; be < 4; be++) s = s + L[al][m] * gks[al][be] * L[be][n];
    g[m][n] = s;
  }
}

double det3(const double m[3][3]) {
  return m[0][0] * (m[1][1] * m[2][2] - m[1][2] * m[2][1]) - m[0][1] * (m[1][0] * m[2][2] - m[1][2] * m[2][0]) +
         m[0][2] * (m[1][0] * m[2][1] - m[1][1] * m[2][0]);
}
// 4x4 inverse by the adjugate (definition); returns det.
double invert4(const double g[4][4], double inv[4][4]) {
  double cof[4][4];
  for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) {
    double m[3][3];
    int rr = 0;
    for (int i = 0; i < 4; i++) {
      if (i == r) continue;
      int cc = 0;
      for (int j = 0; j < 4; j++) { if (j == c) continue; m[rr][cc++] = g[i][j]; }
      rr++;
    }
    cof[r][c] = (((r + c) & 1) ? -1.0 : 1.0) * det3(m);
  }
  double det = 0.0;
  for (int c = 0; c < 4; c++) det += g[0][c] * cof[0][c];
  for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) inv[r][c] = cof[c][r] / det;
  return det;
}

struct Geom { double gcov[4][4], gcon[4][4], gdet, alpha; };

// S6a: g^{mu nu} is the inverse of g_{mu nu} and sqrt(-g) the root of its determinant.  For KS / FMKS both
// are evaluated from their CLOSED FORMS -- the Kerr-Schild inverse metric
//   g^tt = -(1+2r/Sig), g^tr = 2r/Sig, g^rr = Delta/Sig, g^rphi = a/Sig, g^thth = 1/Sig, g^phph = 1/(Sig sin^2 th)
// pushed through the inverse Jacobian of the coordinate map, and sqrt(-g) = Sig |sin th| r |dth/dx2| --
// because the generic cofactor inverse loses ~(condition number) x eps near the polar axis (measured 1e-11
// between two inversion algorithms).  The generic invert4() stays as the definition the closed form is
// pinned against (tests: g * g^-1 = 1, det).
void geom_at(const kho_params& p, double x1, double x2, Geom& G) {
  gcov_native<double>(p, x1, x2, G.gcov);
  if (p.coords == KHO_MINKOWSKI) {
    for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) G.gcon[m][n] = G.gcov[m][n];
    G.gdet = 1.0; G.alpha = 1.0;
    return;
  }
  double r, th, t1 = 0.0, t2 = 1.0, jr = 1.0;     // jr = dr/dx1, t1 = dth/dx1, t2 = dth/dx2
  if (p.coords == KHO_KS) { r = x1; th = x2; }
  else { fmks_map<double>(p, x1, x2, r, th, t1, t2); jr = r; }
  double s = std::sin(th), c = std::cos(th);
  double Sig = r * r + p.a * p.a * c * c, f = 2.0 * r / Sig;
  double ks[4][4] = {{0}};
  ks[0][0] = -(1.0 + f);
  ks[0][1] = ks[1][0] = f;
  ks[1][1] = (r * r - 2.0 * r + p.a * p.a) / Sig;
  ks[1][3] = ks[3][1] = p.a / Sig;
  ks[2][2] = 1.0 / Sig;
  ks[3][3] = 1.0 / (Sig * s * s);
  double M[4][4] = {{0}};                          // M[native][emb] = d X_native / d X_emb
  M[0][0] = 1.0; M[1][1] = 1.0 / jr; M[2][1] = -t1 / (jr * t2); M[2][2] = 1.0 / t2; M[3][3] = 1.0;
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) {
    double acc = 0.0;
    for (int al = 0; al < 4; al++) for (int be = 0; be < 4; be++) acc += M[m][al] * ks[al][be] * M[n][be];
    G.gcon[m][n] = acc;
  }
  G.gdet = std::fabs(Sig * s * jr * t2);
  G.alpha = 1.0 / std::sqrt(-G.gcon[0][0]);
}
void geom_zero(Geom& G) { std::memset(&G, 0, sizeof(G)); }

// Gamma^lam_{mu nu} = 1/2 g^{lam kap} (d_mu g_{kap nu} + d_nu g_{kap mu} - d_kap g_{mu nu}),  d_t = d_3 = 0.
void conn_from_dg(const double gcon[4][4], const double dg[4][4][4] /* dg[k][m][n] = d_k g_mn */, double conn[64]) {
  for (int lam = 0; lam < 4; lam++) for (int mu = 0; mu < 4; mu++) for (int nu = 0; nu < 4; nu++) {
    double s = 0.0;
    for (int kap = 0; kap < 4; kap++) s += gcon[lam][kap] * (dg[mu][kap][nu] + dg[nu][kap][mu] - dg[kap][mu][nu]);
    conn[(lam * 4 + mu) * 4 + nu] = 0.5 * s;
  }
}
void conn_exact(const kho_params& p, double x1, double x2, double conn[64]) {
  Dual g[4][4];
  gcov_native<Dual>(p, Dual(x1, 1.0, 0.0), Dual(x2, 0.0, 1.0), g);
  double dg[4][4][4];
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) {
    dg[0][m][n] = 0.0; dg[1][m][n] = g[m][n].d1; dg[2][m][n] = g[m][n].d2; dg[3][m][n] = 0.0;
  }
  Geom G;
  geom_at(p, x1, x2, G);
  conn_from_dg(G.gcon, dg, conn);
}
void conn_fd(const kho_params& p, double x1, double x2, double h, double conn[64]) {
  double gc[4][4], gi[4][4], dg[4][4][4], gp[4][4], gm[4][4];
  gcov_native<double>(p, x1, x2, gc);
  invert4(gc, gi);
  std::memset(dg, 0, sizeof(dg));
  gcov_native<double>(p, x1 + h, x2, gp); gcov_native<double>(p, x1 - h, x2, gm);
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) dg[1][m][n] = (gp[m][n] - gm[m][n]) / (2 * h);
  gcov_native<double>(p, x1, x2 + h, gp); gcov_native<double>(p, x1, x2 - h, gm);
  for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) dg[2][m][n] = (gp[m][n] - gm[m][n]) / (2 * h);
  conn_from_dg(gi, dg, conn);
}

double radius_at(const kho_params& p, double x1) {
  if (p.coords == KHO_KS) return x1;
  if (p.coords == KHO_FMKS) return std::exp(x1);
  return 1.0;
}

// ---------------------------------------------------------------------------------------------
// C2. Point-wise physics.
// ---------------------------------------------------------------------------------------------
struct FourVec { double ucon[4], ucov[4], bcon[4], bcov[4], bsq; };

void lower(const double gcov[4][4], const double vcon[4], double vcov[4]) {
  for (int m = 0; m < 4; m++) {
    double s = 0.0;
    for (int n = 0; n < 4; n++) s += gcov[m][n] * vcon[n];
    vcov[m] = s;
  }
}

// q^2 = g_ij ut^i ut^j ; gamma = sqrt(1+q^2) ; u^t = gamma/alpha ; u^i = ut^i - gamma alpha g^{ti}   (S1, ref [32])
// b^t = B^i u_i ; b^i = (B^i + b^t u^i)/u^t
void four_vectors(const double gcov[4][4], const double gcon[4][4], const double P[NP], FourVec& D) {
  double qsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) qsq += gcov[i][j] * P[U1 + i - 1] * P[U1 + j - 1];
  double gamma = std::sqrt(1.0 + qsq);
  double alpha = 1.0 / std::sqrt(-gcon[0][0]);
  D.ucon[0] = gamma / alpha;
  for (int i = 1; i < 4; i++) D.ucon[i] = P[U1 + i - 1] - gamma * alpha * gcon[0][i];
  lower(gcov, D.ucon, D.ucov);
  D.bcon[0] = P[B1] * D.ucov[1] + P[B2] * D.ucov[2] + P[B3] * D.ucov[3];
  for (int i = 1; i < 4; i++) D.bcon[i] = (P[B1 + i - 1] + D.bcon[0] * D.ucon[i]) / D.ucon[0];
  lower(gcov, D.bcon, D.bcov);
  D.bsq = 0.0;
  for (int m = 0; m < 4; m++) D.bsq += D.bcon[m] * D.bcov[m];
}

// T^dir_nu = (w + b^2) u^dir u_nu + (p + b^2/2) delta^dir_nu - b^dir b_nu        [eq. 1.1, P:347]
void stress_row(const double P[NP], const FourVec& D, double gam, int dir, double T[4]) {
  double pg = (gam - 1.0) * P[UU];
  double w = P[RHO] + P[UU] + pg;
  double eta = w + D.bsq;
  double ptot = pg + 0.5 * D.bsq;
  for (int nu = 0; nu < 4; nu++)
    T[nu] = eta * D.ucon[dir] * D.ucov[nu] + (dir == nu ? ptot : 0.0) - D.bcon[dir] * D.bcov[nu];
}

// dir = 0: U = sqrt(-g)(rho u^t, T^t_t + rho u^t, T^t_i, B^i)   (S8: rest mass removed from the energy slot)
// dir = d: F^d = sqrt(-g)(rho u^d, T^d_t + rho u^d, T^d_i, b^i u^d - b^d u^i)
void prim_to_flux(const Geom& G, const double P[NP], const FourVec& D, double gam, int dir, double F[NP]) {
  double T[4];
  stress_row(P, D, gam, dir, T);
  double rhou = P[RHO] * D.ucon[dir];
  F[RHO] = G.gdet * rhou;
  F[UU] = G.gdet * (T[0] + rhou);
  F[U1] = G.gdet * T[1];
  F[U2] = G.gdet * T[2];
  F[U3] = G.gdet * T[3];
  for (int i = 1; i < 4; i++) {
    if (dir == 0) F[B1 + i - 1] = G.gdet * P[B1 + i - 1];
    else F[B1 + i - 1] = G.gdet * (D.bcon[i] * D.ucon[dir] - D.bcon[dir] * D.ucon[i]);
  }
}

// Fast-magnetosonic signal speeds in direction dir (S9).
void vchar(const Geom& G, const double P[NP], const FourVec& D, double gam, int dir, double& vmax, double& vmin) {
  double ef = P[RHO] + gam * P[UU];
  double ee = D.bsq + ef;
  double va2 = D.bsq / ee;
  double cs2 = gam * (gam - 1.0) * P[UU] / ef;
  double cms2 = cs2 + va2 - cs2 * va2;
  if (!(cms2 >= 0.0)) cms2 = 0.0;    // also catches NaN
  if (cms2 > 1.0) cms2 = 1.0;
  double ut = D.ucon[0], ud = D.ucon[dir];
  double A = ut * ut - (G.gcon[0][0] + ut * ut) * cms2;
  double B = 2.0 * (ud * ut - (G.gcon[0][dir] + ud * ut) * cms2);
  double C = ud * ud - (G.gcon[dir][dir] + ud * ud) * cms2;
  // Discriminant B^2 - 4AC in its algebraically reduced form: the O(1) terms (u^d u^t)^2 - (u^t)^2 (u^d)^2
  // cancel identically, leaving  4 c_m^2 [ (1-c_m^2)(u^t^2 g^dd - 2 u^t u^d g^td + u^d^2 g^tt) + c_m^2 (g^td^2 - g^tt g^dd) ].
  // Same number; the naive form loses eps/c_m^2 in cold zones (measured 1e-8 relative on ctop).
  double disc = 4.0 * cms2 * ((1.0 - cms2) * (ut * ut * G.gcon[dir][dir] - 2.0 * ut * ud * G.gcon[0][dir] + ud * ud * G.gcon[0][0]) +
                              cms2 * (G.gcon[0][dir] * G.gcon[0][dir] - G.gcon[0][0] * G.gcon[dir][dir]));
  if (!(disc >= 0.0)) disc = 0.0;
  double sq = std::sqrt(disc);
  // roots of A v^2 - B v + C = 0 (dispersion relation of a wave (-omega, k e_dir) with v = omega/k)
  double vp = (B + sq) / (2.0 * A), vm = (B - sq) / (2.0 * A);
  vmax = vp > vm ? vp : vm;
  vmin = vp > vm ? vm : vp;
}

// ---------------------------------------------------------------------------------------------
// C3. Reconstruction on a 5-point stencil q[0..4] = q_{i-2..i+2}: the zone's left (i-1/2) and
// right (i+1/2) face values.
// ---------------------------------------------------------------------------------------------
void recon_mc(const double q[5], double& left, double& right) {   // S11
  double dm = 2.0 * (q[2] - q[1]), dp = 2.0 * (q[3] - q[2]), dc = 0.5 * (q[3] - q[1]);
  double slope = 0.0;
  if (dm * dp > 0.0) {
    slope = dc;
    if (std::fabs(dm) < std::fabs(slope)) slope = dm;
    if (std::fabs(dp) < std::fabs(slope)) slope = dp;
  }
  left = q[2] - 0.5 * slope;
  right = q[2] + 0.5 * slope;
}
double weno5_right(double x1, double x2, double x3, double x4, double x5) {   // S12, Jiang-Shu
  const double eps = 1e-26;
  double b1 = 13.0 / 12.0 * (x1 - 2 * x2 + x3) * (x1 - 2 * x2 + x3) + 0.25 * (x1 - 4 * x2 + 3 * x3) * (x1 - 4 * x2 + 3 * x3);
  double b2 = 13.0 / 12.0 * (x2 - 2 * x3 + x4) * (x2 - 2 * x3 + x4) + 0.25 * (x4 - x2) * (x4 - x2);
  double b3 = 13.0 / 12.0 * (x3 - 2 * x4 + x5) * (x3 - 2 * x4 + x5) + 0.25 * (3 * x3 - 4 * x4 + x5) * (3 * x3 - 4 * x4 + x5);
  double v1 = x1 / 3.0 - 7.0 * x2 / 6.0 + 11.0 * x3 / 6.0;
  double v2 = -x2 / 6.0 + 5.0 * x3 / 6.0 + x4 / 3.0;
  double v3 = x3 / 3.0 + 5.0 * x4 / 6.0 - x5 / 6.0;
  double w1 = 0.1 / ((eps + b1) * (eps + b1));
  double w2 = 0.6 / ((eps + b2) * (eps + b2));
  double w3 = 0.3 / ((eps + b3) * (eps + b3));
  return (w1 * v1 + w2 * v2 + w3 * v3) / (w1 + w2 + w3);
}
void recon_weno5(const double q[5], double& left, double& right) {
  right = weno5_right(q[0], q[1], q[2], q[3], q[4]);
  left = weno5_right(q[4], q[3], q[2], q[1], q[0]);   // mirror image
}
void recon(int kind, const double q[5], double& left, double& right) {
  if (kind == KHO_RECON_WENO5) recon_weno5(q, left, right); else recon_mc(q, left, right);
}

// ---------------------------------------------------------------------------------------------
// C4. Local Lax-Friedrichs flux at one face (S14).
// ---------------------------------------------------------------------------------------------
void llf(const Geom& G, const double PL[NP], const double PR[NP], double gam, int dir, double F[NP], double& ctop) {
  FourVec DL, DR;
  double UL[NP], UR[NP], FL[NP], FR[NP];
  four_vectors(G.gcov, G.gcon, PL, DL);
  four_vectors(G.gcov, G.gcon, PR, DR);
  prim_to_flux(G, PL, DL, gam, 0, UL);
  prim_to_flux(G, PR, DR, gam, 0, UR);
  prim_to_flux(G, PL, DL, gam, dir, FL);
  prim_to_flux(G, PR, DR, gam, dir, FR);
  double vmaxL, vminL, vmaxR, vminR;
  vchar(G, PL, DL, gam, dir, vmaxL, vminL);
  vchar(G, PR, DR, gam, dir, vmaxR, vminR);
  double cmax = std::fmax(0.0, std::fmax(vmaxL, vmaxR));
  double cmin = std::fmax(0.0, std::fmax(-vminL, -vminR));
  ctop = std::fmax(cmax, cmin);
  for (int v = 0; v < NP; v++) F[v] = 0.5 * (FL[v] + FR[v] - ctop * (UR[v] - UL[v]));
}

// ---------------------------------------------------------------------------------------------
// C6. Geometric source  S_nu = sqrt(-g) T^kap_lam Gamma^lam_{nu kap}  -> slots UU, U1..U3.
// ---------------------------------------------------------------------------------------------
void source(const Geom& G, const double conn[64], const double P[NP], double gam, double S[NP]) {
  FourVec D;
  four_vectors(G.gcov, G.gcon, P, D);
  double T[4][4];
  for (int kap = 0; kap < 4; kap++) stress_row(P, D, gam, kap, T[kap]);
  for (int v = 0; v < NP; v++) S[v] = 0.0;
  for (int nu = 0; nu < 4; nu++) {
    double s = 0.0;
    for (int kap = 0; kap < 4; kap++) for (int lam = 0; lam < 4; lam++) s += T[kap][lam] * conn[(lam * 4 + nu) * 4 + kap];
    S[UU + nu] = G.gdet * s;
  }
}

// ---------------------------------------------------------------------------------------------
// C7. U -> P: the 1D_W scheme of ref [37] in the W' = W - D variable (S16).
// ---------------------------------------------------------------------------------------------
struct U2PCtx { double D, Bsq, QdotB, QdotBsq, Qtsq, Ep, gam; };

double u2p_vsq(const U2PCtx& c, double W) {
  return (c.Qtsq * W * W + c.QdotBsq * (c.Bsq + 2.0 * W)) / ((c.Bsq + W) * (c.Bsq + W) * W * W);
}
// f(W') and f'(W') with v^2 clamped to [0, 1-1e-12] inside the iteration
void u2p_func(const U2PCtx& c, double Wp, double& f, double& df) {
  double W = Wp + c.D;
  double vsq = u2p_vsq(c, W);
  if (vsq < 0.0) vsq = 0.0;
  if (vsq > 1.0 - 1e-12) vsq = 1.0 - 1e-12;
  double gsq = 1.0 / (1.0 - vsq), g = std::sqrt(gsq);
  double k = (c.gam - 1.0) / c.gam;
  double p = k * (Wp - c.D * vsq * gsq / (1.0 + g)) / gsq;
  f = Wp - p + 0.5 * c.Bsq * (1.0 + vsq) - c.QdotBsq / (2.0 * W * W) - c.Ep;
  double W3 = W * W * W, WB = W + c.Bsq;
  double dvsq = -2.0 * (c.Qtsq * W3 + c.QdotBsq * (3.0 * W * W + 3.0 * W * c.Bsq + c.Bsq * c.Bsq)) / (W3 * WB * WB * WB);
  double dp = k * ((1.0 - vsq) - (W - 0.5 * c.D * g) * dvsq);
  df = 1.0 - dp + 0.5 * c.Bsq * dvsq + c.QdotBsq / W3;
}

int u2p(const Geom& G, const double U[NP], const double Pg[NP], double gam, double Pout[NP]) {
  for (int v = 0; v < NP; v++) Pout[v] = Pg[v];
  // B is always updated (primitive B^i = U_{5..7}/sqrt(-g))
  for (int i = 0; i < 3; i++) Pout[B1 + i] = U[B1 + i] / G.gdet;
  bool finite = true;
  for (int v = 0; v < NP; v++) if (!std::isfinite(U[v])) finite = false;
  if (!finite || !(U[RHO] > 0.0)) return 1;

  double alpha = G.alpha, k = alpha / G.gdet;
  U2PCtx c;
  c.gam = gam;
  c.D = k * U[RHO];
  double Bc[4] = {0.0, k * U[B1], k * U[B2], k * U[B3]};   // script-B^i = alpha B^i_prim
  double Qcov[4] = {k * (U[UU] - U[RHO]), k * U[U1], k * U[U2], k * U[U3]};
  double Qcon[4];
  for (int m = 0; m < 4; m++) { double s = 0.0; for (int n = 0; n < 4; n++) s += G.gcon[m][n] * Qcov[n]; Qcon[m] = s; }
  c.Bsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) c.Bsq += G.gcov[i][j] * Bc[i] * Bc[j];
  c.QdotB = Qcov[1] * Bc[1] + Qcov[2] * Bc[2] + Qcov[3] * Bc[3];
  c.QdotBsq = c.QdotB * c.QdotB;
  double Qdotn = -alpha * Qcon[0];
  c.Ep = -Qdotn - c.D;
  double ncon[4];
  for (int m = 0; m < 4; m++) ncon[m] = -alpha * G.gcon[m][0];
  double Qtcon[4];
  for (int m = 0; m < 4; m++) Qtcon[m] = Qcon[m] + Qdotn * ncon[m];
  // Qt^2 = Q.Q + (Q.n)^2, evaluated as the spatial norm g_ij Qt^i Qt^j of the projected vector (Qt^t = 0
  // identically): the same number without the cancellation of two O(W^2) terms, so it can never come out
  // negative by round-off and flip the v^2 >= 0 post-check (S16 / S15b: flags must not depend on rounding).
  c.Qtsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) c.Qtsq += G.gcov[i][j] * Qtcon[i] * Qtcon[j];

  // guess from the guess primitives: W0 = (rho + Gamma u)(1 + q^2)
  double qsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) qsq += G.gcov[i][j] * Pg[U1 + i - 1] * Pg[U1 + j - 1];
  double W = (Pg[RHO] + gam * Pg[UU]) * (1.0 + qsq);
  if (!(W > 0.0) || !std::isfinite(W)) W = c.D;
  for (int it = 0; it < 30 && !(u2p_vsq(c, W) < 1.0); it++) W *= 10.0;
  double Wp = W - c.D;

  bool converged = false;
  for (int it = 0; it < 20; it++) {
    double f, df;
    u2p_func(c, Wp, f, df);
    double Wold = Wp + c.D;
    double Wpn = Wp - f / df;
    if (!(Wpn + c.D > 0.0)) Wpn = 0.5 * Wold - c.D;     // new W <= 0: halve the old W instead
    double dW = Wpn - Wp;
    Wp = Wpn;
    if (std::fabs(dW) <= 1e-12 * (Wp + c.D)) { converged = true; break; }
  }
  if (!converged) return 2;

  W = Wp + c.D;
  double vsq = u2p_vsq(c, W);
  if (!(vsq >= 0.0) || !(vsq < 1.0) || !(W > 0.0)) return 3;
  double gsq = 1.0 / (1.0 - vsq), g = std::sqrt(gsq);
  double rho = c.D / g;
  double u = (Wp - c.D * vsq * gsq / (1.0 + g)) / (gsq * gam);
  double ut[3];
  for (int i = 1; i < 4; i++) ut[i - 1] = g / (W + c.Bsq) * (Qtcon[i] + c.QdotB * Bc[i] / W);
  if (!std::isfinite(rho) || !std::isfinite(u) || !std::isfinite(ut[0]) || !std::isfinite(ut[1]) || !std::isfinite(ut[2]))
    return 7;
  bool badrho = !(rho > 0.0), badu = (u < 0.0);
  if (badrho && badu) return 6;
  if (badrho) return 4;
  if (badu) return 5;
  Pout[RHO] = rho; Pout[UU] = u;
  Pout[U1] = ut[0]; Pout[U2] = ut[1]; Pout[U3] = ut[2];
  return 0;
}

// ---------------------------------------------------------------------------------------------
// C7b. U -> P by the bracketed root find of Kastaun, Kalinani & Ciolfi ("the robust primitive
// variable recovery of [27], which greatly improves stability"; reading S24 in DESIGN.md).  Written in the
// paper's notation.  Inputs seen by the normal observer (same as in u2p above): D, tau = E - D, S_i, B^i;
//   q = tau/D,  r_i = S_i/D,  b^i = B^i/sqrt(D),  h0 = 1 (ideal gas, eps >= 0),  v0^2 = r^2/(h0^2 + r^2);
// functions of the unknown mu = 1/(W h):
//   x = 1/(1 + mu b^2),  rbar^2 = r^2 x^2 + mu x (1 + x) (r.b)^2,  qbar = q - b^2/2 - mu^2 x^2 (b^2 r_perp^2)/2,
//   b^2 r_perp^2 = b^2 r^2 - (r.b)^2;
// master function: vhat^2 = min(mu^2 rbar^2, v0^2), What = (1 - vhat^2)^(-1/2), rhohat = D/What,
//   epshat = What (qbar - mu rbar^2) + vhat^2 What^2/(1 + What), clamped to eps >= 0 inside f only,
//   ahat = p(rhohat, epshat)/(rhohat (1 + epshat)),  nuA = (1 + ahat)(1 + epshat)/What,
//   nuB = (1 + ahat)(1 + qbar - mu rbar^2),  f(mu) = mu - 1/(max(nuA, nuB) + rbar^2 mu);
// bracket (0, mu+], mu+ = 1/h0 if r < h0, else the root of fa(mu) = mu sqrt(h0^2 + rbar^2(mu)) - 1 in (0, 1/h0];
// velocity v^i = mu x (r^i + mu (r.b) b^i), ut^i = What v^i.
// Root finder (the paper uses a library bracketing method; S24): Illinois regula falsi on the bracket for 40 evaluations,
// plain bisection after that; stop when the bracket is narrower than 4e-16 of its upper end, cannot be split any more or
// f vanishes; at most 100 evaluations (flag 2 otherwise: reached only through NaN).
// Flags as for u2p: 1 bad input, 2 not converged, 3 speed limit v0 acted at the root, 5 eps < 0 at the root (the
// hydro primitives keep the guess), 7 non-finite result.
// ---------------------------------------------------------------------------------------------
struct KastaunCtx {
  double D, q, rsq, bsq, rbsq, brperp, v0sq, gam;
};
void kastaun_aux(const KastaunCtx& c, double mu, double& x, double& rbarsq, double& qbar) {
  x = 1.0 / (1.0 + mu * c.bsq);
  rbarsq = c.rsq * x * x + mu * x * (1.0 + x) * c.rbsq;
  qbar = c.q - 0.5 * c.bsq - 0.5 * mu * mu * x * x * c.brperp;
}
// the master function; also returns the (unclamped) pieces evaluated at mu
double kastaun_f(const KastaunCtx& c, double mu, double& vsq_raw, double& W, double& eps_raw) {
  double x, rbarsq, qbar;
  kastaun_aux(c, mu, x, rbarsq, qbar);
  vsq_raw = mu * mu * rbarsq;
  double vsq = vsq_raw < c.v0sq ? vsq_raw : c.v0sq;
  W = 1.0 / std::sqrt(1.0 - vsq);
  eps_raw = W * (qbar - mu * rbarsq) + vsq * W * W / (1.0 + W);
  double eps = eps_raw > 0.0 ? eps_raw : 0.0;
  double a = (c.gam - 1.0) * eps / (1.0 + eps);          // p/(rho (1 + eps)), p = (Gamma - 1) rho eps
  double nuA = (1.0 + a) * (1.0 + eps) / W;
  double nuB = (1.0 + a) * (1.0 + qbar - mu * rbarsq);
  double nu = nuA > nuB ? nuA : nuB;
  return mu - 1.0 / (nu + rbarsq * mu);
}
double kastaun_fa(const KastaunCtx& c, double mu) {
  double x, rbarsq, qbar;
  kastaun_aux(c, mu, x, rbarsq, qbar);
  return mu * std::sqrt(1.0 + rbarsq) - 1.0;              // h0 = 1
}
// Illinois regula falsi on [a, b] with fn(a) < 0 <= fn(b).  Returns false if 100 evaluations do not converge.
template <class Fn>
bool illinois(Fn fn, double a, double fa, double b, double fb, double& lo, double& hi) {
  int side = 0;
  for (int it = 0; it < 100; it++) {
    if (!(b - a > 4e-16 * b)) { lo = a; hi = b; return true; }
    double m = (it < 40) ? b - fb * (b - a) / (fb - fa) : 0.5 * (a + b);    // after 40 evaluations: plain bisection
    if (!(m > a && m < b)) m = 0.5 * (a + b);
    if (!(m > a && m < b)) { lo = a; hi = b; return true; }                 // a and b are neighbouring numbers
    double fm = fn(m);
    if (fm == 0.0) { lo = hi = m; return true; }
    if (fm > 0.0) { b = m; fb = fm; if (side == 1) fa *= 0.5; side = 1; }
    else if (fm < 0.0) { a = m; fa = fm; if (side == -1) fb *= 0.5; side = -1; }
    else return false;                                      // NaN
  }
  return false;
}

int u2p_kastaun(const Geom& G, const double U[NP], const double Pg[NP], double gam, double Pout[NP]) {
  for (int v = 0; v < NP; v++) Pout[v] = Pg[v];
  for (int i = 0; i < 3; i++) Pout[B1 + i] = U[B1 + i] / G.gdet;
  bool finite = true;
  for (int v = 0; v < NP; v++) if (!std::isfinite(U[v])) finite = false;
  if (!finite || !(U[RHO] > 0.0)) return 1;

  // normal-observer quantities, as in u2p
  double alpha = G.alpha, k = alpha / G.gdet;
  double D = k * U[RHO];
  double Bc[4] = {0.0, k * U[B1], k * U[B2], k * U[B3]};
  double Qcov[4] = {k * (U[UU] - U[RHO]), k * U[U1], k * U[U2], k * U[U3]};
  double Qcon[4];
  for (int m = 0; m < 4; m++) { double s = 0.0; for (int n = 0; n < 4; n++) s += G.gcon[m][n] * Qcov[n]; Qcon[m] = s; }
  double Qdotn = -alpha * Qcon[0];
  double tau = -Qdotn - D;
  double Scon[4];                                          // S^i = gamma^{ij} S_j: projection of Q^mu normal to n
  for (int m = 0; m < 4; m++) Scon[m] = Qcon[m] + Qdotn * (-alpha * G.gcon[m][0]);
  double Ssq = 0.0, Bsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) { Ssq += G.gcov[i][j] * Scon[i] * Scon[j]; Bsq += G.gcov[i][j] * Bc[i] * Bc[j]; }
  double SdotB = Qcov[1] * Bc[1] + Qcov[2] * Bc[2] + Qcov[3] * Bc[3];

  KastaunCtx c;
  c.gam = gam; c.D = D;
  c.q = tau / D;
  c.rsq = Ssq / (D * D);
  c.bsq = Bsq / D;
  c.rbsq = SdotB * SdotB / (D * D * D);
  c.brperp = c.bsq * c.rsq - c.rbsq;
  if (c.brperp < 0.0) c.brperp = 0.0;                      // Cauchy-Schwarz up to rounding
  c.v0sq = c.rsq / (1.0 + c.rsq);

  double mu_hi = 1.0;                                      // 1/h0
  if (!(c.rsq < 1.0)) {
    double fa1 = kastaun_fa(c, 1.0);
    if (fa1 > 0.0) {
      double lo, hi;
      if (!illinois([&](double m) { return kastaun_fa(c, m); }, 0.0, -1.0, 1.0, fa1, lo, hi)) return 2;
      mu_hi = hi;
    }
  }
  double vr, W, er;
  double f0 = kastaun_f(c, 0.0, vr, W, er);
  double f1 = kastaun_f(c, mu_hi, vr, W, er);
  double mu;
  if (!(f0 < 0.0) || !std::isfinite(f1)) return 2;
  if (f1 <= 0.0) mu = mu_hi;                               // root at the upper end (to rounding)
  else {
    double lo, hi;
    if (!illinois([&](double m) { double a_, b_, c_; return kastaun_f(c, m, a_, b_, c_); }, 0.0, f0, mu_hi, f1, lo, hi)) return 2;
    mu = 0.5 * (lo + hi);
  }
  double vsq_raw, eps_raw;
  kastaun_f(c, mu, vsq_raw, W, eps_raw);
  if (!(vsq_raw <= c.v0sq * (1.0 + 1e-12))) return 3;
  double x, rbarsq, qbar;
  kastaun_aux(c, mu, x, rbarsq, qbar);
  double rho = D / W;
  double u = rho * eps_raw;
  double rb = SdotB / (D * std::sqrt(D));                  // r.b
  double ut[3];
  for (int i = 1; i < 4; i++) ut[i - 1] = W * mu * x * (Scon[i] / D + mu * rb * Bc[i] / std::sqrt(D));
  if (!std::isfinite(rho) || !std::isfinite(u) || !std::isfinite(ut[0]) || !std::isfinite(ut[1]) || !std::isfinite(ut[2]))
    return 7;
  if (eps_raw < 0.0) return 5;
  Pout[RHO] = rho; Pout[UU] = u;
  Pout[U1] = ut[0]; Pout[U2] = ut[1]; Pout[U3] = ut[2];
  return 0;
}

// ---------------------------------------------------------------------------------------------
// C8. Floors and ceilings (S18).  Returns the fflag bits.
// p.floor_frame = KHO_FRAME_FLUID: rho, u overwritten in place, velocity and field untouched.
// p.floor_frame = KHO_FRAME_DRIFT ("the most common of which is the drift frame"; SURVEY 8(f)
// NEXT-4; reading S26): the material is added in the frame that moves with the E x B drift, so that with the normal
// observer's velocity v^i = ut^i/gamma split along the field, v = v_perp + v_par B/|B|,
//   * the drift velocity v_perp is unchanged, and
//   * the momentum along the field, S_i B^i/|B| = w gamma^2 v_par (w = rho + Gamma u), is conserved:
//       A = w gamma^2 v_par / w',   v_par' / (1 - v_perp^2 - v_par'^2) = A
//       =>  v_par' = 2 A (1 - v_perp^2) / (1 + sqrt(1 + 4 A^2 (1 - v_perp^2))).
// (b^2 = B^2 (1 - v_perp^2) is then unchanged too, so the magnetisation limits stay consistent.)  B^2 <= 1e-12 w': no
// direction, the velocity is kept.  The Lorentz-factor ceiling acts on the adjusted velocity.
// ---------------------------------------------------------------------------------------------
void drift_frame_velocity(const Geom& G, double gam, double rho_old, double u_old, double rho_new, double u_new, double P[NP]) {
  double Bcov[4] = {0, 0, 0, 0}, qsq = 0.0, Bsq = 0.0, uB = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) {
    qsq += G.gcov[i][j] * P[U1 + i - 1] * P[U1 + j - 1];
    Bcov[i] += G.gcov[i][j] * P[B1 + j - 1];
  }
  for (int i = 1; i < 4; i++) { Bsq += Bcov[i] * P[B1 + i - 1]; uB += Bcov[i] * P[U1 + i - 1]; }
  // no field direction to speak of: B^2 below 1e-12 of the enthalpy (a magnetisation double precision cannot see in T^mu_nu;
  // such fields are often pure round-off, whose direction is noise) keeps the velocity
  if (!(Bsq > 1e-12 * (rho_new + gam * u_new))) return;
  double gamma = std::sqrt(1.0 + qsq), B = std::sqrt(Bsq);
  double vpar = uB / (gamma * B);                          // v^i B_i / |B|
  double vsq = qsq / (gamma * gamma);
  double omp = 1.0 - (vsq - vpar * vpar);                  // 1 - v_perp^2
  if (omp > 1.0) omp = 1.0;
  double vperp[3];
  for (int i = 0; i < 3; i++) vperp[i] = P[U1 + i] / gamma - vpar * P[B1 + i] / B;
  double w_old = rho_old + gam * u_old, w_new = rho_new + gam * u_new;
  double A = w_old * gamma * gamma * vpar / w_new;
  double vpar_new = 2.0 * A * omp / (1.0 + std::sqrt(1.0 + 4.0 * A * A * omp));
  double gamma_new = 1.0 / std::sqrt(omp - vpar_new * vpar_new);
  for (int i = 0; i < 3; i++) P[U1 + i] = gamma_new * (vperp[i] + vpar_new * P[B1 + i] / B);
}

int floors(const kho_params& p, const Geom& G, double r, double P[NP]);

// p.floor_frame = KHO_FRAME_NORMAL ("any of a number of different frames"; SURVEY 8(f) NEXT-4;
// reading S27): the floor material (rho_inj, u_inj) = (max(rho_fl - rho, 0), max(u_fl - u, 0)) is added AT REST IN THE
// NORMAL OBSERVER'S FRAME, i.e. as conserved variables: with u^mu = n^mu the added gas has T^t_i = 0 and
//   U_add = sqrt(-g) ( rho_inj/alpha,  -(rho_inj + u_inj) + rho_inj/alpha,  0, 0, 0,  0, 0, 0 ),
// so the momentum density is untouched; the primitives follow from inverting U(P) + U_add (guess: the fluid-frame
// result), and the fluid-frame limits and ceilings then act once more on them.  If that inversion fails the fluid-frame
// result is kept (fflag bit 64).
int floors_normal_frame(const kho_params& p, const Geom& G, double r, double P[NP]) {
  kho_params pf = p;
  pf.floor_frame = KHO_FRAME_FLUID;
  double P0[NP];
  for (int v = 0; v < NP; v++) P0[v] = P[v];
  // the limits, as in the fluid frame
  double s = (p.coords == KHO_MINKOWSKI) ? 1.0 : 1.0 / (r * r) / (1.0 + r / p.r_char);
  FourVec D;
  four_vectors(G.gcov, G.gcon, P0, D);
  double rho_g = p.rho_min * s, rho_b = D.bsq / p.bsq_over_rho_max;
  double u_g = p.u_min * std::pow(s, p.gamma), u_b = D.bsq / p.bsq_over_u_max;
  double rho_fl = rho_b > rho_g ? rho_b : rho_g, u_fl = u_b > u_g ? u_b : u_g;
  double rho_inj = rho_fl > P0[RHO] ? rho_fl - P0[RHO] : 0.0;
  double u_inj = u_fl > P0[UU] ? u_fl - P0[UU] : 0.0;
  int flag = floors(pf, G, r, P);                       // provisional: the fluid-frame result
  if (!(rho_inj > 0.0) && !(u_inj > 0.0)) return flag;
  double U[NP];
  prim_to_flux(G, P0, D, p.gamma, 0, U);
  U[RHO] += G.gdet * (rho_inj / G.alpha);
  U[UU] += G.gdet * (-(rho_inj + u_inj) + rho_inj / G.alpha);
  double Pn[NP];
  int pfl = (p.inverter == KHO_INV_KASTAUN) ? u2p_kastaun(G, U, P, p.gamma, Pn) : u2p(G, U, P, p.gamma, Pn);
  if (pfl != 0) return flag | 64;
  int flag2 = floors(pf, G, r, Pn);
  for (int v = 0; v < NP; v++) P[v] = Pn[v];
  return (flag & 15) | flag2;
}

int floors(const kho_params& p, const Geom& G, double r, double P[NP]) {
  if (p.floor_frame == KHO_FRAME_NORMAL) return floors_normal_frame(p, G, r, P);
  int flag = 0;
  double s = (p.coords == KHO_MINKOWSKI) ? 1.0 : 1.0 / (r * r) / (1.0 + r / p.r_char);
  FourVec D;
  four_vectors(G.gcov, G.gcon, P, D);
  double rho_g = p.rho_min * s, rho_b = D.bsq / p.bsq_over_rho_max;
  double u_g = p.u_min * std::pow(s, p.gamma), u_b = D.bsq / p.bsq_over_u_max;
  double rho_fl = rho_b > rho_g ? rho_b : rho_g;
  double u_fl = u_b > u_g ? u_b : u_g;
  const double rho_old = P[RHO], u_old = P[UU];
  if (P[RHO] < rho_fl) { P[RHO] = rho_fl; flag |= (rho_b > rho_g) ? 2 : 1; }
  if (P[UU] < u_fl) { P[UU] = u_fl; flag |= (u_b > u_g) ? 8 : 4; }
  if (P[UU] > p.u_over_rho_max * P[RHO]) { P[UU] = p.u_over_rho_max * P[RHO]; flag |= 16; }
  if (p.floor_frame == KHO_FRAME_DRIFT && flag != 0) drift_frame_velocity(G, p.gamma, rho_old, u_old, P[RHO], P[UU], P);
  double qsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) qsq += G.gcov[i][j] * P[U1 + i - 1] * P[U1 + j - 1];
  double gamma = std::sqrt(1.0 + qsq);
  if (gamma > p.gamma_max) {
    double f = std::sqrt((p.gamma_max * p.gamma_max - 1.0) / (gamma * gamma - 1.0));
    P[U1] *= f; P[U2] *= f; P[U3] *= f;
    flag |= 32;
  }
  return flag;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// Grid object
// ---------------------------------------------------------------------------------------------
struct kho_grid {
  kho_params p;
  int n[3], nt[3];
  long ntot;          // zones with ghosts
  long n2d;           // (n2+6)(n1+6)
  double dx[3];
  std::vector<Geom> G[4];
  std::vector<double> conn;      // [n2d][64]
  std::vector<double> sfloor_r;  // radius per (j,i)
  std::vector<double> P, Ps, Pf; // [8][ntot]
  std::vector<double> F[3];      // [8][ntot]
  std::vector<double> ctop[3];   // [ntot]
  std::vector<double> emf[3];    // [ntot]
  std::vector<int> pflag, fflag; // [ntot]
  std::vector<double> Bf[3], Bfs[3], Bff[3];   // face-centred CT (S28): sqrt(-g) B^d on the lower d-face of each zone, [ntot]; n / * / n+1
  long idx(int i, int j, int k) const { return ((long)(k + NG) * nt[1] + (j + NG)) * nt[0] + (i + NG); }
  long idx2(int i, int j) const { return (long)(j + NG) * nt[0] + (i + NG); }
  double xc(int d, int i) const { return p.xmin[d] + (i + 0.5) * dx[d]; }
  double xf(int d, int i) const { return p.xmin[d] + i * dx[d]; }
};

namespace {

bool polar_face(const kho_grid& g, int j) {
  return (j == 0 && g.p.bc[2] == KHO_BC_POLAR) || (j == g.n[1] && g.p.bc[3] == KHO_BC_POLAR);
}

// C10. Ghost fill (S20): x1, then x2, then x3, each pass spanning the full extent of the others.
void fill_dir(const kho_grid& g, double* A, int d, bool is_prim_array, int var) {
  int lo[3] = {-NG, -NG, -NG}, hi[3] = {g.n[0] + NG, g.n[1] + NG, g.n[2] + NG};
  int N = g.n[d];
  for (int side = 0; side < 2; side++) {
    int bc = g.p.bc[2 * d + side];
    if (bc == KHO_BC_FIXED) continue;
    for (int m = 0; m < NG; m++) {
      int gi = side == 0 ? -1 - m : N + m;     // ghost index along d
      int si;                                  // source index along d
      double sign = 1.0;
      if (bc == KHO_BC_PERIODIC) { si = ((gi % N) + N) % N; }
      else if (bc == KHO_BC_OUTFLOW) { si = side == 0 ? 0 : N - 1; }
      else { /* polar reflect */
        si = side == 0 ? m : N - 1 - m;
        if (is_prim_array && (var == U2 || var == B2)) sign = -1.0;
      }
      int a[3], b[3];
      for (a[2] = (d == 2 ? gi : lo[2]); a[2] < (d == 2 ? gi + 1 : hi[2]); a[2]++)
        for (a[1] = (d == 1 ? gi : lo[1]); a[1] < (d == 1 ? gi + 1 : hi[1]); a[1]++)
          for (a[0] = (d == 0 ? gi : lo[0]); a[0] < (d == 0 ? gi + 1 : hi[0]); a[0]++) {
            b[0] = a[0]; b[1] = a[1]; b[2] = a[2]; b[d] = si;
            double val = sign * A[g.idx(b[0], b[1], b[2])];
            // S20b: outflow ghosts keep sqrt(-g) B^i (HARM-family practice), not B^i itself
            if (bc == KHO_BC_OUTFLOW && is_prim_array && var >= B1)
              val *= g.G[0][g.idx2(b[0], b[1])].gdet / g.G[0][g.idx2(a[0], a[1])].gdet;
            A[g.idx(a[0], a[1], a[2])] = val;
          }
    }
  }
}
void fill_ghosts_prims(const kho_grid& g, double* P) {
  for (int d = 0; d < 3; d++) for (int v = 0; v < NP; v++) fill_dir(g, P + v * g.ntot, d, true, v);
}
void fill_ghosts_flag(const kho_grid& g, int* flag) {
  std::vector<double> tmp(g.ntot);
  for (long n = 0; n < g.ntot; n++) tmp[n] = flag[n];
  for (int d = 0; d < 3; d++) fill_dir(g, tmp.data(), d, false, 0);
  for (long n = 0; n < g.ntot; n++) flag[n] = (int)tmp[n];
}

void get_prim(const kho_grid& g, const double* P, long n, double out[NP]) {
  for (int v = 0; v < NP; v++) out[v] = P[v * g.ntot + n];
}

// C3 + C4: fluxes of direction d (0,1,2) on faces i_d in [0,N_d], transverse in [-1,N_t].
void compute_flux(kho_grid& g, const double* Ps, int d) {
  int lo[3], hi[3];
  for (int e = 0; e < 3; e++) { lo[e] = (e == d) ? 0 : -1; hi[e] = g.n[e] + 1; }   // exclusive hi
  long stride = (d == 0) ? 1 : (d == 1 ? g.nt[0] : (long)g.nt[0] * g.nt[1]);
  double* F = g.F[d].data();
  double* ct = g.ctop[d].data();
#ifdef _OPENMP
#pragma omp parallel for collapse(2) schedule(static)
#endif
  for (int k = lo[2]; k < hi[2]; k++)
    for (int j = lo[1]; j < hi[1]; j++)
      for (int i = lo[0]; i < hi[0]; i++) {
        long n = g.idx(i, j, k);
        const Geom& G = g.G[1 + d][g.idx2(i, j)];
        double Fl[NP], c = 0.0;
        if (d == 1 && polar_face(g, j)) {        // S7 / S10: nothing crosses the axis
          for (int v = 0; v < NP; v++) Fl[v] = 0.0;
        } else {
          double PL[NP], PR[NP], q[5], l, r;
          for (int v = 0; v < NP; v++) {
            const double* A = Ps + v * g.ntot;
            for (int s = 0; s < 5; s++) q[s] = A[n + (s - 3) * stride];   // zone i_d - 1
            recon(g.p.recon, q, l, r);
            PL[v] = r;
            for (int s = 0; s < 5; s++) q[s] = A[n + (s - 2) * stride];   // zone i_d
            recon(g.p.recon, q, l, r);
            PR[v] = l;
          }
          llf(G, PL, PR, g.p.gamma, d + 1, Fl, c);
        }
        for (int v = 0; v < NP; v++) F[v * g.ntot + n] = Fl[v];
        ct[n] = c;
      }
}

// C5. Flux-CT (S15a).  Works on raw face-flux arrays so the invariant can be tested on arbitrary fluxes.
void flux_ct(const kho_grid& g, double* F1, double* F2, double* F3, double* e1, double* e2, double* e3, bool have_emf = false) {
  const long nt = g.ntot;
  const int N1 = g.n[0], N2 = g.n[1], N3 = g.n[2];
  auto X = [&](int i, int j, int k) { return g.idx(i, j, k); };
  if (!have_emf)
  for (int k = 0; k <= N3; k++) for (int j = 0; j <= N2; j++) for (int i = 0; i <= N1; i++) {
    long n = X(i, j, k);
    if (k < N3)
      e3[n] = 0.25 * (F1[B2 * nt + n] + F1[B2 * nt + X(i, j - 1, k)] - F2[B1 * nt + n] - F2[B1 * nt + X(i - 1, j, k)]);
    if (j < N2)
      e2[n] = -0.25 * (F1[B3 * nt + n] + F1[B3 * nt + X(i, j, k - 1)] - F3[B1 * nt + n] - F3[B1 * nt + X(i - 1, j, k)]);
    if (i < N1)
      e1[n] = 0.25 * (F2[B3 * nt + n] + F2[B3 * nt + X(i, j, k - 1)] - F3[B2 * nt + n] - F3[B2 * nt + X(i, j - 1, k)]);
    if (polar_face(g, j)) { e1[n] = 0.0; e3[n] = 0.0; }    // S10
  }
  for (int k = 0; k <= N3; k++) for (int j = 0; j <= N2; j++) for (int i = 0; i <= N1; i++) {
    long n = X(i, j, k);
    if (j < N2 && k < N3) {
      F1[B1 * nt + n] = 0.0;
      F1[B2 * nt + n] = 0.5 * (e3[n] + e3[X(i, j + 1, k)]);
      F1[B3 * nt + n] = -0.5 * (e2[n] + e2[X(i, j, k + 1)]);
    }
    if (i < N1 && k < N3) {
      F2[B2 * nt + n] = 0.0;
      F2[B1 * nt + n] = -0.5 * (e3[n] + e3[X(i + 1, j, k)]);
      F2[B3 * nt + n] = 0.5 * (e1[n] + e1[X(i, j, k + 1)]);
    }
    if (i < N1 && j < N2) {
      F3[B3 * nt + n] = 0.0;
      F3[B1 * nt + n] = 0.5 * (e2[n] + e2[X(i + 1, j, k)]);
      F3[B2 * nt + n] = -0.5 * (e1[n] + e1[X(i, j + 1, k)]);
    }
  }
}

// Upwinded edge EMFs (EMFs "along zone edges with and without upwinding"; reading
// S29): the contact-upwind construction of Gardiner & Stone (2005), restated for the three components.  For component c
// with (a, b) cyclic, eps_c = F^a[B^b] = -F^b[B^a]; per zone n (lower faces / lower edge):
//   efa(n) = F^a[B^b](n),  efb(n) = -F^b[B^a](n),  ec(n) = sqrt(-g) (B^b u^a - B^a u^b)/u^t at the zone centre,
//   gradients across half zones:  da_m(n) = 2 (efa(n) - ec(n - s_a)),  da_p(n) = 2 (ec(n) - efa(n))   (and b likewise),
//   each upwinded in the OTHER direction by the sign of the mass flux through the face between the two candidates,
//   eps_edge = 1/4 (efa(n) + efa(n - s_b) + efb(n) + efb(n - s_a))
//            + 1/8 [ up_a(db_m; M_a(n - s_b)) - up_a(db_p; M_a(n)) ] + 1/8 [ up_b(da_m; M_b(n - s_a)) - up_b(da_p; M_b(n)) ],
//   up_a(d; M) = d(n - s_a) if M > tol Dsum, d(n) if M < -tol Dsum, their mean otherwise, where Dsum is the sum of the
//   conserved densities sqrt(-g) rho u^t of the two zones the face separates and tol = 1e-10: a mass flux that small is
//   "no flow" (by symmetry it is often exactly zero, and then its computed sign is round-off noise).
// For plane-parallel, grid-aligned flow this reduces to the one-dimensional face value (the design condition of that
// paper; pinned in tests/test_oracle_facect.py).  Writes the same emf arrays as flux_ct's first loop.
void emf_upwind(const kho_grid& g, const double* Ps, const double* F1, const double* F2, const double* F3, double* e1, double* e2, double* e3) {
  const long nt = g.ntot;
  const long st[3] = {1, g.nt[0], (long)g.nt[0] * g.nt[1]};
  const double* F[3] = {F1, F2, F3};
  double* E[3] = {e1, e2, e3};
  // zone-centred reference values, zones -1 .. N in every direction
  std::vector<double> ec[3], Dc(nt, 0.0);
  for (int c = 0; c < 3; c++) ec[c].assign(nt, 0.0);
  for (int k = -1; k <= g.n[2]; k++) for (int j = -1; j <= g.n[1]; j++) for (int i = -1; i <= g.n[0]; i++) {
    long n = g.idx(i, j, k);
    const Geom& G = g.G[0][g.idx2(i, j)];
    double P[NP];
    get_prim(g, Ps, n, P);
    FourVec D;
    four_vectors(G.gcov, G.gcon, P, D);
    for (int c = 0; c < 3; c++) {
      int a = (c + 1) % 3, b = (c + 2) % 3;
      ec[c][n] = G.gdet * (P[B1 + b] * D.ucon[1 + a] - P[B1 + a] * D.ucon[1 + b]) / D.ucon[0];
    }
    Dc[n] = G.gdet * P[RHO] * D.ucon[0];
  }
  for (int c = 0; c < 3; c++) {
    const int a = (c + 1) % 3, b = (c + 2) % 3;
    const long sa = st[a], sb = st[b];
    const double* Fa = F[a]; const double* Fb = F[b];
    auto efa = [&](long n) { return Fa[(B1 + b) * nt + n]; };
    auto efb = [&](long n) { return -Fb[(B1 + a) * nt + n]; };
    auto da_m = [&](long n) { return 2.0 * (efa(n) - ec[c][n - sa]); };
    auto da_p = [&](long n) { return 2.0 * (ec[c][n] - efa(n)); };
    auto db_m = [&](long n) { return 2.0 * (efb(n) - ec[c][n - sb]); };
    auto db_p = [&](long n) { return 2.0 * (ec[c][n] - efb(n)); };
    auto up = [&](double lo, double hi, double M, double Dsum) {
      const double t = 1e-10 * Dsum;
      return M > t ? lo : (M < -t ? hi : 0.5 * (lo + hi));
    };
    int hi[3] = {g.n[0] + 1, g.n[1] + 1, g.n[2] + 1};
    hi[c] = g.n[c];                                        // edges along c: zones 0 .. N_c - 1 in that direction
    for (int k = 0; k < hi[2]; k++) for (int j = 0; j < hi[1]; j++) for (int i = 0; i < hi[0]; i++) {
      long n = g.idx(i, j, k);
      double Ma0 = Fa[RHO * nt + n], Ma1 = Fa[RHO * nt + n - sb], Mb0 = Fb[RHO * nt + n], Mb1 = Fb[RHO * nt + n - sa];
      double v = 0.25 * (efa(n) + efa(n - sb) + efb(n) + efb(n - sa))
               + 0.125 * (up(db_m(n - sa), db_m(n), Ma1, Dc[n - sb - sa] + Dc[n - sb]) - up(db_p(n - sa), db_p(n), Ma0, Dc[n - sa] + Dc[n]))
               + 0.125 * (up(da_m(n - sb), da_m(n), Mb1, Dc[n - sa - sb] + Dc[n - sa]) - up(da_p(n - sb), da_p(n), Mb0, Dc[n - sb] + Dc[n]));
      if (c != 1 && polar_face(g, j)) v = 0.0;             // S10
      E[c][n] = v;
    }
  }
}

// C9. Fix-up of failed inversions (S19) followed by floors.
// Edge EMFs of Gardiner & Stone's un-upwinded scheme (their "E-circle"; "a number of schemes for
// determining the EMFs along zone edges with and without upwinding"; S30): the four-point face average corrected by
// the zone-centred reference values,
//   eps_c(edge) = 1/2 (sum of the four face values) - 1/4 (sum of the four zone-centred values around the edge),
// with the face values eps_c = F^a[B^b] = -F^b[B^a] and the centred ones sqrt(-g) (B^b v^a - B^a v^b), v^i = u^i / u^t, (c, a, b)
// cyclic.  It is what the upwinded scheme's general form gives when both candidate gradients are averaged at every face; it
// has the correct limit for plane-parallel, grid-aligned flow (the edge sees the one-dimensional face value), which the plain
// arithmetic average lacks, and no dependence on the direction of the flow.  Written out from this closed form, not through
// emf_upwind().
void emf_centred(const kho_grid& g, const double* Ps, const double* F1, const double* F2, const double* F3, double* e1, double* e2, double* e3) {
  const long nt = g.ntot;
  const long st[3] = {1, g.nt[0], (long)g.nt[0] * g.nt[1]};
  const double* F[3] = {F1, F2, F3};
  double* E[3] = {e1, e2, e3};
  for (int c = 0; c < 3; c++) {
    const int a = (c + 1) % 3, b = (c + 2) % 3;
    const long sa = st[a], sb = st[b];
    std::vector<double> ec(nt, 0.0);
    for (int k = -1; k <= g.n[2]; k++) for (int j = -1; j <= g.n[1]; j++) for (int i = -1; i <= g.n[0]; i++) {
      long n = g.idx(i, j, k);
      const Geom& G = g.G[0][g.idx2(i, j)];
      double P[NP];
      get_prim(g, Ps, n, P);
      FourVec D;
      four_vectors(G.gcov, G.gcon, P, D);
      ec[n] = G.gdet * (P[B1 + b] * D.ucon[1 + a] - P[B1 + a] * D.ucon[1 + b]) / D.ucon[0];
    }
    int hi[3] = {g.n[0] + 1, g.n[1] + 1, g.n[2] + 1};
    hi[c] = g.n[c];
    for (int k = 0; k < hi[2]; k++) for (int j = 0; j < hi[1]; j++) for (int i = 0; i < hi[0]; i++) {
      long n = g.idx(i, j, k);
      double faces = F[a][(B1 + b) * nt + n] + F[a][(B1 + b) * nt + n - sb] - F[b][(B1 + a) * nt + n] - F[b][(B1 + a) * nt + n - sa];
      double centres = ec[n] + ec[n - sa] + ec[n - sb] + ec[n - sa - sb];
      double v = 0.5 * faces - 0.25 * centres;
      if (c != 1 && polar_face(g, j)) v = 0.0;             // S10
      E[c][n] = v;
    }
  }
}

void fixup(kho_grid& g, double* Pf) {
  std::vector<double> snap(Pf, Pf + 5 * g.ntot);   // hydro primitives, pre-fix-up snapshot
  for (int k = 0; k < g.n[2]; k++) for (int j = 0; j < g.n[1]; j++) for (int i = 0; i < g.n[0]; i++) {
    long n = g.idx(i, j, k);
    if (g.pflag[n] == 0) continue;
    double sum[5] = {0, 0, 0, 0, 0}, wsum = 0.0, sum_all[5] = {0, 0, 0, 0, 0}, wsum_all = 0.0;
    for (int dk = -1; dk <= 1; dk++) for (int dj = -1; dj <= 1; dj++) for (int di = -1; di <= 1; di++) {
      if (di == 0 && dj == 0 && dk == 0) continue;
      long m = g.idx(i + di, j + dj, k + dk);
      double w = 1.0 / (std::abs(di) + std::abs(dj) + std::abs(dk) + 1);
      for (int v = 0; v < 5; v++) sum_all[v] += w * snap[v * g.ntot + m];
      wsum_all += w;
      if (g.pflag[m] == 0) {
        for (int v = 0; v < 5; v++) sum[v] += w * snap[v * g.ntot + m];
        wsum += w;
      }
    }
    for (int v = 0; v < 5; v++) Pf[v * g.ntot + n] = (wsum > 0.0) ? sum[v] / wsum : sum_all[v] / wsum_all;
    double Pz[NP];
    get_prim(g, Pf, n, Pz);
    long n2 = g.idx2(i, j);
    g.fflag[n] |= floors(g.p, g.G[0][n2], g.sfloor_r[n2], Pz);
    for (int v = 0; v < NP; v++) Pf[v * g.ntot + n] = Pz[v];
  }
}

// One sub-step (S22): fluxes from Ps, update of U(Pi) by Dt, U->P with guess Pi, floors, fill, fix-up, fill.
// C6 + C7 + C8 on the interior zones: U_f = U(P_i) + Dt [-div F + S(P_s)], inversion with guess P_i, floors.
void update_zones(kho_grid& g, const double* Pi, const double* Ps, double* Pf, double Dt, const std::vector<double>* Bface = nullptr) {
  const long nt = g.ntot;
  const long st[3] = {1, g.nt[0], (long)g.nt[0] * g.nt[1]};
  std::fill(g.pflag.begin(), g.pflag.end(), 0);
  std::fill(g.fflag.begin(), g.fflag.end(), 0);
#ifdef _OPENMP
#pragma omp parallel for collapse(2) schedule(static)
#endif
  for (int k = 0; k < g.n[2]; k++) for (int j = 0; j < g.n[1]; j++) for (int i = 0; i < g.n[0]; i++) {
    long n = g.idx(i, j, k), n2 = g.idx2(i, j);
    const Geom& G = g.G[0][n2];
    double pi[NP], ps[NP], Ui[NP], S[NP], Uf[NP], pf[NP];
    get_prim(g, Pi, n, pi);
    get_prim(g, Ps, n, ps);
    FourVec D;
    four_vectors(G.gcov, G.gcon, pi, D);
    prim_to_flux(G, pi, D, g.p.gamma, 0, Ui);
    source(G, &g.conn[n2 * 64], ps, g.p.gamma, S);
    for (int v = 0; v < NP; v++) {
      double div = 0.0;
      for (int d = 0; d < 3; d++) div += (g.F[d][v * nt + n + st[d]] - g.F[d][v * nt + n]) / g.dx[d];
      Uf[v] = Ui[v] + Dt * (-div + S[v]);
    }
    // face-centred CT (S28): the zone's conserved field is the mean of its two face values
    if (Bface) for (int d = 0; d < 3; d++) Uf[B1 + d] = 0.5 * (Bface[d][n] + Bface[d][n + st[d]]);
    int pf_flag = (g.p.inverter == KHO_INV_KASTAUN) ? u2p_kastaun(G, Uf, pi, g.p.gamma, pf) : u2p(G, Uf, pi, g.p.gamma, pf);
    int ff = 0;
    if (pf_flag == 0) ff = floors(g.p, G, g.sfloor_r[n2], pf);
    g.pflag[n] = pf_flag;
    g.fflag[n] = ff;
    for (int v = 0; v < NP; v++) Pf[v * nt + n] = pf[v];
  }
}

// First-order flux correction (reading S25 in DESIGN.md): the faces of
// every zone of `mask` (ghost images included) get the Local Lax-Friedrichs flux of the donor-cell states, i.e.
// P_L = P_s(zone below the face), P_R = P_s(zone above it).  Same face ranges as compute_flux; axis faces stay zero.
void fofc_reflux(kho_grid& g, const double* Ps, const std::vector<int>& mask) {
  for (int d = 0; d < 3; d++) {
    int lo[3], hi[3];
    for (int e = 0; e < 3; e++) { lo[e] = (e == d) ? 0 : -1; hi[e] = g.n[e] + 1; }
    long stride = (d == 0) ? 1 : (d == 1 ? g.nt[0] : (long)g.nt[0] * g.nt[1]);
    for (int k = lo[2]; k < hi[2]; k++) for (int j = lo[1]; j < hi[1]; j++) for (int i = lo[0]; i < hi[0]; i++) {
      long n = g.idx(i, j, k);
      if (!(mask[n - stride] || mask[n])) continue;
      if (d == 1 && polar_face(g, j)) continue;
      double PL[NP], PR[NP], Fl[NP], c;
      get_prim(g, Ps, n - stride, PL);
      get_prim(g, Ps, n, PR);
      llf(g.G[1 + d][g.idx2(i, j)], PL, PR, g.p.gamma, d + 1, Fl, c);
      for (int v = 0; v < NP; v++) g.F[d][v * g.ntot + n] = Fl[v];
      g.ctop[d][n] = c;
    }
  }
}

// Face-centred constrained transport ("the face-centered constrained transport scheme outlined in [50],
// including a number of schemes for determining the EMFs along zone edges"; reading S28).  The
// magnetic field lives on the faces as Phi^d = sqrt(-g) B^d; it is advanced by the circulation of the edge EMFs around
// each face, so the face-centred divergence sum_d (Phi^d(+1) - Phi^d)/dx_d is constant to round-off:
//   Phi^1_f = Phi^1_i + Dt [ (E3(i,j+1,k) - E3(i,j,k))/dx2 - (E2(i,j,k+1) - E2(i,j,k))/dx3 ]   and cyclic (E = this file's
// emf arrays, lower edge of the zone).  EMF option built: the arithmetic four-point average of the face fluxes (the one
// Flux-CT uses, C5), for which the zone-centred mean of the face field evolves exactly as under Flux-CT (Toth 2000).
// Zone-centred B (primitive) = mean of the zone's two face values / sqrt(-g); ghosts by the ordinary fill.
void face_ct_update(const kho_grid& g, const std::vector<double>* Bi, std::vector<double>* Bf, double Dt) {
  const long s1 = 1, s2 = g.nt[0], s3 = (long)g.nt[0] * g.nt[1];
  const double* e1 = g.emf[0].data(); const double* e2 = g.emf[1].data(); const double* e3 = g.emf[2].data();
  for (int k = 0; k <= g.n[2]; k++) for (int j = 0; j <= g.n[1]; j++) for (int i = 0; i <= g.n[0]; i++) {
    long n = g.idx(i, j, k);
    if (j < g.n[1] && k < g.n[2]) Bf[0][n] = Bi[0][n] + Dt * ((e3[n + s2] - e3[n]) / g.dx[1] - (e2[n + s3] - e2[n]) / g.dx[2]);
    if (i < g.n[0] && k < g.n[2]) Bf[1][n] = Bi[1][n] + Dt * ((e1[n + s3] - e1[n]) / g.dx[2] - (e3[n + s1] - e3[n]) / g.dx[0]);
    if (i < g.n[0] && j < g.n[1]) Bf[2][n] = Bi[2][n] + Dt * ((e2[n + s1] - e2[n]) / g.dx[0] - (e1[n + s2] - e1[n]) / g.dx[1]);
  }
}

void substep(kho_grid& g, const double* Pi, const double* Ps, double* Pf, double Dt, const std::vector<double>* Bfi = nullptr,
             std::vector<double>* Bff = nullptr) {
  for (int d = 0; d < 3; d++) compute_flux(g, Ps, d);
  const long nt = g.ntot;
  if (g.p.fofc) {
    // speculative update with the high-order fluxes: which zones would fail the inversion or hit a floor?
    std::vector<double> raw[3] = {g.F[0], g.F[1], g.F[2]};                      // flux_ct rewrites the B components in place
    if (g.p.emf == KHO_EMF_UPWIND) emf_upwind(g, Ps, g.F[0].data(), g.F[1].data(), g.F[2].data(), g.emf[0].data(), g.emf[1].data(), g.emf[2].data());
    if (g.p.emf == KHO_EMF_CENTRED) emf_centred(g, Ps, g.F[0].data(), g.F[1].data(), g.F[2].data(), g.emf[0].data(), g.emf[1].data(), g.emf[2].data());
    flux_ct(g, g.F[0].data(), g.F[1].data(), g.F[2].data(), g.emf[0].data(), g.emf[1].data(), g.emf[2].data(), g.p.emf != KHO_EMF_ARITHMETIC);
    if (Pf != Pi) std::memcpy(Pf, Pi, sizeof(double) * NP * nt);
    update_zones(g, Pi, Ps, Pf, Dt);
    std::vector<int> mask(nt, 0);
    for (long n = 0; n < nt; n++) mask[n] = (g.pflag[n] != 0 || g.fflag[n] != 0) ? 1 : 0;   // ghosts are 0 here
    fill_ghosts_flag(g, mask.data());                                              // ghost images of troubled zones
    for (int d = 0; d < 3; d++) g.F[d] = raw[d];
    fofc_reflux(g, Ps, mask);
  }
  if (g.p.emf == KHO_EMF_UPWIND) emf_upwind(g, Ps, g.F[0].data(), g.F[1].data(), g.F[2].data(), g.emf[0].data(), g.emf[1].data(), g.emf[2].data());
  if (g.p.emf == KHO_EMF_CENTRED) emf_centred(g, Ps, g.F[0].data(), g.F[1].data(), g.F[2].data(), g.emf[0].data(), g.emf[1].data(), g.emf[2].data());
  flux_ct(g, g.F[0].data(), g.F[1].data(), g.F[2].data(), g.emf[0].data(), g.emf[1].data(), g.emf[2].data(), g.p.emf != KHO_EMF_ARITHMETIC);
  if (Pf != Pi) std::memcpy(Pf, Pi, sizeof(double) * NP * nt);   // ghosts of Pf start from Pi (matters for FIXED)
  if (Bfi) face_ct_update(g, Bfi, Bff, Dt);
  update_zones(g, Pi, Ps, Pf, Dt, Bfi ? Bff : nullptr);
  fill_ghosts_prims(g, Pf);
  fill_ghosts_flag(g, g.pflag.data());
  fixup(g, Pf);
  fill_ghosts_prims(g, Pf);
}

double dt_from_ctop(const kho_grid& g) {
  const long st[3] = {1, g.nt[0], (long)g.nt[0] * g.nt[1]};
  double dtmin = std::numeric_limits<double>::infinity();
  for (int k = 0; k < g.n[2]; k++) for (int j = 0; j < g.n[1]; j++) for (int i = 0; i < g.n[0]; i++) {
    long n = g.idx(i, j, k);
    double s = 0.0;
    for (int d = 0; d < 3; d++) {
      if (g.n[d] <= 1) continue;
      double c = std::fmax(g.ctop[d][n], g.ctop[d][n + st[d]]);
      s += c / g.dx[d];
    }
    double dtz = 1.0 / s;
    if (dtz < dtmin) dtmin = dtz;
  }
  return dtmin;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------------
extern "C" {

const char* kho_strerror(int code) {
  switch (code) {
    case KHO_OK: return "ok";
    case KHO_EINVAL: return "invalid argument";
    case KHO_ENOMEM: return "out of memory";
    default: return "unknown error";
  }
}

int kho_grid_create(const kho_params* p, kho_grid** out) {
  if (!p || !out) return KHO_EINVAL;
  if (p->n1 < 1 || p->n2 < 1 || p->n3 < 1) return KHO_EINVAL;
  if (p->coords < 0 || p->coords > 2 || p->recon < 0 || p->recon > 1) return KHO_EINVAL;
  for (int d = 0; d < 3; d++) {
    if (!(p->xmax[d] > p->xmin[d])) return KHO_EINVAL;
    int N = d == 0 ? p->n1 : (d == 1 ? p->n2 : p->n3);
    for (int s = 0; s < 2; s++) {
      int bc = p->bc[2 * d + s];
      if (bc < 0 || bc > 3) return KHO_EINVAL;
      if (bc == KHO_BC_POLAR && (d != 1 || N < NG)) return KHO_EINVAL;
    }
    if ((p->bc[2 * d] == KHO_BC_PERIODIC) != (p->bc[2 * d + 1] == KHO_BC_PERIODIC)) return KHO_EINVAL;
  }
  kho_grid* g = new (std::nothrow) kho_grid;
  if (!g) return KHO_ENOMEM;
  try {
    g->p = *p;
    g->n[0] = p->n1; g->n[1] = p->n2; g->n[2] = p->n3;
    for (int d = 0; d < 3; d++) { g->nt[d] = g->n[d] + 2 * NG; g->dx[d] = (p->xmax[d] - p->xmin[d]) / g->n[d]; }
    g->ntot = (long)g->nt[0] * g->nt[1] * g->nt[2];
    g->n2d = (long)g->nt[0] * g->nt[1];
    for (int l = 0; l < 4; l++) g->G[l].resize(g->n2d);
    g->conn.assign(g->n2d * 64, 0.0);
    g->sfloor_r.assign(g->n2d, 1.0);
    for (int j = -NG; j < g->n[1] + NG; j++) for (int i = -NG; i < g->n[0] + NG; i++) {
      long n2 = g->idx2(i, j);
      // S3: the metric is evaluated AT the zone centre / face centre, never averaged
      geom_at(*p, g->xc(0, i), g->xc(1, j), g->G[KHO_LOC_CENT][n2]);
      geom_at(*p, g->xf(0, i), g->xc(1, j), g->G[KHO_LOC_FACE1][n2]);
      if (polar_face(*g, j)) geom_zero(g->G[KHO_LOC_FACE2][n2]);          // S7
      else geom_at(*p, g->xc(0, i), g->xf(1, j), g->G[KHO_LOC_FACE2][n2]);
      geom_at(*p, g->xc(0, i), g->xc(1, j), g->G[KHO_LOC_FACE3][n2]);
      conn_exact(*p, g->xc(0, i), g->xc(1, j), &g->conn[n2 * 64]);
      g->sfloor_r[n2] = radius_at(*p, g->xc(0, i));
    }
    g->P.assign(NP * g->ntot, 0.0); g->Ps.assign(NP * g->ntot, 0.0); g->Pf.assign(NP * g->ntot, 0.0);
    for (int d = 0; d < 3; d++) { g->F[d].assign(NP * g->ntot, 0.0); g->ctop[d].assign(g->ntot, 0.0); g->emf[d].assign(g->ntot, 0.0); }
    g->pflag.assign(g->ntot, 0); g->fflag.assign(g->ntot, 0);
    if (g->p.transport == KHO_B_FACE_CT) for (int d = 0; d < 3; d++) { g->Bf[d].assign(g->ntot, 0.0); g->Bfs[d].assign(g->ntot, 0.0); g->Bff[d].assign(g->ntot, 0.0); }
  } catch (...) { delete g; return KHO_ENOMEM; }
  *out = g;
  return KHO_OK;
}

int kho_grid_destroy(kho_grid* g) { delete g; return KHO_OK; }

int kho_set_prims(kho_grid* g, const double* p, int with_ghosts) {
  if (!g || !p) return KHO_EINVAL;
  if (with_ghosts) {
    std::memcpy(g->P.data(), p, sizeof(double) * NP * g->ntot);
  } else {
    long nin = (long)g->n[0] * g->n[1] * g->n[2];
    for (int v = 0; v < NP; v++) for (int k = 0; k < g->n[2]; k++) for (int j = 0; j < g->n[1]; j++) for (int i = 0; i < g->n[0]; i++)
      g->P[v * g->ntot + g->idx(i, j, k)] = p[v * nin + ((long)k * g->n[1] + j) * g->n[0] + i];
  }
  fill_ghosts_prims(*g, g->P.data());
  return KHO_OK;
}

int kho_get_prims(kho_grid* g, double* p, int with_ghosts) {
  if (!g || !p) return KHO_EINVAL;
  if (with_ghosts) { std::memcpy(p, g->P.data(), sizeof(double) * NP * g->ntot); return KHO_OK; }
  long nin = (long)g->n[0] * g->n[1] * g->n[2];
  for (int v = 0; v < NP; v++) for (int k = 0; k < g->n[2]; k++) for (int j = 0; j < g->n[1]; j++) for (int i = 0; i < g->n[0]; i++)
    p[v * nin + ((long)k * g->n[1] + j) * g->n[0] + i] = g->P[v * g->ntot + g->idx(i, j, k)];
  return KHO_OK;
}

int kho_get_cons(kho_grid* g, double* u) {
  if (!g || !u) return KHO_EINVAL;
  long nin = (long)g->n[0] * g->n[1] * g->n[2];
  for (int k = 0; k < g->n[2]; k++) for (int j = 0; j < g->n[1]; j++) for (int i = 0; i < g->n[0]; i++) {
    double pz[NP], U[NP];
    get_prim(*g, g->P.data(), g->idx(i, j, k), pz);
    const Geom& G = g->G[0][g->idx2(i, j)];
    FourVec D;
    four_vectors(G.gcov, G.gcon, pz, D);
    prim_to_flux(G, pz, D, g->p.gamma, 0, U);
    for (int v = 0; v < NP; v++) u[v * nin + ((long)k * g->n[1] + j) * g->n[0] + i] = U[v];
  }
  return KHO_OK;
}

int kho_get_flags(kho_grid* g, int* pflag, int* fflag) {
  if (!g) return KHO_EINVAL;
  for (int k = 0; k < g->n[2]; k++) for (int j = 0; j < g->n[1]; j++) for (int i = 0; i < g->n[0]; i++) {
    long m = ((long)k * g->n[1] + j) * g->n[0] + i, n = g->idx(i, j, k);
    if (pflag) pflag[m] = g->pflag[n];
    if (fflag) fflag[m] = g->fflag[n];
  }
  return KHO_OK;
}

// S22: first-step dt from zone-centred signal speeds.
int kho_estimate_dt(kho_grid* g, double* dt) {
  if (!g || !dt) return KHO_EINVAL;
  double dtmin = std::numeric_limits<double>::infinity();
  for (int k = 0; k < g->n[2]; k++) for (int j = 0; j < g->n[1]; j++) for (int i = 0; i < g->n[0]; i++) {
    double pz[NP];
    get_prim(*g, g->P.data(), g->idx(i, j, k), pz);
    const Geom& G = g->G[0][g->idx2(i, j)];
    FourVec D;
    four_vectors(G.gcov, G.gcon, pz, D);
    double s = 0.0;
    for (int d = 0; d < 3; d++) {
      if (g->n[d] <= 1) continue;
      double vmax, vmin;
      vchar(G, pz, D, g->p.gamma, d + 1, vmax, vmin);
      s += std::fmax(std::fabs(vmax), std::fabs(vmin)) / g->dx[d];
    }
    double dtz = 1.0 / s;
    if (dtz < dtmin) dtmin = dtz;
  }
  *dt = g->p.cfl * dtmin;
  return KHO_OK;
}

// C11 (S22): P* = substep(P^n, P^n, dt/2);  P^{n+1} = substep(P^n, P*, dt);  dt_next from the corrector's face speeds.
int kho_step(kho_grid* g, double dt, double* dt_next) {
  if (!g || !(dt > 0.0)) return KHO_EINVAL;
  if (g->p.transport == KHO_B_FACE_CT) {
    substep(*g, g->P.data(), g->P.data(), g->Ps.data(), 0.5 * dt, g->Bf, g->Bfs);
    substep(*g, g->P.data(), g->Ps.data(), g->Pf.data(), dt, g->Bf, g->Bff);
    for (int d = 0; d < 3; d++) g->Bf[d].swap(g->Bff[d]);
  } else {
    substep(*g, g->P.data(), g->P.data(), g->Ps.data(), 0.5 * dt);
    substep(*g, g->P.data(), g->Ps.data(), g->Pf.data(), dt);
  }
  g->P.swap(g->Pf);
  if (dt_next) {
    double d = g->p.cfl * dt_from_ctop(*g);
    double cap = g->p.dt_growth_max * dt;
    *dt_next = d < cap ? d : cap;
  }
  return KHO_OK;
}

// Corner-centred divergence preserved by Flux-CT (C5).
int kho_divB(kho_grid* g, double* max_abs) {
  if (!g || !max_abs) return KHO_EINVAL;
  int lo[3], hi[3];
  for (int d = 0; d < 3; d++) { lo[d] = (g->p.bc[2 * d] == KHO_BC_PERIODIC) ? 0 : 1; hi[d] = g->n[d]; }
  double mx = 0.0;
  const double* P = g->P.data();
  for (int k = lo[2]; k < hi[2]; k++) for (int j = lo[1]; j < hi[1]; j++) for (int i = lo[0]; i < hi[0]; i++) {
    double div = 0.0;
    for (int d = 0; d < 3; d++) {
      double s = 0.0;
      for (int b = 0; b < 2; b++) for (int a = 0; a < 2; a++) {
        int o[3] = {0, 0, 0};
        o[(d + 1) % 3] = -a; o[(d + 2) % 3] = -b;
        int ih = i + o[0], jh = j + o[1], kh = k + o[2];
        int il = ih - (d == 0), jl = jh - (d == 1), kl = kh - (d == 2);
        double hiB = g->G[0][g->idx2(ih, jh)].gdet * P[(B1 + d) * g->ntot + g->idx(ih, jh, kh)];
        double loB = g->G[0][g->idx2(il, jl)].gdet * P[(B1 + d) * g->ntot + g->idx(il, jl, kl)];
        s += hiB - loB;
      }
      div += 0.25 * s / g->dx[d];
    }
    if (std::fabs(div) > mx) mx = std::fabs(div);
  }
  *max_abs = mx;
  return KHO_OK;
}

int kho_get_flux(kho_grid* g, int dir, double* F, double* ctop) {
  if (!g || dir < 1 || dir > 3) return KHO_EINVAL;
  if (F) std::memcpy(F, g->F[dir - 1].data(), sizeof(double) * NP * g->ntot);
  if (ctop) std::memcpy(ctop, g->ctop[dir - 1].data(), sizeof(double) * g->ntot);
  return KHO_OK;
}
int kho_get_emf(kho_grid* g, int dir, double* emf) {
  if (!g || !emf || dir < 1 || dir > 3) return KHO_EINVAL;
  std::memcpy(emf, g->emf[dir - 1].data(), sizeof(double) * g->ntot);
  return KHO_OK;
}

int kho_get_geom(kho_grid* g, int loc, double* gcov16, double* gcon16, double* gdet, double* alpha) {
  if (!g || loc < 0 || loc > 3) return KHO_EINVAL;
  for (long n = 0; n < g->n2d; n++) {
    const Geom& G = g->G[loc][n];
    for (int m = 0; m < 16; m++) {
      if (gcov16) gcov16[n * 16 + m] = G.gcov[m / 4][m % 4];
      if (gcon16) gcon16[n * 16 + m] = G.gcon[m / 4][m % 4];
    }
    if (gdet) gdet[n] = G.gdet;
    if (alpha) alpha[n] = G.alpha;
  }
  return KHO_OK;
}
int kho_get_conn(kho_grid* g, double* conn64) {
  if (!g || !conn64) return KHO_EINVAL;
  std::memcpy(conn64, g->conn.data(), sizeof(double) * 64 * g->n2d);
  return KHO_OK;
}
// test hook: run the C9 fix-up (+ floors) on the current primitives with a caller-supplied flag array (with ghosts)
// test hook: predictor sub-step only; P* becomes the current state
int kho_debug_predictor(kho_grid* g, double dt) {
  if (!g || !(dt > 0.0)) return KHO_EINVAL;
  if (g->p.transport == KHO_B_FACE_CT) {
    substep(*g, g->P.data(), g->P.data(), g->Ps.data(), 0.5 * dt, g->Bf, g->Bfs);
    for (int d = 0; d < 3; d++) g->Bf[d].swap(g->Bfs[d]);
  } else {
    substep(*g, g->P.data(), g->P.data(), g->Ps.data(), 0.5 * dt);
  }
  g->P.swap(g->Ps);
  return KHO_OK;
}
int kho_debug_fixup(kho_grid* g, const int* pflag_with_ghosts) {
  if (!g || !pflag_with_ghosts) return KHO_EINVAL;
  for (long n = 0; n < g->ntot; n++) { g->pflag[n] = pflag_with_ghosts[n]; g->fflag[n] = 0; }
  fixup(*g, g->P.data());
  return KHO_OK;
}
int kho_set_face_B(kho_grid* g, const double* f1, const double* f2, const double* f3) {
  if (!g || !f1 || !f2 || !f3 || g->p.transport != KHO_B_FACE_CT) return KHO_EINVAL;
  const double* f[3] = {f1, f2, f3};
  for (int d = 0; d < 3; d++) g->Bf[d].assign(f[d], f[d] + g->ntot);
  const long st[3] = {1, g->nt[0], (long)g->nt[0] * g->nt[1]};
  for (int k = 0; k < g->n[2]; k++) for (int j = 0; j < g->n[1]; j++) for (int i = 0; i < g->n[0]; i++) {
    long n = g->idx(i, j, k);
    for (int d = 0; d < 3; d++) g->P[(B1 + d) * g->ntot + n] = 0.5 * (g->Bf[d][n] + g->Bf[d][n + st[d]]) / g->G[0][g->idx2(i, j)].gdet;
  }
  fill_ghosts_prims(*g, g->P.data());
  return KHO_OK;
}
int kho_get_face_B(kho_grid* g, double* f1, double* f2, double* f3) {
  if (!g || !f1 || !f2 || !f3 || g->p.transport != KHO_B_FACE_CT) return KHO_EINVAL;
  double* f[3] = {f1, f2, f3};
  for (int d = 0; d < 3; d++) std::memcpy(f[d], g->Bf[d].data(), sizeof(double) * g->ntot);
  return KHO_OK;
}
int kho_divB_face(kho_grid* g, double* max_abs) {
  if (!g || !max_abs || g->p.transport != KHO_B_FACE_CT) return KHO_EINVAL;
  const long st[3] = {1, g->nt[0], (long)g->nt[0] * g->nt[1]};
  double m = 0.0;
  for (int k = 0; k < g->n[2]; k++) for (int j = 0; j < g->n[1]; j++) for (int i = 0; i < g->n[0]; i++) {
    long n = g->idx(i, j, k);
    double div = 0.0;
    for (int d = 0; d < 3; d++) div += (g->Bf[d][n + st[d]] - g->Bf[d][n]) / g->dx[d];
    if (std::fabs(div) > m) m = std::fabs(div);
  }
  *max_abs = m;
  return KHO_OK;
}
int kho_debug_emf(kho_grid* g) {
  if (!g) return KHO_EINVAL;
  const double* P = g->P.data();
  for (int d = 0; d < 3; d++) compute_flux(*g, P, d);
  if (g->p.emf == KHO_EMF_UPWIND) {
    emf_upwind(*g, P, g->F[0].data(), g->F[1].data(), g->F[2].data(), g->emf[0].data(), g->emf[1].data(), g->emf[2].data());
  } else if (g->p.emf == KHO_EMF_CENTRED) {
    emf_centred(*g, P, g->F[0].data(), g->F[1].data(), g->F[2].data(), g->emf[0].data(), g->emf[1].data(), g->emf[2].data());
  } else {
    std::vector<double> raw[3] = {g->F[0], g->F[1], g->F[2]};
    flux_ct(*g, g->F[0].data(), g->F[1].data(), g->F[2].data(), g->emf[0].data(), g->emf[1].data(), g->emf[2].data());
    for (int d = 0; d < 3; d++) g->F[d] = raw[d];
  }
  return KHO_OK;
}
int kho_debug_fofc(kho_grid* g, const int* mask_with_ghosts) {
  if (!g || !mask_with_ghosts) return KHO_EINVAL;
  const double* P = g->P.data();
  for (int d = 0; d < 3; d++) compute_flux(*g, P, d);
  std::vector<int> mask(mask_with_ghosts, mask_with_ghosts + g->ntot);
  fill_ghosts_flag(*g, mask.data());
  fofc_reflux(*g, P, mask);
  return KHO_OK;
}
int kho_fill_ghosts(kho_grid* g) {
  if (!g) return KHO_EINVAL;
  fill_ghosts_prims(*g, g->P.data());
  return KHO_OK;
}

// ---- point-wise pieces ----
static void unpack(const double a[16], double m[4][4]) { for (int i = 0; i < 16; i++) m[i / 4][i % 4] = a[i]; }
static void make_geom(const double gcov[16], const double gcon[16], double gdet, Geom& G) {
  unpack(gcov, G.gcov); unpack(gcon, G.gcon); G.gdet = gdet; G.alpha = 1.0 / std::sqrt(-G.gcon[0][0]);
}

void kho_embed(const kho_params* p, const double X[3], double emb[3]) {
  if (p->coords == KHO_MINKOWSKI) { emb[0] = X[0]; emb[1] = X[1]; emb[2] = X[2]; return; }
  if (p->coords == KHO_KS) { emb[0] = X[0]; emb[1] = X[1]; emb[2] = X[2]; return; }
  double r, th, d1, d2;
  fmks_map<double>(*p, X[0], X[1], r, th, d1, d2);
  emb[0] = r; emb[1] = th; emb[2] = X[2];
}
void kho_metric(const kho_params* p, double x1, double x2, double gcov[16], double gcon[16], double* gdet, double* alpha) {
  Geom G;
  geom_at(*p, x1, x2, G);
  for (int m = 0; m < 16; m++) { gcov[m] = G.gcov[m / 4][m % 4]; gcon[m] = G.gcon[m / 4][m % 4]; }
  *gdet = G.gdet; *alpha = G.alpha;
}
void kho_conn(const kho_params* p, double x1, double x2, double conn[64]) { conn_exact(*p, x1, x2, conn); }
void kho_conn_fd(const kho_params* p, double x1, double x2, double h, double conn[64]) { conn_fd(*p, x1, x2, h, conn); }

void kho_fourvec(const double gcov[16], const double gcon[16], const double P[8], double out[17]) {
  Geom G; make_geom(gcov, gcon, 1.0, G);
  FourVec D;
  four_vectors(G.gcov, G.gcon, P, D);
  for (int m = 0; m < 4; m++) { out[m] = D.ucon[m]; out[4 + m] = D.ucov[m]; out[8 + m] = D.bcon[m]; out[12 + m] = D.bcov[m]; }
  out[16] = D.bsq;
}
void kho_prim_to_flux(const double gcov[16], const double gcon[16], double gdet, const double P[8], double gamma, int dir, double F[8]) {
  Geom G; make_geom(gcov, gcon, gdet, G);
  FourVec D;
  four_vectors(G.gcov, G.gcon, P, D);
  prim_to_flux(G, P, D, gamma, dir, F);
}
void kho_stress(const double gcov[16], const double gcon[16], const double P[8], double gamma, double T[16]) {
  Geom G; make_geom(gcov, gcon, 1.0, G);
  FourVec D;
  four_vectors(G.gcov, G.gcon, P, D);
  for (int mu = 0; mu < 4; mu++) stress_row(P, D, gamma, mu, &T[mu * 4]);
}
void kho_vchar(const double gcov[16], const double gcon[16], const double P[8], double gamma, int dir, double* vmax, double* vmin) {
  Geom G; make_geom(gcov, gcon, 1.0, G);
  FourVec D;
  four_vectors(G.gcov, G.gcon, P, D);
  vchar(G, P, D, gamma, dir, *vmax, *vmin);
}
void kho_recon(int kind, const double q[5], double* left, double* right) { recon(kind, q, *left, *right); }
void kho_llf(const double gcov[16], const double gcon[16], double gdet, const double PL[8], const double PR[8], double gamma, int dir, double F[8], double* ctop) {
  Geom G; make_geom(gcov, gcon, gdet, G);
  llf(G, PL, PR, gamma, dir, F, *ctop);
}
void kho_source(const double gcov[16], const double gcon[16], double gdet, const double conn[64], const double P[8], double gamma, double S[8]) {
  Geom G; make_geom(gcov, gcon, gdet, G);
  source(G, conn, P, gamma, S);
}
// Test hook (tests/test_oracle_forms.py): the norm Qt^2 of the projected momentum exactly as u2p() forms it, from the
// covariant components Q_mu it receives (no arithmetic of its own: the lines below are u2p()'s).
double kho_qtsq(const double gcov16[16], const double gcon16[16], double alpha, const double Qcov[4]) {
  double gcov[4][4], gcon[4][4];
  unpack(gcov16, gcov); unpack(gcon16, gcon);
  double Qcon[4];
  for (int m = 0; m < 4; m++) { double s = 0.0; for (int n = 0; n < 4; n++) s += gcon[m][n] * Qcov[n]; Qcon[m] = s; }
  double Qdotn = -alpha * Qcon[0];
  double ncon[4];
  for (int m = 0; m < 4; m++) ncon[m] = -alpha * gcon[m][0];
  double Qtcon[4];
  for (int m = 0; m < 4; m++) Qtcon[m] = Qcon[m] + Qdotn * ncon[m];
  double Qtsq = 0.0;
  for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) Qtsq += gcov[i][j] * Qtcon[i] * Qtcon[j];
  return Qtsq;
}

int kho_u2p(const double gcov[16], const double gcon[16], double gdet, const double U[8], const double Pguess[8], double gamma, double Pout[8]) {
  Geom G; make_geom(gcov, gcon, gdet, G);
  return u2p(G, U, Pguess, gamma, Pout);
}
int kho_u2p_kastaun(const double gcov[16], const double gcon[16], double gdet, const double U[8], const double Pguess[8], double gamma, double Pout[8]) {
  Geom G; make_geom(gcov, gcon, gdet, G);
  return u2p_kastaun(G, U, Pguess, gamma, Pout);
}
int kho_floors(const kho_params* p, const double gcov[16], const double gcon[16], double x1, double x2, double P[8]) {
  (void)x2;
  Geom G; make_geom(gcov, gcon, 1.0, G);
  return floors(*p, G, radius_at(*p, x1), P);
}
int kho_flux_ct_arrays(const kho_params* p, double* F1, double* F2, double* F3) {
  kho_grid g;
  g.p = *p;
  g.n[0] = p->n1; g.n[1] = p->n2; g.n[2] = p->n3;
  for (int d = 0; d < 3; d++) g.nt[d] = g.n[d] + 2 * NG;
  g.ntot = (long)g.nt[0] * g.nt[1] * g.nt[2];
  std::vector<double> e1(g.ntot, 0.0), e2(g.ntot, 0.0), e3(g.ntot, 0.0);
  flux_ct(g, F1, F2, F3, e1.data(), e2.data(), e3.data());
  return KHO_OK;
}

}  // extern "C"
