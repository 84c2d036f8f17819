// kh_device.cuh -- device-side building blocks of libkharm (sm_100a): packed symmetric metric,
// four-vectors, stress tensor rows, conserved variables / fluxes, fast-magnetosonic speeds,
// MC / WENO5 reconstruction, the 1D_W inversion and the floors.
//
// Written from the published scheme (DESIGN.md readings
// S1..S23).  Shares nothing with oracle/ (the CPU oracle is test infrastructure only).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#define KH_NGH 3
#define KH_NP 8

namespace kh {

enum { RHO = 0, UU = 1, U1 = 2, U2 = 3, U3 = 4, B1 = 5, B2 = 6, B3 = 7 };

// packed symmetric 4x4: (00,01,02,03,11,12,13,22,23,33)
__host__ __device__ __forceinline__ constexpr int sym(int m, int n) {
  return (m <= n) ? (m * 4 - (m * (m - 1)) / 2 + (n - m)) : (n * 4 - (n * (n - 1)) / 2 + (m - n));
}
enum { G00 = 0, G01 = 1, G02 = 2, G03 = 3, G11 = 4, G12 = 5, G13 = 6, G22 = 7, G23 = 8, G33 = 9 };

// geometry table components per location: 10 gcov, 10 gcon, gdet, alpha
#define KH_NGEO 22
#define KH_NCONN 40   // Gamma^lam_{mu nu}: lam * 10 + sym(mu, nu)

struct Geo {
  double gcov[10], gcon[10], gdet, alpha;
};

template <bool FLAT>
__device__ __forceinline__ void load_geo(Geo& G, const double* __restrict__ tab, long n2d, long p) {
  if (FLAT) {
#pragma unroll
    for (int c = 0; c < 10; c++) { G.gcov[c] = 0.0; G.gcon[c] = 0.0; }
    G.gcov[G00] = -1.0; G.gcov[G11] = 1.0; G.gcov[G22] = 1.0; G.gcov[G33] = 1.0;
    G.gcon[G00] = -1.0; G.gcon[G11] = 1.0; G.gcon[G22] = 1.0; G.gcon[G33] = 1.0;
    G.gdet = 1.0; G.alpha = 1.0;
  } else {
#pragma unroll
    for (int c = 0; c < 10; c++) { G.gcov[c] = __ldg(tab + c * n2d + p); G.gcon[c] = __ldg(tab + (10 + c) * n2d + p); }
    G.gdet = __ldg(tab + 20 * n2d + p);
    G.alpha = __ldg(tab + 21 * n2d + p);
  }
}

struct FourVec {
  double ucon[4], ucov[4], bcon[4], bcov[4], bsq;
};

__device__ __forceinline__ void lower(const double* __restrict__ g, const double v[4], double out[4]) {
  out[0] = g[G00] * v[0] + g[G01] * v[1] + g[G02] * v[2] + g[G03] * v[3];
  out[1] = g[G01] * v[0] + g[G11] * v[1] + g[G12] * v[2] + g[G13] * v[3];
  out[2] = g[G02] * v[0] + g[G12] * v[1] + g[G22] * v[2] + g[G23] * v[3];
  out[3] = g[G03] * v[0] + g[G13] * v[1] + g[G23] * v[2] + g[G33] * v[3];
}

__device__ __forceinline__ double spatial_norm2(const double* __restrict__ g, double a, double b, double c) {
  return g[G11] * a * a + g[G22] * b * b + g[G33] * c * c + 2.0 * (g[G12] * a * b + g[G13] * a * c + g[G23] * b * c);
}

// Reciprocal for the hot paths: MUFU.RCP64H seed (rcp.approx.ftz.f64, ~20 bits) + two Newton steps
// (4 DFMA) -> ~1 ulp.  IEEE division (x/y) costs ~3x the fp64-pipe slots; the step is bound by that
// pipe.  NOT for arguments that may be 0, inf or subnormal (gives NaN / flushes):
// callers guarantee a normal, non-zero argument.
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}

// S1: ut^i is the velocity projected into the normal observer's frame:  u^t = gamma/alpha,
// u^i = ut^i - gamma alpha g^{ti};  b^t = B^i u_i,  b^i = (B^i + b^t u^i)/u^t.
// Since n_i = 0, u_i = g_ij ut^j exactly and q^2 = ut^i u_i: 12 products instead of 9 + 12.
// 1/alpha = -g^tt alpha (alpha = (-g^tt)^(-1/2)).
__device__ __forceinline__ void four_vectors(const Geo& G, const double P[KH_NP], FourVec& D) {
  const double* __restrict__ g = G.gcov;
  const double v1 = P[U1], v2 = P[U2], v3 = P[U3];
  D.ucov[1] = g[G11] * v1 + g[G12] * v2 + g[G13] * v3;
  D.ucov[2] = g[G12] * v1 + g[G22] * v2 + g[G23] * v3;
  D.ucov[3] = g[G13] * v1 + g[G23] * v2 + g[G33] * v3;
  double qsq = v1 * D.ucov[1] + v2 * D.ucov[2] + v3 * D.ucov[3];
  double gamma = sqrt(1.0 + qsq);
  double ga = gamma * G.alpha;
  D.ucon[0] = -G.gcon[G00] * ga;
  D.ucon[1] = v1 - ga * G.gcon[G01];
  D.ucon[2] = v2 - ga * G.gcon[G02];
  D.ucon[3] = v3 - ga * G.gcon[G03];
  D.ucov[0] = g[G00] * D.ucon[0] + g[G01] * D.ucon[1] + g[G02] * D.ucon[2] + g[G03] * D.ucon[3];
  D.bcon[0] = P[B1] * D.ucov[1] + P[B2] * D.ucov[2] + P[B3] * D.ucov[3];
  double iut = fast_rcp(D.ucon[0]);
  D.bcon[1] = (P[B1] + D.bcon[0] * D.ucon[1]) * iut;
  D.bcon[2] = (P[B2] + D.bcon[0] * D.ucon[2]) * iut;
  D.bcon[3] = (P[B3] + D.bcon[0] * D.ucon[3]) * iut;
  lower(G.gcov, D.bcon, D.bcov);
  D.bsq = D.bcon[0] * D.bcov[0] + D.bcon[1] * D.bcov[1] + D.bcon[2] * D.bcov[2] + D.bcon[3] * D.bcov[3];
}

// b^2 alone (floors): b^2 = (g_ij B^i B^j + (b^t)^2) / (u^t)^2 with b^t = B^i u_i; also returns q^2.
__device__ __forceinline__ double bsq_only(const Geo& G, const double P[KH_NP], double& qsq) {
  const double* __restrict__ g = G.gcov;
  const double v1 = P[U1], v2 = P[U2], v3 = P[U3], b1 = P[B1], b2 = P[B2], b3 = P[B3];
  double c1 = g[G11] * v1 + g[G12] * v2 + g[G13] * v3;
  double c2 = g[G12] * v1 + g[G22] * v2 + g[G23] * v3;
  double c3 = g[G13] * v1 + g[G23] * v2 + g[G33] * v3;
  qsq = v1 * c1 + v2 * c2 + v3 * c3;
  double bt = b1 * c1 + b2 * c2 + b3 * c3;
  double BB = spatial_norm2(g, b1, b2, b3);
  double iut2 = -fast_rcp((1.0 + qsq) * G.gcon[G00]);      // 1/(u^t)^2 = alpha^2/gamma^2 = -1/(gamma^2 g^tt)
  return (BB + bt * bt) * iut2;
}

// T^dir_nu = (w + b^2) u^dir u_nu + (p + b^2/2) delta^dir_nu - b^dir b_nu       [eq. 1.1, P:347]
__device__ __forceinline__ void stress_row(const double P[KH_NP], const FourVec& D, double gam, int dir, double T[4]) {
  double pg = (gam - 1.0) * P[UU];
  double eta = P[RHO] + P[UU] + pg + D.bsq;
  double ptot = pg + 0.5 * D.bsq;
  double eu = eta * D.ucon[dir], bd = D.bcon[dir];
#pragma unroll
  for (int nu = 0; nu < 4; nu++) T[nu] = eu * D.ucov[nu] - bd * D.bcov[nu];
  T[dir] += ptot;
}

// dir = 0 -> U (S8: energy slot T^t_t + rho u^t);  dir = 1..3 -> F^dir.  Only the five hydro slots
// and, for dir > 0, the two non-trivial induction slots are meaningful; F^dir[B^dir] = 0.
__device__ __forceinline__ void prim_to_flux(const Geo& G, const double P[KH_NP], const FourVec& D, double gam, int dir,
                                             double F[KH_NP]) {
  double T[4];
  stress_row(P, D, gam, dir, T);
  double rhou = P[RHO] * D.ucon[dir];
  F[RHO] = G.gdet * rhou;
  F[UU] = G.gdet * (T[0] + rhou);
  F[U1] = G.gdet * T[1];
  F[U2] = G.gdet * T[2];
  F[U3] = G.gdet * T[3];
  if (dir == 0) {
    F[B1] = G.gdet * P[B1]; F[B2] = G.gdet * P[B2]; F[B3] = G.gdet * P[B3];
  } else {
#pragma unroll
    for (int i = 1; i < 4; i++)
      F[B1 + i - 1] = (i == dir) ? 0.0 : G.gdet * (D.bcon[i] * D.ucon[dir] - D.bcon[dir] * D.ucon[i]);
  }
}

// S9: fast-magnetosonic bound.  Roots of A v^2 - B v + C = 0.
__device__ __forceinline__ void vchar(const Geo& G, const double P[KH_NP], const FourVec& D, double gam, int dir,
                                      double& vmax, double& vmin) {
  double ef = P[RHO] + gam * P[UU];
  double ee = D.bsq + ef;
  double va2 = D.bsq * fast_rcp(ee);
  double cs2 = gam * (gam - 1.0) * P[UU] * fast_rcp(ef);
  double cms2 = cs2 + va2 - cs2 * va2;
  if (!(cms2 >= 0.0)) cms2 = 0.0;
  if (cms2 > 1.0) cms2 = 1.0;
  double ut = D.ucon[0], ud = D.ucon[dir];
  double gtt = G.gcon[G00], gtd = G.gcon[sym(0, dir)], gdd = G.gcon[sym(dir, dir)];
  double A = ut * ut - (gtt + ut * ut) * cms2;
  double B = 2.0 * (ud * ut - (gtd + ud * ut) * cms2);
  // B^2 - 4AC reduced algebraically ((u^d u^t)^2 - u^t^2 u^d^2 cancels identically): well conditioned in cold zones
  double disc = 4.0 * cms2 * ((1.0 - cms2) * (ut * ut * gdd - 2.0 * ut * ud * gtd + ud * ud * gtt) + cms2 * (gtd * gtd - gtt * gdd));
  if (!(disc >= 0.0)) disc = 0.0;
  double sq = sqrt(disc);
  double i2a = 0.5 * fast_rcp(A);
  double vp = (B + sq) * i2a, vm = (B - sq) * i2a;
  vmax = vp > vm ? vp : vm;
  vmin = vp > vm ? vm : vp;
}

// ---------------------------------------------------------------------------------------------
// Reconstruction.  Both return the face value on the side of x3 towards x4 given the
// stencil (x1..x5) centred on x3 ("right" value); the left value is the mirror image.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double mc_slope(double qm, double q0, double qp) {   // S11
  double dm = 2.0 * (q0 - qm), dp = 2.0 * (qp - q0), dc = 0.5 * (qp - qm);
  double s = 0.0;
  if (dm * dp > 0.0) {
    s = dc;
    if (fabs(dm) < fabs(s)) s = dm;
    if (fabs(dp) < fabs(s)) s = dp;
  }
  return s;
}

// S12: Jiang-Shu WENO5 with eps = 1e-26.  The three non-linear weights d_k/(eps+beta_k)^2 are
// formed over the common denominator so that one division serves the whole face value.
__device__ __forceinline__ double weno5_right(double x1, double x2, double x3, double x4, double x5) {
  const double eps = 1e-26;
  double d1 = x1 - 2.0 * x2 + x3, e1 = x1 - 4.0 * x2 + 3.0 * x3;
  double d2 = x2 - 2.0 * x3 + x4, e2 = x4 - x2;
  double d3 = x3 - 2.0 * x4 + x5, e3 = 3.0 * x3 - 4.0 * x4 + x5;
  double b1 = (13.0 / 12.0) * d1 * d1 + 0.25 * e1 * e1 + eps;
  double b2 = (13.0 / 12.0) * d2 * d2 + 0.25 * e2 * e2 + eps;
  double b3 = (13.0 / 12.0) * d3 * d3 + 0.25 * e3 * e3 + eps;
  double a1 = b1 * b1, a2 = b2 * b2, a3 = b3 * b3;
  double w1 = 0.1 * (a2 * a3), w2 = 0.6 * (a1 * a3), w3 = 0.3 * (a1 * a2);
  double v1 = (1.0 / 3.0) * x1 - (7.0 / 6.0) * x2 + (11.0 / 6.0) * x3;
  double v2 = -(1.0 / 6.0) * x2 + (5.0 / 6.0) * x3 + (1.0 / 3.0) * x4;
  double v3 = (1.0 / 3.0) * x3 + (5.0 / 6.0) * x4 - (1.0 / 6.0) * x5;
  return (w1 * v1 + w2 * v2 + w3 * v3) / (w1 + w2 + w3);
}

// Zone-centred forms: both face values of the zone centred on x3 in one pass.  qm = value at the lower
// face (the RIGHT state of face i-1/2), qp = value at the upper face (the LEFT state of face i+1/2).
// The smoothness indicators are shared by the two faces (mirror image: beta1 <-> beta3), and each
// quotient is one fast reciprocal.
__device__ __forceinline__ void weno5_zone(double x1, double x2, double x3, double x4, double x5, double& qm, double& qp) {
  const double eps = 1e-26;
  double d1 = x1 - 2.0 * x2 + x3, e1 = x1 - 4.0 * x2 + 3.0 * x3;
  double d2 = x2 - 2.0 * x3 + x4, e2 = x4 - x2;
  double d3 = x3 - 2.0 * x4 + x5, e3 = 3.0 * x3 - 4.0 * x4 + x5;
  double b1 = (13.0 / 12.0) * d1 * d1 + 0.25 * e1 * e1 + eps;
  double b2 = (13.0 / 12.0) * d2 * d2 + 0.25 * e2 * e2 + eps;
  double b3 = (13.0 / 12.0) * d3 * d3 + 0.25 * e3 * e3 + eps;
  double a1 = b1 * b1, a2 = b2 * b2, a3 = b3 * b3;
  double p23 = a2 * a3, p13 = 0.6 * (a1 * a3), p12 = a1 * a2;
  // upper face: weights (0.1, 0.6, 0.3) on the stencils (x1..x3), (x2..x4), (x3..x5)
  double w1 = 0.1 * p23, w3 = 0.3 * p12;
  double v1 = (1.0 / 3.0) * x1 - (7.0 / 6.0) * x2 + (11.0 / 6.0) * x3;
  double v2 = -(1.0 / 6.0) * x2 + (5.0 / 6.0) * x3 + (1.0 / 3.0) * x4;
  double v3 = (1.0 / 3.0) * x3 + (5.0 / 6.0) * x4 - (1.0 / 6.0) * x5;
  qp = (w1 * v1 + p13 * v2 + w3 * v3) * fast_rcp(w1 + p13 + w3);
  // lower face: the mirror image, weights (0.1, 0.6, 0.3) on (x5..x3), (x4..x2), (x3..x1)
  double m1 = 0.1 * p12, m3 = 0.3 * p23;
  double u1 = (1.0 / 3.0) * x5 - (7.0 / 6.0) * x4 + (11.0 / 6.0) * x3;
  double u2 = -(1.0 / 6.0) * x4 + (5.0 / 6.0) * x3 + (1.0 / 3.0) * x2;
  double u3 = (1.0 / 3.0) * x3 + (5.0 / 6.0) * x2 - (1.0 / 6.0) * x1;
  qm = (m1 * u1 + p13 * u2 + m3 * u3) * fast_rcp(m1 + p13 + m3);
}
__device__ __forceinline__ void mc_zone(double x2, double x3, double x4, double& qm, double& qp) {
  double h = 0.5 * mc_slope(x2, x3, x4);
  qm = x3 - h;
  qp = x3 + h;
}
template <int RECON>
__device__ __forceinline__ void recon_zone(const double* __restrict__ A, long st, double& qm, double& qp) {
  if (RECON == 0) mc_zone(A[-st], A[0], A[st], qm, qp);
  else weno5_zone(A[-2 * st], A[-st], A[0], A[st], A[2 * st], qm, qp);
}

// ---------------------------------------------------------------------------------------------
// 1D_W inversion (ref [37]) in the W' = W - D variable (S16).
// ---------------------------------------------------------------------------------------------
struct U2P {
  double D, Bsq, QdotB, QdotBsq, Qtsq, Ep, gam;
  __device__ __forceinline__ double vsq(double W) const {
    double WB = Bsq + W;
    return (Qtsq * W * W + QdotBsq * (Bsq + 2.0 * W)) / (WB * WB * W * W);
  }
  // f(W') and f'(W') (S16).  Reciprocals by fast_rcp: W, W + B^2, 1 - v^2 (clamped) and 1 + gamma are
  // positive normal numbers here.
  __device__ __forceinline__ void func(double Wp, double& f, double& df) const {
    double W = Wp + D, WB = W + Bsq;
    double iW = fast_rcp(W), iWB = fast_rcp(WB);
    double iW2 = iW * iW, iW3 = iW2 * iW, iWB2 = iWB * iWB, iWB3 = iWB2 * iWB;
    double v2 = (Qtsq * W * W + QdotBsq * (Bsq + 2.0 * W)) * (iWB2 * iW2);
    v2 = fmax(v2, 0.0);
    v2 = fmin(v2, 1.0 - 1e-12);
    double omv = 1.0 - v2;
    double gsq = fast_rcp(omv), g = sqrt(gsq);
    double k = (gam - 1.0) / gam;
    double p = k * (Wp - D * v2 * gsq * fast_rcp(1.0 + g)) * omv;
    f = Wp - p + 0.5 * Bsq * (1.0 + v2) - 0.5 * QdotBsq * iW2 - Ep;
    double dv2 = -2.0 * (Qtsq * W * W * W + QdotBsq * (3.0 * W * W + 3.0 * W * Bsq + Bsq * Bsq)) * iW3 * iWB3;
    double dp = k * (omv - (W - 0.5 * D * g) * dv2);
    df = 1.0 - dp + 0.5 * Bsq * dv2 + QdotBsq * iW3;
  }
};

// Returns the flag; on failure the hydro primitives of Pout keep the guess, B is always updated.
__device__ __forceinline__ int u_to_p(const Geo& G, const double U[KH_NP], const double Pg[KH_NP], double gam,
                                      double Pout[KH_NP]) {
#pragma unroll
  for (int v = 0; v < 5; v++) Pout[v] = Pg[v];
  double igdet = 1.0 / G.gdet;
  Pout[B1] = U[B1] * igdet; Pout[B2] = U[B2] * igdet; Pout[B3] = U[B3] * igdet;
  bool fin = true;
#pragma unroll
  for (int v = 0; v < KH_NP; v++) fin = fin && isfinite(U[v]);
  if (!fin || !(U[RHO] > 0.0)) return 1;

  double alpha = G.alpha, k = alpha * igdet;
  U2P c;
  c.gam = gam;
  c.D = k * U[RHO];
  double Bc[4] = {0.0, k * U[B1], k * U[B2], k * U[B3]};
  double Qcov[4] = {k * (U[UU] - U[RHO]), k * U[U1], k * U[U2], k * U[U3]};
  double Qcon[4];
  lower(G.gcon, Qcov, Qcon);   // raising with the packed inverse metric
  c.Bsq = spatial_norm2(G.gcov, Bc[1], Bc[2], Bc[3]);
  c.QdotB = Qcov[1] * Bc[1] + Qcov[2] * Bc[2] + Qcov[3] * Bc[3];
  c.QdotBsq = c.QdotB * c.QdotB;
  double Qdotn = -alpha * Qcon[0];
  c.Ep = -Qdotn - c.D;
  double Qt1 = Qcon[1] + Qdotn * (-alpha * G.gcon[G01]);
  double Qt2 = Qcon[2] + Qdotn * (-alpha * G.gcon[G02]);
  double Qt3 = Qcon[3] + Qdotn * (-alpha * G.gcon[G03]);
  // Qt^2 = Q.Q + (Q.n)^2 as the spatial norm of the projected vector (its time component vanishes):
  // no cancellation, never negative (S16).
  c.Qtsq = spatial_norm2(G.gcov, Qt1, Qt2, Qt3);

  double qsq = spatial_norm2(G.gcov, Pg[U1], Pg[U2], Pg[U3]);
  double W = (Pg[RHO] + gam * Pg[UU]) * (1.0 + qsq);
  if (!(W > 0.0) || !isfinite(W)) W = c.D;
  for (int it = 0; it < 30 && !(c.vsq(W) < 1.0); it++) W *= 10.0;
  double Wp = W - c.D;

  bool conv = false;
  for (int it = 0; it < 20; it++) {
    double f, df;
    c.func(Wp, f, df);
    double Wold = Wp + c.D;
    double Wpn = Wp - f * fast_rcp(df);
    if (!(Wpn + c.D > 0.0)) Wpn = 0.5 * Wold - c.D;
    double dW = Wpn - Wp;
    Wp = Wpn;
    if (fabs(dW) <= 1e-12 * (Wp + c.D)) { conv = true; break; }
  }
  if (!conv) return 2;

  W = Wp + c.D;
  double v2 = c.vsq(W);
  if (!(v2 >= 0.0) || !(v2 < 1.0) || !(W > 0.0)) return 3;
  double gsq = 1.0 / (1.0 - v2), g = sqrt(gsq);
  double rho = c.D / g;
  double u = (Wp - c.D * v2 * gsq / (1.0 + g)) / (gsq * gam);
  double fac = g / (W + c.Bsq), qbw = c.QdotB / W;
  double ut1 = fac * (Qt1 + qbw * Bc[1]);
  double ut2 = fac * (Qt2 + qbw * Bc[2]);
  double ut3 = fac * (Qt3 + qbw * Bc[3]);
  if (!isfinite(rho) || !isfinite(u) || !isfinite(ut1) || !isfinite(ut2) || !isfinite(ut3)) return 7;
  bool badrho = !(rho > 0.0), badu = (u < 0.0);
  if (badrho && badu) return 6;
  if (badrho) return 4;
  if (badu) return 5;
  Pout[RHO] = rho; Pout[UU] = u; Pout[U1] = ut1; Pout[U2] = ut2; Pout[U3] = ut3;
  return 0;
}

// ---------------------------------------------------------------------------------------------
// Floors and ceilings in the fluid frame (S18).  rho_g, u_g: tabulated geometric floors.
// ---------------------------------------------------------------------------------------------
struct FloorPar {
  double inv_bsq_over_rho_max, inv_bsq_over_u_max, u_over_rho_max, gamma_max;   // inverses formed once on the host
};

__device__ __forceinline__ int apply_floors(const Geo& G, const FloorPar& fp, double rho_g, double u_g, double P[KH_NP]) {
  int flag = 0;
  double qsq;
  const double bsq = bsq_only(G, P, qsq);
  double rho_b = bsq * fp.inv_bsq_over_rho_max, u_b = bsq * fp.inv_bsq_over_u_max;
  double rho_fl = rho_b > rho_g ? rho_b : rho_g;
  double u_fl = u_b > u_g ? u_b : u_g;
  if (P[RHO] < rho_fl) { P[RHO] = rho_fl; flag |= (rho_b > rho_g) ? 2 : 1; }
  if (P[UU] < u_fl) { P[UU] = u_fl; flag |= (u_b > u_g) ? 8 : 4; }
  if (P[UU] > fp.u_over_rho_max * P[RHO]) { P[UU] = fp.u_over_rho_max * P[RHO]; flag |= 16; }
  double gamma = sqrt(1.0 + qsq);
  if (gamma > fp.gamma_max) {
    double f = sqrt((fp.gamma_max * fp.gamma_max - 1.0) / (gamma * gamma - 1.0));
    P[U1] *= f; P[U2] *= f; P[U3] *= f;
    flag |= 32;
  }
  return flag;
}

}  // namespace kh
