// kh_geometry.cuh -- K1: one-time geometry precompute ("caches of expensive-to-calculate
// quantities such as the metric and connection coefficients").  Kerr-Schild metric (S4), the FMKS map
// (P:111, S5), 4x4 inverse, sqrt(-g), lapse, and the connection by EXACT differentiation with
// forward-mode dual numbers (S6b).  One thread per (i, j) table point; x3 does not enter
// (stationary, axisymmetric).
#pragma once
#include "kh_device.cuh"

namespace kh {

struct GeomPar {
  int coords;
  double a, hslope, poly_xt, poly_alpha, mks_smooth, x1_start;
  double xmin1, xmin2, dx1, dx2;
  int nt1, nt2, n2;
  int polar_lo, polar_hi;
  double rho_min, u_min, r_char, gamma;
};

// value + d/dx1 + d/dx2
struct D2 {
  double v, a, b;
};
__device__ __forceinline__ D2 mk(double v) { return D2{v, 0.0, 0.0}; }
__device__ __forceinline__ D2 operator+(D2 x, D2 y) { return D2{x.v + y.v, x.a + y.a, x.b + y.b}; }
__device__ __forceinline__ D2 operator-(D2 x, D2 y) { return D2{x.v - y.v, x.a - y.a, x.b - y.b}; }
__device__ __forceinline__ D2 operator*(D2 x, D2 y) { return D2{x.v * y.v, x.a * y.v + x.v * y.a, x.b * y.v + x.v * y.b}; }
__device__ __forceinline__ D2 operator*(double c, D2 y) { return D2{c * y.v, c * y.a, c * y.b}; }
__device__ __forceinline__ D2 operator+(double c, D2 y) { return D2{c + y.v, y.a, y.b}; }
__device__ __forceinline__ D2 operator/(D2 x, D2 y) {
  double iy = 1.0 / y.v, q = x.v * iy;
  return D2{q, (x.a - q * y.a) * iy, (x.b - q * y.b) * iy};
}
__device__ __forceinline__ D2 dsin(D2 x) { double s, c; sincos(x.v, &s, &c); return D2{s, c * x.a, c * x.b}; }
__device__ __forceinline__ D2 dcos(D2 x) { double s, c; sincos(x.v, &s, &c); return D2{c, -s * x.a, -s * x.b}; }
__device__ __forceinline__ D2 dexp(D2 x) { double e = exp(x.v); return D2{e, e * x.a, e * x.b}; }
__device__ __forceinline__ D2 dpowc(D2 x, double n) {
  double pm1 = pow(x.v, n - 1.0);
  return D2{pm1 * x.v, n * pm1 * x.a, n * pm1 * x.b};
}

// Native covariant metric with its x1, x2 derivatives (packed symmetric), and the radius.
// emb[5] returns (r, theta, dr/dx1, dtheta/dx1, dtheta/dx2) for the closed-form inverse.
__device__ inline void gcov_dual(const GeomPar& p, double x1, double x2, D2 g[10], double& radius, double emb[5]) {
  for (int c = 0; c < 10; c++) g[c] = mk(0.0);
  if (p.coords == 0) {
    g[G00] = mk(-1.0); g[G11] = mk(1.0); g[G22] = mk(1.0); g[G33] = mk(1.0);
    radius = 1.0;
    emb[0] = emb[1] = 0.0; emb[2] = 1.0; emb[3] = 0.0; emb[4] = 1.0;
    return;
  }
  D2 X1{x1, 1.0, 0.0}, X2{x2, 0.0, 1.0};
  D2 r, th, t1 = mk(0.0), t2 = mk(1.0), jr = mk(1.0);   // jr = dr/dx1, t1 = dth/dx1, t2 = dth/dx2
  if (p.coords == 1) {
    r = X1; th = X2;
  } else {
    const double pi = 3.14159265358979323846;
    r = dexp(X1);
    jr = r;
    D2 y = 2.0 * X2 + mk(-1.0);
    D2 arg = (2.0 * pi) * X2;
    D2 thG = pi * X2 + (0.5 * (1.0 - p.hslope)) * dsin(arg);
    D2 dthG = pi * (1.0 + (1.0 - p.hslope) * dcos(arg));
    double norm = 0.5 * pi / (1.0 + pow(p.poly_xt, -p.poly_alpha) / (p.poly_alpha + 1.0));
    D2 ya = dpowc((1.0 / p.poly_xt) * y, p.poly_alpha);
    D2 thJ = norm * (y * (1.0 + (1.0 / (p.poly_alpha + 1.0)) * ya)) + mk(0.5 * pi);
    D2 dthJ = (2.0 * norm) * (1.0 + ya);
    D2 e = dexp(p.mks_smooth * (mk(p.x1_start) - X1));
    th = thG + e * (thJ - thG);
    t1 = (-p.mks_smooth) * (e * (thJ - thG));
    t2 = dthG + e * (dthJ - dthG);
  }
  radius = r.v;
  emb[0] = r.v; emb[1] = th.v; emb[2] = jr.v; emb[3] = t1.v; emb[4] = t2.v;
  // Kerr-Schild in (t, r, theta, phi)
  D2 s = dsin(th), c = dcos(th);
  D2 s2 = s * s;
  D2 Sig = r * r + (p.a * p.a) * (c * c);
  D2 f = (2.0 * r) / Sig;
  D2 one_f = 1.0 + f;
  D2 gtt = mk(-1.0) + f, gtr = f, gtp = (-p.a) * (f * s2), grr = one_f, grp = (-p.a) * (s2 * one_f);
  D2 gthth = Sig, gpp = s2 * (Sig + (p.a * p.a) * (s2 * one_f));
  // native = L^T g L with L = [[1,0,0,0],[0,jr,0,0],[0,t1,t2,0],[0,0,0,1]]
  g[G00] = gtt;
  g[G01] = jr * gtr;
  g[G03] = gtp;
  g[G11] = jr * jr * grr + t1 * t1 * gthth;
  g[G12] = t1 * t2 * gthth;
  g[G13] = jr * grp;
  g[G22] = t2 * t2 * gthth;
  g[G33] = gpp;
}

// Inverse and determinant of a symmetric 4x4 via 2x2 sub-determinants.
__device__ inline double invert_sym4(const double g[10], double inv[10]) {
  double a00 = g[G00], a01 = g[G01], a02 = g[G02], a03 = g[G03];
  double a11 = g[G11], a12 = g[G12], a13 = g[G13], a22 = g[G22], a23 = g[G23], a33 = g[G33];
  double a10 = a01, a20 = a02, a21 = a12, a30 = a03, a31 = a13, a32 = a23;
  double s0 = a00 * a11 - a10 * a01, s1 = a00 * a12 - a10 * a02, s2 = a00 * a13 - a10 * a03;
  double s3 = a01 * a12 - a11 * a02, s4 = a01 * a13 - a11 * a03, s5 = a02 * a13 - a12 * a03;
  double c5 = a22 * a33 - a32 * a23, c4 = a21 * a33 - a31 * a23, c3 = a21 * a32 - a31 * a22;
  double c2 = a20 * a33 - a30 * a23, c1 = a20 * a32 - a30 * a22, c0 = a20 * a31 - a30 * a21;
  double det = s0 * c5 - s1 * c4 + s2 * c3 + s3 * c2 - s4 * c1 + s5 * c0;
  double id = 1.0 / det;
  inv[G00] = (a11 * c5 - a12 * c4 + a13 * c3) * id;
  inv[G01] = (-a01 * c5 + a02 * c4 - a03 * c3) * id;
  inv[G02] = (a31 * s5 - a32 * s4 + a33 * s3) * id;
  inv[G03] = (-a21 * s5 + a22 * s4 - a23 * s3) * id;
  inv[G11] = (a00 * c5 - a02 * c2 + a03 * c1) * id;
  inv[G12] = (-a30 * s5 + a32 * s2 - a33 * s1) * id;
  inv[G13] = (a20 * s5 - a22 * s2 + a23 * s1) * id;
  inv[G22] = (a30 * s4 - a31 * s2 + a33 * s0) * id;
  inv[G23] = (-a20 * s4 + a21 * s2 - a23 * s0) * id;
  inv[G33] = (a20 * s3 - a21 * s1 + a22 * s0) * id;
  return det;
}

// tab[loc]: KH_NGEO components x n2d; conn: KH_NCONN x n2d; dgt: KH_NDG x n2d (source table of the update
// kernel: sqrt(-g) w d_nu g_{kap lam}, nu = 1, 2); floorp: 2 x n2d (rho, u geometric floors)
__global__ void geometry_kernel(GeomPar p, double* __restrict__ tab0, double* __restrict__ tab1, double* __restrict__ tab2,
                                double* __restrict__ tab3, double* __restrict__ conn, double* __restrict__ dgt, double* __restrict__ floorp) {
  int ii = blockIdx.x * blockDim.x + threadIdx.x, jj = blockIdx.y;
  if (ii >= p.nt1 || jj >= p.nt2) return;
  long n2d = (long)p.nt1 * p.nt2, pt = (long)jj * p.nt1 + ii;
  int i = ii - KH_NGH, j = jj - KH_NGH;
  double xc1 = p.xmin1 + (i + 0.5) * p.dx1, xf1 = p.xmin1 + i * p.dx1;
  double xc2 = p.xmin2 + (j + 0.5) * p.dx2, xf2 = p.xmin2 + j * p.dx2;
  double* tabs[4] = {tab0, tab1, tab2, tab3};
  for (int loc = 0; loc < 4; loc++) {
    double x1 = (loc == 1) ? xf1 : xc1, x2 = (loc == 2) ? xf2 : xc2;   // S3: metric AT the face centre
    D2 g[10];
    double radius;
    double emb[5];
    gcov_dual(p, x1, x2, g, radius, emb);
    double gc[10], gi[10], gdet;
    for (int c = 0; c < 10; c++) gc[c] = g[c].v;
    if (p.coords == 0) {
      for (int c = 0; c < 10; c++) gi[c] = gc[c];
      gdet = 1.0;
    } else {
      // S6a: closed-form Kerr-Schild inverse pushed through the inverse Jacobian of the map; the generic
      // inverse (invert_sym4, kept for checking) loses (condition number) x eps near the polar axis.
      double r = emb[0], th = emb[1], ijr = 1.0 / emb[2], t1 = emb[3], it2 = 1.0 / emb[4];
      double sn, cs;
      sincos(th, &sn, &cs);
      double Sig = r * r + p.a * p.a * cs * cs, iS = 1.0 / Sig, f = 2.0 * r * iS;
      double ktt = -(1.0 + f), ktr = f, krr = (r * r - 2.0 * r + p.a * p.a) * iS, krp = p.a * iS, kthth = iS;
      double kpp = 1.0 / (Sig * sn * sn);
      double m11 = ijr, m21 = -t1 * ijr * it2, m22 = it2;      // d x1/dr, d x2/dr, d x2/dtheta
      gi[G00] = ktt;
      gi[G01] = m11 * ktr;
      gi[G02] = m21 * ktr;
      gi[G03] = 0.0;
      gi[G11] = m11 * m11 * krr;
      gi[G12] = m11 * m21 * krr;
      gi[G13] = m11 * krp;
      gi[G22] = m21 * m21 * krr + m22 * m22 * kthth;
      gi[G23] = m21 * krp;
      gi[G33] = kpp;
      gdet = fabs(Sig * sn * emb[2] * emb[4]);
    }
    double alpha = 1.0 / sqrt(-gi[G00]);
    bool axis = (loc == 2) && ((j == 0 && p.polar_lo) || (j == p.n2 && p.polar_hi));   // S7
    double* t = tabs[loc];
    for (int c = 0; c < 10; c++) { t[c * n2d + pt] = axis ? 0.0 : gc[c]; t[(10 + c) * n2d + pt] = axis ? 0.0 : gi[c]; }
    t[20 * n2d + pt] = axis ? 0.0 : gdet;
    t[21 * n2d + pt] = axis ? 0.0 : alpha;
    if (loc == 0) {
      // Gamma^lam_{mu nu} = 1/2 g^{lam kap} (d_mu g_{kap nu} + d_nu g_{kap mu} - d_kap g_{mu nu}), d_t = d_3 = 0
      for (int lam = 0; lam < 4; lam++)
        for (int mu = 0; mu < 4; mu++)
          for (int nu = mu; nu < 4; nu++) {
            double s = 0.0;
            for (int kap = 0; kap < 4; kap++) {
              double dmu = (mu == 1) ? g[sym(kap, nu)].a : (mu == 2 ? g[sym(kap, nu)].b : 0.0);
              double dnu = (nu == 1) ? g[sym(kap, mu)].a : (nu == 2 ? g[sym(kap, mu)].b : 0.0);
              double dka = (kap == 1) ? g[sym(mu, nu)].a : (kap == 2 ? g[sym(mu, nu)].b : 0.0);
              s += gi[sym(lam, kap)] * (dmu + dnu - dka);
            }
            conn[(lam * 10 + sym(mu, nu)) * n2d + pt] = 0.5 * s;
          }
      // source table: S_nu = sqrt(-g) 1/2 T^{kap lam} d_nu g_{kap lam} = sum over packed pairs c of T^c dgt[nu][c]
      for (int c = 0; c < 10; c++) {
        bool diag = (c == G00 || c == G11 || c == G22 || c == G33);
        double w = diag ? 0.5 : 1.0;
        dgt[c * n2d + pt] = gdet * w * g[c].a;
        dgt[(10 + c) * n2d + pt] = gdet * w * g[c].b;
      }
      double sfl = (p.coords == 0) ? 1.0 : 1.0 / (radius * radius) / (1.0 + radius / p.r_char);
      floorp[pt] = p.rho_min * sfl;
      floorp[n2d + pt] = p.u_min * pow(sfl, p.gamma);
    }
  }
}

}  // namespace kh
