// kh_device.cuh -- device-side building blocks of libkharm (sm_100a): packed symmetric metric,
// four-vectors, conserved variables / fluxes, fast-magnetosonic speeds, MC / WENO5 reconstruction,
// the 1D_W inversion and the floors.
//
// Written from the published scheme (DESIGN.md readings
// S1..S23).  Shares nothing with oracle/ (the CPU oracle is test infrastructure only).
//
// The step is bound by the fp64 pipe (one DFMA/DMUL/DADD holds a sub-partition's
// pipe for 2 cycles per warp), so everything here is written for a minimal fp64 INSTRUCTION count:
// algebraically reduced forms, shared sub-expressions between the L and R state of a face and between a
// zone's two faces, reciprocals / square roots from the MUFU seeds with one third-order correction, and
// the structural zeros of the Kerr-Schild family (g_02 = g_23 = g^03 = 0, also in FMKS) skipped.
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
#define KH_NCONN 40   // Gamma^lam_{mu nu}: lam * 10 + sym(mu, nu)       (kh_get_conn only)
#define KH_NDG 20     // source table: sqrt(-g) w_c d_nu g_c, nu = 1,2, c = packed pair (w = 1/2 diagonal, 1 off-diagonal)

// ---------------------------------------------------------------------------------------------
// Fast reciprocal / reciprocal square root / square root: MUFU seed (rcp/rsqrt.approx.ftz.f64,
// relative error < 2^-20) + ONE third-order correction -> error ~ seed^3 < 2^-60, i.e. the result is
// within 1 ulp of the IEEE one.  IEEE x/y and sqrt() cost ~3x the fp64-pipe slots.
// NOT for arguments that may be 0, inf, NaN-producing or subnormal: callers guarantee normal, positive
// (rcp: non-zero) arguments.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);          // 1/x = r / (1 - e) = r (1 + e + e^2 + O(e^3))
  double t = fma(e, e, e);
  return fma(r, t, r);
}
__device__ __forceinline__ double fast_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double xy = x * y;
  double e = fma(-xy, y, 1.0);         // x^(-1/2) = y (1 - e)^(-1/2) = y (1 + e/2 + 3 e^2/8 + O(e^3))
  double p = fma(0.375, e, 0.5);
  return fma(y, p * e, y);
}
__device__ __forceinline__ double fast_sqrt(double x) {   // x > 0 normal
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y;
  double e = fma(-g, y, 1.0);
  double p = fma(0.375, e, 0.5);
  return fma(g, p * e, g);
}

// ---------------------------------------------------------------------------------------------
// Metric at one table point.  FLAT (Minkowski-Cartesian): compile-time constants, no loads (the paper's
// own compile-time switch).  Otherwise the Kerr-Schild family (KS, FMKS): g_02 = g_23 = 0 and
// g^03 = 0 identically (the geometry kernel stores exact zeros), so those entries are neither loaded nor
// multiplied -- bit-identical to the general contraction for finite operands.
// ---------------------------------------------------------------------------------------------
struct Geo {
  double c00, c01, c03, c11, c12, c13, c22, c33;           // g_{mu nu} (non-zero entries)
  double n00, n01, n02, n11, n12, n13, n22, n23, n33;      // g^{mu nu} (non-zero entries)
  double gdet, alpha;
};

// LEVEL 0: what a face flux of direction DIR needs (g^dd and g^td besides the covariant metric);
// LEVEL 1: everything (zone centres: source term, inversion).
template <bool FLAT, int DIR, int LEVEL>
__device__ __forceinline__ void load_geo(Geo& G, const double* __restrict__ tab, long n2d, long p) {
  if (FLAT) {
    G.c00 = -1.0; G.c11 = G.c22 = G.c33 = 1.0; G.c01 = G.c03 = G.c12 = G.c13 = 0.0;
    G.n00 = -1.0; G.n11 = G.n22 = G.n33 = 1.0; G.n01 = G.n02 = G.n12 = G.n13 = G.n23 = 0.0;
    G.gdet = 1.0; G.alpha = 1.0;
    return;
  }
#define KH_LD(c) __ldg(tab + (long)(c) * n2d + p)
  G.c00 = KH_LD(G00); G.c01 = KH_LD(G01); G.c03 = KH_LD(G03); G.c11 = KH_LD(G11); G.c12 = KH_LD(G12);
  G.c13 = KH_LD(G13); G.c22 = KH_LD(G22); G.c33 = KH_LD(G33);
  G.n00 = KH_LD(10 + G00); G.n01 = KH_LD(10 + G01); G.n02 = KH_LD(10 + G02);
  if (LEVEL == 1 || DIR == 1) G.n11 = KH_LD(10 + G11);
  if (LEVEL == 1 || DIR == 2) G.n22 = KH_LD(10 + G22);
  if (LEVEL == 1 || DIR == 3) G.n33 = KH_LD(10 + G33);
  if (LEVEL == 1) { G.n12 = KH_LD(10 + G12); G.n13 = KH_LD(10 + G13); G.n23 = KH_LD(10 + G23); }
  G.gdet = KH_LD(20); G.alpha = KH_LD(21);
#undef KH_LD
}

// g_ij a^i b^j pieces
template <bool FLAT>
__device__ __forceinline__ void lower3(const Geo& G, double a1, double a2, double a3, double& o1, double& o2, double& o3) {
  if (FLAT) { o1 = a1; o2 = a2; o3 = a3; return; }
  o1 = fma(G.c13, a3, fma(G.c12, a2, G.c11 * a1));
  o2 = fma(G.c22, a2, G.c12 * a1);
  o3 = fma(G.c33, a3, G.c13 * a1);
}
template <bool FLAT>
__device__ __forceinline__ double spatial_norm2(const Geo& G, double a, double b, double c) {
  double o1, o2, o3;
  lower3<FLAT>(G, a, b, c, o1, o2, o3);
  return fma(c, o3, fma(b, o2, a * o1));
}

// ---------------------------------------------------------------------------------------------
// Four-vectors of a primitive state (S1): ut^i is the velocity projected into the normal observer's frame,
//   u^t = gamma/alpha, u^i = ut^i - gamma alpha g^{ti};  b^t = B^i u_i,  b^i = (B^i + b^t u^i)/u^t.
// Since n_i = 0, u_i = g_ij ut^j exactly and q^2 = ut^i u_i.  gamma and 1/gamma come from one rsqrt.
// ---------------------------------------------------------------------------------------------
struct FourVec {
  double ucon[4], ucov[4], bcon[4], bcov[4], bsq;
  double x;       // 1 + q^2 = gamma^2
};

template <bool FLAT>
__device__ __forceinline__ void four_vectors(const Geo& G, double ialpha, const double P[KH_NP], FourVec& D) {
  const double v1 = P[U1], v2 = P[U2], v3 = P[U3];
  lower3<FLAT>(G, v1, v2, v3, D.ucov[1], D.ucov[2], D.ucov[3]);
  double qsq = fma(v3, D.ucov[3], fma(v2, D.ucov[2], v1 * D.ucov[1]));
  D.x = 1.0 + qsq;
  double rg = fast_rsqrt(D.x), gamma = D.x * rg;
  if (FLAT) {
    D.ucon[0] = gamma; D.ucon[1] = v1; D.ucon[2] = v2; D.ucon[3] = v3;
    D.ucov[0] = -gamma;
  } else {
    double ga = gamma * G.alpha;
    D.ucon[0] = gamma * ialpha;
    D.ucon[1] = fma(-ga, G.n01, v1);
    D.ucon[2] = fma(-ga, G.n02, v2);
    D.ucon[3] = v3;                                  // g^03 = 0
    D.ucov[0] = fma(G.c03, D.ucon[3], fma(G.c01, D.ucon[1], G.c00 * D.ucon[0]));   // g_02 = 0
  }
  D.bcon[0] = fma(P[B3], D.ucov[3], fma(P[B2], D.ucov[2], P[B1] * D.ucov[1]));
  double iut = FLAT ? rg : G.alpha * rg;             // 1/u^t = alpha/gamma
  D.bcon[1] = fma(D.bcon[0], D.ucon[1], P[B1]) * iut;
  D.bcon[2] = fma(D.bcon[0], D.ucon[2], P[B2]) * iut;
  D.bcon[3] = fma(D.bcon[0], D.ucon[3], P[B3]) * iut;
  if (FLAT) {
    D.bcov[0] = -D.bcon[0]; D.bcov[1] = D.bcon[1]; D.bcov[2] = D.bcon[2]; D.bcov[3] = D.bcon[3];
  } else {
    D.bcov[0] = fma(G.c03, D.bcon[3], fma(G.c01, D.bcon[1], G.c00 * D.bcon[0]));
    D.bcov[1] = fma(G.c13, D.bcon[3], fma(G.c12, D.bcon[2], fma(G.c11, D.bcon[1], G.c01 * D.bcon[0])));
    D.bcov[2] = fma(G.c22, D.bcon[2], G.c12 * D.bcon[1]);
    D.bcov[3] = fma(G.c33, D.bcon[3], fma(G.c13, D.bcon[1], G.c03 * D.bcon[0]));
  }
  D.bsq = fma(D.bcon[3], D.bcov[3], fma(D.bcon[2], D.bcov[2], fma(D.bcon[1], D.bcov[1], D.bcon[0] * D.bcov[0])));
}

// Row `dir` of the flux matrix WITHOUT the sqrt(-g) factor (applied once per face / zone by the caller):
//   dir = 0: U/sqrt(-g) = (rho u^t, T^t_t + rho u^t, T^t_i, B^i)          (S8)
//   dir > 0: F^dir/sqrt(-g) = (rho u^d, T^d_t + rho u^d, T^d_i, b^i u^d - b^d u^i), F^d[B^d] = 0
// with T^mu_nu = (w + b^2) u^mu u_nu + (p + b^2/2) delta^mu_nu - b^mu b_nu  [eq. 1.1, P:347]; eu[nu] = (w+b^2) u_nu.
__device__ __forceinline__ void flux_row(const double P[KH_NP], const FourVec& D, const double eu[4], double ptot, int dir,
                                         double F[KH_NP]) {
  const double ud = D.ucon[dir], bd = D.bcon[dir];
  double T0 = fma(ud, eu[0], -bd * D.bcov[0]);
  double T1 = fma(ud, eu[1], -bd * D.bcov[1]);
  double T2 = fma(ud, eu[2], -bd * D.bcov[2]);
  double T3 = fma(ud, eu[3], -bd * D.bcov[3]);
  if (dir == 0) T0 += ptot;
  if (dir == 1) T1 += ptot;
  if (dir == 2) T2 += ptot;
  if (dir == 3) T3 += ptot;
  F[RHO] = P[RHO] * ud;
  F[UU] = fma(P[RHO], ud, T0);
  F[U1] = T1; F[U2] = T2; F[U3] = T3;
  if (dir == 0) {
    F[B1] = P[B1]; F[B2] = P[B2]; F[B3] = P[B3];
  } else {
#pragma unroll
    for (int i = 1; i < 4; i++) F[B1 + i - 1] = (i == dir) ? 0.0 : fma(D.bcon[i], ud, -bd * D.ucon[i]);
  }
}

// S9: fast-magnetosonic bound.  c_m^2 = c_s^2 + v_A^2 - c_s^2 v_A^2 = (b^2 + Gamma (Gamma-1) u) / (rho + Gamma u + b^2)
// (one quotient).  The characteristic speeds are the roots of A v^2 - 2 Bh v + C = 0; LLF and the CFL rule
// only need max(|v+|, |v-|) = (|Bh| + sqrt(Bh^2 - A C)) / A (A > 0), and Bh^2 - A C reduces algebraically to
//   c_m^2 [ (1 - c_m^2)(u^t^2 g^dd - 2 u^t u^d g^td + u^d^2 g^tt) + c_m^2 (g^td^2 - g^tt g^dd) ]
// (the (u^d u^t)^2 terms cancel identically: well conditioned in cold zones).  k2 = g^td^2 - g^tt g^dd.
template <bool FLAT>
__device__ __forceinline__ double cfast(const FourVec& D, double ee, double gg1u, double gtt, double gtd, double gdd, double k2,
                                        int dir) {
  double cms2 = (D.bsq + gg1u) * fast_rcp(ee);
  // clamp to [0, 1] (NaN -> 0).  A double compare costs two fp64-pipe slots; the high word decides on the integer
  // pipe: 0 <= cms2 <= 1 <=> hi word (unsigned) <= hi(1.0) -- only the rare out-of-range case takes the branch
  if ((unsigned)__double2hiint(cms2) > 0x3ff00000u) cms2 = (cms2 > 1.0) ? 1.0 : 0.0;
  const double ut = D.ucon[0], ud = D.ucon[dir];
  double ut2 = ut * ut, udut = ud * ut, ud2 = ud * ud;
  double A, Bh, inner;
  if (FLAT) {
    A = fma(-(ut2 - 1.0), cms2, ut2);
    Bh = fma(-udut, cms2, udut);
    inner = fma(1.0 - cms2, ut2 - ud2, cms2);
  } else {
    A = fma(-(gtt + ut2), cms2, ut2);
    Bh = fma(-(gtd + udut), cms2, udut);
    double q = fma(ud2, gtt, fma(-2.0 * udut, gtd, ut2 * gdd));
    inner = fma(1.0 - cms2, q, cms2 * k2);
  }
  // floor the discriminant at ~1e-200 (also maps negative values and NaN to the floor; its root, 1e-100, is
  // invisible): one unsigned range test on the high word instead of an fp64 max
  double disc = cms2 * inner;
  if ((unsigned)(__double2hiint(disc) - 0x16687e93) > (0x7fefffffu - 0x16687e93u)) disc = 1e-200;
  return (fabs(Bh) + fast_sqrt(disc)) * fast_rcp(A);
}

// What the LLF flux of a face needs from one reconstructed state.  The flux is assembled as
//   F = sqrt(-g)/2 [ (F_L + c U_L) + (F_R - c U_R) ],   c = c_top (S14),
// and F^d + s U has the same structure as one flux-matrix row with u^d -> u^d + s u^t and b^d -> b^d + s b^t:
//   rho (u^d + s u^t),  (u^d + s u^t)(w + b^2) u_nu - (b^d + s b^t) b_nu + ptot (delta^d_nu + s delta^t_nu),
//   b^i (u^d + s u^t) - (b^d + s b^t) u^i      [since B^i = b^i u^t - b^t u^i],
// so one row per state is evaluated instead of two rows and a difference (30 fp64 instructions fewer per face).
// c is known only after both states' speeds, so the state is kept in this compact form meanwhile.
struct StateQ {
  double rho, ptot, ut, ud, bt, bd;
  double ee;                  // w + b^2
  double ucov[4], bcov[4];
  double uI, uJ, bI, bJ;      // the two spatial directions other than d
};

template <int DIR, bool FLAT>
__device__ __forceinline__ void state_terms(const Geo& G, double ialpha, double gtd, double gdd, double k2, const double P[KH_NP],
                                            double gam, double gm1, StateQ& S, double& c) {
  FourVec D;
  four_vectors<FLAT>(G, ialpha, P, D);
  double pg = gm1 * P[UU];
  double ee = fma(gam, P[UU], P[RHO]) + D.bsq;      // w + b^2 = rho + Gamma u + b^2
  S.rho = P[RHO];
  S.ptot = fma(0.5, D.bsq, pg);
  S.ut = D.ucon[0]; S.ud = D.ucon[DIR]; S.bt = D.bcon[0]; S.bd = D.bcon[DIR];
  S.ee = ee;
#pragma unroll
  for (int m = 0; m < 4; m++) { S.ucov[m] = D.ucov[m]; S.bcov[m] = D.bcov[m]; }
  constexpr int I = (DIR == 1) ? 2 : 1, J = (DIR == 3) ? 2 : 3;
  S.uI = D.ucon[I]; S.uJ = D.ucon[J]; S.bI = D.bcon[I]; S.bJ = D.bcon[J];
  c = cfast<FLAT>(D, ee, gam * pg, G.n00, gtd, gdd, k2, DIR);
}

// Gs = (F^d + s U) / sqrt(-g) of the state (s = +c for the left state, -c for the right one); Gs[B^d] is not formed.
template <int DIR>
__device__ __forceinline__ void llf_row(const StateQ& S, double s, double Gs[KH_NP]) {
  const double us = fma(s, S.ut, S.ud), bs = fma(s, S.bt, S.bd);
  const double ue = us * S.ee;        // (w + b^2) (u^d + s u^t): one product per state instead of the four (w + b^2) u_nu
  double T0 = fma(ue, S.ucov[0], fma(s, S.ptot, -bs * S.bcov[0]));
  double T1 = fma(ue, S.ucov[1], -bs * S.bcov[1]);
  double T2 = fma(ue, S.ucov[2], -bs * S.bcov[2]);
  double T3 = fma(ue, S.ucov[3], -bs * S.bcov[3]);
  if (DIR == 1) T1 += S.ptot;
  if (DIR == 2) T2 += S.ptot;
  if (DIR == 3) T3 += S.ptot;
  // not contractable into the caller's sum of the two states: with mirror-symmetric states the two mass-flux terms are
  // exact negatives and must cancel to an exact zero (an FMA would leave the rounding error of one product), which the
  // contact-upwinded EMFs read as "no flow through this face"
  Gs[RHO] = __dmul_rn(S.rho, us);
  Gs[UU] = fma(S.rho, us, T0);
  Gs[U1] = T1; Gs[U2] = T2; Gs[U3] = T3;
  constexpr int I = (DIR == 1) ? 2 : 1, J = (DIR == 3) ? 2 : 3;
  Gs[B1 + DIR - 1] = 0.0;
  Gs[B1 + I - 1] = fma(S.bI, us, -bs * S.uI);
  Gs[B1 + J - 1] = fma(S.bJ, us, -bs * S.uJ);
}

// ---------------------------------------------------------------------------------------------
// Reconstruction, zone-centred: both face values of the zone centred on x3 in one pass.
// qm = value at the lower face (the RIGHT state of face i-1/2), qp = value at the upper face (the LEFT
// state of face i+1/2).
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
__device__ __forceinline__ void mc_zone(double x2, double x3, double x4, double& qm, double& qp) {
  double h = 0.5 * mc_slope(x2, x3, x4);
  qm = x3 - h;
  qp = x3 + h;
}

// S12: Jiang-Shu WENO5, eps = 1e-26, written on the differences D_k = x_{k+1} - x_k:
//   4 (beta_k + eps) = (13/3) d_k^2 + e_k^2 + 4 eps      (the common factor 4 cancels in the weights)
//   weights d_k / (beta_k + eps)^2 over the common denominator: (1, 6, 3) x products of the other two squares
//   candidate values as offsets from x3, times 6:  upper face (5 D2 - 2 D1, D2 + 2 D3, 4 D3 - D4),
//   lower face the mirror image (2 D4 - 5 D3, -(D3 + 2 D2), D1 - 4 D2); the smoothness indicators are shared.
// 54 fp64 instructions per variable for both faces.
__device__ __forceinline__ void weno5_zone(double x1, double x2, double x3, double x4, double x5, double& qm, double& qp) {
  const double c = 4.0e-26, k13 = 13.0 / 3.0;
  double D1 = x2 - x1, D2 = x3 - x2, D3 = x4 - x3, D4 = x5 - x4;
  double d1 = D2 - D1, d2 = D3 - D2, d3 = D4 - D3;
  double e1 = fma(3.0, D2, -D1), e2 = D2 + D3, e3 = fma(-3.0, D3, D4);
  double b1 = fma(k13 * d1, d1, fma(e1, e1, c));
  double b2 = fma(k13 * d2, d2, fma(e2, e2, c));
  double b3 = fma(k13 * d3, d3, fma(e3, e3, c));
  double a1 = b1 * b1, a2 = b2 * b2, a3 = b3 * b3;
  double p23 = a2 * a3, p13 = 6.0 * (a1 * a3), p12 = a1 * a2;
  {
    double w3 = 3.0 * p12;
    double V1 = fma(2.0, e1, -D2), V2 = fma(2.0, D3, D2), V3 = fma(4.0, D3, -D4);      // 5 D2 - 2 D1 = 2 e1 - D2
    double N = fma(w3, V3, fma(p13, V2, p23 * V1));
    double S = p23 + p13 + w3;
    qp = fma(N * fast_rcp(S), 1.0 / 6.0, x3);
  }
  {
    double m3 = 3.0 * p23;
    double M1 = fma(2.0, e3, D3), M2 = fma(2.0, D2, D3), M3 = fma(-4.0, D2, D1);        // 2 D4 - 5 D3 = 2 e3 + D3
    double N = fma(m3, M3, fma(-p13, M2, p12 * M1));
    double S = p12 + p13 + m3;
    qm = fma(N * fast_rcp(S), 1.0 / 6.0, x3);
  }
}
template <int RECON>
__device__ __forceinline__ void recon_zone(const double* __restrict__ A, long st, double& qm, double& qp) {
  if (RECON == 0) mc_zone(A[-st], A[0], A[st], qm, qp);
  else weno5_zone(A[-2 * st], A[-st], A[0], A[st], A[2 * st], qm, qp);
}

// ---------------------------------------------------------------------------------------------
// Floors and ceilings in the fluid frame (S18).  rho_g, u_g: tabulated geometric floors.
// ---------------------------------------------------------------------------------------------
struct FloorPar {
  double inv_bsq_over_rho_max, inv_bsq_over_u_max, u_over_rho_max, gamma_max;   // inverses formed once on the host
};

// Limits on (rho, u) and the Lorentz-factor ceiling given b^2 and gamma of the state; returns the fflag bits and
// the factor (1 = none) by which the caller scales ut^i.
__device__ __forceinline__ int floor_limits(const FloorPar& fp, double rho_g, double u_g, double bsq, double gamma, double& rho,
                                            double& u, double& vfac, double inj[2]) {
  int flag = 0;
  double rho_b = bsq * fp.inv_bsq_over_rho_max, u_b = bsq * fp.inv_bsq_over_u_max;
  double rho_fl = rho_b > rho_g ? rho_b : rho_g;
  double u_fl = u_b > u_g ? u_b : u_g;
  inj[0] = inj[1] = 0.0;                      // floor material (rho_inj, u_inj): used by the normal-frame injection only
  if (rho < rho_fl) { inj[0] = rho_fl - rho; rho = rho_fl; flag |= (rho_b > rho_g) ? 2 : 1; }
  if (u < u_fl) { inj[1] = u_fl - u; u = u_fl; flag |= (u_b > u_g) ? 8 : 4; }
  double ucap = fp.u_over_rho_max * rho;
  if (u > ucap) { u = ucap; flag |= 16; }
  vfac = 1.0;
  if (gamma > fp.gamma_max) {      // rare: IEEE sqrt and division
    vfac = sqrt((fp.gamma_max * fp.gamma_max - 1.0) / (gamma * gamma - 1.0));
    flag |= 32;
  }
  return flag;
}

// Drift-frame injection (S26): after (rho, u) were moved to (rho', u'), the
// normal observer's velocity v = ut/gamma keeps its part perpendicular to B (the E x B drift) and changes its part
// along B so that the momentum along the field w gamma^2 v_par (w = rho + Gamma u) is conserved:
//   A = w gamma^2 v_par / w',  v_par' = 2 A (1 - v_perp^2) / (1 + sqrt(1 + 4 A^2 (1 - v_perp^2))),  gamma'^2 = 1/(1 - v_perp^2 - v_par'^2).
// B = 0: the velocity is kept.  Acts on the primitive velocities ut^i in place.
template <bool FLAT>
__device__ __forceinline__ void drift_frame_velocity(const Geo& G, double gam, double rho_old, double u_old, double rho_new, double u_new,
                                                     double& ut1, double& ut2, double& ut3, double b1, double b2, double b3) {
  double l1, l2, l3;
  lower3<FLAT>(G, b1, b2, b3, l1, l2, l3);                               // B_i
  const double Bsq = fma(b3, l3, fma(b2, l2, b1 * l1));
  if (!(Bsq > 1e-12 * fma(gam, u_new, rho_new))) return;               // no field direction to speak of (S26): velocity kept
  const double uB = fma(ut3, l3, fma(ut2, l2, ut1 * l1));                // ut^i B_i
  const double qsq = spatial_norm2<FLAT>(G, ut1, ut2, ut3);
  const double gsq = 1.0 + qsq, gamma = sqrt(gsq), iB = 1.0 / sqrt(Bsq), ig = 1.0 / gamma;
  const double vpar = uB * ig * iB;
  double omp = 1.0 - (qsq / gsq - vpar * vpar);                          // 1 - v_perp^2
  if (omp > 1.0) omp = 1.0;
  const double A = (fma(gam, u_old, rho_old) * gsq * vpar) / fma(gam, u_new, rho_new);
  const double vpn = 2.0 * A * omp / (1.0 + sqrt(fma(4.0 * A * A, omp, 1.0)));
  const double gn = 1.0 / sqrt(fma(-vpn, vpn, omp));
  const double dv = (vpn - vpar) * iB;                                   // v' = v + (v_par' - v_par) B/|B|
  ut1 = gn * fma(dv, b1, ut1 * ig);
  ut2 = gn * fma(dv, b2, ut2 * ig);
  ut3 = gn * fma(dv, b3, ut3 * ig);
}

// Limits, injection frame and Lorentz-factor ceiling on a state whose b^2 and gamma are known.  frame 0: fluid frame
// (velocity untouched), 1: drift frame (the ceiling then acts on the adjusted velocity).
template <bool FLAT>
__device__ __forceinline__ int floors_in_frame(const Geo& G, const FloorPar& fp, int frame, double gam, double rho_g, double u_g, double bsq,
                                               double gamma, double& rho, double& u, double& ut1, double& ut2, double& ut3, double b1,
                                               double b2, double b3, double inj[2]) {
  double vfac;
  if (frame != 1) {                            // fluid frame; the normal frame starts from the same provisional result
    const int flag = floor_limits(fp, rho_g, u_g, bsq, gamma, rho, u, vfac, inj);
    if (flag & 32) { ut1 *= vfac; ut2 *= vfac; ut3 *= vfac; }
    return flag;
  }
  const double rho_old = rho, u_old = u;
  int flag = floor_limits(fp, rho_g, u_g, bsq, 1.0, rho, u, vfac, inj);  // limits only (gamma = 1 never trips the ceiling)
  if (flag != 0) {
    drift_frame_velocity<FLAT>(G, gam, rho_old, u_old, rho, u, ut1, ut2, ut3, b1, b2, b3);
    gamma = sqrt(1.0 + spatial_norm2<FLAT>(G, ut1, ut2, ut3));
  }
  if (gamma > fp.gamma_max) {
    vfac = sqrt((fp.gamma_max * fp.gamma_max - 1.0) / (gamma * gamma - 1.0));
    ut1 *= vfac; ut2 *= vfac; ut3 *= vfac;
    flag |= 32;
  }
  return flag;
}

// Floors of a primitive state (fix-up path): b^2 = (g_ij B^i B^j + (b^t)^2)/(u^t)^2 with b^t = B^i u_i.
template <bool FLAT>
__device__ __forceinline__ int apply_floors(const Geo& G, const FloorPar& fp, int frame, double gam, double rho_g, double u_g, double P[KH_NP],
                                            double inj[2]) {
  double c1, c2, c3;
  lower3<FLAT>(G, P[U1], P[U2], P[U3], c1, c2, c3);
  double qsq = fma(P[U3], c3, fma(P[U2], c2, P[U1] * c1));
  double bt = fma(P[B3], c3, fma(P[B2], c2, P[B1] * c1));
  double BB = spatial_norm2<FLAT>(G, P[B1], P[B2], P[B3]);
  double bsq = fma(bt, bt, BB) / (-(1.0 + qsq) * G.n00);      // 1/(u^t)^2 = alpha^2/gamma^2 = -1/(gamma^2 g^tt)
  return floors_in_frame<FLAT>(G, fp, frame, gam, rho_g, u_g, bsq, sqrt(1.0 + qsq), P[RHO], P[UU], P[U1], P[U2], P[U3], P[B1], P[B2], P[B3], inj);
}

// ---------------------------------------------------------------------------------------------
// 1D_W inversion (ref [37]) in the W' = W - D variable (S16), fused with the floors (S18).
// Input Uh = U / sqrt(-g).  W0 = guess (rho + Gamma u)(1 + q^2) of the guess primitives.
// Returns the pflag; on success writes the five hydro primitives to Pout (floors applied, bits in fflag); B is
// always written; on failure the caller keeps the guess primitives (S16).
// Per Newton step: one reciprocal serves 1/W and 1/(W+B^2), one rsqrt gives gamma and gamma^2.
// After convergence b^2 = B^2 (1 - v^2) + (Q.B)^2 / W^2 and gamma are known from the conserved side, so the
// floors need no second pass through the four-vectors.
// ---------------------------------------------------------------------------------------------
template <bool FLAT>
__device__ __forceinline__ int u_to_p_floors(const Geo& G, const double Uh[KH_NP], double W0, double gam, const FloorPar& fp, int frame,
                                             double rho_g, double u_g, double Pout[KH_NP], int& fflag, double inj[2]) {
  fflag = 0;
  Pout[B1] = Uh[B1]; Pout[B2] = Uh[B2]; Pout[B3] = Uh[B3];
  bool fin = true;
#pragma unroll
  for (int v = 0; v < KH_NP; v++) fin = fin && isfinite(Uh[v]);
  if (!fin || !(Uh[RHO] > 0.0)) return 1;

  const double alpha = G.alpha;
  const double D = alpha * Uh[RHO];
  const double Bc1 = alpha * Uh[B1], Bc2 = alpha * Uh[B2], Bc3 = alpha * Uh[B3];        // script-B^i = alpha B^i
  const double Qc0 = alpha * (Uh[UU] - Uh[RHO]), Qc1 = alpha * Uh[U1], Qc2 = alpha * Uh[U2], Qc3 = alpha * Uh[U3];
  double Qdotn, Qt1, Qt2, Qt3;
  if (FLAT) {
    Qdotn = Qc0; Qt1 = Qc1; Qt2 = Qc2; Qt3 = Qc3;
  } else {
    double Q0 = fma(G.n02, Qc2, fma(G.n01, Qc1, G.n00 * Qc0));                           // g^03 = 0
    double Q1 = fma(G.n13, Qc3, fma(G.n12, Qc2, fma(G.n11, Qc1, G.n01 * Qc0)));
    double Q2 = fma(G.n23, Qc3, fma(G.n22, Qc2, fma(G.n12, Qc1, G.n02 * Qc0)));
    double Q3 = fma(G.n33, Qc3, fma(G.n23, Qc2, G.n13 * Qc1));
    Qdotn = -alpha * Q0;
    double qa = -alpha * Qdotn;                       // Qt^i = Q^i + (Q.n) n^i, n^i = -alpha g^{ti}
    Qt1 = fma(qa, G.n01, Q1); Qt2 = fma(qa, G.n02, Q2); Qt3 = Q3;
  }
  const double Bsq = spatial_norm2<FLAT>(G, Bc1, Bc2, Bc3);
  const double QdotB = fma(Qc3, Bc3, fma(Qc2, Bc2, Qc1 * Bc1));
  const double QdotBsq = QdotB * QdotB;
  const double Ep = -Qdotn - D;
  // Qt^2 as the spatial norm of the projected vector (its time component vanishes): no cancellation (S16)
  const double Qtsq = spatial_norm2<FLAT>(G, Qt1, Qt2, Qt3);

  double W = W0;
  if (!(W > 0.0) || !isfinite(W)) W = D;
#pragma unroll 1
  for (int it = 0; it < 30; it++) {                   // v^2(W0) < 1  <=>  numerator < denominator
    double WB = Bsq + W, den = (WB * WB) * (W * W);
    double num = fma(Qtsq * W, W, QdotBsq * fma(2.0, W, Bsq));
    if (num < den) break;
    W *= 10.0;
  }
  double Wp = W - D;
  const double k = (gam - 1.0) / gam, hB = 0.5 * Bsq, hQ = 0.5 * QdotBsq, hD = 0.5 * D, Bsq2 = Bsq * Bsq;
  const double WpmE0 = -Ep;

  bool conv = false;
#pragma unroll 1
  for (int it = 0; it < 20; it++) {
    W = Wp + D;
    double WB = W + Bsq;
    double r = fast_rcp(W * WB), iW = r * WB, iWB = r * W;      // iW iWB = r
    double iW2 = iW * iW, s2 = iW2 * (iWB * iWB);
    double QW = Qtsq * W;
    double v2 = fma(QW, W, QdotBsq * fma(2.0, W, Bsq)) * s2;
    v2 = fmin(fmax(v2, 0.0), 1.0 - 1e-12);
    double omv = 1.0 - v2;
    double g = fast_rsqrt(omv), gsq = g * g;
    double t = (D * v2) * (gsq * fast_rcp(1.0 + g));
    double p = k * ((Wp - t) * omv);
    double f = fma(-hQ, iW2, fma(hB, v2, hB)) + ((Wp + WpmE0) - p);
    double dv2 = -2.0 * (fma(QW, W * W, QdotBsq * fma(3.0 * W, WB, Bsq2)) * (s2 * r));
    double dp = k * fma(-fma(-hD, g, W), dv2, omv);
    double df = fma(hB, dv2, fma(QdotBsq, iW2 * iW, 1.0 - dp));
    double Wold = W;
    double Wpn = fma(-f, fast_rcp(df), Wp);
    if (!(Wpn + D > 0.0)) Wpn = 0.5 * Wold - D;       // new W <= 0: halve the old W instead
    double dW = Wpn - Wp;
    Wp = Wpn;
    if (fabs(dW) <= 1e-12 * (Wp + D)) { conv = true; break; }
  }
  if (!conv) return 2;

  W = Wp + D;
  if (!(W > 0.0)) return 3;
  double WB = W + Bsq;
  double r = fast_rcp(W * WB), iW = r * WB, iWB = r * W;
  double v2 = fma(Qtsq * W, W, QdotBsq * fma(2.0, W, Bsq)) * (r * r);
  if (!(v2 >= 0.0) || !(v2 < 1.0)) return 3;
  double omv = 1.0 - v2;
  double g = fast_rsqrt(omv), gsq = g * g;
  double rho = D * (omv * g);                          // D / gamma
  double u = ((Wp - (D * v2) * (gsq * fast_rcp(1.0 + g))) * omv) * (1.0 / gam);
  double fac = g * iWB, qbw = QdotB * iW;
  double ut1 = fac * fma(qbw, Bc1, Qt1);
  double ut2 = fac * fma(qbw, Bc2, Qt2);
  double ut3 = fac * fma(qbw, Bc3, Qt3);
  if (!isfinite(rho) || !isfinite(u) || !isfinite(ut1) || !isfinite(ut2) || !isfinite(ut3)) return 7;
  bool badrho = !(rho > 0.0), badu = (u < 0.0);
  if (badrho && badu) return 6;
  if (badrho) return 4;
  if (badu) return 5;
  // floors (S18): b^2 and gamma of the recovered state from the conserved side
  double bsq = fma(Bsq, omv, QdotBsq * (iW * iW));
  fflag = floors_in_frame<FLAT>(G, fp, frame, gam, rho_g, u_g, bsq, g, rho, u, ut1, ut2, ut3, Uh[B1], Uh[B2], Uh[B3], inj);
  Pout[RHO] = rho; Pout[UU] = u; Pout[U1] = ut1; Pout[U2] = ut2; Pout[U3] = ut3;
  return 0;
}

// ---------------------------------------------------------------------------------------------
// Second inverter (reading S24): the bracketed root find of Kastaun, Kalinani &
// Ciolfi in the unknown mu = 1/(W h), fused with the floors like the 1D_W path and behind the same flags.
// With D, tau, S_i, B^i of the normal observer:  q = tau/D, r^2 = S^2/D^2, b^2 = B^2/D, (r.b)^2 = (S.B)^2/D^3,
//   x = 1/(1 + mu b^2),  rbar^2 = x (r^2 x + mu (1 + x)(r.b)^2),  qbar = q - b^2/2 - mu^2 x^2 (b^2 r^2 - (r.b)^2)/2,
//   f(mu) = mu - 1/(nu + rbar^2 mu),  nu = max((1 + Gamma eps)/W, (1 + a)(1 + qbar - mu rbar^2)),  a = (Gamma-1) eps/(1+eps),
//   v^2 = min(mu^2 rbar^2, v0^2), W = (1 - v^2)^(-1/2), eps = W (qbar - mu rbar^2) + v^2 W^2/(1 + W) (clamped at 0 in f),
// bracket (0, mu+], mu+ = 1 or the root of mu sqrt(1 + rbar^2) - 1; Illinois regula falsi (bisection after 40 evaluations) to a
// bracket of 4e-16.
// ---------------------------------------------------------------------------------------------
struct KastaunC {
  double q, rsq, bsq, rbsq, brperp, v0sq, gam;
};
__device__ __forceinline__ void kastaun_aux(const KastaunC& c, double mu, double& x, double& rbarsq, double& qbar) {
  x = fast_rcp(fma(mu, c.bsq, 1.0));
  rbarsq = x * fma(c.rsq, x, mu * ((1.0 + x) * c.rbsq));
  const double mx = mu * x;
  qbar = fma(-0.5 * (mx * mx), c.brperp, fma(-0.5, c.bsq, c.q));
}
__device__ __forceinline__ double kastaun_f(const KastaunC& c, double mu, double& vsq_raw, double& W, double& eps_raw, double& omv) {
  double x, rbarsq, qbar;
  kastaun_aux(c, mu, x, rbarsq, qbar);
  const double mr = mu * rbarsq;
  vsq_raw = mu * mr;
  const double vsq = vsq_raw < c.v0sq ? vsq_raw : c.v0sq;
  omv = 1.0 - vsq;
  W = fast_rsqrt(omv);
  const double e0 = qbar - mr;
  eps_raw = fma(W, e0, (vsq * (W * W)) * fast_rcp(1.0 + W));
  const double eps = eps_raw > 0.0 ? eps_raw : 0.0;
  const double ope = 1.0 + eps;
  const double nuA = fma(c.gam, eps, 1.0) * (omv * W);               // (1 + a)(1 + eps)/W, 1/W = (1 - v^2) W
  const double nuB = fma(c.gam, eps, 1.0) * fast_rcp(ope) * (1.0 + e0);
  const double nu = nuA > nuB ? nuA : nuB;
  return mu - fast_rcp(fma(rbarsq, mu, nu));
}
__device__ __forceinline__ double kastaun_fa(const KastaunC& c, double mu) {
  double x, rbarsq, qbar;
  kastaun_aux(c, mu, x, rbarsq, qbar);
  return fma(mu, fast_sqrt(1.0 + rbarsq), -1.0);
}
// Illinois regula falsi on [a, b], fn(a) < 0 <= fn(b); AUX selects the function.  false: no convergence in 100 evaluations.
template <bool AUX>
__device__ __forceinline__ bool kastaun_root(const KastaunC& c, double a, double fa, double b, double fb, double& lo, double& hi) {
  int side = 0;
#pragma unroll 1
  for (int it = 0; it < 100; it++) {
    if (!(b - a > 4e-16 * b)) { lo = a; hi = b; return true; }
    double m = (it < 40) ? fma(-fb, (b - a) / (fb - fa), b) : 0.5 * (a + b);   // after 40 evaluations: plain bisection
    if (!(m > a && m < b)) m = 0.5 * (a + b);
    if (!(m > a && m < b)) { lo = a; hi = b; return true; }                    // a and b are neighbouring numbers
    double t0, t1, t2, t3;
    const double fm = AUX ? kastaun_fa(c, m) : kastaun_f(c, m, t0, t1, t2, t3);
    if (fm == 0.0) { lo = hi = m; return true; }
    if (fm > 0.0) { b = m; fb = fm; if (side == 1) fa *= 0.5; side = 1; }
    else if (fm < 0.0) { a = m; fa = fm; if (side == -1) fb *= 0.5; side = -1; }
    else return false;
  }
  return false;
}

template <bool FLAT>
__device__ __forceinline__ int u_to_p_kastaun_floors(const Geo& G, const double Uh[KH_NP], double mu0, double gam, const FloorPar& fp, int frame,
                                                     double rho_g, double u_g, double Pout[KH_NP], int& fflag, double inj[2]) {
  fflag = 0;
  Pout[B1] = Uh[B1]; Pout[B2] = Uh[B2]; Pout[B3] = Uh[B3];
  bool fin = true;
#pragma unroll
  for (int v = 0; v < KH_NP; v++) fin = fin && isfinite(Uh[v]);
  if (!fin || !(Uh[RHO] > 0.0)) return 1;
  const double alpha = G.alpha;
  const double D = alpha * Uh[RHO];
  const double Bc1 = alpha * Uh[B1], Bc2 = alpha * Uh[B2], Bc3 = alpha * Uh[B3];
  const double Qc0 = alpha * (Uh[UU] - Uh[RHO]), Qc1 = alpha * Uh[U1], Qc2 = alpha * Uh[U2], Qc3 = alpha * Uh[U3];
  double Qdotn, S1, S2, S3;                             // S^i = gamma^{ij} S_j
  if (FLAT) {
    Qdotn = Qc0; S1 = Qc1; S2 = Qc2; S3 = Qc3;
  } else {
    double Q0 = fma(G.n02, Qc2, fma(G.n01, Qc1, G.n00 * Qc0));
    double Q1 = fma(G.n13, Qc3, fma(G.n12, Qc2, fma(G.n11, Qc1, G.n01 * Qc0)));
    double Q2 = fma(G.n23, Qc3, fma(G.n22, Qc2, fma(G.n12, Qc1, G.n02 * Qc0)));
    double Q3 = fma(G.n33, Qc3, fma(G.n23, Qc2, G.n13 * Qc1));
    Qdotn = -alpha * Q0;
    double qa = -alpha * Qdotn;
    S1 = fma(qa, G.n01, Q1); S2 = fma(qa, G.n02, Q2); S3 = Q3;
  }
  const double Bsq = spatial_norm2<FLAT>(G, Bc1, Bc2, Bc3);
  const double SdotB = fma(Qc3, Bc3, fma(Qc2, Bc2, Qc1 * Bc1));
  const double Ssq = spatial_norm2<FLAT>(G, S1, S2, S3);
  const double tau = -Qdotn - D;
  const double iD = 1.0 / D;
  KastaunC c;
  c.gam = gam;
  c.q = tau * iD;
  c.rsq = Ssq * (iD * iD);
  c.bsq = Bsq * iD;
  c.rbsq = (SdotB * SdotB) * (iD * iD * iD);
  c.brperp = fma(c.bsq, c.rsq, -c.rbsq);
  if (c.brperp < 0.0) c.brperp = 0.0;
  c.v0sq = c.rsq / (1.0 + c.rsq);

  double mu_hi = 1.0, lo, hi;
  if (!(c.rsq < 1.0)) {
    const double fa1 = kastaun_fa(c, 1.0);
    if (fa1 > 0.0) {
      if (!kastaun_root<true>(c, 0.0, -1.0, 1.0, fa1, lo, hi)) return 2;
      mu_hi = hi;
    }
  }
  double vr, W, er, omv;
  double mu;
  // A bracket around the guess first (mu0 = 1/(W h) of the guess primitives): the master function has exactly one root in
  // (0, mu_+] and is negative below it, positive above, so f(a) < 0 < f(b) with 0 < a < b <= mu_+ encloses THE root and the
  // end-point evaluations f(0), f(mu_+) (with their flag semantics) are implied.  The root find converges to the same
  // 4e-16 bracket from any start (S24): the result does not depend on the guess; only the number of evaluations does.
  bool bracketed = false;
  if (mu0 > 0.0 && mu0 < mu_hi) {
    double a = mu0 * (1.0 - 4e-3), b = mu0 * (1.0 + 4e-3);
    if (b > mu_hi) b = mu_hi;
    const double fa = kastaun_f(c, a, vr, W, er, omv), fb = kastaun_f(c, b, vr, W, er, omv);
    if (fa < 0.0 && fb > 0.0) {
      if (!kastaun_root<false>(c, a, fa, b, fb, lo, hi)) return 2;
      mu = 0.5 * (lo + hi);
      bracketed = true;
    }
  }
  if (!bracketed) {
    const double f0 = kastaun_f(c, 0.0, vr, W, er, omv);
    const double f1 = kastaun_f(c, mu_hi, vr, W, er, omv);
    if (!(f0 < 0.0) || !isfinite(f1)) return 2;
    if (f1 <= 0.0) mu = mu_hi;
    else {
      if (!kastaun_root<false>(c, 0.0, f0, mu_hi, f1, lo, hi)) return 2;
      mu = 0.5 * (lo + hi);
    }
  }
  double vsq_raw, eps_raw;
  kastaun_f(c, mu, vsq_raw, W, eps_raw, omv);
  if (!(vsq_raw <= c.v0sq * (1.0 + 1e-12))) return 3;
  const double x = 1.0 / fma(mu, c.bsq, 1.0);
  double rho = D * (omv * W);                           // D / W
  double u = rho * eps_raw;
  const double msb = mu * (SdotB * iD);                 // B_i v^i = mu (S.B)/D
  const double fac = W * mu * x * iD;
  double ut1 = fac * fma(msb, Bc1, S1);
  double ut2 = fac * fma(msb, Bc2, S2);
  double ut3 = fac * fma(msb, Bc3, S3);
  if (!isfinite(rho) || !isfinite(u) || !isfinite(ut1) || !isfinite(ut2) || !isfinite(ut3)) return 7;
  if (eps_raw < 0.0) return 5;
  // floors (S18): comoving b^2 = B^2 (1 - v^2) + (B_i v^i)^2 and the Lorentz factor W
  const double bsq = fma(Bsq, omv, msb * msb);
  fflag = floors_in_frame<FLAT>(G, fp, frame, gam, rho_g, u_g, bsq, W, rho, u, ut1, ut2, ut3, Uh[B1], Uh[B2], Uh[B3], inj);
  Pout[RHO] = rho; Pout[UU] = u; Pout[U1] = ut1; Pout[U2] = ut2; Pout[U3] = ut3;
  return 0;
}

// ---------------------------------------------------------------------------------------------
// Inversion + floors with the injection frame resolved.  INVERTER: 0 1D_W, 1 Kastaun.  W0: the guess -- for 1D_W
// W0 = (rho + Gamma u) gamma^2 of the guess primitives, for Kastaun mu0 = 1/(W h) = rho / ((rho + Gamma u) gamma) (<= 0: none).  Frame 2 (normal observer, S27):
// the floor material enters as conserved variables of a gas at rest for the normal observer,
//   U_add/sqrt(-g) = (rho_inj/alpha, -(rho_inj + u_inj) + rho_inj/alpha, 0, 0, 0), and the sum is inverted again (guess: the
// fluid-frame result; the fluid-frame limits and ceilings act on the new state).  A failed re-inversion keeps the
// fluid-frame result and sets fflag bit 64.
// ---------------------------------------------------------------------------------------------
template <bool FLAT, int INVERTER>
__device__ __forceinline__ int invert_any(const Geo& G, const double Uh[KH_NP], double W0, double gam, const FloorPar& fp, int frame,
                                          double rho_g, double u_g, double Pout[KH_NP], int& fflag, double inj[2]) {
  if (INVERTER == 0) return u_to_p_floors<FLAT>(G, Uh, W0, gam, fp, frame, rho_g, u_g, Pout, fflag, inj);
  return u_to_p_kastaun_floors<FLAT>(G, Uh, W0, gam, fp, frame, rho_g, u_g, Pout, fflag, inj);     // W0 carries mu0 for this inverter
}

template <bool FLAT, int INVERTER>
__device__ __forceinline__ int invert_with_floors(const Geo& G, const double Uh[KH_NP], double W0, double gam, const FloorPar& fp, int frame,
                                                  double rho_g, double u_g, double Pout[KH_NP], int& fflag) {
  double inj[2];
  const int pflag = invert_any<FLAT, INVERTER>(G, Uh, W0, gam, fp, frame, rho_g, u_g, Pout, fflag, inj);
  if (frame != 2 || pflag != 0 || !(inj[0] > 0.0 || inj[1] > 0.0)) return pflag;
  const double ialpha = FLAT ? 1.0 : -G.n00 * G.alpha;
  double Ub[KH_NP], Pb[KH_NP], inj2[2];
#pragma unroll
  for (int v = 0; v < KH_NP; v++) Ub[v] = Uh[v];
  Ub[RHO] = fma(inj[0], ialpha, Ub[RHO]);
  Ub[UU] += fma(inj[0], ialpha, -(inj[0] + inj[1]));
  const double xb = 1.0 + spatial_norm2<FLAT>(G, Pout[U1], Pout[U2], Pout[U3]), efb = fma(gam, Pout[UU], Pout[RHO]);
  const double W0b = INVERTER == 0 ? efb * xb : Pout[RHO] / (efb * sqrt(xb));
  int ff2;
  const int p2 = invert_any<FLAT, INVERTER>(G, Ub, W0b, gam, fp, 0, rho_g, u_g, Pb, ff2, inj2);
  if (p2 != 0) { fflag |= 64; return 0; }
#pragma unroll
  for (int v = 0; v < 5; v++) Pout[v] = Pb[v];
  fflag = (fflag & 15) | ff2;
  return 0;
}

}  // namespace kh
