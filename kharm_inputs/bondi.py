"""Config 2: relativistic (Michel) Bondi accretion with a monopole field, in FMKS / KS, a = 0.

Textbook transonic solution: n = 1/(Gamma-1), u_c^2 = 1/(2 r_s), V_c^2 = u_c^2/(1 - 3 u_c^2),
T_c = n V_c^2 / ((n+1)(1 - n V_c^2)), C1 = u_c r_s^2 T_c^n, C2 = (1 + (1+n) T_c)^2 (1 - 2/r_s + u_c^2),
T(r) from (1 + (1+n)T)^2 (1 - 2/r + C1^2/(r^4 T^{2n})) = C2 (subsonic = larger root outside r_s,
supersonic = smaller root inside), u^r = -C1/(T^n r^2), rho = mdot T^n/(4 pi C1), u = n rho T.
"""
import numpy as np

from . import geometry as G
from .params import FMKS, NG


def michel(r, gamma=4.0 / 3.0, rs=8.0, mdot=1.0):
    r = np.asarray(r, float)
    n = 1.0 / (gamma - 1.0)
    uc2 = 1.0 / (2.0 * rs)
    Vc2 = uc2 / (1.0 - 3.0 * uc2)
    Tc = n * Vc2 / ((n + 1.0) * (1.0 - n * Vc2))
    C1 = np.sqrt(uc2) * rs ** 2 * Tc ** n
    C2 = (1.0 + (1.0 + n) * Tc) ** 2 * (1.0 - 2.0 / rs + uc2)

    def f(T):
        return (1.0 + (1.0 + n) * T) ** 2 * (1.0 - 2.0 / r + C1 ** 2 / (r ** 4 * T ** (2 * n))) - C2

    # minimum of f in log T by ternary search, then bisection on the proper side
    lo = np.full(r.shape, np.log(1e-10))
    hi = np.full(r.shape, np.log(1e4))
    for _ in range(200):
        m1 = lo + (hi - lo) / 3.0
        m2 = hi - (hi - lo) / 3.0
        left = f(np.exp(m1)) < f(np.exp(m2))
        hi = np.where(left, m2, hi)
        lo = np.where(left, lo, m1)
    tmin = 0.5 * (lo + hi)
    outside = r >= rs
    a = np.where(outside, tmin, np.log(1e-10))
    b = np.where(outside, np.log(1e4), tmin)
    fa = f(np.exp(a))
    for _ in range(200):
        m = 0.5 * (a + b)
        fm = f(np.exp(m))
        same = np.sign(fm) == np.sign(fa)
        a = np.where(same, m, a)
        fa = np.where(same, fm, fa)
        b = np.where(same, b, m)
    T = np.exp(0.5 * (a + b))
    ur = -C1 / (T ** n * r ** 2)
    rho = mdot * T ** n / (4.0 * np.pi * C1)
    u = n * rho * T
    return rho, u, ur


def config2(p, rs=8.0, mdot=1.0, bsq_over_rho_at_rs=1.0):
    """Primitives WITH ghosts [8][n3+6][n2+6][n1+6]: analytic everywhere (the x1-hi ghosts are the
    FIXED boundary data; the other ghosts are refilled by set_prims)."""
    assert p["coords"] == FMKS and p["a"] == 0.0
    g = NG
    x1, x2, x3 = G.zone_coords(p, g)
    X2, X1 = np.meshgrid(x2, x1, indexing="ij")
    r, th, dth1, dth2 = G.fmks_map(p, X1, X2)
    rho, u, ur = michel(r, p["gamma"], rs, mdot)
    gks = G.gcov_ks(0.0, r, th)
    b = gks[..., 0, 1] * ur
    c = gks[..., 1, 1] * ur ** 2 + 1.0
    utks = c / (-b + np.sqrt(b * b - gks[..., 0, 0] * c))     # regular through the horizon
    ucon = np.zeros(r.shape + (4,))
    ucon[..., 0] = utks
    ucon[..., 1] = ur / r
    ucon[..., 2] = -dth1 * ucon[..., 1] / dth2                   # u^theta = 0
    gcov, gcon, gdet, alpha = G.geom(p, X1, X2)
    ut = G.ucon_to_utilde(gcon, alpha, ucon)

    # monopole: A_phi = C (1 - cos theta) on corners
    xf1, xf2, _ = G.zone_coords(p, g, extra=1)
    XF2, XF1 = np.meshgrid(xf2, xf1, indexing="ij")
    _, thc, _, _ = G.fmks_map(p, XF1, XF2)
    d = G.dx(p)
    A = 1.0 - np.cos(thc)
    B1, B2 = G.field_from_aphi(A, gdet, d[0], d[1])

    # normalisation from the analytic point (r_s, pi/2) in KS: B^r = C / r^2
    rho_s, _, ur_s = michel(np.array([rs]), p["gamma"], rs, mdot)
    gs = G.gcov_ks(0.0, np.array([rs]), np.array([0.5 * np.pi]))
    gsi = np.linalg.inv(gs)
    al_s = 1.0 / np.sqrt(-gsi[..., 0, 0])
    bs = gs[..., 0, 1] * ur_s
    cs = gs[..., 1, 1] * ur_s ** 2 + 1.0
    uc = np.zeros((1, 4))
    uc[:, 0] = cs / (-bs + np.sqrt(bs * bs - gs[..., 0, 0] * cs))
    uc[:, 1] = ur_s
    ut_s = G.ucon_to_utilde(gsi, al_s, uc)
    Bs = np.zeros((1, 3))
    Bs[:, 0] = 1.0 / rs ** 2
    bsq1 = G.bsq_of(gs, gsi, al_s, ut_s, Bs)[0]
    C = np.sqrt(bsq_over_rho_at_rs * rho_s[0] / bsq1)

    n3t = p["n3"] + 2 * g
    P = np.zeros((8, n3t) + r.shape)
    P[0] = rho[None]
    P[1] = u[None]
    for i in range(3):
        P[2 + i] = ut[..., i][None]
    P[5] = (C * B1)[None]
    P[6] = (C * B2)[None]
    return P
