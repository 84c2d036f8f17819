"""Configs 3 and 4: Fishbone-Moncrief torus around a Kerr hole in FMKS coordinates, SANE or MAD
seed field, plus an optional seeded "stress" variant that plants strongly magnetised cold patches.

Stands in for the paper's EHT-style torus workload: same grid shape,
coordinates, value ranges (floors' atmosphere around a rho_max = 1 torus, weak poloidal loop) and
perturbation.  All formulas are the textbook FM solution in Boyer-Lindquist quantities.
"""
import numpy as np

from . import geometry as G
from .params import NG
from .rng import splitmix64_uniform


def fm_ell(a, rmax):
    """FM constant l = u_phi u^t of the prograde circular equatorial geodesic at rmax (BL)."""
    r = rmax
    Om = 1.0 / (r ** 1.5 + a)
    gtt = -(1.0 - 2.0 / r)
    gtp = -2.0 * a / r
    gpp = r * r + a * a + 2.0 * a * a / r
    ut = 1.0 / np.sqrt(-(gtt + 2.0 * gtp * Om + gpp * Om * Om))
    uphi = (gtp + gpp * Om) * ut
    return uphi * ut


def _lnh_raw(a, ell, r, th):
    s = np.sin(th)
    s = np.where(np.abs(s) < 1e-12, 1e-12, s)
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2.0 * r + a * a
    AA = (r * r + a * a) ** 2 - Del * a * a * s * s
    with np.errstate(invalid="ignore", divide="ignore"):
        Psi = np.sqrt(1.0 + 4.0 * ell ** 2 * Sig ** 2 * Del / (AA * s) ** 2)
        val = 0.5 * np.log((1.0 + Psi) / (Sig * Del / AA)) - 0.5 * Psi - 2.0 * a * r * ell / AA
    return val, Psi, Sig, Del, AA, s


def fm_torus(p, rin=6.0, rmax=12.0, kappa=1e-3, ghosts=0):
    """rho, u, u^phi (BL = KS since u^r = 0) and the inside-mask on the zone grid [nj, ni] (+ghosts)."""
    a, gam = p["a"], p["gamma"]
    ell = fm_ell(a, rmax)
    x1, x2, _ = G.zone_coords(p, ghosts)
    X2, X1 = np.meshgrid(x2, x1, indexing="ij")
    r, th = G.embed(p, X1, X2)
    lnh_in = _lnh_raw(a, ell, np.array(rin), np.array(0.5 * np.pi))[0]
    lnh, Psi, Sig, Del, AA, s = _lnh_raw(a, ell, r, th)
    lnh = lnh - lnh_in
    inside = np.isfinite(lnh) & (lnh > 0.0) & (r >= rin) & (Del > 0)
    h = np.exp(np.where(inside, lnh, 0.0))
    rho = np.where(inside, ((h - 1.0) * (gam - 1.0) / (kappa * gam)) ** (1.0 / (gam - 1.0)), 0.0)
    u = kappa * rho ** gam / (gam - 1.0)
    ups2 = 0.5 * (Psi - 1.0)
    with np.errstate(invalid="ignore", divide="ignore"):
        uphi = 2.0 * a * r * np.sqrt(1.0 + ups2) / np.sqrt(AA * Sig * Del) + np.sqrt(Sig / AA) * np.sqrt(ups2) / s
    uphi = np.where(inside, uphi, 0.0)
    return dict(rho=rho, u=u, uphi=uphi, inside=inside, r=r, th=th, X1=X1, X2=X2, ell=ell)


def torus_state(p, mad=False, seed=1, rin=6.0, rmax=12.0, kappa=1e-3, beta_min=100.0, perturb=0.04,
                stress=False, stress_fraction=0.01):
    """Primitives [8][n3][n2][n1] (interior) of config 3 (mad=False) or 4 (mad=True)."""
    g = 1                                          # one ghost layer: corner means need neighbours
    T = fm_torus(p, rin, rmax, kappa, ghosts=g)
    r, th, X1, X2, inside = T["r"], T["th"], T["X1"], T["X2"], T["inside"]
    gcov, gcon, gdet, alpha = G.geom(p, X1, X2)
    a = p["a"]

    # u^t from u.u = -1 in BL with u^r = u^theta = 0
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2.0 * r + a * a
    AA = (r * r + a * a) ** 2 - Del * a * a * s2
    gtt = -(1.0 - 2.0 * r / Sig)
    gtp = -2.0 * a * r * s2 / Sig
    gpp = AA * s2 / Sig
    up = T["uphi"]
    qa, qb, qc = gtt, 2.0 * gtp * up, gpp * up * up + 1.0
    with np.errstate(invalid="ignore", divide="ignore"):
        utbl = (-qb - np.sqrt(qb * qb - 4.0 * qa * qc)) / (2.0 * qa)
    ucon = np.zeros(r.shape + (4,))
    ucon[..., 0] = np.where(inside, utbl, 0.0)
    ucon[..., 3] = up
    ut = np.where(inside[..., None], G.ucon_to_utilde(gcon, alpha, ucon), 0.0)

    rho_max = T["rho"].max()
    rho = T["rho"] / rho_max
    u = T["u"] / rho_max
    # atmosphere at the geometric floors (DESIGN.md "Readings" S18)
    sfl = 1.0 / r ** 2 / (1.0 + r / p["r_char"])
    rho_fl = p["rho_min"] * sfl
    u_fl = p["u_min"] * sfl ** p["gamma"]
    torus_zone = inside & (rho > rho_fl) & (u > u_fl)
    rho = np.where(torus_zone, rho, rho_fl)
    u = np.where(torus_zone, u, u_fl)
    ut = np.where(torus_zone[..., None], ut, 0.0)

    # vector potential on lower corners of the interior (+1): mean of the 4 zones around each corner
    rho_t = np.where(torus_zone, rho, 0.0)
    rbar = 0.25 * (rho_t[:-1, :-1] + rho_t[:-1, 1:] + rho_t[1:, :-1] + rho_t[1:, 1:])   # corners (j,i), j,i = 0..n
    if mad:
        xf1, xf2, _ = G.zone_coords(p, 0, extra=1)
        XF2, XF1 = np.meshgrid(xf2, xf1, indexing="ij")
        rc, thc = G.embed(p, XF1, XF2)
        q = rbar * (rc / rin) ** 3 * np.sin(thc) ** 3 * np.exp(-rc / 400.0) - 0.2
    else:
        q = rbar - 0.2
    A = np.maximum(q, 0.0)
    d = G.dx(p)
    ci = (slice(g, -g), slice(g, -g))                  # interior of the 1-ghost arrays
    B1, B2 = G.field_from_aphi(A, gdet[ci], d[0], d[1])
    B = np.stack([B1, B2, np.zeros_like(B1)], axis=-1)
    bsq = G.bsq_of(gcov[ci], gcon[ci], alpha[ci], ut[ci], B)
    pmax = ((p["gamma"] - 1.0) * u[ci]).max()
    bmax = 0.5 * bsq.max()
    B *= np.sqrt(pmax / (beta_min * bmax)) if bmax > 0 else 0.0

    n1, n2, n3 = p["n1"], p["n2"], p["n3"]
    P = np.zeros((8, n3, n2, n1))
    P[0] = rho[ci][None]
    P[1] = u[ci][None]
    for i in range(3):
        P[2 + i] = ut[ci][..., i][None]
        P[5 + i] = B[..., i][None]

    idx = np.arange(n3 * n2 * n1, dtype=np.uint64).reshape(n3, n2, n1)
    if perturb:
        xi = splitmix64_uniform(seed, idx)
        P[1] = np.where(torus_zone[ci][None], P[1] * (1.0 + perturb * (2.0 * xi - 1.0)), P[1])
    if stress:
        # seeded cold, strongly magnetised patches: b^2/rho in [50,500], u/rho in [1e-8,1e-4]
        # (B is left untouched so div B stays at round-off; rho and u are lowered instead)
        xs = splitmix64_uniform(seed + 1000, idx)
        x2_ = splitmix64_uniform(seed + 2000, idx)
        x3_ = splitmix64_uniform(seed + 3000, idx)
        bsq3 = G.bsq_of(gcov[ci], gcon[ci], alpha[ci], ut[ci], B)[None] + 0.0 * P[0]
        pick = (xs < stress_fraction) & (bsq3 > 0.0)
        ratio = 50.0 * 10.0 ** x2_
        rho_new = bsq3 / ratio
        u_new = rho_new * 10.0 ** (-8.0 + 4.0 * x3_)
        P[0] = np.where(pick, rho_new, P[0])
        P[1] = np.where(pick, u_new, P[1])
    return P
