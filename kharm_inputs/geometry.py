"""numpy coordinate / metric formulas used ONLY to pose initial conditions.

Kerr-Schild metric in (t,r,theta,phi) and the FMKS map (ref [61]) -- the same
mathematics the two implementations realise, written a third time, vectorised, so that the input
generators depend on neither of them.
"""
import numpy as np

from .params import FMKS, KS, MINKOWSKI, NG


def zone_coords(p, ghosts=0, extra=0):
    """Native zone-centre coordinate vectors (x1, x2, x3) with `ghosts` layers per side.
    extra=1 gives the lower-corner/face coordinates instead (one more point)."""
    out = []
    for d, n in enumerate((p["n1"], p["n2"], p["n3"])):
        dx = (p["xmax"][d] - p["xmin"][d]) / n
        if extra:
            i = np.arange(-ghosts, n + ghosts + 1)
            out.append(p["xmin"][d] + i * dx)
        else:
            i = np.arange(-ghosts, n + ghosts)
            out.append(p["xmin"][d] + (i + 0.5) * dx)
    return out


def dx(p):
    return [(p["xmax"][d] - p["xmin"][d]) / n for d, n in enumerate((p["n1"], p["n2"], p["n3"]))]


def fmks_map(p, x1, x2):
    """r, theta and the Jacobian entries dtheta/dx1, dtheta/dx2 of the FMKS map."""
    hs, xt, al, sm = p["hslope"], p["poly_xt"], p["poly_alpha"], p["mks_smooth"]
    r = np.exp(x1)
    y = 2.0 * x2 - 1.0
    thG = np.pi * x2 + 0.5 * (1.0 - hs) * np.sin(2.0 * np.pi * x2)
    dthG = np.pi * (1.0 + (1.0 - hs) * np.cos(2.0 * np.pi * x2))
    norm = 0.5 * np.pi / (1.0 + xt ** (-al) / (al + 1.0))
    ya = (y / xt) ** al if float(al).is_integer() else np.abs(y / xt) ** al
    thJ = norm * y * (1.0 + ya / (al + 1.0)) + 0.5 * np.pi
    dthJ = 2.0 * norm * (1.0 + ya)
    e = np.exp(sm * (p["xmin"][0] - x1))
    th = thG + e * (thJ - thG)
    return r, th, -sm * e * (thJ - thG), dthG + e * (dthJ - dthG)


def embed(p, x1, x2):
    """(r, theta) of native points; Minkowski returns the inputs."""
    if p["coords"] == FMKS:
        r, th, _, _ = fmks_map(p, x1, x2)
        return r, th
    return x1 + 0 * x2, x2 + 0 * x1


def gcov_ks(a, r, th):
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    f = 2.0 * r / Sig
    g = np.zeros(np.broadcast(r, th).shape + (4, 4))
    g[..., 0, 0] = -(1.0 - f)
    g[..., 0, 1] = g[..., 1, 0] = f
    g[..., 0, 3] = g[..., 3, 0] = -a * f * s2
    g[..., 1, 1] = 1.0 + f
    g[..., 1, 3] = g[..., 3, 1] = -a * s2 * (1.0 + f)
    g[..., 2, 2] = Sig
    g[..., 3, 3] = s2 * (Sig + a * a * s2 * (1.0 + f))
    return g


def gcov_native(p, x1, x2):
    """Covariant metric in native coordinates at broadcast(x1, x2) points -> [...,4,4]."""
    x1, x2 = np.broadcast_arrays(np.asarray(x1, float), np.asarray(x2, float))
    if p["coords"] == MINKOWSKI:
        g = np.zeros(x1.shape + (4, 4))
        g[..., 0, 0] = -1.0
        for m in (1, 2, 3):
            g[..., m, m] = 1.0
        return g
    if p["coords"] == KS:
        return gcov_ks(p["a"], x1, x2)
    r, th, d1, d2 = fmks_map(p, x1, x2)
    gks = gcov_ks(p["a"], r, th)
    L = np.zeros(x1.shape + (4, 4))
    L[..., 0, 0] = 1.0
    L[..., 1, 1] = r
    L[..., 2, 1] = d1
    L[..., 2, 2] = d2
    L[..., 3, 3] = 1.0
    return np.einsum("...am,...ab,...bn->...mn", L, gks, L)


def geom(p, x1, x2):
    """gcov, gcon, sqrt(-g), lapse at broadcast points."""
    gcov = gcov_native(p, x1, x2)
    gcon = np.linalg.inv(gcov)
    gdet = np.sqrt(-np.linalg.det(gcov))
    alpha = 1.0 / np.sqrt(-gcon[..., 0, 0])
    return gcov, gcon, gdet, alpha


def ucon_to_utilde(gcon, alpha, ucon):
    """ut^i = u^i + alpha^2 u^t g^{ti}  (the velocity primitive of ref [32])."""
    return ucon[..., 1:] + (alpha ** 2 * ucon[..., 0])[..., None] * gcon[..., 0, 1:]


def bsq_of(gcov, gcon, alpha, ut, B):
    """b^2 of a state given ut^i and B^i (needed to normalise field strengths)."""
    qsq = np.einsum("...i,...ij,...j->...", ut, gcov[..., 1:, 1:], ut)
    gamma = np.sqrt(1.0 + qsq)
    ucon = np.zeros(ut.shape[:-1] + (4,))
    ucon[..., 0] = gamma / alpha
    ucon[..., 1:] = ut - (gamma * alpha)[..., None] * gcon[..., 0, 1:]
    ucov = np.einsum("...mn,...n->...m", gcov, ucon)
    bt = np.einsum("...i,...i->...", B, ucov[..., 1:])
    bcon = np.zeros_like(ucon)
    bcon[..., 0] = bt
    bcon[..., 1:] = (B + bt[..., None] * ucon[..., 1:]) / ucon[..., 0][..., None]
    bcov = np.einsum("...mn,...n->...m", gcov, bcon)
    return np.einsum("...m,...m->...", bcon, bcov)


def field_from_aphi(A, gdet, dx1, dx2):
    """Cell-centred B^1, B^2 from a corner-centred A_phi so that the Flux-CT corner divergence is
    zero to round-off.  A: [nj+1, ni+1] at lower corners (j,i); gdet: [nj, ni] at centres."""
    B1 = (A[1:, :-1] + A[1:, 1:] - A[:-1, :-1] - A[:-1, 1:]) / (2.0 * dx2 * gdet)
    B2 = -(A[:-1, 1:] + A[1:, 1:] - A[:-1, :-1] - A[1:, :-1]) / (2.0 * dx1 * gdet)
    return B1, B2
