"""Linear MHD modes on a periodic Minkowski box (BASELINE.json configs 1 and 5).

The eigen-system comes from the ANALYTIC linearisation of ideal relativistic MHD about a static
background (rho0, u0, v = 0, B0), written in the primitive basis (rho, u, v^i, B^i):

    lam drho = rho0 (n.dv)                 lam du = Gamma u0 (n.dv)
    lam [(w + B0^2) I - B0 B0^T] dv = n ((Gamma-1) du + B0.dB) - (B0.n) dB
    lam dB = -(B0.n) dv + B0 (n.dv)

(lam = phase speed along the unit vector n, w = rho0 + Gamma u0).  It uses no flux function of
either implementation, so it also serves as an independent pin of the oracle's U(P), F(P).
"""
import numpy as np

from .geometry import dx as _dx
from .geometry import zone_coords
from .rng import splitmix64_uniform

FAST, ALFVEN, SLOW = 0, 1, 2


def linear_system(nhat, rho0, u0, B0, gamma):
    """8x8 matrix A with A r = lam r for plane waves along unit vector nhat."""
    nhat = np.asarray(nhat, float)
    B0 = np.asarray(B0, float)
    w = rho0 + gamma * u0
    M = np.eye(8)
    M[2:5, 2:5] = (w + B0 @ B0) * np.eye(3) - np.outer(B0, B0)
    N = np.zeros((8, 8))
    N[0, 2:5] = rho0 * nhat
    N[1, 2:5] = gamma * u0 * nhat
    N[2:5, 1] = (gamma - 1.0) * nhat
    N[2:5, 5:8] = np.outer(nhat, B0) - (B0 @ nhat) * np.eye(3)
    N[5:8, 2:5] = -(B0 @ nhat) * np.eye(3) + np.outer(B0, nhat)
    return np.linalg.solve(M, N)


def eigenmode(nhat, family, rho0=1.0, u0=1.0, B0=(1.0, 0.0, 0.0), gamma=4.0 / 3.0, sign=+1, prefer=3):
    """(phase speed, unit-norm real eigenvector) of the requested family travelling along sign*nhat.

    Families are ordered by |lam|: fast >= Alfven >= slow.  Degenerate eigenvalues (k parallel to
    B0) are resolved by projecting the unit vector of primitive index `prefer` (default ut2) onto
    the eigenspace, which fixes the x2 polarisation.
    """
    A = linear_system(nhat, rho0, u0, B0, gamma)
    lam, vec = np.linalg.eig(A)
    lam, vec = lam.real, vec.real
    pos = np.sort(lam[lam > 1e-9])[::-1]          # three positive speeds, descending
    if pos.size == 0:
        raise ValueError("no propagating mode")
    if family >= pos.size:                        # k perpendicular to B0: only the fast mode propagates
        family = FAST
    target = sign * pos[family]
    sel = np.abs(lam - target) < 1e-8 * max(1.0, abs(target))
    V = vec[:, sel]
    Q, _ = np.linalg.qr(V)
    e = np.zeros(8)
    e[prefer] = 1.0
    r = Q @ (Q.T @ e)
    if np.linalg.norm(r) < 1e-6:                  # preferred component absent: take the first vector
        r = Q[:, 0].copy()
    r /= np.linalg.norm(r)
    k = int(np.argmax(np.abs(r) > 1e-9))           # sign convention: first non-zero component positive
    if r[k] < 0:
        r = -r
    return target, r


def _curl_free_field(p, kvec, bhat, phase, ghosts):
    """Zone-centred dB = bhat cos(k.x + phase) built from an edge-centred vector potential
    A = -(k x bhat)/|k|^2 sin(k.x + phase): face fields by Stokes, centre = mean of the two faces,
    so the Flux-CT corner divergence vanishes to round-off."""
    d = _dx(p)
    xc = zone_coords(p, ghosts + 1)                     # one extra layer so faces exist on both sides
    xf = [c - 0.5 * h for c, h in zip(xc, d)]           # lower faces
    avec = -np.cross(kvec, bhat) / (kvec @ kvec)

    def A(comp, X1, X2, X3):
        return avec[comp] * np.sin(kvec[0] * X1 + kvec[1] * X2 + kvec[2] * X3 + phase)

    # broadcasting helpers: arrays indexed [k, j, i]
    def g(x3, x2, x1):
        return np.meshgrid(x3, x2, x1, indexing="ij")

    # A1 on edges (i centre, j face, k face); A2 on (i face, j centre, k face); A3 on (i face, j face, k centre)
    X3, X2, X1 = g(xf[2], xf[1], xc[0]); A1 = A(0, X1, X2, X3)
    X3, X2, X1 = g(xf[2], xc[1], xf[0]); A2 = A(1, X1, X2, X3)
    X3, X2, X1 = g(xc[2], xf[1], xf[0]); A3 = A(2, X1, X2, X3)
    # face B^1 at (i face, j centre, k centre) = d2 A3 - d3 A2   (valid for j,k < last)
    Bf1 = (A3[:-1, 1:, :] - A3[:-1, :-1, :]) / d[1] - (A2[1:, :-1, :] - A2[:-1, :-1, :]) / d[2]
    Bf2 = (A1[1:, :, :-1] - A1[:-1, :, :-1]) / d[2] - (A3[:-1, :, 1:] - A3[:-1, :, :-1]) / d[0]
    Bf3 = (A2[:, :-1, 1:] - A2[:, :-1, :-1]) / d[0] - (A1[:, 1:, :-1] - A1[:, :-1, :-1]) / d[1]
    # centres: mean of the two faces; drop the extra layer
    Bc1 = 0.5 * (Bf1[:, :, 1:] + Bf1[:, :, :-1])
    Bc2 = 0.5 * (Bf2[:, 1:, :] + Bf2[:, :-1, :])
    Bc3 = 0.5 * (Bf3[1:, :, :] + Bf3[:-1, :, :])
    # all three now have shape [n3+2g+1, n2+2g+1, n1+2g+1] restricted; crop to [.. +2g]
    n3, n2, n1 = (p["n3"] + 2 * ghosts, p["n2"] + 2 * ghosts, p["n1"] + 2 * ghosts)
    sl = (slice(1, 1 + n3), slice(1, 1 + n2), slice(1, 1 + n1))
    return Bc1[sl], Bc2[sl], Bc3[sl]


def mode_state(p, kvec, family, amp, rho0=1.0, u0=1.0, B0=(1.0, 0.0, 0.0), sign=+1, phase=0.0, t=0.0,
               ghosts=0, vector_potential=True):
    """Primitives [8][n3][n2][n1] (+ghosts) of background + amp * r * cos(k.x - omega t + phase).
    Returns (P, omega)."""
    kvec = np.asarray(kvec, float)
    knorm = np.linalg.norm(kvec)
    lam, r = eigenmode(kvec / knorm, family, rho0, u0, B0, p["gamma"], sign)
    omega = lam * knorm
    P = background(p, rho0, u0, B0, ghosts)
    add_mode(p, P, kvec, r, amp, phase - omega * t, ghosts, vector_potential)
    return P, omega


def background(p, rho0, u0, B0, ghosts=0):
    shape = (8, p["n3"] + 2 * ghosts, p["n2"] + 2 * ghosts, p["n1"] + 2 * ghosts)
    P = np.zeros(shape)
    P[0], P[1] = rho0, u0
    for i in range(3):
        P[5 + i] = B0[i]
    return P


def add_mode(p, P, kvec, r, amp, phase, ghosts=0, vector_potential=True):
    x1, x2, x3 = zone_coords(p, ghosts)
    X3, X2, X1 = np.meshgrid(x3, x2, x1, indexing="ij")
    c = np.cos(kvec[0] * X1 + kvec[1] * X2 + kvec[2] * X3 + phase)
    for v in range(5):
        P[v] += amp * r[v] * c
    bvec = r[5:8]
    bn = np.linalg.norm(bvec)
    if vector_potential and bn > 1e-14:
        b1, b2, b3 = _curl_free_field(p, np.asarray(kvec, float), bvec / bn, phase, ghosts)
        P[5] += amp * bn * b1
        P[6] += amp * bn * b2
        P[7] += amp * bn * b3
    else:
        for v in range(5, 8):
            P[v] += amp * r[v] * c


def config1(p, rotated=False, amp=1e-4):
    """Config 1: fast mode, B0 = (1,0,0), k = (2pi,0,0) or rotated (2pi,2pi,0).
    Returns (P interior, period T)."""
    k = np.array([2 * np.pi, 2 * np.pi if rotated else 0.0, 0.0])
    P, omega = mode_state(p, k, FAST, amp)
    return P, 2 * np.pi / abs(omega)


def config5(p, seed=1, amp=1e-3, nmodes=8):
    """Config 5: seeded random-phase superposition of `nmodes` linear modes, k = 2pi (n1,n2,n3),
    n in {-2..2}^3 minus 0, family / direction / phase from the seed."""
    xi = splitmix64_uniform(seed, np.arange(8 * nmodes)).reshape(nmodes, 8)
    P = background(p, 1.0, 1.0, (1.0, 0.0, 0.0))
    for m in range(nmodes):
        n = np.floor(xi[m, 0:3] * 5).astype(int) - 2
        if not n.any():
            n[m % 3] = 1
        fam = int(xi[m, 3] * 3)
        sign = 1 if xi[m, 4] < 0.5 else -1
        phase = 2 * np.pi * xi[m, 5]
        k = 2 * np.pi * n
        _, r = eigenmode(k / np.linalg.norm(k), fam, 1.0, 1.0, (1.0, 0.0, 0.0), p["gamma"], sign)
        add_mode(p, P, k, r, amp, phase)
    return P
