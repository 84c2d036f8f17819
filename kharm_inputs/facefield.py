"""Seeded face-centred magnetic fields for the face-centred CT transport.

Problem definition only: a vector potential on the zone edges and its discrete circulation around each face
(Stokes), which makes the face field divergence-free to round-off by construction.  Array layout as everywhere:
[k][j][i] with 3 ghost layers; an entry belongs to the zone whose LOWER corner / edge / face it sits on.
    Phi^1 = d2 A3 - d3 A2,  Phi^2 = d3 A1 - d1 A3,  Phi^3 = d1 A2 - d2 A1     (Phi^d = sqrt(-g) B^d on the d-face)
"""
import numpy as np

from .rng import splitmix64_uniform

NG = 3


def _dx(p):
    return [(p["xmax"][d] - p["xmin"][d]) / (p["n1"], p["n2"], p["n3"])[d] for d in range(3)]


def face_from_potential(p, A1, A2, A3):
    """Face fluxes from edge potentials (arrays over the ghosted lattice); the last layer in each direction is left 0."""
    dx = _dx(p)
    f = [np.zeros_like(A1) for _ in range(3)]
    d1 = lambda a: a[:-1, :-1, 1:] - a[:-1, :-1, :-1]
    d2 = lambda a: a[:-1, 1:, :-1] - a[:-1, :-1, :-1]
    d3 = lambda a: a[1:, :-1, :-1] - a[:-1, :-1, :-1]
    f[0][:-1, :-1, :-1] = d2(A3) / dx[1] - d3(A2) / dx[2]
    f[1][:-1, :-1, :-1] = d3(A1) / dx[2] - d1(A3) / dx[0]
    f[2][:-1, :-1, :-1] = d1(A2) / dx[0] - d2(A1) / dx[1]
    return f


def corner_coords(p):
    """native coordinates of the lower corner of every zone of the ghosted lattice: x1[i], x2[j], x3[k]"""
    dx = _dx(p)
    return [p["xmin"][d] + (np.arange(-NG, (p["n1"], p["n2"], p["n3"])[d] + NG)) * dx[d] for d in range(3)]


def periodic_potential(p, seed=1, amp=1e-2, nmodes=4):
    """A superposition of periodic Fourier modes on [xmin, xmax]^3 for each component (Minkowski cube)."""
    x1, x2, x3 = corner_coords(p)
    L = [p["xmax"][d] - p["xmin"][d] for d in range(3)]
    X3, X2, X1 = np.meshgrid(x3, x2, x1, indexing="ij")
    out = []
    c = 0
    for comp in range(3):
        A = np.zeros_like(X1)
        for m in range(nmodes):
            r = splitmix64_uniform(seed, np.arange(c, c + 5)); c += 5
            k = [int(r[0] * 3) - 1, int(r[1] * 3) - 1, int(r[2] * 3) - 1]
            if k == [0, 0, 0]:
                k = [1, 0, 0]
            ph = 2 * np.pi * r[3]
            A += amp * (0.5 + r[4]) * np.cos(2 * np.pi * (k[0] * (X1 - p["xmin"][0]) / L[0] + k[1] * (X2 - p["xmin"][1]) / L[1]
                                                          + k[2] * (X3 - p["xmin"][2]) / L[2]) + ph)
        out.append(A)
    return out


def axisymmetric_loop_potential(p, amp=1e-3, x1c=None, width=0.6):
    """A_phi(x1, x2) of a poloidal loop centred on the midplane, vanishing on the polar axis (torus-like SANE field):
    A3 = amp sin^2(pi x2) exp(-((x1 - x1c)/width)^2); A1 = A2 = 0."""
    x1, x2, x3 = corner_coords(p)
    if x1c is None:
        x1c = 0.5 * (p["xmin"][0] + p["xmax"][0])
    a = amp * np.sin(np.pi * np.clip(x2, 0.0, 1.0))[:, None] ** 2 * np.exp(-((x1 - x1c) / width) ** 2)[None, :]
    A3 = np.broadcast_to(a[None], (len(x3), len(x2), len(x1))).copy()
    return [np.zeros_like(A3), np.zeros_like(A3), A3]
