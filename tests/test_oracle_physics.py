"""Pins of the oracle's point-wise physics (C2): invariants, eq. 1.1, special-relativistic
textbook limits, and the eigenvalues of its flux Jacobian against the analytic linearisation."""
import numpy as np
import pytest

import kharm_inputs as ki
from kharm_inputs import modes
from kharm_inputs import params as kp

ETA = np.diag([-1.0, 1, 1, 1])


def _geoms(kho):
    """(name, gcov, gcon, gdet) at a few points of the three coordinate systems."""
    out = [("mink", ETA, ETA, 1.0)]
    Pk = kho.make_params(ki.base_params(coords=kp.KS, a=0.9375))
    for r, th in ((1.6, 0.4), (6.0, 1.3), (40.0, 2.8)):
        g = kho.metric(Pk, r, th)
        out.append(("ks", g[0], g[1], g[2]))
    Pf = kho.make_params(ki.config_params(3))
    for x1, x2 in ((0.3, 0.02), (2.0, 0.4), (5.5, 0.97)):
        g = kho.metric(Pf, x1, x2)
        out.append(("fmks", g[0], g[1], g[2]))
    return out


def _rand_prims(rng, gcov, scale_v=1.0):
    P = np.zeros(8)
    P[0] = 10 ** rng.uniform(-3, 1)
    P[1] = P[0] * 10 ** rng.uniform(-3, 1)
    # velocities / fields sized by the metric so that q^2 and b^2/rho are O(1)
    for i in range(3):
        P[2 + i] = scale_v * rng.normal() / np.sqrt(gcov[i + 1, i + 1])
        P[5 + i] = np.sqrt(P[0]) * rng.normal() / np.sqrt(gcov[i + 1, i + 1])
    return P


def test_four_vector_invariants_and_eq_1_1(kho):
    rng = np.random.default_rng(11)
    gam = 13.0 / 9.0
    for name, gcov, gcon, gdet in _geoms(kho):
        for _ in range(20):
            P = _rand_prims(rng, gcov)
            D = kho.fourvec(gcov, gcon, P)
            u, ul, b, bl = D["ucon"], D["ucov"], D["bcon"], D["bcov"]
            assert abs(u @ ul + 1) < 1e-12 * (1 + u[0] ** 2 * abs(gcov[0, 0]))      # u.u = -1
            assert abs(b @ ul) < 1e-12 * (np.abs(b * ul).sum() + 1e-300)              # b.u = 0
            assert np.allclose(ul, gcov @ u, rtol=1e-13, atol=1e-15) and np.allclose(bl, gcov @ b, rtol=1e-13, atol=1e-14)
            assert abs(D["bsq"] - b @ bl) <= 1e-13 * np.abs(b * bl).sum()
            # B^i = b^i u^t - b^t u^i  (definition of the field primitive)
            assert np.allclose(b[1:] * u[0] - b[0] * u[1:], P[5:8], rtol=1e-11, atol=1e-13)
            # normal-observer decomposition u^mu = gamma n^mu + ut^mu with n_mu = (-alpha,0,0,0)   (S1)
            alpha = (-gcon[0, 0]) ** -0.5
            gamma = alpha * u[0]
            assert np.allclose(P[2:5], u[1:] + gamma * alpha * gcon[0, 1:], rtol=1e-12, atol=1e-14)
            # eq. 1.1: T^{mu nu} = (rho+u+p+b^2) u^mu u^nu + (p + b^2/2) g^{mu nu} - b^mu b^nu, one index lowered
            p = (gam - 1) * P[1]
            Tcon = (P[0] + P[1] + p + D["bsq"]) * np.outer(u, u) + (p + 0.5 * D["bsq"]) * gcon - np.outer(b, b)
            Tmix = Tcon @ gcov
            T = kho.stress(gcov, gcon, P, gam)
            assert np.abs(T - Tmix).max() <= 1e-11 * np.abs(Tmix).max()
            # U and F^d assembled from it (S8: energy slot T^t_t + rho u^t)
            for d in range(4):
                F = kho.prim_to_flux(gcov, gcon, gdet, P, gam, d)
                want = np.zeros(8)
                want[0] = gdet * P[0] * u[d]
                want[1] = gdet * (Tmix[d, 0] + P[0] * u[d])
                want[2:5] = gdet * Tmix[d, 1:]
                want[5:8] = gdet * (b[1:] * u[d] - b[d] * u[1:])
                assert np.abs(F - want).max() <= 1e-10 * max(np.abs(want).max(), 1e-300)
                if d > 0:
                    assert F[4 + d] == 0.0 or abs(F[4 + d]) < 1e-14 * np.abs(F[5:8]).max()     # F^d[B^d] = 0
                else:
                    assert np.allclose(F[5:8], gdet * P[5:8], rtol=1e-15)


def test_rest_frame_and_srhd_textbook(kho):
    gam = 5.0 / 3.0
    P = np.array([2.0, 0.7, 0, 0, 0, 0.3, -0.4, 0.5])
    U = kho.prim_to_flux(ETA, ETA, 1.0, P, gam, 0)
    bsq = 0.3 ** 2 + 0.4 ** 2 + 0.5 ** 2
    assert np.allclose(U, [2.0, -0.7 - 0.5 * bsq, 0, 0, 0, 0.3, -0.4, 0.5], atol=1e-15)
    # special-relativistic hydro, velocity v along x:  D = rho W, S_x = w W^2 v, tau-like slot = -(w W^2 - p) + D
    v = 0.6
    W = 1 / np.sqrt(1 - v * v)
    P = np.array([1.3, 0.9, W * v, 0, 0, 0, 0, 0])
    p = (gam - 1) * 0.9
    w = 1.3 + 0.9 + p
    U = kho.prim_to_flux(ETA, ETA, 1.0, P, gam, 0)
    F = kho.prim_to_flux(ETA, ETA, 1.0, P, gam, 1)
    assert np.allclose(U[:3], [1.3 * W, -(w * W * W - p) + 1.3 * W, w * W * W * v], rtol=1e-14)
    assert np.allclose(F[:3], [1.3 * W * v, -w * W * W * v + 1.3 * W * v, w * W * W * v * v + p], rtol=1e-14)


def test_wave_speeds(kho):
    gam = 4.0 / 3.0
    rho, u = 1.0, 0.8
    cs = np.sqrt(gam * (gam - 1) * u / (rho + gam * u))
    # rest frame, no field: +-c_s in every direction
    P = np.array([rho, u, 0, 0, 0, 0, 0, 0.0])
    for d in (1, 2, 3):
        vmax, vmin = kho.vchar(ETA, ETA, P, gam, d)
        assert abs(vmax - cs) < 1e-14 and abs(vmin + cs) < 1e-14
    # boosted along x: relativistic velocity addition
    for v in (0.3, -0.7, 0.95):
        W = 1 / np.sqrt(1 - v * v)
        P = np.array([rho, u, W * v, 0, 0, 0, 0, 0.0])
        vmax, vmin = kho.vchar(ETA, ETA, P, gam, 1)
        assert abs(vmax - (v + cs) / (1 + v * cs)) < 1e-13 and abs(vmin - (v - cs) / (1 - v * cs)) < 1e-13
    # field perpendicular to k at rest: the bound is the exact fast speed sqrt(vA^2 + cs^2 (1 - vA^2))
    B = 0.9
    P = np.array([rho, u, 0, 0, 0, 0, B, 0.0])
    vA2 = B * B / (B * B + rho + gam * u)
    vmax, vmin = kho.vchar(ETA, ETA, P, gam, 1)
    lam, _ = modes.eigenmode([1, 0, 0], modes.FAST, rho, u, (0, B, 0), gam)
    assert abs(vmax - np.sqrt(vA2 + cs * cs * (1 - vA2))) < 1e-14 and abs(vmax - lam) < 1e-12 and abs(vmin + vmax) < 1e-15
    # causality in curved space: |coordinate speed| bounded by the light cone  g_tt + 2 g_td v + g_dd v^2 <= 0
    rng = np.random.default_rng(3)
    Pk = kho.make_params(ki.config_params(3))
    gcov, gcon, gdet, _ = kho.metric(Pk, 1.1, 0.3)
    for _ in range(20):
        Pz = _rand_prims(rng, gcov)
        for d in (1, 2, 3):
            vmax, vmin = kho.vchar(gcov, gcon, Pz, gam, d)
            A, Bq, C = gcon[0, 0], gcon[0, d], gcon[d, d]
            # light cone in direction d: roots of g^tt v^2 - 2 g^td v + g^dd = 0
            disc = np.sqrt(Bq * Bq - A * C)
            lo, hi = sorted([(Bq + disc) / A, (Bq - disc) / A])
            assert lo - 1e-12 <= vmin <= vmax <= hi + 1e-12


@pytest.mark.parametrize("nhat", [(1, 0, 0), (1, 1, 0), (1, 2, -2), (0, 0, 1)])
def test_flux_jacobian_eigenvalues_match_analytic_linearisation(kho, nhat):
    """(dU/dP)^-1 n_d dF^d/dP built by differencing the oracle's own U(P), F^d(P) has the eigenvalues
    of the analytic linearised RMHD system (kharm_inputs.modes, an independent derivation)."""
    gam = 4.0 / 3.0
    n = np.array(nhat, float) / np.linalg.norm(nhat)
    P0 = np.array([1.0, 1.0, 0, 0, 0, 1.0, 0.0, 0.0])
    h = 1e-6

    def jac(d):
        J = np.zeros((8, 8))
        for v in range(8):
            e = np.zeros(8); e[v] = h
            J[:, v] = (kho.prim_to_flux(ETA, ETA, 1.0, P0 + e, gam, d) - kho.prim_to_flux(ETA, ETA, 1.0, P0 - e, gam, d)) / (2 * h)
        return J

    A = np.linalg.solve(jac(0), sum(n[d - 1] * jac(d) for d in (1, 2, 3)))
    got = np.sort(np.linalg.eigvals(A).real)
    want = np.sort(np.linalg.eigvals(modes.linear_system(n, 1.0, 1.0, (1.0, 0, 0), gam)).real)
    assert np.allclose(got, want, atol=2e-8)
    # and the eigenvector of the fast mode is an eigenvector of the oracle's Jacobian
    lam, r = modes.eigenmode(n, modes.FAST, gamma=gam)
    assert np.abs(A @ r - lam * r).max() < 1e-7
