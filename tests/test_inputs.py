"""kharm_inputs: the seeded generators are deterministic and produce what DESIGN.md's recipe says."""
import numpy as np

import kharm_inputs as ki
from kharm_inputs import bondi, geometry, modes, torus
from kharm_inputs import params as kp


def test_rng_counter_based():
    a = ki.splitmix64_uniform(1, np.arange(1000))
    b = ki.splitmix64_uniform(1, np.arange(1000))
    c = ki.splitmix64_uniform(2, np.arange(1000))
    assert np.array_equal(a, b) and not np.array_equal(a, c)
    assert a.min() >= 0.0 and a.max() < 1.0 and abs(a.mean() - 0.5) < 0.05
    # order independence: a counter, not a stream
    assert ki.splitmix64_uniform(1, np.array([517]))[0] == a[517]


def test_mode_speeds_closed_forms():
    # k parallel to B0: transverse pair at v_A = sqrt(b^2/(w+b^2)), sound at c_s = sqrt(Gamma p / w)
    g = 4.0 / 3.0
    w = 1.0 + g * 1.0
    vA = np.sqrt(1.0 / (w + 1.0))
    cs = np.sqrt(g * (g - 1.0) / w)
    lam, r = modes.eigenmode([1, 0, 0], modes.FAST, gamma=g)
    assert abs(lam - vA) < 1e-12 and abs(vA - 0.5477226) < 1e-7 and abs(cs - 0.4364358) < 1e-7
    assert np.allclose(r[[3, 6]], [0.480384, -0.877058], atol=1e-6) and np.abs(np.delete(r, [3, 6])).max() < 1e-12
    lam_s, _ = modes.eigenmode([1, 0, 0], modes.SLOW, gamma=g)
    assert abs(lam_s - cs) < 1e-12
    # rotated 45 degrees: closed-form fast / Alfven / slow speeds
    n = np.array([1, 1, 0]) / np.sqrt(2)
    cth2 = 0.5
    A = vA ** 2 + cs ** 2 * (1 - vA ** 2 * (1 - cth2))
    disc = np.sqrt(A * A - 4 * cs ** 2 * vA ** 2 * cth2)
    want = [np.sqrt(0.5 * (A + disc)), vA * np.sqrt(cth2), np.sqrt(0.5 * (A - disc))]
    got = [modes.eigenmode(n, f, gamma=g)[0] for f in (modes.FAST, modes.ALFVEN, modes.SLOW)]
    assert np.allclose(got, want, atol=1e-12)
    assert np.allclose(want, [0.6231609, 0.3872983, 0.2712475], atol=1e-7)


def test_config1_and_5_shapes_and_determinism():
    p = ki.config_params(1, n=16)
    P, T = modes.config1(p)
    assert P.shape == (8, 16, 16, 16) and abs(T - 1.8257419) < 1e-6
    P2, T2 = modes.config1(p, rotated=True)
    assert abs(T2 - 1.0 / (np.sqrt(2) * 0.6231609)) < 1e-6
    p5 = ki.config_params(5, n=(12, 10, 8))
    a, b = modes.config5(p5, seed=3), modes.config5(p5, seed=3)
    assert np.array_equal(a, b) and a.shape == (8, 8, 10, 12)
    assert 1e-4 < np.abs(a[0] - 1).max() < 1e-2


def test_fm_constant_and_torus_structure():
    a = 0.9375
    ell = torus.fm_ell(a, 12.0)
    assert abs(ell - 4.281284) < 2e-6
    # Schwarzschild limit of the FM constant: l = r^{3/2}/(r-3)... as u_phi u^t: r^2 Omega (u^t)^2 = sqrt(r) r/(r-3)
    assert abs(torus.fm_ell(0.0, 12.0) - 12.0 ** 1.5 / 9.0) < 1e-12
    p = ki.config_params(3, n=(48, 32, 4))
    P = torus.torus_state(p, seed=1)
    assert P.shape == (8, 4, 32, 48) and np.isfinite(P).all()
    assert abs(P[0].max() - 1.0) < 0.05 and P[0].min() > 0 and P[1].min() > 0
    assert np.abs(P[7]).max() == 0.0 and np.abs(P[5]).max() > 0
    # seeded perturbation differs by seed but keeps everything else
    Q = torus.torus_state(p, seed=2)
    assert not np.array_equal(P[1], Q[1]) and np.array_equal(P[0], Q[0])
    # beta_min reading: max p_gas / max (b^2/2) = 100 before the perturbation
    R = torus.torus_state(p, seed=1, perturb=0.0)
    x1, x2, _ = geometry.zone_coords(p)
    X2, X1 = np.meshgrid(x2, x1, indexing="ij")
    gcov, gcon, gdet, alpha = geometry.geom(p, X1, X2)
    ut = np.moveaxis(R[2:5, 0], 0, -1)
    B = np.moveaxis(R[5:8, 0], 0, -1)
    bsq = geometry.bsq_of(gcov, gcon, alpha, ut, B)
    assert abs(((p["gamma"] - 1) * R[1, 0]).max() / (0.5 * bsq.max()) - 100.0) < 1e-9
    M = torus.torus_state(ki.config_params(4, n=(48, 32, 4)), mad=True)
    assert np.isfinite(M).all() and np.abs(M[5]).max() > 0


def test_michel_solution_is_transonic_and_conserves():
    r = np.exp(np.linspace(np.log(1.8), np.log(50.0), 200))
    g = 4.0 / 3.0
    rho, u, ur = bondi.michel(r, g, 8.0, 1.0)
    # mass flux 4 pi r^2 rho |u^r| = mdot
    assert np.allclose(4 * np.pi * r ** 2 * rho * np.abs(ur), 1.0, rtol=1e-10)
    # relativistic Bernoulli: (h u_t)^2 = h^2 (1 - 2/r + u^r^2) constant
    h = 1.0 + g * u / rho
    bern = h ** 2 * (1 - 2 / r + ur ** 2)
    assert np.allclose(bern, bern[0], rtol=1e-9)
    # monotone: density rises inwards, flow is sonic at r_s
    assert np.all(np.diff(rho) < 0)
    cs2 = g * (g - 1) * u / (rho + g * u)
    v2 = ur ** 2 / (1 - 2 / r + ur ** 2)         # radial 3-velocity^2 measured by static observers
    k = np.argmin(np.abs(r - 8.0))
    assert abs(v2[k] / cs2[k] - 1.0) < 0.05
    assert v2[0] > cs2[0] and v2[-1] < cs2[-1]


def test_config2_state():
    p = ki.config_params(2, n=(32, 32, 1))
    P = bondi.config2(p)
    assert P.shape == (8, 7, 38, 38) and np.isfinite(P).all()
    assert (P[0] > 0).all() and (P[1] > 0).all() and np.abs(P[5]).min() > 0
    assert np.abs(P[7]).max() == 0
