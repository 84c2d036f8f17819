"""Pins of the oracle's face-centred constrained transport (S28).

  * the face-centred divergence stays at round-off over a run, for a field that starts divergence-free (Stokes) --
    and a non-solenoidal face field keeps exactly the divergence it started with (the update is a pure circulation);
  * Toth (2000): with the arithmetic four-point EMF the zone-centred mean of the face field evolves exactly as under
    Flux-CT, so a step of either transport from consistent data gives the same primitives to round-off;
  * the zone-centred field the scheme uses is the mean of the two face values over sqrt(-g); axis faces carry no flux.
"""
import numpy as np

import kharm_inputs as ki
from kharm_inputs import facefield, modes, torus
from kharm_inputs import params as kp

NG = 3


def _grids(kho, p, P0, faces):
    out = []
    for tr in (kp.B_FLUX_CT, kp.B_FACE_CT):
        g = kho.Grid(dict(p, transport=tr))
        if tr == kp.B_FACE_CT:
            g.set_prims(P0)
            g.set_face_B(*faces)
        out.append(g)
    # the Flux-CT grid starts from the zone-centred field the face grid derived
    Pc = out[1].get_prims()
    out[0].set_prims(Pc)
    return out


def test_face_divergence_and_equivalence_with_flux_ct_minkowski(kho):
    p = ki.config_params(5, n=(12, 10, 8), recon=kp.RECON_WENO5)
    P0 = modes.config5(p, seed=2, amp=1e-2)
    faces = facefield.face_from_potential(p, *facefield.periodic_potential(p, seed=3, amp=5e-2))
    g_flux, g_face = _grids(kho, p, P0, faces)
    assert g_face.divB_face() < 1e-13
    f = g_face.get_face_B()
    Pc = g_face.get_prims()
    I = (slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
    assert np.allclose(Pc[5], 0.5 * (f[0][I] + f[0][NG:-NG, NG:-NG, NG + 1:-NG + 1]), rtol=0, atol=1e-16)
    dt = g_flux.estimate_dt()
    for _ in range(5):
        d1, d2 = g_flux.step(dt), g_face.step(dt)
        assert abs(d1 / d2 - 1) < 1e-12
        dt = d1
    a, b = g_flux.get_prims(), g_face.get_prims()
    for v in range(8):
        assert np.abs(a[v] - b[v]).max() <= 1e-12 * max(np.abs(a[v]).max(), 1e-3), v
    assert g_face.divB_face() < 1e-12
    # periodic: face 0 and face N are the same face and must hold the same number
    f = g_face.get_face_B()
    assert np.allclose(f[0][NG:-NG, NG:-NG, NG], f[0][NG:-NG, NG:-NG, NG + p["n1"]], rtol=0, atol=1e-14)
    assert np.allclose(f[2][NG, NG:-NG, NG:-NG], f[2][NG + p["n3"], NG:-NG, NG:-NG], rtol=0, atol=1e-14)


def test_a_non_solenoidal_face_field_keeps_its_divergence_exactly(kho):
    p = dict(ki.config_params(5, n=(8, 8, 8)), transport=kp.B_FACE_CT)
    P0 = modes.config5(p, seed=1, amp=1e-2)
    rng = np.random.default_rng(0)
    shape = (p["n3"] + 6, p["n2"] + 6, p["n1"] + 6)
    faces = [0.01 * rng.normal(size=shape) for _ in range(3)]
    for d, ax in enumerate((2, 1, 0)):                         # make it periodic: face N := face 0
        sl_lo = [slice(None)] * 3; sl_hi = [slice(None)] * 3
        sl_lo[ax] = NG; sl_hi[ax] = NG + (p["n1"], p["n2"], p["n3"])[d]
        faces[d][tuple(sl_hi)] = faces[d][tuple(sl_lo)]
    g = kho.Grid(p)
    g.set_prims(P0); g.set_face_B(*faces)

    def div(f):
        I = (slice(NG, -NG),) * 3
        dx = [1.0 / 8] * 3
        return ((f[0][NG:-NG, NG:-NG, NG + 1:-NG + 1] - f[0][I]) / dx[0] + (f[1][NG:-NG, NG + 1:-NG + 1, NG:-NG] - f[1][I]) / dx[1]
                + (f[2][NG + 1:-NG + 1, NG:-NG, NG:-NG] - f[2][I]) / dx[2])
    d0 = div(g.get_face_B())
    dt = g.estimate_dt()
    for _ in range(3):
        dt = g.step(dt)
    d1 = div(g.get_face_B())
    assert np.abs(d0).max() > 0.01 and np.abs(d1 - d0).max() <= 1e-12 * np.abs(d0).max()


def test_torus_face_ct_matches_flux_ct_and_axis_faces_stay_empty(kho):
    p = ki.config_params(3, n=(24, 16, 4))
    P0 = torus.torus_state(p, seed=2)
    faces = facefield.face_from_potential(p, *facefield.axisymmetric_loop_potential(p, amp=2e-3, x1c=2.3))
    g_flux, g_face = _grids(kho, p, P0, faces)
    assert g_face.divB_face() < 1e-15
    dt = g_flux.estimate_dt()
    for _ in range(3):
        d1, d2 = g_flux.step(dt), g_face.step(dt)
        dt = d1
    a, b = g_flux.get_prims(), g_face.get_prims()
    assert np.array_equal(g_flux.get_flags()[0], g_face.get_flags()[0])
    for v in range(8):
        assert np.abs(a[v] - b[v]).max() <= 1e-11 * max(np.abs(a[v]).max(), 1e-12), v
    f = g_face.get_face_B()
    for jj in (NG, NG + p["n2"]):                                 # theta = 0, pi faces: no EMF circulates around them
        assert np.array_equal(f[1][NG:-NG, jj, NG:-NG], faces[1][NG:-NG, jj, NG:-NG])
        assert np.abs(f[1][NG:-NG, jj, NG:-NG]).max() < 1e-30
    assert g_face.divB_face() < 1e-14


# ------------------------------------------------------------------------------------------ upwinded edge EMFs (S29)
def _one_d_state(p, d, seed):
    """A state that varies only along direction d (1..3), moving along d, with all three field components."""
    rng = np.random.default_rng(seed)
    n = (p["n1"], p["n2"], p["n3"])[d - 1]
    x = (np.arange(n) + 0.5) / n
    prof = lambda a, b: a + b * np.sin(2 * np.pi * x + rng.uniform(0, 6.28))
    shp = [1, 1, 1]; shp[3 - d] = n
    P = np.zeros((8, p["n3"], p["n2"], p["n1"]))
    P[0] = prof(1.0, 0.3).reshape(shp); P[1] = prof(0.5, 0.2).reshape(shp)
    P[1 + d] = prof(0.1, 0.4).reshape(shp)                       # velocity along d, changing sign
    for e in (1, 2, 3):
        P[4 + e] = 0.3 if e == d else prof(0.2, 0.5).reshape(shp)
    return P


def test_upwinded_emf_reduces_to_the_face_value_for_grid_aligned_flow(kho):
    """The design condition of the contact-upwind EMF: plane-parallel flow along a grid direction must see the
    one-dimensional face value at the edge (no multidimensional averaging left)."""
    p = dict(ki.config_params(5, n=(12, 10, 8), recon=kp.RECON_WENO5), emf=kp.EMF_UPWIND)
    I = (slice(NG, -NG),) * 3
    for d in (1, 2, 3):
        g = kho.Grid(p)
        g.set_prims(_one_d_state(p, d, seed=d))
        g.debug_emf()
        F, _ = g.get_flux(d)                                       # raw face fluxes of direction d
        a, b = d % 3 + 1, (d + 1) % 3 + 1                          # (d, a, b) cyclic
        e_b, e_a = g.get_emf(b), g.get_emf(a)
        # eps_b = F^d[B^a] ... with (b; d, a) cyclic: eps_b = F^d[B^a];  eps_a = -F^d[B^b] with (a; b, d) cyclic
        assert np.abs(e_b[I] - F[4 + a][I]).max() <= 1e-14 * np.abs(F[4 + a][I]).max(), d
        assert np.abs(e_a[I] + F[4 + b][I]).max() <= 1e-14 * np.abs(F[4 + b][I]).max(), d
        # the arithmetic average does NOT have this property (it mixes in the zone-centred values)
        g0 = kho.Grid(dict(p, emf=kp.EMF_ARITHMETIC))
        g0.set_prims(_one_d_state(p, d, seed=d)); g0.debug_emf()
        assert np.abs(g0.get_emf(b)[I] - F[4 + a][I]).max() > 1e-4


def test_upwinded_emf_uniform_state_and_face_divergence(kho):
    from kharm_inputs import facefield
    p = dict(ki.config_params(5, n=(8, 8, 8)), emf=kp.EMF_UPWIND)
    P0 = np.zeros((8, 8, 8, 8)); P0[0] = 1.0; P0[1] = 0.7; P0[2] = 0.3; P0[3] = -0.2; P0[4] = 0.1; P0[5] = 0.4; P0[6] = -0.3; P0[7] = 0.2
    g = kho.Grid(p); g.set_prims(P0); g.debug_emf()
    gamma = np.sqrt(1 + 0.3 ** 2 + 0.2 ** 2 + 0.1 ** 2)
    v = np.array([0.3, -0.2, 0.1]) / gamma; B = np.array([0.4, -0.3, 0.2])
    I = (slice(NG, -NG),) * 3
    for c in range(3):
        a, b = (c + 1) % 3, (c + 2) % 3
        assert np.allclose(g.get_emf(c + 1)[I], B[b] * v[a] - B[a] * v[b], rtol=1e-13, atol=1e-15)
    # a run: the face divergence stays at round-off, and the result differs from the arithmetic-EMF run
    q = ki.config_params(5, n=(12, 10, 8), recon=kp.RECON_WENO5)
    P0 = modes.config5(q, seed=2, amp=5e-2)
    faces = facefield.face_from_potential(q, *facefield.periodic_potential(q, seed=3, amp=5e-2))
    res = []
    for emf in (kp.EMF_ARITHMETIC, kp.EMF_UPWIND):
        g = kho.Grid(dict(q, transport=kp.B_FACE_CT, emf=emf))
        g.set_prims(P0); g.set_face_B(*faces)
        dt = g.estimate_dt()
        for _ in range(5):
            dt = g.step(dt)
        assert g.divB_face() < 1e-12
        res.append(g.get_prims())
    d = np.abs(res[0][5:] - res[1][5:]).max()
    assert 1e-9 < d < 0.2 * np.abs(res[0][5:]).max()          # a different, but not a wildly different, discretisation


def test_upwinded_emf_keeps_second_order_convergence_of_a_rotated_mode(kho):
    errs = []
    for n in (16, 32):
        p = dict(ki.config_params(1, n=(n, n, 4)), emf=kp.EMF_UPWIND)
        P0, T = modes.config1(p, rotated=True)
        g = kho.Grid(p, omp=True); g.set_prims(P0)
        dt, t = g.estimate_dt(), 0.0
        while t < T * (1 - 1e-12):
            dt = min(dt, T - t); t += dt
            dt = g.step(dt)
        errs.append(np.abs(g.get_prims() - P0).mean(axis=(1, 2, 3)).max())
    slope = np.log2(errs[0] / errs[1])
    assert 1.7 < slope < 2.4, (errs, slope)


# ------------------------------------------------------------------------------------------ un-upwinded Gardiner-Stone EMF (S30)
def test_centred_emf_design_condition_uniform_state_and_difference_from_the_other_two(kho):
    """KH_EMF_CENTRED = 1/2 (faces) - 1/4 (centres): (1) plane-parallel flow along each grid direction sees the
    one-dimensional face value at the edge (the design condition the arithmetic average fails); (2) a uniform state gives
    the zone-centred value; (3) it does not depend on the direction of the flow the way the upwinded scheme does: for
    grid-aligned 1-D flow all three agree with (1) except the arithmetic one, for a 3-D state all three differ."""
    p0 = ki.config_params(5, n=(12, 10, 8), recon=kp.RECON_WENO5)
    I = (slice(NG, -NG),) * 3
    for d in (1, 2, 3):
        g = kho.Grid(dict(p0, emf=kp.EMF_CENTRED))
        g.set_prims(_one_d_state(p0, d, seed=d))
        g.debug_emf()
        F, _ = g.get_flux(d)
        a, b = d % 3 + 1, (d + 1) % 3 + 1
        assert np.abs(g.get_emf(b)[I] - F[4 + a][I]).max() <= 1e-14 * np.abs(F[4 + a][I]).max(), d
        assert np.abs(g.get_emf(a)[I] + F[4 + b][I]).max() <= 1e-14 * np.abs(F[4 + b][I]).max(), d
    P0 = np.zeros((8, 8, 10, 12)); P0[0] = 1.0; P0[1] = 0.7; P0[2] = 0.3; P0[3] = -0.2; P0[4] = 0.1; P0[5] = 0.4; P0[6] = -0.3; P0[7] = 0.2
    g = kho.Grid(dict(p0, emf=kp.EMF_CENTRED)); g.set_prims(P0); g.debug_emf()
    gamma = np.sqrt(1 + 0.3 ** 2 + 0.2 ** 2 + 0.1 ** 2)
    v = np.array([0.3, -0.2, 0.1]) / gamma; B = np.array([0.4, -0.3, 0.2])
    for c in range(3):
        a, b = (c + 1) % 3, (c + 2) % 3
        assert np.allclose(g.get_emf(c + 1)[I], B[b] * v[a] - B[a] * v[b], rtol=1e-13, atol=1e-15)
    # a genuinely 3-D state: three different discretisations; the centred one is the mean of the upwinded scheme's two
    # one-sided choices, so it lies between "upwinded with the flow" and "upwinded against it" (the flow reversed)
    P3 = modes.config5(p0, seed=4, amp=5e-2)
    e = {}
    for kind in (kp.EMF_ARITHMETIC, kp.EMF_UPWIND, kp.EMF_CENTRED):
        g = kho.Grid(dict(p0, emf=kind)); g.set_prims(P3); g.debug_emf()
        e[kind] = np.stack([g.get_emf(c)[I] for c in (1, 2, 3)])
    scale = np.abs(e[kp.EMF_ARITHMETIC]).max()
    assert np.abs(e[kp.EMF_CENTRED] - e[kp.EMF_ARITHMETIC]).max() > 1e-6 * scale
    assert np.abs(e[kp.EMF_CENTRED] - e[kp.EMF_UPWIND]).max() > 1e-6 * scale


def test_centred_emf_keeps_divergence_and_second_order(kho):
    from kharm_inputs import facefield
    q = ki.config_params(5, n=(12, 10, 8), recon=kp.RECON_WENO5)
    P0 = modes.config5(q, seed=2, amp=5e-2)
    faces = facefield.face_from_potential(q, *facefield.periodic_potential(q, seed=3, amp=5e-2))
    g = kho.Grid(dict(q, transport=kp.B_FACE_CT, emf=kp.EMF_CENTRED))
    g.set_prims(P0); g.set_face_B(*faces)
    dt = g.estimate_dt()
    for _ in range(5):
        dt = g.step(dt)
    assert g.divB_face() < 1e-12
    g = kho.Grid(dict(q, emf=kp.EMF_CENTRED)); g.set_prims(P0)                 # Flux-CT transport: corner divergence
    d0 = g.divB(); dt = g.estimate_dt()
    for _ in range(5):
        dt = g.step(dt)
    assert abs(g.divB() - d0) < 1e-12
    errs = []
    for n in (16, 32):
        p = dict(ki.config_params(1, n=(n, n, 4)), emf=kp.EMF_CENTRED)
        Pm, T = modes.config1(p, rotated=True)
        g = kho.Grid(p, omp=True); g.set_prims(Pm)
        dt, t = g.estimate_dt(), 0.0
        while t < T * (1 - 1e-12):
            dt = min(dt, T - t); t += dt
            dt = g.step(dt)
        errs.append(np.abs(g.get_prims() - Pm).mean(axis=(1, 2, 3)).max())
    slope = np.log2(errs[0] / errs[1])
    assert 1.7 < slope < 2.4, (errs, slope)


def test_face_ct_equals_flux_ct_for_any_emf_and_option_mix(kho):
    """The zone-centred mean of the face field obeys the Flux-CT update for ANY edge EMFs (the identity is algebra on the
    EMF arrays), so the two transports must agree to round-off whatever the EMF kind, inverter, floor frame or FOFC."""
    rng = np.random.default_rng(9)
    for trial in range(6):
        n = (int(rng.integers(8, 20)), int(rng.integers(6, 14)), int(rng.integers(1, 6)))
        opts = dict(recon=int(rng.integers(0, 2)), inverter=int(rng.integers(0, 2)), floor_frame=int(rng.integers(0, 3)),
                    fofc=int(rng.integers(0, 2)), emf=int(rng.integers(0, 3)))
        p = dict(ki.config_params(3, n=n), **opts)
        P0 = torus.torus_state(p, seed=trial)
        faces = facefield.face_from_potential(p, *facefield.axisymmetric_loop_potential(p, amp=2e-3, x1c=2.3))
        g_flux, g_face = _grids(kho, p, P0, faces)
        dt = g_flux.estimate_dt()
        for _ in range(2):
            d1, d2 = g_flux.step(dt), g_face.step(dt)
            dt = d1
        a, b = g_flux.get_prims(), g_face.get_prims()
        assert np.array_equal(g_flux.get_flags()[0], g_face.get_flags()[0]), opts
        for v in range(8):
            assert np.abs(a[v] - b[v]).max() <= 1e-10 * max(np.abs(a[v]).max(), 1e-12), (opts, v)
        assert g_face.divB_face() < 1e-13
