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
