"""Unit cases on either side of the two thresholds this build added to the extension rows:

  S29  the upwind switch of the contact-upwinded edge EMFs has a dead zone |M| <= 1e-10 (D_1 + D_2): inside it the two
       candidate gradients are averaged, outside it the one upwind of the face's mass flux M is taken;
  S26  the drift-frame floor injection keeps the velocity where B^2 <= 1e-12 (rho' + Gamma u') (no field direction to
       speak of), and adjusts the velocity along B above it.

Each test places states just below and just above the threshold and checks the behaviour that DEFINES the two branches
(not a value): averaging makes the edge EMF an odd-analytic function of a uniform drift velocity, upwinding adds a jump that
does not scale with it; below the drift cut-off the velocity is returned bit for bit, above it the momentum along the field
is what is conserved.  A build with another threshold value, or with the plain sign test, fails them.
"""
import numpy as np
import pytest

import kharm_inputs as ki
from kharm_inputs import params as kp

NG = 3
ETA = np.diag([-1.0, 1, 1, 1])


# ------------------------------------------------------------------------------------------ S29: dead zone of the upwind switch
def _emfs(kho, p, v, Bfield):
    """edge EMFs (interior) of a uniform gas (rho = 1, u = 0.5) drifting with ut^i = v in every direction through a smooth
    field: the mass flux of every face is M = rho v, the conserved density D = rho gamma, so M / (D_1 + D_2) = v / 2."""
    P = np.zeros((8, p["n3"], p["n2"], p["n1"]))
    P[0], P[1] = 1.0, 0.5
    P[2:5] = v
    P[5:8] = Bfield
    g = kho.Grid(p)
    g.set_prims(P)
    g.debug_emf()
    I = (slice(NG, -NG),) * 3
    return np.stack([g.get_emf(c)[I] for c in (1, 2, 3)])


def _odd_part_per_v(kho, p, v, B):
    return (_emfs(kho, p, v, B) - _emfs(kho, p, -v, B)) / v


def test_upwind_switch_dead_zone_sits_at_1e_minus_10_of_the_conserved_density(kho):
    p = dict(ki.config_params(5, n=(10, 8, 6), recon=kp.RECON_MC), emf=kp.EMF_UPWIND)
    x = [(np.arange(n) + 0.5) / n for n in (p["n1"], p["n2"], p["n3"])]
    X3, X2, X1 = np.meshgrid(x[2], x[1], x[0], indexing="ij")
    two_pi = 2 * np.pi
    B = np.stack([0.3 + 0.2 * np.sin(two_pi * (X2 + X3)) * np.cos(two_pi * X1),
                  0.2 + 0.2 * np.cos(two_pi * (X1 - X3)) * np.sin(two_pi * X2),
                  0.1 + 0.2 * np.sin(two_pi * (X1 + X2)) * np.cos(two_pi * X3)])
    # M / (D_1 + D_2) = v / 2: the threshold 1e-10 sits at v = 2e-10
    s_a = _odd_part_per_v(kho, p, 0.5e-10, B)         # deep inside the dead zone
    s_b = _odd_part_per_v(kho, p, 1.9e-10, B)         # just inside
    s_c = _odd_part_per_v(kho, p, 2.1e-10, B)         # just outside: upwinded
    s_d = _odd_part_per_v(kho, p, 8.0e-10, B)         # well outside
    scale = np.abs(s_a).max()
    assert scale > 1e-2                                # the EMFs do respond to the drift (E ~ B v)
    # inside: both candidates averaged whatever the sign of v -> E is odd-analytic in v, (E(v) - E(-v)) / v does not depend on v
    assert np.abs(s_b - s_a).max() < 1e-4 * scale, np.abs(s_b - s_a).max() / scale
    # outside: +v and -v pick opposite candidates; their difference J does not scale with v, so J / v dwarfs the slope
    jump_c, jump_d = np.abs(s_c - s_a).max(), np.abs(s_d - s_a).max()
    assert jump_c > 1e4 * scale and jump_d > 1e3 * scale, (jump_c / scale, jump_d / scale)
    # and it is the SAME jump J on both sides of 2.1e-10 -> 8e-10 (a switch, not a ramp): J = (s - s_a) v is constant
    J_c, J_d = (s_c - s_a) * 2.1e-10, (s_d - s_a) * 8.0e-10
    assert np.abs(J_c - J_d).max() < 1e-6 * np.abs(J_c).max()


def test_arithmetic_emf_has_no_switch_at_all(kho):
    """Control: the four-point average (KH_EMF_ARITHMETIC) is odd-analytic in the drift for every v -- the jump above belongs
    to the upwind switch alone."""
    p = dict(ki.config_params(5, n=(10, 8, 6), recon=kp.RECON_MC), emf=kp.EMF_ARITHMETIC)
    x = [(np.arange(n) + 0.5) / n for n in (p["n1"], p["n2"], p["n3"])]
    X3, X2, X1 = np.meshgrid(x[2], x[1], x[0], indexing="ij")
    B = np.stack([0.3 + 0.2 * np.sin(2 * np.pi * (X2 + X3)), 0.2 + 0.2 * np.cos(2 * np.pi * (X1 - X3)), 0.1 + 0.2 * np.sin(2 * np.pi * (X1 + X2))])
    s_a, s_d = _odd_part_per_v(kho, p, 0.5e-10, B), _odd_part_per_v(kho, p, 8.0e-10, B)
    assert np.abs(s_d - s_a).max() < 1e-4 * np.abs(s_a).max()


# ------------------------------------------------------------------------------------------ S26: cut-off of the drift frame
@pytest.mark.parametrize("curved", [False, True])
def test_drift_frame_cutoff_sits_at_1e_minus_12_of_the_enthalpy(kho, curved):
    if curved:
        gcov, gcon, _, _ = kho.metric(kho.make_params(ki.config_params(3)), 2.5, 0.5)
        x1, x2 = 2.5, 0.5
        base = ki.config_params(3)
    else:
        gcov, gcon, x1, x2 = ETA, ETA, 0.5, 0.5
        base = ki.config_params(5)
    pd = kho.make_params(dict(base, floor_frame=kp.FRAME_DRIFT))
    pf = kho.make_params(dict(base, floor_frame=kp.FRAME_FLUID))
    g3 = gcov[1:, 1:]
    bdir = np.array([0.6, -0.3, 0.7])
    bdir = bdir / np.sqrt(bdir @ g3 @ bdir)                       # unit vector along the field
    ut = 0.5 * bdir + 0.1 * np.array([0.2, 0.5, -0.1]) / np.sqrt(np.diag(g3))      # mostly along B
    hydro = [1e-22, 1e-24]                                        # far below every floor: the floors raise rho and u
    Pfl, _ = kho.floors(pf, gcov, gcon, x1, x2, np.concatenate([hydro, ut, 1e-30 * bdir]))
    w_new = Pfl[0] + pd.gamma * Pfl[1]                            # rho' + Gamma u' (the geometric floors: B is negligible)
    for s, live in ((0.25, False), (0.9, False), (1.1, True), (4.0, True)):
        B = np.sqrt(s * 1e-12 * w_new) * bdir                     # B^2 = s x 1e-12 (rho' + Gamma u')
        P = np.concatenate([hydro, ut, B])
        Pd, f = kho.floors(pd, gcov, gcon, x1, x2, P)
        assert f != 0 and Pd[0] == Pfl[0] and Pd[1] == Pfl[1]     # same limits as the fluid frame
        if not live:
            assert np.array_equal(Pd[2:5], ut), s                # below the cut-off: velocity returned bit for bit
        else:
            # above: the momentum along the field is conserved although w grew by ~20 orders of magnitude, so the
            # velocity along B all but vanishes, and the part perpendicular to B is what remains
            gam_old = np.sqrt(1 + ut @ g3 @ ut)
            v_old = ut / gam_old
            v_perp = v_old - (v_old @ g3 @ bdir) * bdir
            gam_new = np.sqrt(1 + Pd[2:5] @ g3 @ Pd[2:5])
            v_new = Pd[2:5] / gam_new
            assert abs(v_new @ g3 @ bdir) < 1e-10 * abs(v_old @ g3 @ bdir), s     # ~ w_old / w_new of the old parallel velocity
            assert np.abs(v_new - v_perp).max() < 1e-10 * np.abs(v_old).max(), s
            assert not np.allclose(Pd[2:5], ut, rtol=1e-3), s
