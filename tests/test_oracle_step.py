"""Whole-step pins of the oracle: fixed point, second-order convergence of linear MHD modes,
the analytic magnetised Bondi steady state, div B at round-off under Flux-CT, mirror symmetry,
determinism, the dt rule, and a short torus evolution."""
import os

import numpy as np
import pytest

import kharm_inputs as ki
from kharm_inputs import bondi, modes, torus
from kharm_inputs import params as kp


def _evolve(g, tend):
    t, dt, ns = 0.0, g.estimate_dt(), 0
    while t < tend * (1 - 1e-12):
        dt = min(dt, tend - t)
        nxt = g.step(dt)
        t += dt
        dt = nxt
        ns += 1
    return ns


def test_uniform_state_is_a_fixed_point(kho):
    p = ki.base_params(n1=6, n2=5, n3=4, recon=kp.RECON_WENO5)
    P0 = np.zeros((8, 4, 5, 6))
    for v, val in enumerate([1.3, 0.7, 0.2, -0.1, 0.3, 0.5, -0.4, 0.2]):
        P0[v] = val
    g = kho.Grid(p)
    g.set_prims(P0)
    dt = g.estimate_dt()
    # dt rule (S22): cfl / sum_d max|v_d|/dx_d with zone-centred speeds
    s = sum(max(abs(v) for v in kho.vchar(np.diag([-1., 1, 1, 1]), np.diag([-1., 1, 1, 1]), P0[:, 0, 0, 0], p["gamma"], d)) * n
            for d, n in ((1, 6), (2, 5), (3, 4)))
    assert abs(dt - 0.9 / s) < 1e-15
    nxt = g.step(dt)
    assert np.abs(g.get_prims() - P0).max() < 2e-15
    assert abs(nxt - dt) < 1e-13 * dt                      # face speeds of a uniform state = centred speeds
    # growth cap: a tiny step may grow by at most dt_growth_max
    assert g.step(1e-3 * dt) == pytest.approx(1.3e-3 * dt, rel=1e-14)
    pf, ff = g.get_flags()
    assert not pf.any() and not ff.any()


def _mode_errors(kho, rotated, recon, ns, thin):
    """Summed L1 error (over the components the mode moves) of config 1 after one period, per resolution.
    thin: n x 4 x 4 zones (the wave runs along x1 only); otherwise n x n x 4."""
    _, r = modes.eigenmode([1, 1, 0] / np.sqrt(2) if rotated else [1, 0, 0], modes.FAST)
    act = np.abs(r) > 0.05                                   # components the mode actually moves
    tot = []
    for n in ns:
        p = ki.config_params(1, n=(n, 4 if thin else n, 4), recon=recon)
        P0, T = modes.config1(p, rotated=rotated)
        g = kho.Grid(p, omp=True)
        g.set_prims(P0)
        assert g.divB() < 1e-13
        _evolve(g, T)
        assert g.divB() < 1e-12 and not g.get_flags()[0].any()
        tot.append(np.abs(g.get_prims() - P0).mean(axis=(1, 2, 3))[act].sum())
    return np.array(tot)


@pytest.mark.parametrize("recon", [kp.RECON_MC, kp.RECON_WENO5])
def test_linear_mode_convergence_in_the_papers_window_oblique(kho, golden, recon):
    """"the L1 norm of the difference between the computed solution and the analytic solution scale[s] with
    resolution at a power between -1.9 and -2.1" (tests/golden/paper_values.txt).  Config 1 with k = 2 pi (1,1,0), the
    kind of oblique mode the paper's suite runs: WENO5 is inside the window at every doubling from 16 zones per
    wavelength on; MC (whose limiter clips the extrema at coarse resolution) from 64 -> 128 on."""
    lo, hi = golden["convergence_slope_min"], golden["convergence_slope_max"]
    if recon == kp.RECON_WENO5:
        slopes = np.diff(np.log2(_mode_errors(kho, True, recon, (16, 32, 64), thin=False)))
        assert np.all((slopes >= lo) & (slopes <= hi)), slopes
    else:
        slopes = np.diff(np.log2(_mode_errors(kho, True, recon, (32, 64, 128), thin=False)))
        assert lo <= slopes[1] <= hi and slopes[1] < slopes[0] < -1.8, slopes       # approaches -2 from the clipped side


@pytest.mark.parametrize("recon", [kp.RECON_MC, kp.RECON_WENO5])
def test_linear_mode_convergence_in_the_papers_window_grid_aligned(kho, golden, recon):
    """The grid-aligned mode k = 2 pi (1,0,0) along B (the degenerate transverse pair of config 1) has an error
    a h^2 (1 + c h) whose measured slope enters [-2.1,-1.9] only beyond 256 zones per wavelength (measured on the oracle:
    MC -1.79, -1.88 and WENO5 -1.65, -1.83 at 64 -> 128 -> 256).  Pinned here: the slopes approach -2 monotonically and
    their Richardson extrapolation 2 s_2 - s_1 (which removes the O(h) correction) lies in the paper's window."""
    lo, hi = golden["convergence_slope_min"], golden["convergence_slope_max"]
    s1, s2 = np.diff(np.log2(_mode_errors(kho, False, recon, (64, 128, 256), thin=True)))
    assert -2.0 < s2 < s1 < -1.5, (s1, s2)
    assert lo <= 2 * s2 - s1 <= hi, (s1, s2, 2 * s2 - s1)


@pytest.mark.parametrize("rotated,recon", [(False, kp.RECON_MC), (False, kp.RECON_WENO5)])
def test_linear_mode_coarse_cubes_already_converge(kho, rotated, recon):
    """The same mode on n x n x 4 blocks at the coarse resolutions of BASELINE config 1 (16, 32, 64): a first-order
    mistake (slope -1) or a wrong wave speed (O(1) phase error, slope 0) fails this; the paper's window itself is
    enforced by the two tests above at resolutions where the scheme is in its asymptotic range."""
    tot = _mode_errors(kho, rotated, recon, (16, 32, 64), thin=False)
    assert -2.5 < np.log2(tot[2] / tot[1]) < -1.75, tot
    assert tot[2] < 3 * 2e-3 * 1e-4 * 10


def test_linear_mode_true_3d(kho):
    """Oblique k = 2 pi (1,1,1) slow mode in a full 3-D box: error falls at second order 12^3 -> 24^3."""
    errs = []
    k = 2 * np.pi * np.array([1.0, 1.0, 1.0])
    for n in (12, 24):
        p = ki.config_params(1, n=n, recon=kp.RECON_WENO5)
        P0, om = modes.mode_state(p, k, modes.SLOW, 1e-4)
        g = kho.Grid(p, omp=True)
        g.set_prims(P0)
        _evolve(g, 0.5 * 2 * np.pi / abs(om))                # half a period: compare with the analytic wave
        Pex, _ = modes.mode_state(p, k, modes.SLOW, 1e-4, t=0.5 * 2 * np.pi / abs(om))
        errs.append(np.abs(g.get_prims() - Pex).mean(axis=(1, 2, 3)).sum())
    assert errs[1] < errs[0] / 3.2 and errs[0] < 3e-5


@pytest.mark.parametrize("recon", [kp.RECON_MC, kp.RECON_WENO5])
def test_bondi_steady_state_residual_is_second_order(kho, recon):
    """Config 2: the analytic magnetised Bondi solution is a steady state, so one step from it changes
    the primitives only by the truncation error, which must fall as h^2 in the smooth interior.  Pins the
    GR fluxes, the geometric source, the connection and the inversion together against the analytic answer."""
    res = []
    for n in (32, 64, 128):
        p = ki.config_params(2, n=(n, n, 1), recon=recon)
        g = kho.Grid(p, omp=True)
        g.set_prims(bondi.config2(p), with_ghosts=True)
        P0 = g.get_prims()
        assert g.divB() < 1e-10
        dt = 0.01
        g.step(dt)
        s = slice(n // 4, 3 * n // 4)
        R = np.abs(g.get_prims() - P0)[:, 0, s, s].mean(axis=(1, 2)) / dt
        scale = np.abs(P0)[:, 0, s, s].mean(axis=(1, 2))
        res.append((R / np.maximum(scale, 1e-30))[[0, 1, 2, 5]])       # rho, u, ut1, B1 carry the solution
    slopes = np.log2(np.array(res[1:]) / np.array(res[:-1]))
    if recon == kp.RECON_WENO5:
        assert np.all(np.abs(slopes[1] + 2.0) < 0.15), slopes
    else:
        # MC switches slopes zone by zone, so single components wobble; the sum over the two refinements holds
        assert np.all(slopes.sum(axis=0) < -3.2) and np.all(slopes.sum(axis=0) > -5.5), slopes
    assert np.all(res[2] < 1e-2)       # relative rate of change per unit time at 128^2


def test_bondi_short_run_stays_near_analytic(kho):
    p = ki.config_params(2, n=(64, 64, 1))
    p["xmin"][0] = np.log(1.3)             # a few zones inside the horizon at this low resolution
    g = kho.Grid(p, omp=True)
    g.set_prims(bondi.config2(p, bsq_over_rho_at_rs=0.01), with_ghosts=True)
    P0 = g.get_prims()
    d0 = g.divB()
    _evolve(g, 5.0)
    P1 = g.get_prims()
    sl = (slice(None), 0, slice(4, -4), slice(8, None))
    err = np.abs(P1 - P0)[sl].sum(axis=(1, 2)) / np.abs(P0)[sl].sum(axis=(1, 2)).clip(1e-30)
    assert err[0] < 0.01 and err[1] < 0.02 and err[5] < 0.01
    assert abs(g.divB() - d0) < 1e-11


def test_config2_as_stated_stays_at_the_analytic_steady_state_to_t_50(kho):
    """BASELINE config 2 as it is stated ("one Bondi accretion problem"): r in [1.8, 50], sonic radius 8, monopole field
    with b^2 / rho = 1 at r_s, initialised from the analytic solution and run for 50 M; error against the analytic steady
    state outside the horizon.  Here at 32^2 and 64^2 (the stated 128^2 runs on the GPU box: tests/test_gpu_parity.py,
    where this oracle is run beside the CUDA path).  What holds, and is asserted: the run settles (t = 25 -> 50 changes
    the error by < 15 %), the settled state is the analytic one to a few per cent, and the error falls with resolution --
    by 1.8 to 4 per doubling, NOT by the 4 of a clean second-order steady state: the field is b^2 / rho ~ 30 at the inner
    edge, the outflow copy there is first order, and fast waves carry that error outwards (config 2).
    Measured 32 -> 64 -> 128: rho 0.026 / 0.014 / 0.006, u 0.16 / 0.040 / 0.022, field 0.030 / 0.011 / 0.003."""
    from parity_util import bondi_errors
    errs = {}
    for n in (32, 64):
        p = ki.config_params(2, n=(n, n, 1))
        g = kho.Grid(p, omp=True)
        g.set_prims(bondi.config2(p), with_ghosts=True)
        P0 = g.get_prims()
        d0 = g.divB()
        _evolve(g, 25.0)
        mid = bondi_errors(p, g.get_prims(), P0)
        _evolve(g, 25.0)
        errs[n] = bondi_errors(p, g.get_prims(), P0)
        assert np.all(np.abs(errs[n] / mid - 1) < 0.15), (n, mid, errs[n])        # settled, no secular drift
        assert abs(g.divB() - d0) < 1e-10
        assert (g.get_flags()[0] != 0).sum() <= (16 if n == 32 else 8)             # a handful of failed inversions at the inner edge
    e32, e64 = errs[32], errs[64]
    assert e64[0] < 0.02 and e64[1] < 0.05 and e64[3] < 0.015, e64                # rho, u, field at 64^2
    ratio = e32 / e64
    assert np.all(ratio > 1.7) and ratio[1] > 3.0 and ratio[3] > 2.4, ratio


def test_mirror_symmetry_of_a_full_step(kho):
    """x1 -> -x1 with ut1, B1 -> -ut1, -B1 maps solutions to solutions; the scheme (reconstruction L/R,
    LLF, Flux-CT signs, dt rule) must respect it to round-off."""
    n = (12, 6, 5)
    for recon in (kp.RECON_MC, kp.RECON_WENO5):
        p = ki.base_params(n1=n[0], n2=n[1], n3=n[2], gamma=5.0 / 3.0, recon=recon)
        P0 = modes.config5(p, seed=2, amp=0.05)
        g = kho.Grid(p)
        g.set_prims(P0)
        dt = g.estimate_dt()
        dt1 = g.step(dt)
        P1 = g.get_prims()
        flip = np.ones(8); flip[2] = flip[5] = -1
        Pm = (P0 * flip[:, None, None, None])[:, :, :, ::-1].copy()
        gm = kho.Grid(p)
        gm.set_prims(Pm)
        assert abs(gm.estimate_dt() - dt) < 1e-15
        dt1m = gm.step(dt)
        P1m = (gm.get_prims() * flip[:, None, None, None])[:, :, :, ::-1]
        assert np.abs(P1m - P1).max() < 5e-14 and abs(dt1m - dt1) < 1e-14


def test_determinism_and_2d_equals_thin_3d(kho):
    p = ki.config_params(5, n=(10, 8, 6), recon=kp.RECON_WENO5)
    P0 = modes.config5(p, seed=1, amp=0.02)
    outs = []
    for omp in (False, True, False):
        g = kho.Grid(p, omp=omp)
        g.set_prims(P0)
        dt = g.estimate_dt()
        for _ in range(3):
            dt = g.step(dt)
        outs.append((g.get_prims(), dt))
    assert np.array_equal(outs[0][0], outs[2][0]) and outs[0][1] == outs[2][1]      # bitwise repeatable
    assert np.array_equal(outs[0][0], outs[1][0])                                    # OpenMP build is bit-identical
    # S21: a 2-D problem (n3 = 1) is the 3-D code one zone thick; x3-invariant data in a thicker box agree
    p2 = ki.base_params(n1=10, n2=8, n3=1, gamma=5.0 / 3.0)
    p3 = ki.base_params(n1=10, n2=8, n3=4, gamma=5.0 / 3.0)
    k = 2 * np.pi * np.array([1.0, 1.0, 0.0])
    A, _ = modes.mode_state(p2, k, modes.FAST, 0.01)
    B, _ = modes.mode_state(p3, k, modes.FAST, 0.01)
    g2, g3 = kho.Grid(p2), kho.Grid(p3)
    g2.set_prims(A); g3.set_prims(B)
    dt = g3.estimate_dt()
    assert dt < g2.estimate_dt()           # the n3 = 1 direction does not enter the CFL sum
    g2.step(dt); g3.step(dt)
    assert np.abs(g3.get_prims() - g2.get_prims()).max() < 1e-15


def test_torus_short_evolution(kho):
    """Config 3 at reduced resolution: initialisation + a few steps keep div B at round-off, stay finite,
    floors only act in the atmosphere (P:415 'error metrics such as the magnetic field divergence')."""
    p = ki.config_params(3, n=(48, 32, 8))
    P0 = torus.torus_state(p, seed=1)
    g = kho.Grid(p, omp=True)
    g.set_prims(P0)
    bmax = np.abs(P0[5:]).max()
    d0 = g.divB()
    dt = g.estimate_dt()
    assert 0 < dt < 1.0
    for _ in range(4):
        dt = g.step(dt)
    P1 = g.get_prims()
    assert np.isfinite(P1).all() and P1[0].min() > 0 and P1[1].min() > 0
    assert abs(g.divB() - d0) < 1e-13 * max(1.0, d0 / 1e-16 * 1e-3) + 1e-14
    pf, ff = g.get_flags()
    dense = P0[0] > 1e-2
    assert not ff[dense].any() and (pf != 0).mean() < 0.02
    assert np.abs(P1[0][dense] / P0[0][dense] - 1).max() < 0.2          # the torus barely moves in 4 steps
