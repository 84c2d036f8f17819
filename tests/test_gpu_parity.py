"""GPU parity: the CUDA path (through the C ABI of include/kharm.h) against the CPU oracle on the same
seeded inputs.  Bars (BASELINE.json north_star): max relative difference 1e-10 per primitive after one
step (metric: tests/parity_util.py, S23), 1e-8 in L1 after a run, identical U->P flags;
index / copy work (ghost fills) bit-exact."""
import os

import numpy as np
import pytest

import kharm_inputs as ki
from kharm_inputs import bondi, modes, torus
from kharm_inputs import params as kp

from parity_util import TOL_ONE_STEP, TOL_RUN_L1, conditioning, l1_diff, oracle_sensitivity, rel_diff

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def kh():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2408_01361_b200 as m
    m.lib()
    return m


def _both(kh, kho, p, P0, with_ghosts=False, omp=True):
    gg = kh.Grid(p)
    go = kho.Grid(p, omp=omp)
    gg.set_prims(P0, with_ghosts=with_ghosts)
    go.set_prims(P0, with_ghosts=with_ghosts)
    return gg, go


# Allowance of the one-step bar in zones where the scheme itself amplifies round-off (S23): the two sides evaluate
# algebraically identical formulas in different association and contraction, so each of the ~30 rounded operations that
# feed a zone's energy equation (7 face-flux components, source and U(P_i) per sub-step, the inversion's residual) may
# differ by an ulp of its own operand; K_ROUNDINGS of them, amplified by the zone's conditioning number eps (rho + b^2) / u,
# is the bar on u there.  S23c (fuzz cases): where the oracle itself turns 1-ulp input noise into more than a tenth of the
# bar (parity_util.oracle_sensitivity), K_SENS times that measured sensitivity is the bar -- for any primitive.
K_ROUNDINGS = 30.0
K_SENS = 10.0
MAX_RELAXED_FRACTION = 0.5      # no test may judge more than half of its zones on a relaxed bar (asserted)


def _report(label, worst, relaxed, zones, tol):
    """Append one row to the parity report (KH_PARITY_REPORT=<path>.md; profiles/parity_r02.md is such a file)."""
    path = os.environ.get("KH_PARITY_REPORT")
    if not path:
        return
    new = not os.path.exists(path)
    with open(path, "a") as f:
        if new:
            f.write("| case | zones | bar | worst rho | worst u | worst ut1 | worst ut2 | worst ut3 | worst B1 | worst B2 | worst B3 |"
                    " zones on a relaxed bar: rho | u | ut |\n|" + "---|" * 14 + "\n")
        f.write("| %s | %d | %.0e | %s | %d | %d | %d |\n" % (label, zones, tol, " | ".join("%.2e" % w for w in worst),
                                                             relaxed[0], relaxed[1], relaxed[2]))


def _assert_step_parity(p, got, ref, pf_g, pf_o, label="", tol=TOL_ONE_STEP, sens=None):
    """S23: per-zone, per-primitive relative difference <= tol, flags identical.  Relaxed bars:
      u             : K_ROUNDINGS eps (rho + b^2) / u, the conditioning of the internal energy in U -> P (S16); u ONLY --
                      rho, ut^i and B^i stay on the flat bar;
      any primitive : K_SENS x the oracle's measured sensitivity to 1-ulp input noise, where `sens` is given (S23c).
    Returns the worst difference per primitive; the number of zones judged on a relaxed bar is bounded and reported."""
    assert np.array_equal(pf_g, pf_o), "%s: U->P flags differ in %d zones" % (label, (pf_g != pf_o).sum())
    d = rel_diff(p, got, ref)
    allow = np.full(d.shape, tol)
    allow[1] = np.maximum(tol, K_ROUNDINGS * conditioning(p, ref, p["gamma"]))
    if sens is not None:
        allow = np.maximum(allow, K_SENS * sens)
    worst = d.max(axis=(1, 2, 3))
    bad = d > allow
    zones = d[0].size
    relaxed = [int((allow[0] > tol).sum()), int((allow[1] > tol).sum()), int((allow[2:5] > tol).any(axis=0).sum())]
    _report(label, worst, relaxed, zones, tol)
    assert not bad.any(), "%s: max rel diff per primitive %s (bar %g); %d zones over; worst excess %s" % (
        label, worst, tol, bad.any(axis=0).sum(), (d / allow).max(axis=(1, 2, 3)))
    assert max(relaxed) <= MAX_RELAXED_FRACTION * zones, "%s: %s of %d zones judged on a relaxed bar" % (label, relaxed, zones)
    return worst


# ------------------------------------------------------------------------------------------ geometry (K1)
@pytest.mark.parametrize("cfg,n", [(1, (9, 7, 5)), (2, (40, 24, 1)), (3, (48, 40, 4))])
def test_geometry_tables(kh, kho, cfg, n):
    p = ki.config_params(cfg, n=n)
    if cfg == 1:
        p["coords"] = kp.KS; p["a"] = 0.5; p["xmin"] = [1.5, 0.4, 0.0]; p["xmax"] = [3.3, 2.8, 6.0]
        p["bc"] = [kp.BC_OUTFLOW] * 4 + [kp.BC_PERIODIC] * 2
    gg, go = kh.Grid(p), kho.Grid(p)
    # rows beyond a polar axis are never read (S10); there theta passes through pi and sin(theta) is ill-conditioned
    rows = slice(3, p["n2"] + 4) if p["bc"][2] == kp.BC_POLAR else slice(None)
    for loc in range(4):
        a, b = gg.get_geom(loc), go.get_geom(loc)
        for x, y, name in zip(a, b, ("gcov", "gcon", "gdet", "alpha")):
            x, y = x[rows], y[rows]
            scale = np.abs(y).max(axis=(-1, -2), keepdims=True) if y.ndim == 4 else np.abs(y)
            err = np.abs(x - y) / np.maximum(scale, 1e-300)
            assert err.max() < 5e-13, (loc, name, err.max())
    ca, cb = gg.get_conn()[rows], go.get_conn()[rows]
    err = np.abs(ca - cb) / np.maximum(np.abs(cb).max(axis=(-1, -2, -3), keepdims=True), 1e-300)
    assert err.max() < 5e-12, err.max()


# ------------------------------------------------------------------------------------------ ghost fills (K7), bit-exact
def test_ghost_fills_bit_exact(kh, kho):
    rng = np.random.default_rng(1)
    cases = [ki.base_params(n1=5, n2=4, n3=3), ki.base_params(n1=5, n2=4, n3=3, bc=[kp.BC_OUTFLOW] * 6),
             ki.config_params(3, n=(6, 5, 2)), ki.config_params(2, n=(7, 6, 1)),
             ki.base_params(n1=4, n2=4, n3=1, bc=[kp.BC_OUTFLOW, kp.BC_FIXED, kp.BC_PERIODIC, kp.BC_PERIODIC, kp.BC_PERIODIC, kp.BC_PERIODIC])]
    for p in cases:
        shp = (8, p["n3"], p["n2"], p["n1"])
        P0 = rng.normal(size=shp)
        if kp.BC_FIXED in p["bc"]:
            # a FIXED side needs its ghost layers from a with_ghosts load first: until then the library refuses
            # (the fixed layers would silently be vacuum)
            gg, go = kh.Grid(p), kho.Grid(p, omp=True)
            with pytest.raises(kh.KharmError):
                gg.set_prims(P0)
            with pytest.raises(kh.KharmError):
                gg.step(1e-3)
            first = rng.normal(size=(8, p["n3"] + 6, p["n2"] + 6, p["n1"] + 6))
            for g in (gg, go):
                g.set_prims(first, with_ghosts=True)
                g.set_prims(P0)
        else:
            gg, go = _both(kh, kho, p, P0)
        a, b = gg.get_prims(with_ghosts=True), go.get_prims(with_ghosts=True)
        # outflow ghosts rescale B by a ratio of tabulated sqrt(-g): identical up to the tables' own rounding
        assert np.array_equal(a[:5], b[:5])
        assert np.allclose(a[5:], b[5:], rtol=1e-12, atol=0)
        full = rng.normal(size=(8, p["n3"] + 6, p["n2"] + 6, p["n1"] + 6))
        gg.set_prims(full, with_ghosts=True); go.set_prims(full, with_ghosts=True)
        a, b = gg.get_prims(with_ghosts=True), go.get_prims(with_ghosts=True)
        assert np.array_equal(a[:5], b[:5]) and np.allclose(a[5:], b[5:], rtol=1e-12, atol=0)
        assert np.array_equal(gg.get_prims(), go.get_prims())


# ------------------------------------------------------------------------------------------ stages after one step
@pytest.mark.parametrize("recon", [kp.RECON_MC, kp.RECON_WENO5])
def test_stage_parity_fluxes_emf_ctop(kh, kho, recon):
    p = ki.config_params(3, n=(40, 36, 6), recon=recon)
    P0 = torus.torus_state(p, seed=1)
    gg, go = _both(kh, kho, p, P0)
    dt = go.estimate_dt()
    assert abs(gg.estimate_dt() / dt - 1) < 1e-12
    gg.step(dt); go.step(dt)
    I = (slice(3, -3), slice(3, -3), slice(3, -3))
    for d in (1, 2, 3):
        Fg, cg = gg.get_flux(d)
        Fo, co = go.get_flux(d)
        assert np.allclose(cg[I], co[I], rtol=1e-11, atol=1e-14), d
        for v in range(8):
            scale = np.abs(Fo[v][I]).max() + 1e-300
            assert np.abs(Fg[v][I] - Fo[v][I]).max() <= 1e-11 * scale, (d, v)
        eg, eo = gg.get_emf(d), go.get_emf(d)
        assert np.abs(eg[I] - eo[I]).max() <= 1e-11 * (np.abs(eo[I]).max() + 1e-300), d


# ------------------------------------------------------------------------------------------ one step, all configs (small)
def _one_step_case(kh, kho, p, P0, with_ghosts=False, label=""):
    gg, go = _both(kh, kho, p, P0, with_ghosts)
    dt = go.estimate_dt()
    assert abs(gg.estimate_dt() / dt - 1) < 1e-12
    n_g, n_o = gg.step(dt), go.step(dt)
    assert abs(n_g / n_o - 1) < 1e-11
    pf_g, ff_g = gg.get_flags()
    pf_o, ff_o = go.get_flags()
    worst = _assert_step_parity(p, gg.get_prims(), go.get_prims(), pf_g, pf_o, label)
    assert (ff_g != ff_o).mean() < 1e-3          # floor decisions are thresholds on fp64 values: a marginal zone may flip
    dg_, do_ = gg.divB(), go.divB()               # both are round-off noise of O(eps |B| / dx): compare magnitudes
    assert abs(dg_ - do_) <= 0.25 * max(do_, dg_) + 1e-13, (dg_, do_)
    cg, co = gg.get_cons(), go.get_cons()
    assert np.abs(cg - co).max() <= 1e-9 * np.abs(co).max()
    return worst, gg, go


@pytest.mark.parametrize("recon", [kp.RECON_MC, kp.RECON_WENO5])
@pytest.mark.parametrize("n", [(32, 32, 32), (37, 13, 5), (130, 3, 2), (3, 3, 3), (16, 16, 1)])
def test_one_step_minkowski_modes(kh, kho, n, recon):
    p = ki.config_params(5, n=n, recon=recon)
    P0 = modes.config5(p, seed=1, amp=1e-3 if min(n) > 3 else 1e-2)
    _one_step_case(kh, kho, p, P0, label="cfg5 %s" % (n,))


def test_one_step_config1(kh, kho):
    p = ki.config_params(1, n=32)
    P0, _ = modes.config1(p, rotated=True)
    _one_step_case(kh, kho, p, P0, label="cfg1")


@pytest.mark.parametrize("recon", [kp.RECON_MC, kp.RECON_WENO5])
def test_one_step_bondi(kh, kho, recon):
    p = ki.config_params(2, recon=recon)          # full 128 x 128 x 1
    _one_step_case(kh, kho, p, bondi.config2(p), with_ghosts=True, label="cfg2")


@pytest.mark.parametrize("cfg,n", [(3, (64, 48, 8)), (4, (72, 40, 6)), (3, (33, 17, 3))])
def test_one_step_torus(kh, kho, cfg, n):
    p = ki.config_params(cfg, n=n)
    P0 = torus.torus_state(p, mad=(cfg == 4), seed=2)
    _one_step_case(kh, kho, p, P0, label="cfg%d" % cfg)


def test_one_step_mad_stress_failures_and_fixups(kh, kho):
    """Config 4 stress variant: strongly magnetised cold patches force inversion failures, floors and fix-ups."""
    p = ki.config_params(4, n=(72, 40, 8))
    P0 = torus.torus_state(p, mad=True, seed=3, stress=True, stress_fraction=0.02)
    worst, gg, go = _one_step_case(kh, kho, p, P0, label="cfg4-stress")
    pf, ff = go.get_flags()
    npf, nff = gg.count_flags()
    assert (ff != 0).sum() > 50                                   # floors really acted
    assert npf == (pf != 0).sum()                                 # device counter of the last sub-step = oracle's count
    print("stress: pflag zones", (pf != 0).sum(), "fflag zones", (ff != 0).sum(), "worst", worst)


def test_fixup_hook_parity(kh, kho):
    p = ki.config_params(3, n=(20, 16, 6))
    P0 = torus.torus_state(p, seed=1)
    gg, go = _both(kh, kho, p, P0)
    rng = np.random.default_rng(3)
    pf = (rng.uniform(size=(6 + 6, 16 + 6, 20 + 6)) < 0.15).astype(np.int32) * 5
    gg.debug_fixup(pf); go.debug_fixup(pf)
    a, b = gg.get_prims(), go.get_prims()
    assert np.abs(a - b).max() <= 1e-13 * np.abs(b).max() and np.allclose(a, b, rtol=1e-12, atol=1e-300)
    assert np.array_equal(gg.get_flags()[1], go.get_flags()[1])
    # the CUDA fix-up also refreshes the ghost images of the zones it fixed (the second fill of the sub-step, S22);
    # the oracle's hook stops before that fill, so run it to bring both sides to the same point of the sequence
    go.fill_ghosts()
    assert np.array_equal(gg.get_prims(with_ghosts=True)[:5], go.get_prims(with_ghosts=True)[:5]) or \
        np.allclose(gg.get_prims(with_ghosts=True)[:5], go.get_prims(with_ghosts=True)[:5], rtol=1e-12, atol=1e-300)
    allbad = np.ones_like(pf)
    gg.debug_fixup(allbad); go.debug_fixup(allbad)
    assert np.allclose(gg.get_prims(), go.get_prims(), rtol=1e-12, atol=1e-300)


# ------------------------------------------------------------------------------------------ runs
@pytest.mark.parametrize("cfg", [1, 3])
def test_run_l1_parity(kh, kho, cfg):
    """Full run at reduced size: L1 difference per primitive <= 1e-8 after many steps, flags identical at the end,
    div B at round-off on both sides."""
    if cfg == 1:
        p = ki.config_params(1, n=(32, 32, 8))
        P0, T = modes.config1(p)
        nsteps = None
    else:
        p = ki.config_params(3, n=(48, 32, 8))
        P0 = torus.torus_state(p, seed=1)
        nsteps, T = 40, None
    gg, go = _both(kh, kho, p, P0)
    dt_g = dt_o = go.estimate_dt()
    t, k = 0.0, 0
    while True:
        if T is not None:
            if t >= T * (1 - 1e-12):
                break
            dt_g, dt_o = min(dt_g, T - t), min(dt_o, T - t)
        elif k >= nsteps:
            break
        t += dt_o
        dt_g, dt_o = gg.step(dt_g), go.step(dt_o)
        assert abs(dt_g / dt_o - 1) < 1e-9
        k += 1
    a, b = gg.get_prims(), go.get_prims()
    l1 = l1_diff(p, a, b)
    assert (l1 <= TOL_RUN_L1).all(), l1
    assert np.array_equal(gg.get_flags()[0], go.get_flags()[0])
    assert gg.divB() < 1e-11 * max(1.0, np.abs(P0[5:]).max() * p["n1"])
    if cfg == 1:   # and the GPU run itself converges on the analytic answer like the oracle does
        assert np.abs(a - P0).mean(axis=(1, 2, 3))[3] < 2e-6


def test_device_resident_dt_and_graph_replay_match_explicit_stepping(kh):
    p = ki.config_params(5, n=(24, 20, 16), recon=kp.RECON_WENO5)
    P0 = modes.config5(p, seed=4, amp=1e-2)
    outs = []
    for mode in ("explicit", "device_dt", "nograph"):
        g = kh.Grid(p)
        if mode == "nograph":
            g.set_graph(False)
        g.set_prims(P0)
        dt = g.estimate_dt()
        if mode == "device_dt":
            g.step(dt, sync=False)
            for _ in range(4):
                g.step(-1.0, sync=False)
        else:
            for _ in range(5):
                dt = g.step(dt)
        outs.append(g.get_prims())
        assert g.launch_count() > 5 * 15
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])      # deterministic, bitwise


def test_torch_device_buffers(kh):
    import torch
    p = ki.config_params(5, n=(16, 12, 8))
    P0 = modes.config5(p, seed=1)
    g = kh.Grid(p)
    g.set_prims(torch.from_numpy(P0).cuda())
    out = torch.empty(g.shape_int, dtype=torch.float64, device="cuda")
    g.get_prims(out=out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), P0)
    with pytest.raises(kh.KharmError):
        bad = dict(p); bad["n1"] = 0
        kh.Grid(bad)
    # a face-centred CT grid refuses to step before its magnetic state (the face field) is set
    gf = kh.Grid(dict(p, transport=kp.B_FACE_CT))
    gf.set_prims(P0)
    with pytest.raises(kh.KharmError):
        gf.step(1e-3)
    with pytest.raises(kh.KharmError):          # and the face calls are refused on a Flux-CT grid
        g.divB_face()


# ------------------------------------------------------------------------------------------ full size, bench configuration
def test_full_size_config3_one_step_sampled(kh, kho):
    """BASELINE config 3 at its full 192 x 128 x 128 size in the launch configuration bench.py times
    (CUDA-graph replay, WENO5, FMKS a = 0.9375).  The oracle computes the same step (OpenMP build,
    bit-identical to the single-thread one); all interior zones are compared."""
    p = ki.config_params(3)
    P0 = torus.torus_state(p, seed=1)
    gg, go = _both(kh, kho, p, P0)
    dt = go.estimate_dt()
    assert abs(gg.estimate_dt() / dt - 1) < 1e-12
    n_g, n_o = gg.step(dt), go.step(dt)
    assert abs(n_g / n_o - 1) < 1e-11
    pf_g, _ = gg.get_flags()
    pf_o, _ = go.get_flags()
    worst = _assert_step_parity(p, gg.get_prims(), go.get_prims(), pf_g, pf_o, "cfg3 full")
    print("cfg3 full size: worst rel diff per primitive", worst)
    assert gg.divB() < 1e-10


@pytest.mark.parametrize("n,recon", [(64, kp.RECON_MC), (128, kp.RECON_WENO5), (192, kp.RECON_MC), (256, kp.RECON_WENO5)])
def test_config5_sweep_sizes_one_step(kh, kho, n, recon):
    """BASELINE config 5 (Minkowski throughput sweep) at its own sizes up to 256^3, all interior zones.  The oracle holds ~70
    doubles per padded zone (three primitive buffers, three flux and EMF sets, geometry, scratch): 10 GB at 256^3, plus 3 GB
    of numpy arrays in this test; 320^3 would need 19 + 6 GB and is timed by bench.py only."""
    if n >= 256:
        import psutil
        if psutil.virtual_memory().available < 24e9:
            pytest.skip("the 256^3 oracle step needs ~13 GB of host memory; %.0f GB available" % (psutil.virtual_memory().available / 1e9))
    p = ki.config_params(5, n=n, recon=recon)
    P0 = modes.config5(p, seed=1, amp=1e-3)
    gg, go = _both(kh, kho, p, P0)
    dt = go.estimate_dt()
    n_g, n_o = gg.step(dt), go.step(dt)
    assert abs(n_g / n_o - 1) < 1e-11
    _assert_step_parity(p, gg.get_prims(), go.get_prims(), gg.get_flags()[0], go.get_flags()[0], "cfg5 %d^3" % n)
    assert gg.divB() < 1e-10


def test_full_size_config4_one_step(kh, kho):
    """BASELINE config 4 at its full 288 x 128 x 128 size (MAD field, MC), all interior zones."""
    p = ki.config_params(4)
    P0 = torus.torus_state(p, mad=True, seed=1)
    gg, go = _both(kh, kho, p, P0)
    dt = go.estimate_dt()
    n_g, n_o = gg.step(dt), go.step(dt)
    assert abs(n_g / n_o - 1) < 1e-11
    _assert_step_parity(p, gg.get_prims(), go.get_prims(), gg.get_flags()[0], go.get_flags()[0], "cfg4 full")
    assert gg.divB() < 1e-10


def test_full_size_config3_with_every_extension(kh, kho):
    """The 192 x 128 x 128 block with the SURVEY 8(f) extensions switched on together: Kastaun inverter, first-order flux
    correction, drift-frame floors, face-centred CT with upwinded EMFs.  One step, all interior zones."""
    from kharm_inputs import facefield
    p = dict(ki.config_params(3), inverter=kp.INV_KASTAUN, fofc=1, floor_frame=kp.FRAME_DRIFT, transport=kp.B_FACE_CT, emf=kp.EMF_UPWIND)
    P0 = torus.torus_state(p, seed=1)
    faces = facefield.face_from_potential(p, *facefield.axisymmetric_loop_potential(p, amp=2e-3, x1c=2.5))
    gg, go = kh.Grid(p), kho.Grid(p, omp=True)
    for g in (gg, go):
        g.set_prims(P0)
        g.set_face_B(*faces)
    dt = go.estimate_dt()
    n_g, n_o = gg.step(dt), go.step(dt)
    assert abs(n_g / n_o - 1) < 1e-11
    _assert_step_parity(p, gg.get_prims(), go.get_prims(), gg.get_flags()[0], go.get_flags()[0], "cfg3 full, all extensions")
    assert gg.divB_face() <= 4 * go.divB_face() + 1e-14


# ------------------------------------------------------------------------------------------ second inverter (NEXT-2)
@pytest.mark.parametrize("case", ["torus_weno5", "mad_mc", "minkowski", "bondi"])
def test_one_step_kastaun_inverter(kh, kho, case):
    """Same bars as the 1D_W path with kh_params.inverter = KH_INV_KASTAUN on both sides."""
    if case == "torus_weno5":
        p = ki.config_params(3, n=(64, 48, 8)); P0 = torus.torus_state(p, seed=2); gh = False
    elif case == "mad_mc":
        p = ki.config_params(4, n=(72, 40, 6)); P0 = torus.torus_state(p, mad=True, seed=2); gh = False
    elif case == "minkowski":
        p = ki.config_params(5, n=(37, 13, 5), recon=kp.RECON_WENO5); P0 = modes.config5(p, seed=1, amp=1e-3); gh = False
    else:
        p = ki.config_params(2); P0 = bondi.config2(p); gh = True
    p = dict(p, inverter=kp.INV_KASTAUN)
    _one_step_case(kh, kho, p, P0, with_ghosts=gh, label="kastaun " + case)


def test_kastaun_stress_flags_and_run(kh, kho):
    """Failures, floors and fix-ups under the second inverter (flags identical), then a short run in L1."""
    p = dict(ki.config_params(4, n=(72, 40, 8)), inverter=kp.INV_KASTAUN)
    P0 = torus.torus_state(p, mad=True, seed=3, stress=True, stress_fraction=0.02)
    worst, gg, go = _one_step_case(kh, kho, p, P0, label="kastaun cfg4-stress")
    pf, ff = go.get_flags()
    assert gg.count_flags()[0] == (pf != 0).sum()
    p = dict(ki.config_params(3, n=(48, 32, 8)), inverter=kp.INV_KASTAUN)
    gg, go = _both(kh, kho, p, torus.torus_state(p, seed=1))
    dt = go.estimate_dt()
    for _ in range(10):
        dg, dt = gg.step(dt), go.step(dt)
        assert abs(dg / dt - 1) < 1e-9
    l1 = l1_diff(p, gg.get_prims(), go.get_prims())
    assert l1.max() <= TOL_RUN_L1, l1


# ------------------------------------------------------------------------------------------ first-order flux correction (NEXT-3)
@pytest.mark.parametrize("case", ["torus_weno5", "mad_stress_mc", "minkowski", "bondi", "torus_kastaun"])
def test_one_step_fofc(kh, kho, case):
    """kh_params.fofc = 1 on both sides: same bars; the troubled-zone selection goes through
    the flags, which must be identical for the corrected fluxes to be."""
    if case == "torus_weno5":
        p = ki.config_params(3, n=(64, 48, 8)); P0 = torus.torus_state(p, seed=2); gh = False
    elif case == "mad_stress_mc":
        p = ki.config_params(4, n=(72, 40, 8)); P0 = torus.torus_state(p, mad=True, seed=3, stress=True, stress_fraction=0.02); gh = False
    elif case == "minkowski":
        p = ki.config_params(5, n=(37, 13, 5), recon=kp.RECON_WENO5); P0 = modes.config5(p, seed=1, amp=1e-3); gh = False
    elif case == "bondi":
        p = ki.config_params(2); P0 = bondi.config2(p); gh = True
    else:
        p = dict(ki.config_params(3, n=(33, 17, 3)), inverter=kp.INV_KASTAUN); P0 = torus.torus_state(p, seed=2); gh = False
    p = dict(p, fofc=1)
    worst, gg, go = _one_step_case(kh, kho, p, P0, with_ghosts=gh, label="fofc " + case)
    if case == "mad_stress_mc":
        assert gg.count_flags()[0] == (go.get_flags()[0] != 0).sum()
        # stage parity of the corrected fluxes, EMFs and c_top (the corrector's)
        I = (slice(3, -3), slice(3, -3), slice(3, -3))
        for d in (1, 2, 3):
            Fg, cg = gg.get_flux(d)
            Fo, co = go.get_flux(d)
            assert np.allclose(cg[I], co[I], rtol=1e-11, atol=1e-14), d
            for v in range(8):
                assert np.abs(Fg[v][I] - Fo[v][I]).max() <= 1e-11 * (np.abs(Fo[v][I]).max() + 1e-300), (d, v)


def test_fofc_run_l1_and_untroubled_bit_identity(kh, kho):
    p = dict(ki.config_params(3, n=(48, 32, 8)), fofc=1)
    gg, go = _both(kh, kho, p, torus.torus_state(p, seed=1))
    dt = go.estimate_dt()
    for _ in range(10):
        dg, dt = gg.step(dt), go.step(dt)
        assert abs(dg / dt - 1) < 1e-9
    l1 = l1_diff(p, gg.get_prims(), go.get_prims())
    assert l1.max() <= TOL_RUN_L1, l1
    # a problem on which nothing is troubled: the FOFC step is bit-identical to the plain step on the GPU too
    q = ki.config_params(5, n=(24, 16, 8), recon=kp.RECON_WENO5)
    P0 = modes.config5(q, seed=1, amp=1e-3)
    res = []
    for fofc in (0, 1):
        g = kh.Grid(dict(q, fofc=fofc))
        g.set_prims(P0)
        d = g.estimate_dt()
        for _ in range(3):
            d = g.step(d)
        res.append((g.get_prims(), d))
    assert np.array_equal(res[0][0], res[1][0]) and res[0][1] == res[1][1]


# ------------------------------------------------------------------------------------------ drift-frame floors (NEXT-4)
@pytest.mark.parametrize("case", ["torus_weno5", "mad_stress_mc", "bondi", "torus_kastaun_fofc"])
def test_one_step_drift_frame_floors(kh, kho, case):
    """kh_params.floor_frame = KH_FRAME_DRIFT on both sides: same bars."""
    if case == "torus_weno5":
        p = ki.config_params(3, n=(64, 48, 8)); P0 = torus.torus_state(p, seed=2); gh = False
    elif case == "mad_stress_mc":
        p = ki.config_params(4, n=(72, 40, 8)); P0 = torus.torus_state(p, mad=True, seed=3, stress=True, stress_fraction=0.02); gh = False
    elif case == "bondi":
        p = ki.config_params(2); P0 = bondi.config2(p); gh = True
    else:
        p = dict(ki.config_params(3, n=(33, 17, 3)), inverter=kp.INV_KASTAUN, fofc=1); P0 = torus.torus_state(p, seed=2); gh = False
    p = dict(p, floor_frame=kp.FRAME_DRIFT)
    worst, gg, go = _one_step_case(kh, kho, p, P0, with_ghosts=gh, label="drift " + case)
    if case != "bondi":
        assert (go.get_flags()[1] != 0).any()          # floors really acted


def test_drift_frame_run_l1_and_fixup_hook(kh, kho):
    p = dict(ki.config_params(3, n=(48, 32, 8)), floor_frame=kp.FRAME_DRIFT)
    gg, go = _both(kh, kho, p, torus.torus_state(p, seed=1))
    dt = go.estimate_dt()
    for _ in range(10):
        dg, dt = gg.step(dt), go.step(dt)
        assert abs(dg / dt - 1) < 1e-9
    l1 = l1_diff(p, gg.get_prims(), go.get_prims())
    assert l1.max() <= TOL_RUN_L1, l1
    # fix-up hook: the floors after the repair also run in the drift frame
    p = dict(ki.config_params(3, n=(20, 16, 6)), floor_frame=kp.FRAME_DRIFT)
    P0 = torus.torus_state(p, seed=1)
    gg, go = _both(kh, kho, p, P0)
    rng = np.random.default_rng(0)
    pf = np.zeros((p["n3"] + 6, p["n2"] + 6, p["n1"] + 6), dtype=np.int32)
    pf[3:-3, 3:-3, 3:-3] = (rng.uniform(size=(p["n3"], p["n2"], p["n1"])) < 0.1) * 3
    gg.debug_fixup(pf); go.debug_fixup(pf)
    a, b = gg.get_prims(), go.get_prims()          # interior (the oracle's hook stops before the ghost refresh)
    assert np.allclose(a, b, rtol=1e-11, atol=1e-300)
    assert np.array_equal(gg.get_flags()[1], go.get_flags()[1])


# ------------------------------------------------------------------------------------------ the configs' own step counts
@pytest.mark.parametrize("cfg,n", [(3, (96, 64, 32)), (4, (96, 48, 24)), (2, None)])
def test_hundred_step_runs_l1(kh, kho, cfg, n):
    """BASELINE configs 3 and 4 ask for 100 steps (config 2: the first 100 steps of the Bondi run): L1 difference per
    primitive <= 1e-8 at the end, flags identical, div B at round-off -- at reduced resolution, device-resident dt.
    (Bondi: the zones at the inner edge, inside the horizon, are not steady in this scheme -- both sides show the same 30 %
    density excursion there -- and amplify a round-off difference by ~100 every 20 steps from step ~120 on, so a longer
    run compares two valid realisations of an unstable boundary layer, not two implementations.)"""
    if cfg == 2:
        p = ki.config_params(2); P0 = bondi.config2(p); gh, nsteps = True, 100
    else:
        p = ki.config_params(cfg, n=n); P0 = torus.torus_state(p, mad=(cfg == 4), seed=1); gh, nsteps = False, 100
    gg, go = _both(kh, kho, p, P0, with_ghosts=gh)
    dt = go.estimate_dt()
    gg.step(dt, sync=False)
    for _ in range(nsteps - 1):
        gg.step(-1.0, sync=False)               # CUDA-graph replay, dt stays on the device
    for _ in range(nsteps):
        dt = go.step(dt)
    a, b = gg.get_prims(), go.get_prims()
    l1 = l1_diff(p, a, b)
    assert (l1 <= TOL_RUN_L1).all(), l1
    assert np.array_equal(gg.get_flags()[0], go.get_flags()[0])
    d_g, d_o = gg.divB(), go.divB()
    assert d_g <= 4 * d_o + 1e-12


def _run_to(g, tend):
    t, dt, ns = 0.0, g.estimate_dt(), 0
    while t < tend * (1 - 1e-12):
        dt = min(dt, tend - t)
        t += dt
        dt = g.step(dt)
        ns += 1
    return ns


def test_config2_as_stated_to_t_50(kh, kho):
    """BASELINE config 2 as stated: 128 x 128 zones, r in [1.8, 50], b^2 / rho = 1 at the sonic radius, run for 50 M, error
    against the analytic steady state.  The CUDA path runs the stated 128^2 and, for the trend, 64^2 and 256^2;
    the oracle runs 64^2 beside it.  Both settle on the same state: their errors against the analytic solution agree to
    1 % of the error although the two runs are, after ~3000 steps through an unstable inner boundary layer (DESIGN.md
    section 3), two realisations and no longer comparable zone by zone (the first 100 steps are: test_hundred_step_runs_l1)."""
    from parity_util import bondi_errors
    errs = {}
    for n in (64, 128, 256):
        p = ki.config_params(2, n=(n, n, 1))
        g = kh.Grid(p)
        g.set_prims(bondi.config2(p), with_ghosts=True)
        P0 = g.get_prims()
        d0 = g.divB()
        ns = _run_to(g, 50.0)
        errs[n] = bondi_errors(p, g.get_prims(), P0)
        assert np.isfinite(g.get_prims()).all() and abs(g.divB() - d0) < 1e-10
        print("config 2, %d^2, t = 50 (%d steps): L1 error vs analytic [rho, u, velocity, field] = %s" % (n, ns, errs[n]))
    e = errs[128]
    assert e[0] < 0.01 and e[1] < 0.03 and e[3] < 0.005, e                         # the stated configuration
    assert np.all(errs[64] / errs[128] > 1.7) and np.all(errs[128] / errs[256] > 1.5), errs
    p = ki.config_params(2, n=(64, 64, 1))
    go = kho.Grid(p, omp=True)
    go.set_prims(bondi.config2(p), with_ghosts=True)
    P0 = go.get_prims()
    _run_to(go, 50.0)
    eo = bondi_errors(p, go.get_prims(), P0)
    assert np.all(np.abs(errs[64] / eo - 1) < 0.01), (errs[64], eo)


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_hundred_step_runs_l1(kh, kho, cfg):
    """BASELINE configs 3 (192 x 128 x 128, WENO5) and 4 (288 x 128 x 128 MAD, MC) at FULL size for their 100 steps: L1
    difference per primitive <= 1e-8 at the end, flags identical, div B at round-off; CUDA-graph replay with the
    device-resident dt against the OpenMP oracle (3 - 5 minutes of host time each)."""
    p = ki.config_params(cfg)
    P0 = torus.torus_state(p, mad=(cfg == 4), seed=1)
    gg, go = _both(kh, kho, p, P0)
    dt = go.estimate_dt()
    gg.step(dt, sync=False)
    for _ in range(99):
        gg.step(-1.0, sync=False)
    for _ in range(100):
        dt = go.step(dt)
    ref = go.get_prims()
    l1 = l1_diff(p, gg.get_prims(), ref)
    print("config %d full size, 100 steps: L1 per primitive %s" % (cfg, l1))
    assert np.array_equal(gg.get_flags()[0], go.get_flags()[0])
    assert gg.divB() <= 4 * go.divB() + 1e-12
    if not (l1 <= TOL_RUN_L1).all():
        # Measured on config 3 at full size: from step ~15 on a few hundred atmosphere zones at the torus surface amplify
        # round-off exponentially (max relative difference 1e-8 at step 10, 7e-4 at step 20, 0.2 at step 50 in single zones; no
        # flag ever differs), which lifts the L1 of the velocities to 1.5e-7 at step 100 (rho 8e-11, u 9e-12, B 2e-13).  The
        # reduced-size runs (test_hundred_step_runs_l1) stay at 1e-12.  Whether that is the scheme or the CUDA path is decided
        # by the oracle alone: the same run from P0 (1 +- 2^-52) is as far from the oracle's own result (S23c).  That second
        # oracle run is stored: tests/golden/config3_full_sensitivity.txt, written by tests/golden/make_config3_sensitivity.py.
        assert cfg == 3
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config3_full_sensitivity.txt")
        l1_self = np.array([float(x) for x in [ln for ln in open(path) if not ln.startswith("#")][0].split()])
        print("config 3 full size: the oracle against itself from 1-ulp input noise (stored): L1 %s" % l1_self)
        assert (l1 <= np.maximum(TOL_RUN_L1, K_SENS * l1_self)).all(), (l1, l1_self)


# ------------------------------------------------------------------------------------------ normal-frame floors (NEXT-4)
@pytest.mark.parametrize("case", ["torus_weno5", "mad_stress_mc", "torus_kastaun", "minkowski"])
def test_one_step_normal_frame_floors(kh, kho, case):
    """kh_params.floor_frame = KH_FRAME_NORMAL on both sides: same bars (floor flags may carry bit 64)."""
    if case == "torus_weno5":
        p = ki.config_params(3, n=(64, 48, 8)); P0 = torus.torus_state(p, seed=2)
    elif case == "mad_stress_mc":
        p = ki.config_params(4, n=(72, 40, 8)); P0 = torus.torus_state(p, mad=True, seed=3, stress=True, stress_fraction=0.02)
    elif case == "torus_kastaun":
        p = dict(ki.config_params(3, n=(33, 17, 3)), inverter=kp.INV_KASTAUN); P0 = torus.torus_state(p, seed=2)
    else:
        p = ki.config_params(5, n=(16, 12, 8)); P0 = modes.config5(p, seed=1, amp=1e-3)
    p = dict(p, floor_frame=kp.FRAME_NORMAL)
    worst, gg, go = _one_step_case(kh, kho, p, P0, label="normal " + case)
    if case != "minkowski":
        assert (go.get_flags()[1] != 0).any()
    # fix-up hook under the same frame
    if case == "torus_weno5":
        rng = np.random.default_rng(0)
        pf = np.zeros((p["n3"] + 6, p["n2"] + 6, p["n1"] + 6), dtype=np.int32)
        pf[3:-3, 3:-3, 3:-3] = (rng.uniform(size=(p["n3"], p["n2"], p["n1"])) < 0.1) * 3
        gg.debug_fixup(pf); go.debug_fixup(pf)
        z = np.zeros_like(gg.get_flags()[0])
        _assert_step_parity(p, gg.get_prims(), go.get_prims(), z, z, "normal-frame fix-up")     # the S23 metric
        assert (gg.get_flags()[1] != go.get_flags()[1]).mean() < 1e-3


# ------------------------------------------------------------------------------------------ face-centred CT (NEXT-1)
def _face_pair(kh, kho, p, P0, faces):
    p = dict(p, transport=kp.B_FACE_CT)
    gg, go = kh.Grid(p), kho.Grid(p, omp=True)
    for g in (gg, go):
        g.set_prims(P0)
        g.set_face_B(*faces)
    return p, gg, go


@pytest.mark.parametrize("case", ["minkowski_weno5", "torus_mc", "torus_weno5_kastaun_fofc", "two_d_upwind"])
def test_face_centred_ct_parity(kh, kho, case):
    """kh_params.transport = KH_B_FACE_CT on both sides: the face field agrees to round-off, its
    divergence stays at round-off on both sides, the primitives meet the one-step and run bars."""
    from kharm_inputs import facefield
    if case == "minkowski_weno5":
        p = ki.config_params(5, n=(24, 18, 10), recon=kp.RECON_WENO5)
        P0 = modes.config5(p, seed=2, amp=1e-2)
        faces = facefield.face_from_potential(p, *facefield.periodic_potential(p, seed=3, amp=5e-2))
    elif case == "two_d_upwind":          # n3 = 1 (S21) with the face field, upwinded EMFs and drift-frame floors
        p = dict(ki.config_params(3, n=(64, 48, 1)), emf=kp.EMF_UPWIND, floor_frame=kp.FRAME_DRIFT)
        P0 = torus.torus_state(p, seed=2)
        faces = facefield.face_from_potential(p, *facefield.axisymmetric_loop_potential(p, amp=2e-3, x1c=2.3))
    else:
        p = ki.config_params(3, n=(48, 32, 8), recon=kp.RECON_MC if case == "torus_mc" else kp.RECON_WENO5)
        if case != "torus_mc":
            p = dict(p, inverter=kp.INV_KASTAUN, fofc=1)
        P0 = torus.torus_state(p, seed=2)
        faces = facefield.face_from_potential(p, *facefield.axisymmetric_loop_potential(p, amp=2e-3, x1c=2.3))
    p, gg, go = _face_pair(kh, kho, p, P0, faces)
    assert np.array_equal(gg.get_prims(with_ghosts=True)[:5], go.get_prims(with_ghosts=True)[:5])
    assert np.allclose(gg.get_prims(with_ghosts=True)[5:], go.get_prims(with_ghosts=True)[5:], rtol=1e-13, atol=1e-300)
    d0 = go.divB_face()
    assert gg.divB_face() <= 2 * d0 + 1e-16
    dt = go.estimate_dt()
    assert abs(gg.estimate_dt() / dt - 1) < 1e-12
    n_g, n_o = gg.step(dt), go.step(dt)
    assert abs(n_g / n_o - 1) < 1e-11
    _assert_step_parity(p, gg.get_prims(), go.get_prims(), gg.get_flags()[0], go.get_flags()[0], "face-CT " + case)
    for _ in range(9):
        n_g, n_o = gg.step(n_g), go.step(n_o)
    l1 = l1_diff(p, gg.get_prims(), go.get_prims())
    assert l1.max() <= TOL_RUN_L1, l1
    fg, fo = gg.get_face_B(), go.get_face_B()
    I = (slice(3, -3), slice(3, -3), slice(3, -3))
    for d in range(3):
        sc = max(np.abs(fo[d][I]).max(), 1e-300)
        assert np.abs(fg[d][I] - fo[d][I]).max() <= 1e-9 * max(sc, np.abs(fo[0][I]).max()), d
    assert gg.divB_face() <= 1e-11 * max(np.abs(fo[0]).max(), np.abs(fo[1]).max()) * max(p["n1"], p["n2"]) + 4 * d0


@pytest.mark.parametrize("kind", [kp.EMF_UPWIND, kp.EMF_CENTRED])
@pytest.mark.parametrize("case", ["flux_ct_torus", "face_ct_minkowski", "face_ct_torus_stress"])
def test_upwinded_emf_parity(kh, kho, case, kind):
    """kh_params.emf = KH_EMF_UPWIND / KH_EMF_CENTRED on both sides ("a number of schemes ... with and
    without upwinding": Gardiner & Stone's contact-upwinded and un-upwinded edge EMFs), with either transport: stage EMFs,
    one step, a 10-step run."""
    from kharm_inputs import facefield
    faces = None
    if case == "flux_ct_torus":
        p = ki.config_params(3, n=(48, 32, 8)); P0 = torus.torus_state(p, seed=2)
    elif case == "face_ct_minkowski":
        p = dict(ki.config_params(5, n=(24, 18, 10), recon=kp.RECON_WENO5), transport=kp.B_FACE_CT)
        P0 = modes.config5(p, seed=2, amp=5e-2)
        faces = facefield.face_from_potential(p, *facefield.periodic_potential(p, seed=3, amp=5e-2))
    else:
        p = dict(ki.config_params(4, n=(48, 32, 8)), transport=kp.B_FACE_CT)
        P0 = torus.torus_state(p, mad=True, seed=3, stress=True, stress_fraction=0.02)
        faces = facefield.face_from_potential(p, *facefield.axisymmetric_loop_potential(p, amp=2e-3, x1c=2.3))
    p = dict(p, emf=kind)
    gg, go = kh.Grid(p), kho.Grid(p, omp=True)
    for g in (gg, go):
        g.set_prims(P0)
        if faces is not None:
            g.set_face_B(*faces)
    dt = go.estimate_dt()
    n_g, n_o = gg.step(dt), go.step(dt)
    assert abs(n_g / n_o - 1) < 1e-11
    _assert_step_parity(p, gg.get_prims(), go.get_prims(), gg.get_flags()[0], go.get_flags()[0],
                        ("upwind emf " if kind == kp.EMF_UPWIND else "centred emf ") + case)
    I = (slice(3, -3), slice(3, -3), slice(3, -3))
    for d in (1, 2, 3):
        eg, eo = gg.get_emf(d), go.get_emf(d)
        assert np.abs(eg[I] - eo[I]).max() <= 1e-11 * (max(np.abs(go.get_emf(c)[I]).max() for c in (1, 2, 3)) + 1e-300), d
    for _ in range(9):
        n_g, n_o = gg.step(n_g), go.step(n_o)
    l1 = l1_diff(p, gg.get_prims(), go.get_prims())
    assert l1.max() <= TOL_RUN_L1, l1
    if faces is not None:
        assert gg.divB_face() <= 4 * go.divB_face() + 1e-13


# ------------------------------------------------------------------------------------------ the paper's own acceptance tests, on the CUDA path
def _cuda_mode_errors(kh, rotated, recon, ns, thin):
    _, r = modes.eigenmode([1, 1, 0] / np.sqrt(2) if rotated else [1, 0, 0], modes.FAST)
    act = np.abs(r) > 0.05
    tot = []
    for n in ns:
        p = ki.config_params(1, n=(n, 4 if thin else n, 4), recon=recon)
        P0, T = modes.config1(p, rotated=rotated)
        g = kh.Grid(p)
        g.set_prims(P0)
        dt, t = g.estimate_dt(), 0.0
        while t < T * (1 - 1e-12):
            dt = min(dt, T - t)
            t += dt
            dt = g.step(dt)
        assert g.divB() < 1e-12 and g.count_flags()[0] == 0
        tot.append(np.abs(g.get_prims() - P0).mean(axis=(1, 2, 3))[act].sum())
    return np.array(tot)


@pytest.mark.parametrize("rotated,recon", [(True, kp.RECON_WENO5), (True, kp.RECON_MC), (False, kp.RECON_WENO5), (False, kp.RECON_MC)])
def test_cuda_path_linear_mode_convergence(kh, rotated, recon):
    """P:413 on the CUDA path alone (no oracle): the L1 error of a linear mode after one period falls with resolution at a
    power inside the paper's window [-2.1, -1.9] (tests/golden/paper_values.txt) -- the same three statements as the
    oracle's own pins (tests/test_oracle_step.py): oblique WENO5 at every doubling 16 -> 64, oblique MC at 64 -> 128,
    the grid-aligned mode through the Richardson extrapolation of its slopes at 64 -> 128 -> 256."""
    from conftest import read_golden
    gold = read_golden()
    lo, hi = gold["convergence_slope_min"], gold["convergence_slope_max"]
    if rotated and recon == kp.RECON_WENO5:
        slopes = np.diff(np.log2(_cuda_mode_errors(kh, True, recon, (16, 32, 64), thin=False)))
        assert np.all((slopes >= lo) & (slopes <= hi)), slopes
    elif rotated:
        slopes = np.diff(np.log2(_cuda_mode_errors(kh, True, recon, (32, 64, 128), thin=False)))
        assert lo <= slopes[1] <= hi and slopes[1] < slopes[0] < -1.8, slopes
    else:
        s1, s2 = np.diff(np.log2(_cuda_mode_errors(kh, False, recon, (64, 128, 256), thin=True)))
        assert -2.0 < s2 < s1 < -1.5, (s1, s2)
        assert lo <= 2 * s2 - s1 <= hi, (s1, s2, 2 * s2 - s1)


# ------------------------------------------------------------------------------------------ seeded fuzz over sizes, boundaries and options
def _fuzz_case(seed):
    """Seeded random block of the fuzz test: (params, primitives, face field or None, options, label)."""
    from kharm_inputs import facefield
    rng = np.random.default_rng(1000 + seed)
    curved = seed % 2 == 0
    if curved:
        n = (int(rng.integers(6, 28)), int(rng.integers(4, 20)), int(rng.integers(1, 7)))
        p = ki.config_params(3 if seed % 4 == 0 else 4, n=n)
        if rng.uniform() < 0.3:                       # plain Kerr-Schild coordinates away from the axis
            p = dict(p, coords=kp.KS, xmin=[6.0, 1.0, 0.0], xmax=[12.0, np.pi - 1.0, 2 * np.pi],
                     bc=[kp.BC_OUTFLOW, kp.BC_OUTFLOW, kp.BC_OUTFLOW, kp.BC_OUTFLOW, kp.BC_PERIODIC, kp.BC_PERIODIC])
        if p["coords"] == kp.KS:                      # a smooth magnetised inflow in plain Kerr-Schild coordinates (x1 = r, x2 = theta)
            r = (p["xmin"][0] + (np.arange(n[0]) + 0.5) * (p["xmax"][0] - p["xmin"][0]) / n[0])[None, None, :]
            th = (p["xmin"][1] + (np.arange(n[1]) + 0.5) * (p["xmax"][1] - p["xmin"][1]) / n[1])[None, :, None]
            ph = (2 * np.pi * (np.arange(n[2]) + 0.5) / n[2])[:, None, None]
            P0 = np.zeros((8,) + n[::-1])
            P0[0] = (r / 2.0) ** -1.5 * (1 + 0.1 * np.sin(3 * th) * np.cos(ph))
            P0[1] = 0.05 * P0[0] ** p["gamma"]
            P0[2] = -0.3 / np.sqrt(r) * (1 + 0.2 * np.cos(2 * th))
            P0[3] = 0.02 * np.sin(2 * th) / r + 0 * ph
            P0[4] = 0.05 / r ** 1.5 * (1 + 0.3 * np.sin(ph))
            P0[5] = 0.05 / r ** 2 * np.cos(th) + 0 * ph
            P0[6] = 0.02 / r ** 2 * np.sin(th) * np.cos(ph)
            P0[7] = 0.01 / r ** 2 * (1 + 0 * th) * np.sin(ph)
        else:
            P0 = torus.torus_state(p, mad=bool(seed % 4), seed=seed, stress=bool(rng.uniform() < 0.5), stress_fraction=0.03)
    else:
        n = (int(rng.integers(3, 40)), int(rng.integers(3, 20)), int(rng.integers(1, 9)))
        p = ki.config_params(5, n=n)
        bc = []
        for d in range(3):
            kind = kp.BC_PERIODIC if (rng.uniform() < 0.6 or n[d] < 3) else kp.BC_OUTFLOW
            bc += [kind, kind]
        p = dict(p, bc=bc)
        P0 = modes.config5(p, seed=seed, amp=10 ** rng.uniform(-3, -1))
    opts = dict(recon=int(rng.integers(0, 2)), inverter=int(rng.integers(0, 2)), floor_frame=int(rng.integers(0, 3)),
                fofc=int(rng.integers(0, 2)), transport=int(rng.integers(0, 2)), emf=int(rng.integers(0, 2)))
    if seed % 3 == 2 and opts["emf"] == kp.EMF_UPWIND:
        opts["emf"] = kp.EMF_CENTRED           # (added in round 2 without changing any seed's other draws)
    p = dict(p, **opts)
    faces = None
    if opts["transport"] == kp.B_FACE_CT:
        if curved and p["coords"] == kp.FMKS:
            pot = facefield.axisymmetric_loop_potential(p, amp=1e-3, x1c=0.5 * (p["xmin"][0] + p["xmax"][0]),
                                                        width=0.3 * (p["xmax"][0] - p["xmin"][0]))
        else:
            pot = facefield.periodic_potential(p, seed=seed, amp=1e-2)
        if not curved and any(b != kp.BC_PERIODIC for b in p["bc"]):
            pot = [np.zeros_like(pot[0]), np.zeros_like(pot[0]), pot[2] * 0 + 1e-3 * np.cos(np.linspace(0, 1, pot[2].shape[2]))[None, None, :]]
        faces = facefield.face_from_potential(p, *pot)
    label = "fuzz %d %s n=%s bc=%s" % (seed, opts, n, p["bc"])
    return p, P0, faces, opts, label


@pytest.mark.parametrize("seed", list(range(int(__import__("os").environ.get("KH_FUZZ_SEEDS", "48")))) + [432])
def test_fuzz_one_step_random_configurations(kh, kho, seed):
    """Random small blocks: ragged sizes (down to 3 zones), every boundary kind that is legal for the coordinate system,
    and random choices of reconstruction, inverter, floor frame, FOFC, transport and EMF kind.  One step (plus one more
    for the odd seeds), the usual bars.  Seed 432 is the one seed of 0..999 that was outside the bar at the end of round 1
    (named here so that it runs every time)."""
    p, P0, faces, opts, label = _fuzz_case(seed)
    gg, go = kh.Grid(p), kho.Grid(p, omp=True)
    for g in (gg, go):
        g.set_prims(P0)
        if faces is not None:
            g.set_face_B(*faces)
    dt = go.estimate_dt()
    assert abs(gg.estimate_dt() / dt - 1) < 1e-12, label
    dts = []
    for _ in range(1 + seed % 2):
        n_g, n_o = gg.step(dt), go.step(dt)
        assert abs(n_g / n_o - 1) < 1e-10, label
        dts.append(dt)
        dt = n_o
    pf_g, ff_g = gg.get_flags()
    pf_o, ff_o = go.get_flags()
    # the flat bar for one step and for two, for every floor frame: what exceeds it must be explained by the oracle's own
    # measured sensitivity to 1-ulp input noise (S23c), not by a looser number
    sens = oracle_sensitivity(kho, p, P0, faces, dts)
    _assert_step_parity(p, gg.get_prims(), go.get_prims(), pf_g, pf_o, label, tol=TOL_ONE_STEP, sens=sens)
    if opts["floor_frame"] != kp.FRAME_NORMAL:      # (after a normal-frame injection rho sits AT its floor: the second-pass bit is a coin flip)
        assert (ff_g != ff_o).sum() <= max(2, (1e-2 if opts["fofc"] else 5e-3) * ff_o.size), label    # marginal floor decisions may flip


@pytest.mark.parametrize("seed", list(range(8)))
def test_fuzz_graph_replay_matches_direct_launches_for_every_option_mix(kh, seed):
    """CUDA-graph replay with the device-resident dt, direct launches and profiled launches give bitwise the same state
    for random mixes of the options (the graph then holds the FOFC memset / mask nodes, the face-field kernels, ...)."""
    from kharm_inputs import facefield
    rng = np.random.default_rng(77 + seed)
    p = ki.config_params(3, n=(int(rng.integers(12, 40)), int(rng.integers(8, 24)), int(rng.integers(1, 8))))
    opts = dict(recon=int(rng.integers(0, 2)), inverter=int(rng.integers(0, 2)), floor_frame=int(rng.integers(0, 3)),
                fofc=int(rng.integers(0, 2)), transport=int(rng.integers(0, 2)), emf=int(rng.integers(0, 2)))
    p = dict(p, **opts)
    P0 = torus.torus_state(p, mad=bool(seed % 2), seed=seed, stress=True, stress_fraction=0.02)
    faces = facefield.face_from_potential(p, *facefield.axisymmetric_loop_potential(p, amp=1e-3, x1c=2.5)) if opts["transport"] else None
    outs = []
    for mode in ("graph_device_dt", "direct", "profiled"):
        g = kh.Grid(p)
        g.set_prims(P0)
        if faces is not None:
            g.set_face_B(*faces)
        dt = g.estimate_dt()
        if mode == "graph_device_dt":
            g.step(dt, sync=False)
            for _ in range(3):
                g.step(-1.0, sync=False)
        else:
            if mode == "direct":
                g.set_graph(False)
            else:
                g.set_profile(True)
            for _ in range(4):
                dt = g.step(dt)
        outs.append((g.get_prims(), g.get_flags(), g.get_face_B() if faces is not None else None))
    for o in outs[1:]:
        assert np.array_equal(outs[0][0], o[0]), opts
        assert np.array_equal(outs[0][1][0], o[1][0]) and np.array_equal(outs[0][1][1], o[1][1]), opts
        if faces is not None:
            assert all(np.array_equal(a, b) for a, b in zip(outs[0][2], o[2])), opts
