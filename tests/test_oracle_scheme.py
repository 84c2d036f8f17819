"""Pins of the oracle's scheme pieces: reconstruction (C3), LLF (C4), Flux-CT (C5), U->P (C7), and
brute-force unit cases of the build-defined parts (floors C8, fix-up C9, ghost fills C10)."""
import numpy as np
import pytest

import kharm_inputs as ki
from kharm_inputs import params as kp

ETA = np.diag([-1.0, 1, 1, 1])
NG = 3


# ------------------------------------------------------------------ reconstruction
def test_recon_exact_on_polynomials(kho):
    x = np.arange(-2, 3, dtype=float)
    for kind in (kho.RECON_MC, kho.RECON_WENO5):
        l, r = kho.recon(kind, np.full(5, 3.25))
        assert l == 3.25 and r == 3.25
        l, r = kho.recon(kind, 1.5 + 0.25 * x)                       # linear data: exact face values
        assert abs(l - (1.5 - 0.125)) < 1e-15 and abs(r - (1.5 + 0.125)) < 1e-15
    # WENO5: cell AVERAGES of a quadratic -> point values at the faces, exact
    a, b, c = 0.7, -0.3, 0.2
    avg = a + b * x + c * (x * x + 1.0 / 12.0)
    l, r = kho.recon(kho.RECON_WENO5, avg)
    assert abs(l - (a - 0.5 * b + 0.25 * c)) < 1e-14 and abs(r - (a + 0.5 * b + 0.25 * c)) < 1e-14
    # smooth data: fifth-order accurate face value
    errs = []
    for h in (0.2, 0.1):
        xs = h * x
        avgs = (np.cos(xs - h / 2) - np.cos(xs + h / 2)) / h          # cell averages of sin
        errs.append(abs(kho.recon(kho.RECON_WENO5, avgs)[1] - np.sin(h / 2)))
    assert errs[0] / errs[1] > 20


def test_recon_limits_and_mirror(kho):
    rng = np.random.default_rng(2)
    for _ in range(200):
        q = rng.normal(size=5)
        for kind in (kho.RECON_MC, kho.RECON_WENO5):
            l, r = kho.recon(kind, q)
            lm, rm = kho.recon(kind, q[::-1])
            assert l == rm and r == lm                                   # mirror symmetry
            lo, hi = q.min(), q.max()
            if kind == kho.RECON_MC:                                     # MC is bounded by the neighbours
                assert min(q[1:4]) - 1e-15 <= l <= max(q[1:4]) + 1e-15 and min(q[1:4]) - 1e-15 <= r <= max(q[1:4]) + 1e-15
    # MC at an extremum: zero slope; across a jump: bounded, no overshoot
    assert kho.recon(kho.RECON_MC, [0, 1, 2, 1, 0]) == (2.0, 2.0)
    l, r = kho.recon(kho.RECON_MC, [0, 0, 0.1, 1, 1])
    assert 0.0 <= l <= 0.1 <= r <= 1.0
    # MC slope is the minimum of (2 dq-, 2 dq+, centred)
    l, r = kho.recon(kho.RECON_MC, [0, 0.0, 1.0, 1.2, 9])
    assert abs((r - l) - 0.4) < 1e-15
    l, r = kho.recon(kho.RECON_WENO5, [1, 1, 1, 0, 0])                   # WENO picks the smooth stencil
    assert abs(r - 1.0) < 1e-10 and abs(l - 1.0) < 1e-10


# ------------------------------------------------------------------ LLF
def test_llf_consistency_and_dissipation(kho):
    gam = 5.0 / 3.0
    Pk = kho.make_params(ki.config_params(3))
    gcov, gcon, gdet, _ = kho.metric(Pk, 1.5, 0.3)
    P = np.array([0.8, 0.3, 0.2 / np.sqrt(gcov[1, 1]), -0.1 / np.sqrt(gcov[2, 2]), 0.3 / np.sqrt(gcov[3, 3]),
                  0.2 / np.sqrt(gcov[1, 1]), 0.1 / np.sqrt(gcov[2, 2]), -0.3 / np.sqrt(gcov[3, 3])])
    for d in (1, 2, 3):
        F, ctop = kho.llf(gcov, gcon, gdet, P, P, gam, d)
        assert np.array_equal(F, kho.prim_to_flux(gcov, gcon, gdet, P, gam, d))     # F(P,P) = F(P)
        vmax, vmin = kho.vchar(gcov, gcon, P, gam, d)
        assert ctop == max(0.0, vmax, -vmin)
        Q = P * (1 + 0.01 * np.arange(8))
        F2, c2 = kho.llf(gcov, gcon, gdet, P, Q, gam, d)
        FL, FR = kho.prim_to_flux(gcov, gcon, gdet, P, gam, d), kho.prim_to_flux(gcov, gcon, gdet, Q, gam, d)
        UL, UR = kho.prim_to_flux(gcov, gcon, gdet, P, gam, 0), kho.prim_to_flux(gcov, gcon, gdet, Q, gam, 0)
        assert np.allclose(F2, 0.5 * (FL + FR - c2 * (UR - UL)), rtol=1e-14, atol=1e-16)
        v2 = kho.vchar(gcov, gcon, Q, gam, d)
        assert c2 == max(0.0, vmax, v2[0], -vmin, -v2[1])


def test_llf_mirror(kho):
    """x -> -x with ut^x, B^x -> -ut^x, -B^x swaps L/R and flips the sign of the parity-even fluxes."""
    gam = 4.0 / 3.0
    rng = np.random.default_rng(8)
    flip = np.array([1, 1, -1, 1, 1, -1, 1, 1.0])
    for _ in range(20):
        PL = np.abs(rng.normal(size=8)) * np.array([1, 1, .3, .3, .3, 1, 1, 1]) * rng.choice([-1, 1], 8)
        PR = np.abs(rng.normal(size=8)) * np.array([1, 1, .3, .3, .3, 1, 1, 1]) * rng.choice([-1, 1], 8)
        PL[:2] = np.abs(PL[:2]) + 0.1; PR[:2] = np.abs(PR[:2]) + 0.1
        F, c = kho.llf(ETA, ETA, 1.0, PL, PR, gam, 1)
        Fm, cm = kho.llf(ETA, ETA, 1.0, PR * flip, PL * flip, gam, 1)
        assert abs(c - cm) <= 1e-15
        # fluxes of scalars / transverse vectors change sign, of x-vectors do not
        assert np.allclose(Fm, -F * flip, rtol=1e-13, atol=1e-14)


# ------------------------------------------------------------------ Flux-CT
def _corner_div_rate(F1, F2, F3, n, dx):
    """d/dt of the corner-centred div(sqrt(-g) B) implied by face fluxes, interior corners (numpy)."""
    n1, n2, n3 = n
    sl = lambda a, o1, o2, o3: a[NG + o3:NG + n3 + o3 + 1, NG + o2:NG + n2 + o2 + 1, NG + o1:NG + n1 + o1 + 1]  # noqa: E731

    def dUdt(comp, o):          # -sum_e (F^e(+1) - F^e)/dx_e for zone offset o, evaluated for zones [-1..n]
        out = 0.0
        for e, F in enumerate((F1, F2, F3)):
            up = [o[0], o[1], o[2]]; up[e] += 1
            out = out - (sl(F[comp], *up) - sl(F[comp], *o)) / dx[e]
        return out

    div = 0.0
    for d in range(3):
        acc = 0.0
        for a in (0, -1):
            for b in (0, -1):
                o = [0, 0, 0]; o[(d + 1) % 3] = a; o[(d + 2) % 3] = b
                lo = list(o); lo[d] -= 1
                acc = acc + dUdt(5 + d, o) - dUdt(5 + d, lo)
        div = div + 0.25 * acc / dx[d]
    # zones used: offsets -1..0 around corners i = 1..n-1 -> restrict to strictly interior corners
    return div[1:n3, 1:n2, 1:n1] if n3 > 1 else div[:, 1:n2, 1:n1]


@pytest.mark.parametrize("n", [(8, 6, 5), (7, 9, 4)])
def test_flux_ct_preserves_corner_divergence_for_arbitrary_fluxes(kho, n):
    p = ki.base_params(n1=n[0], n2=n[1], n3=n[2], bc=[kp.BC_OUTFLOW] * 6)
    P = kho.make_params(p)
    rng = np.random.default_rng(4)
    shape = (8, n[2] + 6, n[1] + 6, n[0] + 6)
    F = [rng.normal(size=shape) for _ in range(3)]
    dx = (0.1, 0.07, 0.13)
    before = np.abs(_corner_div_rate(F[0], F[1], F[2], n, dx)).max()
    raw = [f.copy() for f in F]
    kho.flux_ct_arrays(P, F[0], F[1], F[2])
    after = np.abs(_corner_div_rate(F[0], F[1], F[2], n, dx)).max()
    assert before > 10 and after < 1e-11
    for d in range(3):
        assert np.array_equal(F[d][:5], raw[d][:5])                       # hydro fluxes untouched
        assert np.all(F[d][5 + d][NG:-NG, NG:-NG, NG:-NG] == 0)           # F^d[B^d] = 0
    # the EMF average reproduces a uniform electric field: fluxes from a constant E stay unchanged
    E = np.array([0.3, -0.2, 0.5])
    G = [np.zeros(shape) for _ in range(3)]
    G[0][6], G[0][7] = E[2], -E[1]
    G[1][5], G[1][7] = -E[2], E[0]
    G[2][5], G[2][6] = E[1], -E[0]
    H = [g.copy() for g in G]
    kho.flux_ct_arrays(P, H[0], H[1], H[2])
    I = (slice(None), slice(NG, NG + n[2]), slice(NG, NG + n[1]), slice(NG, NG + n[0]))
    for d in range(3):
        assert np.allclose(H[d][I], G[d][I], atol=1e-15)


# ------------------------------------------------------------------ U -> P
def _geoms(kho):
    out = [(ETA, ETA, 1.0)]
    Pk = kho.make_params(ki.base_params(coords=kp.KS, a=0.9375))
    out += [kho.metric(Pk, r, th)[:3] for r, th in ((1.4, 0.5), (8.0, 1.5), (300.0, 2.9))]
    Pf = kho.make_params(ki.config_params(3))
    out += [kho.metric(Pf, x1, x2)[:3] for x1, x2 in ((0.26, 0.004), (2.5, 0.5), (6.5, 0.8))]
    return out


def test_u2p_round_trip(kho):
    rng = np.random.default_rng(21)
    gam = 13.0 / 9.0
    worst = 0.0
    for gcov, gcon, gdet in _geoms(kho):
        for _ in range(60):
            P = np.zeros(8)
            P[0] = 10 ** rng.uniform(-4, 1)
            P[1] = P[0] * 10 ** rng.uniform(-3, 1)
            gamma_target = 10 ** rng.uniform(-2, 1)                      # q up to ~10 (Lorentz factor ~10)
            vdir = rng.normal(size=3)
            for i in range(3):
                P[2 + i] = vdir[i] / np.sqrt(gcov[i + 1, i + 1])
                P[5 + i] = np.sqrt(P[0] * 10 ** rng.uniform(-3, 1)) * rng.normal() / np.sqrt(gcov[i + 1, i + 1])
            q = np.sqrt(P[2:5] @ gcov[1:, 1:] @ P[2:5])
            P[2:5] *= gamma_target / q
            U = kho.prim_to_flux(gcov, gcon, gdet, P, gam, 0)
            guess = P * (1 + 0.3 * rng.uniform(-1, 1, 8))
            Pr, flag = kho.u2p(gcov, gcon, gdet, U, guess, gam)
            assert flag == 0
            scale = np.array([P[0], P[1]] + [np.sqrt(P[2:5] @ gcov[1:, 1:] @ P[2:5]) / np.sqrt(gcov[i, i]) for i in (1, 2, 3)]
                             + [np.abs(P[5 + i]) + 1e-300 for i in range(3)])
            # conditioning of the energy slot: du/u ~ eps (rho + b^2) gamma^2 / u
            D = kho.fourvec(gcov, gcon, P)
            cond = max(1.0, (P[0] + D["bsq"]) * (1 + gamma_target ** 2) / P[1])
            err = np.abs(Pr - P) / scale
            worst = max(worst, (err / cond).max())
            assert (err <= 1e-12 * cond).all(), (err, cond)
            assert np.array_equal(Pr[5:8], U[5:8] / gdet)
    assert worst < 1e-12


def test_u2p_static_limit_and_flags(kho):
    gam = 4.0 / 3.0
    # B = 0, ut = 0: W = rho + Gamma u exactly, one Newton step from any guess lands on it
    P = np.array([1.7, 0.4, 0, 0, 0, 0, 0, 0.0])
    U = kho.prim_to_flux(ETA, ETA, 1.0, P, gam, 0)
    assert np.allclose(U[:2], [1.7, -0.4], atol=1e-15)
    Pr, flag = kho.u2p(ETA, ETA, 1.0, U, P * 3.0, gam)
    assert flag == 0 and np.abs(Pr - P).max() < 1e-14
    # flags: D <= 0 -> 1 ; NaN -> 1 ; negative internal energy -> 5 (hydro prims keep the guess, B updated)
    guess = np.array([1.0, 1.0, 0.1, 0, 0, 9, 9, 9.0])
    Ub = U.copy(); Ub[0] = -1.0
    Pr, flag = kho.u2p(ETA, ETA, 1.0, Ub, guess, gam)
    assert flag == 1 and np.array_equal(Pr[:5], guess[:5]) and np.array_equal(Pr[5:], U[5:])
    Ub = U.copy(); Ub[3] = np.nan
    assert kho.u2p(ETA, ETA, 1.0, Ub, guess, gam)[1] == 1
    Ub = U.copy(); Ub[1] = +0.5          # energy below rest mass: T^t_t + D = +0.5 means u = -0.5
    Pr, flag = kho.u2p(ETA, ETA, 1.0, Ub, guess, gam)
    assert flag == 5 and np.array_equal(Pr[:5], guess[:5])
    # momentum too large for the energy: v^2 >= 1 or no root -> a failure flag, never a silent answer
    Ub = U.copy(); Ub[2] = 50.0
    assert kho.u2p(ETA, ETA, 1.0, Ub, guess, gam)[1] != 0


# ------------------------------------------------------------------ floors (build-defined; brute-force unit cases)
def test_floors_unit_cases(kho):
    p = ki.config_params(3)
    P = kho.make_params(p)
    x1, x2 = 2.0, 0.5
    gcov, gcon, gdet, _ = kho.metric(P, x1, x2)
    r = np.exp(x1)
    s = 1 / r ** 2 / (1 + r / 10.0)
    rho_fl, u_fl = 1e-6 * s, 1e-8 * s ** p["gamma"]
    ok = np.array([1e-3, 1e-5, 0, 0, 0, 0, 0, 0.0])
    Pz, flag = kho.floors(P, gcov, gcon, x1, x2, ok)
    assert flag == 0 and np.array_equal(Pz, ok)
    Pz, flag = kho.floors(P, gcov, gcon, x1, x2, [rho_fl / 2, 1e-9, 0, 0, 0, 0, 0, 0])
    assert flag == 1 and Pz[0] == rho_fl and Pz[1] == 1e-9
    Pz, flag = kho.floors(P, gcov, gcon, x1, x2, [1e-3, u_fl / 10, 0, 0, 0, 0, 0, 0])
    assert flag == 4 and abs(Pz[1] / u_fl - 1) < 1e-14
    # magnetisation ceilings: b^2 = g_11 B1^2 at rest
    B1 = 1.0 / np.sqrt(gcov[1, 1])
    D = kho.fourvec(gcov, gcon, [1, 1, 0, 0, 0, B1, 0, 0])
    Pz, flag = kho.floors(P, gcov, gcon, x1, x2, [1e-3, 1e-3, 0, 0, 0, B1, 0, 0])
    assert flag == (2 | 0) and abs(Pz[0] - D["bsq"] / 100.0) < 1e-15 and Pz[1] == 1e-3
    Pz, flag = kho.floors(P, gcov, gcon, x1, x2, [1.0, 1e-6, 0, 0, 0, B1, 0, 0])
    assert flag == 8 and abs(Pz[1] - D["bsq"] / 1e4) < 1e-18
    Pz, flag = kho.floors(P, gcov, gcon, x1, x2, [1e-3, 1.0, 0, 0, 0, 0, 0, 0])
    assert flag == 16 and Pz[1] == 100.0 * 1e-3
    # Lorentz-factor ceiling rescales ut to gamma_max = 50 exactly
    ut = 80.0 / np.sqrt(gcov[3, 3])
    Pz, flag = kho.floors(P, gcov, gcon, x1, x2, [1e-3, 1e-4, 0, 0, ut, 0, 0, 0])
    assert flag == 32 and abs(np.sqrt(1 + gcov[3, 3] * Pz[4] ** 2) - 50.0) < 1e-11
    # Minkowski: s = 1
    Pm = kho.make_params(ki.base_params())
    Pz, flag = kho.floors(Pm, ETA, ETA, 0.5, 0.5, [1e-9, 1e-9, 0, 0, 0, 0, 0, 0])
    assert flag == 5 and Pz[0] == 1e-6 and Pz[1] == 1e-8


# ------------------------------------------------------------------ ghost fills
def test_ghost_fills(kho):
    n = (5, 4, 3)
    rng = np.random.default_rng(0)
    Pin = rng.normal(size=(8, n[2], n[1], n[0]))
    # periodic
    g = kho.Grid(ki.base_params(n1=n[0], n2=n[1], n3=n[2]))
    g.set_prims(Pin)
    Pg = g.get_prims(with_ghosts=True)
    want = np.pad(Pin, ((0, 0), (3, 3), (3, 3), (3, 3)), mode="wrap")
    assert np.array_equal(Pg, want)
    # outflow (Minkowski: gdet = 1, plain copy) incl. edges and corners
    g = kho.Grid(ki.base_params(n1=n[0], n2=n[1], n3=n[2], bc=[kp.BC_OUTFLOW] * 6))
    g.set_prims(Pin)
    assert np.array_equal(g.get_prims(with_ghosts=True), np.pad(Pin, ((0, 0), (3, 3), (3, 3), (3, 3)), mode="edge"))
    # polar reflect in x2 with sign flips of ut2, B2; outflow x1 rescales B by gdet; periodic x3
    p = ki.config_params(3, n=(6, 5, 2))
    g = kho.Grid(p)
    Pin = rng.normal(size=(8, 2, 5, 6))
    g.set_prims(Pin)
    Pg = g.get_prims(with_ghosts=True)
    gd = g.get_geom(kho.LOC_CENT)[2]
    I = Pg[:, 3:-3, 3:-3, 3:-3]
    assert np.array_equal(I, Pin)
    sign = np.ones(8); sign[3] = sign[6] = -1
    for m in range(3):
        assert np.array_equal(Pg[:, 3:-3, 2 - m, 3:-3], sign[:, None, None] * Pin[:, :, m, :])
        assert np.array_equal(Pg[:, 3:-3, 3 + 5 + m, 3:-3], sign[:, None, None] * Pin[:, :, 4 - m, :])
        assert np.array_equal(Pg[:5, 3:-3, 3:-3, 2 - m], Pin[:5, :, :, 0])
        assert np.allclose(Pg[5:, 3:-3, 3:-3, 2 - m], Pin[5:, :, :, 0] * (gd[3:-3, 3] / gd[3:-3, 2 - m])[None, None], rtol=1e-15)
        assert np.array_equal(Pg[:, 2 - m, 3:-3, 3:-3], Pin[:, (2 - 1 - m) % 2])
    # corner: x1-ghost then x2-reflect
    assert Pg[3, 3, 2, 1] == -Pg[3, 3, 3, 1] and Pg[0, 3, 2, 1] == Pg[0, 3, 3, 1]
    # fixed: ghosts keep what set_prims(with_ghosts) wrote
    pf = ki.base_params(n1=4, n2=4, n3=4, bc=[kp.BC_FIXED] * 6)
    g = kho.Grid(pf)
    full = rng.normal(size=(8, 10, 10, 10))
    g.set_prims(full, with_ghosts=True)
    assert np.array_equal(g.get_prims(with_ghosts=True), full)


# ------------------------------------------------------------------ fix-up
def test_fixup_hand_built_neighbourhoods(kho):
    """C9 on hand-built flag patterns: the replacement is the 1/(|di|+|dj|+|dk|+1)-weighted mean of the
    good neighbours (pre-fix-up snapshot), all 26 if none is good; then floors; good zones untouched."""
    n = 5
    p = ki.base_params(n1=n, n2=n, n3=n)
    rng = np.random.default_rng(6)
    P0 = rng.uniform(0.5, 1.5, size=(8, n, n, n))
    P0[2:5] *= 0.1
    g = kho.Grid(p)
    g.set_prims(P0)
    Pg = g.get_prims(with_ghosts=True)
    pf = np.zeros((n, n, n), dtype=np.int32)
    pf[2, 2, 2] = 5                                  # isolated failure
    pf[0, 0, 0] = 2; pf[0, 0, 1] = 3                 # adjacent failures at a periodic corner
    pf[3:, 3:, 3:] = 4                               # a 2x2x2 block ...
    pfg = np.pad(pf, 3, mode="wrap")
    g.debug_fixup(pfg)
    P1 = g.get_prims(with_ghosts=True)
    nb = [(dk, dj, di) for dk in (-1, 0, 1) for dj in (-1, 0, 1) for di in (-1, 0, 1) if (dk, dj, di) != (0, 0, 0)]
    for k, j, i in np.argwhere(pf != 0):
        good = [o for o in nb if pfg[k + 3 + o[0], j + 3 + o[1], i + 3 + o[2]] == 0]
        assert good
        w = np.array([1.0 / (abs(a) + abs(b) + abs(c) + 1) for a, b, c in good])
        vals = np.array([Pg[:5, k + 3 + a, j + 3 + b, i + 3 + c] for a, b, c in good])
        want = (w[:, None] * vals).sum(0) / w.sum()
        assert np.allclose(P1[:5, k + 3, j + 3, i + 3], want, rtol=1e-14)
        assert np.array_equal(P1[5:, k + 3, j + 3, i + 3], Pg[5:, k + 3, j + 3, i + 3])     # B untouched
    ok = np.pad(pf, 3, mode="constant") == 0
    assert np.array_equal(P1[:, ok], Pg[:, ok])
    # no good neighbour at all: mean over all 26 regardless of flag
    g.set_prims(P0)
    allbad = np.ones((n + 6, n + 6, n + 6), dtype=np.int32)
    g.debug_fixup(allbad)
    P2 = g.get_prims(with_ghosts=True)
    w = np.array([1.0 / (abs(a) + abs(b) + abs(c) + 1) for a, b, c in nb])
    vals = np.array([Pg[:5, 2 + 3 + a, 2 + 3 + b, 2 + 3 + c] for a, b, c in nb])
    assert np.allclose(P2[:5, 5, 5, 5], (w[:, None] * vals).sum(0) / w.sum(), rtol=1e-14)
    # floors are applied to repaired zones: neighbours at tiny density -> result floored, fflag set
    Pt = P0.copy(); Pt[0] = 1e-9; Pt[1] = 1e-9; Pt[5:] = 0.0
    g.set_prims(Pt)
    one = np.zeros((n + 6, n + 6, n + 6), dtype=np.int32); one[5, 5, 5] = 5
    g.debug_fixup(one)
    assert g.get_prims()[0, 2, 2, 2] == 1e-6 and g.get_flags()[1][2, 2, 2] & 1
