"""Pins of the oracle's geometry (C1) against closed forms and identities -- none of them re-types
the oracle's own code path: sqrt(-g) and lapse closed forms, g*ginv = 1, contraction identity of the
connection, finite differences, and the FMKS map's end points / symmetry / the paper's 2-8x."""
import os

import numpy as np
import pytest

import kharm_inputs as ki
from kharm_inputs import params as kp

A = 0.9375


def _params(kho, coords, **kw):
    return kho.make_params(ki.base_params(coords=coords, a=A, xmin=[0.2, 0.0, 0.0], xmax=[3.0, 1.0, 6.28], **kw))


def test_minkowski_is_flat(kho):
    P = _params(kho, kp.MINKOWSKI)
    gcov, gcon, gdet, alpha = kho.metric(P, 0.3, 0.7)
    eta = np.diag([-1.0, 1, 1, 1])
    assert np.array_equal(gcov, eta) and np.array_equal(gcon, eta) and gdet == 1.0 and alpha == 1.0
    assert np.abs(kho.conn(P, 0.3, 0.7)).max() == 0.0


@pytest.mark.parametrize("r,th", [(1.5, 0.3), (3.7, 1.1), (20.0, 2.9), (800.0, 1.5707)])
def test_ks_closed_forms(kho, r, th):
    P = _params(kho, kp.KS)
    gcov, gcon, gdet, alpha = kho.metric(P, r, th)
    Sig = r * r + A * A * np.cos(th) ** 2
    assert abs(gdet / (Sig * np.sin(th)) - 1) < 1e-13                 # sqrt(-g)_KS = Sigma sin(theta)
    assert abs(alpha / (1 + 2 * r / Sig) ** -0.5 - 1) < 1e-13          # lapse
    assert np.abs(gcov @ gcon - np.eye(4)).max() < 1e-12
    assert np.array_equal(gcov, gcov.T) and np.allclose(gcon, gcon.T, atol=1e-15)
    # signature (-+++)
    ev = np.linalg.eigvalsh(gcov)
    assert (ev < 0).sum() == 1 and (ev > 0).sum() == 3


def test_ks_a0_is_schwarzschild_ingoing(kho):
    P = kho.make_params(ki.base_params(coords=kp.KS, a=0.0))
    r, th = 5.0, 0.9
    gcov = kho.metric(P, r, th)[0]
    want = np.zeros((4, 4))
    want[0, 0] = -(1 - 2 / r); want[0, 1] = want[1, 0] = 2 / r; want[1, 1] = 1 + 2 / r
    want[2, 2] = r * r; want[3, 3] = (r * np.sin(th)) ** 2
    assert np.abs(gcov - want).max() < 1e-14
    # radial null ray dr/dt = -1 (ingoing) is null in these coordinates
    k = np.array([1.0, -1.0, 0, 0])
    assert abs(k @ gcov @ k) < 1e-14


def test_fmks_map_properties(kho, golden):
    gold = golden
    p = ki.config_params(3)
    P = kho.make_params(p)
    for x1 in (p["xmin"][0], 1.0, 3.0, p["xmax"][0]):
        assert abs(kho.embed(P, [x1, 0.0, 0])[1]) < 1e-14                  # theta(x2=0) = 0
        assert abs(kho.embed(P, [x1, 1.0, 0])[1] - np.pi) < 1e-14          # theta(1) = pi
        assert abs(kho.embed(P, [x1, 0.5, 0])[1] - np.pi / 2) < 1e-14
        x2 = np.linspace(0, 1, 401)
        th = np.array([kho.embed(P, [x1, v, 0])[1] for v in x2])
        assert np.all(np.diff(th) > 0)                                     # monotone
        assert np.abs(th + th[::-1] - np.pi).max() < 1e-13                 # theta(1-x2) = pi - theta(x2)
        assert abs(kho.embed(P, [x1, 0.3, 0])[0] - np.exp(x1)) < 1e-12 * np.exp(x1)
    # far from the hole the map tends to the hslope-only map theta_G
    thG = np.pi * 0.2 + 0.5 * (1 - p["hslope"]) * np.sin(2 * np.pi * 0.2)
    assert abs(kho.embed(P, [40.0, 0.2, 0])[1] - thG) < 1e-8
    # polar zones are widened near the horizon: first zone's dtheta vs uniform spacing, paper's "2-8x"
    gain = kho.embed(P, [p["xmin"][0], 1.0 / p["n2"], 0])[1] / (np.pi / p["n2"])
    assert gold["fmks_dt_gain_min"] <= gain <= gold["fmks_dt_gain_max"]
    assert abs(kho.embed(P, [p["xmin"][0], 1.0 / 128, 0])[1] - 0.1829) < 1e-4


@pytest.mark.parametrize("x1,x2", [(0.3, 0.05), (1.2, 0.31), (2.3, 0.5), (5.0, 0.93), (6.8, 0.999)])
def test_fmks_metric_closed_forms(kho, x1, x2):
    p = ki.config_params(3)
    P = kho.make_params(p)
    gcov, gcon, gdet, alpha = kho.metric(P, x1, x2)
    r, th, _ = kho.embed(P, [x1, x2, 0])
    h = 1e-6
    dth2 = (kho.embed(P, [x1, x2 + h, 0])[1] - kho.embed(P, [x1, x2 - h, 0])[1]) / (2 * h)
    Sig = r * r + A * A * np.cos(th) ** 2
    assert abs(gdet / (Sig * np.sin(th) * r * dth2) - 1) < 1e-8          # sqrt(-g) = Sigma sin(th) r dtheta/dx2
    assert abs(alpha / (1 + 2 * r / Sig) ** -0.5 - 1) < 1e-12             # lapse is a scalar under spatial maps
    assert np.abs(gcov @ gcon - np.eye(4)).max() < 1e-10
    # independent numpy construction of the same metric (kharm_inputs.geometry)
    from kharm_inputs import geometry
    g2 = geometry.gcov_native(p, x1, x2)
    assert np.abs(gcov - g2).max() <= 1e-13 * np.abs(gcov).max()


@pytest.mark.parametrize("coords", [kp.KS, kp.FMKS])
def test_connection_identities(kho, coords):
    p = ki.config_params(3)
    p["coords"] = coords
    if coords == kp.KS:
        p["xmin"], p["xmax"] = [1.3, 0.0, 0.0], [50.0, np.pi, 2 * np.pi]
    P = kho.make_params(p)
    rng = np.random.default_rng(5)
    for _ in range(10):
        x1 = rng.uniform(p["xmin"][0], min(p["xmax"][0], 6.0))
        x2 = rng.uniform(0.03, 0.97) * p["xmax"][1]
        cn = kho.conn(P, x1, x2)
        assert np.abs(cn - cn.transpose(0, 2, 1)).max() < 1e-12 * max(1, np.abs(cn).max())   # symmetric
        # Gamma^mu_{mu nu} = d_nu ln sqrt(-g)
        h = 1e-5

        def dlog(e1, e2, hh):
            return (np.log(kho.metric(P, x1 + e1 * hh, x2 + e2 * hh)[2]) - np.log(kho.metric(P, x1 - e1 * hh, x2 - e2 * hh)[2])) / (2 * hh)

        d1 = (4 * dlog(1, 0, 1e-4) - dlog(1, 0, 2e-4)) / 3      # Richardson-extrapolated centred differences
        d2 = (4 * dlog(0, 1, 1e-4) - dlog(0, 1, 2e-4)) / 3
        tr = np.einsum("mmn->n", cn)
        assert abs(tr[0]) < 1e-12 and abs(tr[3]) < 1e-12
        assert abs(tr[1] - d1) < 1e-7 * max(1, abs(d1)) and abs(tr[2] - d2) < 1e-7 * max(1, abs(d2))
        # exact derivative agrees with Richardson-extrapolated centred differences
        c1, c2 = kho.conn_fd(P, x1, x2, 2e-4), kho.conn_fd(P, x1, x2, 1e-4)
        rich = (4 * c2 - c1) / 3
        assert np.abs(cn - rich).max() < 1e-8 * max(1, np.abs(cn).max())
        # metric compatibility: d_k g_mn = Gamma_{m,nk} + Gamma_{n,mk}
        gcov = kho.metric(P, x1, x2)[0]
        low = np.einsum("la,amn->lmn", gcov, cn)
        for k, (e1, e2) in ((1, (h, 0)), (2, (0, h))):
            dg = (kho.metric(P, x1 + e1, x2 + e2)[0] - kho.metric(P, x1 - e1, x2 - e2)[0]) / (2 * h)
            assert np.abs(dg - (low[:, :, k] + low[:, :, k].T)).max() < 1e-5 * max(1, np.abs(dg).max())


def test_schwarzschild_connection_textbook(kho):
    # a = 0 KS: Gamma^theta_{r theta} = 1/r, Gamma^phi_{theta phi} = cot(theta), Gamma^r_{theta theta} = -(r - 2)
    P = kho.make_params(ki.base_params(coords=kp.KS, a=0.0))
    r, th = 7.0, 1.1
    cn = kho.conn(P, r, th)
    assert abs(cn[2, 1, 2] - 1 / r) < 1e-14
    assert abs(cn[3, 2, 3] - 1 / np.tan(th)) < 1e-13
    assert abs(cn[1, 2, 2] + (r - 2)) < 1e-13
    assert abs(cn[2, 3, 3] + np.sin(th) * np.cos(th)) < 1e-14


def test_grid_tables_and_polar_faces(kho):
    p = ki.config_params(3, n=(16, 12, 4))
    g = kho.Grid(p)
    P = kho.make_params(p)
    gcov, gcon, gdet, alpha = g.get_geom(kho.LOC_FACE2)
    assert np.all(gdet[3, :] == 0) and np.all(gdet[3 + 12, :] == 0) and np.all(gcon[3] == 0)   # S7: axis faces zeroed
    assert np.all(gdet[4:15, :] > 0)
    gc, _, gd, _ = g.get_geom(kho.LOC_CENT)
    dx1 = (p["xmax"][0] - p["xmin"][0]) / 16
    i, j = 5, 7
    ref = kho.metric(P, p["xmin"][0] + (i + 0.5) * dx1, (j + 0.5) / 12)
    assert np.array_equal(gc[j + 3, i + 3], ref[0]) and gd[j + 3, i + 3] == ref[2]
    f1 = g.get_geom(kho.LOC_FACE1)
    ref = kho.metric(P, p["xmin"][0] + i * dx1, (j + 0.5) / 12)
    assert np.array_equal(f1[0][j + 3, i + 3], ref[0])
    cn = g.get_conn()
    assert np.array_equal(cn[j + 3, i + 3], kho.conn(P, p["xmin"][0] + (i + 0.5) * dx1, (j + 0.5) / 12))
