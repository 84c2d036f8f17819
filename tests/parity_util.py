"""Comparison metric between the CUDA path and the oracle (reading S23).

Per zone: rho, u: |d|/|ref|; velocities: |d ut^i| sqrt(g_ii) / max(sqrt(q^2), 1e-3);
field: |d B^i| sqrt(g_ii) / max(|B|, 1e-3 max_block |B|).  "After one step": max over interior zones
<= 1e-10 (BASELINE.json north_star).  "Full run": L1 = sum|d| / sum|ref| per primitive <= 1e-8.
"""
import numpy as np

from kharm_inputs import geometry

TOL_ONE_STEP = 1e-10
TOL_RUN_L1 = 1e-8
EPS = 2.220446049250313e-16


def zone_metric(p):
    """gcov at zone centres, interior, [n2, n1, 4, 4] (numpy formulas of kharm_inputs)."""
    x1, x2, _ = geometry.zone_coords(p)
    X2, X1 = np.meshgrid(x2, x1, indexing="ij")
    return geometry.gcov_native(p, X1, X2)


def rel_diff(p, got, ref):
    """Per-primitive, per-zone relative difference [8][n3][n2][n1] in the S23 metric."""
    gcov = zone_metric(p)
    gs = gcov[..., 1:, 1:]
    out = np.zeros_like(ref)
    out[0] = np.abs(got[0] - ref[0]) / np.abs(ref[0])
    out[1] = np.abs(got[1] - ref[1]) / np.abs(ref[1])
    v = np.moveaxis(ref[2:5], 0, -1)
    q = np.sqrt(np.einsum("kjia,jiab,kjib->kji", v, gs, v))
    B = np.moveaxis(ref[5:8], 0, -1)
    bn = np.sqrt(np.einsum("kjia,jiab,kjib->kji", B, gs, B))
    bfloor = 1e-3 * bn.max() if bn.max() > 0 else 1.0
    for i in range(3):
        gii = np.sqrt(gcov[..., i + 1, i + 1])[None]
        out[2 + i] = np.abs(got[2 + i] - ref[2 + i]) * gii / np.maximum(q, 1e-3)
        out[5 + i] = np.abs(got[5 + i] - ref[5 + i]) * gii / np.maximum(bn, bfloor)
    return out


def conditioning(p, ref, gamma):
    """eps (rho + b^2) / u: the inherent round-off amplification of the internal energy in U -> P
    (S16 'conditioning caveat').  b^2 is bounded by |B|^2 gamma^2-ish; we use g_ij B^i B^j."""
    gcov = zone_metric(p)
    B = np.moveaxis(ref[5:8], 0, -1)
    b2 = np.einsum("kjia,jiab,kjib->kji", B, gcov[..., 1:, 1:], B)
    return EPS * (ref[0] + b2) / ref[1]


def oracle_sensitivity(kho, p, P0, faces, dts, realizations=5, seed=100):
    """What 1-ulp noise on the INPUT does to the oracle's own result (S23c): the oracle is run on P0 (1 +- 2^-52)
    with seeded random signs, for the same steps dts, and the per-zone, per-primitive difference to its unperturbed result
    (S23 metric, maximum over the realisations) is returned, [8][n3][n2][n1].  It measures, from the oracle alone, how much
    the step amplifies round-off in each zone -- the scale on which two correct fp64 evaluations of the scheme can differ."""
    def run(P):
        g = kho.Grid(p, omp=True)
        g.set_prims(P)
        if faces is not None:
            g.set_face_B(*faces)
        for dt in dts:
            g.step(dt)
        return g.get_prims()
    ref = run(P0)
    worst = np.zeros_like(ref)
    for r in range(realizations):
        rng = np.random.default_rng(seed + r)
        worst = np.maximum(worst, rel_diff(p, run(P0 * (1.0 + 2.0 ** -52 * rng.choice([-1.0, 1.0], size=P0.shape))), ref))
    return worst


def l1_diff(p, got, ref):
    """L1 difference per primitive: sum|d| / sum|ref| for rho, u; for the vector components the denominator
    is the sum of the vector's norm (sum sqrt(g_ii)|d v^i| / sum |v|), so that a component that vanishes by
    symmetry is judged against the size of the vector it belongs to (S23)."""
    gcov = zone_metric(p)
    gs = gcov[..., 1:, 1:]
    out = np.zeros(8)
    for v in (0, 1):
        out[v] = np.abs(got[v] - ref[v]).sum() / max(np.abs(ref[v]).sum(), 1e-300)
    for base in (2, 5):
        vec = np.moveaxis(ref[base:base + 3], 0, -1)
        norm = np.sqrt(np.einsum("kjia,jiab,kjib->kji", vec, gs, vec)).sum()
        for i in range(3):
            gii = np.sqrt(gcov[..., i + 1, i + 1])[None]
            out[base + i] = (np.abs(got[base + i] - ref[base + i]) * gii).sum() / max(norm, 1e-300)
    return out


def bondi_errors(p, P1, P0, rmin=2.5):
    """Config 2 ("error against the analytic steady state"): L1 difference between a state and the analytic initial
    state over the zones with r > rmin (outside the horizon and its boundary layer), [rho, u, velocity, field] -- scalars
    relative to sum |ref|, vectors as sum sqrt(g_ii) |d v^i| over i relative to the sum of the vector's norm (S23)."""
    x1, _, _ = geometry.zone_coords(p)
    keep = np.exp(x1) > rmin
    gcov = zone_metric(p)
    out = []
    for v in (0, 1):
        out.append(np.abs(P1[v] - P0[v])[..., keep].sum() / np.abs(P0[v])[..., keep].sum())
    for base in (2, 5):
        vec = np.moveaxis(P0[base:base + 3], 0, -1)
        norm = np.sqrt(np.einsum("kjia,jiab,kjib->kji", vec, gcov[..., 1:, 1:], vec))[..., keep].sum()
        num = sum((np.abs(P1[base + i] - P0[base + i]) * np.sqrt(gcov[..., i + 1, i + 1])[None])[..., keep].sum() for i in range(3))
        out.append(num / norm)
    return np.array(out)
