"""GPU: kh_divB_noalloc, the allocation-free variant of kh_divB (include/kharm.h), gives what kh_divB gives.

Collected last on purpose (the suite runs with `pytest -x`).  The entry point keeps its reduction scratch in one static device
array that every call shares and that keeps the last call's contents, so every case makes TWO calls in a row on different
data -- a large divergence first (its partial maxima stay in the scratch), then a field whose divergence is round-off -- and
both must agree with kh_divB to the bar the suite uses for this quantity (the two kernels add the same terms in the same
order; REL below allows for a different contraction of the products, nothing more).
"""
import numpy as np
import pytest

import kharm_inputs as ki
from kharm_inputs import modes, torus
from kharm_inputs import params as kp

pytestmark = pytest.mark.gpu

REL = 1e-12          # relative; the round-off-sized divergences (1e-14 of B / dx) are compared to ABS as well
ABS = 1e-15


@pytest.fixture(scope="module")
def kh():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2408_01361_b200 as m
    m.lib()
    return m


def _lower_mask(p):
    return sum(1 << d for d in range(3) if p["bc"][2 * d] in (kp.BC_PERIODIC, kp.BC_BLOCK))


def _device_inputs(g, p, curved):
    """(B, gdet) of the grid's current state as device tensors in the layout kh_divB_noalloc reads."""
    import torch
    P = g.get_prims(with_ghosts=True)
    B = torch.from_numpy(np.ascontiguousarray(P[5:8])).cuda()
    gd = torch.from_numpy(np.ascontiguousarray(g.get_geom(0)[2])).cuda() if curved else None
    return B, gd


def _noalloc(kh, p, B, gd, out, stream):
    dx = [(p["xmax"][d] - p["xmin"][d]) / p[("n1", "n2", "n3")[d]] for d in range(3)]
    kh.divB_noalloc(B.data_ptr(), gd.data_ptr() if gd is not None else 0, (p["n1"], p["n2"], p["n3"]), dx, _lower_mask(p),
                    out.data_ptr(), stream.cuda_stream)


CASES = [
    ("minkowski periodic, ragged", lambda: ki.config_params(5, n=(38, 20, 14), recon=kp.RECON_MC), lambda p: modes.config5(p, seed=11, amp=1e-2), False),
    ("fmks torus, several blocks per row", lambda: ki.config_params(3, n=(72, 40, 12)), lambda p: torus.torus_state(p, seed=5), True),
]


@pytest.mark.parametrize("label,mkp,mkP,curved", CASES, ids=[c[0] for c in CASES])
def test_noalloc_divB_matches_divB_on_two_calls_in_a_row(kh, label, mkp, mkP, curved):
    import torch
    p = mkp()
    P0 = mkP(p)
    stream = torch.cuda.Stream()
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    # state 1: the field shuffled between zones -- a divergence of order |B| / dx at every corner
    rough = P0.copy()
    rng = np.random.default_rng(3)
    rough[5:8] = rng.permutation(rough[5:8].reshape(3, -1), axis=1).reshape(rough[5:8].shape) + 0.1 * rng.standard_normal(rough[5:8].shape)
    g1 = kh.Grid(p)
    g1.set_prims(rough)
    # state 2: the seeded initial state advanced three steps -- Flux-CT keeps its divergence at round-off
    g2 = kh.Grid(p)
    g2.set_prims(P0)
    dt = g2.estimate_dt()
    for _ in range(3):
        dt = g2.step(dt)
    inputs = [_device_inputs(g, p, curved) for g in (g1, g2)]
    want = [g1.divB(), g2.divB()]
    torch.cuda.synchronize()
    _noalloc(kh, p, *inputs[0], out[0:1], stream)          # warm-up: the first call on a device looks up the scratch address
    stream.synchronize()
    out.fill_(-1.0)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    _noalloc(kh, p, *inputs[0], out[0:1], stream)          # two calls in a row on one stream, no synchronisation between them
    _noalloc(kh, p, *inputs[1], out[1:2], stream)
    stream.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "kh_divB_noalloc must not allocate device memory"
    got = out.cpu().numpy()
    assert want[0] > 1e3 * max(want[1], 1e-300), (label, want)        # the two states do differ by orders of magnitude
    for a, b in zip(got, want):
        assert abs(a - b) <= REL * abs(b) + ABS, (label, got, want)
    # and once more in the other order: the small result first, the scratch full of the large call's partial maxima before it
    _noalloc(kh, p, *inputs[1], out[0:1], stream)
    _noalloc(kh, p, *inputs[0], out[1:2], stream)
    stream.synchronize()
    got = out.cpu().numpy()
    for a, b in zip(got, want[::-1]):
        assert abs(a - b) <= REL * abs(b) + ABS, (label, got, want)


def test_noalloc_divB_rejects_what_its_scratch_cannot_cover(kh):
    import torch
    B = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    n = (258, 258, 258)                                   # 257^3 interior corners > KH_NOALLOC_MAX_CORNERS
    assert 257 ** 3 > kh.NOALLOC_MAX_CORNERS >= 255 ** 3
    with pytest.raises(kh.KharmError, match="static scratch"):
        kh.divB_noalloc(B.data_ptr(), 0, n, (1.0, 1.0, 1.0), 0, out.data_ptr(), 0)       # rejected before anything touches B
    with pytest.raises(kh.KharmError, match="invalid argument"):
        kh.divB_noalloc(0, 0, (8, 8, 8), (1.0, 1.0, 1.0), 0, out.data_ptr(), 0)
    with pytest.raises(kh.KharmError, match="invalid argument"):
        kh.divB_noalloc(B.data_ptr(), 0, (8, 8, 8), (1.0, 0.0, 1.0), 0, out.data_ptr(), 0)
    torch.cuda.synchronize()
    assert float(out[0]) == -1.0                          # nothing was enqueued
    # a block without interior corners: the result is defined (0), still without allocating
    B1 = torch.zeros(3 * 7 * 7 * 7, dtype=torch.float64, device="cuda")
    kh.divB_noalloc(B1.data_ptr(), 0, (1, 1, 1), (1.0, 1.0, 1.0), 0, out.data_ptr(), 0)
    torch.cuda.synchronize()
    assert float(out[0]) == 0.0
