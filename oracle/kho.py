"""ctypes binding of the CPU oracle (oracle/kho.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It never imports the CUDA package.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MINKOWSKI, KS, FMKS = 0, 1, 2
BC_PERIODIC, BC_OUTFLOW, BC_POLAR, BC_FIXED = 0, 1, 2, 3
RECON_MC, RECON_WENO5 = 0, 1
LOC_CENT, LOC_FACE1, LOC_FACE2, LOC_FACE3 = 0, 1, 2, 3
NG = 3


class Params(C.Structure):
    _fields_ = [
        ("coords", C.c_int), ("a", C.c_double),
        ("hslope", C.c_double), ("poly_xt", C.c_double), ("poly_alpha", C.c_double), ("mks_smooth", C.c_double),
        ("n1", C.c_int), ("n2", C.c_int), ("n3", C.c_int),
        ("xmin", C.c_double * 3), ("xmax", C.c_double * 3),
        ("bc", C.c_int * 6),
        ("gamma", C.c_double), ("cfl", C.c_double), ("recon", C.c_int),
        ("rho_min", C.c_double), ("u_min", C.c_double), ("r_char", C.c_double),
        ("bsq_over_rho_max", C.c_double), ("bsq_over_u_max", C.c_double), ("u_over_rho_max", C.c_double),
        ("gamma_max", C.c_double), ("dt_growth_max", C.c_double), ("inverter", C.c_int), ("fofc", C.c_int), ("floor_frame", C.c_int), ("transport", C.c_int), ("emf", C.c_int),
    ]


def make_params(d):
    """dict (kharm_inputs.params style) -> Params"""
    p = Params()
    for k, v in d.items():
        if k in ("xmin", "xmax"):
            setattr(p, k, (C.c_double * 3)(*v))
        elif k == "bc":
            p.bc = (C.c_int * 6)(*v)
        else:
            setattr(p, k, v)
    return p


_libs = {}
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _ptr(a):
    return a.ctypes.data_as(_dp)


def lib(omp=False):
    key = "omp" if omp else "st"
    if key not in _libs:
        san = os.environ.get("KHO_SANITIZE") == "1"        # the ASan / UBSan build of the same source (oracle/build.py --sanitize)
        paths = _build.build(sanitize=san)
        L = C.CDLL(paths[2] if san else (paths[1] if omp else paths[0]))
        L.kho_strerror.restype = C.c_char_p
        for name in ("kho_embed", "kho_metric", "kho_conn", "kho_conn_fd", "kho_fourvec", "kho_prim_to_flux",
                     "kho_stress", "kho_vchar", "kho_recon", "kho_llf", "kho_source"):
            getattr(L, name).restype = None
        _libs[key] = L
    return _libs[key]


def _chk(rc):
    if rc != 0:
        raise RuntimeError("oracle: " + lib().kho_strerror(rc).decode())


def _a(x, n=None):
    a = np.ascontiguousarray(x, dtype=np.float64)
    if n is not None:
        assert a.size == n, (a.size, n)
    return a


# ---- point-wise pieces -------------------------------------------------------------------
def embed(params, X):
    out = np.zeros(3)
    lib().kho_embed(C.byref(params), _ptr(_a(X, 3)), _ptr(out))
    return out


def metric(params, x1, x2):
    gcov, gcon = np.zeros(16), np.zeros(16)
    gdet, alpha = C.c_double(), C.c_double()
    lib().kho_metric(C.byref(params), C.c_double(x1), C.c_double(x2), _ptr(gcov), _ptr(gcon), C.byref(gdet), C.byref(alpha))
    return gcov.reshape(4, 4), gcon.reshape(4, 4), gdet.value, alpha.value


def conn(params, x1, x2):
    out = np.zeros(64)
    lib().kho_conn(C.byref(params), C.c_double(x1), C.c_double(x2), _ptr(out))
    return out.reshape(4, 4, 4)


def conn_fd(params, x1, x2, h):
    out = np.zeros(64)
    lib().kho_conn_fd(C.byref(params), C.c_double(x1), C.c_double(x2), C.c_double(h), _ptr(out))
    return out.reshape(4, 4, 4)


def fourvec(gcov, gcon, P):
    out = np.zeros(17)
    lib().kho_fourvec(_ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), _ptr(_a(P, 8)), _ptr(out))
    return dict(ucon=out[0:4].copy(), ucov=out[4:8].copy(), bcon=out[8:12].copy(), bcov=out[12:16].copy(), bsq=out[16])


def prim_to_flux(gcov, gcon, gdet, P, gamma, d):
    out = np.zeros(8)
    lib().kho_prim_to_flux(_ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), C.c_double(gdet), _ptr(_a(P, 8)), C.c_double(gamma), C.c_int(d), _ptr(out))
    return out


def stress(gcov, gcon, P, gamma):
    out = np.zeros(16)
    lib().kho_stress(_ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), _ptr(_a(P, 8)), C.c_double(gamma), _ptr(out))
    return out.reshape(4, 4)


def vchar(gcov, gcon, P, gamma, d):
    vmax, vmin = C.c_double(), C.c_double()
    lib().kho_vchar(_ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), _ptr(_a(P, 8)), C.c_double(gamma), C.c_int(d), C.byref(vmax), C.byref(vmin))
    return vmax.value, vmin.value


def recon(kind, q):
    l, r = C.c_double(), C.c_double()
    lib().kho_recon(C.c_int(kind), _ptr(_a(q, 5)), C.byref(l), C.byref(r))
    return l.value, r.value


def llf(gcov, gcon, gdet, PL, PR, gamma, d):
    F = np.zeros(8)
    ctop = C.c_double()
    lib().kho_llf(_ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), C.c_double(gdet), _ptr(_a(PL, 8)), _ptr(_a(PR, 8)), C.c_double(gamma), C.c_int(d), _ptr(F), C.byref(ctop))
    return F, ctop.value


def source(gcov, gcon, gdet, cn, P, gamma):
    S = np.zeros(8)
    lib().kho_source(_ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), C.c_double(gdet), _ptr(_a(cn, 64)), _ptr(_a(P, 8)), C.c_double(gamma), _ptr(S))
    return S


def u2p(gcov, gcon, gdet, U, Pguess, gamma):
    P = np.zeros(8)
    flag = lib().kho_u2p(_ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), C.c_double(gdet), _ptr(_a(U, 8)), _ptr(_a(Pguess, 8)), C.c_double(gamma), _ptr(P))
    return P, flag


def u2p_kastaun(gcov, gcon, gdet, U, Pguess, gamma):
    P = np.zeros(8)
    flag = lib().kho_u2p_kastaun(_ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), C.c_double(gdet), _ptr(_a(U, 8)), _ptr(_a(Pguess, 8)), C.c_double(gamma), _ptr(P))
    return P, flag


def floors(params, gcov, gcon, x1, x2, P):
    Pz = _a(P, 8).copy()
    flag = lib().kho_floors(C.byref(params), _ptr(_a(gcov, 16)), _ptr(_a(gcon, 16)), C.c_double(x1), C.c_double(x2), _ptr(Pz))
    return Pz, flag


def flux_ct_arrays(params, F1, F2, F3):
    """In place on three [8][n3+6][n2+6][n1+6] arrays."""
    for F in (F1, F2, F3):
        assert F.dtype == np.float64 and F.flags.c_contiguous
    _chk(lib().kho_flux_ct_arrays(C.byref(params), _ptr(F1), _ptr(F2), _ptr(F3)))


# ---- grid ------------------------------------------------------------------------------------
class Grid:
    def __init__(self, params, omp=False):
        self.params = params if isinstance(params, Params) else make_params(params)
        self.L = lib(omp)
        self.h = C.c_void_p()
        _chk(self.L.kho_grid_create(C.byref(self.params), C.byref(self.h)))
        p = self.params
        self.n = (p.n1, p.n2, p.n3)
        self.shape_int = (8, p.n3, p.n2, p.n1)
        self.shape_gh = (8, p.n3 + 2 * NG, p.n2 + 2 * NG, p.n1 + 2 * NG)

    def close(self):
        if self.h:
            self.L.kho_grid_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_prims(self, P, with_ghosts=False):
        P = _a(P)
        assert P.shape == (self.shape_gh if with_ghosts else self.shape_int), P.shape
        _chk(self.L.kho_set_prims(self.h, _ptr(P), int(with_ghosts)))

    def get_prims(self, with_ghosts=False):
        out = np.zeros(self.shape_gh if with_ghosts else self.shape_int)
        _chk(self.L.kho_get_prims(self.h, _ptr(out), int(with_ghosts)))
        return out

    def get_cons(self):
        out = np.zeros(self.shape_int)
        _chk(self.L.kho_get_cons(self.h, _ptr(out)))
        return out

    def get_flags(self):
        pf = np.zeros(self.shape_int[1:], dtype=np.int32)
        ff = np.zeros(self.shape_int[1:], dtype=np.int32)
        _chk(self.L.kho_get_flags(self.h, pf.ctypes.data_as(_ip), ff.ctypes.data_as(_ip)))
        return pf, ff

    def estimate_dt(self):
        dt = C.c_double()
        _chk(self.L.kho_estimate_dt(self.h, C.byref(dt)))
        return dt.value

    def step(self, dt):
        nxt = C.c_double()
        _chk(self.L.kho_step(self.h, C.c_double(dt), C.byref(nxt)))
        return nxt.value

    def divB(self):
        m = C.c_double()
        _chk(self.L.kho_divB(self.h, C.byref(m)))
        return m.value

    def get_flux(self, d):
        F = np.zeros(self.shape_gh)
        ct = np.zeros(self.shape_gh[1:])
        _chk(self.L.kho_get_flux(self.h, C.c_int(d), _ptr(F), _ptr(ct)))
        return F, ct

    def get_emf(self, d):
        e = np.zeros(self.shape_gh[1:])
        _chk(self.L.kho_get_emf(self.h, C.c_int(d), _ptr(e)))
        return e

    def get_geom(self, loc):
        n2d = self.shape_gh[2] * self.shape_gh[3]
        gcov, gcon, gdet, alpha = np.zeros((n2d, 16)), np.zeros((n2d, 16)), np.zeros(n2d), np.zeros(n2d)
        _chk(self.L.kho_get_geom(self.h, C.c_int(loc), _ptr(gcov), _ptr(gcon), _ptr(gdet), _ptr(alpha)))
        s = self.shape_gh[2:]
        return gcov.reshape(s + (4, 4)), gcon.reshape(s + (4, 4)), gdet.reshape(s), alpha.reshape(s)

    def get_conn(self):
        n2d = self.shape_gh[2] * self.shape_gh[3]
        cn = np.zeros((n2d, 64))
        _chk(self.L.kho_get_conn(self.h, _ptr(cn)))
        return cn.reshape(self.shape_gh[2:] + (4, 4, 4))

    def debug_predictor(self, dt):
        _chk(self.L.kho_debug_predictor(self.h, C.c_double(dt)))

    def debug_fixup(self, pflag_with_ghosts):
        pf = np.ascontiguousarray(pflag_with_ghosts, dtype=np.int32)
        assert pf.shape == self.shape_gh[1:]
        _chk(self.L.kho_debug_fixup(self.h, pf.ctypes.data_as(_ip)))

    def set_face_B(self, f1, f2, f3):
        a = [np.ascontiguousarray(f, dtype=np.float64) for f in (f1, f2, f3)]
        assert all(x.shape == self.shape_gh[1:] for x in a)
        _chk(self.L.kho_set_face_B(self.h, *[x.ctypes.data_as(_dp) for x in a]))

    def get_face_B(self):
        a = [np.empty(self.shape_gh[1:]) for _ in range(3)]
        _chk(self.L.kho_get_face_B(self.h, *[x.ctypes.data_as(_dp) for x in a]))
        return a

    def divB_face(self):
        m = C.c_double()
        _chk(self.L.kho_divB_face(self.h, C.byref(m)))
        return m.value

    def debug_emf(self):
        _chk(self.L.kho_debug_emf(self.h))

    def debug_fofc(self, mask_with_ghosts):
        m = np.ascontiguousarray(mask_with_ghosts, dtype=np.int32)
        assert m.shape == self.shape_gh[1:]
        _chk(self.L.kho_debug_fofc(self.h, m.ctypes.data_as(_ip)))

    def fill_ghosts(self):
        _chk(self.L.kho_fill_ghosts(self.h))
