"""ctypes binding of libkharm.so (include/kharm.h): same names, argument marshalling only.

PyTorch supplies device memory and the CUDA stream; every step of the path runs in the library's
kernels.  Missing library or missing GPU raise KharmError -- there is no fallback of any kind.
"""
import ctypes as C
import os

import numpy as np

MINKOWSKI, KS, FMKS = 0, 1, 2
BC_PERIODIC, BC_OUTFLOW, BC_POLAR, BC_FIXED, BC_BLOCK = 0, 1, 2, 3, 4
RECON_MC, RECON_WENO5 = 0, 1
INV_1DW, INV_KASTAUN = 0, 1
LOC_CENT, LOC_FACE1, LOC_FACE2, LOC_FACE3 = 0, 1, 2, 3
KERNEL_KINDS = ("flux1", "flux2", "flux3", "emf", "update", "fill", "fixup", "fofc")     # KH_K_* of include/kharm.h
MEM_DEVICE, MEM_HOST = 0, 1
NG = 3

EXPORTED_SYMBOLS = (
    "kh_grid_create", "kh_grid_destroy", "kh_set_prims", "kh_get_prims", "kh_get_cons", "kh_get_flags",
    "kh_estimate_dt", "kh_step", "kh_divB", "kh_set_face_B", "kh_get_face_B", "kh_divB_face", "kh_count_flags", "kh_get_geom", "kh_get_conn", "kh_get_flux",
    "kh_get_emf", "kh_debug_fixup", "kh_debug_predictor", "kh_launch_count", "kh_set_graph", "kh_set_profile", "kh_get_profile", "kh_measure_fp64_peak", "kh_strerror",
    "kh_last_cuda_error", "kh_get_stream", "kh_sync", "kh_link_blocks", "kh_exchange_halos", "kh_step_blocks",
    "kh_divB_noalloc",
)


class KharmError(RuntimeError):
    pass


class Params(C.Structure):
    """Mirror of kh_params (include/kharm.h)."""
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
    p = Params()
    for k, v in d.items():
        if k in ("xmin", "xmax"):
            setattr(p, k, (C.c_double * 3)(*v))
        elif k == "bc":
            p.bc = (C.c_int * 6)(*v)
        else:
            setattr(p, k, v)
    return p


_LIB = None
LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libkharm.so")


def lib():
    """Load libkharm.so (built in-tree by paper_2408_01361_b200/build.py); raises if it is missing."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise KharmError("libkharm.so not built: run `python -m paper_2408_01361_b200.build` (needs nvcc); "
                             "there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        L.kh_strerror.restype = C.c_char_p
        L.kh_last_cuda_error.restype = C.c_char_p
        L.kh_launch_count.restype = C.c_longlong
        L.kh_launch_count.argtypes = [C.c_void_p]
        L.kh_grid_create.argtypes = [C.POINTER(Params), C.c_void_p, C.POINTER(C.c_void_p)]
        L.kh_grid_destroy.argtypes = [C.c_void_p]
        L.kh_set_prims.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        L.kh_get_prims.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        L.kh_get_cons.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.kh_get_flags.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.kh_estimate_dt.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.kh_step.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        L.kh_divB.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.kh_divB_face.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.kh_set_face_B.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.kh_get_face_B.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.kh_count_flags.argtypes = [C.c_void_p, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
        L.kh_get_geom.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.kh_get_conn.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.kh_get_flux.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int]
        L.kh_get_emf.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int]
        L.kh_debug_fixup.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.kh_debug_predictor.argtypes = [C.c_void_p, C.c_double]
        L.kh_set_graph.argtypes = [C.c_void_p, C.c_int]
        L.kh_set_profile.argtypes = [C.c_void_p, C.c_int]
        L.kh_get_profile.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.kh_measure_fp64_peak.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.kh_get_stream.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
        L.kh_sync.argtypes = [C.c_void_p]
        L.kh_link_blocks.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.kh_exchange_halos.argtypes = [C.POINTER(C.c_void_p), C.c_int]
        L.kh_step_blocks.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.POINTER(C.c_double)]
        L.kh_divB_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                      C.c_void_p, C.c_void_p]
        _LIB = L
    return _LIB


def _chk(rc):
    if rc != 0:
        L = lib()
        raise KharmError("kharm: %s [%s]" % (L.kh_strerror(rc).decode(), L.kh_last_cuda_error().decode()))


def _np_ptr(a):
    return C.c_void_p(a.ctypes.data)


def measure_fp64_peak():
    """(TFLOP/s, implied SM MHz at 64 fp64 FMA lanes per SM) from the library's DFMA-chain kernel."""
    tf, mhz = C.c_double(), C.c_double()
    _chk(lib().kh_measure_fp64_peak(C.byref(tf), C.byref(mhz)))
    return tf.value, mhz.value


NOALLOC_MAX_CORNERS = 16777216      # KH_NOALLOC_MAX_CORNERS


def divB_noalloc(B_ptr, gdet_ptr, n, dx, lower_mask, out_ptr, stream=0):
    """kh_divB_noalloc: B_ptr, gdet_ptr (0 = Minkowski) and out_ptr are DEVICE addresses (ints); n = (n1, n2, n3), dx likewise.
    Enqueues on `stream` and returns; the caller synchronises before reading the double at out_ptr."""
    _chk(lib().kh_divB_noalloc(C.c_void_p(B_ptr), C.c_void_p(gdet_ptr or None), int(n[0]), int(n[1]), int(n[2]), float(dx[0]),
                               float(dx[1]), float(dx[2]), int(lower_mask), C.c_void_p(out_ptr), C.c_void_p(stream or None)))


def _handles(blocks):
    return (C.c_void_p * len(blocks))(*[b.h for b in blocks])


def link_blocks(lo, hi, direction):
    """`hi` continues `lo` across lo's upper side in direction 1..3 (both sides KH_BC_BLOCK)."""
    _chk(lib().kh_link_blocks(lo.h, hi.h, int(direction)))


def exchange_halos(blocks):
    _chk(lib().kh_exchange_halos(_handles(blocks), len(blocks)))


def step_blocks(blocks, dt, sync=True):
    """One predictor-corrector step of several linked blocks together; returns the common dt_next (sync=True)."""
    if sync:
        nxt = C.c_double()
        _chk(lib().kh_step_blocks(_handles(blocks), len(blocks), C.c_double(dt), C.byref(nxt)))
        return nxt.value
    _chk(lib().kh_step_blocks(_handles(blocks), len(blocks), C.c_double(dt), None))
    return None


class Grid:
    """One mesh block on one GPU.  Host numpy arrays or CUDA torch tensors are accepted wherever a
    buffer is passed; results come back as numpy (host) or fill the given torch tensor (device)."""

    def __init__(self, params, stream=None):
        self.params = params if isinstance(params, Params) else make_params(params)
        self.L = lib()
        self.h = C.c_void_p()
        if stream is None:
            try:
                import torch
                if torch.cuda.is_available():
                    stream = torch.cuda.current_stream().cuda_stream
            except ImportError:
                stream = 0
        self.stream = int(stream or 0)
        _chk(self.L.kh_grid_create(C.byref(self.params), C.c_void_p(self.stream), C.byref(self.h)))
        p = self.params
        self.n = (p.n1, p.n2, p.n3)
        self.shape_int = (8, p.n3, p.n2, p.n1)
        self.shape_gh = (8, p.n3 + 2 * NG, p.n2 + 2 * NG, p.n1 + 2 * NG)
        self.nzones = p.n1 * p.n2 * p.n3

    def close(self):
        if getattr(self, "h", None) and self.h:
            self.L.kh_grid_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- marshalling helpers
    @staticmethod
    def _is_torch(x):
        return type(x).__module__.startswith("torch")

    def _in(self, x, shape, dtype=np.float64):
        if self._is_torch(x):
            assert x.is_cuda and x.is_contiguous() and tuple(x.shape) == tuple(shape), (x.shape, shape)
            return C.c_void_p(x.data_ptr()), MEM_DEVICE, x
        a = np.ascontiguousarray(x, dtype=dtype)
        assert a.shape == tuple(shape), (a.shape, shape)
        return _np_ptr(a), MEM_HOST, a

    def _out(self, out, shape, dtype=np.float64):
        if out is None:
            out = np.empty(shape, dtype=dtype)
        if self._is_torch(out):
            assert out.is_cuda and out.is_contiguous() and tuple(out.shape) == tuple(shape)
            return C.c_void_p(out.data_ptr()), MEM_DEVICE, out
        assert out.flags.c_contiguous and out.shape == tuple(shape) and out.dtype == dtype
        return _np_ptr(out), MEM_HOST, out

    # ---- the calls of include/kharm.h
    def set_prims(self, P, with_ghosts=False):
        ptr, mem, keep = self._in(P, self.shape_gh if with_ghosts else self.shape_int)
        _chk(self.L.kh_set_prims(self.h, ptr, int(with_ghosts), mem))

    def get_prims(self, with_ghosts=False, out=None):
        ptr, mem, out = self._out(out, self.shape_gh if with_ghosts else self.shape_int)
        _chk(self.L.kh_get_prims(self.h, ptr, int(with_ghosts), mem))
        return out

    def get_cons(self, out=None):
        ptr, mem, out = self._out(out, self.shape_int)
        _chk(self.L.kh_get_cons(self.h, ptr, mem))
        return out

    def get_flags(self):
        pf = np.empty(self.shape_int[1:], dtype=np.int32)
        ff = np.empty(self.shape_int[1:], dtype=np.int32)
        _chk(self.L.kh_get_flags(self.h, _np_ptr(pf), _np_ptr(ff), MEM_HOST))
        return pf, ff

    def estimate_dt(self):
        dt = C.c_double()
        _chk(self.L.kh_estimate_dt(self.h, C.byref(dt)))
        return dt.value

    def step(self, dt, sync=True):
        """One predictor-corrector step.  dt <= 0 reuses the device-resident dt_next.  sync=False returns
        None without a host round trip."""
        if sync:
            nxt = C.c_double()
            _chk(self.L.kh_step(self.h, C.c_double(dt), C.byref(nxt)))
            return nxt.value
        _chk(self.L.kh_step(self.h, C.c_double(dt), None))
        return None

    def divB(self):
        m = C.c_double()
        _chk(self.L.kh_divB(self.h, C.byref(m)))
        return m.value

    def set_face_B(self, f1, f2, f3):
        """Face field of the face-centred CT transport (three arrays with ghosts); also sets the zone-centred field."""
        a = [np.ascontiguousarray(f, dtype=np.float64) for f in (f1, f2, f3)]
        assert all(x.shape == self.shape_gh[1:] for x in a)
        _chk(self.L.kh_set_face_B(self.h, _np_ptr(a[0]), _np_ptr(a[1]), _np_ptr(a[2]), MEM_HOST))

    def get_face_B(self):
        a = [np.empty(self.shape_gh[1:]) for _ in range(3)]
        _chk(self.L.kh_get_face_B(self.h, _np_ptr(a[0]), _np_ptr(a[1]), _np_ptr(a[2]), MEM_HOST))
        return a

    def divB_face(self):
        m = C.c_double()
        _chk(self.L.kh_divB_face(self.h, C.byref(m)))
        return m.value

    def count_flags(self):
        a, b = C.c_longlong(), C.c_longlong()
        _chk(self.L.kh_count_flags(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def get_geom(self, loc):
        s = self.shape_gh[2:]
        n2d = s[0] * s[1]
        gcov, gcon, gdet, alpha = np.empty((n2d, 16)), np.empty((n2d, 16)), np.empty(n2d), np.empty(n2d)
        _chk(self.L.kh_get_geom(self.h, loc, _np_ptr(gcov), _np_ptr(gcon), _np_ptr(gdet), _np_ptr(alpha), MEM_HOST))
        return gcov.reshape(s + (4, 4)), gcon.reshape(s + (4, 4)), gdet.reshape(s), alpha.reshape(s)

    def get_conn(self):
        s = self.shape_gh[2:]
        cn = np.empty((s[0] * s[1], 64))
        _chk(self.L.kh_get_conn(self.h, _np_ptr(cn), MEM_HOST))
        return cn.reshape(s + (4, 4, 4))

    def get_flux(self, d):
        F = np.empty(self.shape_gh)
        ct = np.empty(self.shape_gh[1:])
        _chk(self.L.kh_get_flux(self.h, d, _np_ptr(F), _np_ptr(ct), MEM_HOST))
        return F, ct

    def get_emf(self, d):
        e = np.empty(self.shape_gh[1:])
        _chk(self.L.kh_get_emf(self.h, d, _np_ptr(e), MEM_HOST))
        return e

    def debug_predictor(self, dt):
        _chk(self.L.kh_debug_predictor(self.h, C.c_double(dt)))

    def debug_fixup(self, pflag_with_ghosts):
        pf = np.ascontiguousarray(pflag_with_ghosts, dtype=np.int32)
        assert pf.shape == self.shape_gh[1:]
        _chk(self.L.kh_debug_fixup(self.h, _np_ptr(pf), MEM_HOST))

    def get_stream(self):
        s = C.c_void_p()
        _chk(self.L.kh_get_stream(self.h, C.byref(s)))
        return int(s.value or 0)

    def sync(self):
        _chk(self.L.kh_sync(self.h))

    def launch_count(self):
        return int(self.L.kh_launch_count(self.h))

    def set_graph(self, enable):
        _chk(self.L.kh_set_graph(self.h, int(bool(enable))))

    def set_profile(self, enable):
        _chk(self.L.kh_set_profile(self.h, int(bool(enable))))

    def get_profile(self):
        """{kind: (device ms summed, bracketed launch groups)} since set_profile(True)."""
        n = len(KERNEL_KINDS)
        ms, cnt = (C.c_double * n)(), (C.c_longlong * n)()
        _chk(self.L.kh_get_profile(self.h, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(KERNEL_KINDS)}
