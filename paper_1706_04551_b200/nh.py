"""Thin ctypes binding of libnh_b200.so (include/nh_b200.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; there is no CPU fallback and
nothing here computes.  Loading fails loudly when the library has not been built
(`python -m paper_1706_04551_b200.build`) and `NH(...)` fails loudly without an sm_100 device.

Arrays may be NumPy float64 arrays (host pointers) or torch CUDA float64 tensors (device
pointers); cell fields have shape (ny, nx), node fields (ny+1, nx+1), C order (x fastest).  The
names follow the C ABI: NH(...) = nh_create, set_state, get_state, step, hydrostatic_step,
nonhydro_correct, sync, info, and the test hooks.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

BC_PERIODIC, BC_WALL, BC_OUTFLOW = 0, 1, 2
OK, EINVAL, ENOMEM, ECUDA, ENOCONV, ENAN = 0, -1, -2, -3, -4, -5
FLAG_NOCONV, FLAG_NAN, FLAG_BADSTATE, FLAG_STAGNATED = 1, 2, 4, 8   # nh_info.flags
PROF_CATS = ("predictor", "assembly", "solver", "correct")

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libnh_b200.so")


class Params(C.Structure):
    _fields_ = [
        ("g", C.c_double), ("cfl", C.c_double), ("delta", C.c_double), ("eps_dry", C.c_double),
        ("B1", C.c_double), ("B2", C.c_double), ("solver_rtol", C.c_double),
        ("gen_A", C.c_double), ("gen_h0", C.c_double), ("gen_x0", C.c_double), ("gen_Lrel", C.c_double),
        ("manning_n", C.c_double), ("srj_eps", C.c_double), ("srj_rel", C.c_double),
        ("abs_xlo", C.c_double), ("abs_xhi", C.c_double), ("abs_ylo", C.c_double), ("abs_yhi", C.c_double),
        ("breaking", C.c_int), ("nonhydro", C.c_int), ("time_order", C.c_int), ("space_order", C.c_int),
        ("bc_xlo", C.c_int), ("bc_xhi", C.c_int), ("bc_ylo", C.c_int), ("bc_yhi", C.c_int),
        ("solver_maxit", C.c_int), ("gen_on", C.c_int), ("precision", C.c_int), ("solver", C.c_int),
        ("srj_mmax", C.c_int), ("w_advect", C.c_int), ("warm_start", C.c_int), ("reserved", C.c_int),
    ]


class Info(C.Structure):
    _fields_ = [
        ("t", C.c_double), ("dt_last", C.c_double), ("res_last", C.c_double),
        ("steps", C.c_longlong), ("iters_total", C.c_longlong), ("clamps", C.c_longlong),
        ("solves", C.c_longlong),
        ("iters_last", C.c_int), ("iters_max", C.c_int), ("flags", C.c_int), ("reserved", C.c_int),
        ("clamp_max", C.c_double), ("clamp_hist", C.c_longlong * 6),
        ("solver_rtol_effective", C.c_double),
    ]


class NHError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"nh_b200 error {code}: {msg}")
        self.code = code


_lib = None
_vp = C.c_void_p

EXPORTS = (
    "nh_default_params", "nh_create", "nh_destroy", "nh_set_state", "nh_continue_state", "nh_get_state", "nh_set_time", "nh_step",
    "nh_hydrostatic_step", "nh_nonhydro_correct", "nh_sync", "nh_get_info", "nh_last_error",
    "nh_launch_count", "nh_profile", "nh_profile_read", "nh_compute_dt", "nh_apply_A", "nh_coeffs",
    "nh_rhs", "nh_constraint", "nh_solve", "nh_breaking", "nh_w_advect", "nh_fp64_rate", "nh_start_vector",
    "nh_cfl_dt_static", "nh_cfl_dt_static_max_cells", "nh_static_last_error", "nh_stream_mix_rate",
)


def lib():
    """Load libnh_b200.so (built in-tree).  No fallback: a missing library is an error."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1706_04551_b200.build` "
                "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.nh_default_params.argtypes = [C.POINTER(Params)]
        L.nh_default_params.restype = None
        L.nh_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_double, C.c_double, _vp,
                                C.POINTER(Params), _vp]
        L.nh_destroy.argtypes = [_vp]
        L.nh_destroy.restype = None
        L.nh_set_state.argtypes = [_vp] * 6
        L.nh_continue_state.argtypes = [_vp] * 6
        L.nh_get_state.argtypes = [_vp] * 6
        L.nh_set_time.argtypes = [_vp, C.c_double]
        L.nh_step.argtypes = [_vp, C.c_int]
        L.nh_hydrostatic_step.argtypes = [_vp, C.c_double]
        L.nh_nonhydro_correct.argtypes = [_vp, C.c_double]
        L.nh_sync.argtypes = [_vp]
        L.nh_get_info.argtypes = [_vp, C.POINTER(Info)]
        L.nh_last_error.argtypes = [_vp]
        L.nh_last_error.restype = C.c_char_p
        L.nh_launch_count.argtypes = [_vp]
        L.nh_launch_count.restype = C.c_longlong
        L.nh_profile.argtypes = [_vp, C.c_int]
        L.nh_profile_read.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.nh_compute_dt.argtypes = [_vp, C.POINTER(C.c_double)]
        L.nh_apply_A.argtypes = [_vp, _vp, _vp]
        L.nh_coeffs.argtypes = [_vp] * 6
        L.nh_rhs.argtypes = [_vp, C.c_double, _vp]
        L.nh_constraint.argtypes = [_vp, _vp]
        L.nh_solve.argtypes = [_vp, _vp, _vp, C.POINTER(C.c_int), C.POINTER(C.c_double)]
        L.nh_breaking.argtypes = [_vp, C.c_double, _vp, _vp, _vp]
        L.nh_w_advect.argtypes = [_vp, C.c_double, _vp]
        L.nh_start_vector.argtypes = [_vp, _vp]
        L.nh_fp64_rate.argtypes = [_vp, C.POINTER(C.c_double)]
        L.nh_stream_mix_rate.argtypes = [_vp, C.c_int, C.c_int, C.c_longlong, C.POINTER(C.c_double)]
        L.nh_cfl_dt_static.argtypes = [C.c_int, C.c_int] + [C.c_double] * 5 + [_vp] * 5
        L.nh_cfl_dt_static_max_cells.argtypes = []
        L.nh_cfl_dt_static_max_cells.restype = C.c_longlong
        L.nh_static_last_error.argtypes = []
        L.nh_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def fp64_rate(stream=None) -> float:
    """Measured fp64 FMA rate of the current device (thread instructions per second)."""
    r = C.c_double()
    st = lib().nh_fp64_rate(None if stream is None else stream.cuda_stream, C.byref(r))
    if st != OK:
        raise NHError(st, "nh_fp64_rate")
    return r.value


def stream_mix_rate(nread, nwrite, doubles_per_plane, stream=None) -> float:
    """GB/s a plain streaming kernel reaches with `nread` planes read and `nwrite` written (nh_stream_mix_rate)."""
    r = C.c_double()
    st = lib().nh_stream_mix_rate(None if stream is None else stream.cuda_stream, int(nread), int(nwrite),
                                  int(doubles_per_plane), C.byref(r))
    if st != OK:
        raise NHError(st, "nh_stream_mix_rate")
    return r.value


def cfl_dt_static_max_cells() -> int:
    return int(lib().nh_cfl_dt_static_max_cells())


def cfl_dt_static(h, qx, qy, dt_out, dx, dy, g=9.81, cfl=0.5, delta=1e-5, stream=None):
    """nh_cfl_dt_static: the CFL time step of a state in the caller's own device arrays, for callers
    that must not allocate device memory (include/nh_b200.h has the who and why).  h, qx, qy: torch
    CUDA float64 tensors of shape (ny, nx); dt_out: a torch CUDA float64 tensor of one element, which
    the caller provides -- this wrapper creates no tensor either.  Only enqueues on `stream` (default:
    the NULL stream): read dt_out after that stream has got there.  Grids above
    cfl_dt_static_max_cells() raise NHError(EINVAL)."""
    ny, nx = (int(n) for n in h.shape)
    keep = []
    ptrs = [_in(a, (ny, nx), keep) for a in (h, qx, qy)] + [_out_ptr(dt_out, (1,))]
    sp = None if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
    st = lib().nh_cfl_dt_static(nx, ny, float(dx), float(dy), float(g), float(cfl), float(delta), *ptrs, sp)
    if st != OK:
        raise NHError(st, lib().nh_static_last_error().decode(errors="replace"))


def default_params(**kw) -> Params:
    p = Params()
    lib().nh_default_params(C.byref(p))
    for k, v in kw.items():
        if not hasattr(p, k):
            raise AttributeError(k)
        setattr(p, k, v)
    return p


def _is_torch(a):
    return type(a).__module__.startswith("torch")


def _in(a, shape, keep):
    """Pointer of an input array (host NumPy or device torch), shape-checked, fp64, contiguous."""
    if a is None:
        return None
    if _is_torch(a):
        import torch
        if a.dtype != torch.float64 or tuple(a.shape) != shape or not a.is_contiguous():
            raise ValueError(f"expected contiguous float64 tensor of shape {shape}")
        keep.append(a)
        return a.data_ptr()
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    keep.append(a)
    return a.ctypes.data


def _out_ptr(a, shape):
    if _is_torch(a):
        import torch
        if a.dtype != torch.float64 or tuple(a.shape) != shape or not a.is_contiguous():
            raise ValueError(f"expected contiguous float64 tensor of shape {shape}")
        return a.data_ptr()
    if a.dtype != np.float64 or a.shape != shape or not a.flags.c_contiguous:
        raise ValueError(f"expected C-contiguous float64 array of shape {shape}")
    return a.ctypes.data


class NH:
    """One context of the library = one problem of the paper: grid, bathymetry H, parameters."""

    def __init__(self, nx, ny, dx, dy, H, params=None, stream=None, **kw):
        self.nx, self.ny, self.dx, self.dy = int(nx), int(ny), float(dx), float(dy)
        self.params = params if params is not None else default_params(**kw)
        self.cshape, self.nshape = (self.ny, self.nx), (self.ny + 1, self.nx + 1)
        self._h = _vp()
        keep = []
        Hp = _in(H, self.cshape, keep)
        if stream is None:
            sp = None
        elif isinstance(stream, int):
            sp = stream
        else:
            sp = stream.cuda_stream  # torch.cuda.Stream
        st = lib().nh_create(C.byref(self._h), self.nx, self.ny, self.dx, self.dy, Hp,
                             C.byref(self.params), sp)
        if st != OK:
            self._h = None
            raise NHError(st, {EINVAL: "nh_create: invalid argument", ENOMEM: "nh_create: out of memory",
                               ECUDA: "nh_create: no sm_100 CUDA device / CUDA failure"}.get(st, "nh_create"))

    def close(self):
        if getattr(self, "_h", None):
            lib().nh_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st, allow=()):
        if st != OK and st not in allow:
            raise NHError(st, lib().nh_last_error(self._h).decode(errors="replace"))
        return st

    # ---- state -----------------------------------------------------------------------------
    def set_state(self, h, qx, qy, w=None, p=None, keep_history=False):
        """nh_set_state (a new run), or with keep_history=True nh_continue_state (the running state
        coming back: the solver keeps its solution history)."""
        keep = []
        ptrs = [_in(a, self.cshape, keep) for a in (h, qx, qy)] + \
               [_in(a, self.nshape, keep) for a in (w, p)]
        f = lib().nh_continue_state if keep_history else lib().nh_set_state
        self._check(f(self._h, *ptrs))
        # pageable host sources are consumed synchronously; device sources are ordered on the stream

    def get_state(self, out=None):
        """-> dict(h, qx, qy, w, p).  out: optional dict of preallocated arrays/tensors (a missing
        key skips that field); default: new NumPy arrays."""
        if out is None:
            out = dict(h=np.empty(self.cshape), qx=np.empty(self.cshape), qy=np.empty(self.cshape),
                       w=np.empty(self.nshape), p=np.empty(self.nshape))
        ptrs = [None if out.get(k) is None else _out_ptr(out[k], self.cshape) for k in ("h", "qx", "qy")] + \
               [None if out.get(k) is None else _out_ptr(out[k], self.nshape) for k in ("w", "p")]
        self._check(lib().nh_get_state(self._h, *ptrs))
        return out

    def set_time(self, t):
        self._check(lib().nh_set_time(self._h, float(t)))

    # ---- the path --------------------------------------------------------------------------
    def step(self, nsteps=1):
        self._check(lib().nh_step(self._h, int(nsteps)))

    def hydrostatic_step(self, dt=0.0):
        self._check(lib().nh_hydrostatic_step(self._h, float(dt)))

    def nonhydro_correct(self, dt):
        self._check(lib().nh_nonhydro_correct(self._h, float(dt)))

    def sync(self, allow=()):
        return self._check(lib().nh_sync(self._h), allow)

    def info(self) -> Info:
        out = Info()
        self._check(lib().nh_get_info(self._h, C.byref(out)))
        return out

    def launch_count(self) -> int:
        return int(lib().nh_launch_count(self._h))

    def profile(self, enable=True):
        self._check(lib().nh_profile(self._h, int(bool(enable))))

    def profile_read(self):
        """-> {phase: (milliseconds, brackets)} since the last read."""
        ms = (C.c_double * len(PROF_CATS))()
        n = (C.c_longlong * len(PROF_CATS))()
        self._check(lib().nh_profile_read(self._h, ms, n))
        return {k: (ms[i], int(n[i])) for i, k in enumerate(PROF_CATS)}

    # ---- test hooks ------------------------------------------------------------------------
    def compute_dt(self):
        dt = C.c_double()
        self._check(lib().nh_compute_dt(self._h, C.byref(dt)))
        return dt.value

    def apply_A(self, x):
        keep = []
        y = np.empty(self.nshape)
        self._check(lib().nh_apply_A(self._h, _in(x, self.nshape, keep), y.ctypes.data))
        return y

    def coeffs(self):
        out = [np.empty(self.nshape) for _ in range(5)]
        self._check(lib().nh_coeffs(self._h, *[a.ctypes.data for a in out]))
        return dict(zip(("AC", "AE", "AW", "AN", "AS"), out))

    def rhs(self, dt):
        b = np.empty(self.nshape)
        self._check(lib().nh_rhs(self._h, float(dt), b.ctypes.data))
        return b

    def constraint(self):
        b = np.empty(self.nshape)
        self._check(lib().nh_constraint(self._h, b.ctypes.data))
        return b

    def breaking(self, dt):
        qx, qy, w = np.empty(self.cshape), np.empty(self.cshape), np.empty(self.nshape)
        self._check(lib().nh_breaking(self._h, float(dt), qx.ctypes.data, qy.ctypes.data, w.ctypes.data))
        return dict(qx=qx, qy=qy, w=w)

    def w_advect(self, dt):
        w = np.empty(self.nshape)
        self._check(lib().nh_w_advect(self._h, float(dt), w.ctypes.data))
        return w

    def start_vector(self):
        x = np.empty(self.nshape)
        self._check(lib().nh_start_vector(self._h, x.ctypes.data))
        return x

    def solve(self, b, x0=None, allow=()):
        keep = []
        x = np.zeros(self.nshape) if x0 is None else np.array(x0, dtype=np.float64, order="C")
        it, rr = C.c_int(), C.c_double()
        st = lib().nh_solve(self._h, _in(b, self.nshape, keep), x.ctypes.data, C.byref(it), C.byref(rr))
        self._check(st, allow)
        return x, it.value, rr.value
