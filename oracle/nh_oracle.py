"""ctypes binding of oracle/libnh_oracle.so (CPU ORACLE -- test infrastructure, not the product).

Argument marshalling only; every formula lives in nh_oracle.c.  NumPy arrays are (ny, nx) for
cell fields and (ny+1, nx+1) for node fields (C order => x fastest, as the C side expects).
"""
import ctypes as C
import numpy as np

from . import build as _build

BC_PERIODIC, BC_WALL, BC_OUTFLOW = 0, 1, 2
OK, EINVAL, ENOMEM, ENOCONV, ENAN = 0, -1, -2, -4, -5


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
    ]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.nho_default_params.argtypes = [C.POINTER(Params)]
        L.nho_default_params.restype = None
        L.nho_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_double, C.c_double,
                                 _dp, C.POINTER(Params)]
        L.nho_destroy.argtypes = [C.c_void_p]
        L.nho_destroy.restype = None
        L.nho_set_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        L.nho_continue_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        L.nho_get_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        L.nho_set_time.argtypes = [C.c_void_p, C.c_double]
        L.nho_step.argtypes = [C.c_void_p, C.c_int]
        L.nho_hydrostatic_step.argtypes = [C.c_void_p, C.c_double]
        L.nho_nonhydro_correct.argtypes = [C.c_void_p, C.c_double]
        L.nho_get_info.argtypes = [C.c_void_p, C.POINTER(Info)]
        L.nho_last_error.argtypes = [C.c_void_p]
        L.nho_last_error.restype = C.c_char_p
        L.nho_compute_dt.argtypes = [C.c_void_p, _dp]
        L.nho_apply_A.argtypes = [C.c_void_p, _dp, _dp]
        L.nho_coeffs.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        L.nho_rhs.argtypes = [C.c_void_p, C.c_double, _dp]
        L.nho_constraint.argtypes = [C.c_void_p, _dp]
        L.nho_solve.argtypes = [C.c_void_p, _dp, _dp, C.POINTER(C.c_int), _dp]
        L.nho_breaking.argtypes = [C.c_void_p, C.c_double, _dp, _dp, _dp]
        L.nho_w_advect.argtypes = [C.c_void_p, C.c_double, _dp]
        L.nho_start_vector.argtypes = [C.c_void_p, _dp]
        L.nho_face_fluct.argtypes = [C.c_double] * 9 + [_dp, _dp]
        L.nho_face_fluct.restype = None
        L.nho_dsg.argtypes = [C.c_double] * 3
        L.nho_dsg.restype = C.c_double
        L.nho_minmod.argtypes = [C.c_double] * 2
        L.nho_minmod.restype = C.c_double
        for f in (L.nho_cbrt_fixed, L.nho_sech2_fixed):
            f.argtypes = [C.c_double]
            f.restype = C.c_double
        _lib = L
    return _lib


def default_params(**kw) -> Params:
    p = Params()
    lib().nho_default_params(C.byref(p))
    for k, v in kw.items():
        if not hasattr(p, k):
            raise AttributeError(k)
        setattr(p, k, v)
    return p


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c64(a, shape):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.shape != shape:
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"oracle error {code}: {msg}")
        self.code = code


class Oracle:
    """One oracle context.  Mirrors the paper's problem statement: create(grid, H, params),
    set_state / get_state, step(n), hydrostatic_step(dt), nonhydro_correct(dt)."""

    def __init__(self, nx, ny, dx, dy, H, params=None, **kw):
        self.nx, self.ny, self.dx, self.dy = int(nx), int(ny), float(dx), float(dy)
        self.params = params if params is not None else default_params(**kw)
        self.cshape, self.nshape = (self.ny, self.nx), (self.ny + 1, self.nx + 1)
        Hc = _c64(H, self.cshape)
        self._h = C.c_void_p()
        st = lib().nho_create(C.byref(self._h), self.nx, self.ny, self.dx, self.dy, _ptr(Hc),
                              C.byref(self.params))
        if st != OK:
            self._h = None
            raise OracleError(st, "nho_create failed (invalid argument?)")

    def close(self):
        if getattr(self, "_h", None):
            lib().nho_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def _check(self, st, allow=()):
        if st != OK and st not in allow:
            raise OracleError(st, lib().nho_last_error(self._h).decode())
        return st

    def set_state(self, h, qx, qy, w=None, p=None, keep_history=False):
        a = [_c64(h, self.cshape), _c64(qx, self.cshape), _c64(qy, self.cshape)]
        b = [None if x is None else _c64(x, self.nshape) for x in (w, p)]
        f = lib().nho_continue_state if keep_history else lib().nho_set_state
        self._check(f(self._h, *[_ptr(x) for x in a + b]))

    def get_state(self):
        h, qx, qy = (np.empty(self.cshape) for _ in range(3))
        w, p = (np.empty(self.nshape) for _ in range(2))
        self._check(lib().nho_get_state(self._h, _ptr(h), _ptr(qx), _ptr(qy), _ptr(w), _ptr(p)))
        return dict(h=h, qx=qx, qy=qy, w=w, p=p)

    def set_time(self, t):
        self._check(lib().nho_set_time(self._h, float(t)))

    def step(self, nsteps=1, allow_noconv=False):
        return self._check(lib().nho_step(self._h, int(nsteps)), (ENOCONV,) if allow_noconv else ())

    def hydrostatic_step(self, dt=0.0):
        self._check(lib().nho_hydrostatic_step(self._h, float(dt)))

    def nonhydro_correct(self, dt):
        self._check(lib().nho_nonhydro_correct(self._h, float(dt)))

    def info(self) -> Info:
        out = Info()
        self._check(lib().nho_get_info(self._h, C.byref(out)))
        return out

    def compute_dt(self):
        dt = C.c_double()
        self._check(lib().nho_compute_dt(self._h, C.byref(dt)))
        return dt.value

    def apply_A(self, x):
        x = _c64(x, self.nshape)
        y = np.empty(self.nshape)
        self._check(lib().nho_apply_A(self._h, _ptr(x), _ptr(y)))
        return y

    def coeffs(self):
        out = [np.empty(self.nshape) for _ in range(5)]
        self._check(lib().nho_coeffs(self._h, *[_ptr(a) for a in out]))
        return dict(zip(("AC", "AE", "AW", "AN", "AS"), out))

    def rhs(self, dt):
        b = np.empty(self.nshape)
        self._check(lib().nho_rhs(self._h, float(dt), _ptr(b)))
        return b

    def constraint(self):
        b = np.empty(self.nshape)
        self._check(lib().nho_constraint(self._h, _ptr(b)))
        return b

    def breaking(self, dt):
        """S6 alone on the current state: -> dict(qx=q**_x, qy=q**_y, w=w**)."""
        qx, qy, w = np.empty(self.cshape), np.empty(self.cshape), np.empty(self.nshape)
        self._check(lib().nho_breaking(self._h, float(dt), _ptr(qx), _ptr(qy), _ptr(w)))
        return dict(qx=qx, qy=qy, w=w)

    def w_advect(self, dt):
        """S5b alone (R30) on the current state: w transported over dt by the node velocities."""
        w = np.empty(self.nshape)
        self._check(lib().nho_w_advect(self._h, float(dt), _ptr(w)))
        return w

    def start_vector(self):
        """R32: the vector the next pressure solve of a step would start from."""
        x = np.empty(self.nshape)
        self._check(lib().nho_start_vector(self._h, _ptr(x)))
        return x

    def solve(self, b, x0=None, allow_noconv=False):
        b = _c64(b, self.nshape)
        x = np.zeros(self.nshape) if x0 is None else _c64(x0, self.nshape).copy()
        it, rr = C.c_int(), C.c_double()
        st = lib().nho_solve(self._h, _ptr(b), _ptr(x), C.byref(it), C.byref(rr))
        self._check(st, (ENOCONV,) if allow_noconv else ())
        return x, it.value, rr.value


def face_fluct(g, hm, etam, um, vm, hp, etap, up, vp):
    Dm, Dp = np.empty(3), np.empty(3)
    lib().nho_face_fluct(g, hm, etam, um, vm, hp, etap, up, vp, _ptr(Dm), _ptr(Dp))
    return Dm, Dp


def dsg(h, q, delta):
    return lib().nho_dsg(h, q, delta)


def minmod(a, b):
    return lib().nho_minmod(a, b)


def cbrt_fixed(a):
    return lib().nho_cbrt_fixed(a)


def sech2_fixed(a):
    return lib().nho_sech2_fixed(a)
