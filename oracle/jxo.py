"""ctypes binding of the CPU oracle (oracle/libjxo.so).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this module.  It never touches the CUDA library.
Arrays are numpy, SoA [4][ny][nx] (x fastest), float64 or float32.
"""
import ctypes as C

import numpy as np

from . import build as _build

OK, EINVAL, ENOMEM, ESTATE, ENUMERIC = 0, 1, 2, 4, 5
BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_INFLOW = 0, 1, 2, 3
F64, F32 = 0, 1
_BC_NAMES = {"periodic": 0, "transmissive": 1, "reflective": 2, "inflow": 3}


class _Bc(C.Structure):
    _fields_ = [("xlo", C.c_int), ("xhi", C.c_int), ("ylo", C.c_int), ("yhi", C.c_int),
                ("inflow", C.c_double * 4)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.jxo_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                 C.c_double, C.POINTER(_Bc), C.c_int, C.POINTER(vp)]
        L.jxo_destroy.argtypes = [vp]
        L.jxo_destroy.restype = None
        L.jxo_last_error.argtypes = [vp]
        L.jxo_last_error.restype = C.c_char_p
        L.jxo_set_ibm.argtypes = [vp, vp]
        L.jxo_set_flux_mlp.argtypes = [vp, vp, dp, dp, C.c_int]
        L.jxo_set_artificial_viscosity.argtypes = [vp, C.c_double]
        L.jxo_rhs.argtypes = [vp, vp, vp]
        L.jxo_max_wavespeed.argtypes = [vp, vp, dp]
        L.jxo_step.argtypes = [vp, vp, C.c_double, C.c_int]
        L.jxo_step_fixed_dt.argtypes = [vp, vp, C.c_double, C.c_int]
        L.jxo_get_time.argtypes = [vp, dp, dp]
        L.jxo_weno5.argtypes = [dp]
        L.jxo_weno5.restype = C.c_double
        L.jxo_hllc.argtypes = [dp, dp, C.c_double, dp]
        L.jxo_hllc.restype = None
        L.jxo_hllc_star.argtypes = [dp, dp, C.c_double, dp, dp, dp]
        L.jxo_hllc_star.restype = None
        L.jxo_fill_ghosts.argtypes = [vp, vp, vp]
        L.jxo_ibm_ghosts.argtypes = [vp, ip, ip, dp, dp]
        L.jxo_cell_types.argtypes = [vp, vp]
        L.jxo_guard_count.argtypes = [vp]
        L.jxo_guard_count.restype = C.c_longlong
        L.jxo_count_ops.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
        L.jxo_mlp_eval.argtypes = [vp, dp, dp]
        L.jxo_set_flux_cnn.argtypes = [vp, vp, dp, dp, C.c_int]
        L.jxo_cnn_apply.argtypes = [vp, dp, C.c_int, C.c_int, dp]
        L.jxo_cnn_fields.argtypes = [vp, dp, dp, dp, dp, dp]
        L.jxo_step_fixed_dt_tangent.argtypes = [vp, vp, vp, C.c_double, C.c_double, C.c_int]
        L.jxo_rhs_tangent.argtypes = [vp, vp, vp, C.c_double, vp, vp]
        L.jxo_set_flux_mlp_direction.argtypes = [vp, vp]
        L.jxo_weno5_tangent.argtypes = [dp, dp, dp]
        L.jxo_weno5_tangent.restype = None
        L.jxo_hllc_tangent.argtypes = [dp, dp, dp, dp, C.c_double, C.c_double, dp, dp]
        L.jxo_hllc_tangent.restype = None
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def make_bc(bc):
    """bc: dict with xlo/xhi/ylo/yhi in {'periodic','transmissive','reflective','inflow'}
    and optional inflow=(rho,u,v,p)."""
    b = _Bc()
    for side in ("xlo", "xhi", "ylo", "yhi"):
        setattr(b, side, _BC_NAMES[bc[side]])
    inflow = bc.get("inflow", (1.0, 0.0, 0.0, 1.0))
    for k in range(4):
        b.inflow[k] = float(inflow[k])
    return b


def weno5(v):
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert v.shape == (5,)
    return lib().jxo_weno5(_d(v))


def hllc(WL, WR, gamma):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.zeros(4)
    lib().jxo_hllc(_d(WL), _d(WR), float(gamma), _d(F))
    return F


def weno5_tangent(v, vdot):
    """(value, derivative along vdot) of the left-biased WENO5-JS value (O4)."""
    v = np.ascontiguousarray(v, dtype=np.float64)
    vdot = np.ascontiguousarray(vdot, dtype=np.float64)
    assert v.shape == (5,) and vdot.shape == (5,)
    out = np.zeros(2)
    lib().jxo_weno5_tangent(_d(v), _d(vdot), _d(out))
    return out[0], out[1]


def hllc_tangent(WL, WR, WLdot, WRdot, gamma, gamma_dot):
    """(F, Fdot) of the HLLC flux (O5) along the direction (WLdot, WRdot, gamma_dot)."""
    a = [np.ascontiguousarray(x, dtype=np.float64) for x in (WL, WR, WLdot, WRdot)]
    F, Fd = np.zeros(4), np.zeros(4)
    lib().jxo_hllc_tangent(_d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), float(gamma), float(gamma_dot), _d(F), _d(Fd))
    return F, Fd


def mse_tangent(U, Udot, Utarget):
    """Eq. 14 for one step with the mean over all entries (R22): L = mean((U - Utarget)^2) and its derivative
    along Udot, dL = mean(2 (U - Utarget) Udot)."""
    r = np.asarray(U, dtype=np.float64) - np.asarray(Utarget, dtype=np.float64)
    return float(np.mean(r * r)), float(np.mean(2.0 * r * np.asarray(Udot, dtype=np.float64)))


def hllc_star(WL, WR, gamma):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    sp, UL, UR = np.zeros(3), np.zeros(4), np.zeros(4)
    lib().jxo_hllc_star(_d(WL), _d(WR), float(gamma), _d(sp), _d(UL), _d(UR))
    return sp, UL, UR


class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"jxo error {code}: {msg}")
        self.code = code


class Oracle:
    def __init__(self, nx, ny, dx, dy, gamma=1.4, mu=0.0, Pr=0.72, bc=None, dtype=np.float64):
        self.nx, self.ny = int(nx), int(ny)
        self.dtype = np.dtype(dtype)
        assert self.dtype in (np.float64, np.float32)
        self._bc = make_bc(bc)
        self._h = C.c_void_p()
        rc = lib().jxo_create(self.nx, self.ny, dx, dy, gamma, mu, Pr, C.byref(self._bc),
                              F64 if self.dtype == np.float64 else F32, C.byref(self._h))
        if rc != OK:
            raise OracleError(rc, "jxo_create")

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.jxo_destroy(self._h)
            self._h = None

    def _chk(self, rc):
        if rc != OK:
            raise OracleError(rc, lib().jxo_last_error(self._h).decode())

    def _field(self, U):
        U = np.ascontiguousarray(U, dtype=self.dtype)
        assert U.shape == (4, self.ny, self.nx), U.shape
        return U

    def set_ibm(self, phi):
        if phi is None:
            self._chk(lib().jxo_set_ibm(self._h, None))
            return
        phi = np.ascontiguousarray(phi, dtype=np.float64)
        assert phi.shape == (self.ny, self.nx)
        self._chk(lib().jxo_set_ibm(self._h, phi.ctypes.data))

    def set_flux_mlp(self, weights, in_scale=None, out_scale=None, emulate_bf16=False):
        if weights is None:
            self._chk(lib().jxo_set_flux_mlp(self._h, None, None, None, 0))
            return
        w = np.ascontiguousarray(weights, dtype=np.float32)
        assert w.shape == (6020,)
        a = np.ascontiguousarray(in_scale, dtype=np.float64)
        b = np.ascontiguousarray(out_scale, dtype=np.float64)
        self._chk(lib().jxo_set_flux_mlp(self._h, w.ctypes.data, _d(a), _d(b), int(emulate_bf16)))

    def set_flux_cnn(self, weights, in_scale=None, out_scale=None, emulate_bf16=False):
        """O11: the paper's 2D CNN neural flux, 6388 weights in OIHW order (None disables)."""
        if weights is None:
            self._chk(lib().jxo_set_flux_cnn(self._h, None, None, None, 0))
            return
        w = np.ascontiguousarray(weights, dtype=np.float32)
        assert w.shape == (6388,)
        a = np.ascontiguousarray(in_scale, dtype=np.float64)
        b = np.ascontiguousarray(out_scale, dtype=np.float64)
        self._chk(lib().jxo_set_flux_cnn(self._h, w.ctypes.data, _d(a), _d(b), int(emulate_bf16)))

    def cnn_fields(self, U):
        """(Xx, Xy, Yx, Yy) of one rhs evaluation: inputs and raw outputs of the CNN at x- and y-faces"""
        U = np.ascontiguousarray(U, dtype=np.float64)
        shp = ((4, self.ny, self.nx + 1), (4, self.nx, self.ny + 1))
        f = [np.zeros(shp[0]), np.zeros(shp[1]), np.zeros(shp[0]), np.zeros(shp[1])]
        self._chk(lib().jxo_cnn_fields(self._h, _d(U), *[_d(a) for a in f]))
        return f

    def cnn_apply(self, x):
        """the CNN alone on a normalised field x[4][na][nb] (a tangential, b normal)"""
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.zeros_like(x)
        self._chk(lib().jxo_cnn_apply(self._h, _d(x), x.shape[1], x.shape[2], _d(y)))
        return y

    def set_artificial_viscosity(self, nu):
        self._chk(lib().jxo_set_artificial_viscosity(self._h, float(nu)))

    def rhs(self, U):
        U = self._field(U)
        L = np.empty_like(U)
        self._chk(lib().jxo_rhs(self._h, U.ctypes.data, L.ctypes.data))
        return L

    def max_wavespeed(self, U):
        U = self._field(U)
        s = C.c_double()
        self._chk(lib().jxo_max_wavespeed(self._h, U.ctypes.data, C.byref(s)))
        return s.value

    def step(self, U, cfl, nsteps):
        U = self._field(U).copy()
        self._chk(lib().jxo_step(self._h, U.ctypes.data, float(cfl), int(nsteps)))
        return U

    def step_fixed_dt(self, U, dt, nsteps):
        U = self._field(U).copy()
        self._chk(lib().jxo_step_fixed_dt(self._h, U.ctypes.data, float(dt), int(nsteps)))
        return U

    def set_flux_mlp_direction(self, direction):
        """Direction of perturbation of the MLP's 6020 parameters for the tangent O12; None = none."""
        if direction is None:
            self._chk(lib().jxo_set_flux_mlp_direction(self._h, None))
            return
        d = np.ascontiguousarray(direction, dtype=np.float64)
        assert d.shape == (6020,)
        self._chk(lib().jxo_set_flux_mlp_direction(self._h, d.ctypes.data))

    def rhs_tangent(self, U, Udot, gamma_dot):
        """(L(U), its derivative along (Udot, gamma_dot))."""
        U = np.ascontiguousarray(self._field(U), dtype=np.float64)
        Udot = np.ascontiguousarray(Udot, dtype=np.float64)
        assert Udot.shape == U.shape
        L, Ld = np.empty_like(U), np.empty_like(U)
        self._chk(lib().jxo_rhs_tangent(self._h, U.ctypes.data, Udot.ctypes.data, float(gamma_dot), L.ctypes.data,
                                        Ld.ctypes.data))
        return L, Ld

    def step_fixed_dt_tangent(self, U, Udot, gamma_dot, dt, nsteps, scheme="ssprk3"):
        """O12: (U, Udot) after nsteps steps of size dt; Udot is the derivative along (Udot, gamma_dot).
        scheme "euler": the update of PAPER.md Eq. 10 as printed, U <- U + dt L(U), written out here."""
        U = np.ascontiguousarray(self._field(U), dtype=np.float64).copy()
        Udot = np.ascontiguousarray(Udot, dtype=np.float64).copy()
        assert Udot.shape == U.shape
        if scheme == "euler":
            for _ in range(int(nsteps)):
                L, Ld = self.rhs_tangent(U, Udot, gamma_dot)
                U = U + dt * L
                Udot = Udot + dt * Ld
            return U, Udot
        assert scheme == "ssprk3"
        self._chk(lib().jxo_step_fixed_dt_tangent(self._h, U.ctypes.data, Udot.ctypes.data, float(gamma_dot),
                                                  float(dt), int(nsteps)))
        return U, Udot

    def step_fixed_dt_adjoint(self, U, Ubar, dt, nsteps, planar=False, scheme="ssprk3"):
        """O13: the adjoint of nsteps fixed-dt steps, from the definition of a transpose (Eq. 16 read from
        the left): entry j of J^T Ubar is <Ubar, J e_j>, with J e_j from the tangent O12 -- one tangent run per
        entry of the state (small cases only), and gamma_bar = <Ubar, dS/dgamma>.
        planar: U is a field of identical rows standing for a 1D problem; the directions e_j are repeated over the
        rows and Ubar (one row, [4][1][nx]) is paired with row 0: the 1D adjoint.  Returns (Ubar_in, gamma_bar)."""
        U = np.ascontiguousarray(self._field(U), dtype=np.float64)
        Ubar = np.asarray(Ubar, dtype=np.float64)
        shape = (4, 1, self.nx) if planar else U.shape
        assert Ubar.shape == shape
        out = np.zeros(shape)
        pick = (lambda D: D[:, :1]) if planar else (lambda D: D)
        for j in range(out.size):
            e = np.zeros(shape)
            e.flat[j] = 1.0
            _, D = self.step_fixed_dt_tangent(U, np.repeat(e, self.ny, axis=1) if planar else e, 0.0, dt, nsteps, scheme)
            out.flat[j] = float(np.sum(Ubar * pick(D)))
        _, D = self.step_fixed_dt_tangent(U, np.zeros_like(U), 1.0, dt, nsteps, scheme)
        return out, float(np.sum(Ubar * pick(D)))

    def time(self):
        t, dt = C.c_double(), C.c_double()
        self._chk(lib().jxo_get_time(self._h, C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def fill_ghosts(self, U):
        U = self._field(U)
        Up = np.empty((4, self.ny + 6, self.nx + 6), dtype=self.dtype)
        self._chk(lib().jxo_fill_ghosts(self._h, U.ctypes.data, Up.ctypes.data))
        return Up

    def ibm_ghosts(self):
        n = lib().jxo_ibm_ghosts(self._h, None, None, None, None)
        cell = np.zeros(n, dtype=np.int32)
        donors = np.zeros((n, 4), dtype=np.int32)
        w = np.zeros((n, 4))
        nrm = np.zeros((n, 2))
        if n:
            ip = C.POINTER(C.c_int)
            lib().jxo_ibm_ghosts(self._h, cell.ctypes.data_as(ip), donors.ctypes.data_as(ip), _d(w), _d(nrm))
        return cell, donors, w, nrm

    def cell_types(self):
        t = np.zeros((self.ny, self.nx), dtype=np.uint8)
        self._chk(lib().jxo_cell_types(self._h, t.ctypes.data))
        return t

    def guard_count(self):
        return int(lib().jxo_guard_count(self._h))

    def count_ops(self, U):
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.shape == (4, self.ny, self.nx)
        c = (C.c_longlong * 5)()
        self._chk(lib().jxo_count_ops(self._h, _d(U), c))
        return dict(zip(("add", "mul", "div", "sqrt", "cmp"), [int(x) for x in c]))

    def mlp_eval(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.zeros(4)
        self._chk(lib().jxo_mlp_eval(self._h, _d(x), _d(y)))
        return y
