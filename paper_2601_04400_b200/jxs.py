"""Thin ctypes binding of include/jxs.h with the same names (argument marshalling only).

torch is used for device memory and streams; fields are torch CUDA tensors [4, ny, nx]
(float64 or float32, contiguous).  If the CUDA library cannot be built or loaded, or there
is no CUDA device, this module raises: there is no CPU fallback and it never touches oracle/.
"""
import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENUMERIC = 0, 1, 2, 3, 4, 5
BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_INFLOW = 0, 1, 2, 3
F64, F32 = 0, 1
SSPRK3, EULER = 0, 1
_BC_NAMES = {"periodic": 0, "transmissive": 1, "reflective": 2, "inflow": 3}

EXPORTS = ("jxs_create", "jxs_destroy", "jxs_last_error", "jxs_set_ibm", "jxs_set_flux_mlp",
           "jxs_set_artificial_viscosity", "jxs_rhs", "jxs_max_wavespeed", "jxs_step", "jxs_step_fixed_dt",
           "jxs_step_host", "jxs_rhs_host", "jxs_get_time", "jxs_launch_count", "jxs_set_profiling",
           "jxs_stage_time", "jxs_ibm_ghost_count", "jxs_measure_fp64_peak", "jxs_flux_correction",
           "jxs_flux_mlp_time", "jxs_step_async", "jxs_wait", "jxs_set_time_integrator",
           "jxs_set_concurrent_handles", "jxs_set_flux_cnn", "jxs_flux_cnn_inputs",
           "jxs_step_fixed_dt_tangent", "jxs_mse_tangent", "jxs_step_fixed_dt_record", "jxs_adjoint_steps", "jxs_set_gamma",
           "jxs_set_adjoint_checkpointing", "jxs_flux_mlp_gradient", "jxs_adjoint_steps_mse",
           "jxs_tune", "jxs_set_rows_per_segment", "jxs_set_graph_replay", "jxs_create_batch", "jxs_batch_size",
           "jxs_get_time_batch", "jxs_set_active_rows", "jxs_shard_begin", "jxs_shard_smax", "jxs_shard_step_begin",
           "jxs_shard_rows", "jxs_shard_stage", "jxs_shard_end", "jxs_measure_unit_rate", "jxs_mse_tangent_noalloc")


class jxs_bc(C.Structure):
    _fields_ = [("xlo", C.c_int), ("xhi", C.c_int), ("ylo", C.c_int), ("yhi", C.c_int),
                ("inflow", C.c_double * 4)]


class JxsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"jxs error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load (building first if the sources are newer) paper_2601_04400_b200/libjxs.so."""
    global _lib
    if _lib is None:
        path = os.environ.get("JXS_LIB") or _build.LIB  # JXS_LIB: use this prebuilt library as it is
        if path == _build.LIB and os.path.exists(os.path.join(_build.CSRC, "jxs_api.cu")):
            # a failed rebuild raises: loading an older libjxs.so would validate and time code that is not HEAD
            path = _build.build()
        L = C.CDLL(path)
        vp, dp = C.c_void_p, C.POINTER(C.c_double)
        L.jxs_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                 C.POINTER(jxs_bc), C.c_int, vp, C.POINTER(vp)]
        L.jxs_create_batch.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, dp, C.c_double,
                                       C.POINTER(jxs_bc), C.c_int, vp, C.POINTER(vp)]
        L.jxs_batch_size.argtypes = [vp]
        L.jxs_get_time_batch.argtypes = [vp, dp, dp]
        L.jxs_set_active_rows.argtypes = [vp, C.c_int, C.c_int]
        L.jxs_shard_begin.argtypes = [vp, vp]
        L.jxs_shard_smax.argtypes = [vp, vp, C.c_int]
        L.jxs_shard_step_begin.argtypes = [vp, C.c_double, C.c_double]
        L.jxs_shard_rows.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, C.c_int]
        L.jxs_shard_stage.argtypes = [vp, C.c_int]
        L.jxs_shard_end.argtypes = [vp, vp, C.c_int]
        L.jxs_destroy.argtypes = [vp]
        L.jxs_destroy.restype = None
        L.jxs_last_error.argtypes = [vp]
        L.jxs_last_error.restype = C.c_char_p
        L.jxs_set_ibm.argtypes = [vp, vp]
        L.jxs_set_flux_mlp.argtypes = [vp, vp, dp, dp]
        L.jxs_set_artificial_viscosity.argtypes = [vp, C.c_double]
        L.jxs_rhs.argtypes = [vp, vp, vp]
        L.jxs_rhs_host.argtypes = [vp, vp, vp]
        L.jxs_max_wavespeed.argtypes = [vp, vp, dp]
        L.jxs_step.argtypes = [vp, vp, C.c_double, C.c_int]
        L.jxs_step_fixed_dt.argtypes = [vp, vp, C.c_double, C.c_int]
        L.jxs_step_host.argtypes = [vp, vp, C.c_double, C.c_int]
        L.jxs_step_async.argtypes = [vp, vp, C.c_double, C.c_int]
        L.jxs_wait.argtypes = [vp]
        L.jxs_set_time_integrator.argtypes = [vp, C.c_int]
        L.jxs_set_concurrent_handles.argtypes = [vp, C.c_int]
        L.jxs_tune.argtypes = [vp]
        L.jxs_set_rows_per_segment.argtypes = [vp, C.c_int]
        L.jxs_set_graph_replay.argtypes = [vp, C.c_int]
        L.jxs_set_flux_cnn.argtypes = [vp, vp, dp, dp]
        L.jxs_flux_cnn_inputs.argtypes = [vp, vp, vp, vp]
        L.jxs_step_fixed_dt_tangent.argtypes = [vp, vp, vp, C.c_double, C.c_double, C.c_int]
        L.jxs_mse_tangent.argtypes = [vp, vp, vp, vp, dp, dp]
        L.jxs_mse_tangent_noalloc.argtypes = [vp, vp, vp, vp, vp]
        L.jxs_step_fixed_dt_record.argtypes = [vp, vp, C.c_double, C.c_int]
        L.jxs_adjoint_steps.argtypes = [vp, vp, dp]
        L.jxs_set_gamma.argtypes = [vp, C.c_double]
        L.jxs_set_adjoint_checkpointing.argtypes = [vp, C.c_int]
        L.jxs_flux_mlp_gradient.argtypes = [vp, vp]
        L.jxs_adjoint_steps_mse.argtypes = [vp, vp, vp, dp, dp]
        L.jxs_get_time.argtypes = [vp, dp, dp]
        L.jxs_launch_count.argtypes = [vp]
        L.jxs_launch_count.restype = C.c_longlong
        L.jxs_set_profiling.argtypes = [vp, C.c_int]
        L.jxs_stage_time.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
        L.jxs_ibm_ghost_count.argtypes = [vp]
        L.jxs_measure_fp64_peak.argtypes = [vp, C.c_double, dp]
        L.jxs_measure_unit_rate.argtypes = [vp, C.c_int, C.c_double, dp]
        L.jxs_flux_correction.argtypes = [vp, vp, vp, vp]
        L.jxs_flux_mlp_time.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
        _lib = L
    return _lib


def make_bc(bc):
    b = jxs_bc()
    for side in ("xlo", "xhi", "ylo", "yhi"):
        setattr(b, side, _BC_NAMES[bc[side]])
    inflow = bc.get("inflow", (1.0, 0.0, 0.0, 1.0))
    for k in range(4):
        b.inflow[k] = float(inflow[k])
    return b


def measure_fp64_peak(ms=200.0, stream=None):
    t = C.c_double()
    st = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
    rc = lib().jxs_measure_fp64_peak(C.c_void_p(st), float(ms), C.byref(t))
    if rc != OK:
        raise JxsError(rc, "jxs_measure_fp64_peak")
    return t.value


RATE_DFMA, RATE_DFMA3, RATE_TANH = 0, 1, 2
MSE_NOALLOC_MAX_N = 1 << 26   # JXS_MSE_NOALLOC_MAX_N of include/jxs.h


def measure_unit_rate(what, ms=200.0, stream=None):
    t = C.c_double()
    st = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
    rc = lib().jxs_measure_unit_rate(C.c_void_p(st), int(what), float(ms), C.byref(t))
    if rc != OK:
        raise JxsError(rc, "jxs_measure_unit_rate")
    return t.value


class Solver:
    """One jxs_solver handle.  Methods are the C calls of include/jxs.h, name for name."""

    def __init__(self, nx, ny, dx, dy, gamma=1.4, mu=0.0, Pr=0.72, bc=None, dtype=torch.float64, stream=None):
        if not torch.cuda.is_available():
            raise JxsError(ECUDA, "no CUDA device: jxs has no CPU fallback")
        self.nx, self.ny = int(nx), int(ny)
        self.dtype = dtype
        assert dtype in (torch.float64, torch.float32)
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self._bc = make_bc(bc)
        self._h = C.c_void_p()
        rc = lib().jxs_create(self.nx, self.ny, float(dx), float(dy), float(gamma), float(mu), float(Pr),
                              C.byref(self._bc), F64 if dtype == torch.float64 else F32,
                              C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if rc != OK:
            raise JxsError(rc, "jxs_create")

    @classmethod
    def from_cases(cls, cases, dtype=torch.float64, stream=None):
        """jxs_create_batch: one handle for len(cases) independent cases of one grid size; fields are [nb, 4, ny, nx]."""
        if not torch.cuda.is_available():
            raise JxsError(ECUDA, "no CUDA device: jxs has no CPU fallback")
        c0, nb = cases[0], len(cases)
        self = cls.__new__(cls)
        self.nx, self.ny, self.nb, self.dtype = int(c0["nx"]), int(c0["ny"]), nb, dtype
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self._bcs = (jxs_bc * nb)(*[make_bc(c["bc"]) for c in cases])
        mu = (C.c_double * nb)(*[float(c["mu"]) for c in cases])
        self._h = C.c_void_p()
        rc = lib().jxs_create_batch(nb, self.nx, self.ny, float(c0["dx"]), float(c0["dy"]), float(c0["gamma"]), mu,
                                    float(c0["Pr"]), self._bcs, F64 if dtype == torch.float64 else F32,
                                    C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if rc != OK:
            raise JxsError(rc, "jxs_create_batch")
        if cases[0].get("phi") is not None:
            self.set_ibm(np.stack([c["phi"] for c in cases]))
        return self

    # ---- y-slab sharding (driven by sharded.ShardedSolver)
    def set_active_rows(self, j_lo, j_hi):
        self._chk(lib().jxs_set_active_rows(self._h, int(j_lo), int(j_hi)))

    def shard_begin(self, U):
        self._chk(lib().jxs_shard_begin(self._h, self._dev(U)))

    def shard_smax(self, v, set):
        assert v.is_cuda and v.dtype == torch.float64 and v.numel() == 1
        self._chk(lib().jxs_shard_smax(self._h, C.c_void_p(v.data_ptr()), int(bool(set))))

    def shard_step_begin(self, cfl, fixed_dt=0.0):
        self._chk(lib().jxs_shard_step_begin(self._h, float(cfl), float(fixed_dt)))

    def shard_rows(self, k, row0, nrows, rows, unpack):
        assert rows.is_cuda and rows.is_contiguous() and rows.dtype == self.dtype and tuple(rows.shape) == (4, nrows, self.nx)
        self._chk(lib().jxs_shard_rows(self._h, int(k), int(row0), int(nrows), C.c_void_p(rows.data_ptr()), int(bool(unpack))))

    def shard_stage(self, k):
        self._chk(lib().jxs_shard_stage(self._h, int(k)))

    def shard_end(self, U, nsteps):
        self._chk(lib().jxs_shard_end(self._h, self._dev(U), int(nsteps)))

    @classmethod
    def from_slab(cls, case, active, dtype=torch.float64, stream=None):
        """a rank's handle of a sharded run: the active rows are set before the immersed boundary"""
        s = cls(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"],
                dtype=dtype, stream=stream)
        s.set_active_rows(*active)
        if case.get("phi") is not None:
            s.set_ibm(case["phi"])
        return s

    def time_batch(self):
        n = getattr(self, "nb", 1)
        t, dt = (C.c_double * n)(), (C.c_double * n)()
        self._chk(lib().jxs_get_time_batch(self._h, t, dt))
        return list(t), list(dt)

    @classmethod
    def from_case(cls, case, dtype=torch.float64, stream=None):
        s = cls(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"],
                dtype=dtype, stream=stream)
        if case.get("phi") is not None:
            s.set_ibm(case["phi"])
        return s

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.jxs_destroy(self._h)
            self._h = None

    __del__ = close

    def _chk(self, rc):
        if rc != OK:
            raise JxsError(rc, lib().jxs_last_error(self._h).decode())

    def _dev(self, U):
        assert isinstance(U, torch.Tensor) and U.is_cuda and U.is_contiguous(), "device tensor expected"
        assert U.dtype == self.dtype and tuple(U.shape) == self._shape(), (U.dtype, tuple(U.shape))
        return C.c_void_p(U.data_ptr())

    def _shape(self):
        nb = getattr(self, "nb", 1)
        return (4, self.ny, self.nx) if nb == 1 else (nb, 4, self.ny, self.nx)

    def _host(self, U):
        assert isinstance(U, torch.Tensor) and not U.is_cuda and U.is_contiguous(), "host tensor expected"
        assert U.dtype == self.dtype and tuple(U.shape) == self._shape()
        return C.c_void_p(U.data_ptr())

    def set_ibm(self, phi):
        if phi is None:
            self._chk(lib().jxs_set_ibm(self._h, None))
            return
        phi = np.ascontiguousarray(phi, dtype=np.float64)
        nb = getattr(self, "nb", 1)
        assert phi.shape == ((self.ny, self.nx) if nb == 1 else (nb, self.ny, self.nx))
        self._chk(lib().jxs_set_ibm(self._h, phi.ctypes.data))

    def set_flux_mlp(self, weights, in_scale=None, out_scale=None):
        if weights is None:
            self._chk(lib().jxs_set_flux_mlp(self._h, None, None, None))
            return
        w = np.ascontiguousarray(weights, dtype=np.float32)
        assert w.shape == (6020,)
        a = np.ascontiguousarray(in_scale, dtype=np.float64)
        b = np.ascontiguousarray(out_scale, dtype=np.float64)
        dp = C.POINTER(C.c_double)
        self._chk(lib().jxs_set_flux_mlp(self._h, w.ctypes.data, a.ctypes.data_as(dp), b.ctypes.data_as(dp)))

    def set_flux_cnn(self, weights, in_scale=None, out_scale=None):
        """The paper's 2D CNN flux: 6388 weights in OIHW order (None disables)."""
        if weights is None:
            self._chk(lib().jxs_set_flux_cnn(self._h, None, None, None))
            return
        w = np.ascontiguousarray(weights, dtype=np.float32)
        assert w.shape == (6388,)
        a = np.ascontiguousarray(in_scale, dtype=np.float64)
        b = np.ascontiguousarray(out_scale, dtype=np.float64)
        dp = C.POINTER(C.c_double)
        self._chk(lib().jxs_set_flux_cnn(self._h, w.ctypes.data, a.ctypes.data_as(dp), b.ctypes.data_as(dp)))

    def flux_cnn_inputs(self, U):
        """(Xx [4, ny, nx+1], Xy [4, nx, ny+1]) fp32 device tensors: the CNN's normalised input fields."""
        Xx = torch.empty((4, self.ny, self.nx + 1), dtype=torch.float32, device=U.device)
        Xy = torch.empty((4, self.nx, self.ny + 1), dtype=torch.float32, device=U.device)
        self._chk(lib().jxs_flux_cnn_inputs(self._h, self._dev(U), C.c_void_p(Xx.data_ptr()), C.c_void_p(Xy.data_ptr())))
        return Xx, Xy

    def flux_correction(self, U):
        """(dFx [4, ny, nx+1], dGy [4, ny+1, nx]) fp32 device tensors: Eq. 11's Delta F at every face."""
        dFx = torch.empty((4, self.ny, self.nx + 1), dtype=torch.float32, device=U.device)
        dGy = torch.empty((4, self.ny + 1, self.nx), dtype=torch.float32, device=U.device)
        self._chk(lib().jxs_flux_correction(self._h, self._dev(U), C.c_void_p(dFx.data_ptr()),
                                            C.c_void_p(dGy.data_ptr())))
        return dFx, dGy

    def flux_mlp_time(self):
        ms, n = C.c_double(), C.c_longlong()
        self._chk(lib().jxs_flux_mlp_time(self._h, C.byref(ms), C.byref(n)))
        return ms.value, int(n.value)

    def set_artificial_viscosity(self, nu):
        self._chk(lib().jxs_set_artificial_viscosity(self._h, float(nu)))

    def rhs(self, U, dUdt=None):
        if dUdt is None:
            dUdt = torch.empty_like(U)
        self._chk(lib().jxs_rhs(self._h, self._dev(U), self._dev(dUdt)))
        return dUdt

    def rhs_host(self, U, dUdt=None):
        if dUdt is None:
            dUdt = torch.empty_like(U)
        self._chk(lib().jxs_rhs_host(self._h, self._host(U), self._host(dUdt)))
        return dUdt

    def max_wavespeed(self, U):
        """s_max (a single handle) or the list of every member's s_max (a batch handle)"""
        nb = getattr(self, "nb", 1)
        s = (C.c_double * nb)()
        self._chk(lib().jxs_max_wavespeed(self._h, self._dev(U), s))
        return s[0] if nb == 1 else list(s)

    def step(self, U, cfl, nsteps):
        """In place on the device tensor U."""
        self._chk(lib().jxs_step(self._h, self._dev(U), float(cfl), int(nsteps)))
        return U

    def step_async(self, U, cfl, nsteps):
        """Enqueue only (no synchronisation); call wait() before reading U or the time."""
        self._chk(lib().jxs_step_async(self._h, self._dev(U), float(cfl), int(nsteps)))
        return U

    def wait(self):
        self._chk(lib().jxs_wait(self._h))

    def set_concurrent_handles(self, n):
        self._chk(lib().jxs_set_concurrent_handles(self._h, int(n)))

    def tune(self):
        self._chk(lib().jxs_tune(self._h))

    def set_rows_per_segment(self, rows):
        self._chk(lib().jxs_set_rows_per_segment(self._h, int(rows)))

    def set_graph_replay(self, on):
        self._chk(lib().jxs_set_graph_replay(self._h, int(bool(on))))

    def set_time_integrator(self, scheme):
        self._chk(lib().jxs_set_time_integrator(self._h, int(scheme)))

    def step_fixed_dt(self, U, dt, nsteps):
        self._chk(lib().jxs_step_fixed_dt(self._h, self._dev(U), float(dt), int(nsteps)))
        return U

    def step_fixed_dt_tangent(self, U, Udot, gamma_dot, dt, nsteps):
        """In place on the device tensors U and Udot (one-dimensional fp64 handles): the step and its tangent."""
        self._chk(lib().jxs_step_fixed_dt_tangent(self._h, self._dev(U), self._dev(Udot), float(gamma_dot),
                                                  float(dt), int(nsteps)))
        return U, Udot

    def mse_tangent(self, U, Udot, Utarget):
        """(mean((U - Utarget)^2), its derivative along Udot), Eq. 14."""
        loss, dloss = C.c_double(), C.c_double()
        self._chk(lib().jxs_mse_tangent(self._h, self._dev(U), self._dev(Udot), self._dev(Utarget),
                                        C.byref(loss), C.byref(dloss)))
        return loss.value, dloss.value

    def mse_tangent_noalloc(self, U, Udot, Utarget, out):
        """jxs_mse_tangent without any allocation or synchronisation: out (device tensor, 2 float64) receives
        (loss, dloss) when the handle's stream reaches the two kernels.  Shares one scratch array per device."""
        assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= 2
        self._chk(lib().jxs_mse_tangent_noalloc(self._h, self._dev(U), self._dev(Udot), self._dev(Utarget),
                                                C.c_void_p(out.data_ptr())))

    def set_gamma(self, gamma):
        self._chk(lib().jxs_set_gamma(self._h, float(gamma)))

    def adjoint_steps_mse(self, targets, Ubar):
        """Eq. 14 over the recorded steps: fills Ubar with dL/dU^n; returns (loss, gamma_bar).
        targets: device tensor [m][4][1][nx] float64, m = the recorded step count."""
        assert targets.is_cuda and targets.is_contiguous() and targets.dtype == torch.float64
        assert tuple(targets.shape[1:]) == (4, self.ny, self.nx)
        loss, g = C.c_double(), C.c_double()
        self._chk(lib().jxs_adjoint_steps_mse(self._h, C.c_void_p(targets.data_ptr()), self._dev(Ubar),
                                              C.byref(loss), C.byref(g)))
        return loss.value, g.value

    def flux_mlp_gradient(self):
        """The weights' gradient accumulated by the last adjoint_steps (one-dimensional handles), float64[6020]."""
        import numpy as np
        g = np.zeros(6020)
        self._chk(lib().jxs_flux_mlp_gradient(self._h, g.ctypes.data))
        return g

    def set_adjoint_checkpointing(self, on):
        self._chk(lib().jxs_set_adjoint_checkpointing(self._h, int(bool(on))))

    def step_fixed_dt_record(self, U, dt, nsteps):
        """jxs_step_fixed_dt that keeps the trajectory for adjoint_steps (fp64 handles; SSP-RK3 or forward Euler)."""
        self._chk(lib().jxs_step_fixed_dt_record(self._h, self._dev(U), float(dt), int(nsteps)))
        return U

    def adjoint_steps(self, Ubar):
        """In place: adjoint of the final state -> adjoint of the initial state; returns gamma_bar."""
        g = C.c_double()
        self._chk(lib().jxs_adjoint_steps(self._h, self._dev(Ubar), C.byref(g)))
        return g.value

    def step_host(self, U, cfl, nsteps):
        """In place on the host tensor U (copies inside the call)."""
        self._chk(lib().jxs_step_host(self._h, self._host(U), float(cfl), int(nsteps)))
        return U

    def time(self):
        t, dt = C.c_double(), C.c_double()
        self._chk(lib().jxs_get_time(self._h, C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def launch_count(self):
        return int(lib().jxs_launch_count(self._h))

    def set_profiling(self, on=True):
        self._chk(lib().jxs_set_profiling(self._h, int(bool(on))))

    def stage_time(self):
        ms, n = C.c_double(), C.c_longlong()
        self._chk(lib().jxs_stage_time(self._h, C.byref(ms), C.byref(n)))
        return ms.value, int(n.value)

    def ibm_ghost_count(self):
        return int(lib().jxs_ibm_ghost_count(self._h))
