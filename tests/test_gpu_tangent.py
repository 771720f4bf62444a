"""SURVEY.md section 8(f) rank 3, forward mode: the tangent of the one-dimensional step (tangent1d_kernel.cuh) and the
loss of Eq. 14, through the C ABI against the oracle's tangent (O12) on the planar 2D problem of 8 identical rows.
-m gpu.

Tolerances: those BASELINE.json states for the primal path, for the value and for the derivative alike (relative to
each field's max): <= 1e-12 for one step, <= 1e-9 over tens of steps.  The derivative is a sum of the same kind of
terms as the value, each rounded once on either side (measured: 2e-15 after one step, 2e-13 after 300).
"""
import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import dev, jxs, rel_err

pytestmark = pytest.mark.gpu

PER = dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic")


def oracle_rows(case, nu=0.0):
    c = wl.as_rows(case)
    o = jxo.Oracle(c["nx"], c["ny"], c["dx"], c["dy"], c["gamma"], c["mu"], c["Pr"], c["bc"])
    if nu:
        o.set_artificial_viscosity(nu)
    return c, o


def rows(D, ny=8):
    return np.ascontiguousarray(np.repeat(D, ny, axis=1))


def both(case, Udot, gamma_dot, dt, nsteps, nu=0.0):
    c2, o = oracle_rows(case, nu)
    Uo, Do = o.step_fixed_dt_tangent(c2["U0"], rows(Udot), gamma_dot, dt, nsteps)
    s = jxs().Solver.from_case(case)
    if nu:
        s.set_artificial_viscosity(nu)
    U, D = dev(case["U0"]), dev(Udot)
    s.step_fixed_dt_tangent(U, D, gamma_dot, dt, nsteps)
    return (U.cpu().numpy(), D.cpu().numpy()), (Uo[:, :1], Do[:, :1]), s


def smooth1d(nx, mu=0.0, bc=PER):
    case = wl.sod1d(nx)
    x = (np.arange(nx) + 0.5) / nx
    rho = 1.0 + 0.3 * np.sin(2 * np.pi * x)
    u = 0.4 * np.cos(2 * np.pi * x)
    v = 0.2 * np.sin(4 * np.pi * x)
    p = 1.0 + 0.2 * np.cos(2 * np.pi * x + 0.3)
    case["U0"] = wl.cons_from_prim(rho[None, :], u[None, :], v[None, :], p[None, :])
    case["bc"] = dict(bc)
    case["mu"] = mu
    return case


@pytest.mark.parametrize("nx", [100, 126, 127, 1021])  # one CTA short, exactly one, one cell more, ragged
def test_tangent_sod_one_step_and_many(nx):
    case = wl.sod1d(nx)
    Udot = wl.dcons_dgamma(case["U0"], case["gamma"]) + 0.05 * wl.smooth_direction(case["U0"].shape, seed=nx)
    dt = 0.2 * case["dx"]
    (U, D), (Uo, Do), _ = both(case, Udot, 1.0, dt, 1)
    assert rel_err(U, Uo) <= 1e-12
    assert rel_err(D, Do) <= 1e-12
    (U, D), (Uo, Do), s = both(case, Udot, 1.0, dt, 50)
    assert rel_err(U, Uo) <= 1e-9
    assert rel_err(D, Do) <= 1e-9
    assert abs(s.time()[0] - 50 * dt) < 1e-14
    # the value part is the primal path
    s2 = jxs().Solver.from_case(case)
    U2 = dev(case["U0"])
    s2.step_fixed_dt(U2, dt, 50)
    assert rel_err(U, U2.cpu().numpy()) <= 1e-11


@pytest.mark.parametrize("mu,nu,bc", [(0.0, 0.0, PER), (2e-3, 0.0, PER), (2e-3, 1e-3, PER),
                                      (0.0, 0.0, dict(PER, xlo="reflective", xhi="reflective")),
                                      (1e-3, 0.0, dict(PER, xlo="inflow", xhi="transmissive"))])
def test_tangent_smooth_flow_viscous_terms_and_boundaries(mu, nu, bc):
    case = smooth1d(380, mu, bc)
    if bc["xlo"] == "inflow":
        case["bc"]["inflow"] = (1.0, 0.4, 0.0, 1.0)
    Udot = wl.smooth_direction(case["U0"].shape, seed=11) + wl.dcons_dgamma(case["U0"], case["gamma"])
    dt = 0.15 * case["dx"]
    (U, D), (Uo, Do), _ = both(case, Udot, 0.7, dt, 1, nu)
    assert rel_err(U, Uo) <= 1e-12
    assert rel_err(D, Do) <= 1e-12
    (U, D), (Uo, Do), _ = both(case, Udot, 0.7, dt, 30, nu)
    assert rel_err(U, Uo) <= 1e-9
    assert rel_err(D, Do) <= 1e-9


@pytest.mark.parametrize("nsteps", [1, 2, 7])  # the two buffers swap roles every Euler step: odd and even counts
def test_tangent_of_the_paper_literal_euler_update(nsteps):
    """Eq. 10 as printed (forward Euler + nu Lap_h(U)), differentiated: against the oracle's tangent of the same update"""
    case = smooth1d(300, 1e-3, dict(PER, xlo="inflow", xhi="transmissive", inflow=(1.0, 0.4, 0.0, 1.0)))
    nu, dt = 2e-3, 0.1 * case["dx"]
    Udot = wl.smooth_direction(case["U0"].shape, seed=21) + wl.dcons_dgamma(case["U0"], case["gamma"])
    c2, o = oracle_rows(case, nu)
    Uo, Do = o.step_fixed_dt_tangent(c2["U0"], rows(Udot), 0.6, dt, nsteps, scheme="euler")
    s = jxs().Solver.from_case(case)
    s.set_artificial_viscosity(nu)
    s.set_time_integrator(jxs().EULER)
    U, D = dev(case["U0"]), dev(Udot)
    s.step_fixed_dt_tangent(U, D, 0.6, dt, nsteps)
    assert rel_err(U.cpu().numpy(), Uo[:, :1]) <= 1e-12
    assert rel_err(D.cpu().numpy(), Do[:, :1]) <= 1e-12
    assert abs(s.time()[0] - nsteps * dt) < 1e-15


def test_tangent_is_the_derivative_of_the_gpu_step():
    """central differences of jxs_step_fixed_dt itself (no oracle): the kernel differentiates what the primal computes"""
    nx, ns, h = 300, 20, 1e-6
    dt = 0.2 / nx
    U, D = dev(wl.sod1d(nx)["U0"]), dev(wl.dcons_dgamma(wl.sod1d(nx)["U0"], 1.4))
    jxs().Solver.from_case(wl.sod1d(nx)).step_fixed_dt_tangent(U, D, 1.0, dt, ns)
    ends = []
    for g in (1.4 + h, 1.4 - h):
        c = wl.sod1d(nx, gamma=g)
        Ug = dev(c["U0"])
        jxs().Solver.from_case(c).step_fixed_dt(Ug, dt, ns)
        ends.append(Ug.cpu().numpy())
    fd = (ends[0] - ends[1]) / (2 * h)
    assert rel_err(D.cpu().numpy(), fd) <= 1e-5


def test_mse_tangent_matches_the_definition():
    rng = np.random.default_rng(5)
    for nx in (37, 1000, 300001):
        case = wl.sod1d(nx)
        s = jxs().Solver.from_case(case)
        U, D, T = (rng.normal(size=(4, 1, nx)) for _ in range(3))
        loss, dloss = s.mse_tangent(dev(U), dev(D), dev(T))
        want = jxo.mse_tangent(U, D, T)
        assert loss == pytest.approx(want[0], rel=1e-13)
        assert dloss == pytest.approx(want[1], rel=1e-11, abs=1e-15)
        assert (loss, dloss) == s.mse_tangent(dev(U), dev(D), dev(T))  # fixed summation order


def test_gamma_inference_on_the_gpu():
    """PAPER.md L149 / Fig. 3(b): gamma from Sod data, every step in the kernels; the oracle's loop next to it"""
    nx, ns = 500, 100
    dt = 0.2 / nx
    base = wl.sod1d(nx)
    target = dev(base["U0"])
    jxs().Solver.from_case(base).step_fixed_dt(target, dt, ns)   # the data: gamma = 1.4
    g, hist = 1.25, []
    for _ in range(6):
        c = wl.sod1d(nx, gamma=g)
        s = jxs().Solver.from_case(c)
        U, D = dev(c["U0"]), dev(wl.dcons_dgamma(c["U0"], g))
        s.step_fixed_dt_tangent(U, D, 1.0, dt, ns)
        loss, dloss = s.mse_tangent(U, D, target)
        hist.append((g, loss, dloss))
        g -= float(((U - target) * D).sum() / (D * D).sum())     # Gauss-Newton on the one unknown
    assert abs(g - 1.4) < 1e-8, hist
    assert hist[-1][1] < 1e-16 < hist[0][1]
    assert hist[0][2] < 0  # below the true gamma the loss falls with gamma
    # first iterate against the oracle's
    c = wl.sod1d(nx, gamma=1.25)
    c2, o = oracle_rows(c)
    Uo, Do = o.step_fixed_dt_tangent(c2["U0"], rows(wl.dcons_dgamma(c["U0"], 1.25)), 1.0, dt, ns)
    want = jxo.mse_tangent(Uo[:, :1], Do[:, :1], target.cpu().numpy())
    assert hist[0][1] == pytest.approx(want[0], rel=1e-8)
    assert hist[0][2] == pytest.approx(want[1], rel=1e-6)


def test_set_gamma_keeps_one_handle_through_the_inference():
    """jxs_set_gamma: the optimisation loop of P:L149 on one handle; results equal those of a fresh handle"""
    nx, ns = 400, 60
    dt = 0.2 / nx
    target = dev(wl.sod1d(nx)["U0"])
    jxs().Solver.from_case(wl.sod1d(nx)).step_fixed_dt(target, dt, ns)
    s = jxs().Solver.from_case(wl.sod1d(nx, gamma=1.6))
    g = 1.6
    for it in range(6):
        s.set_gamma(g)
        c = wl.sod1d(nx, gamma=g)
        U, D = dev(c["U0"]), dev(wl.dcons_dgamma(c["U0"], g))
        s.step_fixed_dt_tangent(U, D, 1.0, dt, ns)
        if it == 1:   # bitwise what a handle created with this gamma gives (graphs re-captured, nothing stale)
            U2, D2 = dev(c["U0"]), dev(wl.dcons_dgamma(c["U0"], g))
            jxs().Solver.from_case(c).step_fixed_dt_tangent(U2, D2, 1.0, dt, ns)
            assert torch.equal(U, U2) and torch.equal(D, D2)
        g -= float(((U - target) * D).sum() / (D * D).sum())
    assert abs(g - 1.4) < 1e-8
    # the primal calls follow as well, and a recording made before the change is refused
    s.set_gamma(1.4)
    U = dev(wl.sod1d(nx)["U0"])
    s.step_fixed_dt(U, dt, ns)
    assert torch.equal(U, target)
    s.step_fixed_dt_record(dev(wl.sod1d(nx)["U0"]), dt, 3)
    s.set_gamma(1.5)
    with pytest.raises(jxs().JxsError):
        s.adjoint_steps(dev(np.zeros((4, 1, nx))))
    for bad in (1.0, 0.5, float("nan")):
        with pytest.raises(jxs().JxsError):
            s.set_gamma(bad)


def test_tangent_rejects_what_it_does_not_do():
    E = jxs().JxsError
    case = wl.sod1d(64)
    s = jxs().Solver.from_case(case)
    U, D = dev(case["U0"]), dev(np.zeros_like(case["U0"]))
    for bad in (dict(dt=0.0), dict(dt=-1.0), dict(nsteps=-1), dict(gamma_dot=float("nan"))):
        kw = dict(gamma_dot=1.0, dt=1e-3, nsteps=1)
        kw.update(bad)
        with pytest.raises(E):
            s.step_fixed_dt_tangent(U, D, **kw)
    s.step_fixed_dt_tangent(U, D, 1.0, 1e-3, 0)   # zero steps: nothing moves
    assert np.array_equal(U.cpu().numpy(), case["U0"]) and float(D.abs().max()) == 0.0
    s32 = jxs().Solver.from_case(case, dtype=torch.float32)
    with pytest.raises(E):
        s32.step_fixed_dt_tangent(dev(case["U0"], torch.float32), dev(case["U0"], torch.float32), 1.0, 1e-3, 1)
    c2 = wl.vortex(32)                            # two-dimensional handles: tests/test_gpu_deriv2d.py; not with a network
    s2 = jxs().Solver.from_case(c2)
    s2.set_flux_mlp(wl.mlp_weights(), *wl.mlp_scales())
    with pytest.raises(E):
        s2.step_fixed_dt_tangent(dev(c2["U0"]), dev(c2["U0"]), 1.0, 1e-3, 1)
