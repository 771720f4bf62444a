"""SURVEY.md section 8(f) rank 3 in TWO dimensions: the tangent and the adjoint of the 2D step (deriv2d_kernels.cuh;
jxs_step_fixed_dt_tangent / _record / jxs_adjoint_steps / _mse with ny > 1) through the C ABI.  -m gpu.

* tangent: element by element against the oracle's O12 (the solver on dual numbers) on small grids with every
  ingredient: periodic / inflow / transmissive / reflective frames with corners, a cylinder through the ghost-cell IBM,
  viscous fluxes with their cross derivatives, the nu-term, gamma's own direction;
* adjoint: element by element against the oracle's O13 (the transpose from its definition, one tangent run per entry)
  on grids of at most 24 x 24;
* at the size of BASELINE.json configs[2] (1024 x 512), where the oracle's transpose is out of reach, the identity
  every adjoint satisfies with its tangent, <Ubar, J Udot + J_gamma gamma_dot> = <J^T Ubar, Udot> + gamma_bar gamma_dot;
* the use the paper makes of it (Fig. 5d-f): gamma recovered from shock-cylinder data on a restricted
  domain of 8192 cells, by Gauss-Newton on the forward-mode derivative, and dL/dgamma of Eq. 14 by backpropagation.
Tolerance: the derivative is a sum of the same kind of terms as the value: <= 1e-11 of its max for a few steps.
"""
import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import MIXED, PER, dev, jxs, smooth_case

pytestmark = pytest.mark.gpu
G = 1.4


def oracle_of(case, nu=0.0):
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"])
    if case.get("phi") is not None:
        o.set_ibm(case["phi"])
    if nu:
        o.set_artificial_viscosity(nu)
    return o


def solver_of(case, nu=0.0):
    s = jxs().Solver.from_case(case)
    if nu:
        s.set_artificial_viscosity(nu)
    return s


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return max(np.abs(a[k] - b[k]).max() / max(np.abs(b).max(), 1e-300) for k in range(a.shape[0]))


def small_cylinder(nx, ny, Ms=2.0, Re=200.0):
    """shock-cylinder case on a small grid of [0,2] x [0,1]: a body of radius 3.3 dy at mid-domain, at least 8 cells
    from every edge (the library's rule), the shock 2.5 cells ahead of it"""
    dx, dy = 2.0 / nx, 1.0 / ny
    xc, yc, r = (nx // 2) * dx, 0.5, 3.3 * dy
    return wl.shock_cylinder(nx, ny, Ms=Ms, Re=Re, bodies=((xc, yc, r),), x_shock=xc - r - 2.5 * dx)


WALLS = dict(xlo="reflective", xhi="transmissive", ylo="reflective", yhi="periodic")
WALLS["ylo"] = "periodic"

CASES = {
    "vortex_24": (lambda: wl.vortex(24), 0.0),
    "jumps_periodic_40x30": (lambda: smooth_case(40, 30, 1, PER, jump=True), 0.0),
    "jumps_mixed_viscous_nu_130x20": (lambda: smooth_case(130, 20, 2, MIXED, mu=5e-3, jump=True), 2e-3),   # 2 CTAs along x
    "jumps_walls_viscous_20x130": (lambda: smooth_case(20, 130, 3, WALLS, mu=2e-3, jump=True), 0.0),       # 2 CTAs along y
    "cylinder_ns_64x32": (lambda: wl.shock_cylinder(64, 32, Ms=2.0, Re=200.0, x_shock=0.27), 0.0),
}


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("nsteps", [1, 3])
def test_tangent2d_matches_the_oracle(name, nsteps):
    make, nu = CASES[name]
    case = make()
    dt = 0.15 * min(case["dx"], case["dy"])
    Udir = wl.dcons_dgamma(case["U0"], case["gamma"]) + 0.1 * wl.smooth_direction(case["U0"].shape, seed=7)
    Uo, Do = oracle_of(case, nu).step_fixed_dt_tangent(case["U0"], Udir, 1.0, dt, nsteps)
    s = solver_of(case, nu)
    U, D = dev(case["U0"]), dev(Udir)
    s.step_fixed_dt_tangent(U, D, 1.0, dt, nsteps)
    assert rel(U.cpu().numpy(), Uo) <= 1e-12
    assert rel(D.cpu().numpy(), Do) <= 1e-11, (name, rel(D.cpu().numpy(), Do))
    # the value part is the primal step
    U2 = dev(case["U0"])
    solver_of(case, nu).step_fixed_dt(U2, dt, nsteps)
    assert rel(U.cpu().numpy(), U2.cpu().numpy()) <= 1e-12


def test_tangent2d_forward_euler_update():
    case = smooth_case(40, 30, 5, MIXED, mu=5e-3, jump=True)
    dt = 0.1 * min(case["dx"], case["dy"])
    Udir = 0.3 * wl.smooth_direction(case["U0"].shape, seed=3)
    o = oracle_of(case, 1e-3)
    Uo, Do = o.step_fixed_dt_tangent(case["U0"], Udir, 0.5, dt, 3, scheme="euler")
    s = solver_of(case, 1e-3)
    s.set_time_integrator(jxs().EULER)
    U, D = dev(case["U0"]), dev(Udir)
    s.step_fixed_dt_tangent(U, D, 0.5, dt, 3)
    assert rel(U.cpu().numpy(), Uo) <= 1e-12 and rel(D.cpu().numpy(), Do) <= 1e-11


ADJ_CASES = {
    "vortex_16": (lambda: wl.vortex(16), 0.0, 1),
    "jumps_mixed_viscous_nu_24x18": (lambda: smooth_case(24, 18, 2, MIXED, mu=5e-3, jump=True), 2e-3, 2),
    "jumps_walls_viscous_18x24": (lambda: smooth_case(18, 24, 3, WALLS, mu=2e-2, jump=True), 0.0, 2),
    "cylinder_ns_24x24": (lambda: small_cylinder(24, 24), 0.0, 2),
}


@pytest.mark.parametrize("name", list(ADJ_CASES))
def test_adjoint2d_matches_the_transposed_oracle_tangent(name):
    make, nu, nsteps = ADJ_CASES[name]
    case = make()
    dt = 0.15 * min(case["dx"], case["dy"])
    o = oracle_of(case, nu)
    U0 = case["U0"]
    if "cylinder" in name:   # let the shock reach the body first
        U0 = o.step_fixed_dt(U0, dt, 12)
    Ubar = np.random.default_rng(len(name)).normal(size=U0.shape)
    want, gwant = o.step_fixed_dt_adjoint(U0, Ubar, dt, nsteps)
    s = solver_of(case, nu)
    U, B = dev(U0), dev(Ubar)
    s.step_fixed_dt_record(U, dt, nsteps)
    gbar = s.adjoint_steps(B)
    assert rel(U.cpu().numpy(), o.step_fixed_dt(U0, dt, nsteps)) <= 1e-12
    got = B.cpu().numpy()
    assert rel(got, want) <= 1e-11, (name, rel(got, want))
    assert abs(gbar - gwant) <= 1e-11 * max(abs(gwant), np.abs(want).max()), (gbar, gwant)
    # a second sweep on the same recording gives the same bits; the checkpointed recording too
    B2 = dev(Ubar)
    assert s.adjoint_steps(B2) == gbar and torch.equal(B2, B)
    s.set_adjoint_checkpointing(True)
    U3, B3 = dev(U0), dev(Ubar)
    s.step_fixed_dt_record(U3, dt, nsteps)
    assert s.adjoint_steps(B3) == gbar and torch.equal(B3, B)


def test_adjoint2d_of_the_forward_euler_update():
    case = smooth_case(20, 16, 9, MIXED, mu=5e-3, jump=True)
    dt = 0.1 * min(case["dx"], case["dy"])
    o = oracle_of(case, 1e-3)
    Ubar = np.random.default_rng(4).normal(size=case["U0"].shape)
    want, gwant = o.step_fixed_dt_adjoint(case["U0"], Ubar, dt, 2, scheme="euler")
    s = solver_of(case, 1e-3)
    s.set_time_integrator(jxs().EULER)
    U, B = dev(case["U0"]), dev(Ubar)
    s.step_fixed_dt_record(U, dt, 2)
    gbar = s.adjoint_steps(B)
    assert rel(B.cpu().numpy(), want) <= 1e-11 and abs(gbar - gwant) <= 1e-11 * max(abs(gwant), 1.0)


@pytest.mark.parametrize("size", [(256, 128), (1024, 512)])
def test_adjoint_tangent_identity_at_config_size(size):
    """BASELINE.json configs[2] (Mach-2 shock on a cylinder, Navier-Stokes, IBM, inflow / outflow / walls) after the
    shock has reached the body: <Ubar, J Udot + J_gamma gdot> = <J^T Ubar, Udot> + gamma_bar gdot over 2 steps."""
    nx, ny = size
    case = wl.shock_cylinder(nx, ny, Ms=2.0, x_shock=0.29)
    s = solver_of(case)
    U0 = dev(case["U0"])
    s.step(U0, 0.4, 40)
    dt = s.time()[1]
    rng = np.random.default_rng(1)
    Udot = dev(wl.dcons_dgamma(U0.cpu().numpy(), G) + 0.2 * wl.smooth_direction(case["U0"].shape, seed=5))
    Ubar = dev(rng.normal(size=case["U0"].shape))
    gdot = 0.7
    U, D = U0.clone(), Udot.clone()
    s.step_fixed_dt_tangent(U, D, gdot, dt, 2)
    lhs = float((Ubar * D).sum())
    U2, B = U0.clone(), Ubar.clone()
    s.step_fixed_dt_record(U2, dt, 2)
    gbar = s.adjoint_steps(B)
    rhs = float((B * Udot).sum()) + gbar * gdot
    assert torch.allclose(U, U2, rtol=0, atol=1e-12 * float(U.abs().max()))
    scale = float((Ubar.abs() * D.abs()).sum())
    assert abs(lhs - rhs) <= 1e-11 * scale, (lhs, rhs, scale)


def test_gamma_inference_on_the_restricted_shock_cylinder_domain():
    """PAPER.md L170 / Fig. 5d-f: gamma from shock-cylinder data on a restricted domain of 8192 cells (128 x 64).
    Data: the GPU's own primal run at gamma = 1.4 (given in primitives, so the conserved start and the inflow state
    move with gamma).  Gauss-Newton on the forward-mode derivative from gamma = 1.3; then dL/dgamma of Eq. 14 by
    backpropagation through the recorded steps equals the forward-mode value."""
    ns = 30
    def case_at(g):
        return wl.shock_cylinder(128, 64, Ms=2.0, Re=500.0, gamma=g, x_shock=0.27)
    base = case_at(1.4)
    dt = 0.15 * base["dx"]
    target = dev(base["U0"])
    solver_of(base).step_fixed_dt(target, dt, ns)
    g = 1.3
    for _ in range(7):
        c = case_at(g)
        s = solver_of(c)
        U, D = dev(c["U0"]), dev(wl.dcons_dgamma(c["U0"], g))
        s.step_fixed_dt_tangent(U, D, 1.0, dt, ns)
        g -= float(((U - target) * D).sum() / (D * D).sum())
    assert abs(g - 1.4) < 1e-8, g
    # reverse mode: the same gradient of the one-target loss (Eq. 14 with m = 1 ... here over the ns unrolled steps)
    c = case_at(1.33)
    s = solver_of(c)
    U, D = dev(c["U0"]), dev(wl.dcons_dgamma(c["U0"], 1.33))
    s.step_fixed_dt_tangent(U, D, 1.0, dt, ns)
    loss, dloss = s.mse_tangent(U, D, target)
    U2 = dev(c["U0"])
    s.step_fixed_dt_record(U2, dt, ns)
    B = (U2 - target).mul_(2.0 / U2.numel())
    gbar = s.adjoint_steps(B)
    back = gbar + float((B * dev(wl.dcons_dgamma(c["U0"], 1.33))).sum())
    assert back == pytest.approx(dloss, rel=1e-9)


def test_adjoint2d_mse_sweep_and_argument_checks():
    """Eq. 14 over m unrolled steps with one target per step (jxs_adjoint_steps_mse) = the sum of single-target sweeps"""
    m = jxs()
    case = smooth_case(40, 30, 6, MIXED, mu=5e-3, jump=True)
    dt = 0.1 * min(case["dx"], case["dy"])
    s = solver_of(case)
    ns = 3
    rng = np.random.default_rng(2)
    targets = dev(np.stack([case["U0"] * (1 + 0.01 * rng.normal(size=case["U0"].shape)) for _ in range(ns)]))
    U = dev(case["U0"])
    s.step_fixed_dt_record(U, dt, ns)
    B = torch.empty_like(U)
    loss, gbar = s.adjoint_steps_mse(targets, B)
    # the same thing step by step: states from a primal run, gradients from single adjoint sweeps of growing length
    want_loss, want_B, want_g = 0.0, torch.zeros_like(U), 0.0
    for k in range(1, ns + 1):
        Uk = dev(case["U0"])
        s.step_fixed_dt_record(Uk, dt, k)
        r = Uk - targets[k - 1]
        want_loss += float((r * r).sum()) / (ns * U.numel())
        Bk = r * (2.0 / (ns * U.numel()))
        want_g += s.adjoint_steps(Bk)
        want_B += Bk
    assert loss == pytest.approx(want_loss, rel=1e-12)
    assert float((B - want_B).abs().max()) <= 1e-11 * float(want_B.abs().max())
    assert gbar == pytest.approx(want_g, rel=1e-9, abs=1e-13)
    # networks are not differentiated in 2D
    s.set_flux_mlp(wl.mlp_weights(), *wl.mlp_scales())
    with pytest.raises(m.JxsError) as e:
        s.step_fixed_dt_record(U, dt, 1)
    assert e.value.code == m.ESTATE


def test_sweep_graphs_of_the_2d_path_replay_bitwise():
    """The 2D recorded sweep and reverse sweep run as plain launches on the first call with given parameters, are captured
    as CUDA graphs on the second and replayed afterwards (run_sweep in csrc/jxs_api.cu): same bits as with graph replay
    switched off (the 2D reverse sweep has no atomics), also after a change of the step count and back."""
    case = wl.shock_cylinder(96, 48, Ms=2.0, Re=300.0, x_shock=0.28)
    s0 = solver_of(case)
    U0 = dev(case["U0"])
    s0.step(U0, 0.4, 10)
    dt = s0.time()[1]
    rng = np.random.default_rng(2)
    Ubar = dev(rng.normal(size=case["U0"].shape))
    targets = dev(rng.normal(size=(3,) + case["U0"].shape) * 0.01) + U0

    def run(s, steps):
        U, B = U0.clone(), Ubar.clone()
        s.step_fixed_dt_record(U, dt, steps)
        g = s.adjoint_steps(B)
        out = [U, B, g]
        if steps == 3:
            U2, B2 = U0.clone(), torch.zeros_like(U0)
            s.step_fixed_dt_record(U2, dt, steps)
            loss, g2 = s.adjoint_steps_mse(targets, B2)
            out += [B2, loss, g2]
        return out

    plain, graphed = solver_of(case), solver_of(case)
    plain.set_graph_replay(False)
    for steps in (3, 3, 3, 3, 2, 2, 2, 3, 3):
        want, got = run(plain, steps), run(graphed, steps)
        for a, b in zip(got, want):
            assert torch.equal(a, b) if isinstance(a, torch.Tensor) else a == b
