"""SURVEY.md section 8(f) rank 3, reverse mode: the adjoint of the one-dimensional Euler / Navier-Stokes step (adjoint1d_kernel.cuh,
jxs_step_fixed_dt_record / jxs_adjoint_steps) through the C ABI.  -m gpu.

* element by element against the oracle's adjoint O13 (the transpose written out from its definition with the tangent
  O12, one tangent run per entry) on sizes that span several CTAs and a ragged tail, for every boundary condition;
* at sizes the oracle cannot reach: the identity every adjoint satisfies with its tangent,
  <Ubar_out, J Udot + J_gamma gamma_dot> = <J^T Ubar_out, Udot> + gamma_bar gamma_dot, with the tangent kernel;
* the use the paper makes of it (L149): dL/dgamma of the loss of Eq. 14 by backpropagation = the forward-mode value.
Tolerance: the adjoint is a sum of the same kind of terms as the value: <= 1e-11 of its max for a few steps.
"""
import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import dev, jxs, rel_err
from test_gpu_tangent import PER, oracle_rows, smooth1d

pytestmark = pytest.mark.gpu


def gpu_adjoint(case, Ubar, dt, nsteps, nu=0.0):
    s = jxs().Solver.from_case(case)
    if nu:
        s.set_artificial_viscosity(nu)
    U, B = dev(case["U0"]), dev(Ubar)
    s.step_fixed_dt_record(U, dt, nsteps)
    gbar = s.adjoint_steps(B)
    return U.cpu().numpy(), B.cpu().numpy(), gbar, s


@pytest.mark.parametrize("name,nx,nsteps,mu,nu", [("sod", 60, 1, 0.0, 0.0), ("sod", 130, 2, 0.0, 0.0),
                                                  ("smooth_periodic", 122, 2, 0.0, 0.0),
                                                  ("smooth_reflective", 123, 2, 0.0, 0.0),
                                                  ("smooth_inflow", 70, 2, 0.0, 0.0),
                                                  ("smooth_periodic", 90, 2, 3e-3, 0.0),     # Navier-Stokes terms
                                                  ("smooth_inflow", 125, 2, 2e-3, 1e-3),     # ... and nu Lap_h(U)
                                                  ("sod", 64, 2, 0.0, 2e-3)])
def test_adjoint_matches_the_transposed_oracle_tangent(name, nx, nsteps, mu, nu):
    if name == "sod":
        case = wl.sod1d(nx)
        # let the waves exist before differentiating: start from the state after 20 steps
        c2, o = oracle_rows(case)
        case["U0"] = np.ascontiguousarray(o.step_fixed_dt(c2["U0"], 0.2 * case["dx"], 20)[:, :1])
    else:
        bc = dict(PER)
        if name == "smooth_reflective":
            bc.update(xlo="reflective", xhi="reflective")
        if name == "smooth_inflow":
            bc.update(xlo="inflow", xhi="transmissive", inflow=(1.0, 0.4, 0.0, 1.0))
        case = smooth1d(nx, mu, bc)
    dt = 0.2 * case["dx"]
    Ubar = np.random.default_rng(nx).normal(size=case["U0"].shape)
    c2, o = oracle_rows(case, nu)
    want, gwant = o.step_fixed_dt_adjoint(c2["U0"], Ubar, dt, nsteps, planar=True)
    U, got, gbar, _ = gpu_adjoint(case, Ubar, dt, nsteps, nu)
    assert rel_err(U, o.step_fixed_dt(c2["U0"], dt, nsteps)[:, :1]) <= 1e-12
    assert rel_err(got, want) <= 1e-11
    assert gbar == pytest.approx(gwant, rel=1e-10, abs=1e-12 * np.abs(want).max())


@pytest.mark.parametrize("nsteps", [1, 2, 3])
def test_adjoint_of_the_paper_literal_euler_update(nsteps):
    """Eq. 10 as printed, reversed: against the transposed oracle tangent of the same update"""
    case = smooth1d(100, 1e-3, dict(PER, xlo="reflective", xhi="transmissive"))
    nu, dt = 2e-3, 0.1 * case["dx"]
    Ubar = np.random.default_rng(3).normal(size=case["U0"].shape)
    c2, o = oracle_rows(case, nu)
    want, gwant = o.step_fixed_dt_adjoint(c2["U0"], Ubar, dt, nsteps, planar=True, scheme="euler")
    s = jxs().Solver.from_case(case)
    s.set_artificial_viscosity(nu)
    s.set_time_integrator(jxs().EULER)
    U, B = dev(case["U0"]), dev(Ubar)
    s.step_fixed_dt_record(U, dt, nsteps)
    s.set_time_integrator(jxs().SSPRK3)      # the recording remembers its integrator
    gbar = s.adjoint_steps(B)
    assert rel_err(B.cpu().numpy(), want) <= 1e-11
    assert gbar == pytest.approx(gwant, rel=1e-10, abs=1e-12 * np.abs(want).max())


@pytest.mark.parametrize("nx,nsteps", [(1000, 30), (300007, 5)])
def test_adjoint_pairs_with_the_tangent_kernel(nx, nsteps):
    case = wl.sod1d(nx)
    dt = 0.2 * case["dx"]
    s0 = jxs().Solver.from_case(case)
    U0 = dev(case["U0"])
    s0.step_fixed_dt(U0, dt, 40)                       # waves first
    case["U0"] = U0.cpu().numpy()
    rng = np.random.default_rng(1)
    Ubar = rng.normal(size=case["U0"].shape)
    Udot, gdot = rng.normal(size=case["U0"].shape), 0.8
    s = jxs().Solver.from_case(case)
    U, D = dev(case["U0"]), dev(Udot)
    s.step_fixed_dt_tangent(U, D, gdot, dt, nsteps)
    Ur, got, gbar, s2 = gpu_adjoint(case, Ubar, dt, nsteps)
    assert np.array_equal(Ur, jxs().Solver.from_case(case).step_fixed_dt(dev(case["U0"]), dt, nsteps).cpu().numpy())
    lhs = float(np.sum(Ubar * D.cpu().numpy()))
    rhs = float(np.sum(got * Udot)) + gbar * gdot
    assert lhs == pytest.approx(rhs, rel=1e-11, abs=1e-11 * np.sqrt(Ubar.size))
    # a second reverse sweep on the same recording gives the same result, bit for bit
    B2 = dev(Ubar)
    assert s2.adjoint_steps(B2) == gbar and np.array_equal(B2.cpu().numpy(), got)


def test_checkpointed_recording_gives_the_same_adjoint_bit_for_bit():
    case = smooth1d(3000, 1e-5, dict(PER, xlo="inflow", xhi="transmissive", inflow=(1.0, 0.4, 0.0, 1.0)))
    dt = 0.2 * case["dx"]   # (mu small enough for the explicit viscous step at this dx)
    Ubar = np.random.default_rng(5).normal(size=case["U0"].shape)
    U, full, gfull, s = gpu_adjoint(case, Ubar, dt, 12)
    s.step_fixed_dt(dev(case["U0"]), 0.5 * dt, 3)        # another call in between must not disturb the reverse sweep
    s.set_adjoint_checkpointing(True)
    U2, B = dev(case["U0"]), dev(Ubar)
    s.step_fixed_dt_record(U2, dt, 12)
    s.step_fixed_dt(dev(case["U0"]), 0.5 * dt, 3)
    g = s.adjoint_steps(B)
    assert np.isfinite(full).all() and np.abs(full).max() > 0.1
    assert np.array_equal(U2.cpu().numpy(), U) and np.array_equal(B.cpu().numpy(), full) and g == gfull


def test_loss_gradient_by_backpropagation_equals_forward_mode():
    """dL/dgamma of Eq. 14 for the Sod inference, initial condition given in primitives (R23)"""
    nx, ns, g = 500, 60, 1.3
    dt = 0.2 / nx
    target = dev(wl.sod1d(nx)["U0"])
    jxs().Solver.from_case(wl.sod1d(nx)).step_fixed_dt(target, dt, ns)
    case = wl.sod1d(nx, gamma=g)
    seed = wl.dcons_dgamma(case["U0"], g)
    s = jxs().Solver.from_case(case)
    U, D = dev(case["U0"]), dev(seed)
    s.step_fixed_dt_tangent(U, D, 1.0, dt, ns)
    loss, dloss = s.mse_tangent(U, D, target)
    # reverse: Ubar = dL/dU_final = 2 (U - target) / N, then dL/dgamma = gamma_bar + <Ubar_0, dU_0/dgamma>
    s2 = jxs().Solver.from_case(case)
    U2 = dev(case["U0"])
    s2.step_fixed_dt_record(U2, dt, ns)
    B = 2.0 * (U2 - target) / U2.numel()
    gbar = s2.adjoint_steps(B)
    assert gbar + float((B.cpu().numpy() * seed).sum()) == pytest.approx(dloss, rel=1e-10)


def test_adjoint_rejects_what_it_does_not_do():
    E = jxs().JxsError
    case = wl.sod1d(64)
    s = jxs().Solver.from_case(case)
    U, B = dev(case["U0"]), dev(np.zeros_like(case["U0"]))
    with pytest.raises(E):
        s.adjoint_steps(B)                      # nothing recorded
    for dt, n in ((0.0, 1), (1e-3, 0), (1e-3, -2)):
        with pytest.raises(E):
            s.step_fixed_dt_record(U, dt, n)
    s32 = jxs().Solver.from_case(case, dtype=torch.float32)
    with pytest.raises(E):
        s32.step_fixed_dt_record(dev(case["U0"], torch.float32), 1e-3, 1)
    v = wl.vortex(32)                             # two-dimensional handles: tests/test_gpu_deriv2d.py; not with a network
    sv = jxs().Solver.from_case(v)
    sv.set_flux_mlp(wl.mlp_weights(), *wl.mlp_scales())
    with pytest.raises(E):
        sv.step_fixed_dt_record(dev(v["U0"]), 1e-3, 1)
    # a zero adjoint stays zero
    s3 = jxs().Solver.from_case(case)
    s3.step_fixed_dt_record(dev(case["U0"]), 1e-3, 2)
    assert s3.adjoint_steps(B) == 0.0 and float(B.abs().max()) == 0.0


@pytest.mark.parametrize("with_mlp", [False, True])
def test_sweep_graphs_replay_bitwise(with_mlp):
    """The recorded forward sweep and the reverse sweep run as plain launches on the first call with given parameters,
    are captured into CUDA graphs on the second and replayed from the third on (run_sweep in csrc/jxs_api.cu): all of
    them must give the same bits as a handle with graph replay switched off (to round-off where the network's reverse
    sums with atomics), also after the parameters change."""
    case = wl.sod1d(500)
    dt = 0.2 * case["dx"]
    rng = np.random.default_rng(5)
    seed_bar = torch.tensor(rng.normal(size=case["U0"].shape), device="cuda")
    m = 6
    targets = torch.tensor(rng.normal(size=(m,) + case["U0"].shape) * 0.01 + case["U0"], device="cuda")

    def make(graph):
        s = jxs().Solver.from_case(case)
        if with_mlp:
            s.set_flux_mlp(wl.mlp_weights(3), *wl.mlp_scales(out_factor=1e-2))
        s.set_graph_replay(graph)
        return s

    def run(s, steps):
        U = torch.tensor(case["U0"], device="cuda")
        s.step_fixed_dt_record(U, dt, steps)
        B = seed_bar.clone()
        g = s.adjoint_steps(B)
        out = [U.clone(), B.clone(), g]
        if steps == m:
            U2 = torch.tensor(case["U0"], device="cuda")
            s.step_fixed_dt_record(U2, dt, steps)
            B2 = torch.zeros_like(U2)
            loss, g2 = s.adjoint_steps_mse(targets, B2)
            out += [B2.clone(), loss, g2]
            if with_mlp:
                out.append(s.flux_mlp_gradient().copy())
        return out

    plain, graphed = make(False), make(True)
    launches = []
    for steps in (m, m, m, m, 4, 4, 4, m, m):   # plain / capture / replay, a change of key, and back
        want = run(plain, steps)
        l0 = graphed.launch_count()
        got = run(graphed, steps)
        launches.append(graphed.launch_count() - l0)
        for a, b in zip(got, want):
            if isinstance(a, torch.Tensor):
                if with_mlp:   # the network's reverse adds into the cells' adjoints with fp64 atomics
                    assert float((a - b).abs().max()) <= 1e-12 * float(b.abs().max())
                else:
                    assert torch.equal(a, b)
            elif isinstance(a, np.ndarray):   # the weights' gradient is summed with fp64 atomics: order varies
                assert np.allclose(a, b, rtol=1e-11, atol=1e-13 * np.abs(b).max())
            else:   # gamma_bar is a fixed-order sum; the loss of Eq. 14 is accumulated with atomics
                assert a == pytest.approx(b, rel=1e-13, abs=1e-300)
    assert launches[0] == launches[1] == launches[2]    # the replayed launches are still counted
