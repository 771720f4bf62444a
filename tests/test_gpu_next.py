"""SURVEY.md section 8(f) rows built so far, against the oracle / through the C ABI.  -m gpu.

* rank 2, paper-literal stepping (Eq. 10): U^{n+1} = U^n + dt L(U^n) with the nu Lap_h(U) term.
  The oracle side is the equation written out with the oracle's own L and s_max (numpy, one line per term).
* rank 4 (first half), concurrent handles: jxs_step_async / jxs_wait on one stream per handle give bitwise the
  results of the synchronous calls.
"""
import numpy as np
import pytest
import torch

from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import dev, jxs, make_pair, rel_err

pytestmark = pytest.mark.gpu


def oracle_forward_euler(o, U, cfl, nsteps, h):
    """Eq. 10 as printed, dt from the CFL rule R6 evaluated on U^n."""
    U = np.array(U, dtype=np.float64)
    for _ in range(nsteps):
        dt = cfl * h / o.max_wavespeed(U)
        U = U + dt * o.rhs(U)
    return U


@pytest.mark.parametrize("name,nu,nsteps", [("sod", 2e-3, 40), ("cylinder", 0.0, 25), ("cylinder_nu", 1e-3, 25)])
def test_forward_euler_matches_eq10(name, nu, nsteps):
    case = wl.sod(128, 128, 0) if name == "sod" else wl.shock_cylinder(192, 96, Ms=2.0)
    o, s = make_pair(case, nu=nu)
    s.set_time_integrator(jxs().EULER)
    fluid = o.cell_types() == 0 if case.get("phi") is not None else None
    U = dev(case["U0"])
    s.step(U, 0.2, nsteps)
    want = oracle_forward_euler(o, case["U0"], 0.2, nsteps, min(case["dx"], case["dy"]))
    assert rel_err(U.cpu().numpy(), want, fluid) <= 1e-9
    # and back to the default integrator
    s.set_time_integrator(jxs().SSPRK3)
    U2 = dev(case["U0"])
    s.step(U2, 0.2, 3)
    assert rel_err(U2.cpu().numpy(), o.step(case["U0"], 0.2, 3), fluid) <= 1e-9


def test_forward_euler_odd_step_count_and_time():
    """the two padded buffers swap roles every Euler step: odd and even counts both land in U"""
    case = wl.vortex(64)
    o, s = make_pair(case)
    s.set_time_integrator(jxs().EULER)
    for nsteps in (1, 2, 3):
        U = dev(case["U0"])
        s.step(U, 0.3, nsteps)
        assert rel_err(U.cpu().numpy(), oracle_forward_euler(o, case["U0"], 0.3, nsteps, case["dx"])) <= 1e-11
    with pytest.raises(jxs().JxsError):
        s.set_time_integrator(7)


def test_async_handles_on_streams_match_synchronous_calls():
    cases = wl.batch_cases(3, nx=160, ny=96)
    streams = [torch.cuda.Stream() for _ in cases]
    ref = []
    for c in cases:
        s = jxs().Solver.from_case(c)
        U = dev(c["U0"])
        s.step(U, 0.4, 12)
        ref.append((U.cpu().numpy(), s.time()))
    solvers = [jxs().Solver.from_case(c, stream=st) for c, st in zip(cases, streams)]
    for s in solvers:
        s.set_concurrent_handles(len(solvers))  # a performance hint: results must not change
    torch.cuda.synchronize()
    Us = [dev(c["U0"]) for c in cases]
    torch.cuda.synchronize()
    for s, U in zip(solvers, Us):
        s.step_async(U, 0.4, 5)
    for s, U in zip(solvers, Us):
        s.step_async(U, 0.4, 7)
    for s in solvers:
        s.wait()
    for s, U, (want, tm) in zip(solvers, Us, ref):
        assert np.array_equal(U.cpu().numpy(), want)
        assert s.time() == tm


# ------------------------------------------------------------------ rank 2, second half: the 1D path (ny = 1)
def oracle_rows(case):
    """the 2D oracle on the 1D problem repeated over 8 identical rows (periodic in y)"""
    from oracle import jxo
    c = wl.as_rows(case)
    return c, jxo.Oracle(c["nx"], c["ny"], c["dx"], c["dy"], c["gamma"], c["mu"], c["Pr"], c["bc"])


@pytest.mark.parametrize("nx", [200, 254, 255, 1021])  # one CTA short, exactly one, one cell more, ragged
def test_1d_rhs_and_steps_match_the_planar_oracle(nx):
    case = wl.sod1d(nx)
    c2, o = oracle_rows(case)
    s = jxs().Solver.from_case(case)
    got = s.rhs(dev(case["U0"])).cpu().numpy()
    want = o.rhs(c2["U0"])
    assert np.array_equal(want[:, 0], want[:, 5])          # the oracle's rows stay identical
    assert rel_err(got, want[:, :1]) <= 1e-12
    U = dev(case["U0"])
    s.step(U, 0.4, 60)
    assert rel_err(U.cpu().numpy(), o.step(c2["U0"], 0.4, 60)[:, :1]) <= 1e-9
    assert abs(s.max_wavespeed(dev(case["U0"])) / o.max_wavespeed(c2["U0"]) - 1) <= 1e-14


def test_1d_paper_literal_euler_with_nu_and_fp32():
    case = wl.sod1d(300)
    c2, o = oracle_rows(case)
    o.set_artificial_viscosity(1e-3)
    s = jxs().Solver.from_case(case)
    s.set_artificial_viscosity(1e-3)
    s.set_time_integrator(jxs().EULER)
    U = dev(case["U0"])
    s.step(U, 0.2, 50)
    want = oracle_forward_euler(o, c2["U0"], 0.2, 50, case["dx"])
    assert rel_err(U.cpu().numpy(), want[:, :1]) <= 1e-9
    s32 = jxs().Solver.from_case(case, dtype=torch.float32)
    o2 = oracle_rows(case)[1]
    got = s32.rhs(dev(case["U0"], torch.float32)).cpu().numpy()
    assert rel_err(got, o2.rhs(c2["U0"])[:, :1]) <= 1e-4


def test_1d_navier_stokes_matches_the_planar_oracle():
    case = wl.sod1d(400)
    case["mu"] = 2e-3
    x = (np.arange(400) + 0.5) / 400
    rho = 1.0 + 0.3 * np.sin(2 * np.pi * x)
    u = 0.4 * np.cos(2 * np.pi * x)
    v = 0.2 * np.sin(4 * np.pi * x)  # a planar flow may carry a transverse velocity
    p = 1.0 + 0.2 * np.cos(2 * np.pi * x + 0.3)
    case["U0"] = wl.cons_from_prim(rho[None, :], u[None, :], v[None, :], p[None, :])
    case["bc"] = dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic")
    c2, o = oracle_rows(case)
    s = jxs().Solver.from_case(case)
    assert rel_err(s.rhs(dev(case["U0"])).cpu().numpy(), o.rhs(c2["U0"])[:, :1]) <= 1e-12
    U = dev(case["U0"])
    s.step(U, 0.4, 40)
    assert rel_err(U.cpu().numpy(), o.step(c2["U0"], 0.4, 40)[:, :1]) <= 1e-9


def test_1d_sod_converges_to_the_exact_solution():
    """PAPER.md L141-147 (Fig. 2): the solution at t = 0.2 approaches the exact Riemann solution under refinement"""
    import refs
    errs = []
    for nx in (500, 2000):
        case = wl.sod1d(nx)
        s = jxs().Solver.from_case(case)
        U = dev(case["U0"])
        t, dt = 0.0, 0.2 / (2 * nx)  # fixed step well inside the CFL limit (s_max ~ 2.2), lands on t = 0.2 exactly
        s.step_fixed_dt(U, dt, 2 * nx)
        assert abs(s.time()[0] - 0.2) < 1e-12
        rho = U.cpu().numpy()[0, 0]
        x = (np.arange(nx) + 0.5) / nx
        exact = np.array([refs.riemann_sample((xx - 0.5) / 0.2, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)[0] for xx in x])
        errs.append(np.mean(np.abs(rho - exact)))
    assert errs[1] < 0.4 * errs[0] and errs[1] < 2e-3, errs


def test_1d_rejects_what_it_does_not_do():
    case = wl.sod1d(64)
    s = jxs().Solver.from_case(case)
    with pytest.raises(jxs().JxsError):
        s.set_ibm(-np.ones((1, 64)))
    with pytest.raises(jxs().JxsError):
        s.set_flux_cnn(wl.cnn_weights(), *wl.cnn_scales())
