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
