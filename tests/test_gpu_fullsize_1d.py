"""The one-dimensional paths (primal step, tangent, adjoint) at the size bench.py times them on, 3e6 cells, in the same
launch configuration, against the oracle on SAMPLED WINDOWS: one SSP-RK3 step moves information by at most 9 cells
(3 stages x 3-cell stencils), so the oracle run on cells [c-32, c+32) of the input with transmissive ends reproduces
the full problem's result on the window's centre exactly as if it had computed all 3e6 cells.  Inputs are the seeded
generator's (workloads.wavy1d), never a GPU result.  -m gpu.
"""
import numpy as np
import pytest

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import dev, jxs
from test_gpu_tangent import oracle_rows, rows

pytestmark = pytest.mark.gpu

NX = 3_000_000
HALF = 32      # half width of a window
MARGIN = 14    # cells at either end of a window that feel its artificial ends (9 + the 3 ghost cells, rounded up)


def centres():
    rng = np.random.default_rng(31)
    fixed = [HALF, NX // 2 - 3, NX // 2 + 20, NX - HALF, 126 * 1000 + 1, 254 * 5000]   # ends, the jump, CTA seams
    return fixed + [int(c) for c in rng.integers(HALF, NX - HALF, 6)]


def scale(a):
    return np.maximum(np.abs(a).max(axis=(1, 2), keepdims=True), 1e-300)


@pytest.fixture(scope="module")
def big():
    case = wl.wavy1d(NX)
    dt = 0.2 * case["dx"]
    rng = np.random.default_rng(32)
    Udot = wl.dcons_dgamma(case["U0"], case["gamma"]) + 0.1 * rng.normal(size=case["U0"].shape)
    Ubar = rng.normal(size=case["U0"].shape)
    s = jxs().Solver.from_case(case)
    U = dev(case["U0"])
    s.step_fixed_dt(U, dt, 1)
    Ut, Dt = dev(case["U0"]), dev(Udot)
    jxs().Solver.from_case(case).step_fixed_dt_tangent(Ut, Dt, 1.0, dt, 1)
    s2 = jxs().Solver.from_case(case)
    Ur, B = dev(case["U0"]), dev(Ubar)
    s2.step_fixed_dt_record(Ur, dt, 1)
    gbar = s2.adjoint_steps(B)
    return dict(case=case, dt=dt, Udot=Udot, Ubar=Ubar, U=U.cpu().numpy(), Ut=Ut.cpu().numpy(), Dt=Dt.cpu().numpy(),
                Ur=Ur.cpu().numpy(), B=B.cpu().numpy(), gbar=gbar)


def test_full_size_step_and_tangent_on_sampled_windows(big):
    case, dt = big["case"], big["dt"]
    sU, sD = scale(big["U"]), scale(big["Dt"])
    for c in centres():
        lo, hi = c - HALF, c + HALF
        w = wl.window(case, lo, hi)
        c2, o = oracle_rows(w)
        Uo, Do = o.step_fixed_dt_tangent(c2["U0"], rows(big["Udot"][:, :, lo:hi]), 1.0, dt, 1)
        a, b = (MARGIN if lo > 0 else 0), (2 * HALF - MARGIN if hi < NX else 2 * HALF)   # true ends are the tube's own
        sl = slice(lo + a, lo + b)
        assert (np.abs(big["U"][:, :, sl] - Uo[:, :1, a:b]) / sU).max() <= 1e-12, c
        assert (np.abs(big["Ut"][:, :, sl] - Uo[:, :1, a:b]) / sU).max() <= 1e-12, c
        assert (np.abs(big["Ur"][:, :, sl] - Uo[:, :1, a:b]) / sU).max() <= 1e-12, c
        assert (np.abs(big["Dt"][:, :, sl] - Do[:, :1, a:b]) / sD).max() <= 1e-12, c


def test_full_size_adjoint_on_sampled_windows(big):
    case, dt = big["case"], big["dt"]
    sB = scale(big["B"])
    for c in centres()[:8]:
        lo, hi = c - HALF, c + HALF
        w = wl.window(case, lo, hi)
        c2, o = oracle_rows(w)
        want, _ = o.step_fixed_dt_adjoint(c2["U0"], big["Ubar"][:, :, lo:hi], dt, 1, planar=True)
        # an entry of the adjoint collects the results within 9 cells of it, each of which feels an artificial end
        # within another 9 + 3 cells: twice the margin of the forward check
        m = 2 * MARGIN - 4
        a, b = (m if lo > 0 else 0), (2 * HALF - m if hi < NX else 2 * HALF)
        assert (np.abs(big["B"][:, :, lo + a:lo + b] - want[:, :, a:b]) / sB).max() <= 1e-11, c
    # gamma_bar is a sum over all cells: against the tangent kernel's pairing at this size
    lhs = float(np.sum(big["Ubar"] * big["Dt"]))
    rhs = float(np.sum(big["B"] * big["Udot"])) + big["gbar"] * 1.0
    assert lhs == pytest.approx(rhs, rel=1e-11)
