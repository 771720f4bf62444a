"""GPU-versus-oracle parity, element by element, through the C ABI (include/jxs.h).  -m gpu.

Tolerances are BASELINE.json's: fp64 single RHS <= 1e-12 max-norm relative (per field, scaled by
that field's max, fluid cells only), 100 steps of the 128x128 Sod case <= 1e-9; fp32 <= 1e-4 / 1e-3.
"""
import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_RHS64, TOL_STEP64, TOL_RHS32, TOL_STEP32 = 1e-12, 1e-9, 1e-4, 1e-3
G = 1.4
PER = dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic")


def jxs():
    from paper_2601_04400_b200 import jxs as m
    return m


def make_pair(case, dtype=torch.float64, nu=0.0):
    npdt = np.float64 if dtype == torch.float64 else np.float32
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"],
                   dtype=npdt)
    s = jxs().Solver.from_case(case, dtype=dtype)
    if case.get("phi") is not None:
        o.set_ibm(case["phi"])
    if nu:
        o.set_artificial_viscosity(nu)
        s.set_artificial_viscosity(nu)
    return o, s


def dev(U, dtype=torch.float64):
    return torch.tensor(np.ascontiguousarray(U), dtype=dtype, device="cuda")


def rel_err(a, b, fluid=None, zero_tol=1e-6):
    """max-norm error per field, scaled by THAT field's max over the compared cells (BASELINE.json north_star).
    Only a momentum component that is analytically zero in the case at hand — rho*v while a planar x-shock has not
    reached a body, rho*u in the transposed problem — has no scale of its own: what it holds is amplified round-off
    (below zero_tol of the other component; 1e-6 in fp64, where WENO's weights amplify 1e-16 differences), and it
    borrows the other momentum's scale."""
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    m = np.ones(a.shape[1:], bool) if fluid is None else fluid
    peak = [np.max(np.abs(b[k][m])) for k in range(4)]
    mom = max(peak[1], peak[2])
    scale = [peak[0], peak[1] if peak[1] > zero_tol * mom else mom, peak[2] if peak[2] > zero_tol * mom else mom, peak[3]]
    return max(np.max(np.abs(a[k][m] - b[k][m])) / max(scale[k], 1e-300) for k in range(4))


def smooth_case(nx, ny, seed, bc=PER, mu=0.0, amp=0.2, jump=False):
    rng = np.random.default_rng(seed)
    x, y = (np.arange(nx) + 0.5) / nx, (np.arange(ny) + 0.5) / ny
    X, Y = np.meshgrid(x, y)

    def f():
        a, b, c, d = rng.uniform(-1, 1, 4)
        return amp * (a * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + b * np.cos(4 * np.pi * X + 1.0) +
                      c * np.sin(2 * np.pi * Y + 0.5) + d * np.sin(2 * np.pi * (X + Y)))

    rho, u, v, p = 1.0 + f(), 0.5 + f(), -0.3 + f(), 1.0 + f()
    if jump:
        rho = np.where((X - 0.4) ** 2 + (Y - 0.6) ** 2 < 0.05, 2.5 * rho, rho)
        p = np.where(X + 0.3 * Y > 0.9, 0.3 * p, p)
        u = np.where(Y > 0.7, u - 1.2, u)
    return dict(name="smooth", U0=wl.cons_from_prim(rho, u, v, p), nx=nx, ny=ny, dx=1.0 / nx, dy=0.8 / ny, gamma=G,
                mu=mu, Pr=0.72, bc=bc, phi=None)


MIXED = dict(xlo="inflow", xhi="transmissive", ylo="reflective", yhi="reflective", inflow=(1.2, 0.6, 0.1, 1.1))
WALLS = dict(xlo="reflective", xhi="reflective", ylo="transmissive", yhi="periodic")
WALLS["ylo"] = "periodic"

RHS_CASES = {
    "sod_x_128": lambda: wl.sod(128, 128, 0),
    "sod_y_128": lambda: wl.sod(128, 128, 1),
    "vortex_64": lambda: wl.vortex(64),
    "vortex_gauss_96": lambda: wl.vortex(96, quadrature=3),
    "jumps_periodic_euler_130x67": lambda: smooth_case(130, 67, 1, jump=True),          # ragged: 3 strips, odd sizes
    "jumps_mixed_bc_viscous_200x50": lambda: smooth_case(200, 50, 2, MIXED, mu=5e-3, jump=True),
    "jumps_walls_viscous_63x190": lambda: smooth_case(63, 190, 3, WALLS, mu=2e-2, jump=True),
    "minimum_8x8": lambda: smooth_case(8, 8, 4, mu=1e-2),
    "one_strip_62x9": lambda: smooth_case(62, 9, 5, MIXED),
    "strip_edge_124x11": lambda: smooth_case(124, 11, 6, WALLS, mu=1e-3),
    "shock_cylinder_256x128_ns": lambda: wl.shock_cylinder(256, 128, Ms=2.0),
    "shock_cylinders_euler_384x192": lambda: wl.throughput_case(384, 192, viscous=False),
}


@pytest.mark.parametrize("name", list(RHS_CASES))
def test_rhs_parity_fp64(name):
    case = RHS_CASES[name]()
    o, s = make_pair(case)
    ref = o.rhs(case["U0"])
    got = s.rhs(dev(case["U0"])).cpu().numpy()
    fluid = o.cell_types() == 0
    assert np.all(got[:, ~fluid] == 0.0)
    err = rel_err(got, ref, fluid)
    assert err <= TOL_RHS64, (name, err)
    assert o.guard_count() == 0


def test_rhs_parity_with_artificial_viscosity():
    case = smooth_case(100, 40, 7, MIXED, mu=1e-3, jump=True)
    o, s = make_pair(case, nu=2e-3)
    err = rel_err(s.rhs(dev(case["U0"])).cpu().numpy(), o.rhs(case["U0"]))
    assert err <= TOL_RHS64, err


def test_rhs_after_evolution_shock_cylinder():
    """RHS parity on a developed field (reflected shock on the cylinder), not just initial data."""
    case = wl.shock_cylinder(256, 128, Ms=2.0)
    o, s = make_pair(case)
    U = o.step(case["U0"], 0.4, 60)
    fluid = o.cell_types() == 0
    err = rel_err(s.rhs(dev(U)).cpu().numpy(), o.rhs(U), fluid)
    assert err <= TOL_RHS64, err
    assert o.guard_count() == 0


def test_max_wavespeed_parity():
    for case in (wl.sod(128, 128), wl.shock_cylinder(256, 128, Ms=2.0), wl.vortex(64)):
        o, s = make_pair(case)
        a, b = s.max_wavespeed(dev(case["U0"])), o.max_wavespeed(case["U0"])
        assert abs(a - b) <= 1e-14 * b


def test_sod_128_100_steps_fp64():
    """BASELINE.json configs[0]: 128x128 Sod, CFL 0.4, 100 steps, <= 1e-9."""
    case = wl.sod(128, 128)
    o, s = make_pair(case)
    ref = o.step(case["U0"], 0.4, 100)
    U = dev(case["U0"])
    s.step(U, 0.4, 100)
    err = rel_err(U.cpu().numpy(), ref)
    assert err <= TOL_STEP64, err
    (t_o, dt_o), (t_s, dt_s) = o.time(), s.time()
    assert abs(t_o - t_s) <= 1e-12 * t_o and abs(dt_o - dt_s) <= 1e-12 * dt_o
    assert o.guard_count() == 0


@pytest.mark.parametrize("name,nsteps", [("shock_cylinder_256x128_ns", 40), ("jumps_mixed_bc_viscous_200x50", 30),
                                         ("vortex_64", 50)])
def test_steps_parity_fp64(name, nsteps):
    case = RHS_CASES[name]()
    o, s = make_pair(case)
    ref = o.step(case["U0"], 0.4, nsteps)
    U = dev(case["U0"])
    s.step(U, 0.4, nsteps)
    fluid = o.cell_types() == 0
    err = rel_err(U.cpu().numpy(), ref, fluid)
    assert err <= TOL_STEP64, (name, err)
    assert abs(o.time()[0] - s.time()[0]) <= 1e-12 * o.time()[0]


def test_fixed_dt_and_zero_steps():
    case = wl.vortex(64)
    o, s = make_pair(case)
    U = dev(case["U0"])
    s.step(U, 0.4, 0)
    assert np.array_equal(U.cpu().numpy(), case["U0"])
    s.step_fixed_dt(U, 5e-3, 7)
    ref = o.step_fixed_dt(case["U0"], 5e-3, 7)
    assert rel_err(U.cpu().numpy(), ref) <= TOL_STEP64
    assert s.time() == pytest.approx((7 * 5e-3, 5e-3), rel=1e-14)


def test_host_entry_points_match_device_ones():
    case = wl.shock_cylinder(256, 128, Ms=2.0)
    _, s = make_pair(case)
    Uh = torch.tensor(case["U0"]).pin_memory()
    Ud = dev(case["U0"])
    assert torch.equal(s.rhs_host(Uh), s.rhs(Ud).cpu())
    s.step_host(Uh, 0.4, 5)
    _, s2 = make_pair(case)
    s2.step(Ud, 0.4, 5)
    assert torch.equal(Uh, Ud.cpu())


# ----------------------------------------------------------------------------- fp32
@pytest.mark.parametrize("name", ["sod_x_128", "vortex_64", "jumps_mixed_bc_viscous_200x50", "shock_cylinder_256x128_ns"])
def test_rhs_parity_fp32(name):
    case = RHS_CASES[name]()
    o64, _ = make_pair(case)
    o32, s = make_pair(case, dtype=torch.float32)
    got = s.rhs(dev(case["U0"], torch.float32)).cpu().numpy()
    fluid = o64.cell_types() == 0
    # (in fp32 the round-off that fills an analytically zero momentum sits at 1e-6 of the other one)
    assert rel_err(got, o64.rhs(case["U0"]), fluid, zero_tol=1e-4) <= TOL_RHS32
    assert rel_err(got, o32.rhs(case["U0"]), fluid, zero_tol=1e-4) <= TOL_RHS32


def test_sod_128_100_steps_fp32():
    case = wl.sod(128, 128)
    o64, _ = make_pair(case)
    _, s = make_pair(case, dtype=torch.float32)
    U = dev(case["U0"], torch.float32)
    s.step(U, 0.4, 100)
    assert rel_err(U.cpu().numpy(), o64.step(case["U0"], 0.4, 100)) <= TOL_STEP32


# ------------------------------------------------------------- properties on the GPU itself
def test_gpu_periodic_conservation_and_free_stream():
    case = smooth_case(130, 67, 11, mu=1e-2, jump=True)
    _, s = make_pair(case)
    L = s.rhs(dev(case["U0"])).cpu().numpy()
    for k in range(4):
        assert abs(L[k].sum()) <= 1e-11 * np.abs(L[k]).sum()
    one = np.ones((67, 130))
    U = wl.cons_from_prim(1.3 * one, 0.7 * one, -0.4 * one, 0.9 * one)
    assert float(s.rhs(dev(U)).abs().max()) == 0.0


def test_gpu_error_paths():
    m = jxs()
    case = wl.shock_cylinder(256, 128, Ms=2.0)
    s = m.Solver.from_case(case)
    with pytest.raises(m.JxsError) as e:
        s.set_ibm(wl.cylinders_phi(256, 128, case["dx"], case["dy"], [(0.05, 0.5, 0.04)]))
    assert e.value.code == m.EINVAL and s.ibm_ghost_count() == 0
    U = dev(case["U0"])
    with pytest.raises(m.JxsError) as e:
        s.step(U, -1.0, 1)
    assert e.value.code == m.EINVAL
    bad = U.clone()
    bad[3] = -1.0  # negative energy -> NaN sound speed
    with pytest.raises(m.JxsError) as e:
        s.step(bad, 0.4, 2)
    assert e.value.code == m.ENUMERIC
    s.step(U, 0.4, 1)  # the handle stays usable


# ------------------------------------------------------------- full size, bench configuration
@pytest.mark.parametrize("dtype,tol", [(torch.float64, TOL_RHS64), (torch.float32, TOL_RHS32)])
def test_full_size_throughput_case_rhs(dtype, tol):
    """BASELINE.json configs[3] at 4096x2048 in the launch configuration bench.py times: the whole RHS
    against the oracle, element by element (the oracle needs a few seconds per evaluation)."""
    case = wl.throughput_case()
    o, s = make_pair(case)  # fp64 oracle is the truth for both
    if dtype == torch.float32:
        s = jxs().Solver.from_case(case, dtype=dtype)
    ref = o.rhs(case["U0"])
    got = s.rhs(dev(case["U0"], dtype)).cpu().numpy()
    fluid = o.cell_types() == 0
    assert s.ibm_ghost_count() == len(o.ibm_ghosts()[0]) > 5000
    assert rel_err(got, ref, fluid) <= tol
    assert o.guard_count() == 0


def test_full_size_throughput_case_two_steps():
    case = wl.throughput_case()
    o, s = make_pair(case)
    ref = o.step(case["U0"], 0.4, 2)
    U = dev(case["U0"])
    s.step(U, 0.4, 2)
    fluid = o.cell_types() == 0
    assert rel_err(U.cpu().numpy(), ref, fluid) <= TOL_STEP64
    assert abs(o.time()[0] - s.time()[0]) <= 1e-12 * o.time()[0]


def test_gpu_mirror_symmetry_of_the_shock_cylinder_case():
    """C3 is mirror-symmetric about y = 0.5 (rho, rho u, E even, rho v odd): PAPER.md L162 ("arise symmetrically");
    the CUDA path keeps it to round-off over a short run although it sweeps the rows upwards"""
    case = wl.shock_cylinder(512, 256, Ms=2.0)
    s = jxs().Solver.from_case(case)
    U = dev(case["U0"])
    s.step(U, 0.4, 60)
    u = U.cpu().numpy()
    scale = [np.abs(u[k]).max() for k in range(4)]
    for k, sign in ((0, 1.0), (1, 1.0), (2, -1.0), (3, 1.0)):
        assert np.abs(u[k] - sign * u[k][::-1, :]).max() <= 1e-10 * max(scale[k], scale[1])
