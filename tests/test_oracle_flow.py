"""Pins for the oracle's whole path (O1-O9): exact Riemann solution, free stream, conservation,
symmetry, boundary equivalences, RK3 amplification factor, viscous operator, brute force.
-m "not gpu"; sized so the file runs in about a minute.
"""
import math

import numpy as np
import pytest

import refs
from oracle import jxo
from paper_2601_04400_b200 import workloads as wl

G = 1.4
PER = dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic")
TRN = dict(xlo="transmissive", xhi="transmissive", ylo="transmissive", yhi="transmissive")


def make(case, **kw):
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], kw.pop("mu", case["mu"]),
                   case["Pr"], kw.pop("bc", case["bc"]), **kw)
    if case.get("phi") is not None:
        o.set_ibm(case["phi"])
    return o


def run_to(o, U, t_end, cfl=0.4):
    """Advance with the CFL rule and land exactly on t_end with one fixed-dt step."""
    while True:
        t, _ = o.time()
        smax = o.max_wavespeed(U)
        dt = cfl * min(o_dx(o)) / smax
        if t + dt >= t_end:
            return o.step_fixed_dt(U, t_end - t, 1)
        U = o.step(U, cfl, 1)


def o_dx(o):
    return o._dx


def smooth_periodic_field(n, m, seed=0, amp=0.2):
    rng = np.random.default_rng(seed)
    x = (np.arange(n) + 0.5) / n
    y = (np.arange(m) + 0.5) / m
    X, Y = np.meshgrid(x, y)

    def f():
        a, b, c, d = rng.uniform(-1, 1, 4)
        return amp * (a * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + b * np.cos(4 * np.pi * X + 1.0) +
                      c * np.sin(2 * np.pi * Y + 0.5) + d * np.sin(2 * np.pi * (X + Y)))

    return 1.0 + f(), 0.5 + f(), -0.3 + f(), 1.0 + f()


# ----------------------------------------------------------------- Sod vs exact
def _sod_l1(n, axis):
    case = wl.sod(n if axis == 0 else 8, 8 if axis == 0 else n, axis=axis)
    o = make(case)
    o._dx = (case["dx"], case["dy"])
    # keep the short direction from setting dt: it is uniform there, so only the long one matters
    o._dx = (1.0 / n, 1.0 / n)
    U = run_to(o, case["U0"], 0.2)
    assert o.guard_count() == 0
    s = (np.arange(n) + 0.5) / n
    r, u, p = refs.riemann_sample((s - 0.5) / 0.2, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, G)
    line = U[:, 4, :] if axis == 0 else U[:, :, 4]
    rho = line[0]
    vel = line[1 + axis] / rho
    return np.mean(np.abs(rho - r)), np.mean(np.abs(vel - u)), U


def test_sod_converges_to_the_exact_solution_along_x():
    """PAPER.md L134 (Eq. 17): 'the numerical solution converges toward the exact solution'."""
    e = [_sod_l1(n, 0)[0] for n in (64, 128, 256)]
    orders = [math.log2(e[i] / e[i + 1]) for i in range(2)]
    assert e[2] < 2.5e-3 and min(orders) > 0.7, (e, orders)


def test_sod_along_y_is_the_transpose_of_sod_along_x():
    ex, eux, Ux = _sod_l1(128, 0)
    ey, euy, Uy = _sod_l1(128, 1)
    assert ex == pytest.approx(ey, rel=1e-12)
    Ut = np.transpose(Uy, (0, 2, 1))[[0, 2, 1, 3]]
    assert np.max(np.abs(Ut - Ux)) < 1e-13
    assert np.max(np.abs(Ux[2])) == 0.0  # no transverse momentum is ever created


# ------------------------------------------------------- free stream, contacts
@pytest.mark.parametrize("bc", [PER, TRN])
def test_uniform_state_has_exactly_zero_rhs(bc):
    U = wl.cons_from_prim(np.full((12, 16), 1.3), np.full((12, 16), 0.7), np.full((12, 16), -0.4),
                          np.full((12, 16), 0.9))
    o = jxo.Oracle(16, 12, 0.1, 0.07, G, 1e-3, 0.72, bc)
    assert np.array_equal(o.rhs(U), np.zeros_like(U))


def test_moving_contact_keeps_velocity_and_pressure():
    n = 64
    x = (np.arange(n) + 0.5) / n
    rho = np.tile(1.0 + 0.5 * (np.abs(x - 0.5) < 0.2), (8, 1))
    U = wl.cons_from_prim(rho, np.full_like(rho, 0.8), np.full_like(rho, -0.3), np.full_like(rho, 1.0))
    o = jxo.Oracle(n, 8, 1.0 / n, 1.0 / n, G, 0.0, 0.72, PER)
    U1 = o.step(U, 0.4, 20)
    u, v = U1[1] / U1[0], U1[2] / U1[0]
    p = (G - 1) * (U1[3] - 0.5 * U1[0] * (u * u + v * v))
    assert np.max(np.abs(u - 0.8)) < 1e-13 and np.max(np.abs(v + 0.3)) < 1e-13 and np.max(np.abs(p - 1)) < 1e-13
    assert np.max(np.abs(U1[0] - U[0])) > 1e-2  # the density profile did move


# --------------------------------------------------------------- conservation
@pytest.mark.parametrize("mu", [0.0, 2e-2])
def test_periodic_rhs_sums_to_zero(mu):
    rho, u, v, p = smooth_periodic_field(24, 20, seed=1)
    U = wl.cons_from_prim(rho, u, v, p)
    o = jxo.Oracle(24, 20, 1.0 / 24, 1.0 / 20, G, mu, 0.72, PER)
    o.set_artificial_viscosity(1e-3 if mu else 0.0)
    L = o.rhs(U)
    for k in range(4):
        assert abs(L[k].sum()) < 1e-11 * np.abs(L[k]).sum(), k


def test_periodic_steps_conserve_mass_momentum_energy():
    case = wl.vortex(32)
    o = make(case)
    U = o.step(case["U0"], 0.4, 10)
    for k in range(4):
        assert abs(U[k].sum() - case["U0"][k].sum()) < 1e-12 * np.abs(case["U0"][k]).sum()


# ------------------------------------------------------------------- symmetry
def test_periodic_shift_invariance_is_bitwise():
    rho, u, v, p = smooth_periodic_field(16, 16, seed=2)
    U = wl.cons_from_prim(rho, u, v, p)
    o = jxo.Oracle(16, 16, 1.0 / 16, 1.0 / 16, G, 1e-2, 0.72, PER)
    L = o.rhs(U)
    Ls = o.rhs(np.roll(U, (3, -5), axis=(1, 2)))
    assert np.array_equal(Ls, np.roll(L, (3, -5), axis=(1, 2)))


def test_xy_transposition_invariance():
    rho, u, v, p = smooth_periodic_field(16, 12, seed=3)
    U = wl.cons_from_prim(rho, u, v, p)
    o = jxo.Oracle(16, 12, 1.0 / 16, 1.0 / 12, G, 1e-2, 0.72, PER)
    L = o.rhs(U)
    Ut = np.ascontiguousarray(np.transpose(U, (0, 2, 1))[[0, 2, 1, 3]])
    ot = jxo.Oracle(12, 16, 1.0 / 12, 1.0 / 16, G, 1e-2, 0.72, PER)
    Lt = np.transpose(ot.rhs(Ut), (0, 2, 1))[[0, 2, 1, 3]]
    assert np.max(np.abs(Lt - L)) < 1e-12 * np.max(np.abs(L))


def test_mirror_symmetry_in_x():
    rho, u, v, p = smooth_periodic_field(16, 12, seed=4)
    U = wl.cons_from_prim(rho, u, v, p)
    o = jxo.Oracle(16, 12, 1.0 / 16, 1.0 / 12, G, 1e-2, 0.72, PER)
    L = o.rhs(U)
    Um = np.ascontiguousarray(U[:, :, ::-1] * np.array([1, -1, 1, 1])[:, None, None])
    Lm = o.rhs(Um)[:, :, ::-1] * np.array([1, -1, 1, 1])[:, None, None]
    assert np.max(np.abs(Lm - L)) < 1e-12 * np.max(np.abs(L))


# ------------------------------------------------------------------------ BCs
def test_ghost_frame_values():
    """O1 checked cell by cell against the rule written with numpy indexing (reading R11)."""
    rng = np.random.default_rng(9)
    nx, ny = 10, 9
    U = wl.cons_from_prim(rng.uniform(1, 2, (ny, nx)), rng.uniform(-1, 1, (ny, nx)),
                          rng.uniform(-1, 1, (ny, nx)), rng.uniform(1, 2, (ny, nx)))
    inflow = (1.7, 0.9, -0.2, 2.1)
    bc = dict(xlo="inflow", xhi="transmissive", ylo="reflective", yhi="periodic", inflow=inflow)
    with pytest.raises(jxo.OracleError):
        jxo.Oracle(nx, ny, 1, 1, G, 0, 0.72, bc)  # periodic on one side only
    bc["yhi"] = "reflective"
    Up = jxo.Oracle(nx, ny, 1, 1, G, 0, 0.72, bc).fill_ghosts(U)
    assert np.array_equal(Up[:, 3:-3, 3:-3], U)
    Uin = wl.cons_from_prim(*[np.array(x) for x in inflow])
    for g in (1, 2, 3):
        assert np.array_equal(Up[:, 3:-3, 3 - g], np.tile(Uin[:, None], (1, ny)))  # inflow
        assert np.array_equal(Up[:, 3:-3, nx + 2 + g], U[:, :, nx - 1])  # transmissive
        flip = np.array([1, 1, -1, 1])[:, None]
        assert np.array_equal(Up[:, 3 - g, 3:-3], U[:, g - 1, :] * flip)  # reflective bottom
        assert np.array_equal(Up[:, ny + 2 + g, 3:-3], U[:, ny - g, :] * flip)  # reflective top
        # corners: y-fill of the x-ghost columns
        assert np.array_equal(Up[:, 3 - g, 0], Uin * flip[:, 0])
        assert np.array_equal(Up[:, ny + 2 + g, nx + 5], U[:, ny - g, nx - 1] * flip[:, 0])
    per = jxo.Oracle(nx, ny, 1, 1, G, 0, 0.72, PER).fill_ghosts(U)
    assert np.array_equal(per, np.pad(U, ((0, 0), (3, 3), (3, 3)), mode="wrap"))


def test_reflective_wall_equals_mirrored_doubled_domain():
    n = 24
    rho, u, v, p = smooth_periodic_field(n, 10, seed=5)
    U = wl.cons_from_prim(rho, u, v, p)
    bc = dict(xlo="transmissive", xhi="reflective", ylo="periodic", yhi="periodic")
    a = jxo.Oracle(n, 10, 0.05, 0.05, G, 1e-2, 0.72, bc).step_fixed_dt(U, 2e-3, 2)
    Ud = np.concatenate([U, U[:, :, ::-1] * np.array([1, -1, 1, 1])[:, None, None]], axis=2)
    bcd = dict(xlo="transmissive", xhi="transmissive", ylo="periodic", yhi="periodic")
    b = jxo.Oracle(2 * n, 10, 0.05, 0.05, G, 1e-2, 0.72, bcd).step_fixed_dt(Ud, 2e-3, 2)
    assert np.max(np.abs(b[:, :, :n] - a)) < 1e-13


# ------------------------------------------------------------ RK3 and Eq. 10
def test_rk3_amplification_factor_on_the_discrete_heat_equation():
    """u = 0, p uniform, rho = 1 + A sin(kx): the Euler flux is the exact stationary contact, so
    d rho/dt = nu Lap_h rho (Eq. 10's artificial-viscosity term) and one SSP-RK3 step multiplies
    the mode by 1 + z + z^2/2 + z^3/6, z = -nu dt (4/dx^2) sin^2(k dx/2)."""
    n, A, nu, dt = 32, 0.1, 0.02, 3e-3
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    rho = np.tile(1.0 + A * np.sin(2 * np.pi * x), (8, 1))
    z0 = np.zeros_like(rho)
    U = wl.cons_from_prim(rho, z0, z0, np.ones_like(rho))
    o = jxo.Oracle(n, 8, dx, dx, G, 0.0, 0.72, PER)
    o.set_artificial_viscosity(nu)
    U1 = o.step_fixed_dt(U, dt, 1)
    z = -nu * dt * 4.0 / dx ** 2 * math.sin(math.pi * dx) ** 2
    amp = 1 + z + z * z / 2 + z ** 3 / 6
    assert np.max(np.abs((U1[0] - 1.0) - amp * (rho - 1.0))) < 1e-15
    assert abs(amp - (1 + z + z * z / 2)) > 1e-9  # the cubic term is resolved by the tolerance
    assert np.array_equal(U1[1], z0) and np.max(np.abs(U1[3] - U[3])) < 1e-15
    assert o.time() == (dt, dt)


def test_cfl_time_step_rule():
    case = wl.sod(32, 8)
    o = make(case)
    o.step(case["U0"], 0.4, 1)
    smax = math.sqrt(G * 1.0 / 1.0)  # the left state at rest is the fastest: a = sqrt(gamma p / rho)
    assert o.max_wavespeed(case["U0"]) == pytest.approx(smax, rel=1e-15)
    assert o.time()[1] == pytest.approx(0.4 * min(case["dx"], case["dy"]) / smax, rel=1e-15)


def _uniform_with(n, m, base, cells):
    """Conserved field, uniform primitive state `base` except the listed (i, j) -> (rho, u, v, p)."""
    W = np.empty((4, m, n))
    for k in range(4):
        W[k] = base[k]
    for (i, j), w in cells.items():
        W[:, j, i] = w
    return wl.cons_from_prim(W[0], W[1], W[2], W[3])


def test_max_wavespeed_closed_form_on_moving_states():
    """O9 / R6: s_max = max over fluid cells of max(|u| + a, |v| + a), a = sqrt(gamma p / rho).  Hand-built states in
    which the maximum is taken (a) by a cell moving in -x (|u| matters, not u), (b) by the v-branch, (c) by a slow cell
    with a large sound speed; each number is written out with math.sqrt here.  A rule that drops the absolute value,
    ignores v, or uses |u| + |v| + a or sqrt(u^2 + v^2) + a gives another value in at least one of them."""
    n, m = 12, 10
    base = (1.0, 0.1, -0.2, 1.0)
    a0 = math.sqrt(G * 1.0 / 1.0)
    o = jxo.Oracle(n, m, 0.1, 0.1, G, 0.0, 0.72, TRN)
    # uniform: the v-branch wins (|v| = 0.2 > |u| = 0.1)
    assert o.max_wavespeed(_uniform_with(n, m, base, {})) == pytest.approx(0.2 + a0, rel=1e-15)
    # (a) one cell with u = -3 (and v = +1: |u| + a, not |u| + |v| + a, not hypot(u, v) + a)
    fast = (2.0, -3.0, 1.0, 0.5)
    a = math.sqrt(G * 0.5 / 2.0)
    got = o.max_wavespeed(_uniform_with(n, m, base, {(4, 7): fast}))
    assert got == pytest.approx(3.0 + a, rel=1e-15)
    assert abs(got - (4.0 + a)) > 0.5 and abs(got - (math.hypot(3.0, 1.0) + a)) > 0.1 and abs(got - (1.0 + a)) > 1.0
    # (b) the v-branch with a negative v, at the last cell of the grid (loop bounds)
    fastv = (0.5, 0.3, -2.5, 2.0)
    av = math.sqrt(G * 2.0 / 0.5)
    assert o.max_wavespeed(_uniform_with(n, m, base, {(n - 1, m - 1): fastv})) == pytest.approx(2.5 + av, rel=1e-15)
    # (c) a cell at rest with the largest sound speed, at the first cell
    hot = (0.1, 0.0, 0.0, 10.0)
    assert o.max_wavespeed(_uniform_with(n, m, base, {(0, 0): hot})) == pytest.approx(math.sqrt(G * 10.0 / 0.1), rel=1e-15)
    # gamma enters through E -> p and through a: the same primitives with gamma = 1.67
    o2 = jxo.Oracle(n, m, 0.1, 0.1, 1.67, 0.0, 0.72, TRN)
    full = tuple(np.full((m, n), w) for w in fast)
    U2 = wl.cons_from_prim(*full, gamma=1.67)
    assert o2.max_wavespeed(U2) == pytest.approx(3.0 + math.sqrt(1.67 * 0.5 / 2.0), rel=1e-15)


def test_max_wavespeed_ignores_cells_inside_a_body():
    """O9: "fluid interior cells": the fastest cell placed inside the body (solid), and in its
    ghost layer, must not count; the same cell outside the body does."""
    n, m = 48, 40
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    y = (np.arange(m) + 0.5) * dx
    X, Y = np.meshgrid(x, y)
    phi = np.hypot(X - 0.5, Y - 20.5 * dx) - 6.0 * dx
    o = jxo.Oracle(n, m, dx, dx, G, 0.0, 0.72, TRN)
    o.set_ibm(phi)
    types = o.cell_types()
    base = (1.0, 0.4, 0.0, 1.0)
    a0 = math.sqrt(G)
    fast = (1.0, -5.0, 0.5, 4.0)
    af = math.sqrt(G * 4.0)
    centre = (24, 20)                                   # deep inside: solid
    assert types[centre[1], centre[0]] != 0 and phi[centre[1], centre[0]] < -3 * dx
    gj, gi = [(j, i) for j in range(m) for i in range(n) if types[j, i] != 0 and phi[j, i] > -1.2 * dx][0]
    assert types[gj, gi] != 0                           # a non-fluid cell next to the surface: ghost
    fj, fi = 20, 40                                     # far outside: fluid
    assert types[fj, fi] == 0
    assert o.max_wavespeed(_uniform_with(n, m, base, {})) == pytest.approx(0.4 + a0, rel=1e-15)
    assert o.max_wavespeed(_uniform_with(n, m, base, {centre: fast})) == pytest.approx(0.4 + a0, rel=1e-15)
    assert o.max_wavespeed(_uniform_with(n, m, base, {(gi, gj): fast})) == pytest.approx(0.4 + a0, rel=1e-15)
    assert o.max_wavespeed(_uniform_with(n, m, base, {(fi, fj): fast})) == pytest.approx(5.0 + af, rel=1e-15)
    # without the body the same cell counts
    o.set_ibm(None)
    assert o.max_wavespeed(_uniform_with(n, m, base, {centre: fast})) == pytest.approx(5.0 + af, rel=1e-15)


@pytest.mark.parametrize("dx,dy", [(0.05, 0.02), (0.01, 0.04)])
def test_cfl_time_step_uses_the_smaller_spacing(dx, dy):
    """R6: dt = cfl min(dx, dy) / s_max, with dx != dy either way round, on a moving state."""
    n, m = 16, 12
    U = _uniform_with(n, m, (1.0, -0.7, 0.3, 1.0), {(5, 5): (1.5, 0.2, 2.0, 3.0)})
    smax = max(0.7 + math.sqrt(G), 2.0 + math.sqrt(G * 3.0 / 1.5))
    o = jxo.Oracle(n, m, dx, dy, G, 0.0, 0.72, PER)
    assert o.max_wavespeed(U) == pytest.approx(smax, rel=1e-15)
    o.step(U, 0.3, 1)
    t, dt = o.time()
    assert dt == pytest.approx(0.3 * min(dx, dy) / smax, rel=1e-15) and t == dt


def test_operation_tally_of_the_literal_evaluation():
    """The counting scalar (jxo_count_ops): operations of ONE literal evaluation of L(U), one general RK combine and
    one wavespeed pass on the 512x256 throughput case, per interior cell.  These are the figures DESIGN.md section 6
    quotes next to the minimal-work count the roofline uses (the oracle shares nothing between faces and evaluates both
    HLLC sides, so its count is the larger one)."""
    case = wl.throughput_case(512, 256)
    o = make(case)
    c = o.count_ops(case["U0"])
    n = 512 * 256
    per = {k: v / n for k, v in c.items()}
    # literal WENO5 (two sides x 4 variables x 2 directions), both-sided HLLC at every face, viscous fluxes, divergence,
    # combine, wavespeed; the face counts exceed the cell count by the boundary faces, hence the tolerances
    assert 660 < per["add"] < 670 and 686 < per["mul"] < 696, per
    assert 206 < per["div"] < 212 and 4.9 < per["sqrt"] < 5.1, per
    total = per["add"] + per["mul"] + per["div"] + per["sqrt"]
    assert 1560 < total < 1580, total


def test_float_oracle_agrees_with_the_double_oracle():
    """The float instantiation of the oracle (JXO_F32): a uniform state gives L == 0 exactly (identical arithmetic at
    every face), and on the smooth vortex its RHS is within float round-off of the double oracle's."""
    n = 32
    U = _uniform_with(n, n, (1.0, 0.5, -0.25, 2.0), {})
    o32 = jxo.Oracle(n, n, 0.1, 0.1, G, 0.0, 0.72, PER, dtype=np.float32)
    L = o32.rhs(U.astype(np.float32))
    assert L.dtype == np.float32 and np.array_equal(L, np.zeros_like(L))
    case = wl.vortex(64)
    Ld = make(case).rhs(case["U0"])
    Lf = make(case, dtype=np.float32).rhs(case["U0"].astype(np.float32))
    for k in range(4):
        assert np.max(np.abs(Lf[k] - Ld[k])) <= 1e-5 * np.max(np.abs(Ld[k])) + 1e-5, k
    sd = make(case).max_wavespeed(case["U0"])
    sf = make(case, dtype=np.float32).max_wavespeed(case["U0"].astype(np.float32))
    assert abs(sf - sd) <= 1e-6 * sd


# -------------------------------------------------------------------- viscous
def _viscous_part(n, mu=0.05, Pr=0.72):
    rho, u, v, p = smooth_periodic_field(n, n, seed=6)
    U = wl.cons_from_prim(rho, u, v, p)
    a = jxo.Oracle(n, n, 1.0 / n, 1.0 / n, G, mu, Pr, PER).rhs(U)
    b = jxo.Oracle(n, n, 1.0 / n, 1.0 / n, G, 0.0, Pr, PER).rhs(U)
    exact = refs.viscous_operator_spectral(rho, u, v, p, 1.0, 1.0, mu, Pr, G)
    return a - b, exact


def test_viscous_terms_converge_at_second_order_to_navier_stokes():
    """P:L9 names Navier-Stokes; the discretisation is reading R8.  The analytic operator (Stokes
    hypothesis, T = p/rho, k = mu gamma/((gamma-1) Pr)) is evaluated by FFT differentiation."""
    errs = []
    for n in (32, 64, 128):
        d, e = _viscous_part(n)
        assert np.array_equal(d[0], np.zeros_like(d[0]))
        errs.append([np.max(np.abs(d[k] - e[k])) / np.max(np.abs(e[k])) for k in (1, 2, 3)])
    errs = np.array(errs)
    orders = np.log2(errs[:-1] / errs[1:])
    assert errs[-1].max() < 2e-3 and orders.min() > 1.9, (errs, orders)


def test_pure_shear_closed_form():
    n, mu, k = 32, 0.03, 2 * np.pi
    dy = 1.0 / n
    y = (np.arange(n) + 0.5) * dy
    u = np.tile(0.2 * np.sin(k * y)[:, None], (1, 8))
    one = np.ones_like(u)
    U = wl.cons_from_prim(one, u, 0 * u, one)
    L = jxo.Oracle(8, n, dy, dy, G, mu, 0.72, PER).rhs(U)
    lam = -(4.0 / dy ** 2) * math.sin(0.5 * k * dy) ** 2
    assert np.max(np.abs(L[1] - mu * lam * u)) < 1e-13
    assert np.array_equal(L[0], 0 * u) and np.max(np.abs(L[2])) < 1e-15


# ---------------------------------------------------------------- brute force
@pytest.mark.parametrize("bc", [
    PER,
    dict(xlo="inflow", xhi="transmissive", ylo="reflective", yhi="reflective", inflow=(1.2, 0.6, 0.1, 1.1)),
    dict(xlo="reflective", xhi="reflective", ylo="transmissive", yhi="transmissive"),
])
def test_bruteforce_per_cell_evaluator_on_16x16(bc):
    """A stand-alone evaluator (definition-based WENO, Toro-form HLLC, index-mapped boundaries, no
    shared arrays) must agree with the sweep-based oracle at every cell."""
    rng = np.random.default_rng(12)
    n = 16
    rho, u, v, p = smooth_periodic_field(n, n, seed=8, amp=0.15)
    # add a jump so that the nonlinear weights and all HLLC branches are exercised
    rho[:, 9:] *= 0.4
    p[:, 9:] *= 0.3
    u[5:11, :] += 1.5 * rng.uniform(-1, 1)
    U = wl.cons_from_prim(rho, u, v, p)
    dx, dy = 1.0 / n, 0.8 / n
    L = jxo.Oracle(n, n, dx, dy, G, 0.0, 0.72, bc).rhs(U)
    scale = np.max(np.abs(L), axis=(1, 2))
    for j in range(n):
        for i in range(n):
            ref = refs.rhs_cell_bruteforce(U, i, j, dx, dy, bc, G)
            assert np.all(np.abs(ref - L[:, j, i]) <= 2e-11 * scale), (i, j, ref, L[:, j, i])


# ------------------------------------------------------------ planar shock speed
def test_planar_shock_advances_at_mach_times_sound_speed():
    """An undisturbed planar shock of the Eq. 18 family moves at M_s a_1 (here M_s = 2)."""
    case = wl.shock_cylinder(256, 8, Ms=2.0, bodies=(), x_shock=0.2, viscous=False)
    case["dy"] = case["dx"]
    o = make(case)
    o._dx = (case["dx"], case["dx"])
    U = run_to(o, case["U0"], 0.3)
    rho = U[0, 4]
    x = (np.arange(256) + 0.5) * case["dx"]
    mid = 0.5 * (rho.max() + 1.4)
    xs = x[np.argmax(rho < mid)]
    assert abs(xs - (0.2 + 2.0 * 1.0 * 0.3)) < 2.5 * case["dx"]  # a_1 = sqrt(1.4*1/1.4) = 1


# ------------------------------------------------------------ isentropic vortex
def test_isentropic_vortex_returns_after_one_period():
    errs = []
    for n in (24, 48):
        case = wl.vortex(n)
        o = make(case)
        o._dx = (case["dx"], case["dy"])
        U = run_to(o, case["U0"], 10.0)
        errs.append(np.mean(np.abs(U[0] - case["U0"][0])))
    order = math.log2(errs[0] / errs[1])
    assert errs[1] < 5e-3 and order > 2.0, (errs, order)
