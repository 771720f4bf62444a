"""Pins for the oracle's tangent (O12, R21/R22): the forward-mode derivative of the fixed-dt step, i.e. the
Jacobian products of PAPER.md Eq. 16 applied to one direction, and the gamma inference of L149 / Fig. 3(b).

What fixes the answer independently of the Dual arithmetic under test:
  * the definition of a derivative: central differences of the (already pinned) primal oracle and of the
    independent definitions in refs.py (WENO5 from its polynomials, Toro's HLLC);
  * closed forms: the fifth-order upwind coefficients for constant data, the Euler flux Jacobian for equal /
    supersonic states, dF/dgamma = (0, 0, 0, -u p/(gamma-1)^2);
  * invariants: linearity in the direction, conservation of the tangent, d/dgamma of the first moment of rho = 0;
  * the exact Riemann solution's dependence on gamma (refs.riemann_sample);
  * the inference itself: Gauss-Newton on gamma recovers the value the data were made with.
-m "not gpu".
"""
import numpy as np
import pytest

import refs
from oracle import jxo
from paper_2601_04400_b200 import workloads as wl

G = 1.4


def make(case, gamma=None, **kw):
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"] if gamma is None else gamma,
                   kw.pop("mu", case["mu"]), case["Pr"], kw.pop("bc", case["bc"]), **kw)
    if case.get("phi") is not None:
        o.set_ibm(case["phi"])
    return o


def rel(a, b):
    """max-norm difference per component, relative to that component's max."""
    a, b = np.asarray(a), np.asarray(b)
    return max(np.abs(a[k] - b[k]).max() / max(np.abs(b[k]).max(), 1e-300) for k in range(a.shape[0]))


# --------------------------------------------------------------------------- pointwise
def test_weno5_tangent_constant_data_gives_upwind5_coefficients():
    # beta_k = 0 and d(beta_k) = 0 at constant data: the weights are the linear ones and do not move, so the
    # derivative is the fifth-order upwind interpolation (2, -13, 47, 27, -3)/60 of the direction
    rng = np.random.default_rng(0)
    for c in (0.0, 1.0, -3.5):
        d = rng.normal(size=5)
        val, der = jxo.weno5_tangent(np.full(5, c), d)
        assert val == pytest.approx(c, abs=1e-15)
        assert der == pytest.approx(np.dot([2, -13, 47, 27, -3], d) / 60.0, rel=1e-13, abs=1e-14)


def test_weno5_tangent_matches_central_difference_of_the_definition():
    rng = np.random.default_rng(1)
    for trial in range(20):
        v = rng.normal(size=5) * (0.1 if trial % 2 else 1.0) + (trial % 3)
        d = rng.normal(size=5)
        h = 1e-6
        fd = (refs.weno5_definition(v + h * d) - refs.weno5_definition(v - h * d)) / (2 * h)
        val, der = jxo.weno5_tangent(v, d)
        assert val == pytest.approx(refs.weno5_definition(v), rel=1e-12, abs=1e-13)
        assert der == pytest.approx(fd, rel=2e-6, abs=2e-7)


def flux_jacobian_prim(W, g):
    """d(Euler flux)/d(rho, u, v, p), written out by hand."""
    r, u, v, p = W
    q = u * u + v * v
    H = g * p / (g - 1.0) + 0.5 * r * q  # E + p
    return np.array([
        [u, r, 0.0, 0.0],
        [u * u, 2 * r * u, 0.0, 1.0],
        [u * v, r * v, r * u, 0.0],
        [0.5 * u * q, H + r * u * u, r * u * v, u * g / (g - 1.0)],
    ])


def test_hllc_tangent_equal_states_is_the_exact_flux_derivative():
    rng = np.random.default_rng(2)
    for _ in range(10):
        W = np.array([rng.uniform(0.5, 2), rng.uniform(-0.5, 0.5), rng.uniform(-1, 1), rng.uniform(0.5, 2)])
        d = rng.normal(size=4)
        # both sides move together: consistency F(W, W) = F(W) holds along the direction
        F, Fd = jxo.hllc_tangent(W, W, d, d, G, 0.0)
        assert np.allclose(F, refs.euler_flux_x(W, G)[0], rtol=1e-13, atol=1e-14)
        assert np.allclose(Fd, flux_jacobian_prim(W, G) @ d, rtol=1e-11, atol=1e-12)
        # gamma alone: only the energy flux u (p/(gamma-1) + ... + p) depends on it
        F, Fd = jxo.hllc_tangent(W, W, np.zeros(4), np.zeros(4), G, 1.0)
        assert np.allclose(Fd, [0, 0, 0, -W[1] * W[3] / (G - 1.0) ** 2], rtol=1e-11, atol=1e-12)


def test_hllc_tangent_supersonic_is_upwind():
    WL = np.array([1.0, 3.0, 0.2, 1.0])   # u - a > 0 on both sides
    WR = np.array([0.8, 2.8, -0.1, 0.9])
    dL, dR = np.array([0.3, -0.2, 0.5, 0.7]), np.array([1.0, 1.0, 1.0, 1.0])
    F, Fd = jxo.hllc_tangent(WL, WR, dL, dR, G, 0.5)
    want = flux_jacobian_prim(WL, G) @ dL + 0.5 * np.array([0, 0, 0, -WL[1] * WL[3] / (G - 1.0) ** 2])
    assert np.allclose(Fd, want, rtol=1e-12, atol=1e-13)       # nothing of the right state
    F, Fd = jxo.hllc_tangent(WR * [1, -1, 1, 1], WL * [1, -1, 1, 1], dR, dL * [1, -1, 1, 1], G, 0.0)
    mirrored = flux_jacobian_prim(WL * [1, -1, 1, 1], G) @ (dL * [1, -1, 1, 1])
    assert np.allclose(Fd, mirrored, rtol=1e-12, atol=1e-13)   # u + a < 0: the right state alone


def test_hllc_tangent_matches_central_difference_of_toro():
    rng = np.random.default_rng(3)
    n = 0
    for _ in range(40):
        WL = np.array([rng.uniform(0.3, 2), rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(0.3, 2)])
        WR = np.array([rng.uniform(0.3, 2), rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(0.3, 2)])
        sp, _, _ = jxo.hllc_star(WL, WR, G)
        if min(abs(sp)) < 1e-3:  # a wave speed at zero: the flux has a kink there
            continue
        dL, dR, dg = rng.normal(size=4), rng.normal(size=4), rng.normal()
        h = 1e-6
        fd = (refs.hllc_toro(WL + h * dL, WR + h * dR, G + h * dg) -
              refs.hllc_toro(WL - h * dL, WR - h * dR, G - h * dg)) / (2 * h)
        _, Fd = jxo.hllc_tangent(WL, WR, dL, dR, G, dg)
        assert np.allclose(Fd, fd, rtol=2e-6, atol=2e-7)
        n += 1
    assert n >= 30


# --------------------------------------------------------------------------- the step
def central_difference(case, Udir, gdir, dt, nsteps, h, **kw):
    Up = make(case, gamma=case["gamma"] + h * gdir, **kw).step_fixed_dt(case["U0"] + h * Udir, dt, nsteps)
    Um = make(case, gamma=case["gamma"] - h * gdir, **kw).step_fixed_dt(case["U0"] - h * Udir, dt, nsteps)
    return (Up - Um) / (2 * h)


def test_step_tangent_vortex_matches_central_differences():
    case = wl.vortex(24)
    dt, ns = 0.05, 3
    # h: the truncation error grows with the size of the direction (WENO weights with eps = 1e-6 have large third
    # derivatives), the round-off of the quotient is about 1e-16 / h on tangents of 4e-4 .. 6
    for Udir, gdir, h in ((np.zeros_like(case["U0"]), 1.0, 1e-6),                    # gamma alone, conserved state fixed
                          (wl.smooth_direction(case["U0"].shape, seed=4), 0.0, 1e-6),  # the state alone
                          (wl.dcons_dgamma(case["U0"], G), 1.0, 1e-5)):                 # gamma at fixed primitives
        U, Ud = make(case).step_fixed_dt_tangent(case["U0"], Udir, gdir, dt, ns)
        assert np.array_equal(U, make(case).step_fixed_dt(case["U0"], dt, ns))  # the value is the primal, bit for bit
        fd = central_difference(case, Udir, gdir, dt, ns, h)
        assert rel(Ud, fd) < 5e-7


def test_step_tangent_is_linear_in_the_direction():
    case = wl.vortex(16)
    o = make(case)
    d1, d2 = wl.smooth_direction(case["U0"].shape, seed=5), wl.smooth_direction(case["U0"].shape, seed=6)
    _, t1 = o.step_fixed_dt_tangent(case["U0"], d1, 0.0, 0.05, 2)
    _, t2 = o.step_fixed_dt_tangent(case["U0"], d2, 1.0, 0.05, 2)
    _, t3 = o.step_fixed_dt_tangent(case["U0"], 2.0 * d1 - 3.0 * d2, -3.0, 0.05, 2)
    assert rel(t3, 2.0 * t1 - 3.0 * t2) < 1e-12
    _, t0 = o.step_fixed_dt_tangent(case["U0"], np.zeros_like(d1), 0.0, 0.05, 2)
    assert np.all(t0 == 0.0)


def test_step_tangent_uniform_flow_keeps_a_uniform_direction():
    # a uniform state is a fixed point for every gamma; a uniform perturbation of it is again uniform
    n = 16
    U0 = wl.cons_from_prim(np.full((n, n), 1.3), 0.4, -0.2, 0.9, G)
    case = dict(nx=n, ny=n, dx=0.1, dy=0.1, gamma=G, mu=0.0, Pr=0.72, phi=None, U0=U0,
                bc=dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic"))
    Ud0 = np.ones_like(U0) * np.array([0.3, -0.1, 0.2, 0.5])[:, None, None]
    _, Ud = make(case).step_fixed_dt_tangent(U0, Ud0, 1.0, 0.01, 4)
    assert rel(Ud, Ud0) < 1e-13


def test_step_tangent_with_viscosity_walls_and_a_body_matches_central_differences():
    # every branch of the path at once: inflow / transmissive / reflective frame, IBM ghosts, viscous fluxes
    # (kappa depends on gamma), the shock
    case = wl.shock_cylinder(nx=64, ny=32, Ms=2.0, Re=200.0)
    dt, ns = 2e-3, 3
    Udir = wl.dcons_dgamma(case["U0"], G) + 0.1 * wl.smooth_direction(case["U0"].shape, seed=7)
    U, Ud = make(case).step_fixed_dt_tangent(case["U0"], Udir, 1.0, dt, ns)
    fd = central_difference(case, Udir, 1.0, dt, ns, 1e-7)
    fluid = (case["phi"] > 0)[None]
    assert rel(Ud * fluid, fd * fluid) < 5e-6


def sod_rows(nx, ny=8):
    return wl.as_rows(wl.sod1d(nx), ny)


def test_step_tangent_sod_conserves_and_keeps_the_first_moment():
    case = sod_rows(128)
    dx, dt, ns = case["dx"], 0.2 * case["dx"], 40   # waves stay inside the tube: no flux through the ends
    Ud0 = wl.dcons_dgamma(case["U0"], G)
    U, Ud = make(case).step_fixed_dt_tangent(case["U0"], Ud0, 1.0, dt, ns)
    row, row0 = Ud[:, 0, :], Ud0[:, 0, :]
    assert np.abs(Ud - Ud[:, :1, :]).max() < 1e-12                    # planar stays planar
    assert abs(row[0].sum() * dx) < 1e-13                            # d/dgamma of the mass
    assert abs(row[1].sum() * dx) < 1e-12                            # of the momentum (p_L - p_R) t
    assert row[3].sum() * dx == pytest.approx(row0[3].sum() * dx, rel=1e-12)   # of the energy sum(p)/(gamma-1)
    # d/dt int(x rho) = int(rho u) = (p_L - p_R) t for every gamma: the first moment of rho does not feel gamma in
    # the differential equations; the scheme keeps that to truncation error (its mass flux is not the cell momentum)
    x = (np.arange(case["nx"]) + 0.5) * dx
    assert abs((x * row[0]).sum() * dx) < 2e-3 * (x * np.abs(row[0])).sum() * dx
    assert np.abs(row[0]).max() > 0.1                                # and the tangent is far from zero


def test_step_tangent_sod_agrees_with_the_exact_riemann_solution():
    # second moments of the exact solution as functions of gamma (refs.riemann_sample), differentiated by central
    # differences, against the same moments of the tangent; the scheme's smearing is O(dx)
    nx, t_end = 400, 0.15
    case = sod_rows(nx, 8)
    dx = case["dx"]
    ns = 150
    dt = t_end / ns
    U, Ud = make(case).step_fixed_dt_tangent(case["U0"], wl.dcons_dgamma(case["U0"], G), 1.0, dt, ns)
    x = (np.arange(nx) + 0.5) * dx

    def exact_moments(g):
        # the exact solution is smooth between its waves: Gauss-Legendre on each piece, so that the moments are smooth
        # functions of gamma (the wave positions move with it)
        ps, us = refs.riemann_star(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)
        al, ar = np.sqrt(g * 1.0 / 1.0), np.sqrt(g * 0.1 / 0.125)
        tail = us - al * ps ** ((g - 1) / (2 * g))
        shock = ar * np.sqrt((g + 1) / (2 * g) * ps / 0.1 + (g - 1) / (2 * g))
        cuts = np.array([-0.5 / t_end, -al, tail, us, shock, 0.5 / t_end]) * t_end   # in x - 0.5
        xs, ws = np.polynomial.legendre.leggauss(24)
        m = np.zeros(3)
        for a, b in zip(cuts[:-1], cuts[1:]):
            xx = 0.5 * (a + b) + 0.5 * (b - a) * xs
            rho, u, pp = refs.riemann_sample(xx / t_end, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)
            w = 0.5 * (b - a) * ws * xx ** 2
            m += [(w * rho).sum(), (w * rho * u).sum(), (w * (pp / (g - 1) + 0.5 * rho * u * u)).sum()]
        return m

    h = 1e-5
    want = (exact_moments(G + h) - exact_moments(G - h)) / (2 * h)
    w = (x - 0.5) ** 2 * dx
    got = np.array([(w * Ud[0, 0]).sum(), (w * Ud[1, 0]).sum(), (w * Ud[3, 0]).sum()])
    assert np.allclose(got, want, rtol=0.03, atol=2e-4), (got, want)


def test_gamma_inference_recovers_the_value_behind_the_data():
    # PAPER.md L149 / Fig. 3(b): gamma from Sod data.  Data: the primal run at gamma = 1.4.  Unknown: gamma, starting
    # at 1.25; initial condition given in primitives (Eq. 17), so the conserved start depends on gamma as well.
    nx, ns = 64, 30
    base = wl.sod1d(nx)
    dt = 0.2 * base["dx"]
    target = make(sod_rows(nx)).step_fixed_dt(sod_rows(nx)["U0"], dt, ns)
    g = 1.25
    losses = []
    for _ in range(6):
        case = wl.as_rows(wl.sod1d(nx, gamma=g), 8)
        U, Ud = make(case).step_fixed_dt_tangent(case["U0"], wl.dcons_dgamma(case["U0"], g), 1.0, dt, ns)
        loss, dloss = jxo.mse_tangent(U, Ud, target)
        losses.append(loss)
        # Gauss-Newton on the one unknown: r(g) ~ r + Ud dg
        g -= np.sum((U - target) * Ud) / np.sum(Ud * Ud)
    assert abs(g - 1.4) < 1e-8
    assert losses[-1] < 1e-16 < losses[0]
    # and the gradient of Eq. 14 is the derivative of the loss
    case = wl.as_rows(wl.sod1d(nx, gamma=1.3), 8)
    U, Ud = make(case).step_fixed_dt_tangent(case["U0"], wl.dcons_dgamma(case["U0"], 1.3), 1.0, dt, ns)
    _, dloss = jxo.mse_tangent(U, Ud, target)
    h = 1e-6
    lp = [jxo.mse_tangent(make(c).step_fixed_dt(c["U0"], dt, ns), 0 * target, target)[0]
          for c in (wl.as_rows(wl.sod1d(nx, gamma=1.3 + h), 8), wl.as_rows(wl.sod1d(nx, gamma=1.3 - h), 8))]
    assert dloss == pytest.approx((lp[0] - lp[1]) / (2 * h), rel=1e-5)


def test_adjoint_is_the_gradient_of_a_linear_functional():
    # O13 against central differences of the primal oracle: phi(U0, gamma) = <c, S^n(U0; gamma)> has gradient
    # (J^T c, <c, dS/dgamma>); sampled entries of U0
    case = wl.vortex(8)
    dt, ns = 0.05, 2
    rng = np.random.default_rng(8)
    c = rng.normal(size=case["U0"].shape)
    grad, gbar = make(case).step_fixed_dt_adjoint(case["U0"], c, dt, ns)
    h = 1e-7  # a one-cell perturbation: the WENO weights (eps = 1e-6) have large third derivatives
    for j in rng.choice(c.size, 12, replace=False):
        e = np.zeros(c.shape)
        e.flat[j] = 1.0
        fd = np.sum(c * central_difference(case, e, 0.0, dt, ns, h))
        assert grad.flat[j] == pytest.approx(fd, rel=2e-6, abs=1e-8)
    assert gbar == pytest.approx(np.sum(c * central_difference(case, 0 * c, 1.0, dt, ns, 1e-6)), rel=1e-6)
    # planar form = the 1D adjoint: its pairing with any 1D direction equals the tangent's pairing with c
    case = sod_rows(24)
    c1 = rng.normal(size=(4, 1, 24))
    d1 = rng.normal(size=(4, 1, 24))
    g1, gb1 = make(case).step_fixed_dt_adjoint(case["U0"], c1, 0.2 * case["dx"], 2, planar=True)
    _, D = make(case).step_fixed_dt_tangent(case["U0"], np.repeat(d1, 8, axis=1), 0.7, 0.2 * case["dx"], 2)
    assert np.sum(c1 * D[:, :1]) == pytest.approx(np.sum(g1 * d1) + 0.7 * gb1, rel=1e-12)


def test_rhs_tangent_and_the_euler_update():
    case = wl.shock_cylinder(nx=64, ny=32, Ms=2.0, Re=200.0)
    Udir = wl.dcons_dgamma(case["U0"], G) + 0.1 * wl.smooth_direction(case["U0"].shape, seed=12)
    o = make(case)
    L, Ld = o.rhs_tangent(case["U0"], Udir, 1.0)
    assert np.array_equal(L, o.rhs(case["U0"]))
    h = 1e-7
    fd = (make(case, gamma=G + h).rhs(case["U0"] + h * Udir) - make(case, gamma=G - h).rhs(case["U0"] - h * Udir)) / (2 * h)
    fluid = (case["phi"] > 0)[None]
    assert rel(Ld * fluid, fd * fluid) < 5e-6
    # SSP-RK3 composed from rhs_tangent by hand is O12
    dt = 1e-3
    def stage(U, D):
        L, Ld = o.rhs_tangent(U, D, 1.0)
        return U + dt * L, D + dt * Ld
    U1, D1 = stage(case["U0"], Udir)
    U2, D2 = stage(U1, D1)
    U2, D2 = 0.75 * case["U0"] + 0.25 * U2, 0.75 * Udir + 0.25 * D2
    U3, D3 = stage(U2, D2)
    U3, D3 = case["U0"] / 3 + 2 * U3 / 3, Udir / 3 + 2 * D3 / 3
    Us, Ds = o.step_fixed_dt_tangent(case["U0"], Udir, 1.0, dt, 1)
    # (fluid cells: the step also leaves its IBM ghost fill in the non-fluid cells it returns)
    assert rel(U3 * fluid, Us * fluid) < 1e-14 and rel(D3 * fluid, Ds * fluid) < 1e-12
    # Eq. 10: two Euler steps against central differences of the same update written with the primal L
    def euler(c, g, U, n):
        oo = make(c, gamma=g)
        for _ in range(n):
            U = U + dt * oo.rhs(U)
        return U
    Ue, De = o.step_fixed_dt_tangent(case["U0"], Udir, 1.0, dt, 2, scheme="euler")
    assert np.array_equal(Ue, euler(case, G, case["U0"], 2))
    fd = (euler(case, G + h, case["U0"] + h * Udir, 2) - euler(case, G - h, case["U0"] - h * Udir, 2)) / (2 * h)
    assert rel(De * fluid, fd * fluid) < 5e-6


def test_tangent_through_the_exact_mlp_matches_central_differences():
    # O12 with the network: its inputs' dependence on the state and on gamma, and a direction in its 6020 parameters
    case = wl.vortex(12)
    w = wl.mlp_weights(3)
    sc = wl.mlp_scales(out_factor=5e-2)
    dt, ns = 0.04, 2
    rng = np.random.default_rng(14)
    wdir = rng.normal(size=6020)

    def run(U0, g, ww):
        o = make(case, gamma=g)
        o.set_flux_mlp(ww, *sc, emulate_bf16=False)
        return o.step_fixed_dt(U0, dt, ns)

    o = make(case)
    o.set_flux_mlp(w, *sc, emulate_bf16=False)
    assert rel(run(case["U0"], G, w), make(case).step_fixed_dt(case["U0"], dt, ns)) > 1e-4   # the network acts
    Udir = wl.smooth_direction(case["U0"].shape, seed=15)
    h = 2e-7   # a coarse grid: the third derivatives of the WENO weights are large
    # state and gamma
    U, Ud = o.step_fixed_dt_tangent(case["U0"], Udir, 0.7, dt, ns)
    assert np.array_equal(U, run(case["U0"], G, w))
    fd = (run(case["U0"] + h * Udir, G + 0.7 * h, w) - run(case["U0"] - h * Udir, G - 0.7 * h, w)) / (2 * h)
    assert rel(Ud, fd) < 5e-7
    # the parameters: float32 weights perturbed along a float32 direction, the quotient taken with the step made
    hw = np.float32(2.0 ** -12)
    wd32 = wdir.astype(np.float32)
    wp, wm = (w + hw * wd32).astype(np.float32), (w - hw * wd32).astype(np.float32)
    actual = (wp.astype(np.float64) - wm.astype(np.float64)) / (2.0 * float(hw))   # the direction really taken
    o.set_flux_mlp_direction(actual)
    _, Ud = o.step_fixed_dt_tangent(case["U0"], np.zeros_like(Udir), 0.0, dt, ns)
    fd = (run(case["U0"], G, wp) - run(case["U0"], G, wm)) / (2.0 * float(hw))
    assert np.abs(Ud).max() > 1e-6 and rel(Ud, fd) < 1e-5
    o.set_flux_mlp_direction(None)
    _, Ud = o.step_fixed_dt_tangent(case["U0"], np.zeros_like(Udir), 0.0, dt, ns)
    assert np.all(Ud == 0.0)


def test_tangent_argument_checks():
    case = wl.vortex(8)
    o = make(case, dtype=np.float32)
    with pytest.raises(jxo.OracleError):
        o.step_fixed_dt_tangent(case["U0"].astype(np.float32), np.zeros_like(case["U0"]), 1.0, 0.01, 1)
    o = make(case)
    o.set_flux_mlp(wl.mlp_weights(), *wl.mlp_scales(), emulate_bf16=True)   # only the exact MLP is differentiated
    with pytest.raises(jxo.OracleError):
        o.step_fixed_dt_tangent(case["U0"], np.zeros_like(case["U0"]), 1.0, 0.01, 1)
