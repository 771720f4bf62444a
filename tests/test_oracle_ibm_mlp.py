"""Pins for the oracle's immersed boundary (O2) and per-face MLP (O10).  -m "not gpu"."""
import math

import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl

G = 1.4
PER = dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic")


def cyl_case(nx=96, ny=48, r=0.12, viscous=False, Ms=2.0):
    return wl.shock_cylinder(nx, ny, Ms=Ms, bodies=((0.55, 0.5, r),), x_shock=0.2, viscous=viscous, Re=200.0)


def oracle_for(case, **kw):
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"],
                   case["bc"], **kw)
    o.set_ibm(case["phi"])
    return o


def prims(U):
    r = U[0]
    u, v = U[1] / r, U[2] / r
    return np.stack([r, u, v, (G - 1) * (U[3] - 0.5 * r * (u * u + v * v))])


# ------------------------------------------------------------------------ IBM
def test_cell_classification_matches_the_definition():
    """P:L111 'fluid, solid, ghost, or image cells'; reading R9 (I1, I2), rebuilt with array shifts."""
    case = cyl_case()
    t = oracle_for(case).cell_types()
    fluid = case["phi"] > 0
    assert np.array_equal(t == 0, fluid)
    near = np.zeros_like(fluid)
    F = np.pad(fluid, 3, constant_values=False)
    ny, nx = fluid.shape
    for k in (1, 2, 3):
        for (dj, di) in ((0, k), (0, -k), (k, 0), (-k, 0)):
            near |= F[3 + dj:3 + dj + ny, 3 + di:3 + di + nx]
    for (dj, di) in ((1, 1), (1, -1), (-1, 1), (-1, -1)):
        near |= F[3 + dj:3 + dj + ny, 3 + di:3 + di + nx]
    assert np.array_equal(t == 1, ~fluid & near)
    assert np.array_equal(t == 2, ~fluid & ~near)
    assert (t == 2).sum() > 0 and (t == 1).sum() > 0


def test_ghost_list_geometry():
    case = cyl_case()
    o = oracle_for(case)
    cell, donors, w, nrm = o.ibm_ghosts()
    nx, dx, dy = case["nx"], case["dx"], case["dy"]
    t = o.cell_types().ravel()
    assert np.array_equal(np.sort(cell), np.flatnonzero(t == 1))
    assert np.all(w >= 0) and np.allclose(w.sum(axis=1), 1.0, atol=1e-15)
    assert np.all(t[donors[w > 0]] == 0)  # donors with weight are fluid cells
    assert np.allclose(np.hypot(nrm[:, 0], nrm[:, 1]), 1.0, atol=1e-15)
    xg, yg = (cell % nx + 0.5) * dx, (cell // nx + 0.5) * dy
    rad = np.stack([xg - 0.55, yg - 0.5], axis=1)
    rad /= np.linalg.norm(rad, axis=1)[:, None]
    assert np.max(np.abs(nrm - rad)) < 0.02  # central differences of a distance function
    # bilinear weights reproduce linear functions: sum w_k x_k is the image point x_G + 2|phi_G| n
    full = np.all(w > 0, axis=1)
    assert full.sum() > 0.5 * len(cell)
    xd, yd = (donors % nx + 0.5) * dx, (donors // nx + 0.5) * dy
    phi_g = np.abs(case["phi"].ravel()[cell])
    xi, yi = xg + 2 * phi_g * nrm[:, 0], yg + 2 * phi_g * nrm[:, 1]
    assert np.max(np.abs((w * xd).sum(1) - xi)[full]) < 1e-13
    assert np.max(np.abs((w * yd).sum(1) - yi)[full]) < 1e-13
    # every image point lies in the fluid, at the mirror distance from the surface
    d_img = np.hypot(xi - 0.55, yi - 0.5) - 0.12
    assert np.all(d_img[full] > 0) and np.max(np.abs(d_img - phi_g)[full]) < 0.05 * dx


def test_ghost_state_is_the_slip_wall_mirror_of_the_image_state():
    """'zero normal penetration while preserving the tangential component of velocity'."""
    case = cyl_case()
    o = oracle_for(case)
    rng = np.random.default_rng(1)
    ny, nx = case["ny"], case["nx"]
    U = wl.cons_from_prim(rng.uniform(1, 2, (ny, nx)), rng.uniform(-1, 1, (ny, nx)),
                          rng.uniform(-1, 1, (ny, nx)), rng.uniform(1, 2, (ny, nx)))
    Up = o.fill_ghosts(U)[:, 3:-3, 3:-3]
    cell, donors, w, nrm = o.ibm_ghosts()
    W = prims(U).reshape(4, -1)
    WI = (W[:, donors] * w[None]).sum(axis=2)  # [4][nghost]
    WG = prims(Up).reshape(4, -1)[:, cell]
    n, t = nrm.T, np.stack([-nrm[:, 1], nrm[:, 0]])
    assert np.allclose(WG[0], WI[0], rtol=1e-14) and np.allclose(WG[3], WI[3], rtol=1e-13)
    assert np.allclose((WG[1:3] * n).sum(0), -(WI[1:3] * n).sum(0), atol=1e-14)
    assert np.allclose((WG[1:3] * t).sum(0), (WI[1:3] * t).sum(0), atol=1e-14)
    assert np.allclose(np.hypot(WG[1], WG[2]), np.hypot(WI[1], WI[2]), atol=1e-14)
    mask = np.ones(nx * ny, bool)
    mask[cell] = False
    assert np.array_equal(Up.reshape(4, -1)[:, mask], U.reshape(4, -1)[:, mask])  # nothing else touched


@pytest.mark.parametrize("viscous", [False, True])
def test_quiescent_state_is_preserved_around_the_body(viscous):
    case = cyl_case(viscous=viscous)
    ny, nx = case["ny"], case["nx"]
    one = np.ones((ny, nx))
    U = wl.cons_from_prim(1.4 * one, 0 * one, 0 * one, one)
    case["bc"] = dict(xlo="transmissive", xhi="transmissive", ylo="reflective", yhi="reflective")
    o = oracle_for(case)
    # interpolation weights sum to 1 only to round-off, so the ghost states carry 1-ulp noise
    assert np.max(np.abs(o.rhs(U))) < 1e-12
    # the convex RK combinations (3/4 + 1/4, 1/3 + 2/3) round, so "preserved" means to round-off
    assert np.max(np.abs(o.step(U, 0.4, 3) - U)) < 1e-14


def test_body_too_close_to_the_edge_is_rejected():
    case = cyl_case()
    phi = wl.cylinders_phi(case["nx"], case["ny"], case["dx"], case["dy"], [(0.1, 0.5, 0.08)])
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], G, 0, 0.72, case["bc"])
    with pytest.raises(jxo.OracleError) as e:
        o.set_ibm(phi)
    assert e.value.code == jxo.EINVAL


def test_grid_aligned_wall_reproduces_the_reflective_boundary():
    """A rectangular body whose faces lie on cell faces: along rows far from its corners (further than
    the numerical domain of dependence, 3 cells per stage) the IBM ghost fill must reproduce the
    REFLECTIVE domain boundary of a truncated domain to round-off (image point = mirror cell centre)."""
    nx, ny, h = 64, 64, 1.0 / 64
    iw = 40  # wall on the face between cells 39 and 40
    X, Y = wl.cell_centres(nx, ny, h, h)
    x0, x1, y0, y1 = iw * h, (iw + 12) * h, 12 * h, 52 * h
    ddx = np.maximum(np.maximum(x0 - X, X - x1), 0.0)
    ddy = np.maximum(np.maximum(y0 - Y, Y - y1), 0.0)
    outside = np.hypot(ddx, ddy)
    inside = np.minimum(np.minimum(X - x0, x1 - X), np.minimum(Y - y0, y1 - Y))
    phi = np.where((X > x0) & (X < x1) & (Y > y0) & (Y < y1), -inside, outside)
    # y-uniform data: a Mach-2 shock travelling towards the wall plus a smooth perturbation
    rho2, u2, p2, _ = wl.rankine_hugoniot(2.0)
    x = X[0]
    rho = np.where(x < 0.45, rho2, 1.4) * (1 + 0.05 * np.sin(9 * x))
    u = np.where(x < 0.45, u2, 0.0) + 0.1 * np.cos(7 * x)
    p = np.where(x < 0.45, p2, 1.0) * (1 + 0.05 * np.cos(5 * x))
    tile = lambda a: np.tile(a, (ny, 1))
    U = wl.cons_from_prim(tile(rho), tile(u), 0 * tile(u), tile(p))
    bc = dict(xlo="transmissive", xhi="transmissive", ylo="transmissive", yhi="transmissive")
    mu = 1e-3
    a = jxo.Oracle(nx, ny, h, h, G, mu, 0.72, bc)
    a.set_ibm(phi)
    Ua = a.step_fixed_dt(U, 1e-3, 2)  # 2 steps = 6 stages = 18 cells of dependence < 20
    bcw = dict(xlo="transmissive", xhi="reflective", ylo="transmissive", yhi="transmissive")
    b = jxo.Oracle(iw, ny, h, h, G, mu, 0.72, bcw)
    Ub = b.step_fixed_dt(np.ascontiguousarray(U[:, :, :iw]), 1e-3, 2)
    mid = 32
    assert np.max(np.abs(Ua[:, mid, :iw] - Ub[:, mid, :])) < 1e-12
    assert np.max(np.abs(Ua[:, mid, :iw] - U[:, mid, :iw])) > 1e-3  # the wall rows did evolve


def test_shock_cylinder_stays_mirror_symmetric():
    """'two well-defined shock wave triple points arise symmetrically'."""
    case = cyl_case(viscous=True)
    o = oracle_for(case)
    U = o.step(case["U0"], 0.4, 30)
    assert o.guard_count() == 0
    sgn = np.array([1, 1, -1, 1])[:, None, None]
    fluid = (o.cell_types() == 0)[None]
    d = np.abs(U - U[:, ::-1, :] * sgn) * fluid
    assert d.max() < 1e-10 and np.abs(U[2]).max() > 0.05  # symmetric, and the flow is not trivial


# ------------------------------------------------------------------------ MLP
def _mlp_setup(n=16, seed=0):
    rng = np.random.default_rng(seed)
    U = wl.cons_from_prim(rng.uniform(1, 2, (n, n)), rng.uniform(-1, 1, (n, n)),
                          rng.uniform(-1, 1, (n, n)), rng.uniform(1, 2, (n, n)))
    return U, jxo.Oracle(n, n, 1.0 / n, 1.0 / n, G, 0.0, 0.72, PER)


def test_zero_weights_leave_the_flux_unchanged():
    U, o = _mlp_setup()
    base = o.rhs(U)
    o.set_flux_mlp(np.zeros(6020, np.float32), np.ones(4), np.ones(4))
    assert np.array_equal(o.rhs(U), base)
    o.set_flux_mlp(None)
    assert np.array_equal(o.rhs(U), base)


def test_mlp_matches_a_float64_torch_mlp():
    """O10 / BASELINE.json configs[4]: 24 -> 64 tanh -> 64 tanh -> 4 linear, row-major W[out][in]."""
    U, o = _mlp_setup()
    w = wl.mlp_weights(3)
    w[64 * 24:64 * 24 + 64] = 0.1  # non-zero biases so that their placement is tested
    w[-4:] = [0.3, -0.2, 0.1, 0.05]
    o.set_flux_mlp(w, np.ones(4), np.ones(4))
    t = torch.tensor(w, dtype=torch.float64)
    W1, b1, W2, b2, W3, b3 = torch.split(t, [1536, 64, 4096, 64, 256, 4])
    x = np.random.default_rng(2).standard_normal(24)
    h = torch.tanh(torch.nn.functional.linear(torch.tensor(x), W1.view(64, 24), b1))
    h = torch.tanh(torch.nn.functional.linear(h, W2.view(64, 64), b2))
    y = torch.nn.functional.linear(h, W3.view(4, 64), b3).numpy()
    assert np.allclose(o.mlp_eval(x), y, rtol=1e-13, atol=1e-14)


@pytest.mark.parametrize("cell,var", [(0, 0), (5, 3), (2, 1), (3, 2)])
def test_mlp_input_ordering_and_output_mapping(cell, var):
    """One active path: y_m = out_scale[m] * W3[m][0] * tanh(tanh(x[4*cell+var])).  Cells i-2..i+3 in
    order; y-faces take (rho, v, u, p) and map (mass, normal, tangential, energy) back (Eq. 11)."""
    n = 16
    U, o = _mlp_setup(n)
    base = o.rhs(U)
    w = np.zeros(6020, np.float32)
    w[0 * 24 + 4 * cell + var] = 1.0  # W1[0][4*cell+var]
    w[1536 + 64 + 0] = 1.0  # W2[0][0]
    w3 = np.array([0.5, -1.0, 2.0, 0.25], np.float32)
    w[1536 + 64 + 4096 + 64 + np.arange(4) * 64] = w3  # W3[m][0]
    in_scale, out_scale = np.array([1.3, 0.7, 0.7, 2.0]), np.array([1e-2, 2e-2, 3e-2, 4e-2])
    o.set_flux_mlp(w, in_scale, out_scale)
    d = o.rhs(U) - base
    W = prims(U)
    h = 1.0 / n
    # x-faces: face i+1/2 sees cell i-2+cell, variable var
    sx = np.tanh(np.tanh(np.roll(W[var], -(cell - 2), axis=1) / in_scale[var]))  # value for face i+1/2
    dFx = out_scale[:, None, None] * w3[:, None, None] * sx[None]
    # y-faces: variable order (rho, v, u, p); outputs (mass, y-mom, x-mom, energy) -> swap back
    vy = [0, 2, 1, 3][var]
    sy = np.tanh(np.tanh(np.roll(W[vy], -(cell - 2), axis=0) / in_scale[var]))
    dGn = out_scale[:, None, None] * w3[:, None, None] * sy[None]
    dGy = dGn[[0, 2, 1, 3]]
    want = -(dFx - np.roll(dFx, 1, axis=2)) / h - (dGy - np.roll(dGy, 1, axis=1)) / h
    assert np.max(np.abs(d - want)) < 1e-11 * max(1.0, np.max(np.abs(base)))
    assert np.max(np.abs(want)) > 1e-3


def test_bf16_emulation_error_is_small_and_reported():
    U, o = _mlp_setup()
    w = wl.mlp_weights(4)
    ins, outs = wl.mlp_scales()
    o.set_flux_mlp(w, ins, outs)
    base = jxo.Oracle(16, 16, 1.0 / 16, 1.0 / 16, G, 0.0, 0.72, PER).rhs(U)
    exact = o.rhs(U) - base
    o.set_flux_mlp(w, ins, outs, emulate_bf16=True)
    emul = o.rhs(U) - base
    rel = np.max(np.abs(emul - exact)) / np.max(np.abs(exact))
    assert 0 < rel < 5e-2, rel
