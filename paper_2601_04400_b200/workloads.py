"""Seeded synthetic inputs shared by the CPU oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no reconstruction, no Riemann
solver, no boundary fill, no time stepping): it only builds initial fields,
level sets and weight blobs, as numpy arrays, which are handed unchanged to both
the oracle (oracle/) and the CUDA library.  It imports neither of them.

The inputs are synthetic stand-ins shaped like the paper's workloads — the Sod
tube (Eq. 17) and the shock/cylinder interaction (L151-162,
Eq. 18) — with the sizes BASELINE.json's configs name.  The recipe for every
case is restated in DESIGN.md ("Input recipe").

Every case is a dict:
  U0 [4,ny,nx] float64 (rho, rho u, rho v, E), x fastest;  nx, ny, dx, dy,
  gamma, mu, Pr, bc {xlo,xhi,ylo,yhi[,inflow]}, phi [ny,nx] or None, name.
"""
import math

import numpy as np

GAMMA = 1.4
SEED_THROUGHPUT = 260104400


def cons_from_prim(rho, u, v, p, gamma=GAMMA):
    """(rho,u,v,p) -> (rho, rho u, rho v, E) with the ideal-gas EOS (Eq. 2)."""
    rho, u, v, p = np.broadcast_arrays(rho, u, v, p)
    E = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v)
    return np.stack([rho, rho * u, rho * v, E]).astype(np.float64)


def dcons_dgamma(U, gamma=GAMMA):
    """Direction of perturbation of a conserved field when gamma changes at fixed primitives (rho, u, v, p):
    only E = p/(gamma-1) + kinetic moves, dE/dgamma = -p/(gamma-1)^2 = -(E - kinetic)/(gamma-1).  The seed of the
    gamma inference (Fig. 3b), whose initial condition Eq. 17 is given in primitives."""
    U = np.asarray(U, dtype=np.float64)
    kin = 0.5 * (U[1] ** 2 + U[2] ** 2) / U[0]
    D = np.zeros_like(U)
    D[3] = -(U[3] - kin) / (gamma - 1.0)
    return D


def smooth_direction(shape, seed=3, modes=3):
    """A seeded smooth field [4][ny][nx] (a few low Fourier modes per component, amplitude about 1): a direction of
    perturbation of the state for the tangent tests."""
    rng = np.random.default_rng(seed)
    _, ny, nx = shape
    X, Y = np.meshgrid((np.arange(nx) + 0.5) / nx, (np.arange(ny) + 0.5) / ny)
    D = np.zeros(shape)
    for k in range(4):
        for _ in range(modes):
            a, kx, ky, ph = rng.normal(), rng.integers(0, 3), rng.integers(0, 3), rng.uniform(0, 2 * math.pi)
            D[k] += a * np.cos(2 * math.pi * (kx * X + (ky if ny > 1 else 0) * Y) + ph)
    return D


def cell_centres(nx, ny, dx, dy, x0=0.0, y0=0.0):
    x = x0 + (np.arange(nx) + 0.5) * dx
    y = y0 + (np.arange(ny) + 0.5) * dy
    return np.meshgrid(x, y)  # X[j,i], Y[j,i]


def rankine_hugoniot(Ms, rho1=1.4, p1=1.0, gamma=GAMMA):
    """Post-shock state behind a shock of Mach number Ms moving into gas at rest.

    Returns (rho2, u2, p2, shock_speed).  Mach 5 into (1.4, 0, 1) gives exactly
    (7, 4, 29) and speed 5, the states printed in PAPER.md Eq. 18 (L159).
    """
    a1 = math.sqrt(gamma * p1 / rho1)
    rho2 = rho1 * (gamma + 1.0) * Ms * Ms / ((gamma - 1.0) * Ms * Ms + 2.0)
    p2 = p1 * (1.0 + 2.0 * gamma / (gamma + 1.0) * (Ms * Ms - 1.0))
    W = Ms * a1
    u2 = W * (1.0 - rho1 / rho2)
    return rho2, u2, p2, W


# --------------------------------------------------------------------------- C1
def sod(nx=128, ny=128, axis=0, gamma=GAMMA):
    """Config 1: planar Sod problem on [0,1]^2, transmissive BCs, Euler (Eq. 17)."""
    dx, dy = 1.0 / nx, 1.0 / ny
    X, Y = cell_centres(nx, ny, dx, dy)
    s = X if axis == 0 else Y
    left = s < 0.5
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    z = np.zeros_like(rho)
    bc = dict(xlo="transmissive", xhi="transmissive", ylo="transmissive", yhi="transmissive")
    return dict(name=f"sod{'xy'[axis]}_{nx}x{ny}", U0=cons_from_prim(rho, z, z, p, gamma), nx=nx, ny=ny,
                dx=dx, dy=dy, gamma=gamma, mu=0.0, Pr=0.72, bc=bc, phi=None)


def sod1d(nx=500, gamma=GAMMA):
    """The paper's 1D Sod shock tube (Eq. 17) on [0,1]: fields [4][1][nx], ny = 1, dy = dx."""
    dx = 1.0 / nx
    x = (np.arange(nx) + 0.5) * dx
    left = (x < 0.5)[None, :]
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    z = np.zeros_like(rho)
    bc = dict(xlo="transmissive", xhi="transmissive", ylo="transmissive", yhi="transmissive")
    return dict(name=f"sod1d_{nx}", U0=cons_from_prim(rho, z, z, p, gamma), nx=nx, ny=1, dx=dx, dy=dx, gamma=gamma,
                mu=0.0, Pr=0.72, bc=bc, phi=None)


def wavy1d(nx, gamma=GAMMA):
    """A 1D field for parity checks at large nx on sampled windows: the Sod jump at mid-tube carrying short waves
    (37 to 91 cells long) in every primitive, so that every window of a few dozen cells sees a different, varying
    state.  Deterministic; transmissive ends."""
    case = sod1d(nx, gamma)
    i = np.arange(nx, dtype=np.float64)
    left = i < nx // 2
    rho = np.where(left, 1.0, 0.125) * (1.0 + 0.2 * np.sin(2 * math.pi * i / 37.0))
    u = 0.4 * np.cos(2 * math.pi * i / 53.0)
    v = 0.2 * np.sin(2 * math.pi * i / 91.0)
    p = np.where(left, 1.0, 0.1) * (1.0 + 0.15 * np.cos(2 * math.pi * i / 71.0 + 0.3))
    case["U0"] = cons_from_prim(rho[None, :], u[None, :], v[None, :], p[None, :], gamma)
    case["name"] = f"wavy1d_{nx}"
    return case


def window(case, lo, hi):
    """Cells [lo, hi) of a 1D case as a case of its own (transmissive ends)."""
    c = dict(case)
    c["U0"] = np.ascontiguousarray(case["U0"][:, :, lo:hi])
    c["nx"] = hi - lo
    c["name"] = case["name"] + f"[{lo}:{hi}]"
    return c


def as_rows(case, ny=8):
    """A 1D case repeated over ny identical rows, periodic in y: the planar 2D problem whose every row is the 1D one
    (identical rows make the y-fluxes cancel exactly).  This is how the 2D oracle checks the 1D path."""
    c = dict(case)
    c["U0"] = np.ascontiguousarray(np.repeat(case["U0"], ny, axis=1))
    c["ny"] = ny
    c["bc"] = dict(case["bc"], ylo="periodic", yhi="periodic")
    c["name"] = case["name"] + f"_as_{ny}_rows"
    return c


# --------------------------------------------------------------------------- C2
def vortex_primitives(x, y, gamma=GAMMA, strength=5.0, xc=5.0, yc=5.0, u0=1.0, v0=1.0):
    """Isentropic vortex (config 2) point values, free stream (1, u0, v0, 1)."""
    r2 = (x - xc) ** 2 + (y - yc) ** 2
    f = strength / (2.0 * math.pi) * np.exp(0.5 * (1.0 - r2))
    u = u0 - f * (y - yc)
    v = v0 + f * (x - xc)
    T = 1.0 - (gamma - 1.0) * strength ** 2 / (8.0 * gamma * math.pi ** 2) * np.exp(1.0 - r2)
    rho = T ** (1.0 / (gamma - 1.0))
    p = rho ** gamma
    return rho, u, v, p


def vortex(n=64, gamma=GAMMA, quadrature=0, u0=1.0, v0=1.0):
    """Config 2: isentropic vortex on periodic [0,10]^2.

    quadrature = 0 -> point values at cell centres; q > 0 -> cell averages of the
    conserved variables by q x q Gauss-Legendre quadrature.
    """
    L = 10.0
    dx = dy = L / n
    X, Y = cell_centres(n, n, dx, dy)
    if quadrature <= 0:
        U0 = cons_from_prim(*vortex_primitives(X, Y, gamma, u0=u0, v0=v0), gamma)
    else:
        xs, ws = np.polynomial.legendre.leggauss(quadrature)
        U0 = np.zeros((4, n, n))
        for a, wa in zip(xs, ws):
            for b, wb in zip(xs, ws):
                U0 += 0.25 * wa * wb * cons_from_prim(
                    *vortex_primitives(X + 0.5 * dx * a, Y + 0.5 * dy * b, gamma, u0=u0, v0=v0), gamma)
    bc = dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic")
    return dict(name=f"vortex_{n}", U0=U0, nx=n, ny=n, dx=dx, dy=dy, gamma=gamma, mu=0.0, Pr=0.72,
                bc=bc, phi=None)


# ----------------------------------------------------------------------- C3 / C4
def cylinders_phi(nx, ny, dx, dy, bodies):
    """Signed distance (positive in the fluid) to a union of circles [(xc, yc, r), ...]."""
    X, Y = cell_centres(nx, ny, dx, dy)
    phi = np.full((ny, nx), np.inf)
    for (xc, yc, r) in bodies:
        phi = np.minimum(phi, np.sqrt((X - xc) ** 2 + (Y - yc) ** 2) - r)
    return phi


def shock_field(nx, ny, dx, dy, Ms, x_shock, gamma=GAMMA, rho1=1.4, p1=1.0):
    rho2, u2, p2, _ = rankine_hugoniot(Ms, rho1, p1, gamma)
    X, _ = cell_centres(nx, ny, dx, dy)
    left = X < x_shock
    rho = np.where(left, rho2, rho1)
    u = np.where(left, u2, 0.0)
    p = np.where(left, p2, p1)
    return cons_from_prim(rho, u, np.zeros_like(rho), p, gamma), (rho2, u2, 0.0, p2)


def shock_cylinder(nx=1024, ny=512, Ms=2.0, Re=1.0e4, gamma=GAMMA, bodies=((0.4, 0.5, 0.1),),
                   x_shock=0.2, viscous=True, name=None, d_ref=None):
    """Config 3: planar shock hitting a cylinder on [0,2]x[0,1] through the ghost-cell IBM.

    BCs as in PAPER.md L162: left inflow (= post-shock state), right outflow
    (transmissive), top/bottom reflective.  mu = rho2 u2 D / Re with the
    post-shock state and D the (mean) cylinder diameter (reading R12).
    """
    dx, dy = 2.0 / nx, 1.0 / ny
    U0, post = shock_field(nx, ny, dx, dy, Ms, x_shock, gamma)
    phi = cylinders_phi(nx, ny, dx, dy, bodies) if bodies else None
    if d_ref is None:
        d_ref = 2.0 * float(np.mean([b[2] for b in bodies])) if bodies else 0.2
    mu = post[0] * post[1] * d_ref / Re if viscous else 0.0
    bc = dict(xlo="inflow", xhi="transmissive", ylo="reflective", yhi="reflective", inflow=post)
    return dict(name=name or f"shockcyl_{nx}x{ny}_M{Ms:g}", U0=U0, nx=nx, ny=ny, dx=dx, dy=dy,
                gamma=gamma, mu=mu, Pr=0.72, bc=bc, phi=phi, bodies=list(bodies), Ms=Ms)


def random_cylinders(seed=SEED_THROUGHPUT, n=8, r_range=(0.02, 0.06), box=((0.3, 1.8), (0.15, 0.85)),
                     gap=0.04, wall=((0.0, 2.0), (0.0, 1.0))):
    """Non-overlapping circles by rejection sampling (reading R13)."""
    rng = np.random.default_rng(seed)
    bodies = []
    tries = 0
    while len(bodies) < n:
        tries += 1
        if tries > 100000:
            raise RuntimeError("rejection sampling did not converge")
        r = rng.uniform(*r_range)
        xc = rng.uniform(*box[0])
        yc = rng.uniform(*box[1])
        if min(xc - wall[0][0], wall[0][1] - xc, yc - wall[1][0], wall[1][1] - yc) - r < gap:
            continue
        if any(math.hypot(xc - b[0], yc - b[1]) - r - b[2] < gap for b in bodies):
            continue
        bodies.append((float(xc), float(yc), float(r)))
    return bodies


def throughput_case(nx=4096, ny=2048, seed=SEED_THROUGHPUT, Ms=3.0, Re=1.0e5, viscous=True, ibm=True):
    """Config 4 (the timed case): Mach-3 shock over 8 seeded cylinders, Navier-Stokes Re 1e5."""
    bodies = random_cylinders(seed) if ibm else ()
    case = shock_cylinder(nx, ny, Ms=Ms, Re=Re, bodies=tuple(bodies), x_shock=0.1, viscous=viscous,
                          name=f"throughput_{nx}x{ny}", d_ref=0.08)
    return case


# --------------------------------------------------------------------------- C5
MLP_SIZES = ((64, 24), (64, 64), (4, 64))
MLP_NPARAM = 6020


def mlp_weights(seed=5):
    """Glorot-uniform weights, zero biases, packed W1[64][24],b1,W2[64][64],b2,W3[4][64],b3 (fp32)."""
    rng = np.random.default_rng(seed)
    parts = []
    for (fo, fi) in MLP_SIZES:
        lim = math.sqrt(6.0 / (fi + fo))
        parts.append(rng.uniform(-lim, lim, size=(fo, fi)).astype(np.float32).ravel())
        parts.append(np.zeros(fo, dtype=np.float32))
    w = np.concatenate(parts)
    assert w.size == MLP_NPARAM
    return w


def mlp_scales(gamma=GAMMA, rho_ref=1.4, p_ref=1.0, out_factor=1.0e-3):
    """in_scale = (rho, a, a, p)_ref of the pre-shock state; out_scale = f*(rho a, rho a^2, rho a^2, rho a^3)."""
    a = math.sqrt(gamma * p_ref / rho_ref)
    in_scale = np.array([rho_ref, a, a, p_ref])
    out_scale = out_factor * np.array([rho_ref * a, rho_ref * a * a, rho_ref * a * a, rho_ref * a ** 3])
    return in_scale, out_scale


CNN_SIZES = ((32, 4), (16, 32), (4, 16))  # (out, in) channels of the three 3x3 convolutions
CNN_NPARAM = sum(o * i * 9 + o for o, i in CNN_SIZES)  # 6388, the count the paper prints


def cnn_weights(seed=9, bias=0.0):
    """Glorot-uniform 3x3 kernels in OIHW order, constant biases: W1[32][4][3][3], b1, W2[16][32][3][3], b2,
    W3[4][16][3][3], b3 (fp32)."""
    rng = np.random.default_rng(seed)
    parts = []
    for (fo, fi) in CNN_SIZES:
        lim = math.sqrt(6.0 / (9 * (fi + fo)))
        parts.append(rng.uniform(-lim, lim, size=(fo, fi, 3, 3)).astype(np.float32).ravel())
        parts.append(np.full(fo, bias, dtype=np.float32))
    w = np.concatenate(parts)
    assert w.size == CNN_NPARAM
    return w


def cnn_scales(gamma=GAMMA, rho_ref=1.4, p_ref=1.0, out_factor=1.0e-3):
    """in_scale of (rho, rho u_n, rho u_t, E) and out_scale of the flux, from the pre-shock state."""
    a = math.sqrt(gamma * p_ref / rho_ref)
    in_scale = np.array([rho_ref, rho_ref * a, rho_ref * a, p_ref / (gamma - 1.0)])
    out_scale = out_factor * np.array([rho_ref * a, rho_ref * a * a, rho_ref * a * a, rho_ref * a ** 3])
    return in_scale, out_scale


def batch_cases(n=16, seed=16, nx=1024, ny=512):
    """Config 5: n independent shock-cylinder cases with Mach ~ U[1.5, 3] (seeded)."""
    rng = np.random.default_rng(seed)
    return [shock_cylinder(nx, ny, Ms=float(m), name=f"batch{k}_{nx}x{ny}")
            for k, m in enumerate(rng.uniform(1.5, 3.0, size=n))]
