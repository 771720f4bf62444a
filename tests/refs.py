"""Independent yardsticks for pinning the oracle (test-only; imports neither oracle/ nor the CUDA path).

  * exact Riemann solver for the 1D Euler equations (Newton iteration on the
    pressure function — textbook construction, Toro ch. 4),
  * WENO5 built from its DEFINITION: quadratic reconstruction polynomials of the
    three sub-stencils, Jiang-Shu smoothness indicators as integrals of squared
    derivatives, linear weights derived by matching the 5-cell quartic,
  * HLLC in Toro's flux form F* = (s*(s_k U - F) + s_k p* D)/(s_k - s*), which is
    algebraically equivalent to but differently arranged from PAPER.md Eq. 3-4,
  * a brute-force per-cell evaluator of L(U) through index-mapped boundaries,
  * the analytic Navier-Stokes viscous operator by FFT differentiation.
"""
import math

import numpy as np
from numpy.polynomial import polynomial as Pn


# ----------------------------------------------------------------------------
# exact Riemann solver (ideal gas)
# ----------------------------------------------------------------------------
def _pressure_fn(p, rk, pk, ak, g):
    if p > pk:  # shock
        A = 2.0 / ((g + 1.0) * rk)
        B = (g - 1.0) / (g + 1.0) * pk
        f = (p - pk) * math.sqrt(A / (p + B))
        df = math.sqrt(A / (B + p)) * (1.0 - 0.5 * (p - pk) / (B + p))
    else:  # rarefaction
        f = 2.0 * ak / (g - 1.0) * ((p / pk) ** ((g - 1.0) / (2.0 * g)) - 1.0)
        df = 1.0 / (rk * ak) * (p / pk) ** (-(g + 1.0) / (2.0 * g))
    return f, df


def riemann_star(rl, ul, pl, rr, ur, pr, g=1.4):
    al, ar = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    p = max(1e-8, 0.5 * (pl + pr))
    for _ in range(100):
        fl, dfl = _pressure_fn(p, rl, pl, al, g)
        fr, dfr = _pressure_fn(p, rr, pr, ar, g)
        pn = max(1e-12, p - (fl + fr + ur - ul) / (dfl + dfr))
        if abs(pn - p) < 1e-15 * max(p, pn):
            p = pn
            break
        p = pn
    fl, _ = _pressure_fn(p, rl, pl, al, g)
    fr, _ = _pressure_fn(p, rr, pr, ar, g)
    u = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    return p, u


def riemann_sample(xi, rl, ul, pl, rr, ur, pr, g=1.4):
    """(rho,u,p) of the exact solution at similarity coordinate xi = x/t (vectorised over xi)."""
    ps, us = riemann_star(rl, ul, pl, rr, ur, pr, g)
    al, ar = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    xi = np.asarray(xi, dtype=np.float64)
    rho, u, p = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    gm, gp = g - 1.0, g + 1.0
    for n, s in enumerate(xi.ravel()):
        if s <= us:  # left of the contact
            if ps > pl:  # left shock
                sl = ul - al * math.sqrt(gp / (2 * g) * ps / pl + gm / (2 * g))
                if s <= sl:
                    w = (rl, ul, pl)
                else:
                    w = (rl * ((ps / pl + gm / gp) / (gm / gp * ps / pl + 1.0)), us, ps)
            else:  # left rarefaction
                shl = ul - al
                asl = al * (ps / pl) ** (gm / (2 * g))
                stl = us - asl
                if s <= shl:
                    w = (rl, ul, pl)
                elif s >= stl:
                    w = (rl * (ps / pl) ** (1.0 / g), us, ps)
                else:
                    c = 2.0 / gp + gm / (gp * al) * (ul - s)
                    w = (rl * c ** (2.0 / gm), 2.0 / gp * (al + gm / 2.0 * ul + s), pl * c ** (2.0 * g / gm))
        else:
            if ps > pr:  # right shock
                sr = ur + ar * math.sqrt(gp / (2 * g) * ps / pr + gm / (2 * g))
                if s >= sr:
                    w = (rr, ur, pr)
                else:
                    w = (rr * ((ps / pr + gm / gp) / (gm / gp * ps / pr + 1.0)), us, ps)
            else:
                shr = ur + ar
                asr = ar * (ps / pr) ** (gm / (2 * g))
                str_ = us + asr
                if s >= shr:
                    w = (rr, ur, pr)
                elif s <= str_:
                    w = (rr * (ps / pr) ** (1.0 / g), us, ps)
                else:
                    c = 2.0 / gp - gm / (gp * ar) * (ur - s)
                    w = (rr * c ** (2.0 / gm), 2.0 / gp * (-ar + gm / 2.0 * ur + s), pr * c ** (2.0 * g / gm))
        rho.flat[n], u.flat[n], p.flat[n] = w
    return rho, u, p


# ----------------------------------------------------------------------------
# WENO5 from its definition
# ----------------------------------------------------------------------------
def _poly_from_averages(cells, avgs):
    """Polynomial (ascending coeffs) of degree len(cells)-1 whose averages over the unit cells
    centred at `cells` equal `avgs`."""
    n = len(cells)
    A = np.zeros((n, n))
    for r, c in enumerate(cells):
        for k in range(n):
            A[r, k] = ((c + 0.5) ** (k + 1) - (c - 0.5) ** (k + 1)) / (k + 1)
    return np.linalg.solve(A, np.asarray(avgs, dtype=np.float64))


def _smoothness(coef):
    """Jiang-Shu indicator: sum_l int_{-1/2}^{1/2} (d^l p/dx^l)^2 dx, l = 1.. (h = 1)."""
    beta = 0.0
    d = np.array(coef, dtype=np.float64)
    for _ in range(len(coef) - 1):
        d = Pn.polyder(d)
        sq = Pn.polyint(Pn.polymul(d, d))
        beta += Pn.polyval(0.5, sq) - Pn.polyval(-0.5, sq)
    return beta


_LINEAR_W = None


def weno_linear_weights():
    """d_k such that sum_k d_k q_k equals the 5-cell quartic's value at x = 1/2 for all data."""
    global _LINEAR_W
    if _LINEAR_W is None:
        rows, rhs = [], []
        for e in range(5):
            v = np.zeros(5)
            v[e] = 1.0
            q = [Pn.polyval(0.5, _poly_from_averages([k - 2, k - 1, k], v[k:k + 3])) for k in range(3)]
            rows.append(q)
            rhs.append(Pn.polyval(0.5, _poly_from_averages([-2, -1, 0, 1, 2], v)))
        _LINEAR_W = np.linalg.lstsq(np.array(rows), np.array(rhs), rcond=None)[0]
    return _LINEAR_W


def weno5_definition(v, eps=1e-6):
    """Left-biased WENO5-JS value at x_{i+1/2} from cell averages v[i-2..i+2], from the definition."""
    v = np.asarray(v, dtype=np.float64)
    d = weno_linear_weights()
    q, beta = np.zeros(3), np.zeros(3)
    for k in range(3):
        coef = _poly_from_averages([k - 2, k - 1, k], v[k:k + 3])
        q[k] = Pn.polyval(0.5, coef)
        beta[k] = _smoothness(coef)
    alpha = d / (eps + beta) ** 2
    return float(np.dot(alpha, q) / alpha.sum())


# ----------------------------------------------------------------------------
# HLLC, Toro's arrangement
# ----------------------------------------------------------------------------
def euler_flux_x(W, g):
    r, u, v, p = W
    E = p / (g - 1.0) + 0.5 * r * (u * u + v * v)
    return np.array([r * u, r * u * u + p, r * u * v, u * (E + p)]), np.array([r, r * u, r * v, E])


def hllc_toro(WL, WR, g):
    FL, UL = euler_flux_x(WL, g)
    FR, UR = euler_flux_x(WR, g)
    rl, ul, _, pl = WL
    rr, ur, _, pr = WR
    al, ar = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    sl, sr = min(ul - al, ur - ar), max(ul + al, ur + ar)
    ss = (pr - pl + rl * ul * (sl - ul) - rr * ur * (sr - ur)) / (rl * (sl - ul) - rr * (sr - ur))
    if sl >= 0:
        return FL
    if sr <= 0:
        return FR

    def star(F, U, W, sk):
        r, u, _, p = W
        pstar = p + r * (sk - u) * (ss - u)
        D = np.array([0.0, 1.0, 0.0, ss])
        return (ss * (sk * U - F) + sk * pstar * D) / (sk - ss)

    if ss > 0:
        return star(FL, UL, WL, sl)
    if ss < 0:
        return star(FR, UR, WR, sr)
    return 0.5 * (star(FL, UL, WL, sl) + star(FR, UR, WR, sr))


# ----------------------------------------------------------------------------
# brute-force per-cell L(U) through index-mapped boundaries (Euler, no IBM)
# ----------------------------------------------------------------------------
def _map_index(i, n, lo, hi):
    """-> (interior index or None for inflow, sign of the wall-normal momentum)."""
    if 0 <= i < n:
        return i, 1.0
    if i < 0:
        kind, g = lo, -i
        if kind == "periodic":
            return n - g, 1.0
        if kind == "transmissive":
            return 0, 1.0
        if kind == "reflective":
            return g - 1, -1.0
        return None, 1.0
    kind, g = hi, i - (n - 1)
    if kind == "periodic":
        return g - 1, 1.0
    if kind == "transmissive":
        return n - 1, 1.0
    if kind == "reflective":
        return n - g, -1.0
    return None, 1.0


def prim_mapped(U, i, j, bc, g):
    """Primitive state of (possibly ghost) cell (i,j): x-map for rows inside the domain,
    y-map applied on top for rows outside (x sides first, then y sides over the extended range)."""
    _, ny, nx = U.shape
    jj, sy = _map_index(j, ny, bc["ylo"], bc["yhi"])
    if jj is None:
        r, u, v, p = bc["inflow"]
        return np.array([r, u, v, p])
    ii, sx = _map_index(i, nx, bc["xlo"], bc["xhi"])
    if ii is None:
        r, u, v, p = bc["inflow"]
        return np.array([r, u, sy * v, p])
    r, ru, rv, E = U[:, jj, ii]
    u, v = sx * ru / r, sy * rv / r
    p = (g - 1.0) * (E - 0.5 * r * (u * u + v * v))
    return np.array([r, u, v, p])


def rhs_cell_bruteforce(U, i, j, dx, dy, bc, g):
    """L(U) at interior cell (i,j) from scratch: four faces, each from its own 6-cell stencil."""

    def face(axis, f):  # face between cell f and f+1 along axis, through cell (i,j)
        cells = [prim_mapped(U, f + o, j, bc, g) if axis == 0 else prim_mapped(U, i, f + o, bc, g)
                 for o in range(-2, 4)]
        W = np.array(cells)  # [6][4]
        if axis == 1:
            W = W[:, [0, 2, 1, 3]]
        WL = np.array([weno5_definition(W[0:5, k]) for k in range(4)])
        WR = np.array([weno5_definition(W[5:0:-1, k]) for k in range(4)])
        F = hllc_toro(WL, WR, g)
        if axis == 1:
            F = F[[0, 2, 1, 3]]
        return F

    return -(face(0, i) - face(0, i - 1)) / dx - (face(1, j) - face(1, j - 1)) / dy


# ----------------------------------------------------------------------------
# analytic Navier-Stokes viscous operator on a periodic box by FFT differentiation
# ----------------------------------------------------------------------------
def _ddx(f, Lx):
    k = 2j * np.pi * np.fft.fftfreq(f.shape[1], d=Lx / f.shape[1])
    return np.real(np.fft.ifft(np.fft.fft(f, axis=1) * k[None, :], axis=1))


def _ddy(f, Ly):
    k = 2j * np.pi * np.fft.fftfreq(f.shape[0], d=Ly / f.shape[0])
    return np.real(np.fft.ifft(np.fft.fft(f, axis=0) * k[:, None], axis=0))


def viscous_operator_spectral(rho, u, v, p, Lx, Ly, mu, Pr, g):
    """div of the viscous flux (0, tau_x., tau_y., u.tau + k grad T), Stokes hypothesis, T = p/rho."""
    ux, uy, vx, vy = _ddx(u, Lx), _ddy(u, Ly), _ddx(v, Lx), _ddy(v, Ly)
    T = p / rho
    kap = mu * g / ((g - 1.0) * Pr)
    txx = mu * (4.0 / 3.0 * ux - 2.0 / 3.0 * vy)
    tyy = mu * (4.0 / 3.0 * vy - 2.0 / 3.0 * ux)
    txy = mu * (uy + vx)
    ex = u * txx + v * txy + kap * _ddx(T, Lx)
    ey = u * txy + v * tyy + kap * _ddy(T, Ly)
    return np.stack([np.zeros_like(u), _ddx(txx, Lx) + _ddy(txy, Ly), _ddx(txy, Lx) + _ddy(tyy, Ly),
                     _ddx(ex, Lx) + _ddy(ey, Ly)])
