"""Pins for the oracle's pointwise pieces: WENO5 (O4), HLLC (O5), RH initial data, bf16 rounding.

None of these retypes the oracle's formula: they use the definition (reconstruction
polynomials), closed forms, jump conditions and special cases.  -m "not gpu".
"""
import math
import os

import numpy as np
import pytest
import torch

import refs
from oracle import jxo
from paper_2601_04400_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
G = 1.4


def _golden(name):
    rows = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            rows[k] = [float(x) for x in v]
    return rows


# ------------------------------------------------------------------ WENO5 (O4)
def test_weno_linear_weights_are_the_classical_ones():
    # BASELINE.json configs[0]: linear weights 0.1/0.6/0.3 — here derived from the 5-cell quartic
    assert np.allclose(refs.weno_linear_weights(), [0.1, 0.6, 0.3], atol=1e-12)


def test_weno_constant_and_quadratic_data_exact():
    assert jxo.weno5([3.25] * 5) == 3.25
    # cell averages of a quadratic: every sub-stencil reproduces p(1/2) exactly, whatever the weights
    coef = np.array([0.7, -1.3, 0.45])
    avg = []
    for c in range(-2, 3):
        F = np.polynomial.polynomial.polyint(coef)
        avg.append(np.polynomial.polynomial.polyval(c + 0.5, F) - np.polynomial.polynomial.polyval(c - 0.5, F))
    exact = np.polynomial.polynomial.polyval(0.5, coef)
    assert abs(jxo.weno5(avg) - exact) < 1e-14


def test_weno_matches_definition_on_random_data():
    rng = np.random.default_rng(7)
    for scale in (1.0, 1e-2, 1e-4, 30.0):
        for _ in range(40):
            v = 1.0 + scale * rng.standard_normal(5)
            a, b = jxo.weno5(v), refs.weno5_definition(v)
            assert abs(a - b) <= 2e-12 * max(1.0, np.abs(v).max()), (v, a, b)


def test_weno_essentially_non_oscillatory_at_a_step():
    # stencil (0,0,0,1,1): the smooth sub-stencil wins, no overshoot beyond O(eps)
    assert abs(jxo.weno5([0, 0, 0, 1, 1])) < 1e-3
    assert abs(jxo.weno5([1, 1, 1, 0, 0]) - 1.0) < 1e-3
    assert abs(jxo.weno5([0, 0, 1, 1, 1]) - 1.0) < 1e-3


def test_weno_fifth_order_on_exact_line_averages():
    # reading R16: fifth order applies to the reconstruction operator fed exact cell averages
    errs = []
    k = 2 * math.pi
    for n in (40, 80, 160):
        h = 1.0 / n
        worst = 0.0
        for x0 in np.linspace(0, 1, 37, endpoint=False):  # cell i = [x0, x0+h], face at x0+h
            edges = np.arange(-2, 4) * h + x0
            avg = -(np.cos(k * edges[1:]) - np.cos(k * edges[:-1])) / (k * h) + 2.0  # averages of 2+sin(kx)
            worst = max(worst, abs(jxo.weno5(avg) - (2.0 + math.sin(k * (x0 + h)))))
        errs.append(worst)
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert min(orders) > 4.8, (errs, orders)


# ------------------------------------------------------------------- HLLC (O5)
def _flux(W):
    return refs.euler_flux_x(W, G)[0]


def test_hllc_consistency():
    rng = np.random.default_rng(3)
    for _ in range(50):
        W = np.array([rng.uniform(0.1, 5), rng.uniform(-3, 3), rng.uniform(-3, 3), rng.uniform(0.1, 5)])
        F = jxo.hllc(W, W, G)
        assert np.allclose(F, _flux(W), rtol=1e-13, atol=1e-13)


def test_hllc_supersonic_upwinding_is_exact():
    WL, WR = np.array([1.0, 3.0, 0.2, 1.0]), np.array([0.8, 2.8, -0.1, 0.9])
    assert np.array_equal(jxo.hllc(WL, WR, G), _flux(WL))  # sL >= 0
    WL2, WR2 = WL * [1, -1, 1, 1], WR * [1, -1, 1, 1]
    assert np.array_equal(jxo.hllc(WR2, WL2, G), _flux(WL2))  # sR <= 0


def test_hllc_stationary_contact_exact():
    F = jxo.hllc([1.0, 0.0, 0.0, 0.7], [0.125, 0.0, 0.0, 0.7], G)
    assert np.array_equal(F, [0.0, 0.7, 0.0, 0.0])


def test_hllc_moving_contact_is_upwinded():
    WL, WR = np.array([1.0, 0.4, 0.3, 1.0]), np.array([0.3, 0.4, -0.2, 1.0])
    assert np.allclose(jxo.hllc(WL, WR, G), _flux(WL), rtol=1e-14, atol=1e-15)
    WL[1] = WR[1] = -0.4
    assert np.allclose(jxo.hllc(WL, WR, G), _flux(WR), rtol=1e-14, atol=1e-15)


def test_hllc_star_states_satisfy_the_jump_conditions():
    """F_k + s_k (U*_k - U_k) = s* U*_k + p* (0,1,0,s*) with ONE p* for both sides.
    This is what rejects the energy entry printed in Eq. 4 (reading R1)."""
    rng = np.random.default_rng(11)
    for _ in range(50):
        WL = np.array([rng.uniform(0.2, 3), rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(0.2, 3)])
        WR = np.array([rng.uniform(0.2, 3), rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(0.2, 3)])
        (sL, sR, sS), UsL, UsR = jxo.hllc_star(WL, WR, G)
        pstar = []
        for W, Us, sk in ((WL, UsL, sL), (WR, UsR, sR)):
            F, U = refs.euler_flux_x(W, G)
            ps = W[3] + W[0] * (sk - W[1]) * (sS - W[1])
            pstar.append(ps)
            lhs = F + sk * (Us - U)
            rhs = sS * Us + ps * np.array([0.0, 1.0, 0.0, sS])
            assert np.allclose(lhs, rhs, rtol=1e-12, atol=1e-12), (WL, WR)
            assert abs(Us[1] / Us[0] - sS) < 1e-13  # star velocity is s*
            assert abs(Us[2] / Us[0] - W[2]) < 1e-13  # tangential velocity carried
        assert abs(pstar[0] - pstar[1]) < 1e-12 * max(1.0, abs(pstar[0]))  # Eq. 7


def test_hllc_equals_toro_flux_form():
    rng = np.random.default_rng(5)
    for _ in range(200):
        WL = np.array([rng.uniform(0.2, 3), rng.uniform(-2, 2), rng.uniform(-1, 1), rng.uniform(0.2, 3)])
        WR = np.array([rng.uniform(0.2, 3), rng.uniform(-2, 2), rng.uniform(-1, 1), rng.uniform(0.2, 3)])
        a, b = jxo.hllc(WL, WR, G), refs.hllc_toro(WL, WR, G)
        assert np.allclose(a, b, rtol=1e-12, atol=1e-12), (WL, WR, a, b)


def test_hllc_mirror_symmetry():
    WL, WR = np.array([1.0, 0.3, 0.2, 1.0]), np.array([0.5, -0.1, 0.4, 0.6])
    F = jxo.hllc(WL, WR, G)
    Fm = jxo.hllc(WR * [1, -1, 1, 1], WL * [1, -1, 1, 1], G)
    assert np.allclose(Fm, F * [-1, 1, -1, -1], rtol=1e-14, atol=1e-15)


# ------------------------------------------------------------ exact solver + RH
def test_exact_riemann_solver_reproduces_textbook_sod_values():
    g17, tb = _golden("paper_eq17_sod_states.txt"), _golden("sod_exact_textbook.txt")
    (rl, ul, pl, _), (rr, ur, pr, _) = g17["L"], g17["R"]
    ps, us = refs.riemann_star(rl, ul, pl, rr, ur, pr, G)
    assert abs(ps - tb["p_star"][0]) < 6e-6 and abs(us - tb["u_star"][0]) < 6e-6
    r, _, _ = refs.riemann_sample(np.array([us - 1e-6, us + 1e-6]), rl, ul, pl, rr, ur, pr, G)
    assert abs(r[0] - tb["rho_star_L"][0]) < 6e-6 and abs(r[1] - tb["rho_star_R"][0]) < 6e-6


def test_rankine_hugoniot_reproduces_paper_eq18():
    g18 = _golden("paper_eq18_shock_states.txt")
    rho2, u2, p2, W = wl.rankine_hugoniot(5.0, rho1=g18["pre"][0], p1=g18["pre"][3], gamma=g18["pre"][4])
    assert abs(rho2 - g18["post"][0]) < 1e-12 and abs(u2 - g18["post"][1]) < 1e-12
    assert abs(p2 - g18["post"][3]) < 1e-12 and abs(W - g18["shock_speed"][0]) < 1e-12


# -------------------------------------------------------------- bf16 rounding
def test_bf16_rounding_matches_torch():
    """The emulating MLP's weight rounding, read back through a saturated path, equals torch's bf16 cast:
    b2[0] = 20 makes h2[0] = bf16(tanh(20)) = 1, so y0 = bf16(W3[0][0]); biases stay fp32 (b3[1] = 1)."""
    o = jxo.Oracle(8, 8, 1.0, 1.0, bc=dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic"))
    off_b2, off_w3, off_b3 = 64 * 24 + 64 + 64 * 64, 64 * 24 + 64 + 64 * 64 + 64, 64 * 24 + 64 + 64 * 64 + 64 + 4 * 64
    for val in np.random.default_rng(0).standard_normal(64).astype(np.float32):
        w = np.zeros(6020, dtype=np.float32)
        w[off_b2] = 20.0
        w[off_w3] = val
        w[off_b3 + 1] = 1.0
        o.set_flux_mlp(w, np.ones(4), np.ones(4), emulate_bf16=True)
        y = o.mlp_eval(np.zeros(24))
        want = float(torch.tensor(val, dtype=torch.float32).to(torch.bfloat16).to(torch.float32))
        assert y[0] == want and y[1] == 1.0
