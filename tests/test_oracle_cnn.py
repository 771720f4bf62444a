"""Pins of the oracle's CNN neural flux (O11; Eq. 11-13; readings R18-R20).  -m "not gpu".

The CUDA path of this row is not built yet: the oracle comes first and is pinned
here against the paper's parameter count, a library convolution, and the structure Eq. 11-13 prescribe."""
import os

import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))
PER = dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic")


def split(w):
    out, o = [], 0
    for fo, fi in wl.CNN_SIZES:
        out.append(w[o:o + fo * fi * 9].reshape(fo, fi, 3, 3)); o += fo * fi * 9
        out.append(w[o:o + fo]); o += fo
    return out


def torch_cnn(w, x, bf16=False):
    """three library convolutions (zero padding 1), ReLU, ReLU, tanh, in float64"""
    W1, b1, W2, b2, W3, b3 = [torch.tensor(np.asarray(a, dtype=np.float64)) for a in split(w)]
    r = (lambda t: t.to(torch.bfloat16).to(torch.float64)) if bf16 else (lambda t: t)
    h = r(torch.tensor(x)[None])
    h = r(torch.relu(torch.nn.functional.conv2d(h, r(W1), b1, padding=1)))
    h = r(torch.relu(torch.nn.functional.conv2d(h, r(W2), b2, padding=1)))
    return torch.tanh(torch.nn.functional.conv2d(h, r(W3), b3, padding=1))[0].numpy()


def make(case, w=None, scales=None, bf16=False):
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"])
    if w is not None:
        o.set_flux_cnn(w, *(scales or wl.cnn_scales(out_factor=0.05)), emulate_bf16=bf16)
    return o


def test_parameter_count_is_the_papers():
    want = int(open(os.path.join(HERE, "golden", "paper_l94_cnn_parameters.txt")).read().split("parameters")[-1])
    assert wl.CNN_NPARAM == want == 1184 + 4624 + 580
    assert wl.cnn_weights().shape == (want,)


@pytest.mark.parametrize("bf16", [False, True])
def test_network_equals_three_library_convolutions(bf16):
    rng = np.random.default_rng(3)
    w = wl.cnn_weights(11, bias=0.0)
    w += rng.uniform(-0.05, 0.05, w.shape).astype(np.float32)  # non-zero biases too
    o = make(wl.vortex(16), w, bf16=bf16)
    for shape in ((4, 7, 13), (4, 1, 5), (4, 12, 3)):
        x = rng.normal(size=shape)
        got, want = o.cnn_apply(x), torch_cnn(w, x, bf16)
        assert np.abs(got - want).max() <= (2e-2 if bf16 else 1e-13)  # bf16: a hidden value may round the other way
    assert np.abs(o.cnn_apply(x)).max() < 1.0  # tanh output


def test_zero_network_is_bitwise_neutral_and_disable_works():
    case = wl.shock_cylinder(96, 48, Ms=2.0)
    o = make(case)
    o.set_ibm(case["phi"])
    L0 = o.rhs(case["U0"])
    o.set_flux_cnn(np.zeros(wl.CNN_NPARAM, np.float32), *wl.cnn_scales())
    assert np.array_equal(o.rhs(case["U0"]), L0)
    o.set_flux_cnn(wl.cnn_weights(), *wl.cnn_scales(out_factor=1.0))
    assert np.abs(o.rhs(case["U0"]) - L0).max() > 1e-3
    o.set_flux_cnn(None)
    assert np.array_equal(o.rhs(case["U0"]), L0)


def test_bias_only_network_adds_a_constant_flux():
    """all kernels zero: every face gets out_scale * tanh(b3) -> its divergence vanishes"""
    case = wl.vortex(24)
    w = np.zeros(wl.CNN_NPARAM, np.float32)
    w[-4:] = (0.3, -0.2, 0.5, 0.1)
    L0, L1 = make(case).rhs(case["U0"]), make(case, w).rhs(case["U0"])
    assert np.abs(L1 - L0).max() <= 1e-12 * np.abs(L0).max()


def test_assembly_on_a_uniform_state():
    """uniform flow: both reconstructed states are the cell state, so the input field is the constant
    (rho, rho u_n, rho u_t, E) / in_scale and Eq. 11 reduces to L = -div(out_scale o CNN(constant field)); the zero
    padding makes that field non-constant near the borders, which exercises every index of the assembly, the
    normal/tangential ordering of y-faces and the momentum slots."""
    nx, ny, g = 12, 9, 1.4
    rho, u, v, p = 1.3, 0.4, -0.7, 0.9
    case = dict(nx=nx, ny=ny, dx=0.1, dy=0.2, gamma=g, mu=0.0, Pr=0.72, bc=PER, phi=None,
                U0=wl.cons_from_prim(np.full((ny, nx), rho), np.full((ny, nx), u), np.full((ny, nx), v), np.full((ny, nx), p)))
    w = wl.cnn_weights(4, bias=0.01)
    ins, outs = wl.cnn_scales(out_factor=1.0)
    o = make(case, w, (ins, outs))
    L = o.rhs(case["U0"])
    E = p / (g - 1) + 0.5 * rho * (u * u + v * v)
    Xx = np.empty((4, ny, nx + 1)); Xy = np.empty((4, nx, ny + 1))
    for k, val in enumerate((rho, rho * u, rho * v, E)):
        Xx[k] = val / ins[k]
    for k, val in enumerate((rho, rho * v, rho * u, E)):  # normal first
        Xy[k] = val / ins[k]
    Yx, Yy = torch_cnn(w, Xx), torch_cnn(w, Xy)
    want = np.zeros((4, ny, nx))
    for k in range(4):
        want[k] -= outs[k] * (Yx[k][:, 1:] - Yx[k][:, :-1]) / case["dx"]
    for k, slot in enumerate((0, 2, 1, 3)):  # (mass, normal = rho v, tangential = rho u, energy)
        want[slot] -= outs[k] * (Yy[k][:, 1:] - Yy[k][:, :-1]).T / case["dy"]
    assert np.abs(L - want).max() <= 1e-11 * np.abs(want).max()
    assert np.abs(want).max() > 1e-3


def test_shared_weights_make_the_scheme_transposition_invariant():
    """Eq. 13: x- and y-faces use the same network on (tangential, normal) fields, so swapping the axes of the
    problem (and u with v) swaps them in the result"""
    rng = np.random.default_rng(8)
    nx, ny = 14, 10
    X, Y = np.meshgrid((np.arange(nx) + 0.5) / nx, (np.arange(ny) + 0.5) / ny)
    rho = 1 + 0.2 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y)
    u = 0.3 + 0.1 * np.cos(2 * np.pi * (X + Y)); v = -0.2 + 0.1 * np.sin(4 * np.pi * X)
    p = 1 + 0.1 * np.cos(2 * np.pi * Y)
    bc = dict(xlo="transmissive", xhi="reflective", ylo="periodic", yhi="periodic")
    bcT = dict(ylo="transmissive", yhi="reflective", xlo="periodic", xhi="periodic")
    a = dict(nx=nx, ny=ny, dx=0.05, dy=0.08, gamma=1.4, mu=0.0, Pr=0.72, bc=bc, phi=None, U0=wl.cons_from_prim(rho, u, v, p))
    b = dict(nx=ny, ny=nx, dx=0.08, dy=0.05, gamma=1.4, mu=0.0, Pr=0.72, bc=bcT, phi=None,
             U0=wl.cons_from_prim(rho.T, v.T, u.T, p.T))
    w = wl.cnn_weights(21, bias=0.02)
    La, Lb = make(a, w).rhs(a["U0"]), make(b, w).rhs(b["U0"])
    for ka, kb in ((0, 0), (1, 2), (2, 1), (3, 3)):
        assert np.abs(La[ka] - Lb[kb].T).max() <= 1e-12 * np.abs(La).max()
    assert np.abs(La - make(a).rhs(a["U0"])).max() > 1e-6  # the network is really in the loop


def test_argument_checks():
    o = make(wl.vortex(16))
    w = wl.cnn_weights()
    ins, outs = wl.cnn_scales()
    bad = w.copy(); bad[5] = np.nan
    with pytest.raises(jxo.OracleError):
        o.set_flux_cnn(bad, ins, outs)
    with pytest.raises(jxo.OracleError):
        o.set_flux_cnn(w, np.array([1, 0, 1, 1.0]), outs)
    with pytest.raises(jxo.OracleError):
        o.cnn_apply(np.zeros((4, 3, 3)))  # no network set
