"""S5' — per-face MLP flux correction on the tensor cores (tcgen05) versus the oracle.  -m gpu.

BASELINE.json: the bf16 / fp32-accumulate network is held to <= 1e-2 relative on the flux correction,
against the oracle's bf16-emulating mode (same rounding points, wide accumulation).
"""
import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL_MLP = 1e-2


def jxs():
    from paper_2601_04400_b200 import jxs as m
    return m


def make_pair(case, w, ins, outs, dtype=torch.float64):
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"])
    s = jxs().Solver.from_case(case, dtype=dtype)
    if case.get("phi") is not None:
        o.set_ibm(case["phi"])
    o.set_flux_mlp(w, ins, outs, emulate_bf16=True)
    s.set_flux_mlp(w, ins, outs)
    return o, s


def dev(U, dtype=torch.float64):
    return torch.tensor(np.ascontiguousarray(U), dtype=dtype, device="cuda")


def oracle_face_inputs(o, U, ins):
    """The 24 network inputs of every face, assembled from the oracle's own ghost-filled state (R14)."""
    Up = o.fill_ghosts(U).astype(np.float64)  # [4][ny+6][nx+6]
    r = Up[0]
    W = np.stack([r, Up[1] / r, Up[2] / r, (wl.GAMMA - 1.0) * (Up[3] - 0.5 * (Up[1] ** 2 + Up[2] ** 2) / r)])
    ny, nx = U.shape[1], U.shape[2]
    # x-face f of row j: cells f-3..f+2 (interior index) = padded columns f..f+5
    X = np.empty((ny, nx + 1, 24))
    for cc in range(6):
        for k in range(4):
            X[:, :, 4 * cc + k] = W[k][3:ny + 3, cc:cc + nx + 1] / ins[k]
    # y-face f of column i: rows f-3..f+2 = padded rows f..f+5, normal velocity first (rho, v, u, p)
    Y = np.empty((ny + 1, nx, 24))
    perm = (0, 2, 1, 3)
    for cc in range(6):
        for k in range(4):
            Y[:, :, 4 * cc + k] = W[perm[k]][cc:cc + ny + 1, 3:nx + 3] / ins[k]
    return X, Y


def rel_net(a, b, outs):
    """Error of the correction in the network's own output units (Delta F / out_scale), max-norm over all
    faces and components, relative to the max-norm of the expected output.  (One scale for the four
    outputs: a single output can be accidentally tiny on every face of a nearly uniform field.)"""
    a, b = a / outs[:, None], b / outs[:, None]
    return np.max(np.abs(a - b)) / np.max(np.abs(b))


def rel_fields(a, b, zero_tol=1e-6):
    """max-norm error of each component, scaled by that component's max; a momentum component that holds only
    round-off (below zero_tol of the other) borrows the other's scale."""
    peak = [np.max(np.abs(b[k])) for k in range(4)]
    mom = max(peak[1], peak[2])
    scale = [peak[0], peak[1] if peak[1] > zero_tol * mom else mom, peak[2] if peak[2] > zero_tol * mom else mom, peak[3]]
    return [np.max(np.abs(a[k] - b[k])) / scale[k] for k in range(4)]


def rel(a, b):
    return max(rel_fields(a, b))


CASES = {
    "shock_cylinder_256x128": lambda: wl.shock_cylinder(256, 128, Ms=2.0),
    "shock_cylinder_ragged_301x77": lambda: wl.shock_cylinder(301, 77, Ms=2.5, bodies=((0.5, 0.5, 0.12),)),
    "vortex_64": lambda: wl.vortex(64),
    # the smallest grid the library takes (one strip of 9 face columns, 9 face rows) and two lopsided ones: a strip and a
    # half wide with 10 rows (every CTA starts and ends inside its pipeline's warm-up), 17 columns with 151 rows
    "tiny_8x8": lambda: wl.vortex(8),
    "wide_190x9": lambda: _smooth(190, 9),
    "thin_16x150": lambda: _smooth(16, 150),
}


def _smooth(nx, ny):
    from test_gpu_parity import MIXED, smooth_case
    return smooth_case(nx, ny, 3, MIXED, mu=2e-3, jump=True)


@pytest.mark.parametrize("name", list(CASES))
def test_flux_correction_per_face(name):
    """Delta F of jxs_flux_correction against the oracle's network evaluated face by face (sampled)."""
    case = CASES[name]()
    w, (ins, outs) = wl.mlp_weights(7), wl.mlp_scales()
    brng = np.random.default_rng(11)
    for lo, hi in ((1536, 1600), (5696, 5760), (6016, 6020)):  # b1, b2, b3: non-zero
        w[lo:hi] = brng.uniform(-0.2, 0.2, hi - lo).astype(np.float32)
    o, s = make_pair(case, w, ins, outs)
    U = case["U0"]
    if "cylinder" in name:  # a developed field: reflected shock, IBM ghosts in the stencils
        o.set_flux_mlp(None)
        U = o.step(U, 0.4, 40)
        o.set_flux_mlp(w, ins, outs, emulate_bf16=True)
    dFx, dGy = (a.cpu().numpy().astype(np.float64) for a in s.flux_correction(dev(U)))
    X, Y = oracle_face_inputs(o, U, ins)
    ny, nx = case["ny"], case["nx"]
    rng = np.random.default_rng(0)
    # all faces of a few rows / columns (tile edges included) plus a random sample
    fx = [(j, f) for j in (0, 1, ny // 2, ny - 1) for f in range(nx + 1)] + \
         [(int(rng.integers(ny)), int(rng.integers(nx + 1))) for _ in range(3000)]
    fy = [(f, i) for f in (0, 1, ny // 2, ny) for i in range(nx)] + \
         [(int(rng.integers(ny + 1)), int(rng.integers(nx))) for _ in range(3000)]
    ex = np.array([o.mlp_eval(X[j, f]) * outs for j, f in fx]).T          # (mass, normal, tangential, energy)
    ey = np.array([o.mlp_eval(Y[f, i]) * outs for f, i in fy]).T[[0, 2, 1, 3]]  # -> (rho, rho u, rho v, E)
    gx = np.array([dFx[:, j, f] for j, f in fx]).T
    gy = np.array([dGy[:, f, i] for f, i in fy]).T
    ex_scale, ey_scale = outs, outs[[0, 2, 1, 3]]
    assert rel_net(gx, ex, ex_scale) <= TOL_MLP, (name, rel_net(gx, ex, ex_scale))
    assert rel_net(gy, ey, ey_scale) <= TOL_MLP, (name, rel_net(gy, ey, ey_scale))


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_rhs_with_mlp(dtype):
    """The correction as it enters the RHS: L(with network) - L(without) on both sides."""
    case = wl.shock_cylinder(256, 128, Ms=2.0)
    w, (ins, outs) = wl.mlp_weights(7), wl.mlp_scales(out_factor=1e-1)
    o, s = make_pair(case, w, ins, outs, dtype)
    fluid = o.cell_types() == 0
    U = case["U0"]
    with_o = o.rhs(U)
    with_s = s.rhs(dev(U, dtype)).cpu().numpy().astype(np.float64)
    o.set_flux_mlp(None)
    s.set_flux_mlp(None)
    base_o = o.rhs(U)
    base_s = s.rhs(dev(U, dtype)).cpu().numpy().astype(np.float64)
    d_o, d_s = (with_o - base_o)[:, fluid], (with_s - base_s)[:, fluid]
    assert np.abs(d_o).max() > 0
    if dtype == torch.float64:
        assert rel(d_s, d_o) <= TOL_MLP, rel(d_s, d_o)
    # the whole RHS stays within the network's tolerance of the oracle's
    assert rel(with_s[:, fluid], with_o[:, fluid]) <= TOL_MLP


def test_zero_weights_are_bitwise_neutral_and_disable_works():
    case = wl.shock_cylinder(256, 128, Ms=2.0)
    ins, outs = wl.mlp_scales()
    s = jxs().Solver.from_case(case)
    U = dev(case["U0"])
    base = s.rhs(U).clone()
    s.set_flux_mlp(np.zeros(6020, np.float32), ins, outs)
    assert torch.equal(s.rhs(U), base)
    s.set_flux_mlp(wl.mlp_weights(1), ins, outs)
    assert not torch.equal(s.rhs(U), base)
    s.set_flux_mlp(None)
    assert torch.equal(s.rhs(U), base)
    with pytest.raises(jxs().JxsError) as e:
        s.flux_correction(U)
    assert e.value.code == jxs().ESTATE


def test_biases_and_single_paths():
    """Non-zero biases (kept in fp32) and a network with one active path per layer: fixes the operand
    layout of all three layers (a transposed or permuted tile would fail here)."""
    case = wl.vortex(64)
    ins, outs = np.array([1.0, 1.0, 1.0, 1.0]), np.array([1.0, 2.0, 3.0, 4.0])
    rng = np.random.default_rng(3)
    for trial in range(6):
        w = np.zeros(6020, np.float32)
        W1, b1 = w[:1536].reshape(64, 24), w[1536:1600]
        W2, b2 = w[1600:5696].reshape(64, 64), w[5696:5760]
        W3, b3 = w[5760:6016].reshape(4, 64), w[6016:6020]
        i, h1, h2, k = int(rng.integers(24)), int(rng.integers(64)), int(rng.integers(64)), int(rng.integers(4))
        W1[h1, i], W2[h2, h1], W3[k, h2] = 0.75, -1.5, 2.0
        b1[h1], b2[h2], b3[:] = 0.125, -0.3, (0.01, 0.02, 0.03, 0.04)
        o, s = make_pair(case, w, ins, outs)
        dFx, dGy = (a.cpu().numpy().astype(np.float64) for a in s.flux_correction(dev(case["U0"])))
        X, Y = oracle_face_inputs(o, case["U0"], ins)
        for (j, f) in [(0, 0), (5, 17), (63, 64), (31, 32)]:
            e = o.mlp_eval(X[j, f]) * outs
            assert np.allclose(dFx[:, j, f], e, rtol=1e-2, atol=1e-4), (trial, i, h1, h2, k)
        for (f, i2) in [(0, 0), (64, 63), (20, 40)]:
            e = (o.mlp_eval(Y[f, i2]) * outs)[[0, 2, 1, 3]]
            assert np.allclose(dGy[:, f, i2], e, rtol=1e-2, atol=1e-4), (trial, i, h1, h2, k)


def test_steps_with_mlp_stay_close():
    """20 RK3 steps with the network on: GPU vs the bf16-emulating oracle (activations differ at the
    bf16 rounding level every stage, so the bound is the network's, not 1e-9)."""
    case = wl.shock_cylinder(192, 96, Ms=2.0)
    w, (ins, outs) = wl.mlp_weights(7), wl.mlp_scales()
    o, s = make_pair(case, w, ins, outs)
    ref = o.step(case["U0"], 0.4, 20)
    U = dev(case["U0"])
    s.step(U, 0.4, 20)
    fluid = o.cell_types() == 0
    got = U.cpu().numpy()
    e = rel_fields(got[:, fluid], ref[:, fluid])
    # rho, rho u, E: the corrections are 1e-3 of the flux, their 1e-2 errors 1e-5 of it.  rho v exists here only through
    # the network's corrections (the shock has not reached the body), so relative to ITS max it carries the network's bound
    assert max(e[0], e[1], e[3]) <= 1e-4 and e[2] <= 1e-2, e
    assert abs(o.time()[0] - s.time()[0]) <= 1e-6 * o.time()[0]
