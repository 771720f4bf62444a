"""The paper's 2D CNN neural flux on the CUDA path (flux_cnn_kernel.cuh, tcgen05) against the oracle's
bf16-emulating mode (O11; Eq. 11-13; R18-R20).  -m gpu.  Tolerance: BASELINE.json's bound for the
neural flux correction, 1e-2 relative."""
import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import dev, jxs, rel_err, smooth_case, MIXED

pytestmark = pytest.mark.gpu

CASES = {
    "vortex_48": lambda: wl.vortex(48),
    "jumps_mixed_bc_300x70": lambda: smooth_case(300, 70, 2, MIXED, mu=5e-3, jump=True),   # 3 strips of 124 output faces
    "shock_cylinder_256x136": lambda: wl.shock_cylinder(256, 136, Ms=2.0),                 # IBM, exactly 2 strips in y
    "tiny_8x8": lambda: wl.vortex(8),                                                      # the smallest grid the library takes
    "strip_edge_124x9": lambda: smooth_case(124, 9, 4, MIXED, mu=5e-3),                    # 125 x-faces: a second strip of one face
    "thin_16x150": lambda: smooth_case(16, 150, 5, MIXED, mu=5e-3),                        # one narrow strip, several row segments
}


def pair(case, w, scales):
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"])
    s = jxs().Solver.from_case(case)
    if case.get("phi") is not None:
        o.set_ibm(case["phi"])
    o.set_flux_cnn(w, *scales, emulate_bf16=True)
    s.set_flux_cnn(w, *scales)
    return o, s


def bf16(x):
    return torch.tensor(x).to(torch.bfloat16).to(torch.float64).numpy()


@pytest.mark.parametrize("name", list(CASES))
def test_input_fields_and_corrections(name):
    case = CASES[name]()
    w = wl.cnn_weights(3, bias=0.02)
    scales = wl.cnn_scales(out_factor=0.05)
    o, s = pair(case, w, scales)
    Xx, Xy, Yx, Yy = o.cnn_fields(case["U0"])
    gx, gy = [a.cpu().numpy().astype(np.float64) for a in s.flux_cnn_inputs(dev(case["U0"]))]
    for got, want in ((gx, bf16(Xx)), (gy, bf16(Xy))):
        d = np.abs(got - want)
        assert d.max() <= 2.0 ** -7 * np.abs(want).max()          # at most one bf16 step where a value sits on a tie
        # (a wall's normal momentum is zero up to round-off on both sides, 1e-17 here and 1e-8 there: not a mismatch)
        assert (d > 1e-6 * np.abs(want).max()).mean() < 0.02
    dFx, dGy = [a.cpu().numpy().astype(np.float64) for a in s.flux_correction(dev(case["U0"]))]
    outs = scales[1]
    for k in range(4):
        want = outs[k] * Yx[k]
        assert np.abs(dFx[k] - want).max() <= 1e-2 * np.abs(want).max(), (name, "x", k)
    for k, slot in enumerate((0, 2, 1, 3)):  # network output k -> conserved slot
        want = outs[k] * Yy[k].T
        assert np.abs(dGy[slot] - want).max() <= 1e-2 * np.abs(want).max(), (name, "y", k)


def test_rhs_and_steps_with_the_cnn():
    case = CASES["shock_cylinder_256x136"]()
    w = wl.cnn_weights(5, bias=-0.01)
    scales = wl.cnn_scales(out_factor=0.1)
    o, s = pair(case, w, scales)
    fluid = o.cell_types() == 0
    U0 = case["U0"]
    L1o, L1g = o.rhs(U0), s.rhs(dev(U0)).cpu().numpy()
    o.set_flux_cnn(None); s.set_flux_cnn(None)
    L0o, L0g = o.rhs(U0), s.rhs(dev(U0)).cpu().numpy()
    assert rel_err(L0g, L0o, fluid) <= 1e-12
    corr_o, corr_g = L1o - L0o, L1g - L0g
    assert np.abs(corr_o).max() > 1e-3 * np.abs(L0o).max()                     # the network matters here
    assert rel_err(corr_g, corr_o, fluid) <= 1e-2
    o.set_flux_cnn(w, *scales, emulate_bf16=True); s.set_flux_cnn(w, *scales)
    U = dev(U0)
    s.step(U, 0.4, 8)
    # corrections of 10 % of the flux held to 1e-2, fp16 hand-over (5e-4): a few 1e-4 per step on every field's own scale
    assert rel_err(U.cpu().numpy(), o.step(U0, 0.4, 8), fluid) <= 2e-3


def test_zero_network_is_bitwise_neutral_and_one_network_at_a_time():
    case = CASES["vortex_48"]()
    s = jxs().Solver.from_case(case)
    L0 = s.rhs(dev(case["U0"])).cpu().numpy()
    s.set_flux_cnn(np.zeros(wl.CNN_NPARAM, np.float32), *wl.cnn_scales())
    assert np.array_equal(s.rhs(dev(case["U0"])).cpu().numpy(), L0)
    with pytest.raises(jxs().JxsError):
        s.set_flux_mlp(wl.mlp_weights(), *wl.mlp_scales())
    s.set_flux_cnn(None)
    s.set_flux_mlp(wl.mlp_weights(), *wl.mlp_scales())
    with pytest.raises(jxs().JxsError):
        s.set_flux_cnn(wl.cnn_weights(), *wl.cnn_scales())
