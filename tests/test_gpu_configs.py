"""Parity at the sizes BASELINE.json's configs name (C2, C3, C5, and the CNN at the C4 grid), in the launch
configurations bench.py times.  -m gpu.  The oracle runs for tens of seconds per case here (one host core).

Error norm: max-norm per field over fluid cells, scaled by THAT field's max (BASELINE.json north_star), except
where a component is identically zero up to round-off — then it borrows the other momentum's scale, stated per case.
"""
import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import dev, jxs, make_pair, TOL_STEP64, TOL_STEP32

pytestmark = pytest.mark.gpu


def field_err(a, b, fluid=None, zero_fields=()):
    """per-field max-norm error; `zero_fields`: components that are 0 up to round-off in this case and are
    scaled by the largest momentum instead of their own (tiny) maximum"""
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    m = np.ones(a.shape[1:], bool) if fluid is None else fluid
    peak = [np.max(np.abs(b[k][m])) for k in range(4)]
    out = []
    for k in range(4):
        scale = max(peak[1], peak[2]) if k in zero_fields else peak[k]
        out.append(np.max(np.abs(a[k][m] - b[k][m])) / max(scale, 1e-300))
    return max(out), peak


# ----------------------------------------------------------------------------- C3 (BASELINE.json configs[2])
def test_c3_1024x512_first_100_steps():
    """"parity on the first 100 steps" of the Mach-2 shock / cylinder case at 1024x512, Navier-Stokes,
    IBM, CFL step on the device.  In these 100 steps the shock (x = 0.2 -> 0.26) has not reached the body (x = 0.3):
    rho v is zero up to round-off and borrows the scale of rho u."""
    case = wl.shock_cylinder(1024, 512, Ms=2.0)
    o, s = make_pair(case)
    ref = o.step(case["U0"], 0.4, 100)
    U = dev(case["U0"])
    s.step(U, 0.4, 100)
    fluid = o.cell_types() == 0
    err, peak = field_err(U.cpu().numpy(), ref, fluid, zero_fields=(2,))
    assert peak[2] < 1e-9 * peak[1]
    assert err <= TOL_STEP64, err
    assert o.guard_count() == 0
    assert abs(o.time()[0] - s.time()[0]) <= 1e-12 * o.time()[0]


def test_c3_1024x512_shock_on_the_cylinder():
    """The same case with the shock started just ahead of the body (x = 0.29), so that these 100 steps hold the
    reflection off the immersed boundary: every field has its own scale."""
    case = wl.shock_cylinder(1024, 512, Ms=2.0, x_shock=0.29)
    o, s = make_pair(case)
    ref = o.step(case["U0"], 0.4, 100)
    U = dev(case["U0"])
    s.step(U, 0.4, 100)
    fluid = o.cell_types() == 0
    err, peak = field_err(U.cpu().numpy(), ref, fluid)
    assert peak[2] > 1e-2 * peak[1]          # the reflected shock deflects the flow
    assert err <= TOL_STEP64, err
    assert o.guard_count() == 0


# ----------------------------------------------------------------------------- C2 (BASELINE.json configs[1])
@pytest.mark.parametrize("n,nsteps", [(128, 800), (256, 200)])
def test_c2_vortex_fixed_dt_fp64_and_conservation(n, nsteps):
    """jxs_step_fixed_dt on the periodic vortex; 128^2 runs the whole flow-through period (t = 10)."""
    case = wl.vortex(n)
    dt = 10.0 / (800 * n // 128)
    o, s = make_pair(case)
    ref = o.step_fixed_dt(case["U0"], dt, nsteps)
    U = dev(case["U0"])
    s.step_fixed_dt(U, dt, nsteps)
    got = U.cpu().numpy()
    err, _ = field_err(got, ref)
    assert err <= TOL_STEP64, (n, err)
    assert s.time()[0] == pytest.approx(nsteps * dt, rel=1e-13)
    # discrete conservation over the run, on the GPU: sum of every conserved variable unchanged to round-off
    for k in range(4):
        s0, s1 = case["U0"][k].sum(), got[k].sum()
        assert abs(s1 - s0) <= 1e-12 * np.abs(case["U0"][k]).sum(), (k, s0, s1)


@pytest.mark.parametrize("n", [128, 256])
def test_c2_vortex_fp32_steps(n):
    """fp32 stepping on the vortex against the fp64 oracle (BASELINE.json: 100 steps <= 1e-3), and conservation of
    the fp32 run to fp32 round-off."""
    case = wl.vortex(n)
    dt = 10.0 / (800 * n // 128)
    o64, _ = make_pair(case)
    _, s = make_pair(case, dtype=torch.float32)
    ref = o64.step_fixed_dt(case["U0"], dt, 100)
    U = dev(case["U0"], torch.float32)
    s.step_fixed_dt(U, dt, 100)
    got = U.cpu().numpy().astype(np.float64)
    err, _ = field_err(got, ref)
    assert err <= TOL_STEP32, (n, err)
    U0f = case["U0"].astype(np.float32).astype(np.float64)
    tol = 100 * 3 * 2.0 ** -24      # one fp32 rounding of the combine per stage, all of one sign at worst
    for k in range(4):
        assert abs(got[k].sum() - U0f[k].sum()) <= tol * np.abs(U0f[k]).sum(), k


# ----------------------------------------------------------------------------- C5 (BASELINE.json configs[4])
def _mlp_pair(case, w, ins, outs):
    o = jxo.Oracle(case["nx"], case["ny"], case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"], case["bc"])
    o.set_ibm(case["phi"])
    o.set_flux_mlp(w, ins, outs, emulate_bf16=True)
    s = jxs().Solver.from_case(case)
    s.set_flux_mlp(w, ins, outs)
    return o, s


def test_c5_one_1024x512_handle_correction_after_20_steps():
    """One member of the C5 batch at its full size: 20 RK3 steps with the network in every stage on the GPU, then the
    per-face correction of the reached state against the oracle's bf16-emulating network on sampled faces."""
    from test_gpu_mlp import oracle_face_inputs, rel_net
    case = wl.batch_cases(16)[3]
    w, (ins, outs) = wl.mlp_weights(), wl.mlp_scales()
    o, s = _mlp_pair(case, w, ins, outs)
    U = dev(case["U0"])
    s.step(U, 0.4, 20)
    Uh = U.cpu().numpy()
    assert np.isfinite(Uh).all()
    dFx, dGy = (a.cpu().numpy().astype(np.float64) for a in s.flux_correction(U))
    X, Y = oracle_face_inputs(o, Uh, ins)
    ny, nx = case["ny"], case["nx"]
    rng = np.random.default_rng(5)
    # whole rows / columns through strip and segment boundaries of the 1024x512 launch, plus a random sample
    fx = [(j, f) for j in (0, ny // 2 - 1, ny - 1) for f in range(0, nx + 1, 3)] + \
         [(int(rng.integers(ny)), int(rng.integers(nx + 1))) for _ in range(4000)]
    fy = [(f, i) for f in (0, ny // 2, ny) for i in range(0, nx, 3)] + \
         [(int(rng.integers(ny + 1)), int(rng.integers(nx))) for _ in range(4000)]
    ex = np.array([o.mlp_eval(X[j, f]) * outs for j, f in fx]).T
    ey = np.array([o.mlp_eval(Y[f, i]) * outs for f, i in fy]).T[[0, 2, 1, 3]]
    gx = np.array([dFx[:, j, f] for j, f in fx]).T
    gy = np.array([dGy[:, f, i] for f, i in fy]).T
    assert rel_net(gx, ex, outs) <= 1e-2, rel_net(gx, ex, outs)
    assert rel_net(gy, ey, outs[[0, 2, 1, 3]]) <= 1e-2, rel_net(gy, ey, outs[[0, 2, 1, 3]])


def test_c5_concurrent_handles_with_the_network_equal_the_synchronous_path():
    """bench.py --workload c5 --batch-groups 0: 16 handles x 1024x512 with the flux MLP, one stream each,
    jxs_step_async + jxs_wait — bitwise equal to jxs_step on a handle of its own."""
    m = jxs()
    cases = wl.batch_cases(16)
    w, (ins, outs) = wl.mlp_weights(), wl.mlp_scales()
    streams = [torch.cuda.Stream() for _ in cases]
    solvers, Us = [], []
    for c, st in zip(cases, streams):
        s = m.Solver.from_case(c, stream=st)
        s.set_flux_mlp(w, ins, outs)
        s.set_concurrent_handles(len(cases))
        solvers.append(s)
        Us.append(dev(c["U0"]))
    torch.cuda.synchronize()
    for s, U in zip(solvers, Us):
        s.step_async(U, 0.4, 8)
    for s in solvers:
        s.wait()
    for idx in (0, 7, 15):
        s1 = m.Solver.from_case(cases[idx])
        s1.set_flux_mlp(w, ins, outs)
        U1 = dev(cases[idx]["U0"])
        s1.step(U1, 0.4, 8)
        assert torch.equal(U1, Us[idx]), idx
        assert s1.time() == solvers[idx].time()


# ----------------------------------------------------------------------------- CNN at the C4 grid
def test_cnn_correction_at_4096x2048_on_sampled_windows():
    """bench.py --workload cnn's launch configuration.  A 3-layer 3x3 network has a receptive radius of 3 faces, so
    the oracle's network applied (jxo_cnn_apply) to a window of the oracle's own input field reproduces the full
    field's output at the window's centre: sampled windows across strip and segment boundaries, both directions."""
    case = wl.throughput_case()
    w = wl.cnn_weights(3, bias=0.02)
    scales = wl.cnn_scales(out_factor=0.05)
    ins, outs = scales
    s = jxs().Solver.from_case(case)
    s.set_flux_cnn(w, *scales)
    U = dev(case["U0"])
    gx, gy = [a.cpu().numpy().astype(np.float64) for a in s.flux_cnn_inputs(U)]      # bf16 values the GPU feeds
    dFx, dGy = [a.cpu().numpy().astype(np.float64) for a in s.flux_correction(U)]
    ny, nx = case["ny"], case["nx"]
    small = wl.vortex(16)
    o = jxo.Oracle(16, 16, small["dx"], small["dy"], small["gamma"], 0.0, 0.72, small["bc"])
    o.set_flux_cnn(w, *scales, emulate_bf16=True)       # jxo_cnn_apply only needs the network
    R, Wn = 3, 24
    rng = np.random.default_rng(9)
    # x-faces: field [4][ny][nx+1] (rows tangential, faces normal); windows away from the field's border (zero padding
    # is covered by the small cases of test_gpu_cnn.py), centred on strip edges (multiples of 128) and random places
    shock_col = int(0.1 / case["dx"])
    centres_x = [(j, f) for j in (Wn // 2, 1023, 1024, ny - Wn // 2 - 1) for f in (127, 128, 129, shock_col, 2048, nx - 130)] + \
                [(int(rng.integers(Wn, ny - Wn)), int(rng.integers(Wn, nx - Wn))) for _ in range(24)]
    worst = 0.0
    peak = np.abs(dFx).max(axis=(1, 2))
    for (j, f) in centres_x:
        win = gx[:, j - Wn // 2:j + Wn // 2, f - Wn // 2:f + Wn // 2]
        y = o.cnn_apply(win)
        c = Wn // 2
        for k in range(4):
            want = outs[k] * y[k, R:-R, R:-R]
            got = dFx[k, j - c + R:j + c - R, f - c + R:f + c - R]
            worst = max(worst, np.abs(got - want).max() / peak[k])
    assert worst <= 1e-2, worst
    # y-faces: the network sees (tangential, normal) = (i, f): field [4][nx][ny+1]; dGy is [4][ny+1][nx] in conserved slots
    peak_y = np.abs(dGy).max(axis=(1, 2))
    centres_y = [(i, f) for i in (127, 128, 2048, nx - 129) for f in (Wn // 2, 1024, ny - Wn // 2)] + \
                [(int(rng.integers(Wn, nx - Wn)), int(rng.integers(Wn, ny - Wn))) for _ in range(24)]
    worst = 0.0
    for (i, f) in centres_y:
        win = gy[:, i - Wn // 2:i + Wn // 2, f - Wn // 2:f + Wn // 2]
        y = o.cnn_apply(win)
        c = Wn // 2
        for k, slot in enumerate((0, 2, 1, 3)):
            want = outs[k] * y[k, R:-R, R:-R].T
            got = dGy[slot, f - c + R:f + c - R, i - c + R:i + c - R]
            worst = max(worst, np.abs(got - want).max() / peak_y[slot])
    assert worst <= 1e-2, worst
    # and the input fields themselves on the same windows against the oracle's reconstruction of those windows:
    # sampled rows of the full-size field equal the oracle's field computed on a cropped copy of the state
    # (WENO5 reaches 3 cells: crop with a margin of 8), away from bodies and domain edges
    j0, i0, hh = 1000, 200, 40       # the window holds the Mach-3 shock (column 204)
    crop = dict(case)
    crop["U0"] = np.ascontiguousarray(case["U0"][:, j0 - hh:j0 + hh, i0 - hh:i0 + hh])
    assert np.all(case["phi"][j0 - hh:j0 + hh, i0 - hh:i0 + hh] > 8 * case["dx"])
    oc = jxo.Oracle(2 * hh, 2 * hh, case["dx"], case["dy"], case["gamma"], case["mu"], case["Pr"],
                    dict(xlo="transmissive", xhi="transmissive", ylo="transmissive", yhi="transmissive"))
    oc.set_flux_cnn(w, *scales, emulate_bf16=True)
    Xx, Xy, _, _ = oc.cnn_fields(crop["U0"])
    bf = lambda x: torch.tensor(x).to(torch.bfloat16).to(torch.float64).numpy()
    m = 8
    want = bf(Xx)[:, m:-m, m:-m]
    got = gx[:, j0 - hh + m:j0 + hh - m, i0 - hh + m:i0 + hh + 1 - m]
    assert np.abs(got - want).max() <= 2.0 ** -7 * np.abs(want).max()
    want = bf(Xy)[:, m:-m, m:-m]
    got = gy[:, i0 - hh + m:i0 + hh - m, j0 - hh + m:j0 + hh + 1 - m]
    assert np.abs(got - want).max() <= 2.0 ** -7 * np.abs(want).max()
