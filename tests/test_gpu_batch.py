"""SURVEY.md section 8(f) rank 4, first half: the batched handle (jxs_create_batch) — nb independent simulations
advanced by one launch per kernel and stage — gives bitwise the results of nb separate handles.  -m gpu."""
import numpy as np
import pytest
import torch

from oracle import jxo
from paper_2601_04400_b200 import workloads as wl
from test_gpu_parity import dev, jxs, rel_err

pytestmark = pytest.mark.gpu


def stack(cases, dtype=torch.float64):
    return torch.tensor(np.stack([c["U0"] for c in cases]), dtype=dtype, device="cuda")


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("mlp", [False, True])
def test_batch_equals_separate_handles_bitwise(dtype, mlp):
    m = jxs()
    cases = wl.batch_cases(5, nx=200, ny=96)      # Mach ~ U[1.5, 3]: inflow state, viscosity and CFL step differ
    w, (ins, outs) = wl.mlp_weights(), wl.mlp_scales()
    b = m.Solver.from_cases(cases, dtype=dtype)
    if mlp:
        b.set_flux_mlp(w, ins, outs)
    Ub = stack(cases, dtype)
    Lb = b.rhs(Ub)
    sb = b.max_wavespeed(Ub)
    b.step(Ub, 0.4, 8)
    tb, dtb = b.time_batch()
    launches = b.launch_count()
    for k, c in enumerate(cases):
        s = m.Solver.from_case(c, dtype=dtype)
        if mlp:
            s.set_flux_mlp(w, ins, outs)
        U = torch.tensor(c["U0"], dtype=dtype, device="cuda")
        assert torch.equal(s.rhs(U), Lb[k]), k
        assert s.max_wavespeed(U) == sb[k]
        s.step(U, 0.4, 8)
        assert torch.equal(U, Ub[k]), k
        assert s.time() == (tb[k], dtb[k])
    assert len(set(dtb)) == len(cases)           # every member took its own CFL step
    # one launch per kernel and stage for the whole batch (the tuning launches of the first call aside)
    b2 = m.Solver.from_cases(cases, dtype=dtype)
    b2.set_rows_per_segment(24)
    if mlp:
        b2.set_flux_mlp(w, ins, outs)
    n0 = b2.launch_count()
    b2.step(Ub, 0.4, 10)
    per_step = 1 + 3 * (3 if mlp else 2)
    assert b2.launch_count() - n0 == 10 * per_step + 2      # + pad-with-wavespeed, unpad


def test_batch_member_against_the_oracle_and_fixed_dt():
    cases = wl.batch_cases(3, nx=160, ny=96)
    b = jxs().Solver.from_cases(cases)
    Ub = stack(cases)
    dt = 0.1 * cases[0]["dx"]
    b.step_fixed_dt(Ub, dt, 6)
    c = cases[2]
    o = jxo.Oracle(c["nx"], c["ny"], c["dx"], c["dy"], c["gamma"], c["mu"], c["Pr"], c["bc"])
    o.set_ibm(c["phi"])
    ref = o.step_fixed_dt(c["U0"], dt, 6)
    assert rel_err(Ub[2].cpu().numpy(), ref, o.cell_types() == 0) <= 1e-9
    assert b.time_batch()[0] == pytest.approx([6 * dt] * 3, rel=1e-14)


def test_batch_argument_checks():
    m = jxs()
    cases = wl.batch_cases(2, nx=160, ny=96)
    b = m.Solver.from_cases(cases)
    with pytest.raises(m.JxsError):
        b.set_flux_cnn(wl.cnn_weights(), *wl.cnn_scales())
    with pytest.raises(m.JxsError):
        b.set_artificial_viscosity(1e-3)
    bad = [dict(cases[0]), dict(cases[1])]
    bad[1]["bc"] = dict(bad[1]["bc"], ylo="transmissive")
    with pytest.raises(m.JxsError) as e:
        m.Solver.from_cases(bad)
    assert e.value.code == m.EINVAL
    U = stack(cases)
    with pytest.raises(m.JxsError):
        b.step_fixed_dt_record(U, 1e-4, 1)
