"""SURVEY.md section 8(e) / 8(f) rank 4, second half: y-slab sharding.  All ranks of a sharded run are driven from this
one process on one GPU, one after the other (no kernel waits on another rank's): the CUDA pieces — active rows, halo
pack / unpack kernels, per-stage ghost fills and stage kernel, the s_max hand-over — and the plan of sharded.py give,
on the owned rows of every rank, BITWISE the single-domain result.  -m gpu.  (The transport itself, torch.distributed
send / recv, is tests/test_sharded_plan.py under gloo; UNMEASURED on multi-GPU hardware.)"""
import numpy as np
import pytest
import torch

from paper_2601_04400_b200 import workloads as wl
from paper_2601_04400_b200.sharded import LocalComm, ShardedSolver
from test_gpu_parity import MIXED, dev, jxs, smooth_case

pytestmark = pytest.mark.gpu


def run_sharded(case, world, nsteps, cfl=0.4, fixed_dt=0.0, mlp=None):
    m = jxs()

    def make(c, active):
        s = m.Solver.from_slab(c, active)
        if mlp:
            s.set_flux_mlp(*mlp)
        return s

    sh = ShardedSolver(case, world, range(world), LocalComm(), make,
                       lambda shape: torch.zeros(shape, dtype=torch.float64, device="cuda"))
    Us = [dev(c["U0"]) for c in sh.cases]
    sh.step(Us, cfl, nsteps, fixed_dt)
    out = torch.cat([sh.owned(r, U) for r, U in enumerate(Us)], dim=1)
    return out, sh


@pytest.mark.parametrize("world", [2, 4])
def test_c3_sharded_equals_single_domain_bitwise(world):
    """BASELINE.json configs[2] at 1024 x 512: the cylinder straddles the cut of world = 2 (rows 205..307 vs the cut at
    256) and two of the cuts of world = 4; shock on the body; 6 steps with the CFL step from the all-reduced s_max."""
    case = wl.shock_cylinder(1024, 512, Ms=2.0, x_shock=0.29)
    s = jxs().Solver.from_case(case)
    U = dev(case["U0"])
    s.step(U, 0.4, 6)
    got, sh = run_sharded(case, world, 6)
    assert torch.equal(got, U)
    assert sh.handles[0].time() == s.time()
    assert sum(h.ibm_ghost_count() for h in sh.handles) >= s.ibm_ghost_count()


def test_sharded_periodic_viscous_fixed_dt_and_mlp():
    case = smooth_case(130, 96, 4, mu=5e-3, jump=True)           # periodic in x and y: the slabs wrap around
    s = jxs().Solver.from_case(case)
    U = dev(case["U0"])
    dt = 0.1 * min(case["dx"], case["dy"])
    s.step_fixed_dt(U, dt, 5)
    got, _ = run_sharded(case, 3, 5, fixed_dt=dt)
    assert torch.equal(got, U)
    # inflow / outflow / walls with the flux MLP in every stage
    case = wl.shock_cylinder(256, 128, Ms=2.5, x_shock=0.28)
    mlp = (wl.mlp_weights(), *wl.mlp_scales())
    s = jxs().Solver.from_case(case)
    s.set_flux_mlp(*mlp)
    U = dev(case["U0"])
    s.step(U, 0.4, 4)
    got, _ = run_sharded(case, 2, 4, mlp=mlp)
    assert torch.equal(got, U)


def test_shard_calls_out_of_order():
    m = jxs()
    case = smooth_case(64, 48, 1, MIXED)
    s = m.Solver.from_case(case)
    with pytest.raises(m.JxsError) as e:
        s.shard_stage(0)
    assert e.value.code == m.ESTATE
    with pytest.raises(m.JxsError):
        s.set_active_rows(10, 5)
    s.set_ibm(None)
    s.set_active_rows(12, 36)
    U = dev(case["U0"])
    before = U.clone()
    s.shard_begin(U)
    s.shard_step_begin(0.4)
    for k in range(3):
        s.shard_stage(k)
    s.shard_end(U, 1)
    # inactive rows keep their state (L = 0 there; the Shu-Osher combine of equal states rounds in the last place)
    assert torch.allclose(U[:, :12], before[:, :12], rtol=1e-15, atol=0) and torch.allclose(U[:, 36:], before[:, 36:], rtol=1e-15, atol=0)
    assert not torch.equal(U[:, 12:36], before[:, 12:36])
