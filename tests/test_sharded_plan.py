"""y-slab sharding: the host-side plan (ownership, extended slabs, which rows travel) and the
exchange protocol of paper_2601_04400_b200/sharded.py under torch.distributed (gloo, world size 2, CPU) with a stand-in
handle that packs / unpacks rows of a numpy array.  -m "not gpu".  The CUDA side (pack / unpack kernels, active rows,
bitwise equality with the single-domain run) is tests/test_gpu_sharded.py."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_2601_04400_b200.sharded import OVERLAP, SlabPlan

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("ny,world,periodic", [(512, 2, False), (512, 8, False), (2048, 8, False), (100, 3, False),
                                               (96, 4, True), (512, 1, False), (512, 1, True)])
def test_plan_partitions_the_rows_and_every_overlap_row_has_one_owner(ny, world, periodic):
    p = SlabPlan(ny, world, periodic)
    rows = [j for r in range(world) for j in range(*p.own[r])]
    assert rows == list(range(ny))                                  # owned slabs tile the domain, in order
    assert max(b - a for a, b in p.own) - min(b - a for a, b in p.own) <= 1
    owner = {j: r for r in range(world) for j in range(*p.own[r])}
    covered = {r: set() for r in range(world)}
    for t in p.transfers():
        g_src, g_dst = p.global_rows(t.src), p.global_rows(t.dst)
        a_lo, a_hi = p.active_rows(t.src)
        for q in range(t.n):
            assert a_lo <= t.src_row + q < a_hi                      # only OWNED rows are sent
            assert g_src[t.src_row + q] == g_dst[t.dst_row + q]      # to the local row that stands for the same global row
            assert owner[g_src[t.src_row + q]] == t.src
            covered[t.dst].add(t.dst_row + q)
    for r in range(world):
        lo, hi = p.active_rows(r)
        inactive = set(range(p.local_ny(r))) - set(range(lo, hi))
        assert covered[r] == inactive                                # every overlap row is refreshed, nothing else is touched
        cut_lo, cut_hi = p.cut_sides(r)
        assert lo == (OVERLAP if cut_lo else 0) and p.local_ny(r) - hi == (OVERLAP if cut_hi else 0)
        if not periodic:
            assert cut_lo == (r > 0) and cut_hi == (r < world - 1)


def test_plan_local_cases_and_boundary_conditions():
    from paper_2601_04400_b200 import workloads as wl
    case = wl.shock_cylinder(128, 64, Ms=2.0)
    p = SlabPlan(case["ny"], 2)
    lows = [p.local_case(r, case) for r in range(2)]
    assert lows[0]["bc"]["ylo"] == "reflective" and lows[0]["bc"]["yhi"] == "transmissive"   # real wall / cut
    assert lows[1]["bc"]["ylo"] == "transmissive" and lows[1]["bc"]["yhi"] == "reflective"
    assert lows[0]["bc"]["xlo"] == "inflow"
    assert np.array_equal(lows[0]["U0"], case["U0"][:, :32 + OVERLAP]) and np.array_equal(lows[1]["phi"], case["phi"][32 - OVERLAP:])
    with pytest.raises(ValueError):
        SlabPlan(40, 4)                                              # slabs thinner than the overlap


WORKER = r'''
import os, sys
import numpy as np
import torch
import torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2601_04400_b200.sharded import DistComm, ShardedSolver

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ny, nx = 64, 10
G = np.arange(4 * ny * nx, dtype=np.float64).reshape(4, ny, nx)      # the "global" field: every entry names itself
case = dict(U0=G, phi=None, nx=nx, ny=ny, bc=dict(xlo="periodic", xhi="periodic", ylo=sys.argv[2], yhi=sys.argv[2]), name="g")

class FakeHandle:                                                     # jxs.Solver's sharding calls on a numpy array
    def __init__(self, c, active):
        self.c, self.active, self.buf, self.smax, self.log = c, active, None, None, []
    def shard_begin(self, U):
        self.buf = [U.numpy().copy() for _ in range(3)]
        lo, hi = self.active
        for b in self.buf:                                            # overlap rows start as garbage
            b[:, :lo] = -1.0; b[:, hi:] = -1.0
        self.smax = float(10 + rank)
    def shard_smax(self, v, set):
        if set: self.smax = float(v[0])
        else: v[0] = self.smax
    def shard_step_begin(self, cfl, fixed_dt): self.log.append(("dt", self.smax))
    def shard_rows(self, k, row0, n, rows, unpack):
        if unpack: self.buf[k][:, row0:row0 + n] = rows.numpy()
        else: rows.copy_(torch.from_numpy(self.buf[k][:, row0:row0 + n].copy()))
    def shard_stage(self, k):
        self.log.append(("stage", k, self.buf[k].copy()))
    def shard_end(self, U, nsteps): U.copy_(torch.from_numpy(self.buf[0]))

class HostDist:                                                       # DistComm asks the backend: CPU tensors go as they are
    def __getattr__(self, n): return getattr(dist, n)
    def get_backend(self): return "nccl-like"
comm = DistComm(HostDist(), rank)
s = ShardedSolver(case, world, [rank], comm, lambda c, a: FakeHandle(c, a), lambda shape: torch.zeros(shape, dtype=torch.float64))
U = torch.from_numpy(s.cases[0]["U0"].copy())
s.step([U], 0.4, 2)
h = s.handles[0]
want = G[:, s.plan.global_rows(rank)]
stages = [e for e in h.log if e[0] == "stage"]
assert len(stages) == 6
for _, k, seen in stages:                                             # before every stage the whole extended slab is current
    assert np.array_equal(seen, want), (rank, k)
assert all(e[1] == 10.0 + world - 1 for e in h.log if e[0] == "dt")  # the MAX over the ranks reached everyone
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
'''


@pytest.mark.parametrize("ybc", ["transmissive", "periodic"])
def test_exchange_protocol_under_gloo_world_size_2(tmp_path, ybc):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT, ybc], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o[-2000:]
