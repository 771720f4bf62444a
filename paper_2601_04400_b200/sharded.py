"""y-slab sharding of one simulation over several GPUs: host-side plan and driver.

The path shards naturally — an explicit stencil with one exchange step per stage.  Every rank owns a contiguous slab of
rows and runs an ordinary `jxs` handle on its slab EXTENDED by `overlap` rows on every cut side:

  * the extension rows are *inactive* (`jxs_set_active_rows`): they are overwritten, before every stage, with the rows the
    neighbouring rank owns (pack kernel -> NCCL send/recv -> unpack kernel: `jxs_shard_rows`), their own right-hand side
    is zero and they do not enter s_max, so whatever the dummy boundary condition on the cut puts behind them is never used;
  * `overlap` = 12 rows = 3 (the WENO5 stencil of the owned rows) + 9 (how far the donors of an immersed-boundary ghost
    cell can lie from it: |phi| <= 3.5 cells, image point at twice that, bilinear cell, one probe step): ghost cells in the
    owned rows and in the 3 rows their stencils reach are filled from values inside the extended slab, so bodies may cross
    a cut.  Per stage and neighbour that is 12 nx 4 values (1.5 MB at nx = 4096 in fp64);
  * the CFL step needs the global s_max: one scalar MAX all-reduce per step (`jxs_shard_smax`).

With these three pieces every owned row is computed with the arithmetic of the single-domain run: the sharded result is
bitwise the single-GPU one (tests/test_gpu_sharded.py, all ranks driven from one process on one GPU;
tests/test_sharded_plan.py: the plan and the exchange protocol under gloo, world size 2, on CPU).
UNMEASURED ON HARDWARE: no multi-GPU node was available; `bench.py --gpus N` runs replicas.

This module holds none of the method's arithmetic.  `SlabPlan` is pure Python (no torch, no CUDA).
"""
from dataclasses import dataclass

OVERLAP = 12


@dataclass
class Transfer:
    """rows [src_row, src_row + n) of rank `src`'s extended slab go to rows [dst_row, ...) of rank `dst`'s"""
    src: int
    dst: int
    src_row: int
    dst_row: int
    n: int


class SlabPlan:
    """Who owns which rows, what every rank's extended slab is, and which rows travel before a stage."""

    def __init__(self, ny, world, periodic=False, overlap=OVERLAP):
        if world < 1 or ny < 1:
            raise ValueError("world and ny must be positive")
        if world > 1 and ny // world < overlap:
            raise ValueError(f"slabs of {ny // world} rows are thinner than the overlap of {overlap} rows")
        self.ny, self.world, self.periodic, self.overlap = ny, world, bool(periodic) and world > 1, overlap
        base, extra = divmod(ny, world)
        self.own = []          # [j0, j1) global rows owned by rank r
        j = 0
        for r in range(world):
            n = base + (1 if r < extra else 0)
            self.own.append((j, j + n))
            j += n
        # the extended slab of rank r: `lo` extension rows below, owned rows, `hi` extension rows above
        self.ext = []
        for r, (j0, j1) in enumerate(self.own):
            lo = overlap if (r > 0 or self.periodic) else 0
            hi = overlap if (r < world - 1 or self.periodic) else 0
            self.ext.append((lo, hi))

    def local_ny(self, r):
        j0, j1 = self.own[r]
        lo, hi = self.ext[r]
        return lo + (j1 - j0) + hi

    def active_rows(self, r):
        """[lo, hi) in local row indices: the owned rows"""
        j0, j1 = self.own[r]
        lo, _ = self.ext[r]
        return lo, lo + (j1 - j0)

    def global_rows(self, r):
        """global row index of every local row of rank r (wrapped when the domain is periodic in y)"""
        j0, j1 = self.own[r]
        lo, hi = self.ext[r]
        return [(j % self.ny) for j in range(j0 - lo, j1 + hi)]

    def cut_sides(self, r):
        """(low side is a cut, high side is a cut)"""
        lo, hi = self.ext[r]
        return lo > 0, hi > 0

    def transfers(self):
        """every Transfer of one exchange (the same before every stage)"""
        out = []
        for r in range(self.world):
            lo, hi = self.ext[r]
            j0, j1 = self.own[r]
            n_own = j1 - j0
            if lo:   # my low extension = the top `lo` owned rows of the rank below
                src = (r - 1) % self.world
                s_lo, _ = self.ext[src]
                s_own = self.own[src][1] - self.own[src][0]
                out.append(Transfer(src, r, s_lo + s_own - lo, 0, lo))
            if hi:   # my high extension = the bottom `hi` owned rows of the rank above
                src = (r + 1) % self.world
                s_lo, _ = self.ext[src]
                out.append(Transfer(src, r, s_lo, lo + n_own, hi))
        return out

    def local_bc(self, r, bc):
        """the boundary conditions of rank r's handle: the domain's own on real sides; on a cut a transmissive dummy
        (what it fills is never used: the rows in front of it are inactive)"""
        cut_lo, cut_hi = self.cut_sides(r)
        b = dict(bc)
        if cut_lo or cut_hi:
            if cut_lo or bc["ylo"] == "periodic":
                b["ylo"] = "transmissive"
            if cut_hi or bc["yhi"] == "periodic":
                b["yhi"] = "transmissive"
        return b

    def local_case(self, r, case):
        """rank r's part of a workloads.py case (numpy slicing only)"""
        import numpy as np
        rows = self.global_rows(r)
        c = dict(case)
        c["U0"] = np.ascontiguousarray(case["U0"][:, rows, :])
        c["phi"] = None if case.get("phi") is None else np.ascontiguousarray(case["phi"][rows, :])
        c["ny"] = len(rows)
        c["bc"] = self.local_bc(r, case["bc"])
        c["name"] = f"{case.get('name', 'case')}[rank {r}/{self.world}]"
        return c


class LocalComm:
    """All ranks live in this process (tests on one GPU): a transfer is a pack on the source and an unpack on the
    destination; the MAX over ranks is taken here."""

    def exchange(self, plan, handles, k, buffers):
        for t in plan.transfers():
            buf = buffers(t.n)
            handles[t.src].shard_rows(k, t.src_row, t.n, buf, unpack=False)
            handles[t.dst].shard_rows(k, t.dst_row, t.n, buf, unpack=True)

    def allreduce_max(self, values):
        import torch
        m = torch.stack(values).max()
        return [m.reshape(1).clone() for _ in values]


class DistComm:
    """One rank per process over torch.distributed (NCCL on device tensors; gloo stages through the host)."""

    def __init__(self, dist, rank):
        self.dist, self.rank = dist, rank
        self.host_staging = dist.get_backend() == "gloo"

    def exchange(self, plan, handles, k, buffers):
        import torch
        h = handles[0]
        ops, recvs = [], []
        for t in plan.transfers():   # the same order on every rank: sends and receives pair up
            if t.src == self.rank:
                buf = buffers(t.n)
                h.shard_rows(k, t.src_row, t.n, buf, unpack=False)
                wire = buf.cpu() if self.host_staging else buf
                ops.append(self.dist.P2POp(self.dist.isend, wire, t.dst))
            if t.dst == self.rank:
                buf = buffers(t.n)
                wire = torch.empty(buf.shape, dtype=buf.dtype) if self.host_staging else buf
                ops.append(self.dist.P2POp(self.dist.irecv, wire, t.src))
                recvs.append((t, buf, wire))
        if ops:
            for req in self.dist.batch_isend_irecv(ops):
                req.wait()
        for t, buf, wire in recvs:
            if self.host_staging:
                buf.copy_(wire)
            h.shard_rows(k, t.dst_row, t.n, buf, unpack=True)

    def allreduce_max(self, values):
        v = values[0]
        wire = v.cpu() if self.host_staging else v
        self.dist.all_reduce(wire, op=self.dist.ReduceOp.MAX)
        if self.host_staging:
            v.copy_(wire)
        return [v]


class ShardedSolver:
    """One simulation cut into y-slabs.  `ranks`: the ranks this process drives — [rank] under torch.distributed
    (comm = DistComm), all of them with LocalComm.  make_handle(local_case) -> an object with the jxs.Solver methods
    set_active_rows / shard_begin / shard_smax / shard_step_begin / shard_stage / shard_rows / shard_end."""

    def __init__(self, case, world, ranks, comm, make_handle, new_tensor):
        self.plan = SlabPlan(case["ny"], world, periodic=case["bc"]["ylo"] == "periodic")
        self.ranks, self.comm, self.new_tensor = list(ranks), comm, new_tensor
        self.cases = [self.plan.local_case(r, case) for r in self.ranks]
        self.handles = []
        for r, c in zip(self.ranks, self.cases):
            self.handles.append(make_handle(c, self.plan.active_rows(r)))
        self._pool = {}
        self._next = 0

    def _buffers(self, n):
        """a fresh [4][n][nx] tensor per transfer of one exchange (kept between exchanges)"""
        key = (n, self._next)
        self._next += 1
        if key not in self._pool:
            self._pool[key] = self.new_tensor((4, n, self.cases[0]["nx"]))
        return self._pool[key]

    def step(self, Us, cfl, nsteps, fixed_dt=0.0):
        """Us: one device tensor [4][local ny][nx] per driven rank (extended slabs); advanced in place"""
        hs = self.handles if isinstance(self.comm, LocalComm) else self.handles[:1]
        for h, U in zip(self.handles, Us):
            h.shard_begin(U)
        smax = [self.new_tensor((1,)) for _ in self.handles]
        for _ in range(nsteps):
            if not fixed_dt > 0:
                for h, v in zip(self.handles, smax):
                    h.shard_smax(v, set=False)
                for h, v in zip(self.handles, self.comm.allreduce_max(smax)):
                    h.shard_smax(v, set=True)
            for h in self.handles:
                h.shard_step_begin(cfl, fixed_dt)
            for k in range(3):
                self._next = 0
                self.comm.exchange(self.plan, hs, k, self._buffers)
                for h in self.handles:
                    h.shard_stage(k)
        for h, U in zip(self.handles, Us):
            h.shard_end(U, nsteps)
        return Us

    def owned(self, r_index, U):
        lo, hi = self.plan.active_rows(self.ranks[r_index])
        return U[:, lo:hi, :]
