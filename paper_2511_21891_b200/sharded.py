"""Moment-sharded multi-GPU stepping: host logic only (Q31, section 9).

The Hermite hierarchy is cut into contiguous ranges of moments, one per rank (PAPER.md:832, 975 list multi-device runs as
future work; the paper is single device).  Every rank evolves xi+- redundantly (2 fields, identical on all ranks: same state,
same forcing keys) and its own moments; Eq. 6 couples g_m only to g_{m-1} and g_{m+1}, so a rank needs ONE halo moment from
each neighbour, refreshed after every stage of the RK2 step (twice per step).  The exchange is point to point:
`torch.distributed` P2P ops (NCCL over NVLink between GPUs, gloo in the CPU tests) in place on the library's own buffers.

Nothing here computes: a *shard* is any object with
    step_stage(dt, stage), energy(),
    send_tensor(state, field) / recv_tensor(state, field) -> torch tensor, commit(state, field, tensor), halo_refresh(state)
(`GandalfShard` below wraps the CUDA library; the CPU tests drive the oracle through the same protocol).
"""
from __future__ import annotations

from dataclasses import dataclass


def moment_ranges(M, world):
    """Contiguous, near-equal ranges [lo, hi) of the moments 0..M-1, one per rank (the first M % world ranks get one more)."""
    if world < 1 or M < world:
        raise ValueError(f"cannot give each of {world} ranks at least one of {M} moments")
    base, rem = divmod(M, world)
    out, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < rem else 0)
        out.append((lo, hi))
        lo = hi
    return out


@dataclass(frozen=True)
class ShardLayout:
    """What rank `rank` of `world` holds: owned global moments [lo, hi) plus one halo below (if lo > 0) and above (if hi < M)."""
    rank: int
    world: int
    M: int          # global number of moments
    lo: int
    hi: int

    @classmethod
    def make(cls, M, world, rank):
        lo, hi = moment_ranges(M, world)[rank]
        return cls(rank, world, M, lo, hi)

    @property
    def halo_lo(self):
        return 1 if self.lo > 0 else 0

    @property
    def halo_hi(self):
        return 1 if self.hi < self.M else 0

    @property
    def m_offset(self):            # global index of local moment 0
        return self.lo - self.halo_lo

    @property
    def M_local(self):
        return self.hi - self.lo + self.halo_lo + self.halo_hi

    @property
    def owned_local(self):         # local indices of the owned moments
        return range(self.halo_lo, self.M_local - self.halo_hi)

    def params(self):
        """Library parameters of this shard (include/gandalf.h: M, m_offset, M_global)."""
        if self.world == 1:
            return dict(M=self.M)
        return dict(M=self.M_local, m_offset=self.m_offset, M_global=self.M)

    def take(self, g):
        """The local moment fields (halos included) of a global array g[m, ...]."""
        return g[self.m_offset:self.m_offset + self.M_local]

    def transfers(self):
        """[(kind, peer, local moment)]: what this rank sends and receives in one halo exchange.  A rank's lower halo is its
        lower neighbour's LAST owned moment, its upper halo the upper neighbour's FIRST owned one."""
        t = []
        if self.halo_lo:
            t.append(("send", self.rank - 1, self.halo_lo))                       # first owned -> lower neighbour's upper halo
            t.append(("recv", self.rank - 1, 0))
        if self.halo_hi:
            t.append(("send", self.rank + 1, self.M_local - 1 - self.halo_hi))    # last owned -> upper neighbour's lower halo
            t.append(("recv", self.rank + 1, self.M_local - 1))
        return t


class DistExchange:
    """Halo exchange over a torch.distributed process group (one rank per GPU; NCCL on GPUs, gloo on CPU)."""

    def __init__(self, group=None, device=None):
        """`device`: where reduction operands are placed.  None = decided by the backend: NCCL reduces CUDA tensors only, so
        the operand goes to the current CUDA device (the one the shard's context runs on); gloo reduces on the host."""
        self.group, self.device = group, device

    def _reduce_device(self):
        import torch
        import torch.distributed as dist
        if self.device is not None:
            return torch.device(self.device)
        if dist.get_backend(self.group) == "nccl":
            return torch.device("cuda", torch.cuda.current_device())
        return torch.device("cpu")

    def halos(self, shard, layout, state):
        import torch.distributed as dist
        ops, got = [], []
        for kind, peer, j in layout.transfers():
            if kind == "send":
                ops.append(dist.P2POp(dist.isend, shard.send_tensor(state, 2 + j), peer, self.group))
            else:
                t = shard.recv_tensor(state, 2 + j)
                ops.append(dist.P2POp(dist.irecv, t, peer, self.group))
                got.append((j, t))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        for j, t in got:
            shard.commit(state, 2 + j, t)
        shard.halo_refresh(state)

    def sum(self, x):
        import torch
        import torch.distributed as dist
        t = (x if isinstance(x, torch.Tensor) else torch.as_tensor(x)).to(self._reduce_device())
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
        return t.cpu()


class LocalExchange:
    """The same exchange among shards living in ONE process (several contexts on one GPU, or the CPU tests): the ranks are
    emulated over all ranks' data by plain copies -- no kernel ever waits on another rank."""

    def __init__(self, shards, layouts):
        self.shards, self.layouts = shards, layouts

    def halos_all(self, state):
        for lay, sh in zip(self.layouts, self.shards):
            for kind, peer, j in lay.transfers():
                if kind != "recv":
                    continue
                plan = self.layouts[peer].transfers()
                src = [jj for (k, p, jj) in plan if k == "send" and p == lay.rank][0]
                t = sh.recv_tensor(state, 2 + j)
                t.copy_(self.shards[peer].send_tensor(state, 2 + src))
                sh.commit(state, 2 + j, t)
        for sh in self.shards:
            sh.halo_refresh(state)


class ShardedStepper:
    """One rank's stepping loop: stage 0, halos of the stage state, stage 1, halos of the new state (Alg. 1 with the two
    exchange points of DESIGN.md Q31)."""

    def __init__(self, shard, layout, exchange):
        self.shard, self.layout, self.exchange = shard, layout, exchange

    def step(self, dt, nsteps=1):
        for _ in range(int(nsteps)):
            self.shard.step_stage(dt, 0)
            self.exchange.halos(self.shard, self.layout, 1)
            self.shard.step_stage(dt, 1)
            self.exchange.halos(self.shard, self.layout, 0)

    def energy(self):
        """{E_A, E+, E-, E_kin, E_mag, W_g}: the Alfvenic entries are replicated, W_g is summed over the shards."""
        import torch
        e = torch.as_tensor(self.shard.energy()).clone()
        wg = self.exchange.sum(e[5:6].clone())
        e[5] = wg[0]
        return e.numpy()


def step_all(shards, layouts, dt, nsteps=1):
    """In-process emulation of `world` ranks (see LocalExchange): every shard takes stage 0, halos move, stage 1, halos move."""
    ex = LocalExchange(shards, layouts)
    for _ in range(int(nsteps)):
        for sh in shards:
            sh.step_stage(dt, 0)
        ex.halos_all(1)
        for sh in shards:
            sh.step_stage(dt, 1)
        ex.halos_all(0)


class GandalfShard:
    """The CUDA library as a shard: halos are sent from / received into the library's own device buffers (zero copy)."""

    def __init__(self, nx, ny, nz, layout, device=0, stream=None, **prm):
        from .gandalf import Gandalf
        prm = dict(prm)
        prm.pop("M", None)
        prm.update(layout.params())
        self.layout = layout
        self.g = Gandalf(nx, ny, nz, device=device, stream=stream, **prm)

    def set_state(self, zeta, g_global):
        self.g.set_state(zeta, self.layout.take(g_global))

    def step_stage(self, dt, stage):
        self.g.step_stage(dt, stage)

    def energy(self):
        return self.g.energy()

    def send_tensor(self, state, field):
        return self.g.field_tensor(state, field)

    recv_tensor = send_tensor

    def commit(self, state, field, tensor):      # received in place
        pass

    def halo_refresh(self, state):
        self.g.halo_refresh(state)

    def owned_raw(self):
        """The owned moments' raw retained-mode coefficients, a (n_owned, PS) complex tensor on the device."""
        import torch
        raw = self.g.get_state_raw(device=True)
        per = raw.numel() // (2 + self.layout.M_local)
        fields = torch.view_as_complex(raw.view(2 + self.layout.M_local, per // 2, 2))
        own = self.layout.owned_local
        return fields[2 + own.start:2 + own.stop]

    def close(self):
        self.g.close()
