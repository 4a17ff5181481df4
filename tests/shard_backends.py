"""Test-side shard backend: the CPU oracle driven through the protocol of paper_2511_21891_b200/sharded.py
(step_stage / send_tensor / recv_tensor / commit / halo_refresh).  Test infrastructure: the product never imports it."""
import numpy as np
import torch

from oracle import Oracle


class OracleShard:
    def __init__(self, nx, ny, nz, layout, **prm):
        prm = dict(prm)
        prm.pop("M", None)
        prm.update(layout.params())
        self.layout = layout
        self.o = Oracle(nx, ny, nz, **prm)

    def set_state(self, zeta, g_global):
        self.o.set_state(zeta, self.layout.take(g_global))

    def step_stage(self, dt, stage):
        self.o.step_stage(dt, stage)

    def energy(self):
        return self.o.energy()

    def send_tensor(self, state, field):
        a = self.o.get_stage_full(field) if state == 1 else self.o.get_full(field)
        return torch.from_numpy(np.ascontiguousarray(a).view(np.float64).reshape(-1))

    def recv_tensor(self, state, field):
        return torch.empty(2 * self.o.nz * self.o.ny * self.o.nx, dtype=torch.float64)

    def commit(self, state, field, tensor):
        a = tensor.numpy().view(np.complex128).reshape(self.o.nz, self.o.ny, self.o.nx)
        (self.o.set_stage_full if state == 1 else self.o.set_full)(field, a)

    def halo_refresh(self, state):        # the oracle keeps nothing besides the spectra
        pass

    def owned_full(self):
        return np.stack([self.o.get_full(2 + j) for j in self.layout.owned_local])
