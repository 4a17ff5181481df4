"""Moment-sharded stepping on the CPU (-m "not gpu"): partition and halo plan, and the whole exchange protocol driven with the
oracle as the shard backend -- in one process (LocalExchange) and as a real world_size-2 gloo job (DistExchange).  The bar:
a sharded run reproduces the single-rank oracle BIT FOR BIT on every owned moment and on w+- (Q31)."""
import os
import socket
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

from oracle import Oracle  # noqa: E402
from paper_2511_21891_b200 import sharded  # noqa: E402
from paper_2511_21891_b200.workloads import config2  # noqa: E402
from shard_backends import OracleShard  # noqa: E402


@pytest.mark.parametrize("M,world", [(16, 2), (16, 3), (7, 7), (32, 8), (5, 1)])
def test_ranges_cover_and_halo_plan_pairs_up(M, world):
    rng = sharded.moment_ranges(M, world)
    assert rng[0][0] == 0 and rng[-1][1] == M and all(rng[i][1] == rng[i + 1][0] for i in range(world - 1))
    assert max(h - l for l, h in rng) - min(h - l for l, h in rng) <= 1
    lays = [sharded.ShardLayout.make(M, world, r) for r in range(world)]
    for lay in lays:
        assert lay.m_offset + lay.M_local <= M and len(lay.owned_local) == lay.hi - lay.lo
        for kind, peer, j in lay.transfers():
            gm = lay.m_offset + j                                   # global moment this transfer carries
            other = [(k, p, jj) for (k, p, jj) in lays[peer].transfers() if p == lay.rank and k != kind]
            assert any(lays[peer].m_offset + jj == gm for (_, _, jj) in other), (lay.rank, kind, peer, j)
            if kind == "send":
                assert lay.lo <= gm < lay.hi                        # only owned moments are sent
            else:
                assert not (lay.lo <= gm < lay.hi) and (gm == lay.lo - 1 or gm == lay.hi)
    with pytest.raises(ValueError):
        sharded.moment_ranges(3, 4)


def _reference(shape, prm, z, g, dt, nsteps):
    o = Oracle(*shape, **prm)
    o.set_state(z, g)
    o.step(dt, nsteps)
    return o


@pytest.mark.parametrize("world,extra", [
    (2, {}), (3, {}),
    (2, dict(closure=1, hermite_coeff=1, if_variant=1)),
    (3, dict(force_eps=0.5, force_nperp_min=1, force_nperp_max=2, force_nz_max=1, seed=11, force_g_amp=0.01, force_g_nz=1, g_sign=-1)),
])
def test_sharded_oracle_in_process_is_bit_exact(world, extra):
    shape, M = (16, 16, 8), 7
    prm, z, g, run = config2(*shape, M)
    prm = dict(prm, **extra)
    dt = -1.0 if world == 3 and not extra else run["dt"]            # one case with the CFL dt of Eq. 16 (same on every rank)
    ref = _reference(shape, prm, z, g, dt, 4)
    lays = [sharded.ShardLayout.make(M, world, r) for r in range(world)]
    shards = [OracleShard(*shape, lay, **prm) for lay in lays]
    for sh in shards:
        sh.set_state(z, g)
    sharded.step_all(shards, lays, dt, 4)
    got = np.concatenate([sh.owned_full() for sh in shards])
    want = np.stack([ref.get_full(2 + m) for m in range(M)])
    assert np.array_equal(got, want)
    for sh in shards:
        assert np.array_equal(sh.o.get_full(0), ref.get_full(0)) and np.array_equal(sh.o.get_full(1), ref.get_full(1))
        assert sh.o.time() == ref.time()
    e = np.array([sh.energy() for sh in shards])
    assert np.array_equal(e[:, :5], np.tile(ref.energy()[:5], (world, 1)))          # Alfvenic energies are replicated
    assert abs(e[:, 5].sum() - ref.energy()[5]) <= 1e-14 * ref.energy()[5]            # W_g is the sum over the shards


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _gloo_rank(rank, world, port, shape, M, nsteps, out_dir):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        prm, z, g, run = config2(*shape, M)
        lay = sharded.ShardLayout.make(M, world, rank)
        sh = OracleShard(*shape, lay, **prm)
        sh.set_state(z, g)
        st = sharded.ShardedStepper(sh, lay, sharded.DistExchange())
        st.step(run["dt"], nsteps)
        np.save(os.path.join(out_dir, f"own{rank}.npy"), sh.owned_full())
        np.save(os.path.join(out_dir, f"w{rank}.npy"), np.stack([sh.o.get_full(0), sh.o.get_full(1)]))
        np.save(os.path.join(out_dir, f"e{rank}.npy"), st.energy())
    finally:
        dist.destroy_process_group()


def test_sharded_oracle_gloo_world2_is_bit_exact(tmp_path):
    import torch.multiprocessing as mp
    shape, M, world, nsteps = (16, 16, 8), 6, 2, 3
    mp.spawn(_gloo_rank, args=(world, _free_port(), shape, M, nsteps, str(tmp_path)), nprocs=world, join=True)
    prm, z, g, run = config2(*shape, M)
    ref = _reference(shape, prm, z, g, run["dt"], nsteps)
    got = np.concatenate([np.load(tmp_path / f"own{r}.npy") for r in range(world)])
    assert np.array_equal(got, np.stack([ref.get_full(2 + m) for m in range(M)]))
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"w{r}.npy"), np.stack([ref.get_full(0), ref.get_full(1)]))
        e = np.load(tmp_path / f"e{r}.npy")                          # every rank holds the reduced record
        assert np.array_equal(e[:5], ref.energy()[:5]) and abs(e[5] - ref.energy()[5]) <= 1e-14 * ref.energy()[5]


def test_shard_parameters_are_validated():
    with pytest.raises(Exception):
        Oracle(16, 16, 8, M=4, m_offset=2, M_global=5)                 # 2 + 4 > 5
    with pytest.raises(Exception):
        Oracle(16, 16, 8, M=4, m_offset=1)                             # offset without M_global
    with pytest.raises(Exception):
        Oracle(16, 16, 8, M=4, m_offset=0, M_global=8, hermite_exact=1)


def test_oracle_stages_must_alternate():
    """Stage 1 without a stage 0 has no half-step state to read (it used to index empty arrays); the oracle refuses it the
    way gandalf_step_stage does, and refuses a full step while one is half done."""
    prm, z, g, run = config2(16, 16, 8, 2)
    o = Oracle(16, 16, 8, **prm)
    o.set_state(z, g)
    with pytest.raises(Exception):
        o.step_stage(run["dt"], 1)
    o.step_stage(run["dt"], 0)
    with pytest.raises(Exception):
        o.step_stage(run["dt"], 0)
    with pytest.raises(Exception):
        o.step(run["dt"], 1)
    o.step_stage(run["dt"], 1)
    ref = Oracle(16, 16, 8, **prm)
    ref.set_state(z, g)
    ref.step(run["dt"], 1)
    assert np.array_equal(o.get_full(2), ref.get_full(2)) and o.time() == ref.time()
    o.step_stage(run["dt"], 0)
    o.set_state(z, g)                        # a new state abandons the half-done step
    o.step(run["dt"], 1)
    assert np.array_equal(o.get_full(0), ref.get_full(0))
