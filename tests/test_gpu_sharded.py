"""Moment-sharded stepping with the CUDA library (-m gpu): `world` shard contexts on ONE GPU, halos moved by LocalExchange
(device copies between the contexts' own buffers -- the ranks are emulated over all ranks' data; no kernel waits on another
rank).  The sharded run must reproduce the unsharded library bit for bit on w+- and to round-off on every owned moment (the
x-pass transforms the moment brackets in PAIRS packed into one complex FFT, and a shard pairs different neighbours, so the
last bits differ -- on the CPU, where the oracle transforms every field alone, the sharded run is bit exact:
tests/test_sharded_cpu.py), and match the oracle within the stepped-state tolerance (Q31)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import Oracle  # noqa: E402
from paper_2511_21891_b200 import sharded  # noqa: E402
from paper_2511_21891_b200.gandalf import Gandalf  # noqa: E402
from paper_2511_21891_b200.workloads import config2, rel_l2  # noqa: E402


def _close(a, b, tol=1e-13):
    return float(torch.linalg.vector_norm(a - b) / torch.linalg.vector_norm(b)) <= tol


def _raw_fields(g, nfields):
    raw = g.get_state_raw(device=True)
    return torch.view_as_complex(raw.view(nfields, -1, 2))


@pytest.mark.parametrize("shape,M,world,extra", [
    ((32, 32, 16), 8, 2, {}),
    ((64, 32, 16), 7, 3, dict(closure=1, if_variant=1)),
    ((32, 32, 16), 9, 4, dict(force_eps=0.5, force_nperp_min=1, force_nperp_max=2, force_nz_max=1, seed=5, force_g_amp=0.01, force_g_nz=1)),
])
def test_sharded_library_matches_unsharded(shape, M, world, extra):
    prm, z, g, run = config2(*shape, M)
    prm = dict(prm, **extra)
    nsteps = 6
    ref = Gandalf(*shape, **prm)
    ref.set_state(z, g)
    ref.step(run["dt"], nsteps)
    want = _raw_fields(ref, 2 + M)
    lays = [sharded.ShardLayout.make(M, world, r) for r in range(world)]
    shards = [sharded.GandalfShard(*shape, lay, **prm) for lay in lays]
    for sh in shards:
        sh.set_state(z, g)
    sharded.step_all(shards, lays, run["dt"], nsteps)
    got = torch.cat([sh.owned_raw() for sh in shards])
    assert _close(got, want[2:])
    for sh, lay in zip(shards, lays):
        assert torch.equal(_raw_fields(sh.g, 2 + lay.M_local)[:2], want[:2])
    e = np.array([sh.energy() for sh in shards])
    er = ref.energy()
    assert np.array_equal(e[:, :5], np.tile(er[:5], (world, 1)))
    assert abs(e[:, 5].sum() - er[5]) <= 1e-13 * er[5]
    # and the oracle agrees with the sharded run
    o = Oracle(*shape, **prm)
    o.set_state(z, g)
    o.step(run["dt"], nsteps)
    zs, gs = shards[0].g.get_state()
    zo, go = o.get_state()
    assert rel_l2(zs, zo) <= 1e-10
    own = lays[0].owned_local
    assert rel_l2(gs[own.start:own.stop], go[lays[0].lo:lays[0].hi]) <= 1e-10


def test_sharded_cfl_step_and_stage_protocol():
    shape, M, world = (32, 32, 16), 6, 2
    prm, z, g, run = config2(*shape, M)
    ref = Gandalf(*shape, **prm)
    ref.set_state(z, g)
    ref.step(-1.0, 3)                                               # Eq. 16 dt on the device, identical on every shard
    lays = [sharded.ShardLayout.make(M, world, r) for r in range(world)]
    shards = [sharded.GandalfShard(*shape, lay, **prm) for lay in lays]
    for sh in shards:
        sh.set_state(z, g)
    sharded.step_all(shards, lays, -1.0, 3)
    assert _close(torch.cat([sh.owned_raw() for sh in shards]), _raw_fields(ref, 2 + M)[2:])
    assert shards[0].g.time() == ref.time() == shards[1].g.time()
    # the stages must alternate, and a half-done step refuses step() and rhs()
    sh = shards[0]
    sh.step_stage(run["dt"], 0)
    with pytest.raises(Exception):
        sh.g.step(run["dt"], 1)
    with pytest.raises(Exception):
        sh.step_stage(run["dt"], 0)
    sh.step_stage(run["dt"], 1)
    with pytest.raises(Exception):
        sh.step_stage(run["dt"], 1)


def test_staged_step_equals_step():
    shape, M = (32, 32, 16), 5
    prm, z, g, run = config2(*shape, M)
    a, b = Gandalf(*shape, **prm), Gandalf(*shape, **prm)
    a.set_state(z, g)
    b.set_state(z, g)
    a.step(run["dt"], 4)
    for _ in range(4):
        b.step_stage(run["dt"], 0)
        b.step_stage(run["dt"], 1)
    assert torch.equal(a.get_state_raw(device=True), b.get_state_raw(device=True))
    assert np.array_equal(a.energy_history(), b.energy_history())


def _nccl_world1(rank, port, shape, M, nsteps, out_path):
    """One rank, NCCL backend: the path bench.py --parallelism mshard takes (DistExchange on the library's buffers), as far as
    one GPU can take it -- no halo moves with a single rank, but W_g goes through an NCCL all-reduce, which accepts CUDA tensors
    only (the energy record comes back from the library as a host array)."""
    import os
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=rank, world_size=1, device_id=torch.device("cuda", 0))
    try:
        prm, z, g, run = config2(*shape, M)
        lay = sharded.ShardLayout.make(M, 1, 0)
        sh = sharded.GandalfShard(*shape, lay, device=0, stream=torch.cuda.current_stream().cuda_stream, **prm)
        sh.set_state(z, g)
        st = sharded.ShardedStepper(sh, lay, sharded.DistExchange())
        st.step(run["dt"], nsteps)
        np.save(out_path, np.stack([st.energy(), sh.energy()]))
        sh.close()
    finally:
        dist.destroy_process_group()


def test_stepper_energy_reduces_over_nccl(tmp_path):
    import socket
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    out = str(tmp_path / "e.npy")
    mp.spawn(_nccl_world1, args=(port, (32, 32, 16), 4, 3, out), nprocs=1, join=True)
    e = np.load(out)
    assert np.array_equal(e[0], e[1]) and e[0, 5] > 0            # one rank: the reduced record is the shard's own
