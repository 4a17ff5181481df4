"""CPU-only checks of bench.py's multi-rank plumbing ("replicas only": no data-path collective):
the max-over-ranks reduction under gloo with world_size 2, and the reference arm launched by torchrun with 2 ranks."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")        # rank 1 is the slow replica
    out[rank] = (ms, bench.whole_job_steps_per_s(ms, 50, world))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    port = _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms, sps = res[0]
    assert ms == 15.0                                  # the slowest replica sets the job time
    assert sps == pytest.approx(2 * 50 / 15e-3)        # whole-job aggregate: both replicas' steps over that time


def test_reference_arm_under_torchrun_two_ranks():
    """`bench.py --impl reference` under torchrun with 2 ranks: rank 0 alone runs the oracle and prints ONE JSON line."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--workload", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_algorithmic_bytes_match_the_survey_table():
    """bench.py's roofline numerators are SURVEY.md 8(d)'s formulas: 30.6 GB per step at config 4(a), 19.1 GB at 4(b), and the
    per-pass figures P1 8.5, P2 9.6, P3 5.1, P4 7.4 GB per step (two launches each)."""
    import bench
    per, step = bench.algorithmic_bytes((256, 256, 128), 32)
    assert abs(step / 1e9 - 30.63) < 0.01
    assert abs(2 * per["y_inverse_P1"] / 1e9 - 8.54) < 0.01 and abs(2 * per["x_pass_P2"] / 1e9 - 9.56) < 0.01
    assert abs(2 * per["y_forward_P3"] / 1e9 - 5.11) < 0.01 and abs(2 * per["z_step_P4"] / 1e9 - 7.42) < 0.01
    _, step_b = bench.algorithmic_bytes((512, 512, 256), 0)
    assert abs(step_b / 1e9 - 19.12) < 0.01


def test_moment_shard_layouts_used_by_the_bench():
    from paper_2511_21891_b200 import sharded
    lays = [sharded.ShardLayout.make(32, 4, r) for r in range(4)]
    assert [lay.hi - lay.lo for lay in lays] == [8, 8, 8, 8] and [lay.M_local for lay in lays] == [9, 10, 10, 9]
    assert lays[1].params() == dict(M=10, m_offset=7, M_global=32) and sharded.ShardLayout.make(32, 1, 0).params() == dict(M=32)


def test_bound_and_l2_note_follow_the_workload():
    """The bench line must not call a launch-bound small grid 'hbm', nor claim 'no flush needed' for a working set that fits
    the L2; on the large grids the larger of the two floors is the bound."""
    import bench
    per_launch, _ = bench.algorithmic_bytes((32, 32, 16), 0)
    b, note = bench.classify_bound(max(per_launch.values()), 1e-3, None)
    assert b == "launch/latency" and note.startswith("NOT flushed")
    per_launch, _ = bench.algorithmic_bytes((256, 256, 128), 32)
    dom = per_launch["x_pass_P2"]
    assert bench.classify_bound(dom, 0.73, 0.79)[0] == "alu"
    assert bench.classify_bound(dom, 0.73, 0.60)[0] == "hbm"
    b, note = bench.classify_bound(dom, 0.73, None)
    assert b == "hbm" and note.startswith("no flush needed") and "4.78 GB" in note
    per_launch, _ = bench.algorithmic_bytes((128, 128, 64), 32)
    assert bench.classify_bound(per_launch["x_pass_P2"], 0.1, None)[0] == "hbm"


def test_committed_ncu_figures_belong_to_the_current_kernel_sources():
    """roofline.traffic and roofline.alu.instr are copied from committed captures; the hash beside them must be the one of
    the kernel sources in this tree (re-capture and update profiles/r02_capture_sources.md after touching a kernel)."""
    import bench
    assert bench.captures_stale("r02") is False
    assert bench.captures_stale("no_such_round") is None
