"""N > 1 path of bench.py on CPU (gloo, world_size 2): the method does not shard ("replicas
only"), so the only multi-process logic is the barrier, the MAX of the timed regions over the ranks and the whole-job
throughput; the reference arm must run on rank 0 alone."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["HFFT_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
dist.barrier()
mine = [10.0 + 5.0 * rank, 3.0 - rank]          # rank 1 is slower in the first region, rank 0 in the second
got = bench.max_over_ranks(mine)
value = bench.whole_job_value(world, 4, 10, got[0])
with open(os.path.join(os.environ["HFFT_OUT"], "r%d.json" % rank), "w") as fh:
    json.dump({"rank": rank, "world": world, "max": got, "value": value}, fh)
dist.destroy_process_group()
"""


def test_max_over_ranks_and_whole_job_value_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, HFFT_ROOT=ROOT, HFFT_OUT=str(tmp_path))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
           "127.0.0.1", "--master-port", "29517", str(script)]
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    outs = [json.loads((tmp_path / ("r%d.json" % k)).read_text()) for k in range(2)]
    for o in outs:
        assert o["world"] == 2
        assert o["max"] == [15.0, 3.0]                       # slowest rank per region, same on every rank
        assert abs(o["value"] - 2 * 4 * 10 / 15e-3) < 1e-6     # both replicas' evaluations over the slowest time


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert bench.whole_job_value(1, 32, 5, 10.0) == 32 * 5 / 10e-3


def test_reference_arm_runs_on_rank0_only(tmp_path):
    """Under torchrun the other ranks of `--impl reference` exit 0 without work and print nothing."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--config", "1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
