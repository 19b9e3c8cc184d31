"""The N > 1 path of bench.py on CPU: two `gloo` ranks.  The hot path has no exchange step (states
are independent, "replicas only"), so the multi-rank logic is the MAX of the
device-timed milliseconds over the ranks, the whole-job value, and rank 0 alone printing."""
import json
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, {root!r})
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")      # rank 1 is the slow one
    value = bench.whole_job_value(world, 1000, ms / 4)
    dist.barrier()
    if rank == 0:
        print(json.dumps({{"ms": ms, "value": value, "n_gpus": world}}))
    dist.destroy_process_group()
""")


def test_two_gloo_ranks_take_the_max_and_rank0_prints(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29611", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2
    assert d["ms"] == 15.0                                   # max over ranks
    assert abs(d["value"] - 2 * 1000 / (15.0 / 4 * 1e-3)) < 1e-6


def test_single_rank_is_a_no_op():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.whole_job_value(1, 100000, 2.0) == 100000 / 2.0e-3


def test_reference_arm_non_zero_ranks_do_no_work():
    """`--impl reference` under torchrun: rank 0 alone runs and prints; the others exit 0 silently."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0
    assert res.stdout.strip() == ""
