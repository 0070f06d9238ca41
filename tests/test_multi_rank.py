"""The N > 1 path is "replicas only": its whole host logic is the max-over-ranks reduction of
bench.py and the rule that the reference arm runs on rank 0 alone.  Both are covered here on CPU with gloo, world size 2."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    got = bench.max_over_ranks([1.0 + rank, 10.0 - rank, 0.5], torch.device("cpu"), world)
    dist.barrier()
    dist.destroy_process_group()
    out[rank] = got


def test_max_over_ranks_gloo_world2():
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, 29611, out), nprocs=2, join=True)
        assert out[0] == out[1] == [2.0, 10.0, 0.5]


def test_max_over_ranks_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks([3.0, 4.5], None, 1) == [3.0, 4.5]


def test_reference_arm_under_torchrun_prints_one_line():
    """torchrun, 2 ranks, --impl reference on the tiny workload: rank 0 alone runs the oracle and prints ONE JSON line
    carrying impl / cpu_baseline / e2e; the other rank exits 0 without work."""
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
                        "--master-port", "29612", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--workload", "tiny"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["n_gpus"] == 2 and j["cpu_baseline"]["kind"] == "oracle"
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["value"] > 0
