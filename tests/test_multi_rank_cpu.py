"""N > 1 path on CPU (gloo, world_size 2): the path does not shard ("replicas only", DESIGN.md
section 9), so what there is to cover is bench.py's aggregation (bytes of all ranks over the
MAX of the ranks' times) and the reference arm's rank-0-only rule under torchrun."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank 1 is the slow one: the job's time is ITS time, the job's bytes are both ranks' bytes
    value, ms = bench.whole_job_value(step_bytes=10 ** 9, steps=4, world=world, ms_local=10.0 * (rank + 1),
                                      dist=dist, device="cpu")
    out[rank] = (value, ms)
    dist.barrier()
    dist.destroy_process_group()


def test_whole_job_value_is_all_bytes_over_max_time():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29731, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    value, ms = res[0]
    assert ms == 20.0
    assert abs(value - (10 ** 9 * 4 * 2) / 20e-3 / 1e9) < 1e-9


def test_reference_arm_prints_on_rank0_only_under_torchrun(tmp_path):
    """`bench.py --impl reference` under torchrun with 2 ranks: one JSON line, from rank 0."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29733", os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=str(tmp_path))
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["n_gpus"] == 2 and rec["value"] > 0
    assert rec["cpu_baseline"]["kind"] == "oracle" and rec["e2e"]["h2d_bytes_per_step"] == 0
