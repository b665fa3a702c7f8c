"""N > 1 path of bench.py on CPU (world_size 2, gloo): the path shards only across independent
sequences ("replicas only"), so what there is to check is the harness:
rank-distinct prompts, max-over-ranks timing, whole-job aggregation, and that the reference arm
(--impl reference) runs and prints on rank 0 only under torchrun."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    import dex_synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 * (rank + 1)                          # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, world)
    prompt = dex_synth.make_prompt(1024, 16, 4321, seq=bench.replica_prompt_seq(rank))
    out[rank] = (ms, bench.job_tokens_per_s(world, 3, 64, ms), prompt.tolist())
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_prompts_world2():
    import torch.multiprocessing as mp
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29611, out), nprocs=2, join=True)
    (ms0, v0, p0), (ms1, v1, p1) = out[0], out[1]
    assert ms0 == ms1 == 20.0                              # slowest rank's device time on every rank
    assert v0 == v1 == 2 * 3 * 64 / 20e-3                  # tokens of ALL ranks / that time
    assert p0 != p1                                        # independent sequences per replica
    assert len(p0) == 16 and max(p0) < 1024


def test_world1_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, 1) == 12.5
    assert bench.job_tokens_per_s(1, 2, 256, 1000.0) == 512.0


def test_reference_arm_rank0_only_under_torchrun():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29612", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--workload", "c1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                 # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "committed_tokens_per_s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["n_gpus"] == 2
