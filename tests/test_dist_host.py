"""N > 1 host logic of bench.py on CPU: gloo backend, world size 2 (no GPU, no CUDA path).

The hot path shards by (sequence, KV head) row with no exchange step, so the only
multi-process code is bench.py's plumbing: rank environment, per-rank seeds, the max-over-ranks of the device
time, rank-0-only output, and the reference arm in which only rank 0 works."""
import json
import os
import subprocess
import sys

import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench
    r, l, w = bench.rank_env()
    dist = bench.dist_init(w, l, use_cuda=False)
    ms = 10.0 + 5.0 * r                          # rank 1 is the slow one
    dist.barrier()
    whole = bench.max_over_ranks(ms, dist)
    q.put((r, l, w, whole, bench.rank_seed_offset(r)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_rank_env_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [x[0] for x in res] == [0, 1] and all(x[2] == 2 for x in res)
    assert all(x[3] == 15.0 for x in res)         # every rank sees the slowest rank's time
    assert res[0][4] != res[1][4]                 # different seeds: different sequences per rank


def test_single_process_needs_no_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.dist_init(1, 0, use_cuda=False) is None
    assert bench.max_over_ranks(3.5, None) == 3.5


def test_reference_arm_under_torchrun_world2():
    """`bench.py --impl reference` launched like the driver does for N = 2: rank 0 alone times the oracle and prints
    ONE JSON line, rank 1 exits 0 without work."""
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--config", "C0", "--steps", "2", "--warmup", "1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT,
                       env=dict(os.environ, CUDA_VISIBLE_DEVICES=""))
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["higher_is_better"] is False
