"""N > 1 launch ("replicas only"): the host-side logic under a world_size-2 gloo group on CPU,
and the contract that `bench.py --impl reference` prints one line from rank 0 only."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_1409_4923_b200 import replicas
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    elapsed = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    q.put((rank, replicas.max_over_ranks(elapsed, dist), replicas.replica_seed(14094923, rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_seeds_world_size_2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [15.0, 15.0]        # both ranks see the slowest rank's time
    assert got[0][2] != got[1][2]                     # distinct ensembles


def test_single_process_identities():
    from paper_1409_4923_b200 import replicas
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.whole_job_value(1000, 4, 2.0) == 4 * 1000 / 2e-3
    assert replicas.replica_seed(2 ** 64 - 1, 1) == 0


def test_replica_seeds_give_independent_words(orc):
    a = np.array([orc.philox_call(14094923, g, 1, 0) for g in range(64)], dtype=np.uint64)
    b = np.array([orc.philox_call(14094924, g, 1, 0) for g in range(64)], dtype=np.uint64)
    assert not np.any(a == b)
    # bit agreement between the two ensembles is that of independent words: 50 % +- 4 sigma
    same = np.unpackbits((a ^ b).astype(">u4").view(np.uint8)).size - np.unpackbits((a ^ b).astype(">u4").view(np.uint8)).sum()
    n = 64 * 4 * 32
    assert abs(same - n / 2) < 4 * (n / 4) ** 0.5


def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(29700 + (os.getpid() % 200)), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--workload", "C0", "--cpu-seconds", "0.5"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
