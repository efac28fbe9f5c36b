"""N > 1 path on CPU: world_size-2 gloo run of the replica plumbing bench.py uses (seed offsets, barrier, MAX over
ranks, whole-job aggregate), and `bench.py --impl reference` under a 2-rank launch (rank 0 alone prints the line)."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    from paper_2410_09189_b200 import replicas as R
    from paper_2410_09189_b200.workloads import WORKLOADS, eigenvalues_occ
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert R.rank_env() == (rank, world, rank)
    w = R.replica_workload(WORKLOADS["tiny"], rank)
    eps, _ = eigenvalues_occ(w)
    dist.barrier()
    ms = [10.0 + 5.0 * rank, 7.0 - rank]                      # rank 1 is slower on the first, faster on the second
    mx = R.max_over_ranks(ms)
    dist.barrier()
    q.put((rank, w.seed, float(eps[0]), mx, R.whole_job_steps_per_s(4, world, mx[0])))
    dist.destroy_process_group()


def test_replicas_world2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, e0, m0, v0), (r1, s1, e1, m1, v1) = out
    assert (r0, r1) == (0, 1) and s1 == s0 + 100 and e0 != e1          # independent seeded systems
    assert m0 == m1 == [15.0, 7.0]                                      # MAX over ranks, seen by every rank
    assert v0 == v1 == 2 * 4 / 15.0e-3                                  # whole-job steps/s over the slowest rank


def test_reference_arm_two_ranks_prints_once():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", WORLD_SIZE="2", OMP_NUM_THREADS="2")
    outs = []
    for rank in (0, 1):
        e = dict(env, RANK=str(rank), LOCAL_RANK=str(rank))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny",
                            "--gpus", "2", "--steps", "2", "--warmup", "1"], env=e, capture_output=True, text=True,
                           timeout=300)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["unit"] == "steps/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["config"]["workload"] == "tiny"
