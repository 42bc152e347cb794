"""Timing aggregation of the multi-GPU benchmark (barrier, MAX over ranks of the device time, summed work) and the
rank-0-only reference arm, with world_size 2 on the gloo backend.  The data path of the N > 1 run -- one lattice split into
x-slabs -- is covered by tests/test_slab_gloo.py."""
import json
import os
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    from paper_2603_22553_b200 import replicas

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = 10.0 + 5.0 * rank            # rank 1 is the slow one
    updates = 1e9 * (rank + 1)
    glups, ms_max = replicas.aggregate_glups(updates, ms)
    q.put((rank, glups, ms_max, replicas.max_over_ranks(rank), replicas.sum_over_ranks(1.0)))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregation_takes_max_time_and_sums_work_over_two_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, glups, ms_max, mx, sm in got:
        assert ms_max == 15.0 and mx == 1.0 and sm == 2.0
        assert abs(glups - 3e9 / 15e-3 / 1e9) < 1e-9


def test_single_process_aggregation_is_the_identity():
    sys.path.insert(0, ROOT)
    from paper_2603_22553_b200 import replicas

    assert replicas.env_world()[0] >= 1
    glups, ms = replicas.aggregate_glups(2e9, 4.0)
    assert ms == 4.0 and abs(glups - 2e9 / 4e-3 / 1e9) < 1e-12


def test_reference_arm_runs_on_rank0_only_under_two_ranks():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 prints the line, rank 1 exits 0 silently."""
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), OMP_NUM_THREADS="2",
                   LPC_REF_SAMPLE_L="32")
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "3",
                            "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
