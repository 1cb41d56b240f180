"""The N>1 host logic of bench.py on CPU: two ranks over gloo (world_size 2, 127.0.0.1).

The path shards by blocks with no data-path collective: every rank evaluates its own
seeded block(s); the only communication is the barrier and the max-over-ranks reduction of the step time.  The
test checks that reduction, the whole-job rate, that the ranks' workloads have the same shape but different data,
and that the reference arm leaves all work to rank 0."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        t_local = 0.010 * (rank + 1)                       # rank 1 is the slow one
        t_max = bench.max_over_ranks(t_local, world, "cpu")
        prob = bench.load_workload("c5-32", rank, nbox=2)
        dist.barrier()
        rate = bench.whole_job_rate(prob.cells, world, 4, t_max)
        np.savez(os.path.join(out, f"rank{rank}.npz"), t_max=t_max, rate=rate, cells=prob.cells,
                 shape=np.array(prob.prim.shape), head=prob.prim[0, 0, 5, 5, :8])
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0, r1 = (np.load(tmp_path / f"rank{r}.npz") for r in (0, 1))
    assert r0["t_max"] == pytest.approx(0.020) and r1["t_max"] == pytest.approx(0.020)      # max, on both ranks
    assert np.array_equal(r0["shape"], r1["shape"]) and r0["cells"] == r1["cells"] == 2 * 32 ** 3
    assert not np.array_equal(r0["head"], r1["head"])                                       # own seeds per rank
    assert r0["rate"] == pytest.approx(2 * 2 * 32 ** 3 * 4 / 0.020) == r1["rate"]           # all ranks' cells / max time


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
