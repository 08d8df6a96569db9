"""world_size-2 gloo test (CPU) of bench.py's N > 1 arithmetic: columns shard over ranks with no data-path collective (band
partitioning with n_r = 1); the only cross-rank step is the MAX of the per-rank durations, and `value` is the
whole-job aggregate: world x units per rank / max time.  Also: under torchrun the reference arm runs on rank 0 alone."""
import io
import os
import socket
import sys
from contextlib import redirect_stdout

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r "measured" 10 (r + 1) ms for 5e9 units: the job took the slower rank's 20 ms for 2 x 5e9 units
    ms, value = bench.aggregate_over_ranks(10.0 * (rank + 1), 5e9, world, dist, "cpu")
    with open(os.path.join(out, f"r{rank}.txt"), "w") as f:
        f.write(f"{ms} {value}")
    # the reference arm (CPU oracle): every rank but 0 returns without work or output
    if rank != 0:
        buf = io.StringIO()
        with redirect_stdout(buf):
            bench.run_reference(None, None)
        assert buf.getvalue() == ""
    dist.barrier()
    dist.destroy_process_group()


def test_value_is_the_whole_job_aggregate_over_the_slowest_rank(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for r in range(2):
        ms, value = [float(t) for t in open(tmp_path / f"r{r}.txt").read().split()]
        assert ms == 20.0 and abs(value - 2 * 5e9 / 20e-3) < 1.0


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    ms, value = bench.aggregate_over_ranks(4.0, 8e9, 1)
    assert ms == 4.0 and value == 8e9 / 4e-3
