"""Multi-GPU path of bench.py (replicas only, no data-path collective): the
whole-job value is work summed over ranks divided by the MAX time over ranks.  world_size 2, gloo,
on CPU."""
import os
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 100.0 if rank == 0 else 250.0          # rank 1 is the slow replica
    value, ms = bench.whole_job(ms_local, 1_000_000, dist, "cpu")
    out.put((rank, value, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_whole_job_value_is_sum_of_work_over_max_time():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms in res:
        assert ms == 250.0                             # max over ranks
        assert value == 2 * 1_000_000 / 0.25           # both replicas' work


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    value, ms = bench.whole_job(50.0, 10)
    assert ms == 50.0 and value == 200.0


def test_reference_arm_other_ranks_do_no_work(monkeypatch, capsys):
    """--impl reference under torchrun: rank 0 alone runs and prints; the others exit 0."""
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")

    class A:
        workload, steps, warmup, gpus = "cfg1", 1, 0, 2
    bench.run_reference(A)
    assert capsys.readouterr().out == ""
