"""N > 1 path of bench.py on CPU: two gloo ranks exercise the rank/seed assignment and the
max-over-ranks aggregation (replicas only, no data-path collective)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import bench
    from ttn_inputs import make_batch
    dist.init_process_group("gloo", rank=rank, world_size=world)
    r, lr, w = bench.rank_env()
    assert (r, lr, w) == (rank, rank, world)
    seed = bench.seed_for_rank(r)
    Jh, Jv, _ = make_batch(6, [seed], "pmj")
    local_ms = 100.0 + 10.0 * rank                       # rank 1 is the slow one
    step_ms = bench.max_over_ranks(local_ms, dist, "cpu")
    gathered = [None] * world
    dist.all_gather_object(gathered, (seed, Jv.tobytes().hex()))
    out.put((rank, step_ms, bench.whole_job_ms_per_instance(step_ms, w), gathered))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_aggregation():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, step_ms, per_inst, gathered in res:
        assert step_ms == 110.0                       # max over ranks, on every rank
        assert per_inst == 55.0                       # two instances per step in flight
        assert [g[0] for g in gathered] == [4000, 4001]   # distinct instances per rank
    assert res[0][3][0][1] != res[0][3][1][1]         # the two ranks really drew different couplings


def test_single_process_defaults(monkeypatch):
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        monkeypatch.delenv(k, raising=False)
    import bench
    assert bench.rank_env() == (0, 0, 1)
    assert bench.max_over_ranks(3.5, None) == 3.5
    assert bench.bytes_min(32) == 31 * 2 * 4 * 2.0 ** 32
    assert bench.updates(32) == 31 * 32 * 2.0 ** 32
