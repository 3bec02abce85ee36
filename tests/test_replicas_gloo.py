"""N>1 path of bench.py on CPU: world_size-2 gloo.  The path is 'replicas only' - no data-path collective -
so what is covered is the timing/aggregation protocol: barrier, MAX over ranks of time, SUM of units,
per-rank seeds giving different replicas."""
import os
import sys

import torch.multiprocessing as mpx

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2606_13126_b200 import dist, workloads as W
    r, lr, ws = dist.init(backend="gloo")
    assert (r, ws) == (rank, world)
    dist.barrier()
    w = W.small_variants(seed=11 + 1000 * rank)[0]          # replica seed = base + 1000 * rank, as bench.py does
    agg = dist.aggregate(units_this_rank=w.num_q_tokens, seconds_this_rank=0.5 + rank)
    dist.barrier()
    q.put((rank, agg, int(w.q.view("int16").astype("int64").sum())))
    dist.shutdown()


def test_two_replicas_aggregate_max_time_sum_units():
    ctx = mpx.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29631, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (r0, a0, s0), (r1, a1, s1) = got
    assert a0 == a1
    assert a0["seconds"] == 1.5 and a0["units"] == 2 * 720 and abs(a0["throughput"] - 1440 / 1.5) < 1e-9
    assert s0 != s1                                            # different seeds -> different replicas
