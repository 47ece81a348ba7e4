"""Host-side logic of the N > 1 path (replicas only: no data-path collective): one seed per rank, the
max-over-ranks reduction of the timings, under a world_size-2 gloo group on CPU."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench

    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = dict(bench.WORKLOADS["cfg4_unbounded_256_f32"], n=16)
    inp = bench.make_input(w, rank)
    red = bench.max_over_ranks([1.0 + rank, 5.0 - rank], world, "cpu")
    q.put((rank, bench.rank_seed(4, rank), float(np.abs(inp["f"]).sum()), red))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, c0, m0), (r1, s1, c1, m1) = res
    assert s0 != s1 and c0 != c1          # independent problems per rank
    assert m0 == m1 == [2.0, 5.0]          # max over ranks, identical on every rank


def test_model_bytes_match_the_survey_table():
    import bench

    mb = bench.model_bytes(bench.WORKLOADS["cfg4_unbounded_256_f32"])
    assert [round(v / 1e6, 1) for v in mb] == [201.9, 404.2, 606.9, 404.2, 201.9]
    assert round(sum(mb) / 1e6) == 1819
    mb = bench.model_bytes(bench.WORKLOADS["cfg2_periodic_256_f32"])
    assert round(sum(mb) / 1e6) == 675
    mb = bench.model_bytes(bench.WORKLOADS["cfg5_vector_512_f32_curl"])
    assert abs(sum(mb) / 1e9 - 42.49) < 0.02
