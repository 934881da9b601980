"""N > 1 path of bench.py on CPU: two gloo ranks shard the events, time is reduced with MAX, rank 0
aggregates (events are independent, no data-path collective)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2508_07423_b200 import synth
    cfg = synth.CONFIGS["c2"]
    ids = list(bench.shard_event_ids(cfg, rank, 3))
    batch = synth.generate_events(cfg, ids)
    ms = bench.reduce_max(10.0 * (rank + 1))               # rank 1 is the slow one
    out.put((rank, ids, int(len(batch["r"])), ms, bench.aggregate_events_per_s(world, 3, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_sharding():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ids0, n0, ms0, v0), (r1, ids1, n1, ms1, v1) = res
    assert ids0 == [0, 1, 2] and ids1 == [3, 4, 5]           # disjoint shards of the same stream
    assert ms0 == ms1 == 20.0                                # max over ranks
    assert v0 == v1 == 2 * 3 / 0.020                         # all ranks' events / slowest rank's time
    # the shards are what a single process would generate for those ids
    from paper_2508_07423_b200 import synth
    both = synth.generate_events(synth.CONFIGS["c2"], range(6))
    assert n0 + n1 == len(both["r"])


def test_single_process_helpers():
    import bench
    assert bench.reduce_max(3.5) == 3.5
    assert bench.aggregate_events_per_s(1, 1000, 100.0) == 10000.0
    fl = bench.path_flops(__import__("paper_2508_07423_b200.synth", fromlist=["x"]).CONFIGS["c2"], 10, 60)
    H = 128
    assert fl["edge_net"] == 6 * 60 * 2 * (3 * H * H + H * H + H * H)      # 10 H^2 FLOP per edge and step
    assert fl["scatter"] == 6 * 2 * 60 * H


def test_pair_test_count_is_the_edge_count_at_infinite_radius():
    """bench.py's pair-test count (the denominator of the graph stage's ALU fraction) against the oracle's search
    with r -> infinity on a ragged multi-event batch, for G = 1..3 (SURVEY 8(c) closed form)."""
    import bench
    from oracle import etx_oracle as orc
    from paper_2508_07423_b200 import synth
    cfg = synth.CONFIGS["c2"]
    batch = synth.generate_events(cfg, [5, 6, 300])
    emb = np.zeros((len(batch["r"]), 4), np.float32)
    for gap in (1, 2, 3):
        s, _ = orc.build_graph(batch["event_ptr"], batch["plane"], emb, np.inf, gap)
        assert bench.pair_tests(batch, gap) == len(s)
    assert bench.pair_tests(synth.generate_events(cfg, []), 3) == 0
