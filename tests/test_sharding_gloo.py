"""N > 1 host logic on CPU: two gloo ranks split the heads / layers of a layer and agree on a partition; the
max-over-ranks timing reduction returns the slowest rank's time (what bench.py reports under torchrun)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import saf3r_synth as sy


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import paper_2607_03612_b200 as sf
        from paper_2607_03612_b200 import sharding
        sh = sy.shape_c2()
        _, cfgs = sy.mixed_heads(sh)
        shape = sf.make_shape(sh.S, sh.T, sh.H, sh.D, sh.B)
        costs = sharding.head_costs(shape, cfgs)
        parts = sharding.assign_heads(costs, world)
        mine = parts[rank]
        gathered = [None] * world
        dist.all_gather_object(gathered, {"heads": mine, "costs": costs, "layers": sharding.layers_for_rank(24, rank, world)})
        slowest = sharding.max_over_ranks(10.0 + rank)          # rank r "took" 10 + r ms
        # the head-parallel split end to end on the host side (bench.py --shard heads): the sub-layer this rank would run
        sub_shape = sf.make_shape(sh.S, sh.T, len(mine), sh.D, sh.B)
        sub_entries, sub_ws = sf.query_sizes(sub_shape, [cfgs[h] for h in mine])
        full_entries, _ = sf.query_sizes(shape, cfgs)
        q.put((rank, gathered, slowest, sum(costs[h] for h in mine), sub_entries, full_entries, sub_ws))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_rank_partition_and_timing_reduction():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=100) for _ in range(world)]
    for p in procs:
        p.join(timeout=30)
        assert p.exitcode == 0
    res.sort()
    g0 = res[0][1]
    assert res[1][1] == g0                                       # both ranks saw the same gathered view
    assert g0[0]["costs"] == g0[1]["costs"]                      # closed-form costs agree without communication
    heads = sorted(g0[0]["heads"] + g0[1]["heads"])
    assert heads == list(range(16))                              # a partition: every head exactly once
    assert sorted(g0[0]["layers"] + g0[1]["layers"]) == list(range(24))
    assert res[0][2] == res[1][2] == 11.0                        # max over ranks
    loads = [res[0][3], res[1][3]]
    assert max(loads) <= 0.5 * sum(loads) + max(g0[0]["costs"])  # LPT bound: within one head of the even split
    # the two sub-layers list exactly the block pairs of the whole layer, and each rank's executed FLOP is 4*B^2*D per listed pair
    assert res[0][4] + res[1][4] == res[0][5] == res[1][5]
    sh = sy.shape_c2()
    assert [r[4] * 4 * sh.B * sh.B * sh.D for r in res] == loads
    assert res[0][6] > 0 and res[1][6] > 0


def test_assign_heads_properties():
    from paper_2607_03612_b200.sharding import assign_heads, layers_for_rank
    costs = [5, 9, 1, 9, 3, 3, 7]
    for world in (1, 2, 3, 8, 10):
        parts = assign_heads(costs, world)
        assert len(parts) == world and sorted(h for p in parts for h in p) == list(range(len(costs)))
        assert parts == assign_heads(costs, world)               # deterministic
    assert assign_heads(costs, 2) == [[1, 4, 5, 6], [0, 2, 3]] or sum(costs[h] for h in assign_heads(costs, 2)[0]) in (18, 19)
    assert layers_for_rank(5, 1, 2) == [1, 3]
    with pytest.raises(ValueError):
        assign_heads(costs, 0)
