"""N > 1 path on CPU: world_size 2 over gloo.  Functions are independent, so a batch sharded
by functions and lifted rank by rank must equal the batch lifted in one piece; here each rank lifts its shard
with the CPU oracle (this is a test: the product path has no CPU fallback), the columns are gathered with
gloo and compared == with the unsharded oracle result; the bench's max-over-ranks rule is checked too."""
import os
import socket

import numpy as np
import pytest

from paper_2505_24256_b200 import sharding, workloads as wl


def test_shard_functions_partition_is_exact_and_cost_balanced():
    ts = [7, 300, 5, 5, 5, 120, 64, 1, 90, 33]
    off = np.concatenate([[0], np.cumsum(ts)]).astype(np.int64)
    for world in (1, 2, 3, 4, 16):
        shards = [sharding.shard_functions(off, world, r) for r in range(world)]
        assert shards[0].f_lo == 0 and shards[-1].f_hi == len(ts)
        for a, b in zip(shards, shards[1:]):
            assert a.f_hi == b.f_lo and a.term_hi == b.term_lo
        for s in shards:
            assert s.offsets[0] == 0 and s.offsets[-1] == s.term_hi - s.term_lo
            assert (np.diff(s.offsets) == np.array(ts[s.f_lo:s.f_hi])).all()
    two = [sharding.shard_functions(off, 2, r) for r in range(2)]
    cost = [sum(t * t for t in ts[s.f_lo:s.f_hi]) for s in two]
    assert max(cost) <= 0.9 * sum(cost)  # the 300-term function does not drag everything to one rank
    with pytest.raises(ValueError):
        sharding.shard_functions(off, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist

    from oracle import ref

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.make_box_workload("shard", wl.SEED_BASE + 77, 5, 3, [40, 9, 65, 1, 30], 6, 4, dense=True)
        nodes = ref.eval_nodes(w.exps, w.anchors, w.p)
        vals = ref.power_sums(nodes, w.offsets, ref.poly_rows_eval(w.samples, w.planted, w.p), w.p, 0)
        sh = sharding.shard_functions(w.offsets, world, rank)
        lo, hi = sh.term_lo, sh.term_hi
        out, _, st = ref.zippel_lift_step(np.ascontiguousarray(w.exps[lo:hi]), sh.offsets, w.anchors, w.samples,
                                          np.ascontiguousarray(vals[:, lo:hi]), w.p, 0, 1)
        assert not st.any()
        full = sharding.gather_columns(torch.from_numpy(out.view(np.int64)), sh, w.T_tot).numpy().view(np.uint64)
        ms = sharding.max_over_ranks(10.0 + rank)
        seeds = [None] * world
        dist.all_gather_object(seeds, sharding.rank_seed_shift(rank))
        q.put((rank, bool((full == w.planted).all()), ms, seeds, (sh.f_lo, sh.f_hi)))
    finally:
        dist.destroy_process_group()


def test_sharded_lift_world_size_2_gloo():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    res = sorted(q.get(timeout=300) for _ in procs)
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    assert all(r[1] for r in res), "gathered sharded result differs from the planted coefficients"
    assert all(r[2] == 11.0 for r in res)  # max over ranks of (10, 11)
    assert res[0][3] == [0, 1000] and len({r[4] for r in res}) == 2
