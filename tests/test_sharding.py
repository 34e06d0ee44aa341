"""The N > 1 path: events sharded over ranks, one all-reduce of the tallies.
Covered here on CPU with the `gloo` backend and world_size 2; the per-rank engine is the oracle
(the GPU library needs a device), the sharding and reduction code is the product's
(paper_2302_08252_b200/sharding.py)."""
import os
import socket

import numpy as np
import pytest

from paper_2302_08252_b200.sharding import reduce_results, run_sharded, shard_range
from workloads import CONFIGS, gen_primaries, geometry_for, tables_for


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 16, 1000, 1001):
        for world in (1, 2, 3, 8):
            cuts = [shard_range(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


class _OracleCtx:
    """The oracle behind the four calls run_sharded() makes on a Context."""

    def __init__(self, seed):
        from oracle import Oracle
        self.o = Oracle(geometry_for("tiny"), tables_for("tiny"), seed=seed)
        self.device = None

    def set_primary_index(self, i):
        self.o.set_primary_index(i)

    def inject(self, p):
        self.o.inject(p)

    def run(self):
        self.o.run()
        return self.o.result()


def _rank_main(rank, world, port, n_primaries, seed, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        prim = gen_primaries(n_primaries, CONFIGS["tiny"]["e_primary"])
        res = run_sharded(_OracleCtx(seed), prim, rank, world)
        if rank == 0:
            q.put({k: (v.tolist() if isinstance(v, np.ndarray) else v) for k, v in res.items()})
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_run_equals_single_rank_run():
    import torch.multiprocessing as mp
    from oracle import build
    build()                                   # compile once, before the ranks race for it
    n, seed, world = 13, 7, 2                 # odd count: ranks get 7 and 6 primaries
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, n, seed, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    got = q.get()
    ref = _OracleCtx(seed)
    ref.inject(gen_primaries(n, CONFIGS["tiny"]["e_primary"]))
    want = ref.run()
    for k in ("steps", "secondaries", "killed", "escaped_n", "live"):
        assert list(want[k]) == list(got[k]), k
    assert got["iterations"] == want["iterations"]       # ranks iterate side by side: max
    assert np.allclose(got["edep_slab"], want["edep_slab"], rtol=1e-12, atol=1e-12)
    assert abs(got["e_escaped"] - want["e_escaped"]) <= 1e-12 * max(1.0, want["e_escaped"])
    assert abs(got["e_injected"] - want["e_injected"]) <= 1e-12 * want["e_injected"]
    # a split that ignored the global primary index re-uses the ids 0..5 for the second slice:
    # other random streams, another result
    prim = gen_primaries(n, CONFIGS["tiny"]["e_primary"])
    a, b = _OracleCtx(seed), _OracleCtx(seed)
    a.inject(prim[:7])
    b.inject(prim[7:])
    naive = [int(x) + int(y) for x, y in zip(a.run()["steps"], b.run()["steps"])]
    assert naive != [int(x) for x in want["steps"]]


def test_reduce_results_single_process_group_is_identity():
    import torch.distributed as dist
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=0, world_size=1)
    try:
        c = _OracleCtx(3)
        c.inject(gen_primaries(4, 10.0))
        r = c.run()
        out = reduce_results(r)
        assert np.array_equal(out["edep_slab"], r["edep_slab"]) and out["iterations"] == r["iterations"]
        assert np.allclose(out["edep_layer"], r["edep_layer"], rtol=1e-15)
        for k in ("steps", "secondaries", "killed", "escaped_n", "live", "slots_used"):
            assert list(out[k]) == list(r[k])
    finally:
        dist.destroy_process_group()
