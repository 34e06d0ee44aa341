"""Multi-GPU use of the library: one process per GPU, events sharded, one reduction at the end.

Showers started by different primaries never interact: geometry and tables are
replicated, every rank runs its own context on a contiguous slice of the primary list, and the only
exchange is one all-reduce of the tallies (2*n_layers + 2 doubles and a few integers) when the run
is over -- there is no collective on the data path.  Primary ids depend only on the *global*
primary index (rule R4, `adept_set_primary_index`), so the summed result does not depend on how
the list was split.  Plumbing only: nothing here touches a track.
"""
from __future__ import annotations

import numpy as np

SUM_KEYS = ("steps", "secondaries", "killed", "escaped_n", "live")


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous slice [lo, hi) of n items owned by `rank`; sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world of %d" % (rank, world))
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def reduce_results(res: dict, device=None, group=None) -> dict:
    """All-reduce one rank's `Context.run()` / `Context.result()` dict over the process group.
    Energies and counts add up; `iterations`, `slots_used` and `overflow` take the maximum (ranks
    iterate side by side, and slot use is a per-GPU high-water mark)."""
    import torch
    import torch.distributed as dist
    n_slabs = res["edep_slab"].shape[0]
    f = torch.tensor(np.concatenate([res["edep_slab"], [res["e_escaped"], res["e_injected"]]]),
                     dtype=torch.float64, device=device)
    s = torch.tensor(np.concatenate([np.asarray(res[k], dtype=np.int64) for k in SUM_KEYS]),
                     dtype=torch.int64, device=device)
    m = torch.tensor(np.concatenate([[res["iterations"], res.get("overflow", 0)],
                                     np.asarray(res["slots_used"], dtype=np.int64)]),
                     dtype=torch.int64, device=device)
    dist.all_reduce(f, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(s, op=dist.ReduceOp.SUM, group=group)
    dist.all_reduce(m, op=dist.ReduceOp.MAX, group=group)
    f, s, m = f.cpu().numpy(), s.cpu().numpy(), m.cpu().numpy()
    out = {k: s[3 * i:3 * i + 3].astype(np.uint64) for i, k in enumerate(SUM_KEYS)}
    out.update(edep_slab=f[:n_slabs].copy(), edep_layer=f[:n_slabs].reshape(-1, 2).sum(axis=1),
               e_escaped=float(f[n_slabs]), e_injected=float(f[n_slabs + 1]),
               iterations=int(m[0]), overflow=int(m[1]), slots_used=m[2:5].astype(np.uint64))
    return out


def run_sharded(ctx, primaries: np.ndarray, rank: int, world: int, group=None, device=None) -> dict:
    """Inject this rank's slice of `primaries` with their global indices, run to completion, reduce
    (on `device`, default the context's: NCCL reduces device tensors, gloo host tensors)."""
    lo, hi = shard_range(primaries.shape[0], rank, world)
    ctx.set_primary_index(lo)
    ctx.inject(primaries[lo:hi])
    res = ctx.run()
    return reduce_results(res, device=device if device is not None else getattr(ctx, "device", None), group=group)
