"""Process-group plumbing for the data-parallel launch (one process per GPU, torch.distributed).

The TNLM-E hot path has no collective on its data path when whole stacks are sharded over ranks
(independent 4D scans: weak scaling); timing is aggregated as the MAX over ranks.  The z-slab
partition of ONE stack (tnlm_jacobi_step_slab) needs one halo exchange of
M+d planes per sweep; `exchange_halos` implements it with send/recv and is exercised with gloo on
CPU tensors in tests/test_dist_gloo.py.
"""
from __future__ import annotations

import os
from dataclasses import dataclass


@dataclass
class RankInfo:
    rank: int
    local_rank: int
    world: int

    @property
    def distributed(self):
        return self.world > 1


def rank_info() -> RankInfo:
    return RankInfo(int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
                    int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str) -> RankInfo:
    """Join the process group described by RANK/WORLD_SIZE/MASTER_* (no-op for a single process)."""
    info = rank_info()
    if info.distributed:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if not dist.is_initialized():
            dist.init_process_group(backend=backend, rank=info.rank, world_size=info.world)
    return info


def barrier(info: RankInfo):
    if info.distributed:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(info: RankInfo, value: float, device="cpu") -> float:
    """MAX of a per-rank scalar (elapsed time): the job is as slow as its slowest rank."""
    if not info.distributed:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(info: RankInfo, value: float, device="cpu") -> float:
    if not info.distributed:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def finalize(info: RankInfo):
    if info.distributed:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()


def z_slab(n: int, rank: int, world: int):
    """Balanced contiguous split of n planes over world ranks -> (start, stop)."""
    base, rem = divmod(n, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def exchange_halos(info: RankInfo, stack, halo: int):
    """Refresh the `halo` planes on each side of this rank's z-slab of `stack` ([P][Z][Y][X], every
    rank holds the full-size array but owns only its slab) from the ranks that own them.

    One exchange per Gauss-Jacobi sweep: a sweep of the slab reads f/ref within M+d planes of it
    (PAPER.md:176 with the window of PAPER.md:223), so halo = M + d.  Pure point-to-point, no
    reduction.  Works on any backend (gloo on CPU tensors in the tests, nccl on the GPUs).
    """
    if not info.distributed or halo <= 0:
        return stack
    import torch.distributed as dist
    Z = stack.shape[1]
    slabs = [z_slab(Z, r, info.world) for r in range(info.world)]
    a, b = slabs[info.rank]
    ops, keep = [], []
    for r, (ra, rb) in enumerate(slabs):
        if r == info.rank or ra == rb or a == b:
            continue
        # planes this rank needs that r owns
        need_lo, need_hi = max(a - halo, ra), min(a, rb)          # below my slab
        for lo, hi in ((need_lo, need_hi), (max(b, ra), min(b + halo, rb))):
            if lo < hi:
                buf = stack[:, lo:hi].contiguous()
                keep.append((buf, lo, hi))
                ops.append(dist.P2POp(dist.irecv, buf, r))
        # planes r needs that I own
        for lo, hi in ((max(ra - halo, a), min(ra, b)), (max(rb, a), min(rb + halo, b))):
            if lo < hi:
                ops.append(dist.P2POp(dist.isend, stack[:, lo:hi].contiguous(), r))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    for buf, lo, hi in keep:
        stack[:, lo:hi].copy_(buf)
    return stack


def enhance_z_slabs(info: RankInfo, g, n_iter: int, halo: int, sweep_slab):
    """TNLM-E on ONE stack sharded by z-slab over the ranks.

    Every rank holds full-size arrays `[P][Z][Y][X]` but owns only its slab `[a, b)` of planes (`z_slab`): per
    Gauss-Jacobi sweep it refreshes the `halo = M + d` planes next to its slab from its z-neighbours
    (`exchange_halos`, point-to-point, no reduction) and then computes its slab of Eq. 8 from the old iterate.
    `sweep_slab(f, g, a, b, out)` must write `out[:, a:b]` (on the GPUs: `tnlm_jacobi_step_slab`; the CPU tests
    pass the oracle).  Returns `(f, (a, b))`: the rank's copy after `n_iter` sweeps (valid in `[a, b)`) and its slab.
    Slab results equal the single-device sweep bit for bit (z-tiles are aligned to absolute plane indices).
    """
    Z = g.shape[1]
    a, b = z_slab(Z, info.rank, info.world)
    f = g.clone()
    out = g.clone()
    for _ in range(int(n_iter)):
        exchange_halos(info, f, halo)
        sweep_slab(f, g, a, b, out)
        f, out = out, f
    return f, (a, b)
