"""Process-group plumbing for the data-parallel launch (one process per GPU, torch.distributed).

The TNLM-E hot path has no collective on its data path when whole stacks are sharded over ranks
(independent 4D scans: weak scaling); timing is aggregated as the MAX over ranks.  The z-slab
partition of ONE stack (tnlm_jacobi_step_slab) needs one halo exchange of
M+d planes per sweep.  Two forms:

* `SlabLayout` / `SlabStack` / `enhance_z_slabs_local`: a rank stores only its slab plus the halo planes
  (strong scaling, what `bench.py --scaling strong` times); the exchange of the next iterate's boundary
  planes runs on a side stream while the interior of the current sweep is computed.
* `exchange_halos` / `enhance_z_slabs`: the first, simpler form on full-size arrays (kept for its tests).

Both are exercised with gloo on CPU tensors in tests/test_dist_gloo.py (the oracle stands in for the slab
sweep), and the slab-local form on one GPU by a loop-back exchange in tests/test_parity_gpu.py.
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


# ---------------------------------------------------------------------------------------------------------
# Slab-local storage: a rank holds [P][ZL][Y][X] arrays, ZL = pad + slab + halo


@dataclass
class SlabLayout:
    """Where a rank's planes of a Z-plane volume live in its local arrays.

    The rank owns global planes [a, b); local plane 0 is global plane `origin`, a multiple of the kernels'
    z-tile period (include/tnlm.h: tnlm_z_tile) so that the local tile grid coincides with the global one and the
    slab sweep reproduces the single-device sweep bit for bit.  Local planes: [lo - halo, lo) lower halo,
    [lo, hi) owned, [hi, hi + halo) upper halo; planes below lo - halo are alignment padding that no owned
    output reads."""
    Z: int
    a: int
    b: int
    halo: int
    origin: int

    @property
    def lo(self):
        return self.a - self.origin

    @property
    def hi(self):
        return self.b - self.origin

    @property
    def nz_local(self):
        return self.hi + self.halo


def slab_layout(Z: int, rank: int, world: int, halo: int, z_tile: int = 1) -> SlabLayout:
    a, b = z_slab(Z, rank, world)
    t = max(int(z_tile), 1)
    origin = ((a - halo) // t) * t          # floor: negative for the first rank (planes below 0 are copies of plane 0)
    return SlabLayout(Z, a, b, halo, origin)


class SlabStack:
    """A rank's local copy of one 4D stack: owned slab, halo planes and alignment padding (zeros)."""

    def __init__(self, layout: SlabLayout, own):
        import torch
        P, nb, Y, X = own.shape
        assert nb == layout.b - layout.a, "own must hold exactly the rank's planes [a, b)"
        self.layout = layout
        self.data = torch.zeros((P, layout.nz_local, Y, X), dtype=own.dtype, device=own.device)
        self.data[:, layout.lo:layout.hi].copy_(own)

    def owned(self):
        L = self.layout
        return self.data[:, L.lo:L.hi]


def _neighbours(info: RankInfo, L: SlabLayout):
    """(lower rank or None, upper rank or None) in z; slabs are contiguous and in rank order."""
    return (info.rank - 1 if L.a > 0 else None), (info.rank + 1 if L.b < L.Z else None)


def exchange_slab_halos(info: RankInfo, stack, L: SlabLayout):
    """Fill the halo planes of the local array `stack` ([P][ZL][Y][X]): from the z-neighbours where there is one
    (point-to-point, one message per phase and direction: a phase's planes are contiguous, no staging copy), by
    replicating the end plane where the slab touches the end of the volume (clamp-to-edge along z, reading P4).
    Every slab must hold at least `halo` planes.  Works on any backend; on CUDA tensors the caller picks the stream."""
    h = L.halo
    if h <= 0:
        return stack
    lower, upper = _neighbours(info, L)
    ops = []
    if info.distributed:
        import torch.distributed as dist
        assert L.b - L.a >= h or (lower is None and upper is None), "a slab must be at least M + d planes deep"
        P = stack.shape[0]
        for ph in range(P):
            if lower is not None:
                ops.append(dist.P2POp(dist.irecv, stack[ph, L.lo - h:L.lo], lower))
                ops.append(dist.P2POp(dist.isend, stack[ph, L.lo:L.lo + h], lower))
            if upper is not None:
                ops.append(dist.P2POp(dist.isend, stack[ph, L.hi - h:L.hi], upper))
                ops.append(dist.P2POp(dist.irecv, stack[ph, L.hi:L.hi + h], upper))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
    if lower is None:
        stack[:, L.lo - h:L.lo] = stack[:, L.lo:L.lo + 1]
    if upper is None:
        stack[:, L.hi:L.hi + h] = stack[:, L.hi - 1:L.hi]
    return stack


def halo_bytes_per_sweep(L: SlabLayout, info: RankInfo, shape_pyx, itemsize=4):
    """Bytes this rank sends per sweep (it receives the same amount)."""
    lower, upper = _neighbours(info, L)
    P, Y, X = shape_pyx
    return (int(lower is not None) + int(upper is not None)) * P * L.halo * Y * X * itemsize


def enhance_z_slabs_local(info: RankInfo, g_own, n_iter: int, halo: int, z_tile: int, Z: int, sweep_slab,
                          exchange=exchange_slab_halos):
    """TNLM-E on ONE stack split into z-slabs, every rank storing only its slab, halo and padding.

    g_own: this rank's planes [a, b) of g as [P][b-a][Y][X] (`z_slab(Z, rank, world)`).
    sweep_slab(f, g, z0, z1, out): writes out[:, z0:z1] of Eq. 8 from the local arrays f, g (on the GPUs:
    tnlm_jacobi_step_slab with nz = the local plane count; the CPU tests pass the oracle).

    Per sweep: the boundary planes of the slab (those a neighbour needs: the first and last `halo` rounded up to the
    z-tile) are computed first, their exchange for the NEXT sweep runs on a side stream while the interior planes are
    computed, and the next sweep waits for it.  Returns (SlabStack of f^(n_iter), SlabLayout).
    """
    import torch
    L = slab_layout(Z, info.rank, info.world, halo, z_tile)
    g = SlabStack(L, g_own)
    f = SlabStack(L, g_own)
    out = SlabStack(L, g_own)
    cuda = g_own.is_cuda
    exchange(info, f.data, L)                       # halos of f^0 = g
    t = max(int(z_tile), 1)
    hb = -(-halo // t) * t                          # boundary depth, in whole z-tiles
    lo_end = min(L.lo + hb, L.hi)
    hi_start = max(L.hi - hb, lo_end)
    main = torch.cuda.current_stream(g_own.device) if cuda else None
    side = torch.cuda.Stream(g_own.device) if cuda else None
    for k in range(int(n_iter)):
        sweep_slab(f.data, g.data, L.lo, lo_end, out.data)
        sweep_slab(f.data, g.data, hi_start, L.hi, out.data)
        last = k == int(n_iter) - 1
        if cuda:
            ev = torch.cuda.Event()
            ev.record(main)
            if not last:
                with torch.cuda.stream(side):
                    side.wait_event(ev)
                    exchange(info, out.data, L)
            sweep_slab(f.data, g.data, lo_end, hi_start, out.data)
            if not last:
                main.wait_stream(side)
        else:
            if not last:
                exchange(info, out.data, L)
            sweep_slab(f.data, g.data, lo_end, hi_start, out.data)
        f, out = out, f
    return f, L
