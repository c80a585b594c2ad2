"""The multi-process plumbing (paper_1201_2450_b200/dist.py) on CPU: world_size 2, gloo, 127.0.0.1.

The z-slab partition of one stack: every rank owns a contiguous slab of planes
of every phase and needs the M+d planes next to it from its neighbours before each sweep
(Eq. 8 reads f_{i+-1} inside the window of PAPER.md:223).  The tests check that
  * the slabs tile the volume,
  * exchange_halos delivers exactly the planes a sweep reads (everything else in the rank's copy is
    poisoned with NaN, so a missing plane shows up in the result),
  * two sweeps computed slab-wise on 2 ranks (oracle arithmetic, halo exchange in between) equal two
    sweeps of the whole stack bit for bit,
  * the max / sum reductions that bench.py uses for timing.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, shape, d, M, h, mu, n_sweeps, out_dir):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch
    from paper_1201_2450_b200 import dist as D
    from oracle import tnlm_oracle as O
    from tnlm_inputs import random_stack

    info = D.init("gloo")
    assert info.world == world and info.rank == rank
    P, Z, Y, X = shape
    g_full = random_stack(shape, 7)
    a, b = D.z_slab(Z, rank, world)

    # this rank's copy: its own slab is valid, everything else is poison
    f = np.full(shape, np.nan, dtype=np.float32)
    f[:, a:b] = g_full[:, a:b]
    plane = Y * X
    own = (np.arange(P)[:, None] * Z * plane + (np.arange(a * plane, b * plane))[None, :]).reshape(-1).astype(np.int64)
    for _ in range(n_sweeps):
        ft = torch.from_numpy(f)
        D.exchange_halos(info, ft, M + d)
        lo, hi = max(a - (M + d), 0), min(b + (M + d), Z)
        assert np.isfinite(f[:, lo:hi]).all(), "a plane inside the halo was not delivered"
        # the oracle clamps coordinates to the volume: give it finite values outside the halo that a
        # correct sweep never reads for this slab... it does not read them, so any value works
        work = np.where(np.isfinite(f), f, np.float32(1e30))
        new = O.jacobi_step_at(work, g_full, d, M, np.float32(h), np.float32(mu), own)
        f = np.full(shape, np.nan, dtype=np.float32)
        f.reshape(-1)[own] = new
    np.save(os.path.join(out_dir, f"slab{rank}.npy"), f[:, a:b])

    t = D.max_over_ranks(info, float(rank + 1))
    s = D.sum_over_ranks(info, float(rank + 1))
    assert t == float(world) and s == world * (world + 1) / 2
    D.barrier(info)
    D.finalize(info)


def _worker_enhance(rank, world, port, shape, d, M, h, mu, n_sweeps, out_dir):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch
    from paper_1201_2450_b200 import dist as D
    from oracle import tnlm_oracle as O
    from tnlm_inputs import random_stack

    info = D.init("gloo")
    P, Z, Y, X = shape
    g = torch.from_numpy(random_stack(shape, 7))
    plane = Y * X

    def sweep_slab(f, gg, a, b, out):
        own = (np.arange(P)[:, None] * Z * plane + np.arange(a * plane, b * plane)[None, :]).reshape(-1).astype(np.int64)
        new = O.jacobi_step_at(f.numpy(), gg.numpy(), d, M, np.float32(h), np.float32(mu), own)
        out.view(-1)[torch.from_numpy(own)] = torch.from_numpy(new)

    f, (a, b) = D.enhance_z_slabs(info, g, n_sweeps, M + d, sweep_slab)
    np.save(os.path.join(out_dir, f"enh{rank}.npy"), f[:, a:b].numpy())
    D.barrier(info)
    D.finalize(info)


def _worker_local(rank, world, port, shape, d, M, h, mu, n_sweeps, z_tile, out_dir):
    """Slab-local storage: the rank never sees more than its slab of g; halos travel by exchange_slab_halos."""
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch
    from paper_1201_2450_b200 import dist as D
    from oracle import tnlm_oracle as O
    from tnlm_inputs import random_stack

    info = D.init("gloo")
    P, Z, Y, X = shape
    a, b = D.z_slab(Z, rank, world)
    g_own = torch.from_numpy(np.ascontiguousarray(random_stack(shape, 7)[:, a:b]))
    plane = Y * X

    def sweep_slab(f, gg, z0, z1, out):
        if z1 <= z0:
            return
        ZL = f.shape[1]
        own = (np.arange(P)[:, None] * ZL * plane + np.arange(z0 * plane, z1 * plane)[None, :]).reshape(-1).astype(np.int64)
        new = O.jacobi_step_at(f.numpy(), gg.numpy(), d, M, np.float32(h), np.float32(mu), own)
        out.view(-1)[torch.from_numpy(own)] = torch.from_numpy(new)

    f, L = D.enhance_z_slabs_local(info, g_own, n_sweeps, M + d, z_tile, Z, sweep_slab)
    assert (L.a, L.b) == (a, b) and L.origin % z_tile == 0 and L.lo >= M + d
    assert f.data.shape[1] == L.nz_local < Z + 2 * (M + d) + z_tile
    np.save(os.path.join(out_dir, f"loc{rank}.npy"), f.owned().numpy())
    assert D.halo_bytes_per_sweep(L, info, (P, Y, X)) == (2 if 0 < rank < world - 1 else 1) * P * (M + d) * Y * X * 4
    D.barrier(info)
    D.finalize(info)


@pytest.mark.parametrize("world,Z,d,M,z_tile", [(2, 9, 1, 2, 4), (3, 13, 1, 1, 4), (2, 8, 2, 1, 12)])
def test_slab_local_enhancement_equals_single_process(tmp_path, oracle, world, Z, d, M, z_tile):
    """Every rank stores only slab + halo (+ tile-alignment padding) and the result still equals TNLM-E on the whole
    stack bit for bit: halo exchange, end-plane replication and the local/global index maps are right."""
    import torch.multiprocessing as mp
    shape, h, mu, n_sweeps = (3, Z, 6, 7), 0.3, 0.7, 3
    mp.spawn(_worker_local, args=(world, _free_port(), shape, d, M, h, mu, n_sweeps, z_tile, str(tmp_path)),
             nprocs=world, join=True)
    from tnlm_inputs import random_stack
    want = oracle.enhance(random_stack(shape, 7), d, M, np.float32(h), np.float32(mu), n_sweeps)
    got = np.concatenate([np.load(tmp_path / f"loc{r}.npy") for r in range(world)], axis=1)
    assert np.array_equal(got, want)


def test_slab_layouts():
    from paper_1201_2450_b200 import dist as D
    for Z, world, halo, t in ((128, 8, 3, 4), (100, 8, 4, 6), (128, 4, 3, 12), (9, 2, 3, 4), (5, 1, 2, 1)):
        prev_b = 0
        for r in range(world):
            L = D.slab_layout(Z, r, world, halo, t)
            assert L.a == prev_b and L.origin % t == 0 and halo <= L.lo < halo + t and L.hi - L.lo == L.b - L.a
            prev_b = L.b
        assert prev_b == Z


def test_enhance_z_slabs_two_ranks_equals_single_process(tmp_path, oracle):
    import torch.multiprocessing as mp
    shape, d, M, h, mu, n_sweeps, world = (3, 9, 6, 7), 1, 2, 0.3, 0.7, 3, 2
    mp.spawn(_worker_enhance, args=(world, _free_port(), shape, d, M, h, mu, n_sweeps, str(tmp_path)), nprocs=world,
             join=True)
    from tnlm_inputs import random_stack
    g = random_stack(shape, 7)
    want = oracle.enhance(g, d, M, np.float32(h), np.float32(mu), n_sweeps)
    got = np.concatenate([np.load(tmp_path / f"enh{r}.npy") for r in range(world)], axis=1)
    assert np.array_equal(got, want)


def test_z_slabs_tile_the_volume():
    from paper_1201_2450_b200 import dist as D
    for n in (1, 5, 16, 100, 128):
        for world in (1, 2, 3, 8):
            slabs = [D.z_slab(n, r, world) for r in range(world)]
            assert slabs[0][0] == 0 and slabs[-1][1] == n
            assert all(slabs[i][1] == slabs[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in slabs]
            assert max(sizes) - min(sizes) <= 1


@pytest.mark.parametrize("d,M,Z", [(1, 2, 9), (1, 1, 4), (2, 1, 7)])
def test_two_rank_slab_sweeps_equal_the_full_sweeps(tmp_path, oracle, d, M, Z):
    import torch.multiprocessing as mp
    shape = (3, Z, 6, 7)
    h, mu, n_sweeps, world = 0.3, 0.7, 2, 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, shape, d, M, h, mu, n_sweeps, str(tmp_path)), nprocs=world, join=True)

    from tnlm_inputs import random_stack
    from paper_1201_2450_b200 import dist as D
    g = random_stack(shape, 7)
    want = g
    for _ in range(n_sweeps):
        want = oracle.jacobi_step(want, g, d, M, np.float32(h), np.float32(mu))
    got = np.concatenate([np.load(tmp_path / f"slab{r}.npy") for r in range(world)], axis=1)
    assert got.shape == want.shape
    assert np.array_equal(got, want), "slab-wise sweeps with halo exchange differ from the full sweeps"


def test_single_process_is_a_no_op():
    import torch
    from paper_1201_2450_b200 import dist as D
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    info = D.init("gloo")
    assert not info.distributed
    x = torch.arange(24.0).reshape(1, 4, 2, 3)
    assert D.exchange_halos(info, x, 2) is x
    assert D.max_over_ranks(info, 3.5) == 3.5 and D.sum_over_ranks(info, 3.5) == 3.5
    D.barrier(info)
    D.finalize(info)
