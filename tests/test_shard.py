"""Host logic of the multi-GPU path on CPU: row-block partition arithmetic and the gather of the
blocks over torch.distributed with the gloo backend, world size 2.  No method arithmetic runs here: the per-block
"map" is a stand-in that writes each pixel's own coordinates."""
import os
import socket

import numpy as np
import pytest

from paper_1902_03252_b200 import shard, workloads


def test_row_blocks_partition():
    for ny in (0, 1, 2, 7, 64, 1023, 4096):
        for world in (1, 2, 3, 8, 16):
            b = shard.row_blocks(ny, world)
            assert len(b) == world and b[0][0] == 0 and b[-1][1] == ny
            assert all(b[r][1] == b[r + 1][0] for r in range(world - 1))
            sizes = [j1 - j0 for j0, j1 in b]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard.row_blocks(5, 0)


def test_local_block_halo_and_origin():
    y_min, dx, ny = -100.0, 0.25, 101
    for world in (1, 2, 4):
        for rank in range(world):
            plain = shard.local_block(y_min, dx, ny, rank, world)
            halo = shard.local_block(y_min, dx, ny, rank, world, halo_below=True)
            assert plain.halo == 0 and plain.ny == plain.j1 - plain.j0 and plain.y_min == y_min + plain.j0 * dx
            assert halo.halo == (1 if rank > 0 else 0)          # the first block uses the forward neighbour (R12)
            assert halo.ny == plain.ny + halo.halo and halo.y_min == y_min + (plain.j0 - halo.halo) * dx
    # more ranks than rows: empty blocks get no halo
    b = shard.local_block(0.0, 1.0, 2, 3, 4, halo_below=True)
    assert b.j0 == b.j1 and b.halo == 0 and b.ny == 0


def _coords_map(lenses, x_min, y_min, dx, nx, ny, mode):
    """stand-in for lt_gradient_grid: pixel (i, j) -> its own coordinates (x, y)"""
    import torch
    j, i = torch.meshgrid(torch.arange(ny, dtype=torch.float64), torch.arange(nx, dtype=torch.float64), indexing="ij")
    return torch.stack([x_min + i * dx, y_min + j * dx], dim=-1)


def _stencil_map(lenses, x_min, y_min, dx, nx, ny, mode):
    """CPU stand-in for lt_gradient_grid with the data dependence of the mixed mode (eq. 24 / 27): in mode 2
    a pixel's value also depends on its LOWER neighbour's, and the first row of a call uses the forward neighbour (R12).
    Values are exact integers derived from the GLOBAL pixel indices (recovered from the coordinates), so the sharded and
    the unsharded maps can be compared bit for bit."""
    import torch
    jg = torch.round((y_min + torch.arange(ny, dtype=torch.float64) * dx - 5.0) / dx)           # global row index
    ig = torch.arange(nx, dtype=torch.float64)
    base = torch.stack([(jg[:, None] * 131.0 + ig[None, :] * 7.0) % 1009.0,
                        (jg[:, None] * 17.0 + ig[None, :] * 313.0) % 997.0], dim=-1)
    if mode != 2 or ny < 2:
        return base
    out = base.clone()
    out[1:] += 0.5 * base[:-1]
    out[0] += 0.5 * base[1]
    return out


def _worker_stencil(rank, world, port, ny, nx, ret):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        x_min, y_min, dx = -3.0, 5.0, 0.5
        ok = True
        for mode in (0, 2):
            b, out = shard.compute_block(_stencil_map, None, x_min, y_min, dx, nx, ny, mode, rank, world)
            assert b.halo == (1 if (mode == 2 and rank > 0) else 0)
            full = shard.all_gather_rows(out, ny, nx, rank, world)
            ref = _stencil_map(None, x_min, y_min, dx, nx, ny, mode)
            ok = ok and bool(torch.equal(full, ref))
            if mode == 2 and rank > 0:
                # without the halo row the block's first row would have used its forward neighbour: a different map
                wrong = _stencil_map(None, x_min, y_min + b.j0 * dx, dx, nx, b.j1 - b.j0, mode)
                ok = ok and not bool(torch.equal(wrong, ref[b.j0:b.j1]))
        ret[rank] = ok
    finally:
        dist.destroy_process_group()


def _worker(rank, world, port, ny, nx, mode, ret):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        x_min, y_min, dx = -3.0, 5.0, 0.5
        b, out = shard.compute_block(_coords_map, None, x_min, y_min, dx, nx, ny, mode, rank, world)
        if out is None:
            out = torch.zeros((0, nx, 2), dtype=torch.float64)
        assert out.shape[0] == b.j1 - b.j0
        full = shard.all_gather_rows(out, ny, nx, rank, world)
        ref = _coords_map(None, x_min, y_min, dx, nx, ny, mode)
        ok = bool(torch.allclose(full, ref, rtol=0, atol=1e-12)) and full.shape == ref.shape
        # the bench's per-rank catalogues (seed + rank) differ, and its max-over-ranks reduction works on gloo too
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ok = ok and t.item() == float(world)
        ret[rank] = ok
    finally:
        dist.destroy_process_group()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


@pytest.mark.parametrize("ny,mode", [(9, 0), (8, 2), (1, 2)])
def test_gather_world_size_2_gloo(ny, mode):
    import torch.multiprocessing as mp
    world = 2
    with mp.Manager() as m:
        ret = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), ny, 5, mode, ret), nprocs=world, join=True)
        assert dict(ret) == {0: True, 1: True}


@pytest.mark.parametrize("ny", [9, 16])
def test_mixed_halo_through_the_gather_world_size_2_gloo(ny):
    """compute_block with a map function that has the mixed mode's neighbour dependence, the blocks gathered over gloo:
    bit-equal to the unsharded map in both modes; the self-computed halo row is what makes it so."""
    import torch.multiprocessing as mp
    world = 2
    with mp.Manager() as m:
        ret = m.dict()
        mp.spawn(_worker_stencil, args=(world, _free_port(), ny, 6, ret), nprocs=world, join=True)
        assert dict(ret) == {0: True, 1: True}


def test_ranks_draw_their_own_catalogues():
    a = workloads.make(1, seed_offset=0)
    b = workloads.make(1, seed_offset=1)
    assert a.lenses.shape == b.lenses.shape and not np.array_equal(a.lenses, b.lenses)
    assert np.array_equal(a.lenses, workloads.make(1).lenses)
