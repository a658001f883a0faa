"""Row-block sharding of one deflection map across ranks.

Pixels are independent: a map of ny rows is cut into `world` contiguous row blocks, the lens catalogue is
replicated (56 B per lens) and nothing is exchanged while computing.  The mixed rule needs the lower neighbour of a
pixel (eq. 24 / 27): a block that does not start at row 0 computes one halo row below itself and drops
it, instead of receiving it from the neighbouring rank.  Only if one contiguous map is wanted on every rank are the
blocks gathered (`all_gather_rows`, torch.distributed; NCCL on GPUs, gloo in the CPU tests).

This module holds host logic only (index arithmetic and the optional collective).  The map of a block comes from the
callable `compute(lenses, x_min, y_min, dx, nx, ny, mode)` -- `lt.lt_gradient_grid` in production.  A block's first row
sits at fl(y_min + j0*dx), so its pixel coordinates can differ from the unsharded call's fl(y_min + fl(j*dx)) by one
rounding (1e-16 relative): blocks agree with the unsharded map to rounding level, not bit for bit.
"""
from collections import namedtuple

RowBlock = namedtuple("RowBlock", "rank j0 j1 halo y_min ny")


def row_blocks(ny, world):
    """[(j0, j1)] * world: contiguous, disjoint, covering [0, ny), sizes differing by at most one row (the first
    ny % world blocks are the longer ones).  Blocks may be empty when world > ny."""
    if ny < 0 or world < 1:
        raise ValueError("row_blocks: ny >= 0 and world >= 1 required")
    base, extra = divmod(ny, world)
    out, j = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((j, j + n))
        j += n
    return out


def local_block(y_min, dx, ny, rank, world, halo_below=False):
    """The rows rank `rank` computes: RowBlock(rank, j0, j1, halo, y_min_local, ny_local) with ny_local = j1 - j0 + halo
    rows starting `halo` rows below j0 (halo is 1 only if requested and j0 > 0)."""
    j0, j1 = row_blocks(ny, world)[rank]
    halo = 1 if (halo_below and j0 > 0 and j1 > j0) else 0
    return RowBlock(rank, j0, j1, halo, y_min + (j0 - halo) * dx, j1 - j0 + halo)


def compute_block(compute, lenses, x_min, y_min, dx, nx, ny, mode, rank, world, mixed_mode=2):
    """This rank's rows [j0, j1) of the global map as an array/tensor [j1 - j0, nx, 2] (None for an empty block)."""
    b = local_block(y_min, dx, ny, rank, world, halo_below=(mode == mixed_mode))
    if b.j1 == b.j0:
        return b, None
    out = compute(lenses, x_min, b.y_min, dx, nx, b.ny, mode)
    return b, out[b.halo:]


def all_gather_rows(block_out, ny, nx, rank, world, group=None):
    """Gathers the row blocks into the full [ny, nx, 2] map on every rank.  Blocks are padded to the longest block so
    that a plain all_gather serves (uneven blocks differ by at most one row)."""
    import torch
    import torch.distributed as dist
    blocks = row_blocks(ny, world)
    longest = max(j1 - j0 for j0, j1 in blocks)
    ref = block_out if block_out is not None else None
    if ref is None:
        raise ValueError("all_gather_rows: every rank needs a (possibly zero-row) tensor to fix dtype and device")
    pad = torch.zeros((longest, nx, 2), dtype=ref.dtype, device=ref.device)
    pad[: ref.shape[0]] = ref
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([parts[r][: j1 - j0] for r, (j0, j1) in enumerate(blocks)], dim=0)
