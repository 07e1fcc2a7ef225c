"""Slab decomposition of a periodic box over ranks: host-side bookkeeping only.

The arithmetic of the method stays in the kernels: a rank's context (MPC(..., sub=(z0, nz))) streams its own particles
and adds the cell sums of the brick layers it shares with its neighbours into the neighbours' memory inside the sweep
kernel. This module holds what the processes have to agree on: who owns which cell layers, who the neighbours are,
and which rank a particle belongs to."""
import numpy as np


def slab_partition(nz, world, bz):
    """Own cell layers [z0, z0 + n) of every rank: whole brick layers (bz cell layers each), as even as possible.
    Every rank needs at least two brick layers and, with its halo of one brick layer on either side, at most nz."""
    nb = nz // bz
    if nz % bz or world < 2 or nb < 2 * world:
        raise ValueError("slab decomposition needs whole brick layers and at least two of them per rank")
    base, extra = divmod(nb, world)
    out, z = [], 0
    for r in range(world):
        n = (base + (1 if r < extra else 0)) * bz
        if n + 2 * bz > nz:
            raise ValueError("a slab and its two halo brick layers must fit into the box")
        out.append((z, n))
        z += n
    return out


def slab_neighbours(rank, world):
    """(rank below, rank above) along z, periodic"""
    return (rank - 1) % world, (rank + 1) % world


def slab_owner(z, a, parts):
    """rank that owns a particle at height z: the slab whose layers contain floor(z / a) (a particle exactly at the top
    of the box, which the wrap never produces, would go to rank 0)"""
    layer = np.floor(np.asarray(z, dtype=np.float64) / a).astype(np.int64)
    starts = np.array([p[0] for p in parts], dtype=np.int64)
    owner = np.searchsorted(starts, layer, side="right") - 1
    return np.clip(owner, 0, len(parts) - 1)
