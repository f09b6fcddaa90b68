"""Host logic of the regular domain decomposition whose halo exchange is fused into the ghost-fill kernel (include/mhd.h,
"Domain decomposition"; PAPER.md:592 spatial decomposition). No arithmetic of the method lives here:
brick layout, neighbour table, local boundary codes, and the exchange of device-pointer handles between the processes (one per GPU).

A decomposition is a grid of px x py x pz bricks of equal size; rank = cx + px (cy + py cz). A face of a brick is
  bc 2  if another brick lies behind it (also across a periodic domain boundary when the axis is split over several bricks),
  the global code (0 periodic, 1 outflow) otherwise.
"""
import itertools

import numpy as np

DIRS = [d for d in itertools.product((-1, 0, 1), repeat=3) if d != (0, 0, 0)]      # (dx, dy, dz)


def brick_grid(world, grid=None):
    """(px, py, pz); default: slabs along z (x rows stay whole: the kernels' coalescing axis)"""
    if grid is None:
        return (1, 1, int(world))
    grid = tuple(int(g) for g in grid)
    if len(grid) != 3 or grid[0] * grid[1] * grid[2] != world or min(grid) < 1:
        raise ValueError("brick grid %r does not hold %d ranks" % (grid, world))
    return grid


def brick_coords(rank, grid):
    return (rank % grid[0], (rank // grid[0]) % grid[1], rank // (grid[0] * grid[1]))


def brick_rank(coords, grid):
    return coords[0] + grid[0] * (coords[1] + grid[1] * coords[2])


def local_bc(rank, grid, global_bc):
    """bc[6] of this brick: {x-, x+, y-, y+, z-, z+}"""
    c = brick_coords(rank, grid)
    bc = []
    for a in range(3):
        for side in (0, 1):
            g = int(global_bc[2 * a + side])
            if grid[a] == 1:
                bc.append(g)
            elif (side == 0 and c[a] > 0) or (side == 1 and c[a] < grid[a] - 1):
                bc.append(2)
            else:                                   # brick at the domain boundary of a split axis
                bc.append(2 if g == 0 else g)
    return bc


def neighbor_table(rank, grid, global_bc):
    """{(dx, dy, dz): neighbour rank} for every direction whose non-zero components all cross a bc = 2 face"""
    c = brick_coords(rank, grid)
    bc = local_bc(rank, grid, global_bc)
    out = {}
    for d in DIRS:
        ok = all(d[a] == 0 or bc[2 * a + (1 if d[a] > 0 else 0)] == 2 for a in range(3))
        if ok:
            out[d] = brick_rank(tuple((c[a] + d[a]) % grid[a] for a in range(3)), grid)
    return out


def local_box(rank, grid, n_global):
    """interior index ranges [(lo, hi)] * 3 (x, y, z) of this brick in the global interior index space"""
    c = brick_coords(rank, grid)
    box = []
    for a in range(3):
        if n_global[a] % grid[a]:
            raise ValueError("global size %r is not divisible by the brick grid %r" % (n_global, grid))
        m = n_global[a] // grid[a]
        box.append((c[a] * m, (c[a] + 1) * m))
    return box


def cut_local(arr, rank, grid, n_global, ng):
    """the brick's ghosted sub-array of a ghosted global array (fields, MZ, MY, MX); ghost layers are taken along (they are refilled)"""
    (x0, x1), (y0, y1), (z0, z1) = local_box(rank, grid, n_global)
    return np.ascontiguousarray(arr[:, z0:z1 + 2 * ng, y0:y1 + 2 * ng, x0:x1 + 2 * ng])


def state_slots(patch):
    """slots whose buffers the stage loop reads through the ghost fill or rotates: name -> (slot, tensor)"""
    from . import binding as b
    out = {"U": (b.SLOT_U, patch.U), "U0": (b.SLOT_U0, patch.U0)}
    if getattr(patch, "U1", None) is not None:
        out["U1"] = (b.SLOT_U1, patch.U1)
    if hasattr(patch, "V"):
        out["V"] = (b.SLOT_V, patch.V)
        out["V0"] = (b.SLOT_V0, patch.V0)
    return out


def connect_local(patches, grid, global_bc):
    """All bricks live in this process (one stream, or several GPUs with peer access): wire them by plain device pointers.
    Returns the list of local bc codes, one per brick. No epoch words: the caller's stream order is the ordering."""
    from . import binding as b
    bcs = []
    for r, p in enumerate(patches):
        for d, nb in neighbor_table(r, grid, global_bc).items():
            for name, (slot, _) in state_slots(p).items():
                t = state_slots(patches[nb])[name][1]
                b.mhd_patch_set_neighbor(p.h, slot, d, t.data_ptr(), patches[nb].npts)
        bcs.append(local_bc(r, grid, global_bc))
    return bcs


def connect_distributed(patch, rank, grid, global_bc, gather=None):
    """One process per GPU: export this brick's state buffers and halo words (CUDA IPC), all-gather the handles over
    torch.distributed (any backend: the payload is a few hundred bytes of host data), import the neighbours' and register them.
    Returns (bc, imported) — keep `imported` alive and pass it to disconnect() before the tensors are freed."""
    from . import binding as b
    if gather is None:
        import torch.distributed as dist

        def gather(obj):
            out = [None] * dist.get_world_size()
            dist.all_gather_object(out, obj)
            return out
    mine = {name: b.mhd_ipc_export(t.data_ptr()) + (patch.npts,) for name, (_, t) in state_slots(patch).items()}
    mine["words"] = b.mhd_ipc_export(b.mhd_patch_halo_words(patch.h))
    everyone = gather(mine)
    bases = {}                                                   # one mapping per remote allocation (a handle opens once per process)

    def remote(handle, off):
        if handle not in bases:
            bases[handle] = b.mhd_ipc_import(handle, 0)
        return bases[handle] + off

    for d, nb in neighbor_table(rank, grid, global_bc).items():
        theirs = everyone[nb]
        for name, (slot, t) in state_slots(patch).items():
            ptr = t.data_ptr() if nb == rank else remote(*theirs[name][:2])      # nb == rank: a periodic axis with this brick on both sides
            b.mhd_patch_set_neighbor(patch.h, slot, d, ptr, theirs[name][2])
        words = b.mhd_patch_halo_words(patch.h) if nb == rank else remote(*theirs["words"])
        b.mhd_patch_set_neighbor_word(patch.h, d, words)
    return local_bc(rank, grid, global_bc), list(bases.values())


def disconnect(imported):
    from . import binding as b
    for base in imported:
        try:
            b.mhd_ipc_close(base, 0)
        except b.MhdError:
            pass
