"""Halo exchange fused with the ghost fill, on ONE GPU: the bricks of a decomposition are separate patches whose
neighbour faces (bc = 2) read each other's interiors inside k_fill_ghosts. The definition it must meet: a decomposed evolution is the
undecomposed one, bit for bit (every kernel computes a point from the same operands in the same order wherever the tile seams fall).
All bricks are driven from one stream in lock step (no kernel ever waits on another); the epoch words of the multi-process path are
exercised on a brick that is its own neighbour, and the CUDA-IPC mapping by a child process that reads this process's patch."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2510_13965_b200 import decomp, synth

pytestmark = pytest.mark.gpu
NG = 3


def _drive(binding, patches, bcs, tab, stages, dt, steps):
    """the stage loop of mhd_advance, all bricks in lock step: every brick fills before any brick's con2prim may repair a cell"""
    for _ in range(steps):
        for st in range(1, stages + 1):
            for p, bc in zip(patches, bcs):
                p.fill_ghosts(bc)
            for p in patches:
                p.con2prim()
            if st == 1:
                for p in patches:
                    p.rk_stage(tab, 0, dt)
            for p in patches:
                p.rhs(st)
            for p in patches:
                p.rk_stage(tab, st, dt)
    for p, bc in zip(patches, bcs):
        p.fill_ghosts(bc)
    for p in patches:
        p.con2prim()


def _split_run(oracle_mod, cfg, grid, steps=2):
    from paper_2510_13965_b200 import binding
    n = cfg["n"]
    o = oracle_mod.Oracle(cfg["params"], n[0], n[1], n[2], NG, cfg["dx"], table=cfg.get("table"))
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    o.fill_ghosts(U, cfg["bc"])
    a, w = synth.tableau("rk4")
    tab = binding.make_tableau(a, w)
    dt = 0.25 * cfg["dx"]
    whole = binding.Patch(cfg["params"], n, NG, cfg["dx"], stages=4, table=cfg.get("table"))
    whole.upload(U=U)
    _drive(binding, [whole], [cfg["bc"]], tab, 4, dt, steps)
    world = grid[0] * grid[1] * grid[2]
    bricks = []
    for r in range(world):
        box = decomp.local_box(r, grid, n)
        nl = tuple(hi - lo for lo, hi in box)
        p = binding.Patch(cfg["params"], nl, NG, cfg["dx"], stages=4, table=cfg.get("table"))
        p.upload(U=decomp.cut_local(U, r, grid, n, NG))
        bricks.append(p)
    bcs = decomp.connect_local(bricks, grid, cfg["bc"])
    _drive(binding, bricks, bcs, tab, 4, dt, steps)
    Uw, Pw, Fw = whole.U.cpu().numpy(), whole.P.cpu().numpy(), whole.flags.cpu().numpy()
    for r, p in enumerate(bricks):
        # the brick's whole ghosted array must equal the same window of the undecomposed array: interior and every ghost layer
        assert np.array_equal(p.U.cpu().numpy(), decomp.cut_local(Uw, r, grid, n, NG)), "state of brick %d" % r
        assert np.array_equal(p.P.cpu().numpy(), decomp.cut_local(Pw, r, grid, n, NG)), "primitives of brick %d" % r
        assert np.array_equal(p.flags.cpu().numpy(), decomp.cut_local(Fw, r, grid, n, NG)), "flags of brick %d" % r
        assert p.status()["halo_timeout"] == 0
    for p in bricks + [whole]:
        p.close()
    return Uw


@pytest.mark.parametrize("grid", [(1, 1, 2), (2, 2, 1), (2, 1, 2)])
def test_decomposed_periodic_box_is_bit_identical(oracle_mod, grid):
    """config 1 (all terms live, periodic): slabs, pencils with edge neighbours, and a split of x (the coalescing axis)"""
    _split_run(oracle_mod, synth.config1(n=24, gauge_perturbation=True), grid)


def test_decomposed_star_with_outflow_and_atmosphere(oracle_mod):
    """config 3 (TOV star, atmosphere resets, outflow): the split puts the cut through the star; outer faces stay outflow"""
    _split_run(oracle_mod, synth.config3(n=32), (2, 1, 2), steps=1)


def test_missing_neighbour_and_thin_brick_are_refused():
    from paper_2510_13965_b200 import binding
    p = binding.Patch(synth.default_params(), (8, 8, 8), NG, 0.1, stages=1)
    with pytest.raises(binding.MhdError):
        p.fill_ghosts([0, 0, 0, 0, 2, 2])                      # no neighbour registered
    with pytest.raises(binding.MhdError):
        p.fill_ghosts([0, 0, 0, 0, 3, 0])
    p.close()
    q = binding.Patch(synth.default_params(), (8, 8, 2), NG, 0.1, stages=1)
    with pytest.raises(binding.MhdError):
        q.fill_ghosts([0] * 6)                                 # periodic wrap of a 2-point axis through 3 ghost layers
    q.fill_ghosts([0, 0, 0, 0, 1, 1])
    q.close()


def test_epoch_words_on_a_brick_that_is_its_own_neighbour(oracle_mod):
    """The multi-process protocol (signal / wait kernels around the fill) with the brick wired to itself across z: every wait is
    satisfied by the signal that precedes it in the same stream. mhd_advance must equal the periodic run and report no time-out."""
    from paper_2510_13965_b200 import binding
    cfg = synth.config1(n=16, gauge_perturbation=True)
    o = oracle_mod.Oracle(cfg["params"], 16, 16, 16, NG, cfg["dx"])
    U, P = cfg["U"].copy(), cfg["P"].copy()
    o.prim2con(U, P)
    a, w = synth.tableau("rk4")
    tab = binding.make_tableau(a, w)
    dt = 0.25 * cfg["dx"]
    out = []
    for wired in (False, True):
        p = binding.Patch(cfg["params"], cfg["n"], NG, cfg["dx"], stages=4)
        p.upload(U=U)
        bc = [0] * 6
        if wired:
            bc, imported = decomp.connect_distributed(p, 0, (1, 1, 1), [0] * 6, gather=lambda obj: [obj])
            assert bc == [0] * 6 and imported == []            # a single brick per axis stays periodic
            for d in ((0, 0, 1), (0, 0, -1)):
                for name, (slot, t) in decomp.state_slots(p).items():
                    binding.mhd_patch_set_neighbor(p.h, slot, d, t.data_ptr(), p.npts)
                binding.mhd_patch_set_neighbor_word(p.h, d, binding.mhd_patch_halo_words(p.h))
            bc = [0, 0, 0, 0, 2, 2]
        p.advance(tab, bc, dt, 3)
        st = p.status()
        assert st["halo_timeout"] == 0
        out.append(p.U.cpu().numpy())
        p.close()
    assert np.array_equal(out[0], out[1])


_CHILD = r"""
import sys, numpy as np, torch
from paper_2510_13965_b200 import binding, synth
handle = bytes.fromhex(sys.argv[1]); off = int(sys.argv[2]); npts = int(sys.argv[3])
ptr = binding.mhd_ipc_import(handle, off)
p = binding.Patch(synth.default_params(), (8, 8, 8), 3, 0.1, stages=1)
p.U.fill_(-1.0)
for d in ((0, 0, 1), (0, 0, -1)):
    binding.mhd_patch_set_neighbor(p.h, binding.SLOT_U, d, ptr, npts)
p.fill_ghosts([0, 0, 0, 0, 2, 2])
torch.cuda.synchronize()
U = p.U.cpu().numpy()
idx = np.arange(32 * 14 ** 3, dtype=np.float64).reshape(32, 14, 14, 14)       # the parent's pattern
ok = np.array_equal(U[:, 11:14, 3:11, 3:11], idx[:, 3:6, 3:11, 3:11]) and np.array_equal(U[:, 0:3, 3:11, 3:11], idx[:, 8:11, 3:11, 3:11])
ok = ok and np.all(U[:, 3:11, 3:11, 3:11] == -1.0)
binding.mhd_ipc_close(ptr, off)
print("CHILD_OK" if ok else "CHILD_BAD")
"""


def test_ipc_mapping_read_by_another_process():
    """One process per GPU in miniature: this process exports its state buffer (CUDA IPC handle + offset inside the caching allocator's
    block); a child process maps it and its ghost-fill kernel reads the z faces straight out of this process's memory. The parent only
    waits for the child process to exit."""
    import torch
    from paper_2510_13965_b200 import binding
    p = binding.Patch(synth.default_params(), (8, 8, 8), NG, 0.1, stages=1)
    p.U.copy_(torch.arange(p.U.numel(), dtype=torch.float64, device="cuda").reshape(p.U.shape))
    torch.cuda.synchronize()
    handle, off = binding.mhd_ipc_export(p.U.data_ptr())
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", _CHILD, handle.hex(), str(off), str(p.npts)], cwd=root, capture_output=True, text=True, timeout=300)
    assert "CHILD_OK" in r.stdout, (r.stdout, r.stderr[-2000:])
    p.close()
