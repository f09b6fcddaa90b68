"""The N > 1 path of bench.py is replicas only: N independent patches, no data-path collective; the
one exchange is the MAX reduction of the timed region over ranks. Covered here with world_size 2 on the gloo backend."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local)
    value = bench.aggregate_throughput(world, zones=64 ** 3, stages=4, steps=3, ms_max=ms)
    out.put((rank, ms, value))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_world2():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value in res:
        assert ms == 15.0                                              # every rank sees the slowest rank's time
        assert abs(value - 2 * 64 ** 3 * 4 * 3 / 15.0e-3) < 1e-6 * value    # whole-job aggregate over both replicas


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5) == 7.5


# ---- domain decomposition with the halo exchange fused into the ghost fill: host logic on CPU ----------
def _emulated_fill(local, bc, table, arrays, ng):
    """numpy restatement of the fused ghost fill's index map (test code): wrap / clamp / wrap in the neighbour's array"""
    n = [local.shape[3] - 2 * ng, local.shape[2] - 2 * ng, local.shape[1] - 2 * ng]
    out = local.copy()

    def src(i, a):
        if i < ng:
            b = bc[2 * a]
            return (ng, 0) if b == 1 else (i + n[a], -1 if b == 2 else 0)
        if i >= ng + n[a]:
            b = bc[2 * a + 1]
            return (ng + n[a] - 1, 0) if b == 1 else (i - n[a], 1 if b == 2 else 0)
        return i, 0

    for k in range(local.shape[1]):
        sk, dz = src(k, 2)
        for j in range(local.shape[2]):
            sj, dy = src(j, 1)
            for i in range(local.shape[3]):
                si, dx = src(i, 0)
                if (si, sj, sk) == (i, j, k):
                    continue
                from_arr = local if (dx, dy, dz) == (0, 0, 0) else arrays[table[(dx, dy, dz)]]
                out[:, k, j, i] = from_arr[:, sk, sj, si]
    return out


def _halo_worker(rank, world, port, out):
    import numpy as np
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import oracle
    from paper_2510_13965_b200 import decomp
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ng, n = 3, (8, 6, 8)
    ok = True
    for grid, gbc in (((1, 1, 2), [0] * 6), ((2, 1, 1), [1, 1, 0, 0, 0, 1]), ((1, 2, 1), [0, 0, 0, 0, 1, 1])):
        rng = np.random.default_rng(11)                          # same global array on every rank
        G = rng.standard_normal((2, n[2] + 2 * ng, n[1] + 2 * ng, n[0] + 2 * ng))
        o = oracle.Oracle(dict(), n[0], n[1], n[2], ng, 1.0)
        want = G.copy()
        o.fill_ghosts(want, gbc)                                 # the undecomposed ghost fill is the definition
        mine = decomp.cut_local(G, rank, grid, n, ng)
        t = [torch.zeros(mine.shape, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(t, torch.from_numpy(mine))               # the exchange (on GPUs: direct peer reads inside the kernel)
        arrays = [x.numpy() for x in t]
        table = decomp.neighbor_table(rank, grid, gbc)
        # the table is symmetric: my neighbour in direction d sees me in direction -d
        tables = [None] * world
        dist.all_gather_object(tables, table)
        for d, nb in table.items():
            ok = ok and tables[nb][tuple(-c for c in d)] == rank
        got = _emulated_fill(mine, decomp.local_bc(rank, grid, gbc), table, arrays, ng)
        ok = ok and np.array_equal(got, decomp.cut_local(want, rank, grid, n, ng))
    out.put((rank, bool(ok)))
    dist.barrier()
    dist.destroy_process_group()


def test_decomposed_ghost_fill_equals_global_fill_world2():
    """world 2 over gloo: brick layout, local boundary codes, neighbour table and windows of paper_2510_13965_b200.decomp reproduce the
    undecomposed (oracle) ghost fill exactly, for a periodic split, an outflow split along x and a mixed case."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_halo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True), (1, True)]


def test_decomp_tables():
    sys.path.insert(0, ROOT)
    from paper_2510_13965_b200 import decomp
    assert decomp.brick_grid(4) == (1, 1, 4)
    assert decomp.local_bc(1, (1, 1, 4), [0, 0, 1, 1, 1, 1]) == [0, 0, 1, 1, 2, 2]
    assert decomp.local_bc(0, (1, 1, 4), [0, 0, 1, 1, 1, 1]) == [0, 0, 1, 1, 1, 2]          # outflow end of a split axis stays outflow
    assert decomp.local_bc(3, (1, 1, 4), [0] * 6) == [0, 0, 0, 0, 2, 2]                      # periodic end wraps to brick 0
    assert decomp.neighbor_table(3, (1, 1, 4), [0] * 6) == {(0, 0, -1): 2, (0, 0, 1): 0}
    t = decomp.neighbor_table(0, (2, 2, 2), [0] * 6)
    assert len(t) == 26 and t[(1, 1, 1)] == 7 and t[(-1, 0, 0)] == 1
    assert decomp.local_box(5, (2, 2, 2), (8, 8, 8)) == [(4, 8), (0, 4), (4, 8)]
