"""World-size-2 (and 3) `gloo` tests of the N > 1 host logic: band bounds,
the all-gather of the per-rank slices through the preallocated padded blocks, their reassembly, and a
row-sharded RK4 trajectory driven through `binding.Shard`'s exchange callback.  No GPU here, so what a
rank's kernels would compute for its rows is stood in for by the oracle evaluated on that band of rows;
what is under test is `paper_2107_05364_b200.sharding` and the callback plumbing of `binding.Shard`, the
code `bench.py --gpus N` runs over NCCL (the library side of the same protocol is covered on one GPU by
tests/test_gpu_sharded.py).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2107_05364_b200 import sharding as S
from paper_2107_05364_b200 import workloads as W
from tests import harness as H


def test_row_bands_tile_the_rows_in_rank_order():
    for n in (1, 2, 7, 512, 6400, 36384, 65536):
        for world in (1, 2, 3, 4, 8):
            bands = [S.row_band(r, world, n) for r in range(world)]
            assert bands[0][0] == 0 and bands[-1][1] == n
            assert all(bands[r][1] == bands[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in bands]
            assert max(sizes) - min(sizes) <= 1 and max(sizes) == S.max_band_rows(world, n)
    with pytest.raises(ValueError):
        S.row_band(2, 2, 10)


def test_blocks_reassemble_through_the_precomputed_index():
    """pack [world, B, 3, pad] (block g = rows of rank g, padded to the widest band) -> [B, 3, n]: the torch
    mirror of the library's scatter kernel, for even and uneven bands."""
    for world, n in ((1, 5), (2, 90), (3, 40), (4, 7), (8, 65536)):
        pad = S.max_band_rows(world, n)
        full = torch.arange(2 * 3 * n, dtype=torch.float64).reshape(2, 3, n)
        pack = torch.full((world, 2, 3, pad), -1.0, dtype=torch.float64)
        for g in range(world):
            a, b = S.row_band(g, world, n)
            pack[g, :, :, : b - a] = full[:, :, a:b]
        assert torch.equal(S.unpack(pack, n), full)
        idx = S.unpack_index(world, n, pad)
        assert idx.shape == (n,) and int(idx.max()) < world * pad and len(set(idx.tolist())) == n


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, grid, batch: int, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import mt_oracle as O
        w = W.config5(*grid, batch=batch)
        r0, r1 = S.row_band(rank, world, w.n)
        rows = np.arange(r0, r1, dtype=np.int64)
        # the rank's band of the tensor and its slice of the field (every rank holds all of m)
        N_band = O.assemble_rows(H.oracle_tiles(O, w), rows=rows, long_double=False, nthreads=1)
        local = torch.from_numpy(O.demag_field(N_band, w.Ms, w.m, nthreads=1))
        full = S.all_gather_field(dist, local, w.n, rank, world)
        assert full.shape == (batch, 3, w.n)
        # the exchange is also what feeds the next evaluation: every rank must hold the same vector
        chk = full.clone()
        dist.broadcast(chk, src=0)
        assert torch.equal(chk, full)
        if rank == 0:
            q.put(full.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,grid", [(2, (6, 5, 3)), (3, (5, 4, 2))])
def test_sharded_field_reassembles_to_the_full_field(oracle, world, grid):
    """Uneven bands (90 rows over 2 ranks is even; 40 over 3 is not) gathered in rank order equal the
    oracle's field of the unsharded tensor."""
    batch = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, grid, batch, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = q.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    w = W.config5(*grid, batch=batch)
    N = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=False)
    want = oracle.demag_field(N, w.Ms, w.m)
    np.testing.assert_array_equal(got, want)


def _rk4_worker(rank: int, world: int, port: int, grid, steps: int, dt: float, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import mt_oracle as O
        from paper_2107_05364_b200 import binding as B
        w = W.config3(grid)          # exchange + anisotropy + demag: neighbours cross the band boundary
        n = w.n
        r0, r1 = S.row_band(rank, world, n)
        rows = np.arange(r0, r1, dtype=np.int64)
        N_band = O.assemble_rows(H.oracle_tiles(O, w), rows=rows, long_double=False, nthreads=1)
        prob = H.oracle_problem(O, w, N_band, rows=rows)
        shard = B.Shard(rank, world, n, 1, "cpu", S.dist_exchange(dist, rank))
        assert shard.rows == (r0, r1)

        def f(y):  # this rank's rows of the right-hand side at the full state y [1, 3, n]
            k, _ = O.llg_rhs(prob, y, nthreads=1)
            return k[0]

        def stage(y_rows):  # what the library does per stage: own block -> gather -> full state
            shard.pack[rank, 0, :, : r1 - r0] = torch.from_numpy(y_rows)
            assert shard._cb(None, S.GATHER_STATE, None) == 0, shard.error
            return S.unpack(shard.pack, n).numpy()

        m = w.m[:1].copy()
        for _ in range(steps):
            mr = m[0][:, r0:r1]
            k1 = f(m)
            k2 = f(stage(mr + 0.5 * dt * k1))
            k3 = f(stage(mr + 0.5 * dt * k2))
            k4 = f(stage(mr + dt * k3))
            new = mr + (dt / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)
            new = new / np.linalg.norm(new, axis=0, keepdims=True)
            m = stage(new)
        # the two reduction words: every rank ends with the maximum
        shard.scal[0], shard.scal[1] = 10 + rank, 100 - rank
        assert shard._cb(None, S.MAX_SCALARS, None) == 0, shard.error
        assert shard.scal.tolist() == [10 + world - 1, 100]
        chk = torch.from_numpy(m.copy())
        dist.broadcast(chk, src=0)
        assert torch.equal(chk, torch.from_numpy(m))  # every rank holds the same state, bit for bit
        if rank == 0:
            q.put(m)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_row_sharded_rk4_trajectory_matches_the_oracle(oracle, world):
    """RK4 with every stage's state exchanged through the Shard callback (blocks [world, 1, 3, pad], in-place
    all-gather, index reassembly; 125 rows over 2 and 3 ranks: uneven bands) against the oracle's own
    unsharded RK4."""
    grid, steps, dt = 5, 6, 2e-3
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rk4_worker, args=(r, world, port, grid, steps, dt, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = q.get(timeout=180)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    w = W.config3(grid)
    N = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=False)
    want, _, res = oracle.integrate(H.oracle_problem(oracle, w, N), w.m[0], method=oracle.RK4, dt=dt, t_end=steps * dt)
    assert res["accepted"] == steps
    assert np.max(np.abs(got[0] - want)) < 1e-13
    assert np.max(np.abs(want - w.m[0])) > 1e-3  # the state moved
