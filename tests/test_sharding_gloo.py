"""World-size-2 (and 3) `gloo` test of the N > 1 host logic: band bounds,
the all-gather of the per-rank field slices and their reassembly.  No GPU here, so the per-band field a
rank's kernels would produce is stood in for by the oracle evaluated on that band of rows; what is under
test is `paper_2107_05364_b200.sharding`, the code `bench.py --gpus N` runs over NCCL.
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
