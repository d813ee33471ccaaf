"""-m gpu: mt_demag_field_noalloc (mt.h) — the field of one state with all scratch in the library's static
device array, no mt_ctx and no allocation — against the existing path (mt_demag_field), on calls in a row
that share the array: different states, dtypes, shapes (a full tensor, a ragged one, a row band whose columns
are split), so that anything a call left in the array would show in the next one.  Collected last on purpose
(the file name): the suite runs with -x.
"""
import numpy as np
import pytest
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W
from tests import harness as H

pytestmark = pytest.mark.gpu

TOL_HD = {"f64": 1e-12, "f32": 1e-5}  # the tolerances of tests/test_gpu_small.py


def existing_path(ctx, N, dtype, n, n_rows, ld, Ms, m):
    Hd = torch.empty((1, 3, n_rows), dtype=torch.float64, device="cuda")
    B.mt_demag_field(ctx, N, H.dtype_code(dtype), n, n_rows, ld, Ms, m.view(1, 3, n), 1, Hd)
    torch.cuda.synchronize()
    return Hd[0].cpu().numpy()


def no_alloc(N, dtype, n, n_rows, ld, Ms, m, Hd):
    B.mt_demag_field_noalloc(0, torch.cuda.current_stream().cuda_stream, N, H.dtype_code(dtype), n, n_rows, ld,
                             Ms, m, Hd)


def test_two_calls_in_a_row_match_the_existing_path(oracle):
    ctx = B.mt_create(0)
    w_big = W.config3(16, batch=2)            # n = 4096
    rng = np.random.default_rng(105)
    w_rag = W._cuboid_workload("ragged", 7, 5, 3, (1.0, 0.7, 1.3), 1.0, W.random_unit_states(rng, 2, 105),
                               gamma=1.0, alpha_ll=0.2)  # n = 105: scalar tail, npad > n
    cases = []
    for w, dtype, band in ((w_big, "f32", None), (w_rag, "f64", None), (w_big, "f32", (1000, 1064)),
                           (w_rag, "f32", None), (w_big, "f64", (4000, 4096))):
        tiles = H.dev_tiles(w)
        r0, r1 = band if band else (0, w.n)
        N, ld, status = H.assemble(ctx, tiles, dtype, r0, r1)
        assert status == 0
        cases.append((w, dtype, tiles, N, ld, r1 - r0))

    # warm-up: the first call on the device looks the array up and loads the kernels of both dtypes
    for w, dtype, tiles, N, ld, rows in cases[:2]:
        m = torch.from_numpy(np.ascontiguousarray(w.m[0])).cuda()
        no_alloc(N, dtype, w.n, rows, ld, tiles.Ms, m, torch.empty((3, rows), dtype=torch.float64, device="cuda"))
    torch.cuda.synchronize()

    # inputs and outputs of every call exist before the first one: the calls themselves take no device memory
    ms = [[torch.from_numpy(np.ascontiguousarray(w.m[b])).cuda() for b in range(2)] for w, *_ in cases]
    outs = [[torch.full((3, rows), 7.0, dtype=torch.float64, device="cuda") for _ in range(2)]
            for *_, rows in cases]
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(0)[0]
    for k, (w, dtype, tiles, N, ld, rows) in enumerate(cases):
        for b in range(2):  # two calls in a row on the same shape, then the next shape, no sync in between
            no_alloc(N, dtype, w.n, rows, ld, tiles.Ms, ms[k][b], outs[k][b])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(0)[0] >= free_before

    for k, (w, dtype, tiles, N, ld, rows) in enumerate(cases):
        for b in range(2):
            ref = existing_path(ctx, N, dtype, w.n, rows, ld, tiles.Ms, ms[k][b])
            got = outs[k][b].cpu().numpy()
            assert np.isfinite(got).all() and np.abs(ref).max() > 0
            assert H.rel_l2(got, ref) <= TOL_HD[dtype], (k, b, dtype)
        assert not np.array_equal(outs[k][0].cpu().numpy(), outs[k][1].cpu().numpy())

    # the same call twice gives the same bits (fixed reduction order, nothing left over from other calls)
    w, dtype, tiles, N, ld, rows = cases[2]
    again = torch.empty_like(outs[2][1])
    no_alloc(N, dtype, w.n, rows, ld, tiles.Ms, ms[2][1], again)
    torch.cuda.synchronize()
    assert torch.equal(again, outs[2][1])

    # and the ragged fp64 case against the oracle's own field
    w = w_rag
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    Hd_ref = oracle.demag_field(N_ref, w.Ms, w.m[:2])
    for b in range(2):
        assert H.rel_l2(outs[1][b].cpu().numpy(), Hd_ref[b]) <= TOL_HD["f64"]
    ctx.close()


def test_sizes_beyond_the_static_array_are_rejected():
    n = B.MT_NOALLOC_MAX_N + 1
    x = torch.zeros(64, dtype=torch.float64, device="cuda")
    Nf = torch.zeros(64, dtype=torch.float32, device="cuda")
    with pytest.raises(B.MtError) as e:
        B.mt_demag_field_noalloc(0, 0, Nf, B.MT_F32, n, 8, n + 3, x, x, x)
    assert e.value.code == B.MT_ERR_INVALID_ARG and "MT_NOALLOC_MAX_N" in str(e.value)
    with pytest.raises(B.MtError) as e:
        B.mt_demag_field_noalloc(0, 0, Nf, B.MT_F32, 8, n, 8, x, x, x)
    assert e.value.code == B.MT_ERR_INVALID_ARG and "MT_NOALLOC_MAX_N" in str(e.value)
    with pytest.raises(B.MtError) as e:
        B.mt_demag_field_noalloc(0, 0, Nf, B.MT_F32, 8, 8, 4, x, x, x)  # ld < n
    assert e.value.code == B.MT_ERR_INVALID_ARG and "ld" in str(e.value)
    with pytest.raises(B.MtError):
        B.mt_demag_field_noalloc(99, 0, Nf, B.MT_F32, 8, 8, 8, x, x, x)  # no such device
    torch.cuda.synchronize()
