"""-m gpu: F1 — thresholded tensor through the C-ABI against oracle/threshold.py.

The dense input of the thresholding calls is the ORACLE's tensor (rounded to the stored dtype on the
host and uploaded), so that threshold value, masks and packed values are integer/bit-exact
comparisons; the field of the compressed tensor is compared with the oracle's field of the truncated
tensor within north_star's H_d tolerances.
"""
import numpy as np
import pytest
import torch

from oracle import threshold as OT
from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W
from tests import harness as H

pytestmark = pytest.mark.gpu
TOL_HD = {"f64": 1e-12, "f32": 1e-5}


@pytest.fixture(scope="module")
def ctx():
    c = B.mt_create(0)
    yield c
    c.close()


def upload(N_ref, dtype):
    """oracle tensor -> stored dtype on the host -> device planes [6][n][ld] (padding zero)."""
    npdt = np.float32 if dtype == "f32" else np.float64
    host = N_ref.astype(npdt)
    n = host.shape[2]
    ld = W.leading_dim(n, dtype)
    dev = torch.zeros((6, host.shape[1], ld), dtype=B.torch_dtype(H.dtype_code(dtype)), device="cuda")
    dev[:, :, :n] = torch.from_numpy(host).cuda()
    return host, dev, ld


def unpack(S, n):
    """bitmap rows -> dense numpy planes (host-side decoding for the comparison only)."""
    mask = S.mask.cpu().numpy().view(np.uint32)
    vals = S.vals.cpu().numpy()
    ptr = S.row_ptr.cpu().numpy()
    out = np.zeros((6, S.n_rows, S.nw * 32), dtype=vals.dtype)
    bits = ((mask[..., None] >> np.arange(32, dtype=np.uint32)) & 1).astype(bool).reshape(6, S.n_rows, -1)
    for c in range(6):
        for i in range(S.n_rows):
            r = c * S.n_rows + i
            out[c, i, bits[c, i]] = vals[ptr[r]:ptr[r + 1]]
    assert not bits[:, :, n:].any()
    return out[:, :, :n]


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("grid", [(8, 8, 8), (13, 7, 3)])
def test_threshold_value_and_bitmap_rows_are_exact(ctx, oracle, grid, dtype):
    w = W.config5(*grid, batch=3)
    n = w.n
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    host, dev, ld = upload(N_ref, dtype)
    code = H.dtype_code(dtype)
    mult = np.array(OT.MULTIPLICITY).reshape(6, 1, 1)
    for X in (0.0, 0.2, 0.4, 0.7, 0.93, 1.0):
        tau_ref = OT.threshold_value(host, X)
        tau, cnt = B.mt_threshold_value(ctx, dev, code, n, n, ld, X)
        assert cnt == int((mult * (host != 0)).sum())
        assert tau == tau_ref, (X, tau, tau_ref)
        S = B.mt_sparse_build(ctx, dev, code, n, n, ld, tau)
        torch.cuda.synchronize()
        trunc = OT.truncate(host, tau_ref)
        assert S.nnz == np.count_nonzero(trunc)
        assert np.array_equal(unpack(S, n), trunc)
        # field of the compressed tensor vs the oracle's field of the truncated tensor
        m = torch.from_numpy(w.m).cuda()
        Hd = torch.empty_like(m)
        B.mt_demag_field_sparse(ctx, S, torch.from_numpy(w.Ms).cuda(), m, 3, Hd)
        torch.cuda.synchronize()
        ref = oracle.demag_field(trunc.astype(np.float64), w.Ms, w.m)
        if S.nnz == 0:
            assert not Hd.cpu().numpy().any()
        else:
            for b in range(3):
                assert H.rel_l2(Hd[b].cpu().numpy(), ref[b]) <= TOL_HD[dtype]
        Hd2 = torch.empty_like(m)
        B.mt_demag_field_sparse(ctx, S, torch.from_numpy(w.Ms).cuda(), m, 3, Hd2)
        assert torch.equal(Hd, Hd2)  # fixed reduction order
        # index rows: the 16-bit column of every packed value = the non-zero columns of the truncated
        # tensor in (plane, row, column) order; the field kernel that walks them, with the mask dropped
        B.mt_sparse_index(ctx, S, drop_mask=True)
        assert S.mask is None
        if S.nnz:
            cols_ref = np.nonzero(trunc.reshape(6 * n, n))[1].astype(np.uint16)
            assert np.array_equal(S.cols16.cpu().numpy(), cols_ref)
        Hi = torch.empty_like(m)
        B.mt_demag_field_sparse(ctx, S, torch.from_numpy(w.Ms).cuda(), m, 3, Hi)
        torch.cuda.synchronize()
        if S.nnz == 0:
            assert not Hi.cpu().numpy().any()
        else:
            for b in range(3):
                assert H.rel_l2(Hi[b].cpu().numpy(), ref[b]) <= TOL_HD[dtype]
        Hi2 = torch.empty_like(m)
        B.mt_demag_field_sparse(ctx, S, torch.from_numpy(w.Ms).cuda(), m, 3, Hi2)
        assert torch.equal(Hi, Hi2)


@pytest.mark.parametrize("batch", [1, 4, 5, 8])
def test_sparse_field_batches_match_dense_path_on_truncated_tensor(ctx, oracle, batch):
    """Dense kernels on the truncated tensor and the bitmap kernel on its compressed form agree."""
    w = W.config5(20, 10, 2, batch=batch)
    n = w.n
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    host, dev, ld = upload(N_ref, "f32")
    tau = OT.threshold_value(host, 0.5)
    S = B.mt_sparse_build(ctx, dev, B.MT_F32, n, n, ld, tau)
    trunc = OT.truncate(host, tau)
    _, dev_t, _ = upload(trunc.astype(np.float64), "f32")
    Ms = torch.from_numpy(w.Ms).cuda()
    m = torch.from_numpy(w.m).cuda()
    Hs, Hd = torch.empty_like(m), torch.empty_like(m)
    B.mt_demag_field_sparse(ctx, S, Ms, m, batch, Hs)
    B.mt_demag_field(ctx, dev_t, B.MT_F32, n, n, ld, Ms, m, batch, Hd)
    torch.cuda.synchronize()
    ref = oracle.demag_field(trunc.astype(np.float64), w.Ms, w.m)
    B.mt_sparse_index(ctx, S)
    Hi = torch.empty_like(m)
    B.mt_demag_field_sparse(ctx, S, Ms, m, batch, Hi)
    torch.cuda.synchronize()
    for b in range(batch):
        assert H.rel_l2(Hs[b].cpu().numpy(), ref[b]) <= 1e-5
        assert H.rel_l2(Hs[b].cpu().numpy(), Hd[b].cpu().numpy()) <= 2e-6
        assert H.rel_l2(Hi[b].cpu().numpy(), ref[b]) <= 1e-5
        assert H.rel_l2(Hi[b].cpu().numpy(), Hd[b].cpu().numpy()) <= 2e-6


def test_thresholded_dynamics_follow_the_oracle_on_the_truncated_tensor(ctx, oracle):
    """The experiment of PAPER.md:239 in small: config-2 physics (film, exchange, applied field) with a
    40 % threshold; RK4 trajectory of the sparse path vs the oracle integrating the truncated tensor,
    and the distance to the un-thresholded trajectory reported by the oracle itself."""
    w = W.config2(24, 6, phase="dynamics")
    n = w.n
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    host, dev, ld = upload(N_ref, "f32")
    tau, _ = B.mt_threshold_value(ctx, dev, B.MT_F32, n, n, ld, 0.4)
    assert tau == OT.threshold_value(host, 0.4)
    S = B.mt_sparse_build(ctx, dev, B.MT_F32, n, n, ld, tau)
    prob = H.dev_problem(w, tiles, None, "f32", ld)
    prob.N_sparse = S
    dt, steps = 1e-13, 200
    m = torch.from_numpy(w.m[:1].copy()).cuda()
    samples = torch.zeros((16, 4), dtype=torch.float64, device="cuda")
    _, res, _ = B.mt_integrate(ctx, prob, m, 1, 0.0, method=B.MT_RK4, dt=dt, t_end=steps * dt, sample_every=20,
                               samples=samples)
    trunc = OT.truncate(host, tau).astype(np.float64)
    m_ref, s_ref, _ = oracle.integrate(H.oracle_problem(oracle, w, trunc), w.m[0], method=oracle.RK4, dt=dt,
                                       t_end=steps * dt, sample_every=20, sample_cap=16, weights=w.vol)
    assert res["n_samples"] == 10
    s = samples[:10].cpu().numpy()
    assert np.max(np.abs(s[:, 1:] - s_ref[:, 1:])) < 1e-4
    assert np.max(np.abs(m[0].cpu().numpy() - m_ref)) < 1e-3
    # energy through the sparse path too (F4 on F1)
    E = torch.empty((1, 5), dtype=torch.float64, device="cuda")
    B.mt_energy(ctx, prob, m, 1, E)
    ref = oracle.energy_terms(H.oracle_problem(oracle, w, trunc), m[0].cpu().numpy(), vol=w.vol)
    assert np.max(np.abs(E[0, :4].cpu().numpy() - ref)) <= 1e-5 * np.abs(ref).sum()
    # the same trajectory and energies with the field kernel on the index rows
    B.mt_sparse_index(ctx, S, drop_mask=True)
    prob.N_sparse = S
    mi = torch.from_numpy(w.m[:1].copy()).cuda()
    samples_i = torch.zeros((16, 4), dtype=torch.float64, device="cuda")
    B.mt_integrate(ctx, prob, mi, 1, 0.0, method=B.MT_RK4, dt=dt, t_end=steps * dt, sample_every=20,
                   samples=samples_i)
    assert np.max(np.abs(samples_i[:10].cpu().numpy()[:, 1:] - s_ref[:, 1:])) < 1e-4
    assert np.max(np.abs(mi[0].cpu().numpy() - m_ref)) < 1e-3
    Ei = torch.empty((1, 5), dtype=torch.float64, device="cuda")
    B.mt_energy(ctx, prob, mi, 1, Ei)
    ref_i = oracle.energy_terms(H.oracle_problem(oracle, w, trunc), mi[0].cpu().numpy(), vol=w.vol)
    assert np.max(np.abs(Ei[0, :4].cpu().numpy() - ref_i)) <= 1e-5 * np.abs(ref_i).sum()


def test_sparse_argument_checks(ctx):
    Ms = torch.ones(4, dtype=torch.float64, device="cuda")
    m = torch.zeros((1, 3, 4), dtype=torch.float64, device="cuda")
    N = torch.zeros((6, 4, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(B.MtError):
        B.mt_threshold_value(ctx, N, B.MT_F32, 4, 4, 4, 1.5)
    tau, cnt = B.mt_threshold_value(ctx, N, B.MT_F32, 4, 4, 4, 0.3)   # all-zero tensor: nothing to rank
    assert cnt == 0 and tau == float("inf")
    S = B.mt_sparse_build(ctx, N, B.MT_F32, 4, 4, 4, 0.0)
    assert S.nnz == 0
    S.nw += 1
    with pytest.raises(B.MtError):
        B.mt_demag_field_sparse(ctx, S, Ms, m, 1, torch.empty_like(m))
    S.nw -= 1
    import ctypes
    S.n, S.nw = 65537, 2052   # more than one panel of 16-bit columns: panel_ptr is required
    rc = ctx.lib.mt_sparse_index(ctx.h, ctypes.byref(S._c()), S.vals.data_ptr(), None)
    assert rc != 0


def test_sparse_row_band(ctx, oracle):
    """Thresholding a ROW BAND of the tensor (the multi-GPU shard unit of mt_assemble_tensor): the band's
    own threshold, bitmap rows and field, against the oracle on the same rows."""
    w = W.config5(12, 9, 3, batch=2)
    n = w.n
    rows = np.arange(70, 70 + 101, dtype=np.int64)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=rows, long_double=True)
    host, dev, ld = upload(N_ref, "f32")
    tau, _ = B.mt_threshold_value(ctx, dev, B.MT_F32, n, len(rows), ld, 0.6)
    assert tau == OT.threshold_value(host, 0.6)
    S = B.mt_sparse_build(ctx, dev, B.MT_F32, n, len(rows), ld, tau)
    torch.cuda.synchronize()
    trunc = OT.truncate(host, tau)
    assert np.array_equal(unpack(S, n), trunc)
    m = torch.from_numpy(w.m).cuda()
    Hd = torch.empty((2, 3, len(rows)), dtype=torch.float64, device="cuda")
    B.mt_demag_field_sparse(ctx, S, torch.from_numpy(w.Ms).cuda(), m, 2, Hd)
    torch.cuda.synchronize()
    ref = oracle.demag_field(trunc.astype(np.float64), w.Ms, w.m)
    B.mt_sparse_index(ctx, S)
    assert np.array_equal(S.cols16.cpu().numpy(), np.nonzero(trunc.reshape(6 * len(rows), n))[1].astype(np.uint16))
    Hi = torch.empty_like(Hd)
    B.mt_demag_field_sparse(ctx, S, torch.from_numpy(w.Ms).cuda(), m, 2, Hi)
    torch.cuda.synchronize()
    for b in range(2):
        assert H.rel_l2(Hd[b].cpu().numpy(), ref[b]) <= 1e-5
        assert H.rel_l2(Hi[b].cpu().numpy(), ref[b]) <= 1e-5


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_streamed_thresholding_equals_the_resident_path_and_the_oracle(ctx, oracle, dtype):
    """PAPER.md:237 (memory): the thresholded tensor built band by band (mt_select_*, mt_sparse_*_band; the
    dense tensor never resident) is bit-identical to the one built from the resident dense tensor — same
    threshold, offsets, bitmaps, values — for band heights that do not divide n; and, with the cut placed
    in a gap of the oracle's magnitudes, its bitmaps equal the oracle's truncation and its field the
    oracle's field of the truncated tensor."""
    w = W.config5(13, 7, 3, batch=2)
    n = w.n
    code = H.dtype_code(dtype)
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, dtype)
    assert status == 0
    for X, band_rows in ((0.0, 64), (0.35, 37), (0.9, 100), (1.0, 273)):
        tau, cnt = B.mt_threshold_value(ctx, N, code, n, n, ld, X)
        S = B.mt_sparse_build(ctx, N, code, n, n, ld, tau)
        T = B.mt_sparse_build_streamed(ctx, tiles, code, X, band_rows)
        torch.cuda.synchronize()
        assert T.tau == tau and T.nnz == S.nnz
        assert torch.equal(T.row_ptr, S.row_ptr) and torch.equal(T.mask, S.mask)
        if S.nnz:
            assert torch.equal(T.vals, S.vals)
        # index rows written by the fill pass itself (bitmap left out) = those derived from the bitmap
        B.mt_sparse_index(ctx, S)
        U = B.mt_sparse_build_streamed(ctx, tiles, code, X, band_rows, index=True, keep_mask=False)
        torch.cuda.synchronize()
        assert U.mask is None and U.nnz == S.nnz and torch.equal(U.row_ptr, S.row_ptr)
        if S.nnz:
            assert torch.equal(U.vals, S.vals) and torch.equal(U.cols16, S.cols16)
    # against the oracle: cut in a gap of the oracle's magnitudes next to the device's 60 % value
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    host = N_ref.astype(np.float32 if dtype == "f32" else np.float64)
    tau_dev, _ = B.mt_threshold_value(ctx, N, code, n, n, ld, 0.6)
    mags = np.unique(np.abs(host[np.abs(host) > 0]).astype(np.float64))
    gaps = np.nonzero(mags[1:] > mags[:-1] * 1.001)[0]
    g = gaps[np.argmin(np.abs(np.log(mags[gaps] / tau_dev)))]
    tau = float(np.sqrt(mags[g] * mags[g + 1]))
    if dtype == "f32":
        tau = float(np.float32(tau))
    assert mags[g] < tau < mags[g + 1]
    T = B.mt_sparse_build_streamed(ctx, tiles, code, 0.6, 50, tau=tau)
    B.mt_sparse_index(ctx, T)
    torch.cuda.synchronize()
    trunc = OT.truncate(host, tau)
    assert np.array_equal(unpack(T, n) != 0, trunc != 0)
    m = torch.from_numpy(w.m).cuda()
    Hd = torch.empty_like(m)
    B.mt_demag_field_sparse(ctx, T, tiles.Ms, m, 2, Hd)
    torch.cuda.synchronize()
    ref = oracle.demag_field(trunc.astype(np.float64), w.Ms, w.m)
    for b in range(2):
        assert H.rel_l2(Hd[b].cpu().numpy(), ref[b]) <= TOL_HD[dtype]


def test_index_rows_beyond_65536_columns(ctx, oracle):
    """n > 65,536: 16-bit columns are relative to panels of 65,536 columns and panel_ptr marks where a
    plane row's second panel starts.  A 40-row band of a 66 x 50 x 20 mesh (n = 66,000), thresholded at
    70 %: columns, panel offsets and field against the oracle's truncated rows."""
    w = W.config5(66, 50, 20, batch=2)
    n = w.n
    assert n == 66000
    rows = np.concatenate([np.arange(0, 20), np.arange(65530, 65545), np.arange(n - 5, n)]).astype(np.int64)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=rows, long_double=True)
    host, dev, ld = upload(N_ref, "f32")
    tau = OT.threshold_value(host, 0.7)
    tau_dev, _ = B.mt_threshold_value(ctx, dev, B.MT_F32, n, len(rows), ld, 0.7)
    assert tau_dev == tau
    S = B.mt_sparse_build(ctx, dev, B.MT_F32, n, len(rows), ld, tau)
    m = torch.from_numpy(w.m).cuda()
    Ms = torch.from_numpy(w.Ms).cuda()
    Hb = torch.empty((2, 3, len(rows)), dtype=torch.float64, device="cuda")
    B.mt_demag_field_sparse(ctx, S, Ms, m, 2, Hb)
    B.mt_sparse_index(ctx, S)
    torch.cuda.synchronize()
    trunc = OT.truncate(host, tau)
    flat = trunc.reshape(6 * len(rows), n)
    cols_ref = np.nonzero(flat)[1]
    assert (cols_ref >= 65536).any()
    assert np.array_equal(S.cols16.cpu().numpy(), (cols_ref & 0xFFFF).astype(np.uint16))
    ptr = S.row_ptr.cpu().numpy()
    first_panel = np.count_nonzero(flat[:, :65536], axis=1)
    assert S.panel_ptr.shape == (6 * len(rows), 1)
    assert np.array_equal(S.panel_ptr.cpu().numpy()[:, 0], ptr[:-1] + first_panel)
    Hi = torch.empty_like(Hb)
    B.mt_demag_field_sparse(ctx, S, Ms, m, 2, Hi)
    torch.cuda.synchronize()
    ref = oracle.demag_field(trunc.astype(np.float64), w.Ms, w.m)
    for b in range(2):
        assert H.rel_l2(Hb[b].cpu().numpy(), ref[b]) <= 1e-5
        assert H.rel_l2(Hi[b].cpu().numpy(), ref[b]) <= 1e-5


def test_stream_calls_tau_given_and_argument_errors(ctx):
    """mt_sparse_stream_count / _fill (the streamed build as two library calls): a threshold handed in
    (fraction < 0) skips the selection and reproduces the selected build; bad arguments come back as
    MT_ERR_INVALID_ARG with a message, nothing is launched."""
    import ctypes as C
    w = W.config5(9, 6, 2, batch=1)
    tiles = H.dev_tiles(w)
    A = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, 0.6, 32)
    G = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, 0.0, 50, tau=A.tau)
    torch.cuda.synchronize()
    assert G.tau == A.tau and G.nnz == A.nnz and torch.equal(G.row_ptr, A.row_ptr)
    assert torch.equal(G.mask, A.mask) and torch.equal(G.vals, A.vals)
    n = w.n
    ld = W.leading_dim(n, "f32")
    band = torch.empty(6 * 16 * ld, dtype=torch.float32, device="cuda")
    row_ptr = torch.empty(6 * n + 1, dtype=torch.int64, device="cuda")
    t = tiles._c()
    tau, nnz = C.c_double(0.0), C.c_int64(0)

    def count(fraction, r0, r1, band_rows, band_ptr=band.data_ptr(), rp=row_ptr.data_ptr()):
        return ctx.lib.mt_sparse_stream_count(ctx.h, C.byref(t), B.MT_F32, fraction, r0, r1, band_ptr, band_rows, ld, rp,
                                              None, B.ALLREDUCE_FN(), None, None, C.byref(tau), C.byref(nnz))

    l0 = ctx.launches
    assert count(1.5, 0, n, 16) == B.MT_ERR_INVALID_ARG and b"fraction" in ctx.lib.mt_last_error(ctx.h)
    assert count(0.5, 5, 5, 16) == B.MT_ERR_INVALID_ARG        # empty band
    assert count(0.5, 0, n + 1, 16) == B.MT_ERR_INVALID_ARG    # beyond the tiles
    assert count(0.5, 0, n, 0) == B.MT_ERR_INVALID_ARG         # no band rows
    assert count(0.5, 0, n, 16, band_ptr=None) == B.MT_ERR_INVALID_ARG
    assert count(0.5, 0, n, 16, rp=None) == B.MT_ERR_INVALID_ARG
    assert ctx.lib.mt_sparse_stream_fill(ctx.h, C.byref(t), B.MT_F32, 0.1, 0, n, band.data_ptr(), 16, ld, row_ptr.data_ptr(),
                                         None, None, None, None, None) == B.MT_ERR_INVALID_ARG   # no output arrays
    assert ctx.launches == l0
    assert count(0.6, 0, n, 16) == B.MT_OK and tau.value == A.tau and nnz.value == A.nnz


def test_streamed_thresholding_row_sharded_with_histogram_allreduce(ctx, oracle):
    """DESIGN.md section 9 on F1: two "ranks" (threads with their own mt_ctx and stream on this one GPU)
    each build the thresholded rows of their half, exchanging only the selection histogram after every
    pass (an in-place sum, what dist.all_reduce does).  Both fix the whole tensor's threshold, and their
    bitmap rows / values / fields are the corresponding rows of the single-rank result."""
    import threading
    w = W.config5(13, 7, 3, batch=2)
    n = w.n
    tiles = H.dev_tiles(w)
    whole = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, 0.8, 64)
    B.mt_sparse_index(ctx, whole)
    m = torch.from_numpy(w.m).cuda()
    Hw = torch.empty_like(m)
    B.mt_demag_field_sparse(ctx, whole, tiles.Ms, m, 2, Hw)
    torch.cuda.synchronize()
    cut = 150
    bounds = [(0, cut), (cut, n)]
    barrier = threading.Barrier(2)
    slots, parts, errors = [None, None], [None, None], []

    def rank_main(rank):
        try:
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                c = B.mt_create(0, stream)

                def allreduce(hist):
                    stream.synchronize()
                    slots[rank] = hist.clone()
                    barrier.wait()
                    total = slots[0] + slots[1]
                    barrier.wait()
                    hist.copy_(total)

                S = B.mt_sparse_build_streamed(c, tiles, B.MT_F32, 0.8, 40, row_begin=bounds[rank][0],
                                               row_end=bounds[rank][1], allreduce=allreduce)
                B.mt_sparse_index(c, S)
                Hd = torch.empty((2, 3, S.n_rows), dtype=torch.float64, device="cuda")
                B.mt_demag_field_sparse(c, S, tiles.Ms, m, 2, Hd)
                stream.synchronize()
                parts[rank] = (S, Hd)
                c.close()
        except Exception as exc:  # surfaced in the main thread
            errors.append(exc)
            barrier.abort()

    threads = [threading.Thread(target=rank_main, args=(r,)) for r in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for rank, (r0, r1) in enumerate(bounds):
        S, Hd = parts[rank]
        assert S.tau == whole.tau and S.n_rows == r1 - r0
        assert torch.equal(S.mask, whole.mask[:, r0:r1])
        wp, sp = whole.row_ptr.cpu().numpy(), S.row_ptr.cpu().numpy()
        for p in range(6):
            a, b = wp[p * n + r0], wp[p * n + r1]
            c0, c1 = sp[p * (r1 - r0)], sp[(p + 1) * (r1 - r0)]
            assert b - a == c1 - c0 and torch.equal(whole.vals[a:b], S.vals[c0:c1])
        assert torch.equal(Hd, Hw[:, :, r0:r1])   # same kernel, same rows, same order: bit-identical


def test_morton_ordered_problem_through_the_device_path(ctx, oracle):
    """Tiles listed along a Z-order curve (workloads.morton_order / reorder): the right-hand side with
    exchange (renumbered neighbours), from the dense tensor and from index rows at a gap-placed 60 % cut,
    against the oracle on the reordered problem."""
    w0 = W.config3(6, batch=2)
    w = W.reorder(w0, W.morton_order(w0))
    n = w.n
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, "f32")
    assert status == 0
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    prob = H.dev_problem(w, tiles, N, "f32", ld)
    m = torch.from_numpy(w.m).cuda()
    k = torch.empty_like(m)
    B.mt_llg_rhs(ctx, prob, m, 2, k, None)
    torch.cuda.synchronize()
    k_ref, _ = oracle.llg_rhs(H.oracle_problem(oracle, w, N_ref), w.m)
    for b in range(2):
        assert H.rel_l2(k[b].cpu().numpy(), k_ref[b]) <= 1e-5
    host = N_ref.astype(np.float32)
    tau_dev, _ = B.mt_threshold_value(ctx, N, B.MT_F32, n, n, ld, 0.6)
    mags = np.unique(np.abs(host[np.abs(host) > 0]).astype(np.float64))
    gaps = np.nonzero(mags[1:] > mags[:-1] * 1.001)[0]
    g = gaps[np.argmin(np.abs(np.log(mags[gaps] / tau_dev)))]
    tau = float(np.float32(np.sqrt(mags[g] * mags[g + 1])))
    S = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, 0.6, 50, tau=tau)
    B.mt_sparse_index(ctx, S, drop_mask=True)
    prob.N = None
    prob.N_sparse = S
    B.mt_llg_rhs(ctx, prob, m, 2, k, None)
    torch.cuda.synchronize()
    trunc = OT.truncate(host, tau).astype(np.float64)
    k_ref, _ = oracle.llg_rhs(H.oracle_problem(oracle, w, trunc), w.m)
    for b in range(2):
        assert H.rel_l2(k[b].cpu().numpy(), k_ref[b]) <= 1e-5
