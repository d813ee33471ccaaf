"""-m gpu: the row-sharded right-hand side and integrators (mt.h section 8(e)) through the
C-ABI on ONE GPU: `world` threads, each with its own mt_ctx, stream, row band of the tensor and
`binding.Shard`; the exchange callback is a host-side hand-over between the threads (stream
synchronise, barrier, device copies of the peers' blocks, barrier) — no kernel waits on another.
What is under test is the library side of the protocol: band launches with global row indices in the
fused epilogue, stage states routed through the gather blocks, the scatter kernel, the reduced
error / torque words and a host controller that takes the same decisions on every rank.  The
torch.distributed side of the same protocol is covered by tests/test_sharding_gloo.py.
"""
import threading

import numpy as np
import pytest
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import sharding as S
from paper_2107_05364_b200 import workloads as W
from tests import harness as H

pytestmark = pytest.mark.gpu


class ThreadExchange:
    """exchange callbacks of `world` ranks living in threads of one process on one device."""

    def __init__(self, world):
        self.world = world
        self.barrier = threading.Barrier(world, timeout=60)
        self.shards = [None] * world
        self.streams = [None] * world
        self.calls = [0, 0]

    def make(self, rank):
        def exchange(what, pack, scal, cuda_stream):
            st = self.streams[rank]
            st.synchronize()           # my block / my words are written
            self.barrier.wait()
            with torch.cuda.stream(st):
                if what == S.GATHER_STATE:
                    for g in range(self.world):
                        if g != rank:
                            pack[g].copy_(self.shards[g].pack[g])
                    new = None
                else:
                    new = torch.stack([self.shards[g].scal for g in range(self.world)]).max(dim=0).values
            st.synchronize()           # everyone has read the peers' data ...
            self.barrier.wait()
            if new is not None:        # ... before anyone's words change
                with torch.cuda.stream(st):
                    scal.copy_(new)
            if rank == 0:
                self.calls[what] += 1
        return exchange


def run_sharded(world, w, dtype, fn, batch=1):
    """Runs fn(ctx, prob, rank) in `world` threads, each holding its row band; returns the results."""
    xch = ThreadExchange(world)
    out, errs = [None] * world, []

    def worker(rank):
        try:
            st = torch.cuda.Stream()
            xch.streams[rank] = st
            with torch.cuda.stream(st):
                ctx = B.mt_create(0, st)
                tiles = H.dev_tiles(w)
                r0, r1 = S.row_band(rank, world, w.n)
                N, ld, status = H.assemble(ctx, tiles, dtype, r0, r1)
                assert status == 0
                shard = B.Shard(rank, world, w.n, batch, "cuda:0", xch.make(rank))
                xch.shards[rank] = shard
                prob = H.dev_problem(w, tiles, N, dtype, ld)
                prob.shard = shard
                xch.barrier.wait()
                out[rank] = fn(ctx, prob, rank)
                st.synchronize()
                if shard.error is not None:
                    raise shard.error
                ctx.close()
        except Exception as exc:  # noqa: BLE001
            errs.append((rank, exc))
            xch.barrier.abort()

    threads = [threading.Thread(target=worker, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=600)
    assert not errs, errs
    return out, xch


def run_single(w, dtype, fn):
    ctx = B.mt_create(0)
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, dtype)
    assert status == 0
    res = fn(ctx, H.dev_problem(w, tiles, N, dtype, ld), 0)
    torch.cuda.synchronize()
    ctx.close()
    return res


def integrate_fn(w, batch, **kw):
    def fn(ctx, prob, rank):
        m = torch.from_numpy(np.ascontiguousarray(w.m[:batch])).cuda()
        cap = kw.get("sample_cap", 0)
        samples = torch.zeros((max(cap, 1), 1 + 3 * batch), dtype=torch.float64, device="cuda")
        args = {k: v for k, v in kw.items() if k != "sample_cap"}
        t, res, rc = B.mt_integrate(ctx, prob, m, batch, 0.0, samples=samples if cap else None, **args)
        ctx.stream.synchronize()
        return m.cpu().numpy(), samples[: res["n_samples"]].cpu().numpy(), res, t
    return fn


@pytest.mark.parametrize("world,n1,dtype", [(2, 8, "f64"), (3, 8, "f64"), (2, 16, "f32")])
def test_sharded_rhs_rows(world, n1, dtype):
    """mt_llg_rhs on a band writes exactly the band's rows (global positions), equal to the full call's."""
    w = W.config3(n1, batch=2)

    def fn(ctx, prob, rank):
        m = torch.from_numpy(np.ascontiguousarray(w.m)).cuda()
        k = torch.full_like(m, 7.0)
        h = torch.full_like(m, 7.0)
        B.mt_llg_rhs(ctx, prob, m, 2, k, h)
        ctx.stream.synchronize()
        return k.cpu().numpy(), h.cpu().numpy()

    k_full, h_full = run_single(w, dtype, fn)
    outs, _ = run_sharded(world, w, dtype, fn, batch=2)
    tol = 1e-13 if dtype == "f64" else 2e-6
    for rank, (k, h) in enumerate(outs):
        r0, r1 = S.row_band(rank, world, w.n)
        scale = np.abs(k_full).max()
        assert np.max(np.abs(k[:, :, r0:r1] - k_full[:, :, r0:r1])) <= tol * scale
        assert np.max(np.abs(h[:, :, r0:r1] - h_full[:, :, r0:r1])) <= tol * np.abs(h_full).max()
        mask = np.ones(w.n, bool)
        mask[r0:r1] = False
        assert np.all(k[:, :, mask] == 7.0) and np.all(h[:, :, mask] == 7.0)


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_rk4_matches_single_ctx_and_oracle(oracle, world):
    """8^3 replica of config 3 (exchange neighbours cross the band boundaries; 512 rows over 3 ranks:
    uneven bands): sharded RK4 = the single-context run to rounding = the oracle's RK4."""
    w = W.config3(8, batch=2)
    kw = dict(method=B.MT_RK4, dt=2e-3, t_end=0.08, sample_every=10, sample_cap=8)
    m1, s1, r1, _ = run_single(w, "f64", integrate_fn(w, 2, **kw))
    outs, xch = run_sharded(world, w, "f64", integrate_fn(w, 2, **kw), batch=2)
    for m, s, r, t in outs:
        assert r["accepted"] == 40 and r["rhs_calls"] == 160 and t == pytest.approx(0.08)
        assert np.max(np.abs(m - m1)) < 1e-12 and np.max(np.abs(s - s1)) < 1e-12
        assert np.array_equal(m, outs[0][0])  # every rank holds the same state, bit for bit
    assert xch.calls[S.GATHER_STATE] == 160  # one exchange per stage
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    m_o, _, _ = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.RK4, dt=2e-3, t_end=0.08)
    assert np.max(np.abs(outs[0][0][0] - m_o)) < 1e-10
    assert np.max(np.abs(m_o - w.m[0])) > 1e-2


def test_sharded_dp45_takes_the_same_steps(oracle):
    """DP45 with the error / torque words max-reduced over the ranks: same accept / reject sequence and
    samples as the single-context run and as the oracle (fp64 tensor), torque stop included."""
    w = W.config3(8)
    x = w.extra
    kw = dict(method=B.MT_DP45, dt=x["dt0"], t_end=3.0, rtol=x["rtol"], atol=x["atol"], torque_tol=1e-4,
              sample_dt=0.5, sample_cap=8)
    m1, s1, r1, _ = run_single(w, "f64", integrate_fn(w, 1, **kw))
    outs, xch = run_sharded(2, w, "f64", integrate_fn(w, 1, **kw))
    for m, s, r, t in outs:
        assert (r["accepted"], r["rejected"], r["rhs_calls"]) == (r1["accepted"], r1["rejected"], r1["rhs_calls"])
        assert r["rejected"] > 0 and len(s) == 6 and np.array_equal(s[:, 0], s1[:, 0])
        assert np.max(np.abs(m - m1)) < 1e-10 and np.max(np.abs(s - s1)) < 1e-10
        assert abs(r["max_torque"] - r1["max_torque"]) <= 1e-9 * r1["max_torque"]
    assert xch.calls[S.MAX_SCALARS] == 1 + r1["accepted"] + r1["rejected"]
    assert xch.calls[S.GATHER_STATE] == 6 * (r1["accepted"] + r1["rejected"]) + r1["accepted"]
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    kwo = {k: v for k, v in kw.items() if k != "method"}
    m_o, s_o, r_o = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.DP45, weights=w.vol, **kwo)
    assert (r_o["accepted"], r_o["rejected"]) == (outs[0][2]["accepted"], outs[0][2]["rejected"])
    assert np.max(np.abs(outs[0][1][:, 1:] - s_o[:, 1:])) < 1e-9


def test_sharded_rk4_tma_bands_fp32():
    """16^3 (N = 4,096, fp32): the 2,048-row bands run the TMA pipeline kernel (row groups split between
    CTAs, fix-up kernel with global row indices); trajectory equal to the single-context run to fp32
    summation-order differences, far inside the 1e-3 gate."""
    w = W.config3(16, batch=1)
    kw = dict(method=B.MT_RK4, dt=2e-3, t_end=0.04, sample_every=5, sample_cap=8)
    m1, s1, r1, _ = run_single(w, "f32", integrate_fn(w, 1, **kw))
    outs, _ = run_sharded(2, w, "f32", integrate_fn(w, 1, **kw))
    for m, s, r, t in outs:
        assert r["accepted"] == 20
        assert np.max(np.abs(m - m1)) < 1e-6 and np.max(np.abs(s - s1)) < 1e-7
        assert np.max(np.abs(np.linalg.norm(m[0], axis=0) - 1.0)) < 1e-14


def test_sharded_rk4_on_a_row_sharded_thresholded_tensor():
    """The thresholded tensor (F1) shards by rows like the dense one: every rank compresses its band with the
    whole tensor's threshold (index rows) and runs the sharded RK4 on it; the result equals the single-context
    run on the whole thresholded tensor."""
    w = W.config3(8, batch=1)
    kw = dict(method=B.MT_RK4, dt=2e-3, t_end=0.04)

    def with_sparse(ctx, prob, rank, tau_box=[None]):
        n = w.n
        rows = prob.N.shape[1]
        if tau_box[0] is None:          # the single-context call comes first and fixes the threshold
            tau_box[0], _ = B.mt_threshold_value(ctx, prob.N, B.MT_F64, n, rows, prob.ld, 0.5)
        S = B.mt_sparse_build(ctx, prob.N, B.MT_F64, n, rows, prob.ld, tau_box[0])
        B.mt_sparse_index(ctx, S, drop_mask=True)
        prob.N_sparse, prob.N = S, None
        return integrate_fn(w, 1, **kw)(ctx, prob, rank)

    m1, _, r1, _ = run_single(w, "f64", with_sparse)
    outs, xch = run_sharded(2, w, "f64", with_sparse)
    for m, _, r, _ in outs:
        assert r["accepted"] == 20
        assert np.max(np.abs(m - m1)) < 1e-12
    assert np.array_equal(outs[0][0], outs[1][0]) and xch.calls[S.GATHER_STATE] == 80
    # and thresholding did change the dynamics a little (the test is not run on an untouched tensor)
    m0, _, _, _ = run_single(w, "f64", integrate_fn(w, 1, **kw))
    assert 1e-9 < np.max(np.abs(m0 - m1)) < 1e-2


def test_sharded_argument_errors():
    w = W.config3(4)
    ctx = B.mt_create(0)
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(ctx, tiles, "f64")       # all 64 rows: not a band
    prob = H.dev_problem(w, tiles, N, "f64", ld)
    prob.shard = B.Shard(0, 2, w.n, 1, "cuda:0", lambda *a: None)
    m = torch.from_numpy(np.ascontiguousarray(w.m[:1])).cuda()
    E = torch.zeros((1, 5), dtype=torch.float64, device="cuda")
    with pytest.raises(B.MtError) as ei:
        B.mt_energy(ctx, prob, m, 1, E)
    assert ei.value.code == B.MT_ERR_INVALID_ARG
    prob.shard = B.Shard(0, 2, w.n, 1, "cuda:0", lambda *a: None)
    prob.shard._c_struct.slice_pad = 3  # shorter than the band
    with pytest.raises(B.MtError) as ei:
        B.mt_llg_rhs(ctx, prob, m, 1, torch.empty_like(m), None)
    assert ei.value.code == B.MT_ERR_INVALID_ARG
    ctx.close()
