"""-m gpu: the TMA bulk-tensor pipeline variant of the demag kernel (csrc/demag_tma.cu), forced with
mt_set_demag_variant(ctx, 2) at sizes where the default dispatch would pick the register-streaming
kernel: few tiles (CTAs with empty ranges, row groups split between many CTAs -> the fixed-order
second pass), ragged rows/columns (hardware zero fill), row bands, all batch sizes, both dtypes,
the fused right-hand side and the integrators.  Oracle tolerances as in test_gpu_small.py.
"""
import numpy as np
import pytest
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W
from tests import harness as H

pytestmark = pytest.mark.gpu

TOL_HD = {"f64": 1e-12, "f32": 1e-5}


@pytest.fixture(scope="module")
def ctx():
    c = B.mt_create(0)
    B.mt_set_demag_variant(c, 2)
    yield c
    c.close()


def field(ctx, N, dtype, n, n_rows, ld, Ms, m_np):
    m = torch.from_numpy(np.ascontiguousarray(m_np)).cuda()
    Hd = torch.full((m.shape[0], 3, n_rows), float("nan"), dtype=torch.float64, device="cuda")
    B.mt_demag_field(ctx, N, H.dtype_code(dtype), n, n_rows, ld, Ms, m, m.shape[0], Hd)
    torch.cuda.synchronize()
    return Hd.cpu().numpy()


@pytest.mark.parametrize("grid,dtype,batch", [
    ((1, 1, 1), "f64", 1), ((3, 1, 1), "f32", 2), ((7, 5, 3), "f32", 1), ((7, 5, 3), "f64", 4),
    ((33, 31, 1), "f32", 3), ((16, 12, 4), "f32", 8), ((16, 12, 4), "f64", 8), ((41, 11, 3), "f32", 5),
    ((41, 11, 3), "f64", 6), ((41, 11, 3), "f32", 6), ((50, 30, 2), "f32", 7), ((50, 30, 2), "f32", 1)])
def test_tma_field_matches_oracle(ctx, oracle, grid, dtype, batch):
    nx, ny, nz = grid
    n = nx * ny * nz
    rng = np.random.default_rng(1000 + n + batch)
    w = W._cuboid_workload("tma", nx, ny, nz, (1.0, 0.8, 1.25), 1.0, W.random_unit_states(rng, batch, n))
    w.Ms = rng.uniform(0.5, 2.0, size=n)
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    Hd_ref = oracle.demag_field(N_ref, w.Ms, w.m)
    ld = W.leading_dim(n, dtype) + 4
    N, ld, _ = H.assemble(ctx, tiles, dtype, ld=ld)
    l0 = ctx.launches
    Hd = field(ctx, N, dtype, n, n, ld, tiles.Ms, w.m)
    # stage_M + demag_tma, split row groups finished inside it (+ the B-fragment re-layout of M in front of
    # the tensor-core kernel that serves 5..8 states on fp32 tensors)
    assert ctx.launches - l0 == (3 if dtype == "f32" and batch >= 5 else 2)
    assert np.isfinite(Hd).all()
    for b in range(batch):
        assert H.rel_l2(Hd[b], Hd_ref[b]) <= TOL_HD[dtype]
    # bitwise reproducible run to run
    for _ in range(3):
        assert np.array_equal(field(ctx, N, dtype, n, n, ld, tiles.Ms, w.m), Hd)
    # a row band gives the band's field
    if n >= 8:
        r0, r1 = n // 5, n - 3
        Nb, _, _ = H.assemble(ctx, tiles, dtype, r0, r1, ld=ld)
        Hb = field(ctx, Nb, dtype, n, r1 - r0, ld, tiles.Ms, w.m)
        for b in range(batch):
            assert H.rel_l2(Hb[b], Hd_ref[b][:, r0:r1]) <= TOL_HD[dtype]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_tma_fused_rhs_and_integrators(ctx, oracle, dtype):
    w = W.config3(10, batch=2)  # 1000 tiles: exchange + anisotropy, ragged in rows and columns
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    N, ld, _ = H.assemble(ctx, tiles, dtype)
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    oprob = H.oracle_problem(oracle, w, N_ref)
    m = torch.from_numpy(w.m).cuda()
    k = torch.empty_like(m)
    heff = torch.empty_like(m)
    B.mt_llg_rhs(ctx, prob, m, 2, k, heff)
    torch.cuda.synchronize()
    k_ref, h_ref, _ = oracle.llg_rhs(oprob, w.m, want_heff=True)
    assert H.rel_l2(k.cpu().numpy(), k_ref) <= TOL_HD[dtype]
    assert H.rel_l2(heff.cpu().numpy(), h_ref) <= TOL_HD[dtype]
    tol = 1e-9 if dtype == "f64" else 1e-4
    m1 = torch.from_numpy(w.m[:1].copy()).cuda()
    B.mt_integrate(ctx, prob, m1, 1, 0.0, method=B.MT_RK4, dt=0.005, t_end=0.4)
    m_ref, _, _ = oracle.integrate(oprob, w.m[0], method=oracle.RK4, dt=0.005, t_end=0.4)
    assert np.max(np.abs(m1.cpu().numpy()[0] - m_ref)) < tol
    m1 = torch.from_numpy(w.m[:1].copy()).cuda()
    B.mt_integrate(ctx, prob, m1, 1, 0.0, method=B.MT_DP45, dt=1e-3, t_end=0.3, rtol=1e-6, atol=1e-8)
    m_ref, _, _ = oracle.integrate(oprob, w.m[0], method=oracle.DP45, dt=1e-3, t_end=0.3, rtol=1e-6, atol=1e-8)
    assert np.max(np.abs(m1.cpu().numpy()[0] - m_ref)) < 1e-4


def test_tma_and_ldg_variants_agree(ctx):
    w = W.config5(32, 16, 4, batch=8)  # n = 2048
    tiles = H.dev_tiles(w)
    c1 = B.mt_create(0)
    B.mt_set_demag_variant(c1, 1)
    try:
        for dtype in ("f32", "f64"):
            N, ld, _ = H.assemble(ctx, tiles, dtype)
            a = field(ctx, N, dtype, w.n, w.n, ld, tiles.Ms, w.m)
            b = field(c1, N, dtype, w.n, w.n, ld, tiles.Ms, w.m)
            assert H.rel_l2(a, b) <= (1e-6 if dtype == "f32" else 1e-14)
    finally:
        c1.close()
