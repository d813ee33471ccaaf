"""-m gpu: F3 — field, right-hand side and trajectories from the pair-symmetric half of the tensor
 against the oracle's FULL tensor (the half is a storage choice: the result is the same
product), on grids that are ragged against the 32-row blocks and the 128/64-column tiles."""
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
    yield c
    c.close()


def build_sym(ctx, tiles, dtype):
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    S = B.mt_assemble_tensor_sym(ctx, tiles, H.dtype_code(dtype), status)
    torch.cuda.synchronize()
    return S, int(status.item())


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [(8, 8, 8), (13, 7, 3), (20, 10, 2), (5, 3, 1), (31, 9, 5)])
def test_sym_field_matches_oracle_full_tensor(ctx, oracle, grid, dtype):
    w = W.config5(*grid, batch=3)
    tiles = H.dev_tiles(w)
    S, status = build_sym(ctx, tiles, dtype)
    assert status == 0
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    ref = oracle.demag_field(N_ref, w.Ms, w.m)
    m = torch.from_numpy(w.m).cuda()
    Hd = torch.empty_like(m)
    B.mt_demag_field_sym(ctx, S, tiles.Ms, m, 3, Hd)
    torch.cuda.synchronize()
    for b in range(3):
        assert H.rel_l2(Hd[b].cpu().numpy(), ref[b]) <= TOL_HD[dtype]
    Hd2 = torch.empty_like(m)
    B.mt_demag_field_sym(ctx, S, tiles.Ms, m, 3, Hd2)
    assert torch.equal(Hd, Hd2)


def test_sym_storage_is_about_half(ctx):
    n = 4096
    full = 6 * n * n
    elems = int(ctx.lib.mt_sym_tensor_elems(n, B.MT_F32))
    assert 0.5 * full < elems < 0.53 * full


def test_sym_rejects_non_congruent_meshes(ctx):
    w = W.config5(8, 8, 2, batch=1)
    w.size = w.size.copy()
    w.size[77] = [0.5, 1.0, 1.0]  # one cuboid of another size
    _, status = build_sym(ctx, H.dev_tiles(w), "f32")
    assert status & 2
    w = W.config4(n_tets=200, n_cub=56, n_points=100)
    _, status = build_sym(ctx, H.dev_tiles(w), "f32")
    assert status & 2


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_sym_rhs_energy_and_trajectory(ctx, oracle, dtype):
    """Fused right-hand side, energies and a short RK4 + DP45 run through mt_problem.N_sym."""
    w = W.config3(7, batch=2)
    tiles = H.dev_tiles(w)
    S, status = build_sym(ctx, tiles, dtype)
    assert status == 0
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    op = H.oracle_problem(oracle, w, N_ref)
    prob = H.dev_problem(w, tiles, None, dtype, 0)
    prob.N_sym = S
    m = torch.from_numpy(w.m).cuda()
    k = torch.empty_like(m)
    B.mt_llg_rhs(ctx, prob, m, 2, k, None)
    torch.cuda.synchronize()
    k_ref, _ = oracle.llg_rhs(op, w.m)
    assert H.rel_l2(k.cpu().numpy(), k_ref) <= TOL_HD[dtype]
    E = torch.empty((2, 5), dtype=torch.float64, device="cuda")
    B.mt_energy(ctx, prob, m, 2, E)
    for b in range(2):
        ref = oracle.energy_terms(op, w.m[b], vol=w.vol)
        assert np.max(np.abs(E[b, :4].cpu().numpy() - ref)) <= TOL_HD[dtype] * np.abs(ref).sum()
    tol = 1e-9 if dtype == "f64" else 1e-4
    m1 = torch.from_numpy(w.m[:1].copy()).cuda()
    B.mt_integrate(ctx, prob, m1, 1, 0.0, method=B.MT_RK4, dt=0.01, t_end=0.3)
    m_ref, _, _ = oracle.integrate(op, w.m[0], method=oracle.RK4, dt=0.01, t_end=0.3)
    assert np.max(np.abs(m1[0].cpu().numpy() - m_ref)) < tol
    m1 = torch.from_numpy(w.m[:1].copy()).cuda()
    B.mt_integrate(ctx, prob, m1, 1, 0.0, method=B.MT_DP45, dt=1e-3, t_end=0.5, rtol=1e-6, atol=1e-8)
    m_ref, _, _ = oracle.integrate(op, w.m[0], method=oracle.DP45, dt=1e-3, t_end=0.5, rtol=1e-6, atol=1e-8)
    assert np.max(np.abs(m1[0].cpu().numpy() - m_ref)) < max(tol, 1e-6)
