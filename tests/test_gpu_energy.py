"""-m gpu: F4 — energy terms (mt_energy) and the field-sweep loop (mt_field_sweep) through the C-ABI
against the oracle (oracle.energy_terms / oracle.field_sweep), plus the invariants that hold at
any size (energy non-increasing under damping on a uniform grid, bitwise reproducibility).
"""
import numpy as np
import pytest
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W
from tests import harness as H

pytestmark = pytest.mark.gpu

# relative to sum |terms| of the state: the fp64 path differs by summation order only, the fp32 path
# carries the H_d tolerance of north_star (1e-5 relative L2) into the demagnetisation term
TOL_E = {"f64": 1e-12, "f32": 1e-5}


@pytest.fixture(scope="module")
def ctx():
    c = B.mt_create(0)
    yield c
    c.close()


def gpu_energy(ctx, prob, m_np):
    m = torch.from_numpy(np.ascontiguousarray(m_np)).cuda()
    E = torch.empty((m.shape[0], 5), dtype=torch.float64, device="cuda")
    B.mt_energy(ctx, prob, m, m.shape[0], E)
    torch.cuda.synchronize()
    return E.cpu().numpy()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_energy_terms_cube_with_all_fields(ctx, oracle, dtype):
    """9^3 cube (ragged against every tile width) with exchange, anisotropy, applied field; 3 states."""
    w = W.config3(9, batch=3)
    w.H_a = np.array([0.05, -0.02, 0.03])
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    N, ld, _ = H.assemble(ctx, tiles, dtype)
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    E = gpu_energy(ctx, prob, w.m)
    op = H.oracle_problem(oracle, w, N_ref)
    for b in range(3):
        ref = oracle.energy_terms(op, w.m[b], vol=w.vol)
        scale = np.abs(ref).sum()
        assert np.max(np.abs(E[b, :4] - ref)) <= TOL_E[dtype] * scale, (E[b], ref)
        assert abs(E[b, 4] - ref.sum()) <= TOL_E[dtype] * scale
        assert E[b, 4] == ((E[b, 0] + E[b, 1]) + E[b, 2]) + E[b, 3]
    assert np.array_equal(E, gpu_energy(ctx, prob, w.m))  # fixed-order reductions


def test_energy_mixed_tiles_volume_weights(ctx, oracle):
    """Tetrahedra + octree cuboids (config 4 recipe, small): unequal volumes weight the sums."""
    w = W.config4(n_tets=300, n_cub=212, n_points=120, batch=2)
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    N, ld, _ = H.assemble(ctx, tiles, "f64")
    prob = H.dev_problem(w, tiles, N, "f64", ld)
    E = gpu_energy(ctx, prob, w.m)
    op = H.oracle_problem(oracle, w, N_ref)
    for b in range(2):
        ref = oracle.energy_terms(op, w.m[b], vol=w.vol)
        assert np.max(np.abs(E[b, :4] - ref)) <= 1e-12 * np.abs(ref).sum()


def test_energy_non_increasing_along_gpu_trajectory(ctx):
    """P14 on the device: with alpha > 0 and a constant field the total energy of a
    uniform-grid problem never increases along the integrated trajectory."""
    w = W.config3(8)
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(ctx, tiles, "f32")
    prob = H.dev_problem(w, tiles, N, "f32", ld)
    m = torch.from_numpy(w.m[:1].copy()).cuda()
    E = torch.empty((1, 5), dtype=torch.float64, device="cuda")
    hist = []
    t = 0.0
    for _ in range(12):
        B.mt_energy(ctx, prob, m, 1, E)
        hist.append(float(E[0, 4].item()))
        t, _, _ = B.mt_integrate(ctx, prob, m, 1, t, method=B.MT_RK4, dt=0.01, t_end=t + 0.1)
    assert np.all(np.diff(hist) < 0), hist


@pytest.mark.parametrize("method", ["rk4", "dp45"])
def test_field_sweep_matches_oracle(ctx, oracle, method):
    """Hysteresis-loop driver on a 12x6x2 film with exchange (SP2-like shape): five
    field steps, each relaxed for a fixed time from the previous end state; <m> and the energy terms
    of every step against the oracle's loop."""
    g = W._cuboid_workload("film", 12, 6, 2, (0.5, 0.5, 0.25), 1.0, W.random_unit_states(W.rng_for(3, 5), 2, 144),
                           nbr=W.grid_neighbours(12, 6, 2), inv_d2=np.array([4.0, 4.0, 16.0]), c_ex=1.0, c_an=0.05,
                           easy=np.array([1.0, 0.0, 0.0]), H_a=np.zeros(3), gamma=1.0, alpha_ll=1.0)
    tiles = H.dev_tiles(g)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, g), long_double=True)
    N, ld, _ = H.assemble(ctx, tiles, "f64")
    prob = H.dev_problem(g, tiles, N, "f64", ld)
    fields = [[0.3 * c, 0.05, 0.0] for c in (1.0, 0.5, 0.0, -0.5, -1.0)]
    if method == "rk4":
        kw_o = dict(method=oracle.RK4, dt=0.02, t_end=1.0)
        kw_g = dict(method=B.MT_RK4, dt=0.02, t_end=1.0)
    else:
        kw_o = dict(method=oracle.DP45, dt=1e-2, t_end=1.0, rtol=1e-7, atol=1e-9)
        kw_g = dict(method=B.MT_DP45, dt=1e-2, t_end=1.0, rtol=1e-7, atol=1e-9)
    # DP45 batches share one step sequence (max error over the states): compare it state by state
    nb = 2 if method == "rk4" else 1
    m = torch.from_numpy(g.m[:nb].copy()).cuda()
    rows = torch.zeros((len(fields), nb, 8), dtype=torch.float64, device="cuda")
    res, rc = B.mt_field_sweep(ctx, prob, fields, m, nb, rows, **kw_g)
    assert rc == 0 and abs(res["t"] - len(fields) * 1.0) < 1e-12
    got = rows.cpu().numpy()
    op = H.oracle_problem(oracle, g, N_ref)
    for b in range(nb):
        m_ref, ref = oracle.field_sweep(op, g.m[b], fields, vol=g.vol, **kw_o)
        assert np.max(np.abs(got[:, b, :3] - ref[:, :3])) < 1e-8
        scale = np.abs(ref[:, 3:]).sum(axis=1, keepdims=True)
        assert np.max(np.abs(got[:, b, 3:7] - ref[:, 3:]) / scale) < 1e-8
        assert np.allclose(got[:, b, 7], got[:, b, 3:7].sum(axis=1), rtol=1e-14)
        assert np.max(np.abs(m[b].cpu().numpy() - m_ref)) < 1e-7
    # once the random start has relaxed (first step), <m_x> follows the falling field
    assert np.all(np.diff(got[1:, 0, 0]) < 0)
