"""-m gpu: F2 — far-field-stable assembly (mt_set_assembly_mode(1)) against the long-double oracle,
per BLOCK (max-norm relative error of each 3x3 block), on geometries whose pair distances reach
~190 tile edges; and the documented loss of the closed form in fp64 with mode 0.
The long-double closed form is itself good to ~3e-12 at 200 edges, which bounds what can be gated."""
import numpy as np
import pytest
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W
from tests import harness as H

pytestmark = pytest.mark.gpu


@pytest.fixture()
def ctx():
    c = B.mt_create(0)
    yield c
    c.close()


def block_rel_err(got, ref):
    """[rows, n] max-norm error of each block relative to the block's max-norm."""
    return np.max(np.abs(got - ref), axis=0) / np.max(np.abs(ref), axis=0)


def distances(w, rows):
    d = w.center[rows][:, None, :] - w.center[None, :, :]
    return np.linalg.norm(d, axis=2) / (w.size.max(axis=1)[None, :])


@pytest.mark.parametrize("grid,edge", [((192, 4, 2), 1.0), ((160, 40, 1), (3.125e-9, 3.125e-9, 3e-9)), ((70, 9, 5), (0.5, 0.25, 0.125))])
def test_far_field_stable_assembly_per_block(ctx, oracle, grid, edge):
    nx, ny, nz = grid
    n = nx * ny * nz
    w = W._cuboid_workload("bar", nx, ny, nz, edge, 1.0, W.random_unit_states(W.rng_for(5, 3), 1, n))
    tiles = H.dev_tiles(w)
    rows = np.array(sorted({0, nx - 1, n // 2, n - 1, n - nx, 17 % n}), dtype=np.int64)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=rows, long_double=True)
    r = distances(w, rows)
    assert r.max() > 60
    errs = {}
    for mode in (0, 1):
        B.mt_set_assembly_mode(ctx, mode)
        N, ld, status = H.assemble(ctx, tiles, "f64")
        assert status == 0
        got = N[:, torch.from_numpy(rows).cuda(), :n].cpu().numpy()
        errs[mode] = block_rel_err(got, N_ref)
    # mode 1: every block within 1e-10 of the long-double value, at every distance
    assert errs[1].max() <= 1e-10, errs[1].max()
    # near field (closed form in both modes) is bit-identical between the modes
    near = r < 15.9
    assert np.array_equal(errs[0][near], errs[1][near])
    # mode 0 shows the growth the paper warns about: beyond 60 edges it is worse than mode 1 by > 10x
    far = r > 60
    assert errs[0][far].max() > 10 * errs[1][far].max()
    # the fp32 tensor of mode 1 is within 1 ulp of the rounded oracle value as well
    B.mt_set_assembly_mode(ctx, 1)
    N32, ld32, _ = H.assemble(ctx, tiles, "f32")
    got32 = N32[:, torch.from_numpy(rows).cuda(), :n].cpu().numpy()
    ulp = H.f32_ulp_distance(got32, N_ref)
    assert ((ulp <= 1) | (np.abs(got32.astype(np.float64) - N_ref) < 1e-15 * np.abs(N_ref).max())).all()


def test_far_field_mode_field_matches_oracle(ctx, oracle):
    """H_d from a mode-1 tensor on a 96x6x3 bar: same tolerance as the closed-form tensor."""
    w = W.config5(96, 6, 3, batch=2)
    tiles = H.dev_tiles(w)
    B.mt_set_assembly_mode(ctx, 1)
    N, ld, _ = H.assemble(ctx, tiles, "f64")
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    m = torch.from_numpy(w.m).cuda()
    Hd = torch.empty_like(m)
    B.mt_demag_field(ctx, N, B.MT_F64, w.n, w.n, ld, tiles.Ms, m, 2, Hd)
    torch.cuda.synchronize()
    ref = oracle.demag_field(N_ref, w.Ms, w.m)
    for b in range(2):
        assert H.rel_l2(Hd[b].cpu().numpy(), ref[b]) <= 1e-12
    with pytest.raises(B.MtError):
        B.mt_set_assembly_mode(ctx, 7)


def test_far_field_mode_applies_to_the_symmetric_half(ctx, oracle):
    """mt_assemble_tensor_sym honours mt_set_assembly_mode: on a 160x3x1 bar (pairs out to 159 edges)
    the field from the mode-1 half is closer to the oracle than from the mode-0 half, and both pass
    the fp64 tolerance north_star sets for H_d."""
    w = W.config5(160, 3, 1, batch=2)
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    ref = oracle.demag_field(N_ref, w.Ms, w.m)
    m = torch.from_numpy(w.m).cuda()
    err = {}
    for mode in (0, 1):
        B.mt_set_assembly_mode(ctx, mode)
        status = torch.zeros(1, dtype=torch.int32, device="cuda")
        S = B.mt_assemble_tensor_sym(ctx, tiles, B.MT_F64, status)
        Hd = torch.empty_like(m)
        B.mt_demag_field_sym(ctx, S, tiles.Ms, m, 2, Hd)
        torch.cuda.synchronize()
        assert int(status.item()) == 0
        err[mode] = max(H.rel_l2(Hd[b].cpu().numpy(), ref[b]) for b in range(2))
        assert err[mode] <= 1e-12
    assert err[1] <= err[0]


def test_far_field_stable_assembly_tetrahedron_sources(ctx, oracle):
    """F2 for tetrahedra: Delaunay tetrahedra of a small ball as sources, targets spread out to ~60
    of their edges (config 4's range: ball of radius 1, slab at +3, edges ~0.1).  Mode 1 keeps every
    block within 1e-10 of the long-double oracle; the fp64 polyhedron closed form (mode 0) is more
    than 10x worse beyond 20 edges."""
    w = W.config4(n_tets=400, n_cub=0, n_points=150, batch=1, body="tets")
    n = w.n
    edge = np.max(np.linalg.norm(w.verts[:, :, None, :] - w.verts[:, None, :, :], axis=3), axis=(1, 2))
    # move every second tile's evaluation point far away along a seeded direction: the tensor only uses
    # `center` of the TARGET and `verts` of the SOURCE, so this probes far-field blocks of real tetrahedra
    rng = W.rng_for(4, 9)
    far = np.arange(n) % 2 == 1
    u = rng.standard_normal((n, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    w.center = w.center.copy()
    w.center[far] = u[far] * rng.uniform(3.0, 30.0, size=(far.sum(), 1))
    tiles = H.dev_tiles(w)
    rows = np.flatnonzero(far)[:40].astype(np.int64)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=rows, long_double=True)
    src_cent = w.verts.mean(axis=1)
    r = np.linalg.norm(w.center[rows][:, None, :] - src_cent[None, :, :], axis=2) / edge[None, :]
    assert r.max() > 40
    errs = {}
    for mode in (0, 1):
        B.mt_set_assembly_mode(ctx, mode)
        N, ld, status = H.assemble(ctx, tiles, "f64")
        assert status == 0
        got = N[:, torch.from_numpy(rows).cuda(), :n].cpu().numpy()
        errs[mode] = block_rel_err(got, N_ref)
    assert errs[1].max() <= 1e-10, errs[1].max()
    near = r < 7.9  # closed form in both modes (the two instantiations may contract FMAs differently)
    assert errs[0][near].max() <= 1e-10 and errs[1][near].max() <= 1e-10
    sel = r > 20
    assert errs[0][sel].max() > 10 * errs[1][sel].max()
