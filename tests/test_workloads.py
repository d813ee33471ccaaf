"""-m "not gpu": host logic of the seeded input generators (no method arithmetic)."""
import numpy as np
import pytest

from paper_2107_05364_b200 import workloads as W


def test_seeds_are_reproducible_and_distinct():
    a, b = W.config1(), W.config1()
    assert np.array_equal(a.m, b.m)
    assert not np.array_equal(W.config1().m[0], W.config5(8, 8, 8, 1).m[0])
    assert np.allclose(np.linalg.norm(a.m, axis=1), 1.0, atol=1e-15)


def test_grid_layout_and_neighbours():
    c, s = W.cuboid_grid(4, 3, 2, (1.0, 2.0, 3.0))
    assert np.array_equal(c[0], [0.5, 1.0, 1.5]) and np.array_equal(c[1], [1.5, 1.0, 1.5])  # x fastest
    assert np.array_equal(c[4], [0.5, 3.0, 1.5]) and np.array_equal(c[12], [0.5, 1.0, 4.5])
    nbr = W.grid_neighbours(4, 3, 2)
    assert nbr.shape == (24, 6) and nbr.dtype == np.int32
    assert list(nbr[0]) == [-1, 1, -1, 4, -1, 12]
    assert list(nbr[23]) == [22, -1, 19, -1, 11, -1]
    # symmetric relation
    for i in range(24):
        for d in range(6):
            j = nbr[i, d]
            if j >= 0:
                assert nbr[j, d ^ 1] == i


def test_config2_parameters():
    w = W.config2()
    assert w.n == 6400 and w.dtype == "f32"
    assert np.allclose(w.size[0], [3.125e-9, 3.125e-9, 3e-9])
    assert abs(w.c_ex - 2.58627e-11) < 1e-15            # 2A/(mu0 Ms)
    assert abs(np.hypot(*w.H_a[:2]) - 19894.37) < 0.01   # 25 mT / mu0
    assert abs(w.alpha_ll - 4422.0) < 1e-9               # gamma * 0.02 (reading Q5)
    r = W.config2(phase="relax")
    assert r.H_a == (0.0, 0.0, 0.0) and r.alpha_ll == r.gamma
    assert np.array_equal(r.m, w.m)
    dev = w.m[0] - 1 / np.sqrt(3)
    assert 0.003 < dev.std() < 0.02                      # 1 % perturbation


def test_config4_mesh_is_valid():
    w = W.config4(n_tets=2000, n_cub=2048, n_points=500)
    tets = w.verts[w.type == 1]
    det = np.einsum("ij,ij->i", np.cross(tets[:, 1] - tets[:, 0], tets[:, 2] - tets[:, 0]), tets[:, 3] - tets[:, 0])
    edge = np.linalg.norm(tets[:, 1] - tets[:, 0], axis=1)
    assert np.all(det > 1e-14 * edge**3)                 # positive, non-degenerate
    assert np.allclose(w.center[w.type == 1], tets.mean(axis=1))
    assert np.all(np.linalg.norm(tets, axis=2) <= 1.0 + 1e-12)
    cub = w.type == 0
    lo, hi = w.center[cub] - w.size[cub] / 2, w.center[cub] + w.size[cub] / 2
    assert lo[:, 0].min() >= 3.0 and hi[:, 0].max() <= 4.0 + 1e-12 and hi[:, 2].max() <= 0.25 + 1e-12
    assert set(np.unique(w.size[cub])) <= {1 / 16, 1 / 32, 1 / 64}
    # leaves do not overlap: total volume <= slab volume, and no two centres coincide
    assert w.vol[cub].sum() <= 0.25 + 1e-12
    assert len(np.unique(np.round(w.center[cub] * 1024).astype(np.int64), axis=0)) == cub.sum()


def test_octree_is_two_to_one_balanced():
    rng = W.rng_for(4, 1)
    c, s = W.octree_cuboids(rng, 3000)
    # face neighbours differ by at most a factor 2 in edge length: probe just across every face
    key = {tuple(np.round(ci * 128).astype(int)): si[0] for ci, si in zip(c, s)}
    cells = [(ci, si[0]) for ci, si in zip(c, s)]

    def size_at(p):
        for e in (1 / 64, 1 / 32, 1 / 16):
            cc = (np.floor(p / e) + 0.5) * e
            k = tuple(np.round(cc * 128).astype(int))
            if key.get(k) == e:
                return e
        return None

    for ci, e in cells[::7]:
        for ax in range(3):
            for sg in (-1, 1):
                p = ci.copy()
                p[ax] += sg * (e / 2 + 1 / 256)
                q = size_at(p)
                if q is not None:
                    assert 0.5 <= q / e <= 2.0


def test_sample_rows_and_leading_dim():
    r = W.sample_rows(5, 65536, 1024, extra=(0, 65535, 32768))
    assert r.dtype == np.int64 and len(r) >= 1024 and r[0] == 0 and r[-1] == 65535
    assert np.array_equal(r, W.sample_rows(5, 65536, 1024, extra=(0, 65535, 32768)))
    assert W.leading_dim(513, "f32") == 516 and W.leading_dim(513, "f64") == 514 and W.leading_dim(512, "f32") == 512


def test_morton_order_and_reorder():
    w = W.config3(4, batch=2)          # 4 x 4 x 4 cube with exchange neighbours
    perm = W.morton_order(w)
    assert np.array_equal(np.sort(perm), np.arange(w.n))
    # the first eight tiles along the curve are the 2 x 2 x 2 block at the origin, x fastest, then y, then z
    edge = w.size[0, 0]
    first = np.rint((w.center[perm[:8]] - w.center.min(axis=0)) / edge).astype(int)
    assert [tuple(c) for c in first] == [(0, 0, 0), (1, 0, 0), (0, 1, 0), (1, 1, 0), (0, 0, 1), (1, 0, 1), (0, 1, 1),
                                         (1, 1, 1)]
    r = W.reorder(w, perm)
    assert r.grid is None and np.array_equal(r.center, w.center[perm]) and np.array_equal(r.m, w.m[:, :, perm])
    # neighbour relation carried over: the neighbour of new tile k in direction d is the same physical tile
    for k in range(w.n):
        for d in range(6):
            j_old = w.nbr[perm[k], d]
            if j_old < 0:
                assert r.nbr[k, d] == -1
            else:
                assert np.array_equal(r.center[r.nbr[k, d]], w.center[j_old])
    # composing two reorderings records the composed permutation
    rr = W.reorder(r, np.arange(w.n)[::-1].copy())
    assert np.array_equal(rr.center, w.center[rr.extra["perm"]])


def test_fields_of_a_reordered_problem_are_the_permuted_fields(oracle):
    from tests import harness as H
    w = W.config3(3, batch=2)
    perm = W.morton_order(w)
    r = W.reorder(w, perm)
    N_w = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    N_r = oracle.assemble_rows(H.oracle_tiles(oracle, r), long_double=True)
    k_w, _ = oracle.llg_rhs(H.oracle_problem(oracle, w, N_w), w.m)
    k_r, _ = oracle.llg_rhs(H.oracle_problem(oracle, r, N_r), r.m)
    assert np.max(np.abs(k_r - k_w[:, :, perm])) <= 1e-13 * np.max(np.abs(k_w))


def test_sp2_and_sp3_shaped_seeds():
    """The report-only F4 workloads (PAPER.md:163-199 shapes): unit vectors, the stated tile counts and aspect
    ratios, Neumann neighbour tables; the flower seed points along z, the vortex seed circulates about x."""
    w = W.sp2_film(10.0)
    assert w.n == 6000 and w.grid == (100, 20, 3) and w.gamma == 0.0
    L = np.array(w.grid) * w.size[0]
    assert np.allclose(L, [50.0, 10.0, 1.0])          # L = 5 d, d, d / 10 in exchange lengths
    assert np.allclose(np.linalg.norm(w.m, axis=1), 1.0) and np.allclose(w.m[0, :, 0], 1 / np.sqrt(3))
    for kind in ("flower", "vortex"):
        c = W.sp3_cube(8, 8.5, kind)
        assert c.n == 512 and np.allclose(np.linalg.norm(c.m, axis=1), 1.0, atol=1e-14)
        assert np.allclose(c.size, 8.5 / 8) and c.c_an == 0.1 and tuple(c.easy) == (0.0, 0.0, 1.0)
    f, v = W.sp3_cube(8, 8.5, "flower"), W.sp3_cube(8, 8.5, "vortex")
    assert f.m[0, 2].min() > 0.9 and abs(f.m[0, 0].mean()) < 1e-12
    r = v.center / 8.5 - 0.5
    circ = (r[:, 1] * v.m[0, 2] - r[:, 2] * v.m[0, 1]).sum()   # x component of sum r x m: the circulation
    assert circ > 0.5 * np.sqrt(r[:, 1] ** 2 + r[:, 2] ** 2).sum() * 0.5
    with pytest.raises(ValueError):
        W.sp3_cube(4, 8.0, "onion")
