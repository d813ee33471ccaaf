"""Pins of the oracle's tensor assembly (O1) against what the mathematics fixes — none of these
re-types the oracle's closed forms: they are the surface-charge definition integrated by brute
force, textbook limits, invariants and 40-digit fixtures.  Pin numbers are SURVEY.md 8(c) P1-P11.
"""
import os

import numpy as np
import pytest

from tests import quadrature as Q

GOLD = os.path.join(os.path.dirname(__file__), "golden", "tensor_fixtures.txt")

UNIT_TET = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1]], dtype=np.float64)


def six(N33):
    return Q.six(N33)


def cuboid6(oracle, size, d, ld=True):
    return oracle.cuboid_block(0.5 * np.asarray(size, dtype=np.float64), d, long_double=ld)


# ---- P1 / P2 / P3 ---------------------------------------------------------------------------------
@pytest.mark.parametrize("size", [(1, 1, 1), (3.125, 3.125, 3.0), (1, 2, 5), (0.1, 7, 0.3)])
def test_p1_self_trace_is_one_cuboid(oracle, size):
    b = cuboid6(oracle, size, (0, 0, 0))
    assert abs(b[0] + b[3] + b[5] - 1.0) < 1e-15
    assert np.all(np.abs(b[[1, 2, 4]]) < 1e-16)


@pytest.mark.parametrize("d", [(1, 0, 0), (3, 2, 1), (0.7, -1.9, 0.2), (10, 7, 3)])
def test_p1_exterior_trace_is_zero(oracle, d):
    b = cuboid6(oracle, (1, 1.5, 0.5), d)
    assert abs(b[0] + b[3] + b[5]) < 1e-16


def test_p1_tet_trace(oracle):
    rng = np.random.default_rng(11)
    for _ in range(5):
        v = rng.normal(size=(4, 3))
        N = oracle.tet_block(v, v.mean(axis=0))
        assert abs(np.trace(N) - 1.0) < 1e-14
        N = oracle.tet_block(v, v.mean(axis=0) + np.array([4.0, -3.0, 2.5]))
        assert abs(np.trace(N)) < 1e-15


def test_p2_cube_self_is_third_identity(oracle):
    for edge in (1.0, 0.25, 3e-9):
        b = cuboid6(oracle, (edge,) * 3, (0, 0, 0))
        assert np.allclose(b, [1 / 3, 0, 0, 1 / 3, 0, 1 / 3], rtol=0, atol=2e-16)


def test_p3_self_block_closed_form(oracle):
    # N_xx(0) = (2/pi) atan( bc / (a sqrt(a^2+b^2+c^2)) ), half-edges a,b,c (cyclic) — the classical
    # demagnetizing factor of a prism at its centre.
    rng = np.random.default_rng(3)
    for _ in range(10):
        a, b, c = rng.uniform(0.1, 5.0, size=3)
        R = np.sqrt(a * a + b * b + c * c)
        exp = (2 / np.pi) * np.array([np.arctan(b * c / (a * R)), np.arctan(a * c / (b * R)),
                                      np.arctan(a * b / (c * R))])
        got = cuboid6(oracle, (2 * a, 2 * b, 2 * c), (0, 0, 0))
        assert np.allclose(got[[0, 3, 5]], exp, rtol=0, atol=3e-16)


# ---- P4: symmetry of the polyhedron form is not manifest ------------------------------------------
def test_p4_polyhedron_block_symmetric(oracle):
    rng = np.random.default_rng(4)
    for _ in range(20):
        v = rng.normal(size=(4, 3))
        r = rng.normal(size=3) * 3.0
        N = oracle.tet_block(v, r)
        assert np.max(np.abs(N - N.T)) < 1e-15 * max(1.0, np.max(np.abs(N)) / 1e-3)


# ---- P5: point-dipole far field --------------------------------------------------------------------
def dipole(V, r):
    r = np.asarray(r, dtype=np.float64)
    rn = np.linalg.norm(r)
    return -(V / (4 * np.pi)) * (3 * np.outer(r, r) / rn**5 - np.eye(3) / rn**3)


def test_p5_dipole_limit_cuboid(oracle):
    u = np.array([0.6, 0.48, 0.64])
    prev = None
    for rr, tol in ((5, 1e-3), (20, 5e-6), (80, 2e-8)):
        got = cuboid6(oracle, (1, 1, 1), rr * u)
        exp = six(dipole(1.0, rr * u))
        dev = np.max(np.abs(got - exp)) / np.max(np.abs(exp))
        assert dev < tol
        if prev is not None:
            assert dev < prev / 50  # ~ r^-4 convergence for a cube
        prev = dev


def test_p5_dipole_limit_generic_cuboid_and_tet(oracle):
    size = np.array([1.0, 2.0, 0.5])
    r = 60 * np.array([0.6, 0.48, 0.64])
    got = cuboid6(oracle, size, r)
    exp = six(dipole(size.prod(), r))
    assert np.max(np.abs(got - exp)) / np.max(np.abs(exp)) < 1e-3
    # tetrahedron: dipole at the centroid
    cen = UNIT_TET.mean(axis=0)
    rr = cen + 80 * np.array([0.6, 0.48, 0.64])
    got = six(oracle.tet_block(UNIT_TET, rr))
    exp = six(dipole(1.0 / 6.0, rr - cen))
    assert np.max(np.abs(got - exp)) / np.max(np.abs(exp)) < 3e-4


# ---- P6: brute-force surface-charge quadrature -----------------------------------------------------
@pytest.mark.parametrize("size,center,r", [
    ((1, 1, 1), (0, 0, 0), (1.3, 0.4, -0.9)),
    ((1, 1, 1), (0, 0, 0), (0.1, -0.2, 0.3)),          # interior, generic
    ((3.125, 3.125, 3.0), (1, 2, 3), (1, 2, 3)),        # interior, centre (self term)
    ((1, 2, 0.5), (0.5, -1, 2), (2.5, 1.5, 2.25)),
    ((0.25, 0.5, 1.0), (0, 0, 0), (0.25, 0.5, 0.0)),    # neighbour sharing an edge line
])
def test_p6_cuboid_vs_quadrature(oracle, size, center, r):
    got = cuboid6(oracle, size, np.asarray(r, float) - np.asarray(center, float))
    exp = six(Q.cuboid_tensor_quadrature(center, size, r, npts=400))
    assert np.max(np.abs(got - exp)) < 5e-13


def test_p6_eight_tile_field_vs_quadrature(oracle):
    """2x2x2 cuboid tiles with random M: the oracle's summed field at a tile centre equals the
    quadrature of all 48 charged faces (superposition)."""
    rng = np.random.default_rng(6)
    size = np.array([1.0, 0.8, 0.6])
    centers = np.array([[i, j, k] for k in range(2) for j in range(2) for i in range(2)], float) * size
    M = rng.normal(size=(8, 3))
    tiles = oracle.Tiles(type=np.zeros(8, np.int32), center=centers, size=np.tile(size, (8, 1)),
                         verts=np.zeros((8, 4, 3)), Ms=np.ones(8))
    N = oracle.assemble_rows(tiles)
    Hd = oracle.demag_field(N, np.ones(8), M.T.copy())
    for i in (0, 5):
        H = np.zeros(3)
        for j in range(8):
            H += -Q.cuboid_tensor_quadrature(centers[j], size, centers[i], npts=300) @ M[j]
        assert np.max(np.abs(Hd[:, i] - H)) < 1e-12


@pytest.mark.parametrize("r", [(2, 1.5, 1), (-0.3, 0.2, 0.9), (0.6, 0.6, 0.6), (0.4, -0.5, 0.1)])
def test_p6_tet_exterior_vs_quadrature(oracle, r):
    got = oracle.tet_block(UNIT_TET, r)
    exp = Q.tet_tensor_quadrature(UNIT_TET, r, npts=300)
    assert np.max(np.abs(got - exp)) < 5e-13


def test_p6_tet_interior_vs_quadrature(oracle):
    rng = np.random.default_rng(66)
    v = rng.normal(size=(4, 3))
    r = v.mean(axis=0)
    got = oracle.tet_block(v, r)
    exp = Q.tet_tensor_quadrature(v, r, npts=400)  # a sliver (volume 0.005): converged to ~1e-13
    assert np.max(np.abs(got - exp)) < 1e-11
    # any vertex order gives the same block
    got2 = oracle.tet_block(v[[2, 0, 3, 1]], r)
    assert np.max(np.abs(got - got2)) < 1e-15


# ---- P7: the polyhedron form applied to a box equals the cuboid form -------------------------------
def box_faces(center, size):
    c, h = np.asarray(center, float), 0.5 * np.asarray(size, float)
    x0, y0, z0 = c - h
    x1, y1, z1 = c + h
    return [
        [(x1, y0, z0), (x1, y1, z0), (x1, y1, z1), (x1, y0, z1)],   # +x
        [(x0, y0, z0), (x0, y0, z1), (x0, y1, z1), (x0, y1, z0)],   # -x
        [(x0, y1, z0), (x0, y1, z1), (x1, y1, z1), (x1, y1, z0)],   # +y
        [(x0, y0, z0), (x1, y0, z0), (x1, y0, z1), (x0, y0, z1)],   # -y
        [(x0, y0, z1), (x1, y0, z1), (x1, y1, z1), (x0, y1, z1)],   # +z
        [(x0, y0, z0), (x0, y1, z0), (x1, y1, z0), (x1, y0, z0)],   # -z
    ]


@pytest.mark.parametrize("r", [(1.7, 0.3, -0.4), (0.1, 0.05, -0.2), (6, 5, 4)])
def test_p7_polyhedron_equals_cuboid(oracle, r):
    size = (1.0, 0.6, 1.4)
    N = oracle.polyhedron_block(box_faces((0, 0, 0), size), r)
    assert np.max(np.abs(six(N) - cuboid6(oracle, size, r))) < 5e-15


# ---- P8: six Kuhn tetrahedra tile a cube -----------------------------------------------------------
def test_p8_kuhn_additivity(oracle):
    import itertools
    tets = []
    for perm in itertools.permutations(range(3)):
        v = [np.zeros(3)]
        for ax in perm:
            nxt = v[-1].copy()
            nxt[ax] = 1.0
            v.append(nxt)
        tets.append(np.array(v))
    for r in [(1.8, 0.7, -0.6), (0.31, 0.52, 0.77), (0.5, 0.5, 3.0)]:
        tot = sum(oracle.tet_block(t, r) for t in tets)
        exp = cuboid6(oracle, (1, 1, 1), np.asarray(r) - 0.5)
        assert np.max(np.abs(six(tot) - exp)) < 5e-15


# ---- P9: inversion and mirror symmetries ----------------------------------------------------------
def test_p9_inversion_and_mirror(oracle):
    size, d = (1.0, 1.5, 0.7), np.array([1.2, -0.8, 2.1])
    a = cuboid6(oracle, size, d)
    assert np.max(np.abs(a - cuboid6(oracle, size, -d))) < 1e-17
    b = cuboid6(oracle, size, d * np.array([-1, 1, 1]))
    flip = np.array([1, -1, -1, 1, 1, 1])
    assert np.max(np.abs(a * flip - b)) < 1e-17


# ---- P10: 40-digit fixtures ------------------------------------------------------------------------
def _fixtures():
    out = []
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        kind, geo, pt, vals = [s.strip() for s in line.split("|")]
        out.append((kind, np.array(geo.split(), float), np.array(pt.split(), float),
                    np.array(vals.split(), float)))
    return out


@pytest.mark.parametrize("fx", _fixtures(), ids=lambda f: f"{f[0]}-{'_'.join(map(str, f[2]))}")
def test_p10_fixtures(oracle, fx):
    kind, geo, pt, vals = fx
    if kind == "cuboid":
        got = cuboid6(oracle, geo, pt, ld=True)
        got_d = cuboid6(oracle, geo, pt, ld=False)
    else:
        got = six(oracle.tet_block(geo.reshape(4, 3), pt, long_double=True))
        got_d = six(oracle.tet_block(geo.reshape(4, 3), pt, long_double=False))
    scale = np.max(np.abs(vals))
    # long double: block-relative 1e-12 (SURVEY A.5 measured 2.8e-13 at r = 90 edges)
    assert np.max(np.abs(got - vals)) / scale < 1e-12
    # double: the cancellation PAPER.md:151 warns about grows ~ r^3; 2e-9 covers r = 90 edges
    tol = 2e-9 if np.linalg.norm(pt) > 50 else 1e-12
    assert np.max(np.abs(got_d - vals)) / scale < tol


# ---- P11: degenerate alignments (guard rules A.3) --------------------------------------------------
@pytest.mark.parametrize("r", [
    (0.5, 1.2, 0.1),      # in the plane of the +x face (X_s = 0), outside the face
    (0.5, 0.5, 2.0),      # on the extension of the edge line x = a, y = b
    (0.5, 1.5, 0.5),      # in two face planes at once
    (0.5, 0.5, 1.5),      # on the extension of an edge through a corner direction
    (0.5, -2.0, -0.5),
])
def test_p11_degenerate_alignments(oracle, r):
    size = (1.0, 1.0, 1.0)  # faces at +-0.5
    got = cuboid6(oracle, size, r)
    assert np.all(np.isfinite(got))
    exp = six(Q.cuboid_tensor_quadrature((0, 0, 0), size, r, npts=400))
    assert np.max(np.abs(got - exp)) < 5e-13
    got_d = cuboid6(oracle, size, r, ld=False)
    assert np.max(np.abs(got_d - exp)) < 5e-13


def test_p11_near_edge_line_is_stable(oracle):
    """1e-7 off an edge line the sign-split log must still be right (A.3: 'use the split always')."""
    size = (1.0, 1.0, 1.0)
    r = (0.5 + 1e-7, 0.5 - 1e-7, 2.0)
    got = cuboid6(oracle, size, r, ld=False)
    exp = six(Q.cuboid_tensor_quadrature((0, 0, 0), size, r, npts=400))
    assert np.max(np.abs(got - exp)) < 5e-13


# ---- O2: the field sum ------------------------------------------------------------------------------
def test_o2_demag_field_is_the_plain_sum(oracle):
    rng = np.random.default_rng(2)
    n = 7
    N = rng.normal(size=(6, n, n))
    Ms = rng.uniform(0.5, 2.0, size=n)
    m = rng.normal(size=(2, 3, n))
    Hd = oracle.demag_field(N, Ms, m)
    full = np.array([[N[0], N[1], N[2]], [N[1], N[3], N[4]], [N[2], N[4], N[5]]])  # [a][b][i][j]
    exp = -np.einsum("abij,sbj->sai", full, m * Ms)
    assert np.allclose(Hd, exp, rtol=0, atol=1e-13)


def test_uniformly_magnetised_cube_of_tiles(oracle):
    """4x4x4 unit tiles magnetised along z: by superposition the summed tensor row at any tile
    centre equals the tensor of the 4-edge cube at that point; at the centre-adjacent tiles it is
    checked against the big-cube closed form (and the mean demag factor is 1/3 by symmetry)."""
    n1 = 4
    idx = np.array([[i, j, k] for k in range(n1) for j in range(n1) for i in range(n1)], float)
    centers = idx + 0.5
    n = n1**3
    tiles = oracle.Tiles(type=np.zeros(n, np.int32), center=centers, size=np.ones((n, 3)),
                         verts=np.zeros((n, 4, 3)), Ms=np.ones(n))
    N = oracle.assemble_rows(tiles)
    rowsum = N.sum(axis=2)  # [6][n]
    for i in (0, 21, 42, 63):
        exp = cuboid6(oracle, (n1,) * 3, centers[i] - n1 / 2)
        assert np.max(np.abs(rowsum[:, i] - exp)) < 1e-14
    assert abs(rowsum[5].mean() - rowsum[0].mean()) < 1e-14


# ---- F3: the pair symmetry the half storage relies on ------------------------------------
def test_pair_symmetry_holds_on_congruent_grids_only(oracle):
    """N_ij = N_ji for congruent axis-aligned cuboids (block even in c_i - c_j, P9); it fails for
    cuboids of different sizes and for tetrahedra (Q2) — which is why F3 checks congruence."""
    import numpy as np
    c = np.array([[i + 0.5, j + 0.5, k + 0.5] for k in range(2) for j in range(3) for i in range(4)]) * [0.5, 0.7, 0.3]
    n = len(c)
    t = oracle.Tiles(type=np.zeros(n, np.int32), center=c, size=np.tile([0.5, 0.7, 0.3], (n, 1)),
                     verts=np.zeros((n, 4, 3)), Ms=np.ones(n))
    N = oracle.assemble_rows(t)
    assert np.max(np.abs(N - N.transpose(0, 2, 1))) < 1e-16
    size = np.tile([0.5, 0.7, 0.3], (n, 1))
    size[3] = [0.25, 0.35, 0.15]
    t2 = oracle.Tiles(type=np.zeros(n, np.int32), center=c, size=size, verts=np.zeros((n, 4, 3)), Ms=np.ones(n))
    N2 = oracle.assemble_rows(t2)
    assert np.max(np.abs(N2 - N2.transpose(0, 2, 1))) > 1e-3
