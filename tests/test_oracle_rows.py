"""Pins of the oracle's ROW paths — the functions the full-size GPU tests use as their checker:
`assemble_rows` with tetrahedron (type 1) tiles and mixed systems ("tetrahedra" §3),
`llg_rhs` on a `rows` subset (row bands of Eq. 1/9/17) and the volume-weighted
observable <m> ("average magnetization", reading Q17).  None of these re-types the
oracle: the expected values come from tests/quadrature.py (the surface-charge definition integrated
by brute force), from additivity of the field of a body cut into pieces, from a plain numpy
evaluation of the printed equations, and from hand values.

What they catch: a wrong 3x3 -> six-component pick in `tile_block` (e.g. o9[3] for yy), a wrong
`verts[12 j + k]` stride, target/source swapped for tetrahedra, a row subset read at the wrong index,
weights ignored or applied to the wrong tile.
"""
import itertools

import numpy as np

from tests import quadrature as Q


def _tiles(oracle, specs):
    """specs: list of ("cuboid", center, size) / ("tet", verts(4,3)); tetrahedron centre = centroid."""
    n = len(specs)
    ty = np.zeros(n, np.int32)
    ce, sz, ve = np.zeros((n, 3)), np.zeros((n, 3)), np.zeros((n, 4, 3))
    for k, s in enumerate(specs):
        if s[0] == "cuboid":
            ce[k], sz[k] = s[1], s[2]
        else:
            ty[k] = 1
            ve[k] = s[1]
            ce[k] = np.asarray(s[1], float).mean(axis=0)
    return oracle.Tiles(type=ty, center=ce, size=sz, verts=ve, Ms=np.ones(n))


def _generic_tets(seed, k, spread=2.5):
    """k well-separated generic tetrahedra (no symmetry: all six components of every block differ)."""
    rng = np.random.default_rng(seed)
    out = []
    for q in range(k):
        while True:
            v = rng.uniform(-0.5, 0.5, size=(4, 3))
            vol = abs(np.linalg.det(v[1:] - v[0])) / 6
            if vol > 0.02:
                break
        out.append(v + spread * np.array([q, 0.3 * q * q, -0.4 * q]))
    return out


def test_tetrahedron_rows_equal_surface_charge_quadrature(oracle):
    """Rows of a 3-tetrahedron system through `assemble_rows` (both precisions, full and `rows=`
    subset) against the brute-force quadrature of each source tetrahedron at each target centroid."""
    tets = _generic_tets(2107, 3)
    tiles = _tiles(oracle, [("tet", v) for v in tets])
    exp = np.empty((6, 3, 3))
    for i in range(3):
        for j in range(3):
            exp[:, i, j] = Q.six(Q.tet_tensor_quadrature(tets[j], tiles.center[i], npts=300))
    # sanity of the pin itself: a yy <-> yx mix-up must be visible (components are all distinct)
    assert np.min(np.abs(exp[3] - exp[1])) > 1e-6
    for ld in (True, False):
        N = oracle.assemble_rows(tiles, long_double=ld)
        assert N.shape == (6, 3, 3)
        off = ~np.eye(3, dtype=bool)
        assert np.max(np.abs(N - exp)[:, off]) < 5e-13          # exterior points
        assert np.max(np.abs(N - exp)[:, ~off]) < 2e-11         # own centroid (interior: slower quadrature)
        sub = oracle.assemble_rows(tiles, rows=[2, 0], long_double=ld)
        assert np.array_equal(sub, N[:, [2, 0], :])
    # self blocks: trace 1 (interior), exterior blocks traceless
    N = oracle.assemble_rows(tiles)
    tr = N[0] + N[3] + N[5]
    assert np.max(np.abs(tr - np.eye(3))) < 1e-14


def test_kuhn_cube_as_six_type1_tiles_sums_to_the_cuboid_row(oracle):
    """P8 through the row path: the unit cube cut into its six Kuhn tetrahedra, listed as six type-1
    tiles beside two cuboid tiles.  Field is additive over the pieces, so in every
    row the six tetrahedron columns sum to the block of the whole cube seen from that row's centre;
    the cuboid columns equal the quadrature of that cuboid."""
    tets = []
    for perm in itertools.permutations(range(3)):
        v = [np.zeros(3)]
        for ax in perm:
            nxt = v[-1].copy()
            nxt[ax] = 1.0
            v.append(nxt)
        tets.append(np.array(v))
    specs = [("tet", t) for t in tets]
    specs += [("cuboid", (2.3, 0.4, -0.9), (1.0, 0.5, 2.0)), ("cuboid", (-1.7, 1.1, 0.6), (0.7, 1.3, 0.4))]
    tiles = _tiles(oracle, specs)
    N = oracle.assemble_rows(tiles)
    assert N.shape == (6, 8, 8)
    for i in range(8):
        d = tiles.center[i] - 0.5
        cube = oracle.cuboid_block(np.array([0.5, 0.5, 0.5]), d)
        assert np.max(np.abs(N[:, i, :6].sum(axis=1) - cube)) < 1e-14, i
        # cross-check the expected value itself against the definition (interior points for i < 6)
        assert np.max(np.abs(cube - Q.six(Q.cuboid_tensor_quadrature((0.5,) * 3, (1, 1, 1), tiles.center[i],
                                                                     npts=400)))) < 5e-12
        for j in (6, 7):
            e = Q.six(Q.cuboid_tensor_quadrature(tiles.center[j], tiles.size[j], tiles.center[i], npts=400))
            assert np.max(np.abs(N[:, i, j] - e)) < 5e-13, (i, j)


def test_mixed_row_field_equals_quadrature_of_all_faces(oracle):
    """A mixed cuboid + tetrahedron system with random M: H_d at a cuboid centre and at a
    tetrahedron centroid = superposition of every tile's brute-force field."""
    rng = np.random.default_rng(5364)
    tets = _generic_tets(99, 2)
    specs = [("cuboid", (4.0, -1.0, 0.5), (1.0, 0.8, 0.6)), ("tet", tets[0]),
             ("cuboid", (-2.0, 2.0, 1.0), (0.5, 1.5, 1.0)), ("tet", tets[1])]
    tiles = _tiles(oracle, specs)
    n = tiles.n
    Ms = rng.uniform(0.5, 2.0, size=n)
    m = rng.normal(size=(3, n))
    N = oracle.assemble_rows(tiles)
    Hd = oracle.demag_field(N, Ms, m)
    for i in range(n):
        H = np.zeros(3)
        for j, s in enumerate(specs):
            if s[0] == "cuboid":
                Nq = Q.cuboid_tensor_quadrature(s[1], s[2], tiles.center[i], npts=400)
            else:
                Nq = Q.tet_tensor_quadrature(s[1], tiles.center[i], npts=400 if i == j else 300)
            H += -Nq @ (Ms[j] * m[:, j])
        assert np.max(np.abs(Hd[:, i] - H)) < 3e-11, i


def _numpy_rhs(N6, Ms, m, nbr, inv_d2, c_ex, c_an, easy, H_a, gamma, alpha):
    """Eq. 9, 12 (3-point stencil, Neumann ghost = self), 16, 17 and Eq. 1 written out in numpy."""
    full = np.array([[N6[0], N6[1], N6[2]], [N6[1], N6[3], N6[4]], [N6[2], N6[4], N6[5]]])
    H = -np.einsum("abij,bj->ai", full, m * Ms)
    n = m.shape[1]
    for i in range(n):
        for ax in range(3):
            for side in range(2):
                j = nbr[i, 2 * ax + side]
                mj = m[:, j] if j >= 0 else m[:, i]
                H[:, i] += c_ex * inv_d2[ax] * (mj - m[:, i])
        H[:, i] += c_an * np.dot(m[:, i], easy) * easy + H_a
    mxH = np.cross(m.T, H.T).T
    return -gamma * mxH - alpha * np.cross(m.T, mxH.T).T, H


def test_rhs_row_subset_equals_rows_of_the_full_call(oracle):
    """`llg_rhs` with held rows (N = those rows of the tensor, `rows` = their targets) returns
    exactly those rows of the full call, and both equal the printed equations in numpy."""
    rng = np.random.default_rng(31)
    nx, ny, nz = 4, 3, 2
    n = nx * ny * nz
    idx = np.array([[i, j, k] for k in range(nz) for j in range(ny) for i in range(nx)])
    size = np.array([0.5, 0.7, 0.3])
    nbr = -np.ones((n, 6), np.int32)
    lin = lambda i, j, k: (k * ny + j) * nx + i
    for q, (i, j, k) in enumerate(idx):
        if i > 0: nbr[q, 0] = lin(i - 1, j, k)
        if i < nx - 1: nbr[q, 1] = lin(i + 1, j, k)
        if j > 0: nbr[q, 2] = lin(i, j - 1, k)
        if j < ny - 1: nbr[q, 3] = lin(i, j + 1, k)
        if k > 0: nbr[q, 4] = lin(i, j, k - 1)
        if k < nz - 1: nbr[q, 5] = lin(i, j, k + 1)
    tiles = oracle.Tiles(type=np.zeros(n, np.int32), center=(idx + 0.5) * size, size=np.tile(size, (n, 1)),
                         verts=np.zeros((n, 4, 3)), Ms=rng.uniform(0.5, 1.5, size=n))
    N = oracle.assemble_rows(tiles)
    m = rng.normal(size=(3, n))
    m /= np.linalg.norm(m, axis=0)
    easy = np.array([0.6, 0.0, 0.8])
    kw = dict(n=n, Ms=tiles.Ms, nbr=nbr, inv_d2=tuple(1.0 / size**2), c_ex=0.37, c_an=0.21,
              easy=tuple(easy), H_a=(0.05, -0.02, 0.11), gamma=1.3, alpha_ll=0.4)
    full, heff, tq = oracle.llg_rhs(oracle.Problem(N=N, **kw), m, want_heff=True)
    exp, H = _numpy_rhs(N, tiles.Ms, m, nbr, 1.0 / size**2, 0.37, 0.21, easy, np.array(kw["H_a"]), 1.3, 0.4)
    assert np.max(np.abs(full - exp)) < 1e-13 and np.max(np.abs(heff - H)) < 1e-13
    assert abs(tq - np.max(np.linalg.norm(np.cross(m.T, H.T), axis=1))) < 1e-13
    rows = np.array([17, 3, 23, 0, 8], dtype=np.int64)
    sub, hsub, tqs = oracle.llg_rhs(oracle.Problem(N=N[:, rows, :].copy(), rows=rows, **kw), m, want_heff=True)
    assert sub.shape == (3, len(rows))
    assert np.array_equal(sub, full[:, rows]) and np.array_equal(hsub, heff[:, rows])
    assert abs(tqs - np.max(np.linalg.norm(np.cross(m.T[rows], H.T[rows]), axis=1))) < 1e-13


def test_weighted_mean_hand_value(oracle):
    """<m> with non-uniform weights (Q17): m = (x, y, z unit vectors), weights (1, 3, 4) ->
    (1/8, 3/8, 4/8); without weights (1/3, 1/3, 1/3).  gamma = alpha = 0 keeps m fixed, so every
    sample the integrator records is the mean of the start state."""
    n = 3
    m0 = np.eye(3)  # m[a][i]: tile i points along axis i
    prob = oracle.Problem(n=n, Ms=np.ones(n), N=None, gamma=0.0, alpha_ll=0.0, H_a=(0.3, 0.2, 0.1))
    for w, exp in ((np.array([1.0, 3.0, 4.0]), [0.125, 0.375, 0.5]), (None, [1 / 3] * 3)):
        _, s, res = oracle.integrate(prob, m0, method=oracle.RK4, dt=0.1, t_end=0.3, sample_every=1,
                                     sample_cap=8, weights=w)
        assert res["n_samples"] == 3
        assert np.allclose(s[:, 1:], exp, rtol=0, atol=1e-16)
        assert np.allclose(s[:, 0], [0.1, 0.2, 0.3], rtol=0, atol=1e-15)
        _, s, _ = oracle.integrate(prob, m0, method=oracle.DP45, dt=0.05, t_end=0.35, sample_dt=0.1,
                                   sample_cap=8, weights=w)
        assert np.allclose(s[:, 1:], exp, rtol=0, atol=1e-16) and len(s) == 3
