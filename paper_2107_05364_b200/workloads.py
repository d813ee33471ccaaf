"""Seeded synthetic inputs for the five BASELINE.json configs (host side, numpy only).

This module holds NONE of the method's arithmetic: it only lays out tiles, neighbour tables,
material constants and random magnetisation states.  It is the one module that both the CUDA
path's harness (tests, bench.py) and the oracle's harness use, so that both sides see identical
inputs.  It imports neither `oracle/` nor the binding.

Recipes: seeds 20210705 + k for config k, numpy PCG64, sub-streams via spawn().
Configs 2 and 3 take shapes and parameters from the µmag standard problems 4 and 3 as the paper
ran them and stand in for them; no µmag solution data is used.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field

import numpy as np

SEED0 = 20210705
MU0 = 4.0e-7 * np.pi


@dataclass
class Workload:
    name: str
    type: np.ndarray            # [n] int32 (0 cuboid, 1 tetrahedron)
    center: np.ndarray          # [n, 3]
    size: np.ndarray            # [n, 3]
    verts: np.ndarray           # [n, 4, 3]
    Ms: np.ndarray              # [n]
    vol: np.ndarray             # [n]
    m: np.ndarray               # [B, 3, n] unit vectors
    nbr: np.ndarray | None = None
    inv_d2: tuple = (0.0, 0.0, 0.0)
    c_ex: float = 0.0
    c_an: float = 0.0
    easy: tuple = (0.0, 0.0, 1.0)
    H_a: tuple = (0.0, 0.0, 0.0)
    gamma: float = 1.0
    alpha_ll: float = 0.0
    dtype: str = "f32"
    grid: tuple | None = None
    extra: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.type.shape[0])


def rng_for(config: int, stream: int = 0) -> np.random.Generator:
    ss = np.random.SeedSequence(SEED0 + config)
    return np.random.default_rng(ss.spawn(stream + 1)[stream])


def random_unit_states(rng: np.random.Generator, batch: int, n: int) -> np.ndarray:
    """Normal then normalised (BASELINE.json 'seeded random unit m')."""
    m = rng.standard_normal(size=(batch, 3, n))
    return m / np.linalg.norm(m, axis=1, keepdims=True)


def cuboid_grid(nx: int, ny: int, nz: int, edge) -> tuple:
    """Centres ((i+1/2) dx, (j+1/2) dy, (k+1/2) dz), x fastest; returns (center, size)."""
    e = np.broadcast_to(np.asarray(edge, dtype=np.float64), (3,)).copy()
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    c = np.stack([(i.ravel() + 0.5) * e[0], (j.ravel() + 0.5) * e[1], (k.ravel() + 0.5) * e[2]], axis=1)
    return np.ascontiguousarray(c), np.tile(e, (nx * ny * nz, 1))


def grid_neighbours(nx: int, ny: int, nz: int) -> np.ndarray:
    """[n, 6] int32: -x, +x, -y, +y, -z, +z neighbour index, -1 outside (Neumann)."""
    idx = np.arange(nx * ny * nz, dtype=np.int32).reshape(nz, ny, nx)
    nbr = -np.ones((nz, ny, nx, 6), dtype=np.int32)
    nbr[:, :, 1:, 0] = idx[:, :, :-1]
    nbr[:, :, :-1, 1] = idx[:, :, 1:]
    nbr[:, 1:, :, 2] = idx[:, :-1, :]
    nbr[:, :-1, :, 3] = idx[:, 1:, :]
    nbr[1:, :, :, 4] = idx[:-1, :, :]
    nbr[:-1, :, :, 5] = idx[1:, :, :]
    return np.ascontiguousarray(nbr.reshape(-1, 6))


def _cuboid_workload(name, nx, ny, nz, edge, Ms, m, **kw) -> Workload:
    center, size = cuboid_grid(nx, ny, nz, edge)
    n = nx * ny * nz
    return Workload(name=name, type=np.zeros(n, np.int32), center=center, size=size,
                    verts=np.zeros((n, 4, 3)), Ms=np.full(n, float(Ms)), vol=size.prod(axis=1), m=m,
                    grid=(nx, ny, nz), **kw)


def config1(batch: int = 4) -> Workload:
    """512 unit cubes on 8x8x8, Ms = 1, gamma = 1, alpha = 0.1, no exchange; fp64 tensor."""
    rng = rng_for(1)
    return _cuboid_workload("config1_8x8x8", 8, 8, 8, 1.0, 1.0, random_unit_states(rng, batch, 512),
                            gamma=1.0, alpha_ll=0.1, dtype="f64")


def config2(nx: int = 160, ny: int = 40, batch: int = 1, phase: str = "dynamics") -> Workload:
    """Thin film nx x ny x 1 of (500/nx x 125/ny x 3) nm tiles (µmag SP4 shape).
    phase 'relax': H_a = 0, alpha_ll = gamma*1; 'dynamics': 25 mT at 170 deg, alpha_ll = gamma*0.02."""
    rng = rng_for(2)
    n = nx * ny
    edge = (500e-9 / nx, 125e-9 / ny, 3e-9)
    Ms, A, gamma = 8.0e5, 1.3e-11, 2.211e5
    g = rng.standard_normal(size=(batch, 3, n))
    m = np.full((batch, 3, n), 1.0 / np.sqrt(3.0)) + 0.01 * g
    m /= np.linalg.norm(m, axis=1, keepdims=True)
    if phase == "relax":
        H_a, alpha = (0.0, 0.0, 0.0), gamma * 1.0
    else:
        Hmag = 25e-3 / MU0
        ang = np.deg2rad(170.0)
        H_a, alpha = (Hmag * np.cos(ang), Hmag * np.sin(ang), 0.0), gamma * 0.02
    return _cuboid_workload(f"config2_{nx}x{ny}x1_{phase}", nx, ny, 1, edge, Ms, m,
                            nbr=grid_neighbours(nx, ny, 1), inv_d2=tuple(1.0 / np.asarray(edge) ** 2),
                            c_ex=2.0 * A / (MU0 * Ms), gamma=gamma, alpha_ll=alpha, H_a=H_a, dtype="f32",
                            extra={"dt": 1e-13, "relax_steps": 20000, "dynamics_steps": 10000})


def config3(n1: int = 32, batch: int = 1, dtype: str = "f32") -> Workload:
    """Cube of n1^3 tiles, edge 8/n1 exchange lengths (µmag SP3 shape),
    dimensionless units: Ms = 1, gamma = 1, c_ex = 1, K_u = 0.1 K_m along z, alpha = 0.5."""
    rng = rng_for(3)
    edge = 8.0 / n1
    n = n1**3
    return _cuboid_workload(f"config3_{n1}^3", n1, n1, n1, edge, 1.0, random_unit_states(rng, batch, n),
                            nbr=grid_neighbours(n1, n1, n1), inv_d2=(1.0 / edge**2,) * 3, c_ex=1.0, c_an=0.1,
                            easy=(0.0, 0.0, 1.0), gamma=1.0, alpha_ll=0.5, dtype=dtype,
                            extra={"rtol": 1e-6, "atol": 1e-8, "dt0": 1e-3, "torque_tol": 1e-5, "t_end": 200.0})


def sp3_cube(n1: int, L: float, kind: str) -> Workload:
    """µmag standard problem 3 shape as the paper ran it: a cube of side L exchange
    lengths, n1^3 tiles, K_u = 0.1 K_m along z, started in a `flower`-like state (m along z, tilted
    outwards/inwards with height) or a `vortex`-like state (m circulating about the x axis with an
    x core).  Only the seeds of the two relaxations; the states themselves come out of the integrator."""
    edge = L / n1
    n = n1**3
    center, _ = cuboid_grid(n1, n1, n1, edge)
    r = center / L - 0.5                      # in [-0.5, 0.5]^3
    m = np.zeros((1, 3, n))
    if kind == "flower":
        m[0, 0] = 0.4 * r[:, 0] * r[:, 2]
        m[0, 1] = 0.4 * r[:, 1] * r[:, 2]
        m[0, 2] = 1.0
    elif kind == "vortex":
        rho = np.sqrt(r[:, 1] ** 2 + r[:, 2] ** 2) + 1e-12
        core = np.exp(-(rho / 0.15) ** 2)
        m[0, 0] = core
        m[0, 1] = -r[:, 2] / rho * (1.0 - core)
        m[0, 2] = r[:, 1] / rho * (1.0 - core)
    else:
        raise ValueError(kind)
    m /= np.linalg.norm(m, axis=1, keepdims=True)
    return _cuboid_workload(f"sp3_{kind}_{n1}^3_L{L}", n1, n1, n1, edge, 1.0, m, nbr=grid_neighbours(n1, n1, n1),
                            inv_d2=(1.0 / edge**2,) * 3, c_ex=1.0, c_an=0.1, easy=(0.0, 0.0, 1.0), gamma=1.0,
                            alpha_ll=0.5, dtype="f64", extra={"rtol": 1e-6, "atol": 1e-8, "dt0": 1e-3})


def sp2_film(d_over_lex: float, nx: int = 100, ny: int = 20, nz: int = 3) -> Workload:
    """µmag standard problem 2 shape as the paper ran it: film of length L = 5 d, width
    d, thickness d/10 on 100 x 20 x 3 tiles, no anisotropy, gamma = 0 (only the steady state matters),
    dimensionless units (lengths in l_ex, fields in Ms); started saturated along [1, 1, 1]."""
    d = float(d_over_lex)
    edge = (5.0 * d / nx, d / ny, 0.1 * d / nz)
    n = nx * ny * nz
    m = np.full((1, 3, n), 1.0 / np.sqrt(3.0))
    return _cuboid_workload(f"sp2_d{d}", nx, ny, nz, edge, 1.0, m, nbr=grid_neighbours(nx, ny, nz),
                            inv_d2=tuple(1.0 / np.asarray(edge) ** 2), c_ex=1.0, gamma=0.0, alpha_ll=1.0, dtype="f32")


def config5(nx: int = 64, ny: int = 64, nz: int = 16, batch: int = 8) -> Workload:
    """64x64x16 unit cubes (65,536 tiles), Ms = 1, eight seeded random unit states; fp32 tensor."""
    rng = rng_for(5)
    return _cuboid_workload(f"config5_{nx}x{ny}x{nz}", nx, ny, nz, 1.0, 1.0,
                            random_unit_states(rng, batch, nx * ny * nz), gamma=1.0, alpha_ll=0.1, dtype="f32")


# ---- config 4: unstructured tetrahedra + 2:1-balanced octree of cuboids ----------------------------
def sphere_tets(rng: np.random.Generator, n_points: int = 4000, n_tets: int = 20000) -> np.ndarray:
    """Delaunay tetrahedralisation (Qhull) of uniform random points in the unit ball; the first
    n_tets simplices in the order returned, re-oriented to positive volume.  [n_tets, 4, 3]."""
    from scipy.spatial import Delaunay
    pts = np.empty((0, 3))
    while len(pts) < n_points:  # rejection sampling from the cube
        c = rng.uniform(-1.0, 1.0, size=(2 * n_points, 3))
        pts = np.concatenate([pts, c[np.sum(c * c, axis=1) <= 1.0]])
    pts = pts[:n_points]
    simp = Delaunay(pts).simplices
    if len(simp) < n_tets:
        raise ValueError(f"Delaunay returned only {len(simp)} tetrahedra")
    v = pts[simp[:n_tets]]
    det = np.einsum("ij,ij->i", np.cross(v[:, 1] - v[:, 0], v[:, 2] - v[:, 0]), v[:, 3] - v[:, 0])
    flip = det < 0
    v[flip] = v[flip][:, [0, 2, 1, 3]]
    return np.ascontiguousarray(v)


def octree_cuboids(rng: np.random.Generator, n_leaves: int = 16384, base=(16, 16, 4), max_level: int = 2) -> tuple:
    """2:1 face-balanced octree of a 1 x 1 x 0.25 slab: base cells of edge 1/16 (level 0), refined by
    seeded uniform picks among the refinable leaves down to edge 1/64 (level 2) until >= n_leaves leaves; Morton order; the
    first n_leaves are kept.  Returns (center [n,3], size [n,3])."""
    leaves = {(0, i, j, k) for i in range(base[0]) for j in range(base[1]) for k in range(base[2])}
    dims = np.asarray(base)

    def find_leaf(level, i, j, k):
        """The leaf covering cell (level, i, j, k), searching coarser levels."""
        for L in range(level, -1, -1):
            s = level - L
            key = (L, i >> s, j >> s, k >> s)
            if key in leaves:
                return key
        return None

    def split(key):
        L, i, j, k = key
        if key not in leaves or L >= max_level:
            return
        # 2:1 balance: a face neighbour coarser than this leaf must be split first
        for d in ((1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)):
            ni, nj, nk = i + d[0], j + d[1], k + d[2]
            lim = dims << L
            if not (0 <= ni < lim[0] and 0 <= nj < lim[1] and 0 <= nk < lim[2]):
                continue
            nb = find_leaf(L, ni, nj, nk)
            if nb is not None and nb[0] < L:
                split(nb)
        leaves.remove(key)
        for a in range(2):
            for b in range(2):
                for c in range(2):
                    leaves.add((L + 1, 2 * i + a, 2 * j + b, 2 * k + c))

    while len(leaves) < n_leaves:
        refinable = sorted(k for k in leaves if k[0] < max_level)  # sorted: set order is not seeded
        split(refinable[int(rng.integers(0, len(refinable)))])

    def morton(key):
        L, i, j, k = key
        s = max_level - L
        x, y, z = i << s, j << s, k << s
        code = 0
        for bit in range(10):
            code |= ((x >> bit) & 1) << (3 * bit) | ((y >> bit) & 1) << (3 * bit + 1) | ((z >> bit) & 1) << (3 * bit + 2)
        return (code, L)

    keys = sorted(leaves, key=morton)[:n_leaves]
    h0 = 1.0 / base[0]
    center = np.empty((len(keys), 3))
    size = np.empty((len(keys), 3))
    for q, (L, i, j, k) in enumerate(keys):
        e = h0 / (1 << L)
        center[q] = ((i + 0.5) * e, (j + 0.5) * e, (k + 0.5) * e)
        size[q] = e
    return center, size


def config4(n_tets: int = 20000, n_cub: int = 16384, n_points: int = 4000, batch: int = 1,
            body: str = "both") -> Workload:
    """Unstructured mix (Q15/Q16): tetrahedra first, then octree cuboids shifted by +3 x."""
    rng_t, rng_c, rng_m = rng_for(4, 0), rng_for(4, 1), rng_for(4, 2)
    parts_type, parts_center, parts_size, parts_verts, parts_vol = [], [], [], [], []
    if body in ("both", "tets") and n_tets > 0:
        v = sphere_tets(rng_t, n_points, n_tets)
        parts_type.append(np.ones(len(v), np.int32))
        parts_center.append(v.mean(axis=1))
        parts_size.append(np.zeros((len(v), 3)))
        parts_verts.append(v)
        det = np.einsum("ij,ij->i", np.cross(v[:, 1] - v[:, 0], v[:, 2] - v[:, 0]), v[:, 3] - v[:, 0])
        parts_vol.append(np.abs(det) / 6.0)
    if body in ("both", "cuboids") and n_cub > 0:
        c, s = octree_cuboids(rng_c, n_cub)
        c = c + np.array([3.0, 0.0, 0.0])
        parts_type.append(np.zeros(len(c), np.int32))
        parts_center.append(c)
        parts_size.append(s)
        parts_verts.append(np.zeros((len(c), 4, 3)))
        parts_vol.append(s.prod(axis=1))
    ty = np.concatenate(parts_type)
    n = len(ty)
    return Workload(name=f"config4_{body}_{n}", type=ty, center=np.ascontiguousarray(np.concatenate(parts_center)),
                    size=np.ascontiguousarray(np.concatenate(parts_size)),
                    verts=np.ascontiguousarray(np.concatenate(parts_verts)), Ms=np.ones(n),
                    vol=np.concatenate(parts_vol), m=random_unit_states(rng_m, batch, n), gamma=1.0,
                    alpha_ll=0.1, dtype="f32")


def sample_rows(config: int, n: int, count: int, extra=()) -> np.ndarray:
    """Seeded sample of target rows for sampled-row parity at sizes the oracle cannot finish."""
    rng = rng_for(config, 7)
    rows = set(int(r) for r in rng.choice(n, size=min(count, n), replace=False))
    rows.update(int(r) for r in extra if 0 <= int(r) < n)
    return np.array(sorted(rows), dtype=np.int64)


def leading_dim(n: int, dtype: str) -> int:
    """Row pitch in elements: rows 16-byte aligned (A3)."""
    v = 4 if dtype == "f32" else 2
    return (n + v - 1) // v * v


def reorder(w: Workload, perm: np.ndarray) -> Workload:
    """The same problem with tile k of the result = tile perm[k] of `w` (every per-tile array permuted,
    neighbour indices renumbered).  Tile order is free in the method (`PAPER.md:124`: a list of tiles);
    fields of the reordered problem are the permuted fields of the original."""
    perm = np.asarray(perm, dtype=np.int64)
    n = w.n
    assert perm.shape == (n,) and np.array_equal(np.sort(perm), np.arange(n))
    inv = np.empty(n, dtype=np.int64)
    inv[perm] = np.arange(n)
    nbr = None
    if w.nbr is not None:
        old = w.nbr[perm]
        nbr = np.where(old >= 0, inv[np.maximum(old, 0)], -1).astype(w.nbr.dtype)
    extra = dict(w.extra)
    extra["perm"] = perm if "perm" not in w.extra else w.extra["perm"][perm]
    return dataclasses.replace(
        w, name=w.name + " (reordered)", type=np.ascontiguousarray(w.type[perm]),
        center=np.ascontiguousarray(w.center[perm]), size=np.ascontiguousarray(w.size[perm]),
        verts=np.ascontiguousarray(w.verts[perm]), Ms=np.ascontiguousarray(w.Ms[perm]),
        vol=np.ascontiguousarray(w.vol[perm]), m=np.ascontiguousarray(w.m[:, :, perm]),
        nbr=None if nbr is None else np.ascontiguousarray(nbr), grid=None, extra=extra)


def morton_order(w: Workload, cell: float | None = None) -> np.ndarray:
    """Permutation that sorts the tiles along a Z-order (Morton) curve through their centres (cell =
    quantisation step, default the smallest tile edge).  Spatially close tiles get close indices, so the
    kept entries of a thresholded tensor row (the near field, `PAPER.md:243`) form longer contiguous
    column runs: the index-row kernel's gathers of M touch fewer lines."""
    cell = float(w.size.min()) if cell is None else float(cell)
    ijk = np.floor((w.center - w.center.min(axis=0)) / cell + 0.5).astype(np.uint64)
    assert int(ijk.max()) < (1 << 21)

    def spread(v):  # 21 bits -> every third bit
        v = v & np.uint64(0x1FFFFF)
        v = (v | (v << np.uint64(32))) & np.uint64(0x1F00000000FFFF)
        v = (v | (v << np.uint64(16))) & np.uint64(0x1F0000FF0000FF)
        v = (v | (v << np.uint64(8))) & np.uint64(0x100F00F00F00F00F)
        v = (v | (v << np.uint64(4))) & np.uint64(0x10C30C30C30C30C3)
        v = (v | (v << np.uint64(2))) & np.uint64(0x1249249249249249)
        return v

    code = spread(ijk[:, 0]) | (spread(ijk[:, 1]) << np.uint64(1)) | (spread(ijk[:, 2]) << np.uint64(2))
    return np.argsort(code, kind="stable").astype(np.int64)
