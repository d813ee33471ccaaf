"""Brute-force surface-charge quadrature: the definition the closed forms must reproduce.

Independent of oracle/ and of the CUDA path (numpy only).  A uniformly magnetised body is the
surface charge sigma = M.n on its faces ("assuming that the tile is uniformly
magnetized"), so
    H(r) = (1/4pi) sum_f (M.n_f) int_f (r - r')/|r - r'|^3 dS',      H = -N.M,
and column b of N is -H for M = e_b.  Faces are integrated with tensor Gauss-Legendre rules.
"""
import numpy as np


def _gl01(npts):
    x, w = np.polynomial.legendre.leggauss(npts)
    return 0.5 * (x + 1.0), 0.5 * w


def _face_integral_parallelogram(P0, e1, e2, r, npts):
    """int over {P0 + u e1 + v e2, u,v in [0,1]} of (r - r')/|r - r'|^3 dS'."""
    u, wu = _gl01(npts)
    U, V = np.meshgrid(u, u, indexing="ij")
    W = np.outer(wu, wu) * np.linalg.norm(np.cross(e1, e2))
    pts = P0[None, None, :] + U[..., None] * e1 + V[..., None] * e2
    d = r[None, None, :] - pts
    R3 = np.sum(d * d, axis=-1) ** 1.5
    return np.sum(W[..., None] * d / R3[..., None], axis=(0, 1))


def _face_integral_triangle(P0, P1, P2, r, npts):
    """Duffy map (u, v) -> P0 + u (P1 - P0) + u v (P2 - P1), Jacobian u * 2 * area."""
    u, wu = _gl01(npts)
    U, V = np.meshgrid(u, u, indexing="ij")
    area2 = np.linalg.norm(np.cross(P1 - P0, P2 - P0))
    W = np.outer(wu, wu) * U * area2
    pts = P0 + U[..., None] * (P1 - P0) + (U * V)[..., None] * (P2 - P1)
    d = r - pts
    R3 = np.sum(d * d, axis=-1) ** 1.5
    return np.sum(W[..., None] * d / R3[..., None], axis=(0, 1))


def cuboid_tensor_quadrature(center, size, r, npts=300):
    """3x3 N of an axis-aligned cuboid (full edge lengths `size`) at field point r."""
    center, size, r = (np.asarray(a, dtype=np.float64) for a in (center, size, r))
    h = 0.5 * size
    N = np.zeros((3, 3))
    for ax in range(3):
        a1, a2 = (ax + 1) % 3, (ax + 2) % 3
        for sgn in (+1.0, -1.0):
            n = np.zeros(3)
            n[ax] = sgn
            P0 = center - h
            P0 = P0.copy()
            P0[ax] = center[ax] + sgn * h[ax]
            e1 = np.zeros(3)
            e1[a1] = size[a1]
            e2 = np.zeros(3)
            e2[a2] = size[a2]
            I = _face_integral_parallelogram(P0, e1, e2, r, npts)
            # H = (1/4pi) (M.n) I  ->  N[:, b] = -(1/4pi) n_b I
            N += -np.outer(I, n) / (4.0 * np.pi)
    return N


def _triangle_integral_split(P0, P1, P2, r, npts):
    """Triangle integral; when the foot of r on the face plane lies inside the triangle, split at the
    foot point so that the Duffy-collapsed vertex sits where the integrand peaks."""
    n = np.cross(P1 - P0, P2 - P0)
    n /= np.linalg.norm(n)
    foot = r - np.dot(r - P0, n) * n
    T = np.array([P1 - P0, P2 - P0]).T
    lam, *_ = np.linalg.lstsq(T, foot - P0, rcond=None)
    b = np.array([1.0 - lam.sum(), lam[0], lam[1]])
    if np.all(b > 1e-12):
        tot = np.zeros(3)
        for A, B in ((P0, P1), (P1, P2), (P2, P0)):
            tot += _face_integral_triangle(foot, A, B, r, npts)
        return tot
    return _face_integral_triangle(P0, P1, P2, r, npts)


def tet_tensor_quadrature(verts, r, npts=300):
    """3x3 N of a tetrahedron (4, 3), any vertex order, at field point r."""
    v = np.asarray(verts, dtype=np.float64).reshape(4, 3)
    r = np.asarray(r, dtype=np.float64)
    cen = v.mean(axis=0)
    N = np.zeros((3, 3))
    for f in ((0, 1, 2), (0, 1, 3), (0, 2, 3), (1, 2, 3)):
        P0, P1, P2 = v[f[0]], v[f[1]], v[f[2]]
        n = np.cross(P1 - P0, P2 - P0)
        n /= np.linalg.norm(n)
        if np.dot(n, P0 - cen) < 0:  # make it outward
            n = -n
        I = _triangle_integral_split(P0, P1, P2, r, npts)
        N += -np.outer(I, n) / (4.0 * np.pi)
    return N


def six(N33):
    """(xx, xy, xz, yy, yz, zz) of a 3x3."""
    return np.array([N33[0, 0], N33[0, 1], N33[0, 2], N33[1, 1], N33[1, 2], N33[2, 2]])
