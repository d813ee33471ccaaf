"""ctypes front-end of the CPU oracle (oracle/mt_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the cpu_baseline /
``--impl reference`` legs of bench.py.  The product package never imports this module and this
module never imports the product package.  Argument marshalling only; all arithmetic is in the C++
translation unit, which cites the passages it follows (PAPER.md line + section / SURVEY appendix).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mt_oracle.cpp")
_LIB = os.path.join(_HERE, "libmt_oracle.so")
_lib = None

COMPONENTS = ("xx", "xy", "xz", "yy", "yz", "zz")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (plain -O2, OpenMP over independent rows only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [
        ("n", C.c_int64), ("N", C.c_void_p), ("nrows", C.c_int64), ("rows", C.c_void_p),
        ("Ms", C.c_void_p), ("nbr", C.c_void_p), ("inv_d2", C.c_double * 3),
        ("c_ex", C.c_void_p), ("c_ex_scalar", C.c_double),
        ("c_an", C.c_void_p), ("c_an_scalar", C.c_double),
        ("easy", C.c_void_p), ("easy_const", C.c_double * 3),
        ("H_a", C.c_void_p), ("H_a_const", C.c_double * 3),
        ("gamma", C.c_double), ("alpha_ll", C.c_double),
    ]


class _Opts(C.Structure):
    _fields_ = [
        ("method", C.c_int), ("dt", C.c_double), ("t_end", C.c_double), ("max_steps", C.c_int64),
        ("rtol", C.c_double), ("atol", C.c_double), ("torque_tol", C.c_double),
        ("renormalize", C.c_int), ("sample_every", C.c_int64), ("sample_dt", C.c_double),
    ]


class _Result(C.Structure):
    _fields_ = [
        ("accepted", C.c_int64), ("rejected", C.c_int64), ("rhs_calls", C.c_int64),
        ("n_samples", C.c_int64), ("t", C.c_double), ("dt_last", C.c_double),
        ("max_torque", C.c_double), ("status", C.c_int),
    ]


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.mto_max_threads.restype = C.c_int
        _lib.mto_energy.restype = C.c_double
        for name in ("mto_assemble_rows", "mto_demag_field", "mto_llg_rhs", "mto_integrate"):
            getattr(_lib, name).restype = C.c_int
    return _lib


def max_threads() -> int:
    return int(lib().mto_max_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def cuboid_block(half, d, long_double: bool = True) -> np.ndarray:
    """Six components (xx, xy, xz, yy, yz, zz) of a cuboid with half-edges `half` seen at offset d."""
    half, d, out = _f64(half), _f64(d), np.empty(6)
    lib().mto_cuboid_block(_p(half), _p(d), C.c_int(int(long_double)), _p(out))
    return out


def polyhedron_block(faces, r, long_double: bool = True) -> np.ndarray:
    """Full 3x3 block of a planar-faced polyhedron; `faces` = list of (nv, 3) arrays, CCW from outside."""
    nv = np.array([len(f) for f in faces], dtype=np.int32)
    fv = _f64(np.concatenate([np.asarray(f, dtype=np.float64).reshape(-1, 3) for f in faces], axis=0))
    r, out = _f64(r), np.empty(9)
    lib().mto_polyhedron_block(C.c_int(len(faces)), _p(nv), _p(fv), _p(r), C.c_int(int(long_double)), _p(out))
    return out.reshape(3, 3)


def tet_block(verts, r, long_double: bool = True) -> np.ndarray:
    """Full 3x3 block of a tetrahedron (4, 3) (any orientation) at field point r."""
    verts, r, out = _f64(verts).reshape(12), _f64(r), np.empty(9)
    lib().mto_tet_block(_p(verts), _p(r), C.c_int(int(long_double)), _p(out))
    return out.reshape(3, 3)


@dataclass
class Tiles:
    """Host-side tile list: type 0 = axis-aligned cuboid, 1 = tetrahedron."""
    type: np.ndarray
    center: np.ndarray
    size: np.ndarray
    verts: np.ndarray
    Ms: np.ndarray

    @property
    def n(self) -> int:
        return int(self.type.shape[0])


def assemble_rows(tiles: Tiles, rows=None, long_double: bool = True, nthreads: int = 0) -> np.ndarray:
    """Tensor rows out[6][nrows][n]; rows=None gives the full tensor."""
    n = tiles.n
    ty = np.ascontiguousarray(tiles.type, dtype=np.int32)
    ce, sz, ve = _f64(tiles.center), _f64(tiles.size), _f64(tiles.verts)
    if rows is None:
        rows_a, nrows = None, n
    else:
        rows_a = np.ascontiguousarray(rows, dtype=np.int64)
        nrows = int(rows_a.shape[0])
    out = np.empty((6, nrows, n), dtype=np.float64)
    rc = lib().mto_assemble_rows(C.c_int64(n), _p(ty), _p(ce), _p(sz), _p(ve), _p(rows_a),
                                 C.c_int64(nrows), C.c_int(int(long_double)), _p(out),
                                 C.c_int(nthreads or max_threads()))
    if rc != 0:
        raise RuntimeError(f"mto_assemble_rows failed: {rc}")
    return out


def demag_field(N: np.ndarray, Ms, m, nthreads: int = 0) -> np.ndarray:
    """Hd[b][3][nrows] = -sum_j N_rj Ms_j m_j for the held rows; m is [B][3][n] or [3][n]."""
    N = _f64(N)
    _, nrows, n = N.shape
    Ms, m = _f64(Ms), _f64(m)
    squeeze = m.ndim == 2
    mb = m.reshape(-1, 3, n)
    out = np.empty((mb.shape[0], 3, nrows))
    rc = lib().mto_demag_field(_p(N), C.c_int64(n), C.c_int64(nrows), _p(Ms), _p(mb),
                               C.c_int(mb.shape[0]), _p(out), C.c_int(nthreads or max_threads()))
    if rc != 0:
        raise RuntimeError(f"mto_demag_field failed: {rc}")
    return out[0] if squeeze else out


@dataclass
class Problem:
    """Everything the effective field / LL right-hand side needs (Eq. 1, 7, 12, 16, 17)."""
    n: int
    Ms: np.ndarray
    N: np.ndarray | None = None          # [6][nrows][n] fp64, or None (demag off)
    rows: np.ndarray | None = None       # target index of each held row (None: all rows)
    nbr: np.ndarray | None = None        # [n, 6] int32
    inv_d2: tuple = (0.0, 0.0, 0.0)
    c_ex: object = 0.0                   # scalar or [n]
    c_an: object = 0.0
    easy: object = (0.0, 0.0, 1.0)       # 3-vector or [n, 3]
    H_a: object = (0.0, 0.0, 0.0)
    gamma: float = 1.0
    alpha_ll: float = 0.0
    _keep: list = field(default_factory=list, repr=False)

    def _c(self) -> _Problem:
        s = _Problem()
        keep = self._keep = []

        def arr(a, dt):
            a = np.ascontiguousarray(a, dtype=dt)
            keep.append(a)
            return a.ctypes.data

        s.n = self.n
        s.Ms = arr(self.Ms, np.float64)
        if self.N is not None:
            s.N = arr(self.N, np.float64)
            s.nrows = self.N.shape[1]
        else:
            s.N = None
            s.nrows = self.n if self.rows is None else len(self.rows)
        s.rows = arr(self.rows, np.int64) if self.rows is not None else None
        s.nbr = arr(self.nbr, np.int32) if self.nbr is not None else None
        s.inv_d2 = (C.c_double * 3)(*self.inv_d2)
        for name in ("c_ex", "c_an"):
            v = getattr(self, name)
            if np.ndim(v) == 0:
                setattr(s, name, None)
                setattr(s, name + "_scalar", float(v))
            else:
                setattr(s, name, arr(v, np.float64))
        for name in ("easy", "H_a"):
            v = np.asarray(getattr(self, name), dtype=np.float64)
            if v.ndim == 1:
                setattr(s, name, None)
                setattr(s, name + "_const", (C.c_double * 3)(*v))
            else:
                setattr(s, name, arr(v, np.float64))
        s.gamma, s.alpha_ll = float(self.gamma), float(self.alpha_ll)
        return s


def llg_rhs(prob: Problem, m, want_heff: bool = False, nthreads: int = 0):
    """dmdt[b][3][nrows] (and H_eff, max torque per state) by Eq. 1 on H_eff of Eq. 17."""
    m = _f64(m)
    squeeze = m.ndim == 2
    mb = m.reshape(-1, 3, prob.n)
    cp = prob._c()
    B, nrows = mb.shape[0], int(cp.nrows)
    dmdt = np.empty((B, 3, nrows))
    heff = np.empty((B, 3, nrows)) if want_heff else None
    tq = np.empty(B)
    rc = lib().mto_llg_rhs(C.byref(cp), _p(mb), C.c_int(B), _p(dmdt), _p(heff), _p(tq),
                           C.c_int(nthreads or max_threads()))
    if rc != 0:
        raise RuntimeError(f"mto_llg_rhs failed: {rc}")
    if squeeze:
        dmdt, tq = dmdt[0], tq[0]
        heff = heff[0] if want_heff else None
    return (dmdt, heff, tq) if want_heff else (dmdt, tq)


RK4, DP45 = 0, 1


def integrate(prob: Problem, m0, *, method: int, dt: float, t_end: float, t0: float = 0.0,
              max_steps: int = 0, rtol: float = 1e-6, atol: float = 1e-8, torque_tol: float = 0.0,
              renormalize: bool = True, sample_every: int = 0, sample_dt: float = 0.0,
              sample_cap: int = 0, weights=None, nthreads: int = 0):
    """Integrate one state; returns (m_end [3][n], samples [k][4], result dict)."""
    m = _f64(m0).copy().reshape(3, prob.n)
    cp = prob._c()
    o = _Opts(method, dt, t_end, max_steps, rtol, atol, torque_tol, int(renormalize), sample_every, sample_dt)
    res = _Result()
    t = C.c_double(t0)
    samples = np.zeros((max(sample_cap, 1), 4))
    w = _f64(weights) if weights is not None else None
    rc = lib().mto_integrate(C.byref(cp), C.byref(o), _p(m), C.byref(t), _p(w), _p(samples),
                             C.c_int64(sample_cap), C.byref(res), C.c_int(nthreads or max_threads()))
    if rc != 0:
        raise RuntimeError(f"mto_integrate failed: {rc}")
    out = {k: getattr(res, k) for k, _ in _Result._fields_}
    return m, samples[: res.n_samples].copy(), out


def energy(prob: Problem, m, vol=None) -> float:
    m = _f64(m).reshape(3, prob.n)
    cp = prob._c()
    v = _f64(vol) if vol is not None else None
    return float(lib().mto_energy(C.byref(cp), _p(m), _p(v)))


def energy_terms(prob: Problem, m, vol=None) -> np.ndarray:
    """(E_demag, E_exch, E_anis, E_zeeman) of one state — Eq. 8, 11, 15, 6 through the fields."""
    m = _f64(m).reshape(3, prob.n)
    cp = prob._c()
    v = _f64(vol) if vol is not None else None
    out = np.empty(4)
    lib().mto_energy_terms(C.byref(cp), _p(m), _p(v), _p(out))
    return out


def field_sweep(prob: Problem, m0, fields, *, vol=None, **integrate_kw):
    """F4, the loop of the paper's hysteresis experiment ("the applied field is changed
    in steps ... for each field the system is relaxed"): for every applied field H_a in `fields`
    ([k][3]) in order, integrate from the previous end state over [0, t_end] with `integrate_kw`,
    then record <m> (volume weighted) and the four energy terms.  Returns (m_end, rows [k][3+4])."""
    import dataclasses
    m = _f64(m0).copy().reshape(3, prob.n)
    rows = []
    for Hk in np.asarray(fields, dtype=np.float64).reshape(-1, 3):
        pk = dataclasses.replace(prob, H_a=tuple(float(x) for x in Hk))
        m, _, _ = integrate(pk, m, weights=vol, **integrate_kw)
        w = np.ones(prob.n) if vol is None else _f64(vol)
        mean = (m * w).sum(axis=1) / w.sum()
        rows.append(np.concatenate([mean, energy_terms(pk, m, vol)]))
    return m, np.array(rows)


def dp45_tableau():
    c, a, b5, b4 = np.empty(7), np.empty(42), np.empty(7), np.empty(7)
    lib().mto_dp45_tableau(_p(c), _p(a), _p(b5), _p(b4))
    return c, a.reshape(7, 6), b5, b4
