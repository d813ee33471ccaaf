"""Pins of the oracle's effective field, LL right-hand side and integrators (O3-O5):
SURVEY.md 8(c) P12-P16.  Closed forms, invariants and order conditions; no oracle formula is
re-typed here except Eq. 1 itself in vector form (numpy cross products) as the definition.
"""
from fractions import Fraction as F

import numpy as np
import pytest


def grid_nbr(nx, ny, nz):
    """-x,+x,-y,+y,-z,+z neighbour table, x fastest, -1 at the boundary."""
    idx = np.arange(nx * ny * nz).reshape(nz, ny, nx)
    nbr = -np.ones((nz, ny, nx, 6), dtype=np.int32)
    nbr[:, :, 1:, 0] = idx[:, :, :-1]
    nbr[:, :, :-1, 1] = idx[:, :, 1:]
    nbr[:, 1:, :, 2] = idx[:, :-1, :]
    nbr[:, :-1, :, 3] = idx[:, 1:, :]
    nbr[1:, :, :, 4] = idx[:-1, :, :]
    nbr[:-1, :, :, 5] = idx[1:, :, :]
    return nbr.reshape(-1, 6)


def grid_tiles(oracle, nx, ny, nz, edge=(1.0, 1.0, 1.0)):
    e = np.asarray(edge, float)
    c = np.array([[i + 0.5, j + 0.5, k + 0.5] for k in range(nz) for j in range(ny) for i in range(nx)]) * e
    n = len(c)
    return oracle.Tiles(type=np.zeros(n, np.int32), center=c, size=np.tile(e, (n, 1)),
                        verts=np.zeros((n, 4, 3)), Ms=np.ones(n))


def unit_m(rng, n):
    m = rng.normal(size=(3, n))
    return m / np.linalg.norm(m, axis=0)


# ---- Eq. 1 -----------------------------------------------------------------------------------------
def test_rhs_is_eq1_and_orthogonal_to_m(oracle):
    """P12: dm/dt = -gamma m x H - alpha m x (m x H) and m . dm/dt = 0."""
    rng = np.random.default_rng(12)
    n = 50
    m = unit_m(rng, n)
    Ha = rng.normal(size=(n, 3))
    prob = oracle.Problem(n=n, Ms=np.ones(n), H_a=Ha, gamma=1.7, alpha_ll=0.3)
    dmdt, heff, tq = oracle.llg_rhs(prob, m, want_heff=True)
    assert np.allclose(heff, Ha.T, atol=0)
    mxH = np.cross(m.T, Ha)
    exp = (-1.7 * mxH - 0.3 * np.cross(m.T, mxH)).T
    assert np.allclose(dmdt, exp, rtol=0, atol=1e-14)
    assert np.max(np.abs(np.sum(m * dmdt, axis=0))) < 1e-14
    assert abs(tq - np.max(np.linalg.norm(mxH, axis=1))) < 1e-14


# ---- P13: single spin in a constant field -----------------------------------------------------------
def single_spin(oracle, method, dt, T=2.0, gamma=1.3, alpha=0.7, H=0.9, **kw):
    prob = oracle.Problem(n=1, Ms=np.ones(1), H_a=(0.0, 0.0, H), gamma=gamma, alpha_ll=alpha)
    m0 = np.array([[1.0], [0.0], [0.0]])
    m, samples, res = oracle.integrate(prob, m0, method=method, dt=dt, t_end=T, renormalize=False, **kw)
    mz = np.tanh(alpha * H * T)
    phi = gamma * H * T
    exact = np.array([np.cos(phi) * np.sqrt(1 - mz**2), np.sin(phi) * np.sqrt(1 - mz**2), mz])
    return np.max(np.abs(m[:, 0] - exact)), res


def test_p13_single_spin_rk4_order(oracle):
    """m_z(t) = tanh(alpha H t), azimuth = +gamma H t: fixes the signs of both terms of Eq. 1."""
    e1, _ = single_spin(oracle, oracle.RK4, 0.1)
    e2, _ = single_spin(oracle, oracle.RK4, 0.05)
    assert e1 < 5e-6
    assert 12 < e1 / e2 < 20  # 4th order


def test_p13_single_spin_dp45_order(oracle):
    """One DP45 step of size h (tolerances huge so it is accepted as is): local error O(h^6)."""
    e1, r1 = single_spin(oracle, oracle.DP45, 0.1, T=0.1, rtol=1e9, atol=1e9)
    e2, r2 = single_spin(oracle, oracle.DP45, 0.05, T=0.05, rtol=1e9, atol=1e9)
    assert r1["rejected"] == 0 and r1["accepted"] == 1 and r1["rhs_calls"] == 7
    assert e1 < 1e-8
    assert 50 < e1 / e2 < 80  # 2^6 = 64


def test_p13_single_spin_dp45_adaptive(oracle):
    e, res = single_spin(oracle, oracle.DP45, 1e-3, rtol=1e-8, atol=1e-10)
    assert e < 1e-7
    assert res["accepted"] > 5 and abs(res["t"] - 2.0) == 0.0
    assert res["rhs_calls"] == 1 + 6 * (res["accepted"] + res["rejected"])


# ---- P12: |m| drift ---------------------------------------------------------------------------------
def test_p12_norm_drift_is_fifth_order(oracle):
    rng = np.random.default_rng(5)
    n = 27
    tiles = grid_tiles(oracle, 3, 3, 3)
    N = oracle.assemble_rows(tiles)
    m0 = unit_m(rng, n)
    prob = oracle.Problem(n=n, Ms=np.ones(n), N=N, gamma=1.0, alpha_ll=0.1)
    drift = []
    for dt in (0.2, 0.1):
        m, _, _ = oracle.integrate(prob, m0, method=oracle.RK4, dt=dt, t_end=dt, renormalize=False)
        drift.append(np.max(np.abs(np.linalg.norm(m, axis=0) - 1.0)))
    assert drift[0] < 1e-5
    assert drift[0] / drift[1] > 20  # O(dt^5)
    m, _, _ = oracle.integrate(prob, m0, method=oracle.RK4, dt=0.1, t_end=1.0, renormalize=True)
    assert np.max(np.abs(np.linalg.norm(m, axis=0) - 1.0)) < 1e-15


# ---- P15: exchange stencil ---------------------------------------------------------------------------
def test_p15_exchange_linear_and_cosine(oracle):
    nx, ny, nz = 32, 3, 1
    n = nx * ny * nz
    dx = 0.37
    nbr = grid_nbr(nx, ny, nz)
    x = (np.arange(n) % nx + 0.5) * dx
    prob = oracle.Problem(n=n, Ms=np.ones(n), nbr=nbr, inv_d2=(1 / dx**2, 1.0, 1.0), c_ex=2.5)
    # linear profile: zero in the interior; Neumann ghost = self gives +-slope/dx at the ends
    m = np.stack([3.0 * x, 0 * x + 1.0, -x])
    _, heff, _ = oracle.llg_rhs(prob, m, want_heff=True)
    interior = (np.arange(n) % nx > 0) & (np.arange(n) % nx < nx - 1)
    assert np.max(np.abs(heff[:, interior])) < 1e-10
    left = np.arange(n) % nx == 0
    assert np.allclose(heff[0, left], 2.5 * 3.0 * dx / dx**2)
    assert np.allclose(heff[2, ~interior & ~left], 2.5 * (+1.0) * dx / dx**2)
    assert np.max(np.abs(heff[1])) == 0.0  # single cell in z and constant in y contribute nothing
    # cos(kx) with kL = pi*j satisfies the Neumann condition: lap = -(2 - 2cos(k dx))/dx^2 cos(kx)
    k = np.pi * 3 / (nx * dx)
    m = np.stack([np.cos(k * x), 0 * x, 0 * x])
    _, heff, _ = oracle.llg_rhs(prob, m, want_heff=True)
    exp = -2.5 * (2 - 2 * np.cos(k * dx)) / dx**2 * np.cos(k * x)
    assert np.allclose(heff[0], exp, rtol=0, atol=1e-12)
    assert np.allclose(exp, -2.5 * k * k * np.cos(k * x), rtol=0, atol=2.5 * k**4 * dx**2 / 12 * 1.01)


def test_anisotropy_and_zeeman_fields(oracle):
    rng = np.random.default_rng(16)
    n = 9
    m = unit_m(rng, n)
    e = unit_m(rng, n).T.copy()
    can = rng.uniform(0.1, 1.0, n)
    prob = oracle.Problem(n=n, Ms=np.ones(n), c_an=can, easy=e, H_a=(0.1, -0.2, 0.3))
    _, heff, _ = oracle.llg_rhs(prob, m, want_heff=True)
    exp = (can * np.sum(m.T * e, axis=1))[:, None] * e + np.array([0.1, -0.2, 0.3])  # Eq. 16 + Eq. 7
    assert np.allclose(heff, exp.T, rtol=0, atol=1e-15)


# ---- P14: energy decreases under damping --------------------------------------------------------------
def test_p14_energy_monotone(oracle):
    rng = np.random.default_rng(14)
    nx = ny = nz = 4
    n = nx * ny * nz
    edge = 0.5
    tiles = grid_tiles(oracle, nx, ny, nz, edge=(edge,) * 3)
    N = oracle.assemble_rows(tiles)
    prob = oracle.Problem(n=n, Ms=np.ones(n), N=N, nbr=grid_nbr(nx, ny, nz), inv_d2=(1 / edge**2,) * 3,
                          c_ex=1.0, c_an=0.1, easy=(0, 0, 1), H_a=(0.05, 0.0, 0.02), gamma=1.0, alpha_ll=0.5)
    m = unit_m(rng, n)
    E = [oracle.energy(prob, m)]
    t = 0.0
    for _ in range(15):
        m, _, res = oracle.integrate(prob, m, method=oracle.RK4, dt=0.01, t_end=t + 0.05, t0=t)
        t = res["t"]
        E.append(oracle.energy(prob, m))
    assert np.all(np.diff(E) < 0)
    # and dE/dt = -alpha * sum |m x H|^2 * Ms V at the start (Eq. 5 + Eq. 1), to first order
    m = unit_m(np.random.default_rng(14), n)
    _, heff, _ = oracle.llg_rhs(prob, m, want_heff=True)
    rate = -0.5 * np.sum(np.linalg.norm(np.cross(m.T, heff.T), axis=1) ** 2)
    m1, _, _ = oracle.integrate(prob, m, method=oracle.RK4, dt=1e-4, t_end=1e-4)
    assert abs((oracle.energy(prob, m1) - oracle.energy(prob, m)) / 1e-4 - rate) < 2e-3 * abs(rate)


# ---- P16: Dormand-Prince order conditions, exact rational arithmetic ----------------------------------
def test_p16_dp45_tableau_order_conditions(oracle):
    c, a, b5, b4 = oracle.dp45_tableau()
    fr = lambda x: F(x).limit_denominator(10**7)
    c, b5, b4 = [fr(x) for x in c], [fr(x) for x in b5], [fr(x) for x in b4]
    a = [[fr(x) for x in row] for row in a]
    # the limit_denominator round trip reproduces the doubles exactly
    assert all(float(x) == y for x, y in zip(b5, oracle.dp45_tableau()[2]))
    for s in range(7):
        assert sum(a[s]) == c[s]
    assert [a[6][j] for j in range(6)] == b5[:6]  # FSAL: a7 = b5
    for b, order in ((b5, 5), (b4, 4)):
        for k in range(order):
            assert sum(bi * ci**k for bi, ci in zip(b, c)) == F(1, k + 1)
        A = [[a[s][j] if j < 6 else F(0) for j in range(7)] for s in range(7)]
        Ac = [sum(A[s][j] * c[j] for j in range(7)) for s in range(7)]
        Ac2 = [sum(A[s][j] * c[j] ** 2 for j in range(7)) for s in range(7)]
        AAc = [sum(A[s][j] * Ac[j] for j in range(7)) for s in range(7)]
        assert sum(b[s] * Ac[s] for s in range(7)) == F(1, 6)             # order 3
        assert sum(b[s] * c[s] * Ac[s] for s in range(7)) == F(1, 8)      # order 4
        assert sum(b[s] * Ac2[s] for s in range(7)) == F(1, 12)
        assert sum(b[s] * AAc[s] for s in range(7)) == F(1, 24)
    # b5 is really 5th order, b4 is not: one 5th-order condition separates them
    assert sum(bi * ci**4 for bi, ci in zip(b5, c)) == F(1, 5)
    assert sum(bi * ci**4 for bi, ci in zip(b4, c)) != F(1, 5)


def test_dp45_sampling_lands_on_sample_times(oracle):
    prob = oracle.Problem(n=1, Ms=np.ones(1), H_a=(0.0, 0.0, 1.0), gamma=1.0, alpha_ll=0.5)
    m0 = np.array([[1.0], [0.0], [0.0]])
    m, samples, res = oracle.integrate(prob, m0, method=oracle.DP45, dt=1e-3, t_end=1.0, rtol=1e-7,
                                       atol=1e-9, renormalize=True, sample_dt=0.25, sample_cap=8)
    assert np.array_equal(samples[:, 0], [0.25, 0.5, 0.75, 1.0])
    assert np.allclose(samples[:, 3], np.tanh(0.5 * samples[:, 0]), atol=1e-6)
    assert res["status"] == 0 and res["t"] == 1.0


def test_torque_stop(oracle):
    prob = oracle.Problem(n=1, Ms=np.ones(1), H_a=(0.0, 0.0, 1.0), gamma=0.0, alpha_ll=1.0)
    m0 = np.array([[1.0], [0.0], [0.0]])
    m, _, res = oracle.integrate(prob, m0, method=oracle.DP45, dt=1e-2, t_end=100.0, rtol=1e-6,
                                 atol=1e-8, torque_tol=1e-5)
    assert res["max_torque"] <= 1e-5 and res["t"] < 100.0
    # |m x H| = sech(t): the stop time is acosh(1e5) up to one step
    assert abs(res["t"] - np.arccosh(1e5)) < 2.0


# ---- readings Q10c / Q11b: behaviour at the edge of the domain --------------------------
def test_dp45_nonfinite_state_ends_the_run_and_zero_m_stays_zero(oracle):
    """A NaN in the state reaches the error estimate (it is not dropped by a max) and ends the run
    with the step-underflow status instead of being 'accepted' with err = 0; a zero-length m_i is a
    fixed point (no 0/0 on renormalisation)."""
    n = 3
    prob = oracle.Problem(n=n, Ms=np.ones(n), N=None, gamma=1.0, alpha_ll=0.5, H_a=(0.0, 0.0, 1.0))
    m0 = np.array([[1.0, 0.0, 0.6], [0.0, 1.0, 0.0], [0.0, 0.0, 0.8]])
    bad = m0.copy()
    bad[1, 2] = np.nan
    _, _, res = oracle.integrate(prob, bad, method=oracle.DP45, dt=1e-2, t_end=1.0, max_steps=50)
    assert res["status"] == -4 and res["accepted"] == 0
    zero = m0.copy()
    zero[:, 1] = 0.0
    for method in (oracle.RK4, oracle.DP45):
        m, _, res = oracle.integrate(prob, zero, method=method, dt=1e-2, t_end=0.5)
        assert res["status"] == 0 and np.all(m[:, 1] == 0.0) and np.all(np.isfinite(m))
        assert np.allclose(np.linalg.norm(m[:, [0, 2]], axis=0), 1.0, atol=1e-14)
