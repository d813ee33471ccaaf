"""Pins of the oracle's energy terms and field-sweep loop (Eq. 4-16,
PAPER.md:163-181 hysteresis loop).  Closed forms and identities only; nothing here re-types the
oracle's loops.
"""
import numpy as np

from tests.test_oracle_dynamics import grid_nbr, grid_tiles, unit_m


def test_single_cube_demag_energy_is_ms2_v_over_6(oracle):
    """A uniformly magnetised cube has N = I/3 (P2): E_d = (1/2) Ms^2 V m.N.m = Ms^2 V / 6 (Eq. 8)."""
    edge, Ms = 2.0, 3.0
    tiles = oracle.Tiles(type=np.zeros(1, np.int32), center=np.zeros((1, 3)), size=np.full((1, 3), edge),
                         verts=np.zeros((1, 4, 3)), Ms=np.array([Ms]))
    N = oracle.assemble_rows(tiles)
    prob = oracle.Problem(n=1, Ms=np.array([Ms]), N=N)
    m = np.array([[0.6], [0.0], [0.8]])
    E = oracle.energy_terms(prob, m, vol=np.array([edge**3]))
    assert abs(E[0] - Ms**2 * edge**3 / 6.0) < 1e-13
    assert E[1] == 0.0 and E[2] == 0.0 and E[3] == 0.0


def test_anisotropy_and_zeeman_closed_forms(oracle):
    """E_anis = -(1/2) Ms V c_an (m.e)^2 (Eq. 15-16 up to the constant), E_z = -Ms V m.H_a (Eq. 6-7)."""
    rng = np.random.default_rng(4)
    n = 7
    m = unit_m(rng, n)
    Ms = rng.uniform(0.5, 2.0, n)
    vol = rng.uniform(0.1, 3.0, n)
    e = np.array([1.0, 2.0, -2.0]) / 3.0
    Ha = np.array([0.3, -0.1, 0.25])
    prob = oracle.Problem(n=n, Ms=Ms, c_an=0.7, easy=tuple(e), H_a=tuple(Ha))
    E = oracle.energy_terms(prob, m, vol=vol)
    assert abs(E[2] - np.sum(-0.5 * Ms * vol * 0.7 * (e @ m) ** 2)) < 1e-14
    assert abs(E[3] - np.sum(-Ms * vol * (Ha @ m))) < 1e-14
    assert E[0] == 0.0 and E[1] == 0.0


def test_exchange_energy_of_a_uniform_spiral(oracle):
    """Chain of n cells whose m turns by delta from cell to cell: every bond carries
    c_ex Ms V (1 - cos delta)/dx^2 (3-point stencil, Neumann ends: Eq. 11-12)."""
    n, dx, delta, cex, Ms, V = 12, 0.4, 0.17, 1.3, 0.9, 0.4**3
    phi = delta * np.arange(n)
    m = np.stack([np.cos(phi), np.sin(phi), np.zeros(n)])
    prob = oracle.Problem(n=n, Ms=np.full(n, Ms), nbr=grid_nbr(n, 1, 1), inv_d2=(1 / dx**2, 1 / dx**2, 1 / dx**2),
                          c_ex=cex)
    E = oracle.energy_terms(prob, m, vol=np.full(n, V))
    assert abs(E[1] - (n - 1) * cex * Ms * V * (1 - np.cos(delta)) / dx**2) < 1e-13


def test_terms_sum_to_the_total_whose_rate_is_pinned(oracle):
    """sum of the four terms == oracle.energy (whose time derivative P14 pins to -alpha |m x H|^2)."""
    rng = np.random.default_rng(15)
    nx, ny, nz, edge = 4, 3, 2, 0.5
    n = nx * ny * nz
    tiles = grid_tiles(oracle, nx, ny, nz, edge=(edge,) * 3)
    N = oracle.assemble_rows(tiles)
    prob = oracle.Problem(n=n, Ms=np.ones(n), N=N, nbr=grid_nbr(nx, ny, nz), inv_d2=(1 / edge**2,) * 3,
                          c_ex=1.0, c_an=0.1, easy=(0, 0, 1), H_a=(0.05, 0.0, 0.02))
    m = unit_m(rng, n)
    vol = np.full(n, edge**3)
    E = oracle.energy_terms(prob, m, vol=vol)
    assert abs(E.sum() - oracle.energy(prob, m, vol=vol)) < 1e-14
    # demagnetisation energy is positive semi-definite for a uniform grid (symmetric operator)
    assert E[0] > 0


def test_field_sweep_single_spin_closed_form(oracle):
    """One spin, fields along z one after the other, gamma = 0: m_z = tanh(alpha sum_k H_k T + atanh m_z0)
    (P13's closed form continued across field steps); the recorded Zeeman energy is -m_z H_k."""
    alpha, T = 0.8, 0.5
    fields = np.array([[0, 0, 0.4], [0, 0, -0.9], [0, 0, 0.3]])
    m0 = np.array([[np.sqrt(1 - 0.2**2)], [0.0], [0.2]])
    prob = oracle.Problem(n=1, Ms=np.ones(1), gamma=0.0, alpha_ll=alpha)
    m, rows = oracle.field_sweep(prob, m0, fields, method=oracle.RK4, dt=1e-3, t_end=T)
    u = np.arctanh(0.2) + alpha * T * np.cumsum(fields[:, 2])
    assert np.allclose(rows[:, 2], np.tanh(u), atol=1e-11)
    assert np.allclose(rows[:, 6], -np.tanh(u) * fields[:, 2], atol=1e-11)
    assert abs(m[2, 0] - np.tanh(u[-1])) < 1e-11
