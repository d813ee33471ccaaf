"""-m gpu: RK4 with the tensor resident in shared memory (csrc/resident.cu, mt_set_resident_mode): one
cooperative launch per chunk of steps.  Checked against the per-stage launches (mode 1) and against the
CPU oracle's trajectory, with the tolerances of tests/test_gpu_small.py, on ragged sizes, both tensor
dtypes, batches, sampling and the stop test (Eq. 2); a problem that does not fit is refused
when the mode is 'required' and runs through the streaming kernels otherwise.
"""
import numpy as np
import pytest
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W
from tests import harness as H
from tests.test_gpu_small import run_gpu_integrate

pytestmark = pytest.mark.gpu


@pytest.fixture()
def ctx():
    c = B.mt_create(0)
    yield c
    c.close()


def setup(ctx, oracle, w, dtype):
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, dtype)
    assert status == 0
    return H.dev_problem(w, tiles, N, dtype, ld), tiles


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [(20, 5, 1), (7, 5, 3), (8, 8, 8)])
def test_resident_rk4_equals_staged_launches_and_oracle(ctx, oracle, grid, dtype):
    """Film physics (exchange + Zeeman) on 100 / 105 (odd n: ragged vectors, uneven rows per CTA) / 512
    tiles: same trajectory from the resident kernel, from the per-stage launches, and from the oracle."""
    nx, ny, nz = grid
    if nz == 1:
        w = W.config2(nx, ny, phase="dynamics")
    elif nx == ny == nz:
        w = W.config3(nx, batch=1, dtype=dtype)
    else:
        rng = np.random.default_rng(nx * ny * nz)
        edge = (1.0, 0.7, 1.3)
        w = W._cuboid_workload("ragged", nx, ny, nz, edge, 1.0, W.random_unit_states(rng, 1, nx * ny * nz),
                               nbr=W.grid_neighbours(nx, ny, nz), inv_d2=tuple(1.0 / e**2 for e in edge), c_ex=0.35,
                               c_an=0.2, easy=(0.0, 0.0, 1.0), H_a=(0.05, 0.02, -0.01), gamma=1.0, alpha_ll=0.3)
        w.Ms = rng.uniform(0.5, 2.0, size=w.n)
    film = nz == 1
    dt, steps, every = (1e-13, 200, 20) if film else (0.01, 160, 16)
    prob, _ = setup(ctx, oracle, w, dtype)
    kw = dict(method=B.MT_RK4, dt=dt, t_end=steps * dt, sample_every=every, sample_cap=32)
    out = {}
    for mode in (1, 2):
        B.mt_set_resident_mode(ctx, mode)
        l0 = B.mt_launch_count(ctx)
        out[mode] = run_gpu_integrate(ctx, prob, w.m[:1], 1, **kw)
        out[mode] += (B.mt_launch_count(ctx) - l0,)
    (m1, s1, r1, rc1, n1), (m2, s2, r2, rc2, n2) = out[1], out[2]
    assert rc1 == 0 and rc2 == 0
    assert r2["accepted"] == steps == r1["accepted"] and r2["rhs_calls"] == 4 * steps
    assert r2["n_samples"] == steps // every == r1["n_samples"]
    tol = 1e-11 if dtype == "f64" else 2e-5
    assert np.array_equal(s1[:, 0], s2[:, 0])
    assert np.max(np.abs(m2 - m1)) < tol and np.max(np.abs(s2 - s1)) < tol
    assert np.max(np.abs(np.linalg.norm(m2[0], axis=0) - 1.0)) < 1e-14
    # one launch per chunk of `every` steps + one per sample + the two initial stagings of M
    assert n2 == 2 + 2 * (steps // every) and n2 < n1 / 10
    if w.n <= 128:  # the oracle's trajectory (seconds at these sizes)
        N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
        m_ref, s_ref, _ = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.RK4, dt=dt,
                                           t_end=steps * dt, sample_every=every, sample_cap=32, weights=w.vol)
        otol = 1e-9 if dtype == "f64" else 1e-4
        assert np.max(np.abs(s2[:, 1:] - s_ref[:, 1:])) < otol
        assert np.max(np.abs(m2[0] - m_ref)) < otol * 10


def test_resident_rk4_batches_and_repeatability(ctx, oracle):
    """A batch of three states on the resident kernel: each state bit-identical to its own run, and two
    runs of the same problem bit-identical (fixed summation order)."""
    w = W.config3(5, batch=3)
    prob, _ = setup(ctx, oracle, w, "f32")
    B.mt_set_resident_mode(ctx, 2)
    kw = dict(method=B.MT_RK4, dt=0.01, t_end=0.5, sample_every=10, sample_cap=8)
    mb, sb, _, _ = run_gpu_integrate(ctx, prob, w.m, 3, **kw)
    mb2, sb2, _, _ = run_gpu_integrate(ctx, prob, w.m, 3, **kw)
    assert np.array_equal(mb, mb2) and np.array_equal(sb, sb2)
    for b in range(3):
        m1, s1, _, _ = run_gpu_integrate(ctx, prob, w.m[b:b + 1], 1, **kw)
        assert np.array_equal(m1[0], mb[b])
        assert np.array_equal(s1[:, 1:4], sb[:, 1 + 3 * b:4 + 3 * b])


def test_resident_rk4_stop_test_against_oracle(ctx, oracle):
    """The stop test inside a resident chunk: every step leaves the torque of its start state in its own
    word; the state returned is the one the oracle's per-step test stops at."""
    w = W.config3(4)
    prob, _ = setup(ctx, oracle, w, "f64")
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    op = H.oracle_problem(oracle, w, N_ref)
    _, _, r_probe = oracle.integrate(op, w.m[0], method=oracle.RK4, dt=0.02, t_end=4.0, torque_tol=1e-30)
    tol = 0.999 * r_probe["max_torque"]
    m_o, _, r_o = oracle.integrate(op, w.m[0], method=oracle.RK4, dt=0.02, t_end=400.0, torque_tol=tol)
    B.mt_set_resident_mode(ctx, 2)
    m, _, r, rc = run_gpu_integrate(ctx, prob, w.m[:1], 1, method=B.MT_RK4, dt=0.02, t_end=400.0, torque_tol=tol)
    assert rc == 0 and r["accepted"] == r_o["accepted"] and r["accepted"] % 64 not in (0, 63)
    assert abs(r["max_torque"] - r_o["max_torque"]) <= 1e-9 * tol and r["max_torque"] <= tol
    assert np.max(np.abs(m[0] - m_o)) < 1e-10


def test_resident_mode_required_refuses_what_does_not_fit(ctx, oracle):
    """40x40x1 = 1,600 tiles in fp64 is 123 MB: not resident.  Mode 2 refuses, mode 0 streams."""
    w = W.config2(40, 40, phase="dynamics")
    prob, _ = setup(ctx, oracle, w, "f64")
    kw = dict(method=B.MT_RK4, dt=1e-13, t_end=8e-13)
    B.mt_set_resident_mode(ctx, 2)
    _, _, _, rc = run_gpu_integrate(ctx, prob, w.m[:1], 1, allow=(B.MT_ERR_INVALID_ARG,), **kw)
    assert rc == B.MT_ERR_INVALID_ARG
    B.mt_set_resident_mode(ctx, 0)
    m, _, r, rc = run_gpu_integrate(ctx, prob, w.m[:1], 1, **kw)
    assert rc == 0 and r["accepted"] == 8 and np.isfinite(m).all()
    with pytest.raises(B.MtError):
        B.mt_set_resident_mode(ctx, 3)
