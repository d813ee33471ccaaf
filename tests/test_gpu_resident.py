"""-m gpu: RK4 and DP45 with the tensor resident in shared memory (csrc/resident.cu, mt_set_resident_mode): one
cooperative launch per chunk of steps / per 64 attempted steps.  Checked against the per-stage launches (mode 1) and against the
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


def test_resident_dp45_equals_host_controller_and_oracle(oracle):
    """DP45 inside the resident kernel (controller of dp_control.cuh run by every CTA on its own copy of the
    state) against the host controller with per-stage launches and against the oracle, on an 8^3 replica of
    config 3 with two states: same accept / reject sequence, same sample times, states and samples to
    rounding; stops by the torque test, by t_end and by max_steps; sample rows capped by sample_cap."""
    w = W.config3(8, batch=2)
    x = w.extra
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    runs = {}
    for key, (ctl, resident) in {"host": (1, 1), "resident": (0, 2)}.items():
        c = B.mt_create(0)
        B.mt_set_step_control(c, ctl)
        B.mt_set_resident_mode(c, resident)
        tiles = H.dev_tiles(w)
        N, ld, _ = H.assemble(c, tiles, "f64")
        prob = H.dev_problem(w, tiles, N, "f64", ld)
        out = []
        for kw in (dict(t_end=2.0, sample_dt=0.25, sample_cap=16),
                   dict(t_end=40.0, sample_dt=1.0, sample_cap=5, torque_tol=0.5),
                   dict(t_end=2.0, max_steps=37, allow=(B.MT_ERR_MAX_STEPS,))):
            l0 = B.mt_launch_count(c)
            out.append(run_gpu_integrate(c, prob, w.m, 2, method=B.MT_DP45, dt=x["dt0"], rtol=x["rtol"], atol=x["atol"], **kw)
                       + (B.mt_launch_count(c) - l0,))
        runs[key] = out
        c.close()
    for (m1, s1, r1, rc1, n1), (m2, s2, r2, rc2, n2) in zip(runs["host"], runs["resident"]):
        assert rc1 == rc2
        for key in ("accepted", "rejected", "rhs_calls", "n_samples"):
            assert r1[key] == r2[key], key
        # (another summation order in H_d: the error estimate, a difference of nearly equal slopes, moves in its
        # ~10th digit and the step sizes with it: a run that ends on a step count ends at t equal to ~1e-10)
        assert abs(r1["t"] - r2["t"]) <= 1e-9 and abs(r1["dt_last"] - r2["dt_last"]) <= 1e-6 * r1["dt_last"]
        assert abs(r1["max_torque"] - r2["max_torque"]) <= 1e-6 * r1["max_torque"]
        assert np.array_equal(s1[:, 0], s2[:, 0]) and (s1.size == 0 or np.max(np.abs(s1 - s2)) < 1e-9)
        assert np.max(np.abs(m1 - m2)) < 1e-9
        # stagings + k1 + one launch per 64 attempts, against ~8 launches per attempt
        assert n2 <= 3 + (r2["accepted"] + r2["rejected"]) // 64 + 1 and n2 < n1 / 20
    (_, s, r, _, _), (_, s_t, r_t, _, _), (_, _, r_m, rc_m, _) = runs["resident"]
    assert r["t"] == 2.0 and r["rejected"] > 0 and np.array_equal(s[:, 0], 0.25 * np.arange(1, 9))
    assert r_t["max_torque"] <= 0.5 and 5.0 < r_t["t"] < 40.0 and r_t["n_samples"] == 5
    assert rc_m == B.MT_ERR_MAX_STEPS and r_m["accepted"] + r_m["rejected"] == 37
    # a single state against the oracle's own step sequence
    m_o, s_o, r_o = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.DP45, dt=x["dt0"],
                                     rtol=x["rtol"], atol=x["atol"], t_end=2.0, sample_dt=0.25, sample_cap=16, weights=w.vol)
    c = B.mt_create(0)
    B.mt_set_resident_mode(c, 2)
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(c, tiles, "f64")
    m, s, r, _ = run_gpu_integrate(c, H.dev_problem(w, tiles, N, "f64", ld), w.m[:1], 1, method=B.MT_DP45, dt=x["dt0"],
                                   rtol=x["rtol"], atol=x["atol"], t_end=2.0, sample_dt=0.25, sample_cap=16)
    c.close()
    assert (r["accepted"], r["rejected"]) == (r_o["accepted"], r_o["rejected"])
    assert np.array_equal(s[:, 0], s_o[:, 0]) and np.max(np.abs(s[:, 1:] - s_o[:, 1:])) < 1e-9
    assert np.max(np.abs(m[0] - m_o)) < 1e-8


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_resident_dp45_small_cube_against_oracle(ctx, oracle, dtype):
    """Config-3 physics on a 6^3 cube (216 tiles: two rows per CTA on 108 CTAs): DP45 to t = 3 on the resident
    kernel, the assertions of test_dp45_trajectory_small_cube; then continued in a second call (k1 = f(m) is
    re-evaluated by the caller, the controller state starts afresh)."""
    w = W.config3(6)
    prob, _ = setup(ctx, oracle, w, dtype)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    kw = dict(dt=1e-3, t_end=3.0, rtol=1e-6, atol=1e-8, sample_dt=0.25)
    m_ref, s_ref, r_ref = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.DP45,
                                           sample_cap=64, weights=w.vol, **kw)
    B.mt_set_resident_mode(ctx, 2)
    m, s, res, _ = run_gpu_integrate(ctx, prob, w.m, 1, method=B.MT_DP45, sample_cap=64, **kw)
    assert res["n_samples"] == 12 == r_ref["n_samples"] and res["t"] == 3.0
    assert np.array_equal(s[:, 0], s_ref[:, 0])
    assert np.max(np.abs(s[:, 1:] - s_ref[:, 1:])) < 1e-3
    if dtype == "f64":
        assert res["accepted"] == r_ref["accepted"] and res["rejected"] == r_ref["rejected"]
        assert np.max(np.abs(m[0] - m_ref)) < 1e-8
    assert res["rhs_calls"] == 1 + 6 * (res["accepted"] + res["rejected"])
    assert np.max(np.abs(np.linalg.norm(m[0], axis=0) - 1.0)) < 1e-14


def test_resident_dp45_nonfinite_state_is_an_error(ctx, oracle):
    """A NaN in the state reaches the error estimate inside the kernel: MT_ERR_STEP_UNDERFLOW (Q11b)."""
    w = W.config3(4)
    prob, _ = setup(ctx, oracle, w, "f64")
    B.mt_set_resident_mode(ctx, 2)
    m0 = w.m[:1].copy()
    m0[0, 1, 7] = np.nan
    _, _, r, rc = run_gpu_integrate(ctx, prob, m0, 1, method=B.MT_DP45, dt=1e-3, t_end=1.0,
                                    allow=(B.MT_ERR_STEP_UNDERFLOW,))
    assert rc == B.MT_ERR_STEP_UNDERFLOW and r["accepted"] == 0


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("grid", [(1, 1, 1), (3, 1, 1), (2, 2, 1)])
def test_resident_tiny_problems_with_padded_rows(ctx, oracle, grid, dtype):
    """One to four tiles (one CTA row each, vectors mostly padding) on a tensor with extra row padding filled
    with NaN beyond column n: both integrators equal the per-stage launches."""
    nx, ny, nz = grid
    n = nx * ny * nz
    rng = np.random.default_rng(10 + n)
    edge = (1.0, 0.8, 1.2)
    w = W._cuboid_workload("tiny", nx, ny, nz, edge, 1.0, W.random_unit_states(rng, 2, n),
                           nbr=W.grid_neighbours(nx, ny, nz), inv_d2=tuple(1.0 / e**2 for e in edge), c_ex=0.2,
                           c_an=0.3, easy=(0.0, 0.6, 0.8), H_a=(0.1, 0.0, 0.05), gamma=1.0, alpha_ll=0.4)
    tiles = H.dev_tiles(w)
    ld = W.leading_dim(n, dtype) + 8
    N, ld, status = H.assemble(ctx, tiles, dtype, ld=ld)
    assert status == 0
    N[:, :, n:] = float("nan")  # what lies beyond column n must never be used
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    tol = 1e-11 if dtype == "f64" else 2e-5
    for kw in (dict(method=B.MT_RK4, dt=0.01, t_end=1.0, sample_every=25, sample_cap=8),
               dict(method=B.MT_DP45, dt=1e-3, t_end=1.0, rtol=1e-7, atol=1e-9, sample_dt=0.25, sample_cap=8)):
        out = {}
        for mode in (1, 2):
            B.mt_set_resident_mode(ctx, mode)
            out[mode] = run_gpu_integrate(ctx, prob, w.m, 2, **kw)
        (m1, s1, r1, _), (m2, s2, r2, _) = out[1], out[2]
        assert np.isfinite(m2).all() and r1["n_samples"] == r2["n_samples"] == 4
        assert (r1["accepted"], r1["rejected"]) == (r2["accepted"], r2["rejected"])
        assert np.max(np.abs(m2 - m1)) < tol and np.max(np.abs(s2 - s1)) < tol


@pytest.mark.parametrize("grid,dtype,batch", [((40, 30, 1), "f32", 1), ((30, 30, 1), "f64", 2), ((11, 11, 11), "f32", 3)])
def test_l2_streamed_persistent_kernel_equals_staged_launches(ctx, oracle, grid, dtype, batch):
    """Tensors too large for shared memory but at most 100 MB (1,200 / 1,331 tiles fp32, 900 tiles fp64) run the same
    persistent kernels with the rows read from L2 at every stage: RK4 and DP45 against the per-stage launches, with
    NaN in the row padding, odd n (1,331: ragged last vector) and batches."""
    nx, ny, nz = grid
    w = W.config2(nx, ny, batch=batch, phase="dynamics") if nz == 1 else W.config3(nx, batch=batch, dtype=dtype)
    n = w.n
    tiles = H.dev_tiles(w)
    ld = W.leading_dim(n, dtype) + 4
    N, ld, status = H.assemble(ctx, tiles, dtype, ld=ld)
    assert status == 0
    N[:, :, n:] = float("nan")
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    film = nz == 1
    rk = dict(method=B.MT_RK4, dt=1e-13 if film else 0.005, sample_every=10, sample_cap=8)
    rk["t_end"] = 40 * rk["dt"]
    dp = dict(method=B.MT_DP45, dt=1e-13 if film else 1e-3, rtol=1e-6, atol=1e-8, sample_cap=8)
    dp["t_end"], dp["sample_dt"] = (40e-13, 10e-13) if film else (0.2, 0.05)
    tol = 1e-11 if dtype == "f64" else 2e-5
    for kw in (rk, dp):
        out = {}
        for mode in (1, 2):
            B.mt_set_resident_mode(ctx, mode)
            l0 = B.mt_launch_count(ctx)
            out[mode] = run_gpu_integrate(ctx, prob, w.m, batch, **kw) + (B.mt_launch_count(ctx) - l0,)
        (m1, s1, r1, _, n1), (m2, s2, r2, _, n2) = out[1], out[2]
        assert np.isfinite(m2).all() and r1["n_samples"] == r2["n_samples"] == 4
        assert (r1["accepted"], r1["rejected"]) == (r2["accepted"], r2["rejected"]) and r2["accepted"] >= 4
        assert np.max(np.abs(m2 - m1)) < tol and np.max(np.abs(s2[:, 1:] - s1[:, 1:])) < tol
        assert n2 <= 12 and n2 < n1 / 8  # a handful of cooperative launches against several per right-hand side
