"""-m gpu: parity of the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element, at sizes the oracle finishes in seconds but that still span several tiles, several column
splits and ragged tails.  Tolerances are north_star's: assembly <= 1e-10 (fp64, per-row relative
L2 and Frobenius, reading Q9), fp32 planes within 1 ulp of the rounded oracle value, H_d <= 1e-12
(fp64 tensor) / <= 1e-5 (fp32 tensor) relative L2, <m>(t) within 1e-3 absolute.
"""
import numpy as np
import pytest
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W
from tests import harness as H

pytestmark = pytest.mark.gpu

TOL_ASM = 1e-10
TOL_HD = {"f64": 1e-12, "f32": 1e-5}


@pytest.fixture(scope="module")
def ctx():
    c = B.mt_create(0)
    yield c
    c.close()


def check_tensor(N_gpu, N_ref, dtype, n):
    got = N_gpu[:, :, :n].cpu().numpy()
    if dtype == "f64":
        row_err = np.linalg.norm((got - N_ref).transpose(1, 0, 2).reshape(got.shape[1], -1), axis=1)
        row_nrm = np.linalg.norm(N_ref.transpose(1, 0, 2).reshape(got.shape[1], -1), axis=1)
        assert np.max(row_err / row_nrm) <= TOL_ASM
        assert H.rel_l2(got, N_ref) <= TOL_ASM
    else:
        # fp32 planes = round-to-nearest of the fp64 closed form: within 1 fp32 ulp of the rounded
        # oracle value, or (entries that are differences of O(1) terms down at fp64 resolution, e.g.
        # symmetry zeros) within the 1e-15 absolute floor of any fp64 evaluation
        ulp = H.f32_ulp_distance(got, N_ref)
        ok = (ulp <= 1) | (np.abs(got.astype(np.float64) - N_ref) < 1e-15)
        assert ok.all(), f"{(~ok).sum()} entries off; worst ulp {ulp[~ok].max()}"
    # padding columns are zero
    if N_gpu.shape[2] > n:
        assert torch.count_nonzero(N_gpu[:, :, n:]).item() == 0


def gpu_field(ctx, N, dtype, n, n_rows, ld, Ms, m_np):
    dev = N.device
    m = torch.from_numpy(np.ascontiguousarray(m_np)).to(dev)
    Bn = m.shape[0]
    Hd = torch.empty((Bn, 3, n_rows), dtype=torch.float64, device=dev)
    B.mt_demag_field(ctx, N, H.dtype_code(dtype), n, n_rows, ld, Ms, m, Bn, Hd)
    torch.cuda.synchronize()
    return Hd.cpu().numpy()


# ---- config 1: 8x8x8 ---------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def cfg1(oracle):
    w = W.config1(batch=4)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    return w, N_ref


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config1_assembly_full_tensor(ctx, oracle, cfg1, dtype):
    w, N_ref = cfg1
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, dtype)
    assert status == 0
    check_tensor(N, N_ref, dtype, w.n)
    # paper-fixed facts hold on the GPU tensor too: self block = I/3, trace of every block
    g = N.cpu().numpy().astype(np.float64)
    i = np.arange(w.n)
    assert np.allclose(g[0, i, i], 1 / 3, atol=1e-7 if dtype == "f32" else 1e-15)
    tr = g[0] + g[3] + g[5]
    assert np.max(np.abs(tr - np.eye(w.n))) < (1e-7 if dtype == "f32" else 1e-14)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config1_field_and_rhs(ctx, oracle, cfg1, dtype):
    w, N_ref = cfg1
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(ctx, tiles, dtype)
    Hd_ref = oracle.demag_field(N_ref, w.Ms, w.m)
    Hd = gpu_field(ctx, N, dtype, w.n, w.n, ld, tiles.Ms, w.m)
    for b in range(w.m.shape[0]):
        assert H.rel_l2(Hd[b], Hd_ref[b]) <= TOL_HD[dtype]
    # fused right-hand side, all four states in one batched call and one by one
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    k_ref, heff_ref, _ = oracle.llg_rhs(H.oracle_problem(oracle, w, N_ref), w.m, want_heff=True)
    m = torch.from_numpy(w.m).cuda()
    k = torch.empty_like(m)
    heff = torch.empty_like(m)
    B.mt_llg_rhs(ctx, prob, m, 4, k, heff)
    torch.cuda.synchronize()
    assert H.rel_l2(k.cpu().numpy(), k_ref) <= TOL_HD[dtype]
    assert H.rel_l2(heff.cpu().numpy(), heff_ref) <= TOL_HD[dtype]
    k1 = torch.empty_like(m[:1])
    B.mt_llg_rhs(ctx, prob, m[2:3].contiguous(), 1, k1, None)
    assert torch.equal(k1[0], k[2])  # batching does not change a state's arithmetic
    # m . dm/dt = 0
    assert torch.max(torch.abs((m * k).sum(dim=1))).item() < 1e-14


def test_config1_hundred_evaluations_are_bitwise_identical(ctx, cfg1):
    w, _ = cfg1
    tiles = H.dev_tiles(w)
    for dtype in ("f64", "f32"):
        N, ld, _ = H.assemble(ctx, tiles, dtype)
        m = torch.from_numpy(w.m[:1].copy()).cuda()
        ref = torch.empty_like(m)
        B.mt_demag_field(ctx, N, H.dtype_code(dtype), w.n, w.n, ld, tiles.Ms, m, 1, ref)
        out = torch.empty_like(m)
        for _ in range(100):
            out.zero_()
            B.mt_demag_field(ctx, N, H.dtype_code(dtype), w.n, w.n, ld, tiles.Ms, m, 1, out)
            assert torch.equal(out, ref)


# ---- ragged sizes, row bands, batches ----------------------------------------------------------------
@pytest.mark.parametrize("grid,dtype", [((7, 5, 3), "f32"), ((7, 5, 3), "f64"), ((33, 31, 1), "f32"),
                                        ((1, 1, 1), "f64"), ((3, 1, 1), "f32")])
def test_ragged_sizes_and_row_bands(ctx, oracle, grid, dtype):
    nx, ny, nz = grid
    n = nx * ny * nz
    rng = np.random.default_rng(n)
    w = W._cuboid_workload("ragged", nx, ny, nz, (1.0, 0.7, 1.3), 1.0, W.random_unit_states(rng, 3, n),
                           gamma=1.0, alpha_ll=0.2)
    w.Ms = rng.uniform(0.5, 2.0, size=n)
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    ld = W.leading_dim(n, dtype) + 8  # extra padding on purpose
    N, ld, status = H.assemble(ctx, tiles, dtype, ld=ld)
    assert status == 0
    check_tensor(N, N_ref, dtype, n)
    Hd_ref = oracle.demag_field(N_ref, w.Ms, w.m)
    Hd = gpu_field(ctx, N, dtype, n, n, ld, tiles.Ms, w.m)
    assert H.rel_l2(Hd, Hd_ref) <= TOL_HD[dtype]
    if n >= 4:
        r0, r1 = n // 3, n - 1
        Nb, _, _ = H.assemble(ctx, tiles, dtype, r0, r1, ld=ld)
        assert torch.equal(Nb, N[:, r0:r1])
        Hb = gpu_field(ctx, Nb, dtype, n, r1 - r0, ld, tiles.Ms, w.m)
        assert H.rel_l2(Hb, Hd_ref[:, :, r0:r1]) <= TOL_HD[dtype]
        # empty band is a no-op
        B.mt_assemble_tensor(ctx, tiles, H.dtype_code(dtype), r0, r0, Nb, ld, None)


@pytest.mark.parametrize("batch", [1, 2, 3, 5, 8])
def test_batched_field_matches_single(ctx, oracle, batch):
    w = W.config5(16, 12, 4, batch=batch)  # n = 768
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    Hd_ref = oracle.demag_field(N_ref, w.Ms, w.m)
    for dtype in ("f32", "f64"):
        N, ld, _ = H.assemble(ctx, tiles, dtype)
        Hd = gpu_field(ctx, N, dtype, w.n, w.n, ld, tiles.Ms, w.m)
        for b in range(batch):
            assert H.rel_l2(Hd[b], Hd_ref[b]) <= TOL_HD[dtype]
            one = gpu_field(ctx, N, dtype, w.n, w.n, ld, tiles.Ms, w.m[b:b + 1])
            assert np.array_equal(one[0], Hd[b])


def test_host_entry_point(ctx, oracle, cfg1):
    w, N_ref = cfg1
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(ctx, tiles, "f64")
    m_host = torch.from_numpy(w.m.copy()).pin_memory()
    Hd_host = torch.empty_like(m_host).pin_memory()
    B.mt_demag_field_host(ctx, N, B.MT_F64, w.n, w.n, ld, tiles.Ms, m_host, 4, Hd_host)
    assert H.rel_l2(Hd_host.numpy(), oracle.demag_field(N_ref, w.Ms, w.m)) <= 1e-12


# ---- argument validation (error behaviour stated in mt.h) -------------------------------------------
def test_invalid_arguments_are_rejected(ctx, cfg1):
    w, _ = cfg1
    tiles = H.dev_tiles(w)
    N = torch.empty((6, w.n, 512), dtype=torch.float32, device="cuda")
    with pytest.raises(B.MtError) as e:
        B.mt_assemble_tensor(ctx, tiles, B.MT_F32, 0, w.n, N, 510, None)  # ld < n
    assert e.value.code == B.MT_ERR_INVALID_ARG
    with pytest.raises(B.MtError):
        B.mt_assemble_tensor(ctx, tiles, B.MT_F32, 0, w.n + 1, N, 512, None)
    with pytest.raises(B.MtError):
        B.mt_assemble_tensor(ctx, tiles, 7, 0, w.n, N.data_ptr(), 512, None)  # unknown dtype
    m = torch.zeros((9, 3, w.n), dtype=torch.float64, device="cuda")
    with pytest.raises(B.MtError):
        B.mt_demag_field(ctx, N, B.MT_F32, w.n, w.n, 512, tiles.Ms, m, 9, m)
    with pytest.raises(B.MtError):
        B.mt_demag_field(ctx, N.view(-1)[1:], B.MT_F32, w.n, w.n, 512, tiles.Ms, m, 1, m)  # misaligned


def test_singular_geometry_sets_status_flag(ctx):
    """A target centre on a source face (overlapping tiles) is a genuine singularity (reading Q8)."""
    n = 2
    w = W._cuboid_workload("sing", 2, 1, 1, 1.0, 1.0, np.zeros((1, 3, n)))
    # (the face-interior point is only a jump of N_xx, finite either side; an edge point is infinite)
    w.center[1] = w.center[0] + np.array([0.5, 0.5, 0.0])
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, "f64")
    assert status == 1
    # the same through the ABI's own status check: MT_ERR_SINGULAR_GEOMETRY, and MT_OK for a clean flag
    flag = torch.ones(1, dtype=torch.int32, device="cuda")
    with pytest.raises(B.MtError) as ei:
        B.mt_check_status(ctx, flag)
    assert ei.value.code == B.MT_ERR_SINGULAR_GEOMETRY
    flag.zero_()
    assert B.mt_check_status(ctx, flag) == B.MT_OK
    flag.fill_(2)
    assert B.mt_check_status(ctx, flag, allow=(B.MT_ERR_INVALID_ARG,)) == B.MT_ERR_INVALID_ARG


# ---- small mixed tetrahedra + octree mesh (config 4 shape) ------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config4_small_full_tensor(ctx, oracle, dtype):
    w = W.config4(n_tets=900, n_cub=700, n_points=300, batch=2)
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    N, ld, status = H.assemble(ctx, tiles, dtype)
    assert status == 0
    check_tensor(N, N_ref, dtype, w.n)
    Hd_ref = oracle.demag_field(N_ref, w.Ms, w.m)
    Hd = gpu_field(ctx, N, dtype, w.n, w.n, ld, tiles.Ms, w.m)
    assert H.rel_l2(Hd, Hd_ref) <= TOL_HD[dtype]


# ---- integrators ---------------------------------------------------------------------------------------
def run_gpu_integrate(ctx, prob, m0, batch, **kw):
    m = torch.from_numpy(np.ascontiguousarray(m0)).cuda()
    cap = kw.pop("sample_cap", 0)
    samples = torch.zeros((cap, 1 + 3 * batch), dtype=torch.float64, device="cuda") if cap else None
    t, res, rc = B.mt_integrate(ctx, prob, m, batch, kw.pop("t0", 0.0), samples=samples, **kw)
    s = samples[: res["n_samples"]].cpu().numpy() if cap else np.zeros((0, 1 + 3 * batch))
    return m.cpu().numpy(), s, res, rc


def test_single_spin_closed_form_on_gpu(ctx):
    """P13 on the CUDA path: m_z = tanh(alpha H t), azimuth = gamma H t (no tensor, N == NULL)."""
    Ms = torch.ones(1, dtype=torch.float64, device="cuda")
    prob = B.Problem(n=1, Ms=Ms, H_a=(0.0, 0.0, 0.9), gamma=1.3, alpha_ll=0.7)
    m0 = np.array([[[1.0], [0.0], [0.0]]])
    T = 2.0
    mz, phi = np.tanh(0.7 * 0.9 * T), 1.3 * 0.9 * T
    exact = np.array([np.cos(phi) * np.sqrt(1 - mz**2), np.sin(phi) * np.sqrt(1 - mz**2), mz])
    m, _, res, _ = run_gpu_integrate(ctx, prob, m0, 1, method=B.MT_RK4, dt=0.05, t_end=T, renormalize=False)
    assert np.max(np.abs(m[0, :, 0] - exact)) < 5e-7 and res["accepted"] == 40 and res["rhs_calls"] == 160
    m, s, res, _ = run_gpu_integrate(ctx, prob, m0, 1, method=B.MT_DP45, dt=1e-3, t_end=T, rtol=1e-8, atol=1e-10,
                                     renormalize=False, sample_dt=0.5, sample_cap=8)
    assert np.max(np.abs(m[0, :, 0] - exact)) < 1e-7
    assert np.array_equal(s[:, 0], [0.5, 1.0, 1.5, 2.0])
    assert np.allclose(s[:, 3], np.tanh(0.63 * s[:, 0]), atol=1e-7)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_rk4_trajectory_small_film(ctx, oracle, dtype):
    """Config-2 physics on a 20x5x1 film: 300 RK4 steps, sampled every 20, with exchange + Zeeman."""
    w = W.config2(20, 5, phase="dynamics")
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    N, ld, _ = H.assemble(ctx, tiles, dtype)
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    dt, steps = 1e-13, 300
    m_ref, s_ref, r_ref = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.RK4, dt=dt,
                                           t_end=steps * dt, sample_every=20, sample_cap=64, weights=w.vol)
    m, s, res, _ = run_gpu_integrate(ctx, prob, w.m, 1, method=B.MT_RK4, dt=dt, t_end=steps * dt,
                                     sample_every=20, sample_cap=64)
    assert res["accepted"] == steps and res["n_samples"] == 15 == r_ref["n_samples"]
    assert np.allclose(s[:, 0], s_ref[:, 0], rtol=1e-12)
    tol = 1e-9 if dtype == "f64" else 1e-4
    assert np.max(np.abs(s[:, 1:] - s_ref[:, 1:])) < tol
    assert np.max(np.abs(m[0] - m_ref)) < tol * 10
    assert np.max(np.abs(np.linalg.norm(m[0], axis=0) - 1.0)) < 1e-14


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_dp45_trajectory_small_cube(ctx, oracle, dtype):
    """Config-3 physics on a 6^3 cube (edge 8/6): DP45 with exchange + anisotropy to t = 3."""
    w = W.config3(6)
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    N, ld, _ = H.assemble(ctx, tiles, dtype)
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    kw = dict(dt=1e-3, t_end=3.0, rtol=1e-6, atol=1e-8, sample_dt=0.25)
    m_ref, s_ref, r_ref = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.DP45,
                                           sample_cap=64, weights=w.vol, **kw)
    m, s, res, _ = run_gpu_integrate(ctx, prob, w.m, 1, method=B.MT_DP45, sample_cap=64, **kw)
    assert res["n_samples"] == 12 == r_ref["n_samples"] and res["t"] == 3.0
    assert np.array_equal(s[:, 0], s_ref[:, 0])
    assert np.max(np.abs(s[:, 1:] - s_ref[:, 1:])) < 1e-3
    if dtype == "f64":  # same arithmetic up to rounding: same step sequence
        assert res["accepted"] == r_ref["accepted"] and res["rejected"] == r_ref["rejected"]
        assert np.max(np.abs(m[0] - m_ref)) < 1e-8
    assert res["rhs_calls"] == 1 + 6 * (res["accepted"] + res["rejected"])


def test_torque_stop_and_max_steps(ctx):
    Ms = torch.ones(1, dtype=torch.float64, device="cuda")
    prob = B.Problem(n=1, Ms=Ms, H_a=(0.0, 0.0, 1.0), gamma=0.0, alpha_ll=1.0)
    m0 = np.array([[[1.0], [0.0], [0.0]]])
    m, _, res, rc = run_gpu_integrate(ctx, prob, m0, 1, method=B.MT_DP45, dt=1e-2, t_end=100.0, rtol=1e-6, atol=1e-8,
                                      torque_tol=1e-5)
    assert rc == 0 and res["max_torque"] <= 1e-5 and abs(res["t"] - np.arccosh(1e5)) < 2.0
    m, _, res, rc = run_gpu_integrate(ctx, prob, m0, 1, method=B.MT_RK4, dt=0.05, t_end=100.0, torque_tol=1e-3)
    assert rc == 0 and res["max_torque"] <= 1e-3 and abs(res["t"] - np.arccosh(1e3)) < 0.2
    m, _, res, rc = run_gpu_integrate(ctx, prob, m0, 1, method=B.MT_DP45, dt=1e-2, t_end=100.0, max_steps=5,
                                      allow=(B.MT_ERR_MAX_STEPS,))
    assert rc == B.MT_ERR_MAX_STEPS and res["accepted"] + res["rejected"] == 5


def test_dp45_device_controller_equals_host_controller(oracle):
    """mt_set_step_control: the one-thread controller kernel replayed from a CUDA graph (default for small
    problems) against the host controller (one read per attempted step) and the oracle on an 8^3 replica of
    config 3: same accept / reject sequence, same sample times, states and samples to rounding, with the
    stop by the torque test, by t_end, and by max_steps, and sample rows capped by sample_cap."""
    w = W.config3(8, batch=2)
    x = w.extra
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    runs = {}
    for mode in (1, 2):
        c = B.mt_create(0)
        B.mt_set_step_control(c, mode)
        B.mt_set_resident_mode(c, 1)  # the graph-replayed attempt (the tensor-resident kernel: test_gpu_resident.py)
        tiles = H.dev_tiles(w)
        N, ld, _ = H.assemble(c, tiles, "f64")
        prob = H.dev_problem(w, tiles, N, "f64", ld)
        out = []
        for kw in (dict(t_end=2.0, sample_dt=0.25, sample_cap=16),
                   dict(t_end=40.0, sample_dt=1.0, sample_cap=5, torque_tol=0.5),
                   dict(t_end=2.0, max_steps=37, allow=(B.MT_ERR_MAX_STEPS,))):
            out.append(run_gpu_integrate(c, prob, w.m, 2, method=B.MT_DP45, dt=x["dt0"], rtol=x["rtol"], atol=x["atol"], **kw))
        runs[mode] = out
        c.close()
    for (m1, s1, r1, rc1), (m2, s2, r2, rc2) in zip(runs[1], runs[2]):
        assert rc1 == rc2
        for key in ("accepted", "rejected", "rhs_calls", "n_samples"):
            assert r1[key] == r2[key], key
        # (the device takes err^(-1/5) from CUDA's pow, the host from the C library's: a last-bit difference
        # in one dt feeds back through the next error estimate, so step sizes agree to ~1e-10, not to the bit)
        assert abs(r1["t"] - r2["t"]) <= 1e-12 and abs(r1["dt_last"] - r2["dt_last"]) <= 1e-6 * r1["dt_last"]
        assert abs(r1["max_torque"] - r2["max_torque"]) <= 1e-6 * r1["max_torque"]
        assert np.array_equal(s1[:, 0], s2[:, 0]) and (s1.size == 0 or np.max(np.abs(s1 - s2)) < 1e-9)
        assert np.max(np.abs(m1 - m2)) < 1e-9
    (_, s, r, _), (_, s_t, r_t, _), (_, _, r_m, rc_m) = runs[2]
    assert r["t"] == 2.0 and r["rejected"] > 0 and np.array_equal(s[:, 0], 0.25 * np.arange(1, 9))
    assert r_t["max_torque"] <= 0.5 and 5.0 < r_t["t"] < 40.0 and r_t["n_samples"] == 5
    assert rc_m == B.MT_ERR_MAX_STEPS and r_m["accepted"] + r_m["rejected"] == 37
    m_o, s_o, r_o = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.DP45, dt=x["dt0"],
                                     rtol=x["rtol"], atol=x["atol"], t_end=2.0, sample_dt=0.25, sample_cap=16, weights=w.vol)
    # (batch of two states shares the step sequence: the controller sees the maximum over both; compare a
    # single-state device run with the oracle)
    c = B.mt_create(0)
    B.mt_set_step_control(c, 2)
    B.mt_set_resident_mode(c, 1)
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(c, tiles, "f64")
    m, s, r, _ = run_gpu_integrate(c, H.dev_problem(w, tiles, N, "f64", ld), w.m[:1], 1, method=B.MT_DP45, dt=x["dt0"],
                                   rtol=x["rtol"], atol=x["atol"], t_end=2.0, sample_dt=0.25, sample_cap=16)
    c.close()
    assert (r["accepted"], r["rejected"]) == (r_o["accepted"], r_o["rejected"])
    assert np.array_equal(s[:, 0], s_o[:, 0]) and np.max(np.abs(s[:, 1:] - s_o[:, 1:])) < 1e-9
    assert np.max(np.abs(m[0] - m_o)) < 1e-8


def test_rk4_stop_test_inside_a_replayed_chunk(ctx, oracle):
    """RK4 with the torque stop test (Eq. 2): the device runs chunks of steps from a CUDA
    graph, every step leaving the torque of its start state in its own word, and the host reads a
    chunk's words at once; a satisfied test inside a chunk sends the state back to the chunk's start and
    repeats the steps before it.  Against the oracle's per-step test: same number of steps, same state,
    with the stop falling well inside a replayed chunk (after the eager first chunk), with and without
    sampling."""
    w = W.config3(4)
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    N, ld, _ = H.assemble(ctx, tiles, "f64")
    prob = H.dev_problem(w, tiles, N, "f64", ld)
    base = dict(dt=0.02, t_end=400.0)
    # torque of a relaxing 4^3 cube falls steadily: pick the tolerance it crosses after ~200 steps
    m_o, _, r_probe = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.RK4, dt=0.02, t_end=4.0,
                                       torque_tol=1e-30)
    tol = 0.999 * r_probe["max_torque"]
    for extra in (dict(), dict(sample_every=16, sample_cap=64)):
        m_o, s_o, r_o = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.RK4,
                                         torque_tol=tol, weights=w.vol, **base, **extra)
        m, s, r, rc = run_gpu_integrate(ctx, prob, w.m[:1], 1, method=B.MT_RK4, torque_tol=tol, **base, **extra)
        assert rc == 0 and r["accepted"] == r_o["accepted"] and 150 < r["accepted"] < 20000
        assert r["accepted"] % 64 not in (0, 63) or extra  # not at a chunk boundary by luck
        assert abs(r["t"] - r_o["t"]) < 1e-9 and r["max_torque"] <= tol
        assert abs(r["max_torque"] - r_o["max_torque"]) <= 1e-9 * tol
        assert np.max(np.abs(m[0] - m_o)) < 1e-10
        assert len(s) == len(s_o) and (len(s) == 0 or np.max(np.abs(s - s_o)) < 1e-10)


def test_batched_rk4_equals_individual_runs(ctx, oracle):
    w = W.config3(5, batch=3)
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(ctx, tiles, "f32")
    prob = H.dev_problem(w, tiles, N, "f32", ld)
    mb, sb, _, _ = run_gpu_integrate(ctx, prob, w.m, 3, method=B.MT_RK4, dt=0.01, t_end=0.5, sample_every=10, sample_cap=8)
    for b in range(3):
        m1, s1, _, _ = run_gpu_integrate(ctx, prob, w.m[b:b + 1], 1, method=B.MT_RK4, dt=0.01, t_end=0.5,
                                         sample_every=10, sample_cap=8)
        assert np.array_equal(m1[0], mb[b])
        assert np.array_equal(s1[:, 1:4], sb[:, 1 + 3 * b:4 + 3 * b])


def test_dp45_nonfinite_state_is_an_error_and_zero_m_stays_zero(ctx):
    """a NaN in m must reach the DP45 error estimate (no fmax laundering) and end the run
    with MT_ERR_STEP_UNDERFLOW instead of MT_OK with a NaN state; m_i = 0 is a fixed point (Q10c, Q11b)."""
    n = 3
    Ms = torch.ones(n, dtype=torch.float64, device="cuda")
    prob = B.Problem(n=n, Ms=Ms, H_a=(0.0, 0.0, 1.0), gamma=1.0, alpha_ll=0.5)
    m0 = np.array([[[1.0, 0.0, 0.6], [0.0, 1.0, 0.0], [0.0, 0.0, 0.8]]])
    bad = m0.copy()
    bad[0, 1, 2] = np.nan
    _, _, res, rc = run_gpu_integrate(ctx, prob, bad, 1, method=B.MT_DP45, dt=1e-2, t_end=1.0, max_steps=50,
                                      allow=(B.MT_ERR_STEP_UNDERFLOW,))
    assert rc == B.MT_ERR_STEP_UNDERFLOW and res["accepted"] == 0
    zero = m0.copy()
    zero[0, :, 1] = 0.0
    for method in (B.MT_RK4, B.MT_DP45):
        m, _, res, rc = run_gpu_integrate(ctx, prob, zero, 1, method=method, dt=1e-2, t_end=0.5)
        assert rc == 0 and np.all(m[0][:, 1] == 0.0) and np.all(np.isfinite(m))
        assert np.allclose(np.linalg.norm(m[0][:, [0, 2]], axis=0), 1.0, atol=1e-14)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_small_problem_field_in_one_launch_equals_staged_path_bitwise(ctx, cfg1, dtype):
    """Where the register-streaming kernel is the default and n is a multiple of the 16-byte vector, mt_demag_field and
    mt_llg_rhs form Ms*m inside the field kernel (one launch per call); forcing the same kernel with
    mt_set_demag_variant(1) keeps the staging launch: the two agree to the bit (same expression for Ms*m)."""
    w, _ = cfg1
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(ctx, tiles, dtype)
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    m = torch.from_numpy(w.m).cuda()
    out = {}
    for variant in (0, 1):
        B.mt_set_demag_variant(ctx, variant)
        Hd, k = torch.empty_like(m), torch.empty_like(m)
        l0 = B.mt_launch_count(ctx)
        B.mt_demag_field(ctx, N, H.dtype_code(dtype), w.n, w.n, ld, tiles.Ms, m, m.shape[0], Hd)
        l1 = B.mt_launch_count(ctx)
        B.mt_llg_rhs(ctx, prob, m, m.shape[0], k, None)
        torch.cuda.synchronize()
        out[variant] = (Hd, k, l1 - l0, B.mt_launch_count(ctx) - l1)
    B.mt_set_demag_variant(ctx, 0)
    assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1])
    assert out[0][2:] == (1, 1) and out[1][2:] == (2, 2)
