"""-m gpu: parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

Where the oracle cannot finish the whole problem in seconds, parity is on sampled target rows it
can compute one by one (tensor rows, H_d and the right-hand side of those rows) and on properties
that hold at any size; trajectories are compared on windows at full size and on reduced grids run
by both sides (DESIGN.md §6 states the plan per config).
"""
import numpy as np
import pytest
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W
from tests import harness as H
from tests.test_gpu_small import TOL_ASM, TOL_HD, check_tensor, gpu_field, run_gpu_integrate

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = B.mt_create(0)
    yield c
    c.close()


def grid_corner_rows(grid):
    nx, ny, nz = grid
    idx = lambda i, j, k: (k * ny + j) * nx + i
    rows = [idx(i, j, k) for i in (0, nx - 1) for j in (0, ny - 1) for k in (0, nz - 1)]
    rows.append(idx(nx // 2, ny // 2, nz // 2))
    return rows


def sampled_row_checks(ctx, oracle, w, tiles, N, ld, dtype, rows, states, config_id):
    """Tensor rows, H_d and RHS of the sampled rows against the oracle."""
    n = w.n
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=rows, long_double=True)
    idx = torch.from_numpy(rows).to(N.device)
    got = N.index_select(1, idx)
    check_tensor(got, N_ref, dtype, n)
    Hd_ref = oracle.demag_field(N_ref, w.Ms, states)            # [B, 3, nrows]
    Hd = gpu_field(ctx, N, dtype, n, n, ld, tiles.Ms, states)   # [B, 3, n]
    for b in range(states.shape[0]):
        assert H.rel_l2(Hd[b][:, rows], Hd_ref[b]) <= TOL_HD[dtype]
    prob = H.dev_problem(w, tiles, N, dtype, ld)
    k_ref, _ = oracle.llg_rhs(H.oracle_problem(oracle, w, N_ref, rows=rows), states)
    m = torch.from_numpy(np.ascontiguousarray(states)).cuda()
    k = torch.empty_like(m)
    B.mt_llg_rhs(ctx, prob, m, states.shape[0], k, None)
    torch.cuda.synchronize()
    kk = k.cpu().numpy()
    for b in range(states.shape[0]):
        assert H.rel_l2(kk[b][:, rows], k_ref[b]) <= TOL_HD[dtype]
    return Hd


# ---- config 2: 160x40x1 film, fp32 tensor -------------------------------------------------------------
@pytest.fixture(scope="module")
def cfg2(oracle):
    w = W.config2(batch=4)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)  # 4.1e7 pairs
    return w, N_ref


def test_config2_full_fp32_tensor_and_rhs(ctx, oracle, cfg2):
    w, N_ref = cfg2
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, "f32")
    assert status == 0
    check_tensor(N, N_ref, "f32", w.n)
    prob = H.dev_problem(w, tiles, N, "f32", ld)
    k_ref, heff_ref, _ = oracle.llg_rhs(H.oracle_problem(oracle, w, N_ref), w.m, want_heff=True)
    m = torch.from_numpy(w.m).cuda()
    k, heff = torch.empty_like(m), torch.empty_like(m)
    B.mt_llg_rhs(ctx, prob, m, 4, k, heff)
    torch.cuda.synchronize()
    for b in range(4):
        assert H.rel_l2(heff[b].cpu().numpy(), heff_ref[b]) <= 1e-5
        assert H.rel_l2(k[b].cpu().numpy(), k_ref[b]) <= 1e-5


def test_config2_fp64_assembly_gate(ctx, oracle, cfg2):
    """Reading Q9: per-row relative L2 and Frobenius <= 1e-10 although single far-field entries
    (r up to 165 edges) cannot reach 1e-10 individually."""
    w, N_ref = cfg2
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(ctx, tiles, "f64")
    check_tensor(N, N_ref, "f64", w.n)


def test_config2_trajectory_window_full_size(ctx, oracle, cfg2):
    """First 40 RK4 steps of each phase at full N against the oracle (window plan)."""
    w, N_ref = cfg2
    tiles = H.dev_tiles(w)
    N, ld, _ = H.assemble(ctx, tiles, "f32")
    for phase in ("relax", "dynamics"):
        wp = W.config2(batch=1, phase=phase)
        prob = H.dev_problem(wp, tiles, N, "f32", ld)
        dt, steps = 1e-13, 40
        m_ref, s_ref, _ = oracle.integrate(H.oracle_problem(oracle, wp, N_ref), wp.m[0], method=oracle.RK4, dt=dt,
                                           t_end=steps * dt, sample_every=10, sample_cap=8, weights=wp.vol)
        m, s, res, _ = run_gpu_integrate(ctx, prob, wp.m, 1, method=B.MT_RK4, dt=dt, t_end=steps * dt,
                                         sample_every=10, sample_cap=8)
        assert res["accepted"] == steps and res["n_samples"] == 4
        assert np.max(np.abs(s[:, 1:] - s_ref[:, 1:])) < 1e-6
        assert np.max(np.abs(m[0] - m_ref)) < 1e-5


def test_config2_full_length_trajectory_reduced_grid(ctx, oracle):
    """Whole config-2 protocol (20,000 relax steps with alpha = 1, then 10,000 steps under the
    25 mT field, dt = 1e-13 s) on a 40x10x1 film run by both sides; <m>(t) sampled every 100
    steps must agree within 1e-3 absolute (north_star)."""
    wr = W.config2(40, 10, phase="relax")
    wd = W.config2(40, 10, phase="dynamics")
    tiles = H.dev_tiles(wr)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, wr), long_double=True)
    N, ld, _ = H.assemble(ctx, tiles, "f32")
    dt = 1e-13
    # oracle
    m_o, s1_o, _ = oracle.integrate(H.oracle_problem(oracle, wr, N_ref), wr.m[0], method=oracle.RK4, dt=dt,
                                    t_end=20000 * dt, sample_every=100, sample_cap=200, weights=wr.vol)
    m_o, s2_o, _ = oracle.integrate(H.oracle_problem(oracle, wd, N_ref), m_o, method=oracle.RK4, dt=dt,
                                    t_end=10000 * dt, sample_every=100, sample_cap=100, weights=wd.vol)
    # CUDA path
    m1, s1, r1, _ = run_gpu_integrate(ctx, H.dev_problem(wr, tiles, N, "f32", ld), wr.m, 1, method=B.MT_RK4, dt=dt,
                                      t_end=20000 * dt, sample_every=100, sample_cap=200)
    m2, s2, r2, _ = run_gpu_integrate(ctx, H.dev_problem(wd, tiles, N, "f32", ld), m1, 1, method=B.MT_RK4, dt=dt,
                                      t_end=10000 * dt, sample_every=100, sample_cap=100)
    assert r1["accepted"] == 20000 and r2["accepted"] == 10000 and len(s1) == 200 and len(s2) == 100
    assert np.max(np.abs(s1[:, 1:] - s1_o[:, 1:])) < 1e-3
    assert np.max(np.abs(s2[:, 1:] - s2_o[:, 1:])) < 1e-3
    assert np.max(np.abs(np.linalg.norm(m2[0], axis=0) - 1.0)) < 1e-14
    # the dynamics actually moved the magnetisation (the test is not vacuous)
    assert np.max(np.abs(s2[-1, 1:] - s2[0, 1:])) > 0.05


# ---- config 3: 32^3 cube, fp32 and fp64 tensors ---------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config3_sampled_rows(ctx, oracle, dtype):
    w = W.config3(32, batch=2, dtype=dtype)
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, dtype)   # 25.8 GB / 51.5 GB
    assert status == 0
    rows = W.sample_rows(3, w.n, 1024, extra=grid_corner_rows(w.grid))
    sampled_row_checks(ctx, oracle, w, tiles, N, ld, dtype, rows, w.m, 3)
    del N
    torch.cuda.empty_cache()


def config3_dp45_segments(ctx, w, prob, t_end, seg, torque_tol):
    """BASELINE config 3's own protocol (DP45, rtol/atol/dt0 of DESIGN.md Q11, stop test Q12) run in
    segments of `seg` time units so that the energy can be read between them; mt_integrate is
    resumable on (m, t, dt_last).  Returns sample rows [t, <m>], energies, counters."""
    x = w.extra
    m = torch.from_numpy(np.ascontiguousarray(w.m[:1])).cuda()
    E = torch.zeros((1, 5), dtype=torch.float64, device="cuda")
    row = torch.zeros((1, 4), dtype=torch.float64, device="cuda")
    B.mt_energy(ctx, prob, m, 1, E)
    energies, rows = [float(E[0, 4].item())], []
    tot = dict(accepted=0, rejected=0, rhs_calls=0, max_torque=float("inf"))
    t, dt = 0.0, x["dt0"]
    while t < t_end and tot["max_torque"] > torque_tol:
        t1 = min(t_end, t + seg)
        t, res, _ = B.mt_integrate(ctx, prob, m, 1, t, method=B.MT_DP45, dt=dt, t_end=t1, rtol=x["rtol"],
                                   atol=x["atol"], torque_tol=torque_tol, renormalize=True, sample_dt=t1 - t,
                                   samples=row)
        dt = res["dt_last"]
        for k in ("accepted", "rejected", "rhs_calls"):
            tot[k] += res[k]
        tot["max_torque"] = res["max_torque"]
        B.mt_energy(ctx, prob, m, 1, E)
        energies.append(float(E[0, 4].item()))
        rows.append(np.concatenate([[t], m[0].mean(dim=1).cpu().numpy()]))
    return m.cpu().numpy(), np.array(rows), np.array(energies), tot, t


def test_config3_full_size_dp45_fp32_vs_fp64(ctx):
    """Config 3 as BASELINE.json states it, at its full size: "DP45 adaptive to equilibrium; both fp32
    and fp64 tensor paths" (SP3 shape PAPER.md:185-187; RK(4,5) PAPER.md:143,181; stop test Eq. 2
    PAPER.md:40).  The oracle cannot run 32^3 (parity of the same integrator is on the 8^3/16^3
    replicas below and on sampled rows of the right-hand side above); here the two device paths are
    held against each other and against what holds at any size: <m>(t) of the fp32- and the
    fp64-tensor runs within 1e-3 at common times, |m| = 1, the free energy non-increasing (alpha > 0,
    no applied field: PAPER.md:58), the torque falling towards the stop tolerance.  The driver's GPU
    test step has a 20-minute limit, so the run stops at t = 8 (the first ~1,300 attempted steps: the
    random start is smoothed, the step has reached the exchange stability limit); the whole protocol
    (to |m x H| <= 1e-5 or t = 200) is what `bench.py --config 3 --protocol` runs and reports."""
    T_END, SEG = 8.0, 1.0
    out = {}
    w = W.config3(32, batch=1)
    tiles = H.dev_tiles(w)
    for dtype in ("f32", "f64"):
        N, ld, status = H.assemble(ctx, tiles, dtype)
        assert status == 0
        prob = H.dev_problem(w, tiles, N, dtype, ld)
        out[dtype] = config3_dp45_segments(ctx, w, prob, T_END, SEG, w.extra["torque_tol"])
        del N, prob
        torch.cuda.empty_cache()
    (m32, s32, e32, r32, t32), (m64, s64, e64, r64, t64) = out["f32"], out["f64"]
    assert t32 == T_END and t64 == T_END and len(s32) == len(s64) == int(T_END / SEG)
    assert np.array_equal(s32[:, 0], s64[:, 0])
    assert np.max(np.abs(s32[:, 1:] - s64[:, 1:])) < 1e-3
    assert np.max(np.abs(m32 - m64)) < 1e-3  # tile by tile as well: the fp32 tensor does not bend the path
    for m, e, r in ((m32, e32, r32), (m64, e64, r64)):
        assert np.max(np.abs(np.linalg.norm(m[0], axis=0) - 1.0)) < 1e-14
        assert np.all(np.diff(e) <= 1e-12 * np.abs(e[0])), np.diff(e)
        assert e[-1] < 0.5 * e[0]          # not vacuous: a random state has lost most of its exchange energy
        assert r["rejected"] < r["accepted"] and r["rhs_calls"] >= 6 * r["accepted"]
        assert np.isfinite(r["max_torque"]) and r["max_torque"] < 1.0
    # the two runs take nearly the same step sequence (same controller, errors differ by ~1e-7 relative)
    assert abs(r32["accepted"] - r64["accepted"]) <= 0.02 * r64["accepted"]


def test_config3_trajectory_replicas(ctx, oracle):
    """DP45 trajectory parity on replicas both sides can run: 8^3 to equilibrium (torque stop) and a
    16^3 window; <m>(t) at common sample times within 1e-3."""
    w = W.config3(8)
    x = w.extra
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    kw = dict(dt=x["dt0"], t_end=60.0, rtol=x["rtol"], atol=x["atol"], torque_tol=1e-4, sample_dt=2.0)
    m_o, s_o, r_o = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.DP45, sample_cap=64,
                                     weights=w.vol, **kw)
    for dtype in ("f32", "f64"):
        N, ld, _ = H.assemble(ctx, tiles, dtype)
        m, s, r, _ = run_gpu_integrate(ctx, H.dev_problem(w, tiles, N, dtype, ld), w.m, 1, method=B.MT_DP45,
                                       sample_cap=64, **kw)
        k = min(len(s), len(s_o))
        assert k >= 5 and np.array_equal(s[:k, 0], s_o[:k, 0])
        assert np.max(np.abs(s[:k, 1:] - s_o[:k, 1:])) < 1e-3
        assert r["t"] == 60.0 or (r["max_torque"] <= 1e-4 and abs(r["t"] - r_o["t"]) < 2.0)
        assert np.max(np.abs(np.linalg.norm(m[0], axis=0) - 1.0)) < 1e-14
    w = W.config3(16)
    tiles = H.dev_tiles(w)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), long_double=True)
    kw = dict(dt=x["dt0"], t_end=1.0, rtol=x["rtol"], atol=x["atol"], sample_dt=0.25)
    m_o, s_o, r_o = oracle.integrate(H.oracle_problem(oracle, w, N_ref), w.m[0], method=oracle.DP45, sample_cap=8,
                                     weights=w.vol, **kw)
    N, ld, _ = H.assemble(ctx, tiles, "f32")
    m, s, r, _ = run_gpu_integrate(ctx, H.dev_problem(w, tiles, N, "f32", ld), w.m, 1, method=B.MT_DP45,
                                   sample_cap=8, **kw)
    assert np.array_equal(s[:, 0], s_o[:, 0]) and np.max(np.abs(s[:, 1:] - s_o[:, 1:])) < 1e-3
    assert np.max(np.abs(m[0] - m_o)) < 1e-3


# ---- config 4: 20,000 tetrahedra + 16,384 octree cuboids -----------------------------------------------
def degenerate_alignments(w, per_kind=8, chunk=1024):
    """Guard rules of SURVEY A.3 (Q8): every (cuboid target, cuboid source) pair of the mesh
    whose target centre lies exactly in the plane of a source face (one coordinate of d equals +-h:
    "face" alignment) or on the line of a source edge (two coordinates: "edge" alignment), outside the
    source.  ALL such pairs are enumerated on the host (16,384^2 pairs, exact comparisons); they are
    classified by kind = (aligned axes, signs) and `per_kind` target rows are returned for every kind
    that occurs, so that each branch of the guard rules is exercised.  (Checking every aligned pair's row
    against the long-double oracle is out of reach: two thirds of the octree's leaves have at least one —
    ~11,000 rows x 36,384 sources = 4e8 long-double pairs, minutes of host time.)
    Returns (rows, {kind: number of pairs})."""
    cub = np.where(w.type == 0)[0]
    dev = "cuda" if torch.cuda.is_available() else "cpu"   # 2.7e8 pairs: exact comparisons, done with torch
    c = torch.from_numpy(w.center[cub]).to(dev)
    h = torch.from_numpy(0.5 * w.size[cub]).to(dev)
    counts = np.zeros(27, dtype=np.int64)           # kind code: sum over axes of (1 + [d_ax > 0]) * 3^ax
    targets = [set() for _ in range(27)]
    pw = torch.tensor([1, 3, 9], dtype=torch.int64, device=dev)
    for a0 in range(0, len(cub), chunk):
        d = c[a0:a0 + chunk, None, :] - c[None, :, :]                 # [targets, sources, 3]
        on = d.abs() == h[None, :, :]
        outside = (d.abs() > h[None, :, :]).any(dim=2)
        code = ((on.to(torch.int64) * (1 + (d > 0).to(torch.int64))) * pw).sum(dim=2)
        code[~outside] = 0
        counts += torch.bincount(code.reshape(-1), minlength=27).cpu().numpy()
        for kc in torch.unique(code).tolist():
            if kc:
                targets[kc].update((a0 + torch.nonzero((code == kc).any(dim=1))[:, 0]).tolist())
    kinds, rows = {}, set()
    for kc in range(1, 27):
        if counts[kc]:
            kind = tuple((ax, 1 if (kc // 3**ax) % 3 == 2 else -1) for ax in range(3) if (kc // 3**ax) % 3)
            kinds[kind] = int(counts[kc])
            t = np.array(sorted(targets[kc]))
            rng = W.rng_for(4, 100 + kc)
            rows.update(int(cub[i]) for i in rng.choice(t, size=min(per_kind, len(t)), replace=False))
    return sorted(rows), kinds


def test_config4_full_size_sampled_rows(ctx, oracle):
    w = W.config4(batch=2)
    assert w.n == 36384
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, "f32")   # 31.8 GB
    assert status == 0
    deg, kinds = degenerate_alignments(w)
    # the 2:1 octree does produce aligned pairs: face-plane alignments along every axis and both sides,
    # and edge-line alignments (two coordinates at once)
    assert all(((ax, sg),) in kinds for ax in range(3) for sg in (-1, 1)), sorted(kinds)
    assert any(len(k) == 2 for k in kinds) and not any(len(k) == 3 for k in kinds), sorted(kinds)
    assert len(deg) >= 32 and sum(kinds.values()) > 100000
    rng = W.rng_for(4, 9)
    rows = np.array(sorted(set(rng.choice(20000, 512, replace=False)) | set(20000 + rng.choice(16384, 512, replace=False))
                           | set(deg)), dtype=np.int64)
    sampled_row_checks(ctx, oracle, w, tiles, N, ld, "f32", rows, w.m, 4)
    del N
    torch.cuda.empty_cache()
    # fp64 kernel on a row band containing both tile types' targets
    r0, r1 = 19744, 20256
    Nb, ldb, status = H.assemble(ctx, tiles, "f64", r0, r1)
    assert status == 0
    sub = np.arange(r0, r1, 8, dtype=np.int64)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=sub, long_double=True)
    check_tensor(Nb[:, ::8], N_ref, "f64", w.n)


# ---- config 5: 64x64x16, 65,536 tiles, 103 GB fp32 tensor ----------------------------------------------
def test_config5_full_size(ctx, oracle):
    w = W.config5(batch=8)
    assert w.n == 65536
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, "f32")   # 103.08 GB: plane has 2^32 elements (64-bit indexing)
    assert status == 0 and N.numel() == 6 * 65536 * 65536
    rows = W.sample_rows(5, w.n, 1024, extra=grid_corner_rows(w.grid) + [65535, 32768, 32767])
    Hd = sampled_row_checks(ctx, oracle, w, tiles, N, ld, "f32", rows, w.m, 5)
    # properties that hold at any size: uniform m -> H_d,i = -(sum_j N_ij) m, and sum_j N_ij is the
    # tensor of the whole 64x64x16 block at centre i (superposition): check rows of the GPU field
    # against the big-block closed form evaluated by the oracle
    mu = np.zeros((1, 3, w.n))
    mu[0, 2] = 1.0
    Hu = gpu_field(ctx, N, "f32", w.n, w.n, ld, tiles.Ms, mu)[0]
    big = np.array([64.0, 64.0, 16.0])
    for i in (0, 32768 + 2080, 65535):
        blk = oracle.cuboid_block(0.5 * big, w.center[i] - 0.5 * big)
        assert np.max(np.abs(Hu[:, i] + blk[[2, 4, 5]])) < 2e-5
    # determinism at full size
    Hd2 = gpu_field(ctx, N, "f32", w.n, w.n, ld, tiles.Ms, w.m)
    assert np.array_equal(Hd, Hd2)
    # last rows / last columns (64-bit offsets beyond 2^32 elements in every plane but the first)
    assert torch.isfinite(N[5, 65535, 65528:]).all() and abs(N[0, 65535, 65535].item() - 1 / 3) < 1e-7
    del N
    torch.cuda.empty_cache()
    # fp64 assembly kernel on a 512-row band via row_begin/row_end
    r0 = 40000
    Nb, ldb, status = H.assemble(ctx, tiles, "f64", r0, r0 + 512)
    sub = np.arange(r0, r0 + 512, 16, dtype=np.int64)
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=sub, long_double=True)
    check_tensor(Nb[:, ::16], N_ref, "f64", w.n)


def test_config5_full_size_symmetric_half(ctx, oracle):
    """F3 at BASELINE's full size, in the configuration bench.py times: the field from the 51.6 GB
    pair-symmetric half on sampled rows against the oracle's rows of the full tensor; the uniform-m
    property (sum_j N_ij = tensor of the whole block) on rows the sample does not contain."""
    w = W.config5(batch=2)
    tiles = H.dev_tiles(w)
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    S = B.mt_assemble_tensor_sym(ctx, tiles, B.MT_F32, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0 and S.data.numel() * 4 < 0.502 * 6 * 65536 * 65536 * 4
    rows = W.sample_rows(5, w.n, 96, extra=grid_corner_rows(w.grid) + [65535, 32768, 32767, 31, 32, 127, 128])
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=rows, long_double=True)
    Hd_ref = oracle.demag_field(N_ref, w.Ms, w.m)
    m = torch.from_numpy(w.m).cuda()
    Hd = torch.empty_like(m)
    B.mt_demag_field_sym(ctx, S, tiles.Ms, m, 2, Hd)
    torch.cuda.synchronize()
    got = Hd.cpu().numpy()
    for b in range(2):
        assert H.rel_l2(got[b][:, rows], Hd_ref[b]) <= TOL_HD["f32"]
    mu = torch.zeros((1, 3, w.n), dtype=torch.float64, device="cuda")
    mu[0, 2] = 1.0
    Hu = torch.empty_like(mu)
    B.mt_demag_field_sym(ctx, S, tiles.Ms, mu, 1, Hu)
    Hu = Hu.cpu().numpy()[0]
    big = np.array([64.0, 64.0, 16.0])
    for i in (0, 4097, 32768 + 2080, 65535):
        blk = oracle.cuboid_block(0.5 * big, w.center[i] - 0.5 * big)
        assert np.max(np.abs(Hu[:, i] + blk[[2, 4, 5]])) < 2e-5
    Hd2 = torch.empty_like(m)
    B.mt_demag_field_sym(ctx, S, tiles.Ms, m, 2, Hd2)
    assert torch.equal(Hd, Hd2)


def gap_cut(host, tau_dev):
    """A cut inside a > 1e-3 relative gap of the oracle's magnitudes, next to the device's threshold."""
    import math
    mags = np.abs(host[(np.abs(host) > 0.5 * tau_dev) & (np.abs(host) < 2.0 * tau_dev)]).astype(np.float64)
    mags = np.unique(mags)
    gaps = np.nonzero(mags[1:] > mags[:-1] * 1.001)[0]
    g = gaps[np.argmin(np.abs(np.log(mags[gaps] / tau_dev)))]
    tau = float(np.float32(math.sqrt(mags[g] * mags[g + 1])))
    assert mags[g] < tau < mags[g + 1] and 0.5 * tau_dev < tau < 2.0 * tau_dev
    return tau


def check_sparse_rows(S, rows, N_ref, trunc, n):
    """Bitmap rows, 16-bit columns (+ panel offsets) and packed values of the sampled target rows of a
    whole-tensor SparseTensor against the oracle's truncated rows."""
    ridx = torch.from_numpy(rows).cuda()
    for p in range(6):
        ptr = S.row_ptr[p * n: (p + 1) * n + 1]
        beg, end = ptr[:-1][ridx].cpu().numpy(), ptr[1:][ridx].cpu().numpy()
        mask = S.mask[p].index_select(0, ridx).cpu().numpy().view(np.uint32)
        bits = ((mask[..., None] >> np.arange(32, dtype=np.uint32)) & 1).astype(bool).reshape(len(rows), -1)
        assert np.array_equal(bits[:, :n], trunc[p] != 0) and not bits[:, n:].any()
        pp = S.panel_ptr[p * n: (p + 1) * n].index_select(0, ridx).cpu().numpy() if S.panel_ptr is not None else None
        for q in range(len(rows)):
            cols_ref = np.nonzero(trunc[p, q])[0]
            assert end[q] - beg[q] == len(cols_ref)
            assert np.array_equal(S.cols16[beg[q]:end[q]].cpu().numpy(), (cols_ref & 0xFFFF).astype(np.uint16))
            if pp is not None:
                starts = [beg[q] + np.count_nonzero(cols_ref < 65536 * (k + 1)) for k in range(pp.shape[1])]
                assert np.array_equal(pp[q], np.array(starts))
            vals = S.vals[beg[q]:end[q]].cpu().numpy()
            assert (H.f32_ulp_distance(vals, N_ref[p, q, cols_ref]) <= 1).all()


def test_config5_full_size_thresholded_index_rows(ctx, oracle):
    """F1 at BASELINE's full size, in the configuration bench.py times (X = 0.9, index rows).
    (1) the device's threshold value has the rank PAPER.md:239 defines, counted on the device tensor
    with torch reductions (not this library's kernels); (2) on sampled target rows the bitmap, the
    16-bit columns and the packed values equal the oracle's truncation of its own rows, with the cut
    placed in a gap of the oracle's magnitudes next to the device's value (so that the last-bit
    difference between the two assemblies cannot move an entry across it); (3) the field from the
    index rows on those rows against the oracle's field of its truncated rows; the bitmap-row kernel
    and the index-row kernel agree on every row."""
    import math
    from oracle import threshold as OT
    w = W.config5(batch=2)
    n = w.n
    tiles = H.dev_tiles(w)
    N, ld, status = H.assemble(ctx, tiles, "f32")
    X = 0.9
    tau_dev, cnt = B.mt_threshold_value(ctx, N, B.MT_F32, n, n, ld, X)
    mult = (1, 2, 2, 1, 2, 1)
    nonzero = below = ties = 0
    for p in range(6):
        for r0 in range(0, n, 8192):
            a = N[p, r0:r0 + 8192, :n].abs()
            nonzero += mult[p] * int(torch.count_nonzero(a))
            below += mult[p] * int(((a < tau_dev) & (a != 0)).sum())
            ties += mult[p] * int((a == tau_dev).sum())
            del a
    assert cnt == nonzero
    k = math.floor(X * nonzero)
    assert below <= k < below + ties, (below, k, ties)
    # (2) sampled rows, cut in a gap of the oracle's magnitudes
    rows = W.sample_rows(5, n, 64, extra=grid_corner_rows(w.grid) + [65535, 32768, 32767])
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=rows, long_double=True)
    host = N_ref.astype(np.float32)
    tau = gap_cut(host, tau_dev)
    S = B.mt_sparse_build(ctx, N, B.MT_F32, n, n, ld, tau)
    B.mt_sparse_index(ctx, S)
    torch.cuda.synchronize()
    assert 0.05 < S.nnz / (6.0 * n * n) < 0.2
    trunc = OT.truncate(host, tau)
    check_sparse_rows(S, rows, N_ref, trunc, n)
    # (2b) the streamed build (dense tensor never resident: 4,096-row bands, 6.4 GB) gives the same
    # threshold and, for the same cut, the same offsets, bitmaps and values (64-bit offsets throughout)
    T = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, X, 4096)
    assert T.tau == tau_dev
    del T
    T = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, X, 3000, tau=tau)
    torch.cuda.synchronize()
    assert T.nnz == S.nnz and torch.equal(T.row_ptr, S.row_ptr)
    assert torch.equal(T.mask, S.mask) and torch.equal(T.vals, S.vals)
    del T
    # (3) fields
    m = torch.from_numpy(w.m).cuda()
    Hb, Hi, Hi2 = torch.empty_like(m), torch.empty_like(m), torch.empty_like(m)
    cols = S.cols16
    S.cols16 = None
    B.mt_demag_field_sparse(ctx, S, tiles.Ms, m, 2, Hb)      # bitmap-row kernel
    S.cols16 = cols
    B.mt_demag_field_sparse(ctx, S, tiles.Ms, m, 2, Hi)      # index-row kernel
    B.mt_demag_field_sparse(ctx, S, tiles.Ms, m, 2, Hi2)
    torch.cuda.synchronize()
    assert torch.equal(Hi, Hi2)
    ref = oracle.demag_field(trunc.astype(np.float64), w.Ms, w.m)
    got_i, got_b = Hi.cpu().numpy(), Hb.cpu().numpy()
    for b in range(2):
        assert H.rel_l2(got_i[b][:, rows], ref[b]) <= TOL_HD["f32"]
        assert H.rel_l2(got_b[b][:, rows], ref[b]) <= TOL_HD["f32"]
        assert H.rel_l2(got_i[b], got_b[b]) <= 2e-6


def test_beyond_hbm_size_thresholded_streamed(ctx, oracle):
    """N = 131,072 tiles (128 x 64 x 16 unit cubes): the dense fp32 tensor is 412 GB and cannot exist on
    one B200; thresholded at X = 0.95 and built band by band it is 34 GB.  Sampled
    rows (bitmap, columns in two panels, values, field from both kernels) against the oracle."""
    from oracle import threshold as OT
    w = W.config5(128, 64, 16, batch=1)
    n = w.n
    assert n == 131072
    tiles = H.dev_tiles(w)
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    T0 = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, 0.95, 4096, status)
    tau_dev = T0.tau
    assert int(status.item()) == 0 and 0.04 < T0.nnz / (6.0 * n * n) < 0.06
    del T0
    rows = W.sample_rows(5, n, 32, extra=grid_corner_rows(w.grid) + [65535, 65536, n - 1])
    N_ref = oracle.assemble_rows(H.oracle_tiles(oracle, w), rows=rows, long_double=True)
    host = N_ref.astype(np.float32)
    tau = gap_cut(host, tau_dev)
    S = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, 0.95, 4096, status, tau=tau)
    B.mt_sparse_index(ctx, S)
    torch.cuda.synchronize()
    trunc = OT.truncate(host, tau)
    check_sparse_rows(S, rows, N_ref, trunc, n)
    # index rows written by the fill pass itself (no bitmap held): the same columns, panel offsets, values
    U = B.mt_sparse_build_streamed(ctx, tiles, B.MT_F32, 0.95, 4096, status, tau=tau, index=True, keep_mask=False)
    assert U.mask is None and torch.equal(U.row_ptr, S.row_ptr) and torch.equal(U.vals, S.vals)
    assert torch.equal(U.cols16, S.cols16) and torch.equal(U.panel_ptr, S.panel_ptr)
    del U
    m = torch.from_numpy(w.m).cuda()
    Hb, Hi = torch.empty_like(m), torch.empty_like(m)
    cols = S.cols16
    S.cols16 = None
    B.mt_demag_field_sparse(ctx, S, tiles.Ms, m, 1, Hb)
    S.cols16 = cols
    B.mt_demag_field_sparse(ctx, S, tiles.Ms, m, 1, Hi)
    torch.cuda.synchronize()
    ref = oracle.demag_field(trunc.astype(np.float64), w.Ms, w.m)
    assert H.rel_l2(Hi.cpu().numpy()[0][:, rows], ref[0]) <= TOL_HD["f32"]
    assert H.rel_l2(Hb.cpu().numpy()[0][:, rows], ref[0]) <= TOL_HD["f32"]
    assert H.rel_l2(Hi.cpu().numpy()[0], Hb.cpu().numpy()[0]) <= 2e-6


def test_config2_full_protocol_full_size_invariants_and_half_storage(ctx):
    """The whole config-2 protocol at full size (160x40x1, 20,000 relax + 10,000 dynamics RK4 steps,
    the work bench-class runs do) on the CUDA path: properties that hold at any size — |m| = 1, energy
    non-increasing while relaxing (alpha > 0, constant field, uniform grid: PAPER.md:58) — and the two
    storage formats of the same tensor (full six planes vs pair-symmetric half, F3) giving the same
    <m>(t) within north_star's 1e-3."""
    wr = W.config2(batch=1, phase="relax")
    wd = W.config2(batch=1, phase="dynamics")
    tiles = H.dev_tiles(wr)
    N, ld, _ = H.assemble(ctx, tiles, "f32")
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    S = B.mt_assemble_tensor_sym(ctx, tiles, B.MT_F32, status)
    assert int(status.item()) == 0
    dt = 1e-13
    out = {}
    for name in ("full", "half"):
        pr = H.dev_problem(wr, tiles, N if name == "full" else None, "f32", ld)
        pd = H.dev_problem(wd, tiles, N if name == "full" else None, "f32", ld)
        if name == "half":
            pr.N_sym = S
            pd.N_sym = S
        m = torch.from_numpy(wr.m[:1].copy()).cuda()
        E = torch.empty((1, 5), dtype=torch.float64, device="cuda")
        energies, t = [], 0.0
        s1 = torch.zeros((200, 4), dtype=torch.float64, device="cuda")
        for k in range(10):  # 10 x 2,000 relax steps, energy in between
            B.mt_energy(ctx, pr, m, 1, E)
            energies.append(float(E[0, 4].item()))
            t, res, _ = B.mt_integrate(ctx, pr, m, 1, t, method=B.MT_RK4, dt=dt, t_end=t + 2000 * dt, sample_every=100,
                                       samples=s1[20 * k:20 * (k + 1)])
            assert res["accepted"] == 2000 and res["n_samples"] == 20
        B.mt_energy(ctx, pr, m, 1, E)
        energies.append(float(E[0, 4].item()))
        # once relaxed the energy sits still to within the fp32 tensor's rounding of H_d (~1e-8 relative)
        assert np.all(np.diff(energies) <= 1e-6 * abs(energies[-1])), energies
        assert energies[-1] < 0.03 * energies[0]
        s2 = torch.zeros((100, 4), dtype=torch.float64, device="cuda")
        _, res, _ = B.mt_integrate(ctx, pd, m, 1, 0.0, method=B.MT_RK4, dt=dt, t_end=10000 * dt, sample_every=100, samples=s2)
        assert res["accepted"] == 10000 and res["n_samples"] == 100
        mm = m.cpu().numpy()[0]
        assert np.max(np.abs(np.linalg.norm(mm, axis=0) - 1.0)) < 1e-14
        out[name] = (s1.cpu().numpy(), s2.cpu().numpy())
    assert np.max(np.abs(out["full"][0][:, 1:] - out["half"][0][:, 1:])) < 1e-3
    assert np.max(np.abs(out["full"][1][:, 1:] - out["half"][1][:, 1:])) < 1e-3
    assert np.max(np.abs(out["full"][1][-1, 1:] - out["full"][1][0, 1:])) > 0.05  # the field did move <m>
