"""Glue shared by the GPU parity tests, smoke() and bench.py: moves a Workload to the device for
the C-ABI path and to the oracle's structs for the CPU path.  No arithmetic of the method here.
"""
from __future__ import annotations

import numpy as np
import torch

from paper_2107_05364_b200 import binding as B
from paper_2107_05364_b200 import workloads as W


def dtype_code(name: str) -> int:
    return B.MT_F32 if name == "f32" else B.MT_F64


def dev_tiles(w: W.Workload, device="cuda:0") -> B.Tiles:
    has_tets = bool((w.type == 1).any())
    return B.Tiles(
        type=torch.from_numpy(w.type).to(device),
        center=torch.from_numpy(w.center).to(device),
        size=torch.from_numpy(w.size).to(device),
        verts=torch.from_numpy(w.verts).to(device) if has_tets else None,
        Ms=torch.from_numpy(w.Ms).to(device),
    )


def assemble(ctx: B.Context, tiles: B.Tiles, dtype: str, row_begin: int = 0, row_end: int | None = None,
             ld: int | None = None):
    """Returns (N [6, rows, ld] device tensor, ld, status int)."""
    n = tiles.n
    row_end = n if row_end is None else row_end
    ld = W.leading_dim(n, dtype) if ld is None else ld
    code = dtype_code(dtype)
    N = torch.empty((6, row_end - row_begin, ld), dtype=B.torch_dtype(code), device=tiles.type.device)
    status = torch.zeros(1, dtype=torch.int32, device=tiles.type.device)
    B.mt_assemble_tensor(ctx, tiles, code, row_begin, row_end, N, ld, status)
    torch.cuda.synchronize()
    return N, ld, int(status.item())


def dev_problem(w: W.Workload, tiles: B.Tiles, N, dtype: str, ld: int) -> B.Problem:
    dev = tiles.type.device
    return B.Problem(
        n=w.n, Ms=tiles.Ms, N=N, dtype=dtype_code(dtype), ld=ld,
        nbr=torch.from_numpy(w.nbr).to(dev) if w.nbr is not None else None,
        inv_d2=tuple(float(x) for x in w.inv_d2), c_ex=float(w.c_ex), c_an=float(w.c_an),
        easy=tuple(w.easy), H_a=tuple(float(x) for x in w.H_a), gamma=w.gamma, alpha_ll=w.alpha_ll,
        vol=torch.from_numpy(w.vol).to(dev),
    )


def oracle_tiles(oracle, w: W.Workload):
    return oracle.Tiles(type=w.type, center=w.center, size=w.size, verts=w.verts, Ms=w.Ms)


def oracle_problem(oracle, w: W.Workload, N=None, rows=None):
    return oracle.Problem(n=w.n, Ms=w.Ms, N=N, rows=rows, nbr=w.nbr, inv_d2=tuple(w.inv_d2), c_ex=w.c_ex,
                          c_an=w.c_an, easy=tuple(w.easy), H_a=tuple(w.H_a), gamma=w.gamma, alpha_ll=w.alpha_ll)


def rel_l2(a, b) -> float:
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def f32_ulp_distance(got_f32: np.ndarray, exact_f64: np.ndarray) -> np.ndarray:
    """|got - float32(exact)| in units of float32 ulps of the exact value."""
    ref = exact_f64.astype(np.float32)
    gi = got_f32.view(np.int32).astype(np.int64)
    ri = ref.view(np.int32).astype(np.int64)
    # map sign-magnitude to a monotone integer line
    gi = np.where(gi < 0, -(gi & 0x7FFFFFFF), gi)
    ri = np.where(ri < 0, -(ri & 0x7FFFFFFF), ri)
    return np.abs(gi - ri)
