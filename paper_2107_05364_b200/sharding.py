"""Row sharding of the demagnetisation tensor across ranks.

The tensor shards by TARGET rows: rank g assembles and keeps rows [g n / G, (g+1) n / G) — the
`row_begin, row_end` band of `mt_assemble_tensor` — with no communication (every pair is independent,
PAPER.md:126).  A field evaluation needs all of m on every rank and yields the rank's slice of H_d;
the one real exchange step is the all-gather of those slices (3 n doubles per state in total).
Host logic only: the same functions run under `gloo` on CPU (tests) and `nccl` on GPUs (bench.py).
"""
from __future__ import annotations

import torch


def row_band(rank: int, world: int, n: int) -> tuple[int, int]:
    """Rows [begin, end) owned by `rank`; bands tile [0, n) in rank order and differ by at most one row."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError("need 0 <= rank < world and n >= 0")
    return rank * n // world, (rank + 1) * n // world


def max_band_rows(world: int, n: int) -> int:
    return max(row_band(r, world, n)[1] - row_band(r, world, n)[0] for r in range(world))


def all_gather_field(dist, local: torch.Tensor, n: int, rank: int, world: int, scratch=None) -> torch.Tensor:
    """local: [B, 3, rows_of_rank] slice of a field -> [B, 3, n] on every rank, bands in rank order.

    Bands may differ by one row, so every rank contributes a buffer padded to the widest band and the
    padding is dropped on reassembly.  `scratch` (optional) is a reusable [world, B, 3, max_rows] tensor.
    """
    B = local.shape[0]
    r0, r1 = row_band(rank, world, n)
    if local.shape != (B, 3, r1 - r0):
        raise ValueError(f"rank {rank} must pass [B, 3, {r1 - r0}], got {tuple(local.shape)}")
    mr = max_band_rows(world, n)
    if scratch is None:
        scratch = torch.empty((world, B, 3, mr), dtype=local.dtype, device=local.device)
    send = local
    if r1 - r0 != mr:
        send = torch.zeros((B, 3, mr), dtype=local.dtype, device=local.device)
        send[:, :, : r1 - r0] = local
    dist.all_gather_into_tensor(scratch.view(-1), send.contiguous().view(-1))
    out = torch.empty((B, 3, n), dtype=local.dtype, device=local.device)
    for g in range(world):
        b0, b1 = row_band(g, world, n)
        out[:, :, b0:b1] = scratch[g, :, :, : b1 - b0]
    return out
