"""Row sharding of the demagnetisation tensor across ranks.

The tensor shards by TARGET rows: rank g assembles and keeps rows [g n / G, (g+1) n / G) — the
`row_begin, row_end` band of `mt_assemble_tensor` — with no communication (every pair is independent,
PAPER.md:126).  An evaluation needs all of m on every rank and yields the rank's rows; the one real
exchange step is the all-gather of those slices (3 n doubles per state in total) — of the next stage
state inside the sharded integrators (`binding.Shard`, mt.h section 8(e)), of the field in the bare
field benchmark.  All buffers are allocated once, equally padded ([world, B, 3, pad] blocks), and the
exchange is ONE `all_gather_into_tensor` in place; reassembly into [B, 3, n] is one gather through a
precomputed index.  Host logic only: the same functions run under `gloo` on CPU (tests) and `nccl` on
GPUs (bench.py).
"""
from __future__ import annotations

import numpy as np
import torch

GATHER_STATE, MAX_SCALARS = 0, 1  # binding.MT_XCHG_*


def row_band(rank: int, world: int, n: int) -> tuple[int, int]:
    """Rows [begin, end) owned by `rank`; bands tile [0, n) in rank order and differ by at most one row."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError("need 0 <= rank < world and n >= 0")
    return rank * n // world, (rank + 1) * n // world


def max_band_rows(world: int, n: int) -> int:
    return max(row_band(r, world, n)[1] - row_band(r, world, n)[0] for r in range(world))


def unpack_index(world: int, n: int, pad: int) -> torch.Tensor:
    """idx[j] = position of row j in the flattened [world * pad] block axis (owner(j) * pad + j - begin)."""
    begins = np.array([row_band(g, world, n)[0] for g in range(world)] + [n], dtype=np.int64)
    j = np.arange(n, dtype=np.int64)
    owner = np.searchsorted(begins, j, side="right") - 1
    return torch.from_numpy(owner * pad + (j - begins[owner]))


def unpack(pack: torch.Tensor, n: int, index: torch.Tensor | None = None) -> torch.Tensor:
    """pack [world, B, 3, pad] (block g = rows of rank g) -> [B, 3, n]; what the library's scatter kernel
    does on the device inside the integrators, as one torch gather (used outside timed regions)."""
    world, B, three, pad = pack.shape
    if index is None:
        index = unpack_index(world, n, pad).to(pack.device)
    flat = pack.permute(1, 2, 0, 3).reshape(B, three, world * pad)
    return flat.index_select(2, index)


def dist_exchange(dist, rank: int, group=None):
    """The exchange callback of `binding.Shard` on torch.distributed (nccl on GPUs, gloo on CPU): one
    in-place all_gather_into_tensor of the preallocated blocks / one MAX all-reduce of the two words."""
    def exchange(what: int, pack: torch.Tensor, scal: torch.Tensor, cuda_stream: int):
        def run():
            if what == GATHER_STATE:
                dist.all_gather_into_tensor(pack.view(-1), pack[rank].view(-1), group=group)
            elif what == MAX_SCALARS:
                dist.all_reduce(scal, op=dist.ReduceOp.MAX, group=group)
            else:
                raise ValueError(f"unknown exchange {what}")
        if pack.is_cuda:
            # the library launches on its ctx stream; the collective must be ordered on the same stream
            s = torch.cuda.ExternalStream(cuda_stream, device=pack.device) if cuda_stream else torch.cuda.default_stream(pack.device)
            with torch.cuda.stream(s):
                run()
        else:
            run()
    return exchange


class FieldGather:
    """All-gather of per-rank field slices [B, 3, rows_of_rank] (bench.py's multi-GPU field step) through
    preallocated, equally padded blocks; nothing is allocated per step."""

    def __init__(self, dist, rank: int, world: int, n: int, batch: int, device, dtype=torch.float64):
        self.dist, self.rank, self.world, self.n = dist, rank, world, n
        self.pad = max_band_rows(world, n)
        self.r0, self.r1 = row_band(rank, world, n)
        self.pack = torch.zeros((world, batch, 3, self.pad), dtype=dtype, device=device)
        self.index = unpack_index(world, n, self.pad).to(device)

    def gather(self, local: torch.Tensor) -> torch.Tensor:
        """Returns the gathered blocks [world, B, 3, pad] (valid on every rank); `full()` reassembles."""
        rows = self.r1 - self.r0
        if tuple(local.shape) != (self.pack.shape[1], 3, rows):
            raise ValueError(f"rank {self.rank} must pass [B, 3, {rows}], got {tuple(local.shape)}")
        self.pack[self.rank, :, :, :rows].copy_(local)
        self.dist.all_gather_into_tensor(self.pack.view(-1), self.pack[self.rank].view(-1))
        return self.pack

    def full(self) -> torch.Tensor:
        return unpack(self.pack, self.n, self.index)


def all_gather_field(dist, local: torch.Tensor, n: int, rank: int, world: int) -> torch.Tensor:
    """local: [B, 3, rows_of_rank] slice of a field -> [B, 3, n] on every rank, bands in rank order
    (convenience form: allocates; steady-state callers keep a FieldGather)."""
    fg = FieldGather(dist, rank, world, n, local.shape[0], local.device, local.dtype)
    fg.gather(local)
    return fg.full()
