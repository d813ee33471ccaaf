"""Thin ctypes binding of libmagtile.so — same names as include/mt.h, argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C-ABI; this module only turns torch
tensors into device pointers and fills the C structs.  PyTorch is used for device memory and
streams, nothing else.  There is no fallback: importing works without a GPU (so that the symbol
check can run on CPU), but `load()` raises if the library is missing and `mt_create` raises if no
CUDA device is usable.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmagtile.so")

MT_OK = 0
MT_ERR_INVALID_ARG, MT_ERR_CUDA, MT_ERR_SINGULAR_GEOMETRY = -1, -2, -3
MT_ERR_STEP_UNDERFLOW, MT_ERR_MAX_STEPS, MT_ERR_UNIMPLEMENTED = -4, -5, -6
MT_F32, MT_F64 = 0, 1
MT_RK4, MT_DP45 = 0, 1
MT_SELECT_HIST_WORDS = 1 << 20
MT_NOALLOC_MAX_N = 65536
MT_NOALLOC_SCRATCH_BYTES = 4718592
COMPONENTS = ("xx", "xy", "xz", "yy", "yz", "zz")
EXPORTS = ("mt_create", "mt_destroy", "mt_last_error", "mt_version", "mt_assemble_tensor",
           "mt_check_status", "mt_demag_field", "mt_demag_field_host", "mt_llg_rhs", "mt_integrate", "mt_energy",
           "mt_field_sweep", "mt_sparse_mask_words", "mt_threshold_value", "mt_sparse_count",
           "mt_sparse_fill", "mt_sparse_index", "mt_select_begin", "mt_select_accumulate", "mt_select_advance",
           "mt_sparse_count_band", "mt_sparse_scan", "mt_sparse_fill_band", "mt_sparse_fill_index_band",
           "mt_sparse_stream_count", "mt_sparse_stream_fill", "mt_demag_field_sparse", "mt_sym_tensor_elems", "mt_assemble_tensor_sym",
           "mt_demag_field_sym", "mt_set_assembly_mode", "mt_launch_count",
           "mt_set_demag_variant", "mt_set_step_control", "mt_set_resident_mode", "mt_profile_begin", "mt_profile_end", "mt_measure_peak",
           "mt_demag_field_noalloc")


class MtError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libmagtile error {code}: {msg}")
        self.code = code


class _Tiles(C.Structure):
    _fields_ = [("n", C.c_int64), ("type", C.c_void_p), ("center", C.c_void_p), ("size", C.c_void_p),
                ("verts", C.c_void_p), ("Ms", C.c_void_p)]


class _Problem(C.Structure):
    _fields_ = [
        ("n", C.c_int64), ("N", C.c_void_p), ("dtype", C.c_int), ("ld", C.c_int64), ("Ms", C.c_void_p),
        ("nbr", C.c_void_p), ("inv_d2", C.c_double * 3),
        ("c_ex", C.c_void_p), ("c_ex_scalar", C.c_double),
        ("c_an", C.c_void_p), ("c_an_scalar", C.c_double),
        ("easy", C.c_void_p), ("easy_const", C.c_double * 3),
        ("H_a", C.c_void_p), ("H_a_const", C.c_double * 3),
        ("gamma", C.c_double), ("alpha_ll", C.c_double), ("vol", C.c_void_p), ("N_sparse", C.c_void_p),
        ("N_sym", C.c_void_p), ("shard", C.c_void_p),
    ]


MT_XCHG_GATHER_STATE, MT_XCHG_MAX_SCALARS = 0, 1
EXCHANGE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int, C.c_void_p)
ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p)


class _Shard(C.Structure):
    _fields_ = [("rank", C.c_int), ("world", C.c_int), ("slice_pad", C.c_int64), ("pack", C.c_void_p),
                ("scal", C.c_void_p), ("exchange", EXCHANGE_FN), ("user", C.c_void_p)]


class _Sym(C.Structure):
    _fields_ = [("n", C.c_int64), ("dtype", C.c_int), ("data", C.c_void_p)]


class _Sparse(C.Structure):
    _fields_ = [("n", C.c_int64), ("n_rows", C.c_int64), ("dtype", C.c_int), ("nw", C.c_int64),
                ("row_ptr", C.c_void_p), ("mask", C.c_void_p), ("vals", C.c_void_p), ("cols16", C.c_void_p), ("panel_ptr", C.c_void_p)]


class _SelectState(C.Structure):
    _fields_ = [("dtype", C.c_int), ("fraction", C.c_double), ("hi", C.c_int), ("prefix", C.c_ulonglong),
                ("k", C.c_ulonglong), ("count", C.c_ulonglong), ("done", C.c_int), ("tau", C.c_double)]


class _Opts(C.Structure):
    _fields_ = [
        ("method", C.c_int), ("dt", C.c_double), ("t_end", C.c_double), ("max_steps", C.c_int64),
        ("rtol", C.c_double), ("atol", C.c_double), ("torque_tol", C.c_double),
        ("renormalize", C.c_int), ("sample_every", C.c_int64), ("sample_dt", C.c_double),
    ]


class _Result(C.Structure):
    _fields_ = [("accepted", C.c_int64), ("rejected", C.c_int64), ("rhs_calls", C.c_int64),
                ("n_samples", C.c_int64), ("t", C.c_double), ("dt_last", C.c_double),
                ("max_torque", C.c_double)]


_lib = None


def load() -> C.CDLL:
    """dlopen the in-tree library; fails loudly when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2107_05364_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.mt_last_error.restype = C.c_char_p
        lib.mt_last_error.argtypes = [C.c_void_p]
        lib.mt_version.restype = C.c_char_p
        lib.mt_launch_count.restype = C.c_int64
        lib.mt_launch_count.argtypes = [C.c_void_p]
        lib.mt_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p]
        lib.mt_destroy.argtypes = [C.c_void_p]
        lib.mt_set_demag_variant.argtypes = [C.c_void_p, C.c_int]
        lib.mt_set_assembly_mode.argtypes = [C.c_void_p, C.c_int]
        lib.mt_set_step_control.argtypes = [C.c_void_p, C.c_int]
        lib.mt_set_resident_mode.argtypes = [C.c_void_p, C.c_int]
        lib.mt_check_status.argtypes = [C.c_void_p, C.c_void_p]
        lib.mt_profile_begin.argtypes = [C.c_void_p]
        lib.mt_measure_peak.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int64, C.POINTER(C.c_double)]
        lib.mt_profile_end.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        lib.mt_assemble_tensor.argtypes = [C.c_void_p, C.POINTER(_Tiles), C.c_int, C.c_int64, C.c_int64,
                                           C.c_void_p, C.c_int64, C.c_void_p]
        lib.mt_demag_field.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                       C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        lib.mt_demag_field_host.argtypes = lib.mt_demag_field.argtypes
        lib.mt_llg_rhs.argtypes = [C.c_void_p, C.POINTER(_Problem), C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        lib.mt_integrate.argtypes = [C.c_void_p, C.POINTER(_Problem), C.POINTER(_Opts), C.c_void_p, C.c_int,
                                     C.POINTER(C.c_double), C.c_void_p, C.c_int64, C.POINTER(_Result)]
        lib.mt_sparse_mask_words.restype = C.c_int64
        lib.mt_sparse_mask_words.argtypes = [C.c_int64]
        lib.mt_threshold_value.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                           C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        lib.mt_sparse_count.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                        C.c_double, C.c_void_p, C.POINTER(C.c_int64)]
        lib.mt_sparse_fill.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                       C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.mt_select_begin.argtypes = [C.c_void_p, C.POINTER(_SelectState), C.c_int, C.c_double, C.c_void_p]
        lib.mt_select_accumulate.argtypes = [C.c_void_p, C.POINTER(_SelectState), C.c_void_p, C.c_int64, C.c_int64,
                                             C.c_int64, C.c_void_p]
        lib.mt_select_advance.argtypes = [C.c_void_p, C.POINTER(_SelectState), C.c_void_p]
        lib.mt_sparse_count_band.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                             C.c_double, C.c_int64, C.c_int64, C.c_void_p]
        lib.mt_sparse_scan.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
        lib.mt_sparse_fill_band.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                            C.c_double, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.mt_sparse_fill_index_band.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64, C.c_int64,
                                                  C.c_double, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p,
                                                  C.c_void_p, C.c_void_p, C.c_void_p]
        lib.mt_sparse_index.argtypes = [C.c_void_p, C.POINTER(_Sparse), C.c_void_p, C.c_void_p]
        lib.mt_sparse_stream_count.argtypes = [C.c_void_p, C.POINTER(_Tiles), C.c_int, C.c_double, C.c_int64, C.c_int64,
                                               C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, ALLREDUCE_FN,
                                               C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        lib.mt_sparse_stream_fill.argtypes = [C.c_void_p, C.POINTER(_Tiles), C.c_int, C.c_double, C.c_int64, C.c_int64,
                                              C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                              C.c_void_p, C.c_void_p, C.c_void_p]
        lib.mt_demag_field_sparse.argtypes = [C.c_void_p, C.POINTER(_Sparse), C.c_void_p, C.c_void_p, C.c_int,
                                              C.c_void_p]
        lib.mt_sym_tensor_elems.restype = C.c_int64
        lib.mt_sym_tensor_elems.argtypes = [C.c_int64, C.c_int]
        lib.mt_assemble_tensor_sym.argtypes = [C.c_void_p, C.POINTER(_Tiles), C.c_int, C.c_void_p, C.c_void_p]
        lib.mt_demag_field_sym.argtypes = [C.c_void_p, C.POINTER(_Sym), C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        lib.mt_energy.argtypes = [C.c_void_p, C.POINTER(_Problem), C.c_void_p, C.c_int, C.c_void_p]
        lib.mt_field_sweep.argtypes = [C.c_void_p, C.POINTER(_Problem), C.POINTER(_Opts), C.c_void_p, C.c_int64,
                                       C.c_void_p, C.c_int, C.c_void_p, C.POINTER(_Result)]
        lib.mt_demag_field_noalloc.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64,
                                               C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_char_p, C.c_int64]
        _lib = lib
    return _lib


def _ptr(t, dtype=None):
    """Device (or pinned host) pointer of a contiguous torch tensor; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected {dtype}, got {t.dtype}")
    return t.data_ptr()


def torch_dtype(dtype: int):
    return torch.float32 if dtype == MT_F32 else torch.float64


class Context:
    """Owns an mt_ctx bound to a device and a torch stream."""

    def __init__(self, device: int = 0, stream: torch.cuda.Stream | None = None):
        if not torch.cuda.is_available():
            raise MtError(MT_ERR_CUDA, "no CUDA device: libmagtile has no CPU fallback")
        self.lib = load()
        self.device = device
        self.stream = stream if stream is not None else torch.cuda.current_stream(device)
        h = C.c_void_p()
        rc = self.lib.mt_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream))
        if rc != MT_OK:
            raise MtError(rc, "mt_create failed")
        self.h = h

    def check(self, rc: int, allow=()):
        if rc != MT_OK and rc not in allow:
            raise MtError(rc, self.lib.mt_last_error(self.h).decode())
        return rc

    def close(self):
        if getattr(self, "h", None):
            self.lib.mt_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launches(self) -> int:
        return int(self.lib.mt_launch_count(self.h))


def mt_create(device: int = 0, stream=None) -> Context:
    return Context(device, stream)


def mt_destroy(ctx: Context):
    ctx.close()


def mt_version() -> str:
    return load().mt_version().decode()


def mt_launch_count(ctx: Context) -> int:
    return ctx.launches


def mt_set_demag_variant(ctx: Context, variant: int):
    ctx.check(ctx.lib.mt_set_demag_variant(ctx.h, variant))


def mt_set_step_control(ctx: Context, mode: int):
    """DP45 controller: 0 auto (device for small unsharded problems), 1 host, 2 device."""
    ctx.check(ctx.lib.mt_set_step_control(ctx.h, mode))


def mt_set_resident_mode(ctx: Context, mode: int):
    """RK4 with the tensor resident in shared memory: 0 auto (when it fits), 1 never, 2 required."""
    ctx.check(ctx.lib.mt_set_resident_mode(ctx.h, mode))


def mt_profile_begin(ctx: Context):
    ctx.check(ctx.lib.mt_profile_begin(ctx.h))


def mt_profile_end(ctx: Context):
    """Returns (summed device time of the demag field kernel in ms, launches timed)."""
    ms, cnt = C.c_double(0.0), C.c_int64(0)
    ctx.check(ctx.lib.mt_profile_end(ctx.h, C.byref(ms), C.byref(cnt)))
    return ms.value, cnt.value


MT_PEAK_DFMA, MT_PEAK_FFMA, MT_PEAK_FFMA2, MT_PEAK_MMA_TF32, MT_PEAK_HBM_READ = 0, 1, 2, 3, 4


def mt_measure_peak(ctx: Context, kind: int, buf: torch.Tensor | None = None):
    """Returns (rate, ms) of one roofline-denominator microbenchmark (see mt.h)."""
    out = (C.c_double * 2)()
    nbytes = int(buf.numel() * buf.element_size()) if buf is not None else 0
    ctx.check(ctx.lib.mt_measure_peak(ctx.h, kind, buf.data_ptr() if buf is not None else None, nbytes, out))
    return out[0], out[1]


@dataclass
class Tiles:
    """A0: device-resident tile geometry (torch tensors on the ctx's device)."""
    type: torch.Tensor      # [n] int32
    center: torch.Tensor    # [n, 3] float64
    size: torch.Tensor      # [n, 3] float64
    verts: torch.Tensor | None  # [n, 4, 3] float64 or None
    Ms: torch.Tensor        # [n] float64

    @property
    def n(self) -> int:
        return int(self.type.shape[0])

    def _c(self) -> _Tiles:
        return _Tiles(self.n, _ptr(self.type, torch.int32), _ptr(self.center, torch.float64),
                      _ptr(self.size, torch.float64), _ptr(self.verts, torch.float64),
                      _ptr(self.Ms, torch.float64))


def mt_assemble_tensor(ctx: Context, tiles: Tiles, dtype: int, row_begin: int, row_end: int,
                       out: torch.Tensor, ld: int, status_flag: torch.Tensor | None = None):
    """out: [6, row_end-row_begin, ld] tensor of the matching dtype on the device."""
    t = tiles._c()
    ctx.check(ctx.lib.mt_assemble_tensor(ctx.h, C.byref(t), dtype, row_begin, row_end,
                                         _ptr(out, torch_dtype(dtype)), ld, _ptr(status_flag, torch.int32)))


def mt_check_status(ctx: Context, status_flag: torch.Tensor, allow=()):
    """Synchronises and raises MtError(MT_ERR_SINGULAR_GEOMETRY / MT_ERR_INVALID_ARG) when the assembly flagged."""
    return ctx.check(ctx.lib.mt_check_status(ctx.h, _ptr(status_flag, torch.int32)), allow=allow)


def mt_demag_field(ctx: Context, N: torch.Tensor, dtype: int, n: int, n_rows: int, ld: int,
                   Ms: torch.Tensor, m: torch.Tensor, batch: int, Hd: torch.Tensor):
    ctx.check(ctx.lib.mt_demag_field(ctx.h, _ptr(N, torch_dtype(dtype)), dtype, n, n_rows, ld,
                                     _ptr(Ms, torch.float64), _ptr(m, torch.float64), batch,
                                     _ptr(Hd, torch.float64)))


def mt_demag_field_host(ctx: Context, N: torch.Tensor, dtype: int, n: int, n_rows: int, ld: int,
                        Ms: torch.Tensor, m_host: torch.Tensor, batch: int, Hd_host: torch.Tensor):
    """m_host / Hd_host are HOST tensors (pinned recommended); synchronises before returning."""
    if m_host.is_cuda or Hd_host.is_cuda:
        raise ValueError("mt_demag_field_host takes host tensors")
    ctx.check(ctx.lib.mt_demag_field_host(ctx.h, _ptr(N, torch_dtype(dtype)), dtype, n, n_rows, ld,
                                          _ptr(Ms, torch.float64), _ptr(m_host, torch.float64), batch,
                                          _ptr(Hd_host, torch.float64)))


def mt_demag_field_noalloc(device: int, cuda_stream: int, N: torch.Tensor, dtype: int, n: int, n_rows: int, ld: int,
                           Ms: torch.Tensor, m: torch.Tensor, Hd: torch.Tensor):
    """One state's field with no allocation anywhere (mt.h): no Context; scratch is the library's static device
    array (n, n_rows <= MT_NOALLOC_MAX_N; calls that overlap on the GPU race on it).  `cuda_stream` is the raw
    stream handle (torch.cuda.Stream.cuda_stream; 0 = legacy default stream).  Enqueues only."""
    err = C.create_string_buffer(256)
    rc = load().mt_demag_field_noalloc(device, C.c_void_p(cuda_stream), _ptr(N, torch_dtype(dtype)), dtype, n, n_rows,
                                       ld, _ptr(Ms, torch.float64), _ptr(m, torch.float64), _ptr(Hd, torch.float64),
                                       err, len(err))
    if rc != MT_OK:
        raise MtError(rc, err.value.decode(errors="replace"))


class Shard:
    """mt_shard (row sharding, mt.h section 8(e)): this rank's place in the partition, the all-gather
    buffer `pack` [world, batch, 3, slice_pad] and the two reduction words `scal`, both preallocated
    here once, and the exchange callback.  `exchange(what, pack, scal, cuda_stream)` must enqueue the
    collective on `cuda_stream` (an int; 0 = legacy default stream): what == MT_XCHG_GATHER_STATE:
    all-gather of pack[rank] into pack, in place; MT_XCHG_MAX_SCALARS: element-wise max of scal over
    the ranks.  `sharding.dist_exchange` builds one from torch.distributed."""

    def __init__(self, rank: int, world: int, n: int, batch: int, device, exchange):
        if not (0 <= rank < world):
            raise ValueError("need 0 <= rank < world")
        self.rank, self.world, self.n, self.batch = rank, world, n, batch
        self.slice_pad = (n + world - 1) // world
        self.pack = torch.zeros((world, batch, 3, self.slice_pad), dtype=torch.float64, device=device)
        self.scal = torch.zeros(2, dtype=torch.int64, device=device)
        self.error = None

        def _cb(_user, what, stream):
            try:
                exchange(int(what), self.pack, self.scal, int(stream or 0))
                return 0
            except Exception as exc:  # nothing may propagate through the C frames
                self.error = exc
                return 1

        self._cb = EXCHANGE_FN(_cb)
        self._c_struct = _Shard(rank, world, self.slice_pad, self.pack.data_ptr(), self.scal.data_ptr(), self._cb, None)

    @property
    def rows(self) -> tuple[int, int]:
        return self.rank * self.n // self.world, (self.rank + 1) * self.n // self.world


@dataclass
class Problem:
    """mt_problem: tensor + local-term parameters.  Scalars or device tensors for c_ex, c_an;
    3-vectors or [n, 3] device tensors for easy, H_a."""
    n: int
    Ms: torch.Tensor
    N: torch.Tensor | None = None
    dtype: int = MT_F32
    ld: int = 0
    nbr: torch.Tensor | None = None
    inv_d2: tuple = (0.0, 0.0, 0.0)
    c_ex: object = 0.0
    c_an: object = 0.0
    easy: object = (0.0, 0.0, 1.0)
    H_a: object = (0.0, 0.0, 0.0)
    gamma: float = 1.0
    alpha_ll: float = 0.0
    vol: torch.Tensor | None = None
    N_sparse: object = None  # SparseTensor (F1): used for the demagnetising term instead of N
    N_sym: object = None     # SymTensor (F3): pair-symmetric half, congruent cuboid meshes only
    shard: object = None     # Shard: N (or N_sparse) holds this rank's row band only

    def _c(self) -> _Problem:
        s = _Problem()
        if self.N_sparse is not None:
            self._sparse_c = self.N_sparse._c()  # keep the struct alive while the call runs
            s.N_sparse = C.addressof(self._sparse_c)
        if self.N_sym is not None:
            self._sym_c = self.N_sym._c()
            s.N_sym = C.addressof(self._sym_c)
        if self.shard is not None:
            s.shard = C.addressof(self.shard._c_struct)
        s.n = self.n
        s.N = _ptr(self.N, torch_dtype(self.dtype)) if self.N is not None else None
        s.dtype, s.ld = self.dtype, self.ld
        s.Ms = _ptr(self.Ms, torch.float64)
        s.nbr = _ptr(self.nbr, torch.int32)
        s.inv_d2 = (C.c_double * 3)(*self.inv_d2)
        for name in ("c_ex", "c_an"):
            v = getattr(self, name)
            if isinstance(v, torch.Tensor):
                setattr(s, name, _ptr(v, torch.float64))
            else:
                setattr(s, name, None)
                setattr(s, name + "_scalar", float(v))
        for name in ("easy", "H_a"):
            v = getattr(self, name)
            if isinstance(v, torch.Tensor):
                setattr(s, name, _ptr(v, torch.float64))
            else:
                setattr(s, name, None)
                setattr(s, name + "_const", (C.c_double * 3)(*[float(x) for x in v]))
        s.gamma, s.alpha_ll = float(self.gamma), float(self.alpha_ll)
        s.vol = _ptr(self.vol, torch.float64)
        return s


def mt_llg_rhs(ctx: Context, prob: Problem, m: torch.Tensor, batch: int, dmdt: torch.Tensor,
               heff: torch.Tensor | None = None):
    p = prob._c()
    ctx.check(ctx.lib.mt_llg_rhs(ctx.h, C.byref(p), _ptr(m, torch.float64), batch,
                                 _ptr(dmdt, torch.float64), _ptr(heff, torch.float64)))


def mt_integrate(ctx: Context, prob: Problem, m: torch.Tensor, batch: int, t0: float, *, method: int,
                 dt: float, t_end: float, max_steps: int = 0, rtol: float = 1e-6, atol: float = 1e-8,
                 torque_tol: float = 0.0, renormalize: bool = True, sample_every: int = 0,
                 sample_dt: float = 0.0, samples: torch.Tensor | None = None, allow=()):
    """Advances m in place; returns (t, result dict, return code)."""
    p = prob._c()
    o = _Opts(method, dt, t_end, max_steps, rtol, atol, torque_tol, int(renormalize), sample_every, sample_dt)
    res = _Result()
    t = C.c_double(t0)
    cap = int(samples.shape[0]) if samples is not None else 0
    rc = ctx.check(ctx.lib.mt_integrate(ctx.h, C.byref(p), C.byref(o), _ptr(m, torch.float64), batch,
                                        C.byref(t), _ptr(samples, torch.float64), cap, C.byref(res)),
                   allow=allow)
    return t.value, {k: getattr(res, k) for k, _ in _Result._fields_}, rc


def mt_energy(ctx: Context, prob: Problem, m: torch.Tensor, batch: int, E_out: torch.Tensor):
    """E_out[batch][5] (device): E_demag, E_exch, E_anis, E_zeeman, E_total."""
    p = prob._c()
    ctx.check(ctx.lib.mt_energy(ctx.h, C.byref(p), _ptr(m, torch.float64), batch, _ptr(E_out, torch.float64)))


def mt_field_sweep(ctx: Context, prob: Problem, fields, m: torch.Tensor, batch: int, rows: torch.Tensor, *,
                   method: int, dt: float, t_end: float, max_steps: int = 0, rtol: float = 1e-6,
                   atol: float = 1e-8, torque_tol: float = 0.0, renormalize: bool = True, allow=()):
    """fields: host sequence [k][3]; rows (device) [k][batch][8]; m advanced in place.  Returns the
    summed counters and the return code."""
    p = prob._c()
    o = _Opts(method, dt, t_end, max_steps, rtol, atol, torque_tol, int(renormalize), 0, 0.0)
    flat = [float(x) for row in fields for x in row]
    nf = len(flat) // 3
    arr = (C.c_double * max(1, len(flat)))(*flat)
    res = _Result()
    rc = ctx.check(ctx.lib.mt_field_sweep(ctx.h, C.byref(p), C.byref(o), arr, nf, _ptr(m, torch.float64), batch,
                                          _ptr(rows, torch.float64), C.byref(res)), allow=allow)
    return {k: getattr(res, k) for k, _ in _Result._fields_}, rc


@dataclass
class SparseTensor:
    """mt_sparse_tensor (F1): bitmap rows of a thresholded tensor; device tensors owned here."""
    n: int
    n_rows: int
    dtype: int
    nw: int
    row_ptr: torch.Tensor  # [6*n_rows + 1] int64
    mask: torch.Tensor     # [6, n_rows, nw] int32 (bit patterns of uint32)
    vals: torch.Tensor     # [nnz]
    nnz: int = 0
    tau: float = 0.0
    cols16: object = None  # [nnz] uint16 index rows (mt_sparse_index) or None; the mask may be dropped then
    panel_ptr: object = None  # n > 65536: [6*n_rows, ceil(n/65536)-1] int64 panel starts

    def _c(self) -> _Sparse:
        return _Sparse(self.n, self.n_rows, self.dtype, self.nw, _ptr(self.row_ptr, torch.int64),
                       _ptr(self.mask, torch.int32) if self.mask is not None else None,
                       _ptr(self.vals, torch_dtype(self.dtype)),
                       _ptr(self.cols16, torch.uint16) if self.cols16 is not None else None,
                       _ptr(self.panel_ptr, torch.int64) if self.panel_ptr is not None else None)

    def nbytes(self) -> int:
        """Bytes one field evaluation streams: values + the index the kernel walks (16-bit columns if present)."""
        idx = self.cols16.numel() * 2 if self.cols16 is not None else self.mask.numel() * 4
        if self.cols16 is not None and self.panel_ptr is not None:
            idx += self.panel_ptr.numel() * 8
        return self.row_ptr.numel() * 8 + idx + self.vals.numel() * self.vals.element_size()


def mt_threshold_value(ctx: Context, N: torch.Tensor, dtype: int, n: int, n_rows: int, ld: int, fraction: float):
    """Returns (tau, number of non-zero elements counted with multiplicity)."""
    tau, cnt = C.c_double(), C.c_int64()
    ctx.check(ctx.lib.mt_threshold_value(ctx.h, _ptr(N, torch_dtype(dtype)), dtype, n, n_rows, ld, float(fraction),
                                         C.byref(tau), C.byref(cnt)))
    return tau.value, cnt.value


def mt_sparse_build(ctx: Context, N: torch.Tensor, dtype: int, n: int, n_rows: int, ld: int, tau: float) -> SparseTensor:
    """mt_sparse_count + allocation (torch) + mt_sparse_fill."""
    dev = N.device
    row_ptr = torch.empty(6 * n_rows + 1, dtype=torch.int64, device=dev)
    nnz = C.c_int64()
    ctx.check(ctx.lib.mt_sparse_count(ctx.h, _ptr(N, torch_dtype(dtype)), dtype, n, n_rows, ld, float(tau),
                                      _ptr(row_ptr), C.byref(nnz)))
    nw = int(ctx.lib.mt_sparse_mask_words(n))
    mask = torch.empty((6, n_rows, nw), dtype=torch.int32, device=dev)
    vals = torch.empty(max(1, nnz.value), dtype=torch_dtype(dtype), device=dev)
    ctx.check(ctx.lib.mt_sparse_fill(ctx.h, _ptr(N, torch_dtype(dtype)), dtype, n, n_rows, ld, float(tau),
                                     _ptr(row_ptr), _ptr(mask), _ptr(vals)))
    return SparseTensor(n, n_rows, dtype, nw, row_ptr, mask, vals, nnz=nnz.value, tau=float(tau))


def mt_sparse_build_streamed(ctx: Context, tiles: Tiles, dtype: int, fraction: float, band_rows: int,
                             status_flag: torch.Tensor | None = None, tau: float | None = None,
                             row_begin: int = 0, row_end: int | None = None, allreduce=None,
                             index: bool = False, keep_mask: bool = True) -> SparseTensor:
    """Thresholded tensor of `tiles` without ever holding the dense tensor: every pass (one per radix
    digit of the selection, one for the counts, one for the fill) assembles the tensor again band by
    band into one [6, band_rows, ld] buffer.  Two library calls, mt_sparse_stream_count and
    mt_sparse_stream_fill (the band loop and the passes run inside the library); this function only
    allocates.  `tau` given: the selection passes are skipped.

    Row-sharded (multi-GPU): `row_begin, row_end` = this rank's target rows; the
    result then has n_rows = row_end - row_begin.  The threshold is a property of the WHOLE tensor: after
    every selection pass `allreduce(hist)` must sum the 2,048-bin int64 device histogram over the ranks in
    place (e.g. `lambda h: dist.all_reduce(h)`: 16 KB, the one exchange step of the build), so that every
    rank fixes the same digit.

    `index=True`: the fill pass writes the index rows (16-bit columns, panel offsets) as well;
    `keep_mask=False` then leaves the bitmap out altogether (values + columns only)."""
    if not index and not keep_mask:
        raise ValueError("keep_mask=False needs index=True")
    n = tiles.n
    row_end = n if row_end is None else row_end
    n_loc = row_end - row_begin
    dev = tiles.type.device
    tdt = torch_dtype(dtype)
    vec = 4 if dtype == MT_F32 else 2
    ld = (n + vec - 1) // vec * vec
    band = torch.empty(6 * band_rows * ld, dtype=tdt, device=dev)
    row_ptr = torch.empty(6 * n_loc + 1, dtype=torch.int64, device=dev)
    hist = torch.empty(MT_SELECT_HIST_WORDS, dtype=torch.int64, device=dev) if allreduce is not None else None
    err = []

    def _cb(_user, _hist, _stream):
        try:
            allreduce(hist)
            return 0
        except Exception as exc:  # nothing may propagate through the C frames
            err.append(exc)
            return 1

    cb = ALLREDUCE_FN(_cb) if allreduce is not None else ALLREDUCE_FN()
    t = tiles._c()
    tau_c = C.c_double(float(tau) if tau is not None else 0.0)
    nnz = C.c_int64()
    rc = ctx.lib.mt_sparse_stream_count(ctx.h, C.byref(t), dtype, float(fraction) if tau is None else -1.0, row_begin,
                                        row_end, _ptr(band, tdt), band_rows, ld, _ptr(row_ptr), _ptr(hist), cb, None,
                                        _ptr(status_flag, torch.int32), C.byref(tau_c), C.byref(nnz))
    if err:
        raise err[0]
    ctx.check(rc)
    tau = tau_c.value
    nw = int(ctx.lib.mt_sparse_mask_words(n))
    mask = torch.empty((6, n_loc, nw), dtype=torch.int32, device=dev) if keep_mask else None
    vals = torch.empty(max(1, nnz.value), dtype=tdt, device=dev)
    panels = (n + 65535) // 65536
    cols = torch.empty(max(1, nnz.value), dtype=torch.uint16, device=dev) if index else None
    pp = torch.empty((6 * n_loc, panels - 1), dtype=torch.int64, device=dev) if index and panels > 1 else None
    ctx.check(ctx.lib.mt_sparse_stream_fill(ctx.h, C.byref(t), dtype, float(tau), row_begin, row_end, _ptr(band, tdt),
                                            band_rows, ld, _ptr(row_ptr), _ptr(mask), _ptr(vals), _ptr(cols), _ptr(pp),
                                            _ptr(status_flag, torch.int32)))
    return SparseTensor(n, n_loc, dtype, nw, row_ptr, mask, vals, nnz=nnz.value, tau=float(tau), cols16=cols,
                        panel_ptr=pp)


def mt_sparse_index(ctx: Context, S: SparseTensor, drop_mask: bool = False) -> SparseTensor:
    """Adds the index rows (16-bit column of every packed value) to S; the field kernel then walks them."""
    cols = torch.empty(max(1, S.nnz), dtype=torch.uint16, device=S.vals.device)
    panels = (S.n + 65535) // 65536
    pp = (torch.empty((6 * S.n_rows, panels - 1), dtype=torch.int64, device=S.vals.device) if panels > 1 else None)
    s = S._c()
    ctx.check(ctx.lib.mt_sparse_index(ctx.h, C.byref(s), _ptr(cols, torch.uint16), _ptr(pp, torch.int64)))
    S.cols16 = cols
    S.panel_ptr = pp
    if drop_mask:
        ctx.stream.synchronize()  # the index kernel reads the mask
        S.mask = None
    return S


def mt_demag_field_sparse(ctx: Context, S: SparseTensor, Ms: torch.Tensor, m: torch.Tensor, batch: int,
                          Hd: torch.Tensor):
    s = S._c()
    ctx.check(ctx.lib.mt_demag_field_sparse(ctx.h, C.byref(s), _ptr(Ms, torch.float64), _ptr(m, torch.float64),
                                            batch, _ptr(Hd, torch.float64)))


@dataclass
class SymTensor:
    """mt_sym_tensor (F3): the kept half in the tiled layout; `data` is a flat device tensor."""
    n: int
    dtype: int
    data: torch.Tensor

    def _c(self) -> _Sym:
        return _Sym(self.n, self.dtype, _ptr(self.data, torch_dtype(self.dtype)))


def mt_assemble_tensor_sym(ctx: Context, tiles: Tiles, dtype: int, status_flag: torch.Tensor | None = None) -> SymTensor:
    """Allocates (torch) and assembles the pair-symmetric half; check status_flag & 2 == 0 afterwards."""
    elems = int(ctx.lib.mt_sym_tensor_elems(tiles.n, dtype))
    data = torch.empty(elems, dtype=torch_dtype(dtype), device=tiles.type.device)
    t = tiles._c()
    ctx.check(ctx.lib.mt_assemble_tensor_sym(ctx.h, C.byref(t), dtype, _ptr(data), _ptr(status_flag, torch.int32)))
    return SymTensor(tiles.n, dtype, data)


def mt_demag_field_sym(ctx: Context, S: SymTensor, Ms: torch.Tensor, m: torch.Tensor, batch: int, Hd: torch.Tensor):
    s = S._c()
    ctx.check(ctx.lib.mt_demag_field_sym(ctx.h, C.byref(s), _ptr(Ms, torch.float64), _ptr(m, torch.float64), batch,
                                         _ptr(Hd, torch.float64)))


def mt_set_assembly_mode(ctx: Context, mode: int):
    """0: closed form everywhere (default, the paper's method); 1: far-field-stable (F2)."""
    ctx.check(ctx.lib.mt_set_assembly_mode(ctx.h, mode))
