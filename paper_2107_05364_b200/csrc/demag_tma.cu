// demag_tma.cu — A4/A7, TMA bulk-tensor pipeline variant of H_d = -N.(Ms m) ("demag_tma").
//
// PAPER.md:17,122,138 name this product as the dominant cost; PAPER.md:145 moves it to CUDA.  The
// kernel is HBM-bound: per call it must stream the six component planes once.
//
// Shape.  A persistent grid of P = (#SMs) CTAs.  The work is the flattened space of tiles
// (row group g of RT target rows) x (column chunk k of CT source columns); CTA c owns the contiguous
// range [T c / P, T (c+1) / P) of it, so every SM streams the same number of bytes (+-1 tile) whatever
// n is.  One producer thread issues, per tile, ONE 3-D TMA box {CT, RT, 6} of the tensor (all six
// planes; out-of-range rows/columns are zero-filled by the hardware, which is the ragged-tail
// handling) and one 2-D box {CT, 3B} of the staged magnetisation M into a ring of STAGES shared
// memory buffers guarded by full/empty mbarriers; eight consumer warps (warp w owns rows
// w*RW .. w*RW+RW-1 of the group) multiply out of shared memory.  The producer is lane 0 of warp 0,
// which tops the ring up (non-blocking probe of the empty barriers) before each of its own tiles:
// a ninth warp would cap every thread at 168 registers (three warps on one SM sub-partition), too
// few for the B = 8 accumulators.  Bytes in flight per SM = the ring
// (up to ~200 KB), independent of registers and occupancy.
//
// Arithmetic (Q19): fp32 tensors: fp32 products, fp32 partial sums over ONE tile (at most
// CT/32*4*3 = 96 terms per lane), then fp64; fp64 tensors: DFMA throughout.  Batches of 5..8 states
// on fp32 tensors use `demag_tma_f32x2_kernel` below (packed FFMA2, the only way to the full FP32
// rate on sm_100a: a three-register FFMA issues every other cycle per scheduler).  Lanes are combined
// with a fixed xor butterfly; a group finished inside one CTA goes straight to the fused epilogue
// (epilogue.cuh); a group split between CTAs leaves per-CTA partial sums, and the CTA that completes the
// group's chunk count adds them in CTA order and runs the epilogue (finish_split_group: nobody waits, the
// order of the sum does not depend on who arrives last) — bitwise reproducible for a given (n, n_rows,
// #SMs), in ONE launch (a second, fix-up launch cost 5-10 us per call: r06, problems of 1,000-8,000 tiles).
#include <cuda.h>
#include <string.h>

#include "epilogue.cuh"
#include "mbar.cuh"

namespace {

constexpr int kConsumerWarps = 8;
constexpr int kMaxDevices = 64;  // device ordinals tracked by the per-device attribute flags (power of two)
// shape of the packed-FMA batched kernel (see demag_tma_f32x2_kernel)
#ifndef MT_B8_WARPS
#define MT_B8_WARPS 8   /* measured at N = 32,768, B = 8 (r01): 8/128/3 4.55 ms; 12/64/4 5.04; 8/64/6 6.2 */
#define MT_B8_CT 128
#define MT_B8_STAGES 3
#endif
#ifndef MT_B4_WARPS
#define MT_B4_WARPS 8
#define MT_B4_CT 128 /* box width; a tile is two boxes */
#endif
constexpr int kThreads = kConsumerWarps * 32;

template <typename T> struct Vec;
template <> struct Vec<float> { typedef float4 type; static constexpr int W = 4; };
template <> struct Vec<double> { typedef double2 type; static constexpr int W = 2; };

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2,
                                            uint32_t bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(bar), "l"(policy)
      : "memory");
}

__device__ __forceinline__ void fma3(float acc[3], const float4 v[6], const float4 m[3]) {
#define MT_BLK(q)                                                            \
  acc[0] = fmaf(v[0].q, m[0].q, fmaf(v[1].q, m[1].q, fmaf(v[2].q, m[2].q, acc[0]))); \
  acc[1] = fmaf(v[1].q, m[0].q, fmaf(v[3].q, m[1].q, fmaf(v[4].q, m[2].q, acc[1]))); \
  acc[2] = fmaf(v[2].q, m[0].q, fmaf(v[4].q, m[1].q, fmaf(v[5].q, m[2].q, acc[2])));
  MT_BLK(x) MT_BLK(y) MT_BLK(z) MT_BLK(w)
#undef MT_BLK
}
__device__ __forceinline__ void fma3(double acc[3], const double2 v[6], const double2 m[3]) {
#define MT_BLK(q)                                                        \
  acc[0] = fma(v[0].q, m[0].q, fma(v[1].q, m[1].q, fma(v[2].q, m[2].q, acc[0]))); \
  acc[1] = fma(v[1].q, m[0].q, fma(v[3].q, m[1].q, fma(v[4].q, m[2].q, acc[1]))); \
  acc[2] = fma(v[2].q, m[0].q, fma(v[4].q, m[1].q, fma(v[5].q, m[2].q, acc[2])));
  MT_BLK(x) MT_BLK(y)
#undef MT_BLK
}

template <typename T, bool Direct> struct RunSel { typedef T type; };
template <typename T> struct RunSel<T, true> { typedef char type; };

#ifndef MT_TMA_MIN_TILES_PER_SM
#define MT_TMA_MIN_TILES_PER_SM 9LL
#endif
#ifndef MT_KEEP_L2_MB
#define MT_KEEP_L2_MB 100
#endif
constexpr size_t kKeepL2Bytes = (size_t)MT_KEEP_L2_MB << 20;  // tensors up to this size are kept in the 126 MB L2 between calls

struct TmaArgs {
  int64_t n_rows;
  int64_t groups;   // ceil(n_rows / RT)
  int64_t chunks;   // ceil(n / CT)
  int64_t tiles;    // groups * chunks
  double* partial;  // [P][2][RT][B][3]
  double* exch;     // tensor-core kernel: [P][MmaCfg::exch_doubles] column parts of a row block
  int* count;       // [groups] chunks of a split row group summed so far; zero between launches
  int keep_l2;      // the tensor fits in L2: load it with the evict-last policy (it is read again at the next right-hand side)
};

// first tile of CTA c: floor(tiles * c / P), c in [0, P]
__host__ __device__ __forceinline__ int64_t range_begin(int64_t tiles, int64_t P, int64_t c) {
  if (tiles < (int64_t(1) << 40) && P < (int64_t(1) << 20))  // every real shape: one 64-bit division
    return (int64_t)((uint64_t)tiles * (uint64_t)c / (uint64_t)P);
  return (int64_t)(((unsigned __int128)tiles * (unsigned __int128)c) / (unsigned __int128)P);
}

// A row group split between CTAs.  Every CTA that covers part of it has left its partial sums in
// a.partial (slot 0: the group its range starts in, slot 1: the group its range ends in) and now adds
// the number of chunks it covered to the group's counter; the CTA whose addition completes the count
// adds the parts in CTA order — the order is fixed whichever CTA arrives last: bitwise reproducible —
// runs the epilogue and puts the counter back to zero for the next launch.  Nobody waits for anybody.
// Called by ALL threads of the CTA after their partial stores; `sh` = 3 ints of shared memory.
template <int RT>
__device__ __forceinline__ void finish_split_group(const TmaArgs& a, int64_t P, int64_t c, const EpiArgs& e, int B,
                                                   int64_t g, int mine, volatile int* sh) {
  __threadfence();  // this thread's partial sums are visible device-wide before the count moves
  __syncthreads();
  if (threadIdx.x == 0) {
    const int last = (atomicAdd(a.count + g, mine) + mine == (int)a.chunks) ? 1 : 0;
    if (last) {
      a.count[g] = 0;  // nobody else touches this word any more in this launch
      const int64_t tb = g * a.chunks, te = tb + a.chunks;
      int64_t lo = c, hi = c;
      while (lo > 0 && range_begin(a.tiles, P, lo) > tb) --lo;
      while (hi + 1 < P && range_begin(a.tiles, P, hi + 1) < te) ++hi;
      sh[1] = (int)lo;
      sh[2] = (int)hi;
    }
    sh[0] = last;
  }
  __syncthreads();
  if (!sh[0]) return;
  __threadfence();
  const int lo = sh[1], hi = sh[2];
  for (int idx = threadIdx.x; idx < RT * B; idx += blockDim.x) {
    const int rg = idx / B, b = idx - rg * B;
    const int64_t row = g * RT + rg;
    if (row >= a.n_rows) continue;
    double s[3] = {0.0, 0.0, 0.0};
    int64_t cb = range_begin(a.tiles, P, lo);
    for (int cc = lo; cc <= hi; ++cc) {
      const int64_t ce = range_begin(a.tiles, P, cc + 1);
      if (cb < ce) {
        const int slot = (cb / a.chunks == g) ? 0 : 1;
        const double* p = a.partial + ((((int64_t)cc * 2 + slot) * RT + rg) * B + b) * 3;
        s[0] += __ldcg(p);  // written by other SMs in this launch: read from L2
        s[1] += __ldcg(p + 1);
        s[2] += __ldcg(p + 2);
      }
      cb = ce;
    }
    const double hd[3] = {-s[0], -s[1], -s[2]};
    row_epilogue(e, row, b, hd);
  }
}

template <typename T, int B, int RW, int CT_, int STAGES, int WARPS_ = kConsumerWarps>
struct TmaCfg {
  static constexpr int WARPS = WARPS_;
  static constexpr int RT = WARPS_ * RW;
  static constexpr int CT = CT_;
  static constexpr int W = Vec<T>::W;
  static constexpr int VPL = CT / (32 * W);  // 16-byte vectors per lane per row-plane per tile
  static constexpr size_t tensor_bytes = (size_t)6 * RT * CT * sizeof(T);
  static constexpr size_t m_bytes = (size_t)3 * B * CT * sizeof(T);
  static constexpr size_t stage_bytes = tensor_bytes + m_bytes;
  static constexpr size_t smem_bytes = STAGES * stage_bytes + 2 * STAGES * sizeof(uint64_t) + 16 + 128;  // ring, barriers, finish_split_group's words, alignment slack
  static_assert(CT % 64 == 0, "tile width must be a whole number of warp-wide 8-byte vectors");
  static_assert(tensor_bytes % 128 == 0 && m_bytes % 128 == 0, "TMA destinations must stay 128-byte aligned");
};

// NBOX > 1: a tile is NBOX boxes side by side (a TMA box is at most 256 elements wide), each laid out
// [plane][row][CT / NBOX] in the stage, so that a row-plane contributes NBOX contiguous kilobytes per tile
template <typename T, int B, int RW, int CT, int STAGES, int NBOX = 1>
__global__ void __launch_bounds__(kThreads, 1)
    demag_tma_kernel(const __grid_constant__ CUtensorMap tmN, const __grid_constant__ CUtensorMap tmM, TmaArgs a,
                     EpiArgs e) {
  typedef TmaCfg<T, B, RW, CT, STAGES> Cfg;
  typedef typename Vec<T>::type V;
  constexpr int RT = Cfg::RT, VPL = Cfg::VPL;
  constexpr int BW = CT / NBOX;  // box width in elements
  static_assert(CT % NBOX == 0 && BW <= 256 && BW % (32 * Cfg::W) == 0, "box width");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // (generic pointer on purpose: with the provenance-preserving form below the tile reads become LDS,
  // measured 0.5 % slower for this HBM-bound kernel — A/B on one box, r02 — while the packed-FMA kernel
  // gains 2.7 % at B = 8 from it)
  unsigned char* smem = (unsigned char*)(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
  uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::stage_bytes);
  volatile int* fin = (volatile int*)(bars + 2 * STAGES);  // finish_split_group's three words
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t P = gridDim.x, c = blockIdx.x;
  if (e.active_dev && !*e.active_dev) return;  // replayed attempt of a finished device-controlled DP45 run
  const int64_t t0 = range_begin(a.tiles, P, c), t1 = range_begin(a.tiles, P, c + 1);

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, kConsumerWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (t0 >= t1) return;

  // ===== producer state (used by lane 0 of warp 0 only) =====
  uint64_t pol_stream = 0, pol_keep = 0;
  int p_stage = 0;
  uint32_t p_phase = 0;
  int64_t p_t = t0, p_g = t0 / a.chunks, p_k = t0 % a.chunks;
  const bool is_producer = (threadIdx.x == 0);
  if (is_producer) {
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
    if (a.keep_l2) pol_stream = pol_keep;
  }
  // issues tiles until the ring is full or a slot is still being read; `must` = tile index that has to
  // be in flight on return (blocking wait for its slot if necessary)
  auto top_up = [&](int64_t must) {
    while (p_t < t1) {
      if (!mbar_test(empty0 + 8 * p_stage, p_phase ^ 1)) {
        if (p_t > must) break;
        mbar_wait(empty0 + 8 * p_stage, p_phase ^ 1);
      }
      const uint32_t dst = smem_u32(smem + (size_t)p_stage * Cfg::stage_bytes);
      mbar_expect_tx(full0 + 8 * p_stage, (uint32_t)Cfg::stage_bytes);
#pragma unroll
      for (int bx = 0; bx < NBOX; ++bx) {
        tma_load_3d(dst + (uint32_t)(bx * (Cfg::tensor_bytes / NBOX)), &tmN, (int)(p_k * CT + bx * BW), (int)(p_g * RT), 0,
                    full0 + 8 * p_stage, pol_stream);
        tma_load_2d(dst + (uint32_t)(Cfg::tensor_bytes + bx * (Cfg::m_bytes / NBOX)), &tmM, (int)(p_k * CT + bx * BW), 0,
                    full0 + 8 * p_stage, pol_keep);
      }
      if (++p_stage == STAGES) { p_stage = 0; p_phase ^= 1; }
      if (++p_k == a.chunks) { p_k = 0; ++p_g; }
      ++p_t;
    }
  };

  // ===== consumers =====
  double acc[RW][B][3];
#pragma unroll
  for (int r = 0; r < RW; ++r)
#pragma unroll
    for (int b = 0; b < B; ++b) acc[r][b][0] = acc[r][b][1] = acc[r][b][2] = 0.0;
  int stage = 0;
  uint32_t phase = 0;
  int64_t g = t0 / a.chunks, k = t0 % a.chunks;
  const int64_t g_first = g;
  bool head_in_range = (k == 0);  // the current group's first chunk belongs to this CTA
  for (int64_t t = t0; t < t1; ++t) {
    if (is_producer) top_up(t);
    __syncwarp();
    mbar_wait(full0 + 8 * stage, phase);
    const T* tile = (const T*)(smem + (size_t)stage * Cfg::stage_bytes);
    const T* mt = (const T*)(smem + (size_t)stage * Cfg::stage_bytes + Cfg::tensor_bytes);
    // fp32: a short fp32 run per tile, flushed into the fp64 accumulators below; fp64: the
    // accumulators themselves (no second register set)
    constexpr bool kDirect = (sizeof(T) == 8);
    typedef typename RunSel<T, kDirect>::type RunT;
    RunT run_store[kDirect ? 1 : RW][kDirect ? 1 : B][3];
    auto run_of = [&](int r, int b) -> T* {
      if constexpr (kDirect) return (T*)acc[r][b]; else return (T*)run_store[r][b];
    };
    if constexpr (!kDirect) {
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int b = 0; b < B; ++b) run_store[r][b][0] = run_store[r][b][1] = run_store[r][b][2] = RunT(0);
    }
#pragma unroll
    for (int v = 0; v < VPL; ++v) {
      const int colt = (v * 32 + lane) * Cfg::W;          // column in the tile
      const int bx = (v * 32 * Cfg::W) / BW;                // its box (compile-time per v)
      const int col = colt - bx * BW;
      const T* tbox = tile + (size_t)bx * (6 * RT * BW);
      const T* mbox = mt + (size_t)bx * (3 * B * BW);
      V tv[RW][6];
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int cc = 0; cc < 6; ++cc)
          tv[r][cc] = *(const V*)(tbox + ((size_t)cc * RT + (warp * RW + r)) * BW + col);
#pragma unroll
      for (int b = 0; b < B; ++b) {
        V mv[3];
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) mv[cc] = *(const V*)(mbox + (size_t)(b * 3 + cc) * BW + col);
#pragma unroll
        for (int r = 0; r < RW; ++r) fma3(run_of(r, b), tv[r], mv);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(empty0 + 8 * stage);
    if (++stage == STAGES) { stage = 0; phase ^= 1; }
    if constexpr (!kDirect) {
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int b = 0; b < B; ++b) {
          acc[r][b][0] += (double)run_store[r][b][0];
          acc[r][b][1] += (double)run_store[r][b][1];
          acc[r][b][2] += (double)run_store[r][b][2];
        }
    }
    const bool group_done = (k + 1 == a.chunks);
    if (group_done || t + 1 == t1) {
      // fixed-order butterfly: every lane ends with the same sums
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int b = 0; b < B; ++b)
#pragma unroll
          for (int cc = 0; cc < 3; ++cc)
#pragma unroll
            for (int off = 16; off > 0; off >>= 1)
              acc[r][b][cc] += __shfl_xor_sync(0xffffffffu, acc[r][b][cc], off);
      const bool whole = head_in_range && group_done;
#pragma unroll
      for (int r = 0; r < RW; ++r) {
        const int rg = warp * RW + r;
        const int64_t row = g * RT + rg;
        double s[3] = {0.0, 0.0, 0.0};
#pragma unroll
        for (int b = 0; b < B; ++b)
          if (lane == b) { s[0] = acc[r][b][0]; s[1] = acc[r][b][1]; s[2] = acc[r][b][2]; }
        if (lane < B && row < a.n_rows) {
          if (whole) {
            const double hd[3] = {-s[0], -s[1], -s[2]};
            row_epilogue(e, row, lane, hd);
          } else {
            const int slot = (g == g_first) ? 0 : 1;
            double* p = a.partial + ((((int64_t)c * 2 + slot) * RT + rg) * B + lane) * 3;
            p[0] = s[0]; p[1] = s[1]; p[2] = s[2];
          }
        }
      }
      if (!whole) finish_split_group<RT>(a, P, c, e, B, g, (int)(t + 1 - max(t0, g * a.chunks)), fin);
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int b = 0; b < B; ++b) acc[r][b][0] = acc[r][b][1] = acc[r][b][2] = 0.0;
    }
    if (group_done) { k = 0; ++g; head_in_range = true; } else { ++k; }
  }
}

// ---- fp32 tensors, batches of 5..8 states: packed-FMA consumer -------------------------------------
// Same ring, same work split, same finish of split groups as above; what differs is the arithmetic of a tile.  At
// B = 8 a tile block (24 B) carries 72 FMAs: at the HBM rate that is 67 FMA/clk/SM, above what
// three-register FFMA sustains (64/clk/SM), so the products are issued as FFMA2 (fma.rn.f32x2): the
// two halves of a 64-bit register pair are two adjacent source columns, so an LDS.128 of a plane row
// and an LDS.128 of a component of M are each two ready-made operands.  Each (row, state, component)
// sum therefore lives in an even-column/odd-column pair of fp32 accumulators (2 rows x 8 states x 3
// x 2 = 96 registers), which leaves no room for per-lane fp64 accumulators; instead, every kFlush
// tiles (<= 96 terms per fp32 accumulator, Q19) and at the end of a row group the 48 fp32
// sums of a lane are combined across the warp by a transposing butterfly (24+12+6+3+3 shuffles) after
// which lane l holds the three components of (row l>>4, state (l>>1)&7) and adds them to three fp64
// accumulators.  The order is fixed: bitwise reproducible.
constexpr int kPackRW = 2;  // rows per consumer warp of the packed-FMA kernel

__device__ __forceinline__ void ffma2(unsigned long long& d, unsigned long long a, unsigned long long b) {
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
}
__device__ __forceinline__ float sum_halves(unsigned long long v) {
  float lo, hi;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
  return lo + hi;
}
// NP column pairs per lane: 1 (LDS.64, CT = 64) or 2 (LDS.128, CT = 128)
template <int NP> struct PairVec;
template <> struct PairVec<1> { unsigned long long p[1]; };
template <> struct alignas(16) PairVec<2> { unsigned long long p[2]; };

template <int B, int WARPS, int CT, int STAGES, int NBOX = 1>
__global__ void __launch_bounds__(WARPS * 32, 1)
    demag_tma_f32x2_kernel(const __grid_constant__ CUtensorMap tmN, const __grid_constant__ CUtensorMap tmM,
                           TmaArgs a, EpiArgs e) {
  typedef TmaCfg<float, B, kPackRW, CT, STAGES, WARPS> Cfg;
  constexpr int RT = Cfg::RT, RW = kPackRW;
  constexpr int NV = RW * B * 3;                 // fp32 sums per lane
  constexpr int kOwnShift = (B == 8) ? 1 : 2;    // lane l ends up owning (row, state) index l >> kOwnShift
  constexpr int BW = CT / NBOX;          // box width (a tile is NBOX boxes side by side, as in demag_tma_kernel)
  constexpr int NP = BW / 64;            // column pairs per lane per box
  constexpr int kFlush = 96 / (3 * NP * NBOX);  // tiles per fp32 run: <= 96 terms per accumulator
  static_assert((NP == 1 || NP == 2) && (B == 4 || B == 8), "lane mapping of the transposing butterfly");
  typedef PairVec<NP> PV;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // 128-byte alignment by an OFFSET into the shared array (not by integer arithmetic on the generic
  // address): the pointer keeps its shared-memory provenance and the tile reads compile to LDS
  // instead of generic LD (which queue behind the global-memory path: r02 ncu, lg_throttle stalls)
  unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::stage_bytes);
  volatile int* fin = (volatile int*)(bars + 2 * STAGES);  // finish_split_group's three words
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t P = gridDim.x, c = blockIdx.x;
  if (e.active_dev && !*e.active_dev) return;  // replayed attempt of a finished device-controlled DP45 run
  const int64_t t0 = range_begin(a.tiles, P, c), t1 = range_begin(a.tiles, P, c + 1);

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (t0 >= t1) return;

  // producer (lane 0 of warp 0), as in demag_tma_kernel
  uint64_t pol_stream = 0, pol_keep = 0;
  int p_stage = 0;
  uint32_t p_phase = 0;
  int64_t p_t = t0, p_g = t0 / a.chunks, p_k = t0 % a.chunks;
  const bool is_producer = (threadIdx.x == 0);
  if (is_producer) {
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
    if (a.keep_l2) pol_stream = pol_keep;
  }
  auto top_up = [&](int64_t must) {
    while (p_t < t1) {
      if (!mbar_test(empty0 + 8 * p_stage, p_phase ^ 1)) {
        if (p_t > must) break;
        mbar_wait(empty0 + 8 * p_stage, p_phase ^ 1);
      }
      const uint32_t dst = smem_u32(smem + (size_t)p_stage * Cfg::stage_bytes);
      mbar_expect_tx(full0 + 8 * p_stage, (uint32_t)Cfg::stage_bytes);
#pragma unroll
      for (int bx = 0; bx < NBOX; ++bx) {
        tma_load_3d(dst + (uint32_t)(bx * (Cfg::tensor_bytes / NBOX)), &tmN, (int)(p_k * CT + bx * BW), (int)(p_g * RT), 0,
                    full0 + 8 * p_stage, pol_stream);
        tma_load_2d(dst + (uint32_t)(Cfg::tensor_bytes + bx * (Cfg::m_bytes / NBOX)), &tmM, (int)(p_k * CT + bx * BW), 0,
                    full0 + 8 * p_stage, pol_keep);
      }
      if (++p_stage == STAGES) { p_stage = 0; p_phase ^= 1; }
      if (++p_k == a.chunks) { p_k = 0; ++p_g; }
      ++p_t;
    }
  };

  unsigned long long run[RW][B][3];  // {even-column sum, odd-column sum}
#pragma unroll
  for (int r = 0; r < RW; ++r)
#pragma unroll
    for (int b = 0; b < B; ++b) run[r][b][0] = run[r][b][1] = run[r][b][2] = 0ull;
  double acc[3] = {0.0, 0.0, 0.0};  // of (row lane>>4, state (lane>>1)&7)
  int since_flush = 0;
  int stage = 0;
  uint32_t phase = 0;
  int64_t g = t0 / a.chunks, k = t0 % a.chunks;
  const int64_t g_first = g;
  bool head_in_range = (k == 0);
  for (int64_t t = t0; t < t1; ++t) {
    if (is_producer) top_up(t);
    __syncwarp();
    mbar_wait(full0 + 8 * stage, phase);
    const float* tile = (const float*)(smem + (size_t)stage * Cfg::stage_bytes);
    const float* mt = (const float*)(smem + (size_t)stage * Cfg::stage_bytes + Cfg::tensor_bytes);
    const int col = lane * (2 * NP);
#pragma unroll
    for (int bx = 0; bx < NBOX; ++bx) {
    const float* tbox = tile + (size_t)bx * (6 * RT * BW);
    const float* mbox = mt + (size_t)bx * (3 * B * BW);
    PV tv[RW][6];
#pragma unroll
    for (int r = 0; r < RW; ++r)
#pragma unroll
      for (int cc = 0; cc < 6; ++cc)
        tv[r][cc] = *(const PV*)(tbox + ((size_t)cc * RT + (warp * RW + r)) * BW + col);
#pragma unroll
    for (int b = 0; b < B; ++b) {
      PV mv[3];
#pragma unroll
      for (int cc = 0; cc < 3; ++cc) mv[cc] = *(const PV*)(mbox + (size_t)(b * 3 + cc) * BW + col);
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int q = 0; q < NP; ++q) {
          // planes xx, xy, xz, yy, yz, zz = 0..5; p[q] = columns {2q, 2q+1} of the lane
          ffma2(run[r][b][0], tv[r][0].p[q], mv[0].p[q]);
          ffma2(run[r][b][1], tv[r][1].p[q], mv[0].p[q]);
          ffma2(run[r][b][2], tv[r][2].p[q], mv[0].p[q]);
          ffma2(run[r][b][0], tv[r][1].p[q], mv[1].p[q]);
          ffma2(run[r][b][1], tv[r][3].p[q], mv[1].p[q]);
          ffma2(run[r][b][2], tv[r][4].p[q], mv[1].p[q]);
          ffma2(run[r][b][0], tv[r][2].p[q], mv[2].p[q]);
          ffma2(run[r][b][1], tv[r][4].p[q], mv[2].p[q]);
          ffma2(run[r][b][2], tv[r][5].p[q], mv[2].p[q]);
        }
    }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(empty0 + 8 * stage);
    if (++stage == STAGES) { stage = 0; phase ^= 1; }
    const bool group_done = (k + 1 == a.chunks);
    const bool emit = group_done || t + 1 == t1;
    if (++since_flush == kFlush || emit) {
      since_flush = 0;
      // val[(r*8 + b)*3 + cc]; halving steps keep the lower or upper half of the index space by one
      // lane bit each, so that after offsets 16, 8, 4, 2 lane l owns (r*8 + b) == l >> 1
      float val[NV];
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int b = 0; b < B; ++b)
#pragma unroll
          for (int cc = 0; cc < 3; ++cc) {
            val[(r * B + b) * 3 + cc] = sum_halves(run[r][b][cc]);
            run[r][b][cc] = 0ull;
          }
#pragma unroll
      for (int half = NV / 2, off = 16; half >= 3; half >>= 1, off >>= 1) {
        const bool upper = (lane & off) != 0;
#pragma unroll
        for (int i = 0; i < half; ++i) {
          const float keep = upper ? val[i + half] : val[i];
          const float send = upper ? val[i] : val[i + half];
          val[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
        }
      }
#pragma unroll
      for (int cc = 0; cc < 3; ++cc) {
#pragma unroll
        for (int off = 1 << (kOwnShift - 1); off > 0; off >>= 1) val[cc] += __shfl_xor_sync(0xffffffffu, val[cc], off);
        acc[cc] += (double)val[cc];
      }
    }
    if (emit) {
      const int own = lane >> kOwnShift;  // == r * B + b
      const int rg = warp * RW + own / B, b = own % B;
      const int64_t row = g * RT + rg;
      if (!(lane & ((1 << kOwnShift) - 1)) && b < e.batch && row < a.n_rows) {
        if (head_in_range && group_done) {
          const double hd[3] = {-acc[0], -acc[1], -acc[2]};
          row_epilogue(e, row, b, hd);
        } else {
          const int slot = (g == g_first) ? 0 : 1;
          double* p = a.partial + ((((int64_t)c * 2 + slot) * RT + rg) * e.batch + b) * 3;
          p[0] = acc[0]; p[1] = acc[1]; p[2] = acc[2];
        }
      }
      if (!(head_in_range && group_done))
        finish_split_group<RT>(a, P, c, e, e.batch, g, (int)(t + 1 - max(t0, g * a.chunks)), fin);
      acc[0] = acc[1] = acc[2] = 0.0;
    }
    if (group_done) { k = 0; ++g; head_in_range = true; } else { ++k; }
  }
}

// ---- fp32 tensors, batches of 5..8 states: tensor-core consumer (error-compensated TF32) ------------
// With 8 states a 24-byte tensor block carries 72 FMAs; at the HBM rate that is ~2/3 of the FP32 pipe
// AND ~2/3 of the shared-memory bandwidth (every warp re-reads the eight states' M), which do not
// overlap well at two warps per scheduler: the packed-FFMA2 kernel above stops at 0.76 of the HBM
// peak (r02/r03 ncu).  Here the batched product is what it really is, a dense contraction
//     H[(i,a), b] = sum_{(j,c)} N^{ac}_{ij} M[(j,c), b]           (3 n_rows x 3 n) x (3 n x 8),
// and runs on the tensor cores (north_star allows them "if the batched form is a real dense
// contraction that holds accuracy").  Accuracy: TF32 alone (10-bit mantissa) cannot hold the 1e-5
// gate, so both operands are split, x = x_hi + x_lo: for the staged M (re-laid out once per call) x_hi =
// RN_tf32(x), x_lo = RN_tf32(x - x_hi); for the streamed tensor x_hi = trunc_tf32(x) — the tensor core reads
// only the top 19 bits of an fp32 operand, so the raw register is the hi operand — and x_lo = x - x_hi (the
// subtraction is exact; r05 A/B: 18.2 -> 17.9 ms against rounding x_hi in software, error 1.21e-7 -> 1.33e-7).
// Three products are accumulated: lo*hi + hi*lo + hi*hi; what is dropped (lo*lo and the truncation of x_lo)
// is ~2^-21 relative per product.  Products of
// tf32 operands are exact in the tensor core; its fp32 accumulator is drained into per-lane fp64
// sums every kMmaFlush tiles (<= 2 x 9 x 3 mma per accumulator in between).
// Shape: RT = 64 rows x CT = 32 columns per stage; the tensor box lands in shared memory with the
// 128-byte swizzle (a 32-float row = one swizzle span), so ldmatrix.x4 fetches a 16 x 8 fp32 A
// fragment (four 8 x 16-byte matrices) without bank conflicts; warp w owns row block w & 3 (16 rows)
// and part w >> 2 of the tile's four 8-column slabs (16 warps: one slab each; 8 warps: two).  M is re-laid out once per call
// by mma_stage_kernel as [component][slab of 8 columns][state g][t][{hi(t), hi(t+4), lo(t), lo(t+4)}],
// so that one LDS.128 per component is a lane's whole B fragment (k = t, t + 4; n = g) for hi and lo.
// mma.sync m16n8k8: D (16 rows x 8 states) += A (16 x 8 columns) . B (8 columns x 8 states); the nine
// plane-component products of a symmetric 3x3 block are nine such mma per split term (27 per slab).
// No cross-lane reduction is needed: the mma sums over columns.  The warps that share a row block
// add their fp64 sums through shared memory at the end of a row group (fixed order).
// Measured at config 5 (r04): 18.4 ms against 20.5 ms for the packed-FFMA2 kernel, error 1.2e-7
// against the fp64 tensor; the board sits at its 1 kW power cap in both (SM clock ~1.5 GHz) and the
// time follows the energy per block: with the two correction products left out (accuracy lost) it is
// 15.6 ms, 8 or 16 warps and early or late release of the stage make no difference.
#ifndef MT_MMA_WARPS
#define MT_MMA_WARPS 16
#endif
#ifndef MT_MMA_FLUSH_TILES
#define MT_MMA_FLUSH_TILES 1  /* measured (N = 32,768, 8 states, vs the fp64 tensor): 1 -> 2.0e-7, 2 -> 4.3e-7, 8 -> 1.8e-6 */
#endif
#ifndef MT_MMA_NBOX
#define MT_MMA_NBOX 2 /* swizzled boxes of 32 columns side by side in a tile (1: three stages of 54 KB, 2: two of 108 KB; r05 A/B at config 5, eight states: 17.7 -> 16.45 ms) */
#endif
constexpr int kMmaNBox = MT_MMA_NBOX;
constexpr int kMmaWarps = MT_MMA_WARPS, kMmaRT = 64, kMmaCT = 32 * kMmaNBox, kMmaStages = kMmaNBox == 1 ? 3 : 2;
constexpr uint32_t kMmaBoxBytes = 6u * kMmaRT * 128u;  // one swizzled box: 6 planes x 64 rows x 128 bytes
constexpr int kMmaKS = kMmaWarps / 4;           // warps that share a row block (column split of a tile)
constexpr int kMmaSPW = (kMmaCT / 8) / kMmaKS;  // 8-column slabs per warp per tile
constexpr int kMmaFlush = MT_MMA_FLUSH_TILES;
static_assert(kMmaWarps == 8 || kMmaWarps == 16, "4 row blocks x 2 or 4 column slabs");
struct MmaCfg {
  static constexpr int WARPS = kMmaWarps, RT = kMmaRT, CT = kMmaCT;
  static constexpr size_t tensor_bytes = (size_t)6 * kMmaRT * kMmaCT * 4;          // 49,152
  static constexpr size_t m_bytes = (size_t)3 * (kMmaCT / 8) * 128 * 4;           // 6,144
  static constexpr size_t stage_bytes = tensor_bytes + m_bytes;                  // 55,296 = 54 KB
  // column parts of a row block meet in a per-CTA global scratch at the end of a row group (rare: once per
  // 64 rows x n columns), not in shared memory: the ring may use all of it
  static constexpr size_t exch_doubles = (size_t)(kMmaKS - 1) * 12 * 4 * 32;
  static constexpr size_t smem_bytes = kMmaStages * stage_bytes + 2 * kMmaStages * sizeof(uint64_t) + 16 + 1024;
  static_assert(stage_bytes % 1024 == 0, "swizzled tiles must start on 1 KB boundaries");
};

__device__ __forceinline__ uint32_t tf32_rn(uint32_t x) { return (x + 0x1000u) & 0xffffe000u; }
__device__ __forceinline__ void mma_tf32(float d[4], const uint32_t a[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// plain staged M [MT_MAX_BATCH][3][npad] fp32 -> Mq[3][npad/8][8 states][4][4] (see above)
__global__ void __launch_bounds__(256) mma_stage_kernel(const float* __restrict__ M, int64_t npad, float4* __restrict__ Mq) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // (comp, slab, g, t)
  const int64_t slabs = npad / 8;
  if (idx >= 3 * slabs * 32) return;
  const int t = (int)(idx & 3), g = (int)((idx >> 2) & 7);
  const int64_t slab = (idx >> 5) % slabs;
  const int comp = (int)((idx >> 5) / slabs);
  const float* src = M + ((int64_t)g * 3 + comp) * npad + slab * 8 + t;
  const float v0 = src[0], v1 = src[4];
  const uint32_t h0 = tf32_rn(__float_as_uint(v0)), h1 = tf32_rn(__float_as_uint(v1));
  const float l0 = v0 - __uint_as_float(h0), l1 = v1 - __uint_as_float(h1);
  Mq[idx] = make_float4(__uint_as_float(h0), __uint_as_float(h1), __uint_as_float(tf32_rn(__float_as_uint(l0))),
                        __uint_as_float(tf32_rn(__float_as_uint(l1))));
}

__global__ void __launch_bounds__(kMmaWarps * 32, 1)
    demag_tma_mma_kernel(const __grid_constant__ CUtensorMap tmN, const __grid_constant__ CUtensorMap tmM, TmaArgs a,
                         EpiArgs e) {
  typedef MmaCfg Cfg;
  constexpr int RT = kMmaRT, CT = kMmaCT, STAGES = kMmaStages, KS = kMmaKS, SPW = kMmaSPW;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint64_t* bars = (uint64_t*)(smem + STAGES * Cfg::stage_bytes);
  volatile int* fin = (volatile int*)(bars + 2 * STAGES);  // finish_split_group's three words
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + STAGES);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t P = gridDim.x, c = blockIdx.x;
  if (e.active_dev && !*e.active_dev) return;  // replayed attempt of a finished device-controlled DP45 run
  double* exch = a.exch + (size_t)c * Cfg::exch_doubles;
  const int64_t t0 = range_begin(a.tiles, P, c), t1 = range_begin(a.tiles, P, c + 1);

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, kMmaWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (t0 >= t1) return;

  // producer (lane 0 of warp 0), as in demag_tma_kernel
  uint64_t pol_stream = 0, pol_keep = 0;
  int p_stage = 0;
  uint32_t p_phase = 0;
  int64_t p_t = t0, p_g = t0 / a.chunks, p_k = t0 % a.chunks;
  const bool is_producer = (threadIdx.x == 0);
  if (is_producer) {
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
    if (a.keep_l2) pol_stream = pol_keep;
  }
  auto top_up = [&](int64_t must) {
    while (p_t < t1) {
      if (!mbar_test(empty0 + 8 * p_stage, p_phase ^ 1)) {
        if (p_t > must) break;
        mbar_wait(empty0 + 8 * p_stage, p_phase ^ 1);
      }
      const uint32_t dst = smem_u32(smem + (size_t)p_stage * Cfg::stage_bytes);
      mbar_expect_tx(full0 + 8 * p_stage, (uint32_t)Cfg::stage_bytes);
#pragma unroll
      for (int bx = 0; bx < kMmaNBox; ++bx)
        tma_load_3d(dst + (uint32_t)bx * kMmaBoxBytes, &tmN, (int)(p_k * CT + bx * 32), (int)(p_g * RT), 0,
                    full0 + 8 * p_stage, pol_stream);
      tma_load_3d(dst + (uint32_t)Cfg::tensor_bytes, &tmM, 0, (int)(p_k * (CT / 8)), 0, full0 + 8 * p_stage, pol_keep);
      if (++p_stage == STAGES) { p_stage = 0; p_phase ^= 1; }
      if (++p_k == a.chunks) { p_k = 0; ++p_g; }
      ++p_t;
    }
  };

  // consumer geometry: warp = (row block rb of 16 rows, column part ks of the tile)
  const int rb = warp & 3, ks = warp >> 2;
  const int g8 = lane >> 2, tig = lane & 3;
  // ldmatrix: lane supplies the address of row (lane & 7) of matrix (lane >> 3); matrices = {rows 0-7,
  // rows 8-15} x {columns 0-3, 4-7} of the slab, in the order of the A fragment registers a0..a3
  const int lm_r = lane & 7, lm_j = lane >> 3;
  const uint32_t lm_row_off = (uint32_t)(rb * 16 + lm_r + 8 * (lm_j & 1)) * 128u;
  uint32_t lm_chunk[SPW];
#pragma unroll
  for (int q = 0; q < SPW; ++q) {
    const int sl = SPW * ks + q;  // slab of the tile: box sl >> 2, 16-byte chunks 2 (sl & 3), 2 (sl & 3) + 1 of the row
    lm_chunk[q] = (uint32_t)(sl >> 2) * kMmaBoxBytes + (uint32_t)(((2 * (sl & 3) + (lm_j >> 1)) ^ lm_r) << 4);
  }

  float d[3][4];
  double acc[3][4];
#pragma unroll
  for (int cc = 0; cc < 3; ++cc)
#pragma unroll
    for (int i = 0; i < 4; ++i) { d[cc][i] = 0.f; acc[cc][i] = 0.0; }
  int since_flush = 0;
  int stage = 0;
  uint32_t phase = 0;
  int64_t g = t0 / a.chunks, k = t0 % a.chunks;
  const int64_t g_first = g;
  bool head_in_range = (k == 0);
  for (int64_t t = t0; t < t1; ++t) {
    if (is_producer) top_up(t);
    __syncwarp();
    mbar_wait(full0 + 8 * stage, phase);
    const uint32_t tile = smem_u32(smem + (size_t)stage * Cfg::stage_bytes);
    const float4* mq = (const float4*)(smem + (size_t)stage * Cfg::stage_bytes + Cfg::tensor_bytes);
    // all fragments of the warp's slabs go to registers first and the stage is handed back to the
    // producer BEFORE the arithmetic: a stage is held for ~10 shared-memory loads instead of the
    // whole tile's mma work
    uint32_t raw[SPW][6][4];
    float4 bq[SPW][3];
#pragma unroll
    for (int q = 0; q < SPW; ++q) {
#pragma unroll
      for (int p = 0; p < 6; ++p)
        asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                     : "=r"(raw[q][p][0]), "=r"(raw[q][p][1]), "=r"(raw[q][p][2]), "=r"(raw[q][p][3])
                     : "r"(tile + (uint32_t)p * (RT * 128u) + lm_row_off + lm_chunk[q]));
#pragma unroll
      for (int cc = 0; cc < 3; ++cc) bq[q][cc] = mq[(cc * (CT / 8) + SPW * ks + q) * 32 + lane];
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(empty0 + 8 * stage);
#pragma unroll
    for (int q = 0; q < SPW; ++q) {
      // plane p multiplies component col(p) of M into row component row(p) and, off the diagonal,
      // component row(p) into col(p): xx, xy, xz, yy, yz, zz
#pragma unroll
      for (int p = 0; p < 6; ++p) {
        constexpr int prow[6] = {0, 0, 0, 1, 1, 2}, pcol[6] = {0, 1, 2, 1, 2, 2};
        // x_hi = trunc_tf32(x): the tensor core reads the top 19 bits of an fp32 operand, so x itself is
        // passed as the hi operand (no instruction); x_lo = x - trunc(x) is exact and is truncated the same way
        uint32_t lo[4];
        const uint32_t* hi = raw[q][p];
#pragma unroll
        for (int i = 0; i < 4; ++i)
          lo[i] = __float_as_uint(__uint_as_float(raw[q][p][i]) - __uint_as_float(raw[q][p][i] & 0xffffe000u));
        const int ra = prow[p], ca = pcol[p];
        const float4* b = bq[q];
        // small terms first, the dominant hi*hi product last
        mma_tf32(d[ra], lo, __float_as_uint(b[ca].x), __float_as_uint(b[ca].y));
        mma_tf32(d[ra], hi, __float_as_uint(b[ca].z), __float_as_uint(b[ca].w));
        mma_tf32(d[ra], hi, __float_as_uint(b[ca].x), __float_as_uint(b[ca].y));
        if (ra != ca) {
          mma_tf32(d[ca], lo, __float_as_uint(b[ra].x), __float_as_uint(b[ra].y));
          mma_tf32(d[ca], hi, __float_as_uint(b[ra].z), __float_as_uint(b[ra].w));
          mma_tf32(d[ca], hi, __float_as_uint(b[ra].x), __float_as_uint(b[ra].y));
        }
      }
    }
    if (++stage == STAGES) { stage = 0; phase ^= 1; }
    const bool group_done = (k + 1 == a.chunks);
    const bool emit = group_done || t + 1 == t1;
    if (++since_flush == kMmaFlush || emit) {
      since_flush = 0;
#pragma unroll
      for (int cc = 0; cc < 3; ++cc)
#pragma unroll
        for (int i = 0; i < 4; ++i) { acc[cc][i] += (double)d[cc][i]; d[cc][i] = 0.f; }
    }
    if (emit) {
      // the KS warps of a row block (column parts of the tiles) add up through shared memory, in order
      if (ks > 0) {
#pragma unroll
        for (int cc = 0; cc < 3; ++cc)
#pragma unroll
          for (int i = 0; i < 4; ++i) exch[(((ks - 1) * 3 + cc) * 4 + i) * 128 + rb * 32 + lane] = acc[cc][i];
      }
      __syncthreads();
      if (ks == 0) {
#pragma unroll 1
        for (int i = 0; i < 4; ++i) {
          const int rg = rb * 16 + g8 + 8 * (i >> 1), b = 2 * tig + (i & 1);
          const int64_t row = g * RT + rg;
          double s3[3];
#pragma unroll
          for (int cc = 0; cc < 3; ++cc) {
            // (dynamic index i: pick without spilling acc to local memory)
            double v = i == 0 ? acc[cc][0] : i == 1 ? acc[cc][1] : i == 2 ? acc[cc][2] : acc[cc][3];
#pragma unroll
            for (int w = 0; w < KS - 1; ++w) v += exch[((w * 3 + cc) * 4 + i) * 128 + rb * 32 + lane];
            s3[cc] = v;
          }
          if (b < e.batch && row < a.n_rows) {
            if (head_in_range && group_done) {
              const double hd[3] = {-s3[0], -s3[1], -s3[2]};
              row_epilogue(e, row, b, hd);
            } else {
              const int slot = (g == g_first) ? 0 : 1;
              double* pp = a.partial + ((((int64_t)c * 2 + slot) * RT + rg) * e.batch + b) * 3;
              pp[0] = s3[0]; pp[1] = s3[1]; pp[2] = s3[2];
            }
          }
        }
      }
      __syncthreads();
      if (!(head_in_range && group_done))
        finish_split_group<RT>(a, P, c, e, e.batch, g, (int)(t + 1 - max(t0, g * a.chunks)), fin);
#pragma unroll
      for (int cc = 0; cc < 3; ++cc)
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[cc][i] = 0.0;
    }
    if (group_done) { k = 0; ++g; head_in_range = true; } else { ++k; }
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

int make_map(mt_ctx* ctx, CUtensorMap* out, int dtype, const void* base, int rank, const uint64_t* dims,
             const uint64_t* strides_bytes, const uint32_t* box, bool swizzle128 = false) {
  static_assert(sizeof(CUtensorMap) == sizeof(ctx->tm_cache[0].map), "tensor map size");
  for (auto& c : ctx->tm_cache) {
    bool hit = c.valid && c.base == base && c.dtype == dtype && c.rank == rank && c.swizzle == (int)swizzle128;
    for (int k = 0; hit && k < rank; ++k) hit = c.dims[k] == dims[k] && c.box[k] == box[k];
    for (int k = 0; hit && k + 1 < rank; ++k) hit = c.strides[k] == strides_bytes[k];
    if (hit) {
      memcpy(out, c.map, sizeof(CUtensorMap));
      return MT_OK;
    }
  }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return mt_fail(ctx, MT_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
  const cuuint32_t ones[3] = {1, 1, 1};
  CUresult r = fn(out, dtype == MT_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64,
                  (cuuint32_t)rank, const_cast<void*>(base), (const cuuint64_t*)dims, (const cuuint64_t*)strides_bytes,
                  (const cuuint32_t*)box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return mt_fail(ctx, MT_ERR_CUDA, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
  auto& c = ctx->tm_cache[ctx->tm_next];
  ctx->tm_next = (ctx->tm_next + 1) % (int)(sizeof(ctx->tm_cache) / sizeof(ctx->tm_cache[0]));
  c.base = base; c.dtype = dtype; c.rank = rank; c.swizzle = (int)swizzle128; c.valid = 1;
  for (int k = 0; k < 3; ++k) { c.dims[k] = k < rank ? dims[k] : 0; c.box[k] = k < rank ? box[k] : 0; }
  for (int k = 0; k < 2; ++k) c.strides[k] = k + 1 < rank ? strides_bytes[k] : 0;
  memcpy(c.map, out, sizeof(CUtensorMap));
  return MT_OK;
}

// the split-group counters (finish_split_group): zeroed when allocated, left at zero by every launch
int ensure_count(mt_ctx* ctx, int64_t groups) {
  const size_t need = (size_t)(groups > 16384 ? groups : 16384) * sizeof(int);
  if (ctx->split_count && ctx->split_count_bytes >= need) return MT_OK;
  int rc = mt_ensure_ws(ctx, (void**)&ctx->split_count, &ctx->split_count_bytes, need);
  if (rc) return rc;
  MT_CUDA_OK(ctx, cudaMemsetAsync(ctx->split_count, 0, need, ctx->stream));
  return MT_OK;
}

// Cfg = tile geometry; kern = the kernel instantiated for it; m_rows = rows of the staged-M box (3 B)
template <typename T, typename Cfg, typename Kern>
int launch_tiles(mt_ctx* ctx, Kern kern, unsigned char* attr_set, int m_rows, const void* N, int dtype, int64_t n,
                 int64_t n_rows, int64_t ld, const void* Mst, int64_t npad, const EpiArgs& e, int nbox = 1) {
  constexpr int RT = Cfg::RT;
  static_assert(Cfg::smem_bytes <= 227 * 1024, "ring does not fit shared memory");
  const int64_t P = ctx->num_sms;
  TmaArgs a;
  a.n_rows = n_rows;
  a.groups = (n_rows + RT - 1) / RT;
  a.chunks = (n + Cfg::CT - 1) / Cfg::CT;
  a.tiles = a.groups * a.chunks;
  const size_t need = (size_t)P * 2 * RT * e.batch * 3 * sizeof(double);
  int rc = mt_ensure_ws(ctx, (void**)&ctx->partial, &ctx->partial_bytes, need);
  if (rc) return rc;
  a.partial = ctx->partial;
  a.exch = nullptr;
  if ((rc = ensure_count(ctx, a.groups))) return rc;
  a.count = ctx->split_count;
  a.keep_l2 = 6 * (size_t)n_rows * (size_t)ld * sizeof(T) <= kKeepL2Bytes;
  alignas(64) CUtensorMap tmN, tmM;
  {
    const uint64_t dims[3] = {(uint64_t)n, (uint64_t)n_rows, 6};
    const uint64_t strides[2] = {(uint64_t)ld * sizeof(T), (uint64_t)n_rows * (uint64_t)ld * sizeof(T)};
    const uint32_t box[3] = {(uint32_t)(Cfg::CT / nbox), (uint32_t)RT, 6};
    if ((rc = make_map(ctx, &tmN, dtype, N, 3, dims, strides, box))) return rc;
  }
  {
    // the staged-M buffers always hold MT_MAX_BATCH states (rows beyond 3*batch: zero or stale, unused)
    const uint64_t dims[2] = {(uint64_t)npad, (uint64_t)(3 * MT_MAX_BATCH)};
    const uint64_t strides[1] = {(uint64_t)npad * sizeof(T)};
    const uint32_t box[2] = {(uint32_t)(Cfg::CT / nbox), (uint32_t)m_rows};
    if ((rc = make_map(ctx, &tmM, dtype, Mst, 2, dims, strides, box))) return rc;
  }
  // the attribute is per DEVICE (a second mt_ctx on another device of the same process needs its own
  // call): one flag per device ordinal and kernel instantiation
  const int dev = ctx->device & (kMaxDevices - 1);
  if (!attr_set[dev]) {
    MT_CUDA_OK(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem_bytes));
    attr_set[dev] = 1;
  }
  kern<<<(unsigned)P, Cfg::WARPS * 32, Cfg::smem_bytes, ctx->stream>>>(tmN, tmM, a, e);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

template <typename T, int B, int RW, int CT, int STAGES, int NBOX = 1>
int launch_cfg(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, const void* Mst,
               int64_t npad, const EpiArgs& e) {
  static unsigned char attr_set[kMaxDevices] = {};
  return launch_tiles<T, TmaCfg<T, B, RW, CT, STAGES>>(ctx, demag_tma_kernel<T, B, RW, CT, STAGES, NBOX>, attr_set, 3 * B,
                                                        N, dtype, n, n_rows, ld, Mst, npad, e, NBOX);
}

// fp32, 5 <= batch <= 8: packed-FMA kernel (states beyond `batch` are computed on unused rows of M
// and dropped)
template <int B, int WARPS, int CT, int STAGES, int NBOX = 1>
int launch_f32x2_shape(mt_ctx* ctx, const void* N, int64_t n, int64_t n_rows, int64_t ld, const void* Mst,
                       int64_t npad, const EpiArgs& e) {
  static unsigned char attr_set[kMaxDevices] = {};
  return launch_tiles<float, TmaCfg<float, B, kPackRW, CT, STAGES, WARPS>>(
      ctx, demag_tma_f32x2_kernel<B, WARPS, CT, STAGES, NBOX>, attr_set, 3 * B, N, MT_F32, n, n_rows, ld, Mst, npad, e, NBOX);
}

// fp32, 5 <= batch <= 8: tensor-core kernel (error-compensated TF32); states beyond `batch` are
// computed on unused rows of M and dropped
int launch_mma(mt_ctx* ctx, const void* N, int64_t n, int64_t n_rows, int64_t ld, const void* Mst, int64_t npad,
               const EpiArgs& e) {
  typedef MmaCfg Cfg;
  constexpr int RT = Cfg::RT;
  static_assert(Cfg::smem_bytes <= 227 * 1024, "ring does not fit shared memory");
  const int64_t P = ctx->num_sms;
  TmaArgs a;
  a.n_rows = n_rows;
  a.groups = (n_rows + RT - 1) / RT;
  a.chunks = (n + Cfg::CT - 1) / Cfg::CT;
  a.tiles = a.groups * a.chunks;
  const size_t partial_doubles = (size_t)P * 2 * RT * e.batch * 3;
  int rc = mt_ensure_ws(ctx, (void**)&ctx->partial, &ctx->partial_bytes,
                        (partial_doubles + (size_t)P * Cfg::exch_doubles) * sizeof(double));
  if (rc) return rc;
  a.partial = ctx->partial;
  a.exch = ctx->partial + partial_doubles;
  if ((rc = ensure_count(ctx, a.groups))) return rc;
  a.count = ctx->split_count;
  a.keep_l2 = 6 * (size_t)n_rows * (size_t)ld * sizeof(float) <= kKeepL2Bytes;
  // M re-laid out for the B fragments: hi/lo split, [3][npad/8][8 states][4][4] fp32
  const size_t mq_bytes = (size_t)3 * (npad / 8) * 32 * sizeof(float4);
  if ((rc = mt_ensure_ws(ctx, &ctx->Mq, &ctx->Mq_bytes, mq_bytes))) return rc;
  {
    const int64_t tot = 3 * (npad / 8) * 32;
    mma_stage_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, ctx->stream>>>((const float*)Mst, npad, (float4*)ctx->Mq);
    ctx->launches++;
    MT_CUDA_OK(ctx, cudaGetLastError());
  }
  alignas(64) CUtensorMap tmN, tmM;
  {
    const uint64_t dims[3] = {(uint64_t)n, (uint64_t)n_rows, 6};
    const uint64_t strides[2] = {(uint64_t)ld * 4, (uint64_t)n_rows * (uint64_t)ld * 4};
    const uint32_t box[3] = {32, (uint32_t)RT, 6};  // one swizzle span wide; a tile is kMmaNBox of them
    if ((rc = make_map(ctx, &tmN, MT_F32, N, 3, dims, strides, box, /*swizzle128=*/true))) return rc;
  }
  {
    const uint64_t dims[3] = {128, (uint64_t)(npad / 8), 3};
    const uint64_t strides[2] = {128 * 4, (uint64_t)(npad / 8) * 128 * 4};
    const uint32_t box[3] = {128, (uint32_t)(Cfg::CT / 8), 3};
    if ((rc = make_map(ctx, &tmM, MT_F32, ctx->Mq, 3, dims, strides, box))) return rc;
  }
  static unsigned char attr_set[kMaxDevices] = {};
  const int dev = ctx->device & (kMaxDevices - 1);
  if (!attr_set[dev]) {
    MT_CUDA_OK(ctx, cudaFuncSetAttribute(demag_tma_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)Cfg::smem_bytes));
    attr_set[dev] = 1;
  }
  demag_tma_mma_kernel<<<(unsigned)P, Cfg::WARPS * 32, Cfg::smem_bytes, ctx->stream>>>(tmN, tmM, a, e);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

// fp32, 3 <= batch <= 8: packed-FMA kernels for 4 or 8 states (states beyond `batch` are computed on
// unused rows of M and dropped)
int launch_f32x2(mt_ctx* ctx, const void* N, int64_t n, int64_t n_rows, int64_t ld, const void* Mst, int64_t npad,
                 const EpiArgs& e) {
  // two boxes of MT_B4_CT columns side by side per tile, two stages (r05 A/B at config 5: batches of 3 and 4
  // 16.4-16.7 -> 15.5-15.6 ms against one-box tiles in four stages)
  if (e.batch <= 4) return launch_f32x2_shape<4, MT_B4_WARPS, MT_B4_CT * 2, 2, 2>(ctx, N, n, n_rows, ld, Mst, npad, e);
  // variant 3 keeps the packed-FFMA2 kernel for A/B comparisons; the default is the tensor-core kernel
  if (ctx->variant != 3) return launch_mma(ctx, N, n, n_rows, ld, Mst, npad, e);
  return launch_f32x2_shape<8, MT_B8_WARPS, MT_B8_CT, MT_B8_STAGES>(ctx, N, n, n_rows, ld, Mst, npad, e);
}

template <typename T>
int launch_T(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, const void* Mst,
             int64_t npad, const EpiArgs& e) {
  constexpr int CT1 = 1024 / sizeof(T);  // 1 KB of one row-plane per tile
  // batches of 1 and 2: tiles of two boxes side by side (2 KB of every row-plane per tile, 96 KB per stage,
  // two stages) — r05 A/B at config 5, batch 1: 14.94 ms with one-box tiles in four stages, 13.97 ms with
  // two-box tiles in two (7.38 TB/s: the rate of the read-only stream microbenchmark)
#ifndef MT_B1_NBOX
#define MT_B1_NBOX 2
#define MT_B1_STAGES 2
#endif
  if (e.batch == 1) return launch_cfg<T, 1, 1, CT1 * MT_B1_NBOX, MT_B1_STAGES, MT_B1_NBOX>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
  // (batch 2 on fp32 tensors is no faster with them: 14.61 vs 14.58 ms; on fp64 tensors 7.36 vs 7.47 ms at config 3)
  if (e.batch == 2 && sizeof(T) == 8)
    return launch_cfg<T, 2, 1, CT1 * MT_B1_NBOX, MT_B1_STAGES, MT_B1_NBOX>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
  if (e.batch == 2) return launch_cfg<T, 2, 1, CT1, 4>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
  if (e.batch >= 3 && e.batch <= MT_MAX_BATCH) {
    if constexpr (sizeof(T) == 4) {
      return launch_f32x2(ctx, N, n, n_rows, ld, Mst, npad, e);
    } else {
      switch (e.batch) {
        case 3: return launch_cfg<T, 3, 1, CT1, 3>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
        case 4: return launch_cfg<T, 4, 1, CT1, 3>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
        case 5: return launch_cfg<T, 5, 2, CT1 / 2, 3>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
        case 6: return launch_cfg<T, 6, 2, CT1 / 2, 3>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
        case 7: return launch_cfg<T, 7, 2, CT1 / 2, 3>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
        case 8: return launch_cfg<T, 8, 2, CT1 / 2, 3>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
      }
    }
  }
  return mt_fail(ctx, MT_ERR_INVALID_ARG, "batch must be in [1, %d]", MT_MAX_BATCH);
}

}  // namespace

bool mt_demag_tma_takes(mt_ctx* ctx, int dtype, int64_t n, int64_t n_rows) {
  const int64_t tiles = ((n_rows + 7) / 8) * ((n * (dtype == MT_F32 ? 4 : 8) + 1023) / 1024);
  return tiles >= MT_TMA_MIN_TILES_PER_SM * ctx->num_sms;
}

// Returns MT_ERR_UNIMPLEMENTED when the shape is better served by the register-streaming kernel
// (too few tiles to give every SM a share); the dispatcher then falls back to it.
int mt_launch_demag_tma(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                        const void* Mst, int64_t npad, const EpiArgs& e) {
  if (ctx->variant < 2) {
    if (!mt_demag_tma_takes(ctx, dtype, n, n_rows)) return MT_ERR_UNIMPLEMENTED;
  }
  if (dtype == MT_F32) return launch_T<float>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
  return launch_T<double>(ctx, N, dtype, n, n_rows, ld, Mst, npad, e);
}
