// sym.cu — F3: field from the pair-symmetric half of the tensor, layout sym_layout.cuh.
//
// Every stored block N_ij (j's 32-column block right of row block I) serves two rows of
// H_d = -N.(Ms m): row i (with M_j) and row j (with M_i), so one evaluation streams half the bytes
// of the full tensor.  Bound: HBM (3 flop/B fp32), same roofline as A4.
//
// One CTA (8 warps) walks the tiles of a row block I and then of its mirror block nrb-1-I, so every
// CTA streams the same number of tiles.  A tile is 96 KiB of CONTIGUOUS storage (sym_layout.cuh), so
// since r05 it is fetched by three 32 KiB bulk copies (cp.async.bulk, L2 evict-first) into a two-stage
// shared-memory ring guarded by full/empty mbarriers — the access pattern of the read-only stream
// microbenchmark — instead of 24 x 16-byte register loads per lane.  Inside a tile warp w owns 4W columns
// for all 32 rows: lane l reads, for g = 0..3, the W-column vector of row 8g + l/4 of the six planes (each
// warp-wide read 512 contiguous bytes of shared memory: conflict-free).
//   * row part:    racc[g] += N_ij M_j over the lane's W columns; summed over the tiles of the row block
//                  in registers (fp32 runs of <= 96 terms, then fp64), reduced over the 4 lanes of a row
//                  and the 8 warps once per row block (shared memory, fixed order);
//   * column part: cacc[e] += N_ij M_i over the lane's 4 rows, reduced over the 8 row-lanes of the warp
//                  by shuffles: the tile's contribution to rows j, written (no atomics) to
//                  colpart[I][3][j] and summed over I < j/32 in fixed order by the finishing kernel,
//                  which also runs the fused epilogue (epilogue.cuh).
// The 32 x 32 diagonal block is stored whole and used for the row part only; the entries left of it
// are zero in storage and masked here.  Results are bitwise reproducible.
#include "epilogue.cuh"
#include "mbar.cuh"
#include "sym_layout.cuh"

namespace {

template <typename T> struct SymVec;
template <> struct SymVec<float> { typedef float4 type; };
template <> struct SymVec<double> { typedef double2 type; };

__device__ __forceinline__ float4 ld_stream(const float4* p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
               : "l"(p));
  return v;
}
__device__ __forceinline__ double2 ld_stream(const double2* p) {
  double2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ float comp(const float4& v, int e) { return e == 0 ? v.x : e == 1 ? v.y : e == 2 ? v.z : v.w; }
__device__ __forceinline__ double comp(const double2& v, int e) { return e == 0 ? v.x : v.y; }

struct SymArgs {
  int64_t n, nrb, ntc, npad, ncolpad, nrowpad;
  const void* data;
  const void* Mst;   // staged Ms*m of ONE state: [3][npad] in the tensor's dtype
  double* rowpart;   // [3][nrowpad]
  void* colpart;     // [nrb][3][ncolpad] in the tensor's dtype
};

constexpr int kSymStages = 2;
constexpr uint32_t kSymTileBytes = 6u * 32u * 32u * 16u;  // 98,304 for both dtypes (TW = 32 W, W = 16 / sizeof(T))
constexpr size_t kSymSmemBytes = (size_t)kSymStages * kSymTileBytes + 2 * kSymStages * sizeof(uint64_t) + 128;

template <typename T>
__global__ void __launch_bounds__(256, 1) sym_field_kernel(SymArgs a) {
  typedef SymCfg<T> Cfg;
  typedef typename SymVec<T>::type V;
  constexpr int W = Cfg::W, TW = Cfg::TW;
  constexpr int kFlushTiles = 96 / (3 * W);  // fp32: 8 tiles of 12 terms per accumulator
  static_assert(Cfg::kTileElems * sizeof(T) == kSymTileBytes, "tile size");
  __shared__ double red[8][32][3];
  extern __shared__ __align__(128) unsigned char sym_smem_raw[];
  unsigned char* ring = sym_smem_raw + ((128u - (smem_u32(sym_smem_raw) & 127u)) & 127u);
  uint64_t* bars = (uint64_t*)(ring + (size_t)kSymStages * kSymTileBytes);
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + kSymStages);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rl = lane >> 2, cq = lane & 3;  // row-lane (0..7), column quad (0..3)
  const T* M = (const T*)a.Mst;
  T* colpart = (T*)a.colpart;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kSymStages; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 8);
    }
    mbar_fence_init();
  }
  __syncthreads();
  // the CTA's tile sequence: all tiles of row block I0 = blockIdx.x, then all of its mirror block I1
  const int64_t I0 = blockIdx.x, I1 = a.nrb - 1 - (int64_t)blockIdx.x;
  const int64_t cnt0 = a.ntc - (32 * I0) / TW;
  const int64_t cnt1 = I1 > I0 ? a.ntc - (32 * I1) / TW : 0;
  const int64_t start0 = sym_tile_prefix(I0, a.ntc, Cfg::kBlocksPerTile);
  const int64_t start1 = cnt1 ? sym_tile_prefix(I1, a.ntc, Cfg::kBlocksPerTile) : 0;
  const int64_t total = cnt0 + cnt1;
  // producer (thread 0): tops the ring up before each of its own tiles, as in demag_tma.cu
  const bool is_producer = threadIdx.x == 0;
  uint64_t policy = 0;
  if (is_producer) policy = l2_policy_evict_first();
  int64_t p_q = 0;
  int p_stage = 0;
  uint32_t p_phase = 0;
  auto top_up = [&](int64_t must) {
    while (p_q < total) {
      if (!mbar_test(empty0 + 8 * p_stage, p_phase ^ 1)) {
        if (p_q > must) break;
        mbar_wait(empty0 + 8 * p_stage, p_phase ^ 1);
      }
      const int64_t tile = p_q < cnt0 ? start0 + p_q : start1 + (p_q - cnt0);
      const unsigned char* src = (const unsigned char*)a.data + tile * (int64_t)kSymTileBytes;
      const uint32_t dst = smem_u32(ring + (size_t)p_stage * kSymTileBytes);
      mbar_expect_tx(full0 + 8 * p_stage, kSymTileBytes);
#pragma unroll
      for (int c = 0; c < 3; ++c)
        bulk_load_1d(dst + c * (kSymTileBytes / 3), src + c * (kSymTileBytes / 3), kSymTileBytes / 3, full0 + 8 * p_stage, policy);
      if (++p_stage == kSymStages) { p_stage = 0; p_phase ^= 1; }
      ++p_q;
    }
  };
  int stage = 0;
  uint32_t phase = 0;
  int64_t q = 0;
  for (int pass = 0; pass < 2; ++pass) {
    const int64_t I = pass == 0 ? I0 : I1;
    if (pass == 1 && cnt1 == 0) break;  // odd count: the middle block was done in pass 0
    const int64_t Jd = (32 * I) / TW;
    T Mi[4][3];
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
      for (int c = 0; c < 3; ++c) Mi[g][c] = M[(int64_t)c * a.npad + 32 * I + 8 * g + rl];
    double racc[4][3];
    T rrun[4][3];
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
      for (int c = 0; c < 3; ++c) { racc[g][c] = 0.0; rrun[g][c] = T(0); }
    int since = 0;
    for (int64_t J = Jd; J < a.ntc; ++J, ++q) {
      if (is_producer) top_up(q);
      __syncwarp();
      mbar_wait(full0 + 8 * stage, phase);
      const V* tp = (const V*)(ring + (size_t)stage * kSymTileBytes) + warp * 32 + lane;
      V v[6][4];
#pragma unroll
      for (int p = 0; p < 6; ++p)
#pragma unroll
        for (int g = 0; g < 4; ++g) v[p][g] = tp[(p * 4 + g) * 256];
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * stage);  // the tile is in registers: hand the stage back
      if (++stage == kSymStages) { stage = 0; phase ^= 1; }
      const int64_t j0 = J * TW + warp * 4 * W + cq * W;
      const int64_t jb = j0 >> 5;
      const bool use_row = jb >= I, use_col = jb > I;
      T Mj[3][W];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const V mv = *(const V*)(M + (int64_t)c * a.npad + j0);
#pragma unroll
        for (int e = 0; e < W; ++e) Mj[c][e] = use_row ? comp(mv, e) : T(0);
      }
      T cacc[W][3];
#pragma unroll
      for (int e = 0; e < W; ++e) cacc[e][0] = cacc[e][1] = cacc[e][2] = T(0);
#pragma unroll
      for (int g = 0; g < 4; ++g)
#pragma unroll
        for (int e = 0; e < W; ++e) {
          const T xx = comp(v[0][g], e), xy = comp(v[1][g], e), xz = comp(v[2][g], e);
          const T yy = comp(v[3][g], e), yz = comp(v[4][g], e), zz = comp(v[5][g], e);
          rrun[g][0] = fma(xx, Mj[0][e], fma(xy, Mj[1][e], fma(xz, Mj[2][e], rrun[g][0])));
          rrun[g][1] = fma(xy, Mj[0][e], fma(yy, Mj[1][e], fma(yz, Mj[2][e], rrun[g][1])));
          rrun[g][2] = fma(xz, Mj[0][e], fma(yz, Mj[1][e], fma(zz, Mj[2][e], rrun[g][2])));
          cacc[e][0] = fma(xx, Mi[g][0], fma(xy, Mi[g][1], fma(xz, Mi[g][2], cacc[e][0])));
          cacc[e][1] = fma(xy, Mi[g][0], fma(yy, Mi[g][1], fma(yz, Mi[g][2], cacc[e][1])));
          cacc[e][2] = fma(xz, Mi[g][0], fma(yz, Mi[g][1], fma(zz, Mi[g][2], cacc[e][2])));
        }
      // column part of this tile: sum over the 8 row-lanes (fixed butterfly), one store per column
#pragma unroll
      for (int e = 0; e < W; ++e)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          T s = cacc[e][c];
          s += __shfl_xor_sync(0xffffffffu, s, 4);
          s += __shfl_xor_sync(0xffffffffu, s, 8);
          s += __shfl_xor_sync(0xffffffffu, s, 16);
          cacc[e][c] = s;
        }
      if (rl == 0 && use_col) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          T* dst = colpart + ((int64_t)I * 3 + c) * a.ncolpad + j0;
#pragma unroll
          for (int e = 0; e < W; ++e) dst[e] = cacc[e][c];
        }
      }
      if (sizeof(T) == 8 || ++since == kFlushTiles) {
        since = 0;
#pragma unroll
        for (int g = 0; g < 4; ++g)
#pragma unroll
          for (int c = 0; c < 3; ++c) { racc[g][c] += (double)rrun[g][c]; rrun[g][c] = T(0); }
      }
    }
    // row part of the block: flush, reduce over the 4 column-quad lanes, then over the 8 warps
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        double s = racc[g][c] + (double)rrun[g][c];
        s += __shfl_xor_sync(0xffffffffu, s, 1);
        s += __shfl_xor_sync(0xffffffffu, s, 2);
        if (cq == 0) red[warp][8 * g + rl][c] = s;
      }
    __syncthreads();
    if (threadIdx.x < 96) {
      const int it = threadIdx.x / 3, c = threadIdx.x % 3;
      double s = 0.0;
#pragma unroll
      for (int w = 0; w < 8; ++w) s += red[w][it][c];
      a.rowpart[(int64_t)c * a.nrowpad + 32 * I + it] = s;
    }
    __syncthreads();
  }
}

// H_d,j = -(rowpart_j + sum_{I < j/32} colpart[I][.][j]) in fixed order, then the fused epilogue
template <typename T>
__global__ void __launch_bounds__(256) sym_finish_kernel(SymArgs a, int b, EpiArgs e) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= a.n) return;
  const T* colpart = (const T*)a.colpart;
  const int64_t jb = j >> 5;
  double s[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) s[c] = a.rowpart[(int64_t)c * a.nrowpad + j];
  for (int64_t I = 0; I < jb; ++I)
#pragma unroll
    for (int c = 0; c < 3; ++c) s[c] += (double)colpart[(I * 3 + c) * a.ncolpad + j];
  const double hd[3] = {-s[0], -s[1], -s[2]};
  row_epilogue(e, j, b, hd);
}

template <typename T>
int launch_sym_T(mt_ctx* ctx, const mt_sym_tensor* S, const void* Mst, int64_t npad, const EpiArgs& e) {
  typedef SymCfg<T> Cfg;
  SymArgs a;
  a.n = S->n;
  a.nrb = sym_row_blocks(S->n);
  a.ntc = sym_col_tiles(S->n, Cfg::TW);
  a.npad = npad;
  a.ncolpad = a.ntc * Cfg::TW;
  a.nrowpad = a.nrb * 32;
  a.data = S->data;
  const size_t row_bytes = (size_t)3 * a.nrowpad * sizeof(double);
  const size_t col_bytes = (size_t)a.nrb * 3 * a.ncolpad * sizeof(T);
  int rc = mt_ensure_ws(ctx, (void**)&ctx->sym_ws, &ctx->sym_ws_bytes, row_bytes + col_bytes);
  if (rc) return rc;
  a.rowpart = (double*)ctx->sym_ws;
  a.colpart = (char*)ctx->sym_ws + row_bytes;
  const unsigned grid = (unsigned)((a.nrb + 1) / 2);
  static unsigned char attr_set[64] = {};  // per device ordinal (the attribute is per device)
  if (!attr_set[ctx->device & 63]) {
    MT_CUDA_OK(ctx, cudaFuncSetAttribute(sym_field_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSymSmemBytes));
    attr_set[ctx->device & 63] = 1;
  }
  for (int b = 0; b < e.batch; ++b) {  // states one after the other: each streams the half once
    a.Mst = (const T*)Mst + (int64_t)b * 3 * npad;
    sym_field_kernel<T><<<grid, 256, kSymSmemBytes, ctx->stream>>>(a);
    ctx->launches++;
    MT_CUDA_OK(ctx, cudaGetLastError());
    sym_finish_kernel<T><<<(unsigned)((S->n + 255) / 256), 256, 0, ctx->stream>>>(a, b, e);
    ctx->launches++;
    MT_CUDA_OK(ctx, cudaGetLastError());
  }
  return MT_OK;
}

}  // namespace

int mt_launch_demag_sym(mt_ctx* ctx, const mt_sym_tensor* S, const void* Mst, int64_t npad, const EpiArgs& e) {
  const bool prof = ctx->prof_on && ctx->prof_ev && ctx->prof_count < MT_PROF_CAP;
  if (prof) MT_CUDA_OK(ctx, cudaEventRecord(ctx->prof_ev[2 * ctx->prof_count], ctx->stream));
  const int rc = S->dtype == MT_F32 ? launch_sym_T<float>(ctx, S, Mst, npad, e) : launch_sym_T<double>(ctx, S, Mst, npad, e);
  if (prof) {
    MT_CUDA_OK(ctx, cudaEventRecord(ctx->prof_ev[2 * ctx->prof_count + 1], ctx->stream));
    ctx->prof_count++;
  }
  return rc;
}
