// sym.cu — F3: field from the pair-symmetric half of the tensor, layout sym_layout.cuh.
//
// Every stored block N_ij (j's 32-column block right of row block I) serves two rows of
// H_d = -N.(Ms m): row i (with M_j) and row j (with M_i), so one evaluation streams half the bytes
// of the full tensor.  Bound: HBM (3 flop/B fp32), same roofline as A4.
//
// One CTA (8 warps) walks the tiles of a row block I and then of its mirror block nrb-1-I, so every
// CTA streams the same number of tiles.  Inside a tile warp w owns 4W columns for all 32 rows:
// lane l holds, for g = 0..3, the W-column vector of row 8g + l/4 of the six planes (24 x 16-byte loads
// in flight per lane, each warp-wide load 512 contiguous bytes).
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

template <typename T>
__global__ void __launch_bounds__(256, 1) sym_field_kernel(SymArgs a) {
  typedef SymCfg<T> Cfg;
  typedef typename SymVec<T>::type V;
  constexpr int W = Cfg::W, TW = Cfg::TW;
  constexpr int kFlushTiles = 96 / (3 * W);  // fp32: 8 tiles of 12 terms per accumulator
  __shared__ double red[8][32][3];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rl = lane >> 2, cq = lane & 3;  // row-lane (0..7), column quad (0..3)
  const T* M = (const T*)a.Mst;
  T* colpart = (T*)a.colpart;
  for (int pass = 0; pass < 2; ++pass) {
    const int64_t I = pass == 0 ? (int64_t)blockIdx.x : a.nrb - 1 - (int64_t)blockIdx.x;
    if (pass == 1 && I <= (int64_t)blockIdx.x) break;  // odd count: the middle block was done in pass 0
    const int64_t Jd = (32 * I) / TW;
    const int64_t tile0 = sym_tile_prefix(I, a.ntc, Cfg::kBlocksPerTile);
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
    for (int64_t J = Jd; J < a.ntc; ++J) {
      const V* tp = (const V*)((const T*)a.data + (tile0 + (J - Jd)) * Cfg::kTileElems) + warp * 32 + lane;
      V v[6][4];
#pragma unroll
      for (int p = 0; p < 6; ++p)
#pragma unroll
        for (int g = 0; g < 4; ++g) v[p][g] = ld_stream(tp + (p * 4 + g) * 256);
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
  for (int b = 0; b < e.batch; ++b) {  // states one after the other: each streams the half once
    a.Mst = (const T*)Mst + (int64_t)b * 3 * npad;
    sym_field_kernel<T><<<grid, 256, 0, ctx->stream>>>(a);
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
