// demag.cu — A4/A7: H_d = -N.(Ms m), register-streaming variant ("LDG"), plus the small O(N)
// kernels around it: staging of Ms*m in the tensor's dtype, split-column reduction, local-only
// right-hand side, stage combine and the <m> observable (A10).
//
// Kernel shape (HBM-bound): one warp owns one target row i and streams the
// six component rows N^{c}_{i,*} once with 128-bit non-allocating loads; the staged vector
// M = Ms*m (same dtype as the tensor) comes through L1/L2.  fp32 tensors accumulate in short fp32
// runs (8 vector iterations = 96 products per accumulator) flushed into fp64; fp64 tensors use
// DFMA directly.  The warp reduces with a fixed xor-butterfly (bitwise reproducible) and lanes
// 0..B-1 run the fused epilogue (epilogue.cuh).  For small n the columns are split over
// gridDim.y and a second kernel adds the partials in a fixed order.
#include <stdarg.h>

#include "dp_control.cuh"
#include "epilogue.cuh"

int mt_fail(mt_ctx* ctx, int code, const char* fmt, ...) {
  if (ctx) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
    va_end(ap);
  }
  return code;
}

int mt_ensure_ws(mt_ctx* ctx, void** p, size_t* cur, size_t need) {
  if (*cur >= need && *p) return MT_OK;
  if (*p) {
    MT_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
    MT_CUDA_OK(ctx, cudaFree(*p));
    *p = nullptr;
    *cur = 0;
  }
  MT_CUDA_OK(ctx, cudaMalloc(p, need));
  *cur = need;
  return MT_OK;
}

namespace {

template <typename T> struct VecOf;
template <> struct VecOf<float> { typedef float4 type; static constexpr int W = 4; };
template <> struct VecOf<double> { typedef double2 type; static constexpr int W = 2; };

// streaming (read-once) 128-bit loads: do not allocate in L1
__device__ __forceinline__ float4 ld_stream(const float4* p) {
  float4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ double2 ld_stream(const double2* p) {
  double2 r;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
  return r;
}

template <typename A>
__device__ __forceinline__ void fma_block(A acc[3], float xx, float xy, float xz, float yy, float yz,
                                          float zz, float mx, float my, float mz) {
  acc[0] = fmaf(xx, mx, fmaf(xy, my, fmaf(xz, mz, acc[0])));
  acc[1] = fmaf(xy, mx, fmaf(yy, my, fmaf(yz, mz, acc[1])));
  acc[2] = fmaf(xz, mx, fmaf(yz, my, fmaf(zz, mz, acc[2])));
}
__device__ __forceinline__ void fma_block(double acc[3], double xx, double xy, double xz, double yy,
                                          double yz, double zz, double mx, double my, double mz) {
  acc[0] = fma(xx, mx, fma(xy, my, fma(xz, mz, acc[0])));
  acc[1] = fma(xy, mx, fma(yy, my, fma(yz, mz, acc[1])));
  acc[2] = fma(xz, mx, fma(yz, my, fma(zz, mz, acc[2])));
}

__device__ __forceinline__ void vec_fma(float acc[3], const float4 v[6], const float4 m[3]) {
  fma_block(acc, v[0].x, v[1].x, v[2].x, v[3].x, v[4].x, v[5].x, m[0].x, m[1].x, m[2].x);
  fma_block(acc, v[0].y, v[1].y, v[2].y, v[3].y, v[4].y, v[5].y, m[0].y, m[1].y, m[2].y);
  fma_block(acc, v[0].z, v[1].z, v[2].z, v[3].z, v[4].z, v[5].z, m[0].z, m[1].z, m[2].z);
  fma_block(acc, v[0].w, v[1].w, v[2].w, v[3].w, v[4].w, v[5].w, m[0].w, m[1].w, m[2].w);
}
__device__ __forceinline__ void vec_fma(double acc[3], const double2 v[6], const double2 m[3]) {
  fma_block(acc, v[0].x, v[1].x, v[2].x, v[3].x, v[4].x, v[5].x, m[0].x, m[1].x, m[2].x);
  fma_block(acc, v[0].y, v[1].y, v[2].y, v[3].y, v[4].y, v[5].y, m[0].y, m[1].y, m[2].y);
}

template <typename T>
struct DemagArgs {
  const T* N;
  int64_t n, n_rows, ld, plane;  // plane = n_rows * ld
  const T* M;                    // [B][3][npad]
  int64_t npad;
  int64_t vec_per_split;         // full vectors per column split
  int nsplit;
  double* partial;               // [nsplit][B][3][n_rows] when nsplit > 1
  const double* Ms;              // FUSE: M is formed on the fly as (T)(Ms[j] * y[b][c][j]) — the same expression,
  const double* y;               // hence the same bits, as stage_M_kernel's — instead of read from the staged M
};

// FUSE: the 16 bytes of M a lane needs, from Ms and the state (n a multiple of the vector width: no tail)
__device__ __forceinline__ void fused_ms(const double* Ms, int64_t v, double (&ms)[4]) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(Ms) + 2 * v), b = __ldg(reinterpret_cast<const double2*>(Ms) + 2 * v + 1);
  ms[0] = a.x; ms[1] = a.y; ms[2] = b.x; ms[3] = b.y;
}
__device__ __forceinline__ void fused_ms(const double* Ms, int64_t v, double (&ms)[2]) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(Ms) + v);
  ms[0] = a.x; ms[1] = a.y;
}
__device__ __forceinline__ float4 fused_m(const double* yrow, int64_t v, const double (&ms)[4]) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(yrow) + 2 * v), b = __ldg(reinterpret_cast<const double2*>(yrow) + 2 * v + 1);
  return make_float4((float)(ms[0] * a.x), (float)(ms[1] * a.y), (float)(ms[2] * b.x), (float)(ms[3] * b.y));
}
__device__ __forceinline__ double2 fused_m(const double* yrow, int64_t v, const double (&ms)[2]) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(yrow) + v);
  return make_double2(ms[0] * a.x, ms[1] * a.y);
}

constexpr int kWarps = 8;
constexpr int kFlush = 8;  // fp32: vector iterations per fp32 run

template <typename T, int B, bool FUSE>
__global__ void __launch_bounds__(kWarps * 32) demag_ldg_kernel(DemagArgs<T> a, EpiArgs e) {
  typedef typename VecOf<T>::type V;
  constexpr int W = VecOf<T>::W;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * kWarps + warp;
  if (row >= a.n_rows) return;
  if (e.active_dev && !*e.active_dev) return;  // replayed attempt of a finished device-controlled DP45 run
  const int split = blockIdx.y;
  const int64_t nvec = a.n / W;
  const int64_t v0 = (int64_t)split * a.vec_per_split;
  const int64_t v1 = min(nvec, v0 + a.vec_per_split);
  const V* p[6];
#pragma unroll
  for (int c = 0; c < 6; ++c) p[c] = reinterpret_cast<const V*>(a.N + c * a.plane + row * a.ld);
  const V* mp = reinterpret_cast<const V*>(a.M);
  const int64_t mstride = a.npad / W;  // vectors per component row of M

  double acc[B][3];
#pragma unroll
  for (int b = 0; b < B; ++b) acc[b][0] = acc[b][1] = acc[b][2] = 0.0;

  for (int64_t vb = v0 + lane; vb < v1; vb += 32 * kFlush) {
    T run[B][3];
#pragma unroll
    for (int b = 0; b < B; ++b) run[b][0] = run[b][1] = run[b][2] = T(0);
#pragma unroll 2
    for (int it = 0; it < kFlush; ++it) {
      const int64_t v = vb + (int64_t)it * 32;
      if (v < v1) {
        V t[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) t[c] = ld_stream(p[c] + v);
        double ms[W];
        if constexpr (FUSE) fused_ms(a.Ms, v, ms);
#pragma unroll
        for (int b = 0; b < B; ++b) {
          V m[3];
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            if constexpr (FUSE) m[c] = fused_m(a.y + (int64_t)(b * 3 + c) * a.n, v, ms);
            else m[c] = __ldg(mp + (b * 3 + c) * mstride + v);
          }
          vec_fma(run[b], t, m);
        }
      }
    }
#pragma unroll
    for (int b = 0; b < B; ++b) {
      acc[b][0] += (double)run[b][0];
      acc[b][1] += (double)run[b][1];
      acc[b][2] += (double)run[b][2];
    }
  }
  // scalar tail (n not a multiple of the vector width): last split, one lane per leftover column
  if (split == a.nsplit - 1) {
    const int64_t j = nvec * W + lane;
    if (j < a.n) {
#pragma unroll
      for (int b = 0; b < B; ++b) {
        T t[6], m[3];
#pragma unroll
        for (int c = 0; c < 6; ++c) t[c] = a.N[c * a.plane + row * a.ld + j];
#pragma unroll
        for (int c = 0; c < 3; ++c) m[c] = a.M[(b * 3 + c) * a.npad + j];
        T run[3] = {T(0), T(0), T(0)};
        fma_block(run, t[0], t[1], t[2], t[3], t[4], t[5], m[0], m[1], m[2]);
        acc[b][0] += (double)run[0];
        acc[b][1] += (double)run[1];
        acc[b][2] += (double)run[2];
      }
    }
  }
  // fixed-order butterfly: every lane ends with the same, reproducible sum
#pragma unroll
  for (int b = 0; b < B; ++b)
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) acc[b][c] += __shfl_xor_sync(0xffffffffu, acc[b][c], off);

  if (a.nsplit > 1) {
    if (lane == 0) {
#pragma unroll
      for (int b = 0; b < B; ++b)
#pragma unroll
        for (int c = 0; c < 3; ++c)
          a.partial[(((int64_t)split * B + b) * 3 + c) * a.n_rows + row] = acc[b][c];
    }
    return;
  }
  // lanes 0..B-1 each finish one state (static selection keeps acc[][] in registers)
  double hd[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int b = 0; b < B; ++b)
    if (lane == b) {
      hd[0] = -acc[b][0];
      hd[1] = -acc[b][1];
      hd[2] = -acc[b][2];
    }
  if (lane < B) row_epilogue(e, row, lane, hd);
}

// second pass for nsplit > 1: add the partials in split order, then the epilogue
__global__ void __launch_bounds__(256) demag_reduce_kernel(const double* partial, int nsplit, int B,
                                                           int64_t n_rows, EpiArgs e) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_rows * B) return;
  const int b = (int)(idx / n_rows);
  const int64_t row = idx % n_rows;
  double hd[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    double s = 0.0;
    for (int sp = 0; sp < nsplit; ++sp) s += partial[(((int64_t)sp * B + b) * 3 + c) * n_rows + row];
    hd[c] = -s;
  }
  row_epilogue(e, row, b, hd);
}

// both walk the launch's rows (all n, or a rank's band [row0, row0 + n_rows) of a sharded problem)
__global__ void __launch_bounds__(256) local_only_kernel(EpiArgs e) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= e.n_rows * e.batch) return;
  const double hd[3] = {0.0, 0.0, 0.0};
  row_epilogue(e, idx % e.n_rows, (int)(idx / e.n_rows), hd);
}

__global__ void __launch_bounds__(256) combine_kernel(EpiArgs e) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= e.n_rows * e.batch) return;
  if (e.active_dev && !*e.active_dev) return;
  stage_combine(e, e.row0 + idx % e.n_rows, (int)(idx / e.n_rows), nullptr);
}

// ---- device-resident DP45 controller (A9): dp_control.cuh's rules run by one thread ----------------------
__global__ void dp_begin_kernel(DpState* s) { dp_begin(s); }
__global__ void dp_decide_kernel(DpState* s) { dp_decide(s); }

// accepted: m <- candidate, k1 <- k7 (FSAL; the host controller swaps pointers, a replayed graph cannot)
__global__ void __launch_bounds__(256) dp_commit_kernel(const DpState* s, double* __restrict__ m,
                                                        const double* __restrict__ mc, double* __restrict__ k1,
                                                        const double* __restrict__ k7, int64_t count) {
  if (!s->accept) return;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  m[i] = mc[i];
  k1[i] = k7[i];
}

// Row-sharded problems (mt.h section 8(e)): after the all-gather, block g of `pack` holds rows
// [g n / world, (g+1) n / world) of the next stage state as [B][3][pad]; scatter into y[B][3][n] and
// stage M = Ms*y in the tensor's dtype (padding j in [n, npad) zeroed as stage_M_kernel does).
template <typename T>
__global__ void __launch_bounds__(256) unpack_kernel(const double* __restrict__ pack, int world, int64_t pad,
                                                     int64_t n, int64_t npad, int rows /* B*3 */,
                                                     const double* __restrict__ Ms, double* __restrict__ y,
                                                     T* __restrict__ M) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int r = blockIdx.y;
  if (j >= npad || r >= rows) return;
  if (j >= n) {
    if (M) M[(int64_t)r * npad + j] = T(0);
    return;
  }
  // owner of row j under the band rule begin(g) = g n / world: the largest g with begin(g) <= j
  int g = (int)(((unsigned __int128)(j + 1) * (unsigned __int128)world - 1) / (unsigned __int128)n);
  while (g + 1 < world && (int64_t)(((unsigned __int128)(g + 1) * (unsigned __int128)n) / (unsigned)world) <= j) ++g;
  while (g > 0 && (int64_t)(((unsigned __int128)g * (unsigned __int128)n) / (unsigned)world) > j) --g;
  const int64_t b0 = (int64_t)(((unsigned __int128)g * (unsigned __int128)n) / (unsigned)world);
  const double v = pack[((int64_t)g * rows + r) * pad + (j - b0)];
  y[(int64_t)r * n + j] = v;
  if (M) M[(int64_t)r * npad + j] = (T)(Ms[j] * v);
}

// M[b][c][j] = T(Ms[j] * m[b][c][j]), zero in the padding j in [n, npad)
template <typename T>
__global__ void __launch_bounds__(256) stage_M_kernel(const double* __restrict__ Ms, const double* __restrict__ m,
                                                      int64_t n, int64_t npad, int rows /* B*3 */, T* __restrict__ M) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int r = blockIdx.y;
  if (j >= npad || r >= rows) return;
  M[(int64_t)r * npad + j] = j < n ? (T)(Ms[j] * m[(int64_t)r * n + j]) : T(0);
}

// A10: <m_c> of state b = sum_i w_i m_i / sum_i w_i; one block per (c, b), fixed-order tree.
__global__ void __launch_bounds__(1024) mean_kernel(const double* __restrict__ m, const double* __restrict__ vol,
                                                    int64_t n, int batch, double t, double* __restrict__ out) {
  __shared__ double sh[1024], shw[1024];
  const int c = blockIdx.x, b = blockIdx.y;
  const double* v = m + ((int64_t)b * 3 + c) * n;
  double s = 0.0, w = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += 1024) {
    const double wi = vol ? vol[i] : 1.0;
    s += wi * v[i];
    w += wi;
  }
  sh[threadIdx.x] = s;
  shw[threadIdx.x] = w;
  __syncthreads();
  for (int off = 512; off > 0; off >>= 1) {
    if ((int)threadIdx.x < off) {
      sh[threadIdx.x] += sh[threadIdx.x + off];
      shw[threadIdx.x] += shw[threadIdx.x + off];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    out[1 + b * 3 + c] = sh[0] / shw[0];
    if (c == 0 && b == 0) out[0] = t;
  }
}

// the same observable, written only when the device-resident DP45 controller flagged a sample
__global__ void __launch_bounds__(1024) mean_cond_kernel(const DpState* st, const double* __restrict__ m,
                                                         const double* __restrict__ vol, int64_t n, int batch,
                                                         double* __restrict__ samples, int64_t stride) {
  if (!st->sample_flag) return;
  __shared__ double sh[1024], shw[1024];
  const int c = blockIdx.x, b = blockIdx.y;
  const double* v = m + ((int64_t)b * 3 + c) * n;
  double s = 0.0, w = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += 1024) {
    const double wi = vol ? vol[i] : 1.0;
    s += wi * v[i];
    w += wi;
  }
  sh[threadIdx.x] = s;
  shw[threadIdx.x] = w;
  __syncthreads();
  for (int off = 512; off > 0; off >>= 1) {
    if ((int)threadIdx.x < off) {
      sh[threadIdx.x] += sh[threadIdx.x + off];
      shw[threadIdx.x] += shw[threadIdx.x + off];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double* out = samples + st->sample_row * stride;
    out[1 + b * 3 + c] = sh[0] / shw[0];
    if (c == 0 && b == 0) out[0] = st->sample_t;
  }
}

// F4: E[b][term] = sum_i e_dens[b][term][i] (one block per (term, b), fixed-order tree: bitwise
// reproducible); the total is added by the last launch's thread 0 of term 0 in a second tiny kernel.
__global__ void __launch_bounds__(1024) energy_reduce_kernel(const double* __restrict__ e_dens, int64_t n,
                                                             double* __restrict__ out) {
  __shared__ double sh[1024];
  const int term = blockIdx.x, b = blockIdx.y;
  const double* v = e_dens + ((int64_t)b * 4 + term) * n;
  double s = 0.0;
  for (int64_t i = threadIdx.x; i < n; i += 1024) s += v[i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int off = 512; off > 0; off >>= 1) {
    if ((int)threadIdx.x < off) sh[threadIdx.x] += sh[threadIdx.x + off];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[b * 5 + term] = sh[0];
}
__global__ void energy_total_kernel(int batch, double* __restrict__ out) {
  const int b = threadIdx.x;
  if (b < batch) out[b * 5 + 4] = ((out[b * 5] + out[b * 5 + 1]) + out[b * 5 + 2]) + out[b * 5 + 3];
}

template <typename T, int B>
int launch_ldg_T(mt_ctx* ctx, const DemagArgs<T>& a, const EpiArgs& e) {
  dim3 grid((unsigned)((a.n_rows + kWarps - 1) / kWarps), (unsigned)a.nsplit);
  if (a.y) demag_ldg_kernel<T, B, true><<<grid, kWarps * 32, 0, ctx->stream>>>(a, e);
  else demag_ldg_kernel<T, B, false><<<grid, kWarps * 32, 0, ctx->stream>>>(a, e);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  if (a.nsplit > 1) {
    const int64_t tot = a.n_rows * B;
    demag_reduce_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, ctx->stream>>>(a.partial, a.nsplit, B, a.n_rows, e);
    ctx->launches++;
    MT_CUDA_OK(ctx, cudaGetLastError());
  }
  return MT_OK;
}

template <typename T>
int launch_ldg(mt_ctx* ctx, const void* N, int64_t n, int64_t n_rows, int64_t ld, const void* Mst,
               int64_t npad, const EpiArgs& e, const double* Ms_fuse, const double* y_fuse) {
  constexpr int W = VecOf<T>::W;
  DemagArgs<T> a;
  a.N = (const T*)N;
  a.n = n;
  a.n_rows = n_rows;
  a.ld = ld;
  a.plane = n_rows * ld;
  a.M = (const T*)Mst;
  a.npad = npad;
  a.Ms = Ms_fuse;
  a.y = y_fuse;
  // split the columns when the rows alone cannot fill the machine twice over
  const int64_t ctas = (n_rows + kWarps - 1) / kWarps;
  const int64_t want = 2LL * ctx->num_sms;
  int nsplit = 1;
  const int64_t nvec = n / W;
  if (ctas < want) {
    nsplit = (int)((want + ctas - 1) / ctas);
    const int64_t max_split = (nvec + 255) / 256;  // keep >= 256 vectors per split
    if (nsplit > max_split) nsplit = (int)(max_split > 0 ? max_split : 1);
    if (nsplit > 64) nsplit = 64;
  }
  int64_t vps = (nvec + nsplit - 1) / nsplit;
  vps = (vps + 31) / 32 * 32;
  if (vps == 0) vps = 32;
  nsplit = (int)((nvec + vps - 1) / vps);
  if (nsplit < 1) nsplit = 1;
  a.vec_per_split = vps;
  a.nsplit = nsplit;
  a.partial = nullptr;
  if (nsplit > 1) {
    const size_t need = (size_t)nsplit * e.batch * 3 * n_rows * sizeof(double);
    int rc = mt_ensure_ws(ctx, (void**)&ctx->partial, &ctx->partial_bytes, need);
    if (rc) return rc;
    a.partial = ctx->partial;
  }
  switch (e.batch) {
    case 1: return launch_ldg_T<T, 1>(ctx, a, e);
    case 2: return launch_ldg_T<T, 2>(ctx, a, e);
    case 3: return launch_ldg_T<T, 3>(ctx, a, e);
    case 4: return launch_ldg_T<T, 4>(ctx, a, e);
    case 5: return launch_ldg_T<T, 5>(ctx, a, e);
    case 6: return launch_ldg_T<T, 6>(ctx, a, e);
    case 7: return launch_ldg_T<T, 7>(ctx, a, e);
    case 8: return launch_ldg_T<T, 8>(ctx, a, e);
  }
  return mt_fail(ctx, MT_ERR_INVALID_ARG, "batch must be in [1, %d]", MT_MAX_BATCH);
}

}  // namespace

int mt_launch_stage_M(mt_ctx* ctx, int dtype, const double* Ms, const double* m, int batch, int64_t n,
                      int64_t npad, void* M_out) {
  dim3 grid((unsigned)((npad + 255) / 256), (unsigned)(batch * 3));
  if (dtype == MT_F32)
    stage_M_kernel<float><<<grid, 256, 0, ctx->stream>>>(Ms, m, n, npad, batch * 3, (float*)M_out);
  else
    stage_M_kernel<double><<<grid, 256, 0, ctx->stream>>>(Ms, m, n, npad, batch * 3, (double*)M_out);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

static int launch_demag_variant(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                                const void* Mst, int64_t npad, const EpiArgs& epi, const double* Ms_fuse,
                                const double* y_fuse) {
  if (y_fuse) {  // the caller checked mt_demag_can_fuse: register-streaming kernel, M formed on the fly
    if (dtype == MT_F32) return launch_ldg<float>(ctx, N, n, n_rows, ld, nullptr, npad, epi, Ms_fuse, y_fuse);
    return launch_ldg<double>(ctx, N, n, n_rows, ld, nullptr, npad, epi, Ms_fuse, y_fuse);
  }
  if (ctx->variant != 1) {
    int rc = mt_launch_demag_tma(ctx, N, dtype, n, n_rows, ld, Mst, npad, epi);
    if (rc != MT_ERR_UNIMPLEMENTED) return rc;
    if (ctx->variant >= 2) return rc;
  }
  if (dtype == MT_F32) return launch_ldg<float>(ctx, N, n, n_rows, ld, Mst, npad, epi, nullptr, nullptr);
  return launch_ldg<double>(ctx, N, n, n_rows, ld, Mst, npad, epi, nullptr, nullptr);
}

// Small problems (the register-streaming kernel's range) with n a multiple of the 16-byte vector: the field
// kernel can form Ms*m itself — one launch per call instead of two (staging + field), same bits.
bool mt_demag_can_fuse(mt_ctx* ctx, int dtype, int64_t n, int64_t n_rows, const double* Ms, const double* y) {
  const int64_t W = dtype == MT_F32 ? 4 : 2;
  if (n % W || ((uintptr_t)Ms & 15) || ((uintptr_t)y & 15) || (n & 1)) return false;
  if (ctx->variant != 0) return false;  // (a forced variant keeps the staged M: mt_set_demag_variant(ctx, 1) is the A/B)
  return !mt_demag_tma_takes(ctx, dtype, n, n_rows);
}

int mt_launch_demag(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                    const void* Mst, int64_t npad, const EpiArgs& epi, const double* Ms_fuse, const double* y_fuse) {
  const bool prof = ctx->prof_on && ctx->prof_ev && ctx->prof_count < MT_PROF_CAP;
  if (prof) MT_CUDA_OK(ctx, cudaEventRecord(ctx->prof_ev[2 * ctx->prof_count], ctx->stream));
  const int rc = launch_demag_variant(ctx, N, dtype, n, n_rows, ld, Mst, npad, epi, Ms_fuse, y_fuse);
  if (prof) {
    MT_CUDA_OK(ctx, cudaEventRecord(ctx->prof_ev[2 * ctx->prof_count + 1], ctx->stream));
    ctx->prof_count++;
  }
  return rc;
}

int mt_launch_unpack(mt_ctx* ctx, const double* pack, int world, int64_t pad, int batch, int64_t n, int64_t npad,
                     const double* Ms, double* y, void* M_out, int M_dtype) {
  dim3 grid((unsigned)((npad + 255) / 256), (unsigned)(batch * 3));
  if (M_dtype == MT_F32)
    unpack_kernel<float><<<grid, 256, 0, ctx->stream>>>(pack, world, pad, n, npad, batch * 3, Ms, y, (float*)M_out);
  else
    unpack_kernel<double><<<grid, 256, 0, ctx->stream>>>(pack, world, pad, n, npad, batch * 3, Ms, y, (double*)M_out);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_local_only(mt_ctx* ctx, const EpiArgs& epi) {
  const int64_t tot = epi.n_rows * epi.batch;
  local_only_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, ctx->stream>>>(epi);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_combine(mt_ctx* ctx, const EpiArgs& epi) {
  const int64_t tot = epi.n_rows * epi.batch;
  combine_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, ctx->stream>>>(epi);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_mean(mt_ctx* ctx, const double* m, const double* vol, int batch, int64_t n, double t,
                   double* sample_row) {
  mean_kernel<<<dim3(3, (unsigned)batch), 1024, 0, ctx->stream>>>(m, vol, n, batch, t, sample_row);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_dp_begin(mt_ctx* ctx, DpState* st) {
  dp_begin_kernel<<<1, 1, 0, ctx->stream>>>(st);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_dp_decide(mt_ctx* ctx, DpState* st) {
  dp_decide_kernel<<<1, 1, 0, ctx->stream>>>(st);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_dp_commit(mt_ctx* ctx, const DpState* st, double* m, const double* mc, double* k1, const double* k7,
                        int64_t count) {
  dp_commit_kernel<<<(unsigned)((count + 255) / 256), 256, 0, ctx->stream>>>(st, m, mc, k1, k7, count);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_mean_cond(mt_ctx* ctx, const DpState* st, const double* m, const double* vol, int batch, int64_t n,
                        double* samples, int64_t stride) {
  mean_cond_kernel<<<dim3(3, (unsigned)batch), 1024, 0, ctx->stream>>>(st, m, vol, n, batch, samples, stride);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_energy_reduce(mt_ctx* ctx, const double* e_dens, int batch, int64_t n, double* E_out) {
  energy_reduce_kernel<<<dim3(4, (unsigned)batch), 1024, 0, ctx->stream>>>(e_dens, n, E_out);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  energy_total_kernel<<<1, 32, 0, ctx->stream>>>(batch, E_out);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}
