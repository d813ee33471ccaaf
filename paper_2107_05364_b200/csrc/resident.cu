// resident.cu — A8 (RK4) for problems whose whole demagnetization tensor fits in the shared memory of
// the GPU's SMs together (148 x 227 KB = 33 MB on a B200: N <= ~740 tiles fp64, ~1,100 fp32 — the sizes the
// paper itself runs, N = 100 n^2 <= 8,100 with SP4 converged from n = 3).
//
// At these sizes a right-hand side is a few microseconds of L2 streaming and the step is bound by launch
// latency ("small N").  Here one cooperative launch integrates a whole chunk of steps:
// every CTA loads its R rows of the six component planes into shared memory ONCE; then, for every stage of
// every step, it reads the stage state of all tiles (3 n doubles per state, from L2) into shared memory,
// rounds Ms*m to the tensor's dtype, multiplies its resident rows with it (H_d = -N.M), and
// one thread per (row, state) adds exchange, anisotropy and the applied field (Eq. 12, 16, 7: PAPER.md:94,114,70;
// neighbours come from the shared-memory copy of the state), forms the Landau-Lifshitz right-hand side (Eq. 1,
// PAPER.md:33) and the Runge-Kutta stage state, of which it writes its three numbers; the row's constants,
// the step's start state and the slopes k1..k3 stay in that thread's registers.  A grid barrier ends the
// stage — the only thing left between two right-hand sides.  The tensor is read from HBM/L2 once per launch
// instead of once per right-hand side; per stage a CTA moves 24 n bytes per state from L2 and 24 bytes per
// row to it.  The arithmetic of a row is that of epilogue.cuh's row_epilogue / stage_combine, term by term.
//
// Deterministic: a row's columns are split over WPR warps, lanes stride the columns, fixed xor butterfly,
// the warps' parts added in warp order.  fp32 tensors: fp32 products and per-lane partial sums over at most
// 36 terms (n <= ~1,100, Q19 allows 128), then fp64.
#include "epilogue.cuh"

namespace {

constexpr int kResThreads = 256;
constexpr int kResWarps = kResThreads / 32;

struct ResArgs {
  const void* N;  // [6][n][ld]
  int64_t n, ld;
  int R;          // rows per CTA
  int wpr;        // warps per row (power of two, R * wpr <= 8)
  int batch;
  int renorm;
  int64_t ldS;    // shared-memory row length in elements (multiple of the 16-byte vector, >= n)
  int64_t count;  // steps of this launch
  unsigned long long* tq;    // per-step torque words (stop test, Eq. 2) or NULL
  unsigned int* bar;         // grid barrier counter (zero at launch)
  const double* y_in[4];     // stage states [B][3][n]: m, ya, yb, ya
  double* y_to[4];           //                          ya, yb, ya, m
  double h[4];               // dt/2, dt/2, dt, dt/6
  EpiArgs prob;              // the problem's constants (fill_problem); no pointers into the integrator
};

template <typename T> struct Vec;
template <> struct Vec<float> { typedef float4 type; static constexpr int W = 4; };
template <> struct Vec<double> { typedef double2 type; static constexpr int W = 2; };

__device__ __forceinline__ void block3(float acc[3], float xx, float xy, float xz, float yy, float yz, float zz,
                                       float mx, float my, float mz) {
  acc[0] = fmaf(xx, mx, fmaf(xy, my, fmaf(xz, mz, acc[0])));
  acc[1] = fmaf(xy, mx, fmaf(yy, my, fmaf(yz, mz, acc[1])));
  acc[2] = fmaf(xz, mx, fmaf(yz, my, fmaf(zz, mz, acc[2])));
}
__device__ __forceinline__ void block3(double acc[3], double xx, double xy, double xz, double yy, double yz,
                                       double zz, double mx, double my, double mz) {
  acc[0] = fma(xx, mx, fma(xy, my, fma(xz, mz, acc[0])));
  acc[1] = fma(xy, mx, fma(yy, my, fma(yz, mz, acc[1])));
  acc[2] = fma(xz, mx, fma(yz, my, fma(zz, mz, acc[2])));
}
__device__ __forceinline__ void vec3(float acc[3], const float4 t[6], const float4 m[3]) {
  block3(acc, t[0].x, t[1].x, t[2].x, t[3].x, t[4].x, t[5].x, m[0].x, m[1].x, m[2].x);
  block3(acc, t[0].y, t[1].y, t[2].y, t[3].y, t[4].y, t[5].y, m[0].y, m[1].y, m[2].y);
  block3(acc, t[0].z, t[1].z, t[2].z, t[3].z, t[4].z, t[5].z, m[0].z, m[1].z, m[2].z);
  block3(acc, t[0].w, t[1].w, t[2].w, t[3].w, t[4].w, t[5].w, m[0].w, m[1].w, m[2].w);
}
__device__ __forceinline__ void vec3(double acc[3], const double2 t[6], const double2 m[3]) {
  block3(acc, t[0].x, t[1].x, t[2].x, t[3].x, t[4].x, t[5].x, m[0].x, m[1].x, m[2].x);
  block3(acc, t[0].y, t[1].y, t[2].y, t[3].y, t[4].y, t[5].y, m[0].y, m[1].y, m[2].y);
}
__device__ __forceinline__ float4 zero_from(float4 v, int64_t j, int64_t n) {
  if (j + 0 >= n) v.x = 0.f;
  if (j + 1 >= n) v.y = 0.f;
  if (j + 2 >= n) v.z = 0.f;
  if (j + 3 >= n) v.w = 0.f;
  return v;
}
__device__ __forceinline__ double2 zero_from(double2 v, int64_t j, int64_t n) {
  if (j + 0 >= n) v.x = 0.0;
  if (j + 1 >= n) v.y = 0.0;
  return v;
}

// Grid barrier: the launch is cooperative (all CTAs co-resident), the counter only grows.  Writes of the
// CTA's threads are ordered before thread 0's releasing add by the CTA barrier, and thread 0's acquiring poll
// before the CTA's later reads by the second one.
__device__ __forceinline__ void grid_barrier(unsigned int* ctr, unsigned int target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(ctr), "r"(1u) : "memory");
    unsigned int seen;
    do {
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(ctr) : "memory");
    } while (seen < target);
  }
  __syncthreads();
}

// Shared memory: tens[R][6][ldS] T | Msh[B][3][ldS] T | ysh[B][3][n] double | Mss[n] double | red[B][8][3] double
template <typename T>
__global__ void __launch_bounds__(kResThreads, 1) rk4_resident_kernel(const __grid_constant__ ResArgs a) {
  typedef typename Vec<T>::type V;
  constexpr int W = Vec<T>::W;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int64_t n = a.n, ldS = a.ldS;
  const int64_t nv = ldS / W;  // vectors per shared-memory row (covers all n columns)
  const int B = a.batch;
  const int64_t r0 = (int64_t)blockIdx.x * a.R;
  const int rows = (int)min((int64_t)a.R, n - r0);
  V* tens = reinterpret_cast<V*>(smem_raw);
  V* Msh = tens + (int64_t)a.R * 6 * nv;
  double* ysh = reinterpret_cast<double*>(Msh + (int64_t)B * 3 * nv);
  double* Mss = ysh + (int64_t)B * 3 * n;
  double* red = Mss + n;
  const EpiArgs& e = a.prob;

  // ---- once per launch: the CTA's rows of the six planes (columns >= n read as zero), Ms, zeroed M ----
  {
    const T* N = (const T*)a.N;
    const int64_t plane = n * a.ld;
    const int64_t tot = (int64_t)rows * 6 * nv;
    for (int64_t idx = tid; idx < tot; idx += kResThreads) {
      const int64_t v = idx % nv;
      const int c = (int)((idx / nv) % 6);
      const int r = (int)(idx / (6 * nv));
      const V x = __ldcs(reinterpret_cast<const V*>(N + c * plane + (r0 + r) * a.ld) + v);
      tens[((int64_t)r * 6 + c) * nv + v] = zero_from(x, v * W, n);
    }
    for (int64_t j = tid; j < n; j += kResThreads) Mss[j] = e.Ms[j];
    T* Mz = reinterpret_cast<T*>(Msh);
    for (int64_t idx = tid; idx < (int64_t)B * 3 * ldS; idx += kResThreads) Mz[idx] = T(0);
  }
  // ---- the epilogue thread of (row i, state b) keeps the row's constants and the step's slopes ----
  const bool epi = tid < rows * B;
  const int er = epi ? tid % rows : 0, eb = epi ? tid / rows : 0;
  const int64_t i = r0 + er;
  int32_t nb[6] = {-1, -1, -1, -1, -1, -1};
  double cex = 0.0, can = 0.0, ax[3] = {0.0, 0.0, 0.0}, ha[3] = {0.0, 0.0, 0.0};
  if (epi) {
    if (e.nbr) {
#pragma unroll
      for (int q = 0; q < 6; ++q) nb[q] = e.nbr[6 * i + q];
      cex = e.c_ex ? e.c_ex[i] : e.c_ex_s;
    }
    can = e.c_an ? e.c_an[i] : e.c_an_s;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      ax[c] = e.easy ? e.easy[3 * i + c] : e.easy_c[c];
      ha[c] = e.H_a ? e.H_a[3 * i + c] : e.H_a_c[c];
    }
  }
  double base[3] = {0.0, 0.0, 0.0}, ks[3][3];
#pragma unroll
  for (int q = 0; q < 3; ++q) ks[q][0] = ks[q][1] = ks[q][2] = 0.0;
  __syncthreads();

  const int row = warp / a.wpr, seg = warp % a.wpr;
  const int64_t per = (nv + a.wpr - 1) / a.wpr;
  const int64_t v0 = (int64_t)seg * per, v1 = min(nv, v0 + per);
  const V* trow = tens + (int64_t)row * 6 * nv;
  unsigned int bar_target = 0;

  for (int64_t step = 0; step < a.count; ++step) {
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      // the stage state of all tiles (written by every CTA's epilogue threads: L2, not L1), and Ms*m in the
      // tensor's dtype, rounded once (Q19)
      {
        const double* yin = a.y_in[s];
        T* Ms_ = reinterpret_cast<T*>(Msh);
        const int n32 = (int)n, ld32 = (int)ldS, total = 3 * B * n32;
        // eight loads in flight per thread: the stage costs one L2 round trip, not one per element
        for (int base0 = 0; base0 < total; base0 += kResThreads * 8) {
          double yv[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            const int idx = base0 + u * kResThreads + tid;
            yv[u] = idx < total ? __ldcg(yin + idx) : 0.0;
          }
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            const int idx = base0 + u * kResThreads + tid;
            if (idx < total) {
              const int bc = idx / n32, j = idx - bc * n32;
              ysh[idx] = yv[u];
              Ms_[bc * ld32 + j] = (T)(Mss[j] * yv[u]);
            }
          }
        }
      }
      __syncthreads();
      if (row < rows) {
        // up to four states per pass over the row: the tensor's shared-memory rows are read once per pass
        for (int b0 = 0; b0 < B; b0 += 4) {
          T acc[4][3];
#pragma unroll
          for (int bb = 0; bb < 4; ++bb) acc[bb][0] = acc[bb][1] = acc[bb][2] = T(0);
          for (int64_t v = v0 + lane; v < v1; v += 32) {
            V t[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) t[c] = trow[c * nv + v];
#pragma unroll
            for (int bb = 0; bb < 4; ++bb)
              if (b0 + bb < B) {
                const V* Mb = Msh + (int64_t)(b0 + bb) * 3 * nv;
                V m[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) m[c] = Mb[c * nv + v];
                vec3(acc[bb], t, m);
              }
          }
#pragma unroll
          for (int bb = 0; bb < 4; ++bb)
            if (b0 + bb < B) {
              double d[3] = {(double)acc[bb][0], (double)acc[bb][1], (double)acc[bb][2]};
#pragma unroll
              for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) d[c] += __shfl_xor_sync(0xffffffffu, d[c], off);
              if (lane == 0) {
                double* o = red + ((int64_t)(b0 + bb) * kResWarps + warp) * 3;
                o[0] = d[0];
                o[1] = d[1];
                o[2] = d[2];
              }
            }
        }
      }
      __syncthreads();
      if (epi) {
        // H_d = -N.M, the warps' column parts added in warp order
        double H[3] = {0.0, 0.0, 0.0};
        for (int w = 0; w < a.wpr; ++w) {
          const double* o = red + ((int64_t)eb * kResWarps + er * a.wpr + w) * 3;
#pragma unroll
          for (int c = 0; c < 3; ++c) H[c] += o[c];
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) H[c] = -H[c];
        const double* y = ysh + (int64_t)eb * 3 * n;
        const double mi[3] = {y[i], y[n + i], y[2 * n + i]};
        // exchange: Eq. 12, 3-point stencil, Neumann ghost = self
        if (e.nbr) {
          double hx[3] = {0.0, 0.0, 0.0};
#pragma unroll
          for (int dir = 0; dir < 3; ++dir) {
            const int32_t jm = nb[2 * dir], jp = nb[2 * dir + 1];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              const double mm = jm >= 0 ? y[c * n + jm] : mi[c];
              const double mp = jp >= 0 ? y[c * n + jp] : mi[c];
              hx[c] += (mp - 2.0 * mi[c] + mm) * e.inv_d2[dir];
            }
          }
#pragma unroll
          for (int c = 0; c < 3; ++c) H[c] += cex * hx[c];
        }
        // uniaxial anisotropy: Eq. 16; applied field: Eq. 7
        const double me = mi[0] * ax[0] + mi[1] * ax[1] + mi[2] * ax[2];
#pragma unroll
        for (int c = 0; c < 3; ++c) H[c] += can * me * ax[c] + ha[c];
        // Landau-Lifshitz: Eq. 1
        double mxH[3], mxmxH[3], k[3];
        cross3(mi, H, mxH);
        cross3(mi, mxH, mxmxH);
#pragma unroll
        for (int c = 0; c < 3; ++c) k[c] = -e.gamma * mxH[c] - e.alpha * mxmxH[c];
        if (s == 0) {
          if (a.tq) atomic_max_nonneg(a.tq + step, sqrt(mxH[0] * mxH[0] + mxH[1] * mxH[1] + mxH[2] * mxH[2]));
#pragma unroll
          for (int c = 0; c < 3; ++c) base[c] = mi[c];  // stage 1 is evaluated at the step's start state
        }
        double yo[3];
        if (s < 3) {
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            ks[s][c] = k[c];
            yo[c] = base[c] + a.h[s] * k[c];
          }
        } else {
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            double sum = 0.0;
            sum += 1.0 * ks[0][c];
            sum += 2.0 * ks[1][c];
            sum += 2.0 * ks[2][c];
            sum += 1.0 * k[c];
            yo[c] = base[c] + a.h[3] * sum;
          }
          if (a.renorm) {
            // a zero-length m_i stays zero (Q10c)
            const double r = sqrt(yo[0] * yo[0] + yo[1] * yo[1] + yo[2] * yo[2]);
            if (r > 0.0) {
#pragma unroll
              for (int c = 0; c < 3; ++c) yo[c] /= r;
            }
          }
        }
        double* yout = a.y_to[s] + (int64_t)eb * 3 * n + i;
#pragma unroll
        for (int c = 0; c < 3; ++c) yout[c * n] = yo[c];
      }
      bar_target += gridDim.x;
      grid_barrier(a.bar, bar_target);  // every CTA's rows of the next stage state are visible to all
    }
  }
}

size_t resident_smem(int dtype, int64_t n, int R, int batch, int64_t* ldS_out) {
  const int64_t W = dtype == MT_F32 ? 4 : 2;
  const size_t sz = dtype == MT_F32 ? 4 : 8;
  const int64_t ldS = (n + W - 1) / W * W;
  if (ldS_out) *ldS_out = ldS;
  return ((size_t)R * 6 + (size_t)batch * 3) * ldS * sz + ((size_t)batch * 3 + 1) * n * sizeof(double) +
         (size_t)batch * kResWarps * 3 * sizeof(double);
}

static_assert(sizeof(ResArgs) <= 4000, "kernel parameter space");

}  // namespace

// Can the dense n x n tensor of this dtype stay resident in shared memory across the GPU (one CTA per SM,
// ceil(n / SMs) <= 8 rows each) together with `batch` stage states?
bool mt_resident_fits(mt_ctx* ctx, int dtype, int64_t n, int batch) {
  if (n <= 0 || n > 65536 || batch < 1 || batch > MT_MAX_BATCH) return false;
  const int R = (int)((n + ctx->num_sms - 1) / ctx->num_sms);
  if (R > kResWarps || R * batch > kResThreads) return false;
  int dev_smem = 0, coop = 0;
  if (cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device) != cudaSuccess ||
      cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device) != cudaSuccess || !coop) {
    cudaGetLastError();
    return false;
  }
  return resident_smem(dtype, n, R, batch, nullptr) <= (size_t)dev_smem;
}

// `count` RK4 steps of m (in place); ya, yb: two scratch states [B][3][n]; `prob`: fill_problem's constants.
int mt_launch_rk4_resident(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t ld, const EpiArgs& prob,
                           double* m, double* ya, double* yb, double dt, int renorm,
                           unsigned long long* tq_slots, unsigned int* bar, int64_t count) {
  if (count <= 0) return MT_OK;
  ResArgs a;
  memset(&a, 0, sizeof(a));
  a.N = N;
  a.n = n;
  a.ld = ld;
  a.R = (int)((n + ctx->num_sms - 1) / ctx->num_sms);
  a.wpr = 1;
  while (a.wpr * 2 * a.R <= kResWarps) a.wpr *= 2;
  a.batch = prob.batch;
  a.renorm = renorm;
  a.count = count;
  a.tq = tq_slots;
  a.bar = bar;
  a.y_in[0] = m;  a.y_to[0] = ya; a.h[0] = 0.5 * dt;
  a.y_in[1] = ya; a.y_to[1] = yb; a.h[1] = 0.5 * dt;
  a.y_in[2] = yb; a.y_to[2] = ya; a.h[2] = dt;
  a.y_in[3] = ya; a.y_to[3] = m;  a.h[3] = dt / 6.0;
  a.prob = prob;
  const size_t smem = resident_smem(dtype, n, a.R, a.batch, &a.ldS);
  if (a.ldS > ld) return mt_fail(ctx, MT_ERR_INVALID_ARG, "resident RK4: ld must cover whole 16-byte vectors");
  const void* fn = dtype == MT_F32 ? (const void*)rk4_resident_kernel<float> : (const void*)rk4_resident_kernel<double>;
  // the attribute is per device, not per process: set it on every launch (a few microseconds per chunk)
  MT_CUDA_OK(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const unsigned grid = (unsigned)((n + a.R - 1) / a.R);
  int per_sm = 0;
  MT_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, kResThreads, smem));
  if ((int64_t)per_sm * ctx->num_sms < (int64_t)grid)
    return mt_fail(ctx, MT_ERR_CUDA, "resident RK4: %u CTAs cannot be co-resident on this device", grid);
  MT_CUDA_OK(ctx, cudaMemsetAsync(bar, 0, sizeof(unsigned int), ctx->stream));
  void* args[] = {(void*)&a};
  MT_CUDA_OK(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(kResThreads), args, smem, ctx->stream));
  ctx->launches++;
  return MT_OK;
}
