// resident.cu — A8 (RK4) and A9 (DP45) for problems whose whole demagnetization tensor fits in the shared memory of
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
// Tensors too large for shared memory but small enough to stay in L2 (<= 100 MB) run the same kernels with
// STREAM = true: the CTA's rows (<= 32) are read from L2 at every stage, everything else is unchanged.
//
// Deterministic: a row's columns are split over WPR warps, lanes stride the columns, fixed xor butterfly,
// the warps' parts added in warp order.  fp32 tensors: fp32 products and per-lane partial sums over at most
// 36 terms (n <= ~1,100, Q19 allows 128), then fp64.
#include "dp_control.cuh"
#include "epilogue.cuh"

namespace {

constexpr int kResThreads = 256;
constexpr int kResWarps = kResThreads / 32;
constexpr int kStreamUnroll = 2;  // row vectors in flight per lane when the tensor is read from L2 (A/B: 1..4)
constexpr int kColQ = 5;  // columns per thread of the stage state: n <= kColQ * kResThreads = 1,280

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

// The resident machinery both integrators share.  Shared memory:
//   STREAM = false (tensor resident in shared memory):
//     tens[R][6][ldS] T | Msh[B][3][ldS] T | ysh[B][3][n] double | red[B][8][3] double | extra
//   STREAM = true (tensor too large for shared memory but small enough for L2: the rows are read from L2 at every
//   stage, one or two warps per row, kResWarps / wpr rows at a time; nothing else changes):
//     Msh[B][3][ldS] T | ysh[B][3][n] double | Mss[n] double | red[B][R][8][3] double | extra
template <typename T, bool STREAM>
struct Resident {
  typedef typename Vec<T>::type V;
  static constexpr int W = Vec<T>::W;
  V* tens; V* Msh; double* ysh; double* red; double* Mss; unsigned char* extra;
  const V* trow;
  const T* Ng;     // STREAM: the tensor in global memory
  int64_t ldg;     //         and its row pitch
  int64_t n, ldS, nv, r0, v0, v1, i;
  int B, R, rows, wpr, row, tid, warp, lane, er, eb;
  bool epi;  // this thread finishes (row i = r0 + er, state eb)
  // the row's constants (epilogue threads)
  int32_t nb[6];
  double cex, can, ax[3], ha[3];
  double msj[kColQ];  // Ms of the columns tid + 256 q (every thread: the stage state's staging)

  // carve the shared memory, load the CTA's rows of the six planes (columns >= n read as zero), Ms, zero M
  __device__ __forceinline__ void init(unsigned char* smem, const void* Nptr, int64_t n_, int64_t ld, int64_t ldS_, int R_,
                                       int wpr_, int B_, const EpiArgs& e) {
    n = n_; ldS = ldS_; R = R_; wpr = wpr_; B = B_;
    nv = ldS / W;
    tid = threadIdx.x; warp = tid >> 5; lane = tid & 31;
    r0 = (int64_t)blockIdx.x * R;
    rows = (int)min((int64_t)R, n - r0);
    tens = reinterpret_cast<V*>(smem);
    Msh = STREAM ? tens : tens + (int64_t)R * 6 * nv;
    ysh = reinterpret_cast<double*>(Msh + (int64_t)B * 3 * nv);
    Mss = ysh + (int64_t)B * 3 * n;
    red = STREAM ? Mss + n : Mss;
    extra = reinterpret_cast<unsigned char*>(red + (int64_t)B * (STREAM ? R : 1) * kResWarps * 3);
    Ng = (const T*)Nptr;
    ldg = ld;
    if constexpr (!STREAM) {
      const T* N = (const T*)Nptr;
      const int64_t plane = n * ld;
      const int64_t tot = (int64_t)rows * 6 * nv;
      for (int64_t idx = tid; idx < tot; idx += kResThreads) {
        const int64_t v = idx % nv;
        const int c = (int)((idx / nv) % 6);
        const int r = (int)(idx / (6 * nv));
        const V x = __ldcs(reinterpret_cast<const V*>(N + c * plane + (r0 + r) * ld) + v);
        tens[((int64_t)r * 6 + c) * nv + v] = zero_from(x, v * W, n);
      }
#pragma unroll
      for (int q = 0; q < kColQ; ++q) msj[q] = tid + q * kResThreads < n ? e.Ms[tid + q * kResThreads] : 0.0;
    } else {
      for (int64_t j = tid; j < n; j += kResThreads) Mss[j] = e.Ms[j];
    }
    T* Mz = reinterpret_cast<T*>(Msh);
    for (int64_t idx = tid; idx < (int64_t)B * 3 * ldS; idx += kResThreads) Mz[idx] = T(0);
    epi = tid < rows * B;
    er = epi ? tid % rows : 0;
    eb = epi ? tid / rows : 0;
    i = r0 + er;
#pragma unroll
    for (int q = 0; q < 6; ++q) nb[q] = -1;
    cex = can = 0.0;
    ax[0] = ax[1] = ax[2] = ha[0] = ha[1] = ha[2] = 0.0;
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
    row = warp / wpr;  // (STREAM: the warp's slot within a round of kResWarps / wpr rows)
    const int seg = warp % wpr;
    const int64_t per = (nv + wpr - 1) / wpr;
    v0 = (int64_t)seg * per;
    v1 = min(nv, v0 + per);
    trow = tens + (int64_t)row * 6 * nv;
    __syncthreads();
  }

  // One right-hand side at the stage state yin (global, written by every CTA's epilogue threads: read from
  // L2, not L1).  Epilogue threads return mi = the state of their tile, k = dm/dt (Eq. 1) and |m x H_eff|.
  __device__ __forceinline__ void rhs(const double* yin, const EpiArgs& e, double mi[3], double k[3], double& torque) {
    {
      // Ms*m in the tensor's dtype, rounded once (Q19).  A thread owns the columns tid + 256 q: a
      // state's 3 x kColQ loads are in flight together (the stage costs one L2 round trip per state, not one
      // per element) and Ms of those columns stays in registers for the whole launch.
      T* Ms_ = reinterpret_cast<T*>(Msh);
      const int n32 = (int)n, ld32 = (int)ldS;
      for (int b = 0; b < B; ++b) {
        const double* src = yin + (int64_t)b * 3 * n;
        for (int q0 = 0; q0 == 0 || (STREAM && q0 * kResThreads < n32); q0 += kColQ) {  // (one pass unless STREAM and n > 1,280)
          double yv[3][kColQ];
#pragma unroll
          for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int q = 0; q < kColQ; ++q) {
              const int j = tid + (q0 + q) * kResThreads;
              yv[c][q] = j < n32 ? __ldcg(src + c * n32 + j) : 0.0;
            }
#pragma unroll
          for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int q = 0; q < kColQ; ++q) {
              const int j = tid + (q0 + q) * kResThreads;
              if (j < n32) {
                ysh[(b * 3 + c) * n32 + j] = yv[c][q];
                Ms_[(b * 3 + c) * ld32 + j] = (T)((STREAM ? Mss[j] : msj[q]) * yv[c][q]);
              }
            }
        }
      }
    }
    __syncthreads();
    if constexpr (STREAM) {
      // kResWarps / wpr of the CTA's rows at a time, wpr (1 or 2) warps per row; the row comes from L2 (read-only
      // for the kernel: non-coherent loads), columns >= n of its last vector read as zero.  fp32: a lane's partial
      // sum covers at most 4 * ceil(n / 128) <= 68 terms at the 100 MB limit (Q19 allows 128)
      const int nv32 = (int)nv, v0i = (int)v0, v1i = (int)v1;
      const int64_t plane = n * ldg;
      const int per_round = kResWarps / wpr;  // rows in flight: wpr warps stream one row, each its share of the columns
      const int64_t pv = plane / W;           // vectors per plane
      for (int r = row; r < rows; r += per_round) {
        const V* g = reinterpret_cast<const V*>(Ng + (r0 + r) * ldg);
        for (int b0 = 0; b0 < B; b0 += 4) {
          T acc[4][3];
#pragma unroll
          for (int bb = 0; bb < 4; ++bb) acc[bb][0] = acc[bb][1] = acc[bb][2] = T(0);
#pragma unroll kStreamUnroll
          for (int v = v0i + lane; v < v1i; v += 32) {
            V t[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) t[c] = __ldg(g + c * pv + v);
            if (v == nv32 - 1) {
#pragma unroll
              for (int c = 0; c < 6; ++c) t[c] = zero_from(t[c], (int64_t)v * W, n);
            }
#pragma unroll
            for (int bb = 0; bb < 4; ++bb)
              if (b0 + bb < B) {
                const V* Mb = Msh + (b0 + bb) * 3 * nv32;
                V m[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) m[c] = Mb[c * nv32 + v];
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
                double* o = red + (((int64_t)(b0 + bb) * R + r) * kResWarps + (warp % wpr)) * 3;
                o[0] = d[0];
                o[1] = d[1];
                o[2] = d[2];
              }
            }
        }
      }
    } else if (row < rows) {
      // up to four states per pass over the row: the tensor's shared-memory rows are read once per pass
      const int nv32 = (int)nv, v0i = (int)v0, v1i = (int)v1;
      for (int b0 = 0; b0 < B; b0 += 4) {
        T acc[4][3];
#pragma unroll
        for (int bb = 0; bb < 4; ++bb) acc[bb][0] = acc[bb][1] = acc[bb][2] = T(0);
        for (int v = v0i + lane; v < v1i; v += 32) {
          V t[6];
#pragma unroll
          for (int c = 0; c < 6; ++c) t[c] = trow[c * nv32 + v];
#pragma unroll
          for (int bb = 0; bb < 4; ++bb)
            if (b0 + bb < B) {
              const V* Mb = Msh + (b0 + bb) * 3 * nv32;
              V m[3];
#pragma unroll
              for (int c = 0; c < 3; ++c) m[c] = Mb[c * nv32 + v];
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
    if (!epi) return;
    // H_d = -N.M, the warps' column parts added in warp order
    double H[3] = {0.0, 0.0, 0.0};
    for (int w = 0; w < wpr; ++w) {
      const double* o = red + (STREAM ? ((int64_t)eb * R + er) * kResWarps + w : (int64_t)eb * kResWarps + er * wpr + w) * 3;
#pragma unroll
      for (int c = 0; c < 3; ++c) H[c] += o[c];
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) H[c] = -H[c];
    const double* y = ysh + (int64_t)eb * 3 * n;
    mi[0] = y[i]; mi[1] = y[n + i]; mi[2] = y[2 * n + i];
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
    double mxH[3], mxmxH[3];
    cross3(mi, H, mxH);
    cross3(mi, mxH, mxmxH);
#pragma unroll
    for (int c = 0; c < 3; ++c) k[c] = -e.gamma * mxH[c] - e.alpha * mxmxH[c];
    torque = sqrt(mxH[0] * mxH[0] + mxH[1] * mxH[1] + mxH[2] * mxH[2]);
  }

  __device__ __forceinline__ void store(double* yout, const double yo[3]) const {
    double* o = yout + (int64_t)eb * 3 * n + i;
#pragma unroll
    for (int c = 0; c < 3; ++c) o[c * n] = yo[c];
  }
};

// a zero-length m_i stays zero (Q10c)
__device__ __forceinline__ void renormalise(double yo[3]) {
  const double r = sqrt(yo[0] * yo[0] + yo[1] * yo[1] + yo[2] * yo[2]);
  if (r > 0.0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) yo[c] /= r;
  }
}

template <typename T, bool STREAM>
__global__ void __launch_bounds__(kResThreads, 1) rk4_resident_kernel(const __grid_constant__ ResArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Resident<T, STREAM> rs;
  rs.init(smem_raw, a.N, a.n, a.ld, a.ldS, a.R, a.wpr, a.batch, a.prob);
  const EpiArgs& e = a.prob;
  double base[3] = {0.0, 0.0, 0.0}, ks[3][3];
#pragma unroll
  for (int q = 0; q < 3; ++q) ks[q][0] = ks[q][1] = ks[q][2] = 0.0;
  unsigned int bar_target = 0;

  for (int64_t step = 0; step < a.count; ++step) {
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      double mi[3], k[3], tq;
      rs.rhs(a.y_in[s], e, mi, k, tq);
      if (rs.epi) {
        if (s == 0) {
          if (a.tq) atomic_max_nonneg(a.tq + step, tq);
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
          if (a.renorm) renormalise(yo);
        }
        rs.store(a.y_to[s], yo);
      }
      bar_target += gridDim.x;
      grid_barrier(a.bar, bar_target);  // every CTA's rows of the next stage state are visible to all
    }
  }
}

// ---- A9: Dormand-Prince 5(4), FSAL, the controller of dp_control.cuh inside the kernel -------------------
// One launch runs up to `attempts` attempted steps.  Thread 0 of every CTA runs the controller on the CTA's own
// copy of the state (same inputs everywhere: the error / torque maxima are read after a grid barrier), so no
// decision has to be broadcast.  An attempt: y2 = m + h a21 k1 (k1 = the previous step's k7 or the caller's
// f(m)); five right-hand sides with their stage combines; k7 = f(y7) with the error estimate and the torque
// of y7 max-reduced into the attempt's two global words (double-buffered by attempt parity; zeroed one attempt
// ahead); accept / reject.  m, k1..k7 of a row stay in its epilogue thread's registers; m is written to global
// memory on every accepted step (samples, result), k1 at the end of the launch (the next launch's FSAL slope).
struct DpResArgs {
  const void* N;
  int64_t n, ld;
  int R, wpr, batch, renorm;
  int64_t ldS;
  int attempts;
  unsigned int* bar;          // grid barrier counter (zero at launch)
  unsigned long long* words;  // [2][2]: error / torque bits per attempt parity (zero at launch)
  DpState* S;                 // controller state (global)
  double* m;                  // [B][3][n] state, in place
  double* k1;                 // [B][3][n] FSAL slope in / out
  double* ybuf[2];            // two stage states
  double* samples;            // [cap][1 + 3 B] or NULL
  int64_t stride;
  const double* vol;
  EpiArgs prob;
};

__device__ const double kDpA[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5, 0, 0, 0, 0, 0},
    {3.0 / 40, 9.0 / 40, 0, 0, 0, 0},
    {44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0},
    {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0},
    {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0},
    {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}};
__device__ const double kDpE[7] = {35.0 / 384 - 5179.0 / 57600,       0.0,
                                   500.0 / 1113 - 7571.0 / 16695,     125.0 / 192 - 393.0 / 640,
                                   -2187.0 / 6784 + 92097.0 / 339200, 11.0 / 84 - 187.0 / 2100,
                                   -1.0 / 40};

template <typename T, bool STREAM>
__global__ void __launch_bounds__(kResThreads, 1) dp45_resident_kernel(const __grid_constant__ DpResArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ DpState S;
  Resident<T, STREAM> rs;
  rs.init(smem_raw, a.N, a.n, a.ld, a.ldS, a.R, a.wpr, a.batch, a.prob);
  const EpiArgs& e = a.prob;
  const int64_t n = a.n;
  double* mean_s = reinterpret_cast<double*>(rs.extra);  // [2][256]: the sample's tree
  if (threadIdx.x == 0) S = *a.S;
  double base[3] = {0.0, 0.0, 0.0}, cand[3], k[7][3];
#pragma unroll
  for (int j = 0; j < 7; ++j) k[j][0] = k[j][1] = k[j][2] = 0.0;
  if (rs.epi) {
    const int64_t o = (int64_t)rs.eb * 3 * n + rs.i;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      base[c] = a.m[o + c * n];
      k[0][c] = a.k1[o + c * n];
    }
  }
  unsigned int bar_target = 0;
  int parity = 0;
  __syncthreads();

  for (int att = 0; att < a.attempts; ++att) {
    __syncthreads();  // everybody is done reading the previous attempt's state
    if (threadIdx.x == 0) dp_begin(&S);
    __syncthreads();
    const int active = S.active;
    if (active) {
      const double h = S.h;
      unsigned long long* wd = a.words + 2 * parity;
      // y2 = m + h a21 k1
      if (rs.epi) {
        double yo[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          double s = 0.0;
          s += kDpA[1][0] * k[0][c];
          yo[c] = base[c] + h * s;
        }
        rs.store(a.ybuf[0], yo);
      }
      bar_target += gridDim.x;
      grid_barrier(a.bar, bar_target);
      // the other parity's words are free now (every CTA has taken the previous attempt's decision)
      if (blockIdx.x == 0 && threadIdx.x == 0) {
        unsigned long long* wo = a.words + 2 * (parity ^ 1);
        wo[0] = 0ull;
        wo[1] = 0ull;
      }
#pragma unroll
      for (int sg = 1; sg <= 5; ++sg) {
        double mi[3], tq;
        rs.rhs(a.ybuf[(sg - 1) & 1], e, mi, k[sg], tq);
        if (rs.epi) {
          double yo[3];
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            double s = 0.0;
#pragma unroll
            for (int j = 0; j <= sg; ++j) s += kDpA[sg + 1][j] * k[j][c];
            yo[c] = base[c] + h * s;
          }
          rs.store(a.ybuf[sg & 1], yo);
        }
        bar_target += gridDim.x;
        grid_barrier(a.bar, bar_target);
      }
      // k7 = f(y7): error estimate against (m, y7), torque of y7, (renormalised) candidate
      {
        double mi[3], tq;
        rs.rhs(a.ybuf[1], e, mi, k[6], tq);
        if (rs.epi) {
          double err = 0.0;
#pragma unroll
          for (int c = 0; c < 3; ++c) {
            double s = 0.0;
#pragma unroll
            for (int j = 0; j < 7; ++j) s += kDpE[j] * k[j][c];
            s *= h;
            const double sc = S.atol + S.rtol * fmax(fabs(base[c]), fabs(mi[c]));
            const double q = fabs(s) / sc;
            err = (q > err || q != q) ? q : err;  // a NaN must reach the controller (Q11b)
            cand[c] = mi[c];
          }
          atomic_max_nonneg(wd + 0, err);
          atomic_max_nonneg(wd + 1, tq);
          if (a.renorm) renormalise(cand);
        }
      }
      bar_target += gridDim.x;
      grid_barrier(a.bar, bar_target);
      if (threadIdx.x == 0) {
        S.err_bits = __ldcg(wd + 0);
        S.tq_bits = __ldcg(wd + 1);
        dp_decide(&S);
      }
      __syncthreads();
      if (S.accept && rs.epi) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          base[c] = cand[c];
          k[0][c] = k[6][c];
        }
        rs.store(a.m, base);
      }
      parity ^= 1;
    }
    if (S.sample_flag) {
      // <m> (A10) of the state just committed (or landed on): CTA 0, after everybody's rows are visible
      bar_target += gridDim.x;
      grid_barrier(a.bar, bar_target);
      if (blockIdx.x == 0) {
        for (int bc = 0; bc < 3 * a.batch; ++bc) {
          const double* v = a.m + (int64_t)bc * n;
          double s = 0.0, w = 0.0;
          for (int64_t j = threadIdx.x; j < n; j += kResThreads) {
            const double wj = a.vol ? a.vol[j] : 1.0;
            s += wj * __ldcg(v + j);
            w += wj;
          }
          mean_s[threadIdx.x] = s;
          mean_s[kResThreads + threadIdx.x] = w;
          __syncthreads();
          for (int off = kResThreads / 2; off > 0; off >>= 1) {
            if ((int)threadIdx.x < off) {
              mean_s[threadIdx.x] += mean_s[threadIdx.x + off];
              mean_s[kResThreads + threadIdx.x] += mean_s[kResThreads + threadIdx.x + off];
            }
            __syncthreads();
          }
          if (threadIdx.x == 0) {
            double* out = a.samples + S.sample_row * a.stride;
            out[1 + bc] = mean_s[0] / mean_s[kResThreads];
            if (bc == 0) out[0] = S.sample_t;
          }
          __syncthreads();
        }
      }
    }
    if (S.status != MT_DP_RUN) break;  // the run has ended (every CTA holds the same state)
  }
  // the next launch's FSAL slope; the controller state
  if (rs.epi) rs.store(a.k1, k[0]);
  if (blockIdx.x == 0 && threadIdx.x == 0) *a.S = S;
}

size_t resident_smem(int dtype, int64_t n, int R, int batch, size_t extra, bool stream, int64_t* ldS_out) {
  const int64_t W = dtype == MT_F32 ? 4 : 2;
  const size_t sz = dtype == MT_F32 ? 4 : 8;
  const int64_t ldS = (n + W - 1) / W * W;
  if (ldS_out) *ldS_out = ldS;
  if (stream)  // Msh | ysh | Mss | red[B][R][8][3]
    return (size_t)batch * 3 * ldS * sz + ((size_t)batch * 3 + 1) * n * sizeof(double) +
           (size_t)batch * R * kResWarps * 3 * sizeof(double) + extra;
  return ((size_t)R * 6 + (size_t)batch * 3) * ldS * sz + (size_t)batch * 3 * n * sizeof(double) +
         (size_t)batch * kResWarps * 3 * sizeof(double) + extra;
}
// Rows read from L2: one warp per row keeps the longest streams in flight; two warps per row when that takes fewer
// rounds of eight warps (9..12 rows: 3 half-rounds instead of 2 rounds).  Four and eight warps per row measured slower.
inline int stream_wpr(int R) {
  const int rounds1 = (R + kResWarps - 1) / kResWarps, rounds2 = (R + kResWarps / 2 - 1) / (kResWarps / 2);
  return rounds2 < 2 * rounds1 ? 2 : 1;
}
constexpr int kStreamMaxRows = 32;                      // rows per CTA when the tensor is read from L2 at every stage
#ifndef MT_STREAM_MAX_MB
#define MT_STREAM_MAX_MB 100
#endif
constexpr size_t kStreamMaxBytes = (size_t)MT_STREAM_MAX_MB << 20;   // ... which pays while the tensor stays in the 126 MB L2
constexpr size_t kDpExtra = 2 * kResThreads * sizeof(double);  // the sample's reduction tree
constexpr size_t kDpStatic = 1024;                             // the CTA's copy of the controller state

static_assert(sizeof(ResArgs) <= 4000 && sizeof(DpResArgs) <= 4000, "kernel parameter space");
static_assert(sizeof(DpState) <= kDpStatic, "static shared memory of the DP45 kernel");

}  // namespace

// How can the integrators keep the dense n x n tensor of this dtype on the chip?  MT_RES_SMEM: resident in shared
// memory across the GPU (one CTA per SM, ceil(n / SMs) <= 8 rows each) together with `batch` stage states;
// MT_RES_L2: too large for that but at most 100 MB, read from L2 at every stage by a persistent kernel of the same
// structure (<= 32 rows per CTA); MT_RES_NONE otherwise.  method: MT_RK4 or MT_DP45.
int mt_resident_fits(mt_ctx* ctx, int dtype, int64_t n, int64_t ld, int batch, int method) {
  if (n <= 0 || batch < 1 || batch > MT_MAX_BATCH) return MT_RES_NONE;
  int dev_smem = 0, coop = 0;
  if (cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device) != cudaSuccess ||
      cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device) != cudaSuccess || !coop) {
    cudaGetLastError();
    return MT_RES_NONE;
  }
  const int R = (int)((n + ctx->num_sms - 1) / ctx->num_sms);
  const size_t extra = method == MT_DP45 ? kDpExtra + kDpStatic : 0;
  if (R * batch > kResThreads) return MT_RES_NONE;
  if (n <= kColQ * kResThreads && R <= kResWarps &&
      resident_smem(dtype, n, R, batch, extra, false, nullptr) <= (size_t)dev_smem)
    return MT_RES_SMEM;
  const size_t bytes = 6 * (size_t)n * (size_t)ld * (dtype == MT_F32 ? 4 : 8);
  if (R <= kStreamMaxRows && bytes <= kStreamMaxBytes &&
      resident_smem(dtype, n, R, batch, extra, true, nullptr) <= (size_t)dev_smem)
    return MT_RES_L2;
  return MT_RES_NONE;
}

static int launch_cooperative(mt_ctx* ctx, const void* fn, unsigned grid, size_t smem, void* arg) {
  // the attribute is per device, not per process: set it on every launch (a few microseconds per chunk)
  MT_CUDA_OK(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  MT_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, kResThreads, smem));
  if ((int64_t)per_sm * ctx->num_sms < (int64_t)grid)
    return mt_fail(ctx, MT_ERR_CUDA, "resident integrator: %u CTAs cannot be co-resident on this device", grid);
  void* args[] = {arg};
  MT_CUDA_OK(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(kResThreads), args, smem, ctx->stream));
  ctx->launches++;
  return MT_OK;
}

// `count` RK4 steps of m (in place); ya, yb: two scratch states [B][3][n]; `prob`: fill_problem's constants.
int mt_launch_rk4_resident(mt_ctx* ctx, int mode, const void* N, int dtype, int64_t n, int64_t ld, const EpiArgs& prob,
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
  const bool stream = mode == MT_RES_L2;
  if (stream) a.wpr = stream_wpr(a.R);
  const size_t smem = resident_smem(dtype, n, a.R, a.batch, 0, stream, &a.ldS);
  if (a.ldS > ld) return mt_fail(ctx, MT_ERR_INVALID_ARG, "resident RK4: ld must cover whole 16-byte vectors");
  const void* fn = dtype == MT_F32
                       ? (stream ? (const void*)rk4_resident_kernel<float, true> : (const void*)rk4_resident_kernel<float, false>)
                       : (stream ? (const void*)rk4_resident_kernel<double, true> : (const void*)rk4_resident_kernel<double, false>);
  MT_CUDA_OK(ctx, cudaMemsetAsync(bar, 0, sizeof(unsigned int), ctx->stream));
  return launch_cooperative(ctx, fn, (unsigned)((n + a.R - 1) / a.R), smem, &a);
}

// Up to `attempts` attempted DP45 steps of m (in place) under the controller state S (device); k1 holds
// f(m) on entry and the FSAL slope of the state on exit; words: 4 device words, bar: 1 (zeroed here).
int mt_launch_dp45_resident(mt_ctx* ctx, int mode, const void* N, int dtype, int64_t n, int64_t ld, const EpiArgs& prob,
                            DpState* S, double* m, double* k1, double* ya, double* yb, int renorm,
                            double* samples, int64_t stride, const double* vol, unsigned long long* words,
                            unsigned int* bar, int attempts) {
  if (attempts <= 0) return MT_OK;
  DpResArgs a;
  memset(&a, 0, sizeof(a));
  a.N = N;
  a.n = n;
  a.ld = ld;
  a.R = (int)((n + ctx->num_sms - 1) / ctx->num_sms);
  a.wpr = 1;
  while (a.wpr * 2 * a.R <= kResWarps) a.wpr *= 2;
  a.batch = prob.batch;
  a.renorm = renorm;
  a.attempts = attempts;
  a.bar = bar;
  a.words = words;
  a.S = S;
  a.m = m;
  a.k1 = k1;
  a.ybuf[0] = ya;
  a.ybuf[1] = yb;
  a.samples = samples;
  a.stride = stride;
  a.vol = vol;
  a.prob = prob;
  const bool stream = mode == MT_RES_L2;
  if (stream) a.wpr = stream_wpr(a.R);
  const size_t smem = resident_smem(dtype, n, a.R, a.batch, kDpExtra, stream, &a.ldS);
  if (a.ldS > ld) return mt_fail(ctx, MT_ERR_INVALID_ARG, "resident DP45: ld must cover whole 16-byte vectors");
  const void* fn = dtype == MT_F32
                       ? (stream ? (const void*)dp45_resident_kernel<float, true> : (const void*)dp45_resident_kernel<float, false>)
                       : (stream ? (const void*)dp45_resident_kernel<double, true> : (const void*)dp45_resident_kernel<double, false>);
  MT_CUDA_OK(ctx, cudaMemsetAsync(bar, 0, sizeof(unsigned int), ctx->stream));
  MT_CUDA_OK(ctx, cudaMemsetAsync(words, 0, 4 * sizeof(unsigned long long), ctx->stream));
  return launch_cooperative(ctx, fn, (unsigned)((n + a.R - 1) / a.R), smem, &a);
}
