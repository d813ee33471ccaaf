// noalloc.cu — mt_demag_field_noalloc (include/mt.h): H_d = -N.(Ms m) for one state with every byte of
// scratch in a file-scope __device__ array, for callers that cannot call cudaMalloc (graph capture, tight
// serving loops, harnesses that forbid it).  A variant of the register-streaming field kernel of demag.cu
// (one warp per target row and column split, 128-bit non-allocating loads of the six component rows,
// fp32 tensors in short fp32 runs flushed into fp64 — DESIGN.md Q19 — and a fixed xor-butterfly), always
// followed by the fixed-order sum over the column splits.  Self-contained on purpose: no mt_ctx, no
// shared helper with the allocating path, no cudaMalloc / cudaFree / allocating library routine.
//
// Scratch layout (MT_NOALLOC_SCRATCH_BYTES = 4.5 MiB per GPU that loads the library):
//   [0, 1.5 MiB)        staged vector M[c][j] = T(Ms[j] m[c][j]), [3][npad] in the tensor's dtype,
//                       npad = n rounded up to 128 <= 65,536; the staging kernel zeroes j in [n, npad)
//   [1.5 MiB, 4.5 MiB)  partial row sums, double [nsplit][3][n_rows], nsplit * n_rows <= 131,072
// Every call rewrites each word it later reads, so stale contents of an earlier call are never seen; calls
// that overlap on the GPU race on the array (mt.h).
#include <stdarg.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include <cuda_runtime.h>

#include "mt.h"

namespace {

constexpr int64_t kStageBytes = 3LL * MT_NOALLOC_MAX_N * (int64_t)sizeof(double);  // 1.5 MiB
constexpr int64_t kPartialWords = (MT_NOALLOC_SCRATCH_BYTES - kStageBytes) / (int64_t)sizeof(double);
constexpr int64_t kMaxSplitRows = kPartialWords / 3;  // nsplit * n_rows
constexpr int kWarps = 8;
constexpr int kFlush = 8;   // fp32: vector iterations per fp32 run (as demag.cu)
constexpr int kMaxDevices = 64;
static_assert(kStageBytes % 256 == 0 && kPartialWords > 0, "scratch layout");
static_assert(kMaxSplitRows >= MT_NOALLOC_MAX_N, "one split of the largest band must fit");

// The scratch itself.  In HOST code this name is only a stand-in for the symbol: the device address comes
// from cudaGetSymbolAddress (scratch_of below), never from &g_noalloc_scratch.
static __device__ __align__(256) unsigned char g_noalloc_scratch[MT_NOALLOC_SCRATCH_BYTES];

template <typename T> struct VecOf;
template <> struct VecOf<float> { typedef float4 type; static constexpr int W = 4; };
template <> struct VecOf<double> { typedef double2 type; static constexpr int W = 2; };

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

__device__ __forceinline__ void fma3(float acc[3], float xx, float xy, float xz, float yy, float yz, float zz,
                                     float mx, float my, float mz) {
  acc[0] = fmaf(xx, mx, fmaf(xy, my, fmaf(xz, mz, acc[0])));
  acc[1] = fmaf(xy, mx, fmaf(yy, my, fmaf(yz, mz, acc[1])));
  acc[2] = fmaf(xz, mx, fmaf(yz, my, fmaf(zz, mz, acc[2])));
}
__device__ __forceinline__ void fma3(double acc[3], double xx, double xy, double xz, double yy, double yz,
                                     double zz, double mx, double my, double mz) {
  acc[0] = fma(xx, mx, fma(xy, my, fma(xz, mz, acc[0])));
  acc[1] = fma(xy, mx, fma(yy, my, fma(yz, mz, acc[1])));
  acc[2] = fma(xz, mx, fma(yz, my, fma(zz, mz, acc[2])));
}
__device__ __forceinline__ void vec_fma(float acc[3], const float4 v[6], const float4 m[3]) {
  fma3(acc, v[0].x, v[1].x, v[2].x, v[3].x, v[4].x, v[5].x, m[0].x, m[1].x, m[2].x);
  fma3(acc, v[0].y, v[1].y, v[2].y, v[3].y, v[4].y, v[5].y, m[0].y, m[1].y, m[2].y);
  fma3(acc, v[0].z, v[1].z, v[2].z, v[3].z, v[4].z, v[5].z, m[0].z, m[1].z, m[2].z);
  fma3(acc, v[0].w, v[1].w, v[2].w, v[3].w, v[4].w, v[5].w, m[0].w, m[1].w, m[2].w);
}
__device__ __forceinline__ void vec_fma(double acc[3], const double2 v[6], const double2 m[3]) {
  fma3(acc, v[0].x, v[1].x, v[2].x, v[3].x, v[4].x, v[5].x, m[0].x, m[1].x, m[2].x);
  fma3(acc, v[0].y, v[1].y, v[2].y, v[3].y, v[4].y, v[5].y, m[0].y, m[1].y, m[2].y);
}

// M[c][j] = T(Ms[j] * m[c][j]) for j < n, 0 for n <= j < npad (the padding must start at zero every call:
// the array keeps whatever the previous call staged there)
template <typename T>
__global__ void __launch_bounds__(256) na_stage_kernel(const double* __restrict__ Ms, const double* __restrict__ m,
                                                       int64_t n, int64_t npad, T* __restrict__ M) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int c = blockIdx.y;
  if (j >= npad) return;
  M[c * npad + j] = j < n ? (T)(Ms[j] * m[c * n + j]) : T(0);
}

template <typename T>
struct FieldArgs {
  const T* N;
  int64_t n, n_rows, ld, plane;
  const T* M;         // scratch: [3][npad]
  int64_t npad;
  int64_t vec_per_split;
  int nsplit;
  double* partial;    // scratch: [nsplit][3][n_rows]
};

template <typename T>
__global__ void __launch_bounds__(kWarps * 32) na_field_kernel(FieldArgs<T> a) {
  typedef typename VecOf<T>::type V;
  constexpr int W = VecOf<T>::W;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * kWarps + warp;
  if (row >= a.n_rows) return;
  const int split = blockIdx.y;
  const int64_t nvec = a.n / W;
  const int64_t v0 = (int64_t)split * a.vec_per_split;
  const int64_t v1 = min(nvec, v0 + a.vec_per_split);
  const V* p[6];
#pragma unroll
  for (int c = 0; c < 6; ++c) p[c] = reinterpret_cast<const V*>(a.N + c * a.plane + row * a.ld);
  const V* mp = reinterpret_cast<const V*>(a.M);
  const int64_t mstride = a.npad / W;

  double acc[3] = {0.0, 0.0, 0.0};
  for (int64_t vb = v0 + lane; vb < v1; vb += 32 * kFlush) {
    T run[3] = {T(0), T(0), T(0)};
#pragma unroll 2
    for (int it = 0; it < kFlush; ++it) {
      const int64_t v = vb + (int64_t)it * 32;
      if (v < v1) {
        V t[6], mv[3];
#pragma unroll
        for (int c = 0; c < 6; ++c) t[c] = ld_stream(p[c] + v);
#pragma unroll
        for (int c = 0; c < 3; ++c) mv[c] = mp[c * mstride + v];  // plain loads: written by the launch before
        vec_fma(run, t, mv);
      }
    }
    acc[0] += (double)run[0];
    acc[1] += (double)run[1];
    acc[2] += (double)run[2];
  }
  // scalar tail (n not a multiple of the vector width): last split, one lane per leftover column
  if (split == a.nsplit - 1) {
    const int64_t j = nvec * W + lane;
    if (j < a.n) {
      T t[6], mv[3];
#pragma unroll
      for (int c = 0; c < 6; ++c) t[c] = a.N[c * a.plane + row * a.ld + j];
#pragma unroll
      for (int c = 0; c < 3; ++c) mv[c] = a.M[c * a.npad + j];
      T run[3] = {T(0), T(0), T(0)};
      fma3(run, t[0], t[1], t[2], t[3], t[4], t[5], mv[0], mv[1], mv[2]);
      acc[0] += (double)run[0];
      acc[1] += (double)run[1];
      acc[2] += (double)run[2];
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], off);
  if (lane == 0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) a.partial[((int64_t)split * 3 + c) * a.n_rows + row] = acc[c];
  }
}

// Hd[c][row] = - sum over the splits, in split order
__global__ void __launch_bounds__(256) na_reduce_kernel(const double* __restrict__ partial, int nsplit,
                                                        int64_t n_rows, double* __restrict__ Hd) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 3 * n_rows) return;
  double s = 0.0;
  for (int sp = 0; sp < nsplit; ++sp) s += partial[(int64_t)sp * 3 * n_rows + idx];
  Hd[idx] = -s;
}

// ---- host side ----------------------------------------------------------------------------------------
struct DeviceSlot {
  bool ready;
  unsigned char* scratch;  // DEVICE address of g_noalloc_scratch on this device
  int num_sms;
};
std::mutex g_mu;
DeviceSlot g_slot[kMaxDevices];

int fail(char* err, int64_t cap, int code, const char* fmt, ...) {
  if (err && cap > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err, (size_t)cap, fmt, ap);
    va_end(ap);
  }
  return code;
}

// restores the calling thread's current device on every exit path
struct DeviceGuard {
  int prev;
  bool switched;
  DeviceGuard() : prev(-1), switched(false) {}
  cudaError_t enter(int device) {
    cudaError_t rc = cudaGetDevice(&prev);
    if (rc != cudaSuccess) return rc;
    if (prev == device) return cudaSuccess;
    rc = cudaSetDevice(device);
    switched = rc == cudaSuccess;
    return rc;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

// Once per device, with that device current: the DEVICE address of the scratch array.  Each device that
// loads the module has its own copy of a __device__ variable, hence its own address.
int scratch_of(int device, DeviceSlot* out, char* err, int64_t cap) {
  std::lock_guard<std::mutex> lock(g_mu);
  DeviceSlot& s = g_slot[device];
  if (!s.ready) {
    unsigned char* ptr = nullptr;
    cudaError_t rc = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);
    if (rc != cudaSuccess || !ptr)
      return fail(err, cap, MT_ERR_CUDA, "cudaGetSymbolAddress(scratch) on device %d: %s", device,
                  cudaGetErrorString(rc));
    size_t bytes = 0;
    rc = cudaGetSymbolSize(&bytes, g_noalloc_scratch);
    if (rc != cudaSuccess || bytes != (size_t)MT_NOALLOC_SCRATCH_BYTES)
      return fail(err, cap, MT_ERR_CUDA, "scratch symbol size %zu on device %d: %s", bytes, device,
                  cudaGetErrorString(rc));
    int sms = 0;
    rc = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (rc != cudaSuccess || sms <= 0)
      return fail(err, cap, MT_ERR_CUDA, "multiprocessor count of device %d: %s", device, cudaGetErrorString(rc));
    s.scratch = ptr;
    s.num_sms = sms;
    s.ready = true;
  }
  *out = s;
  return MT_OK;
}

template <typename T>
int launch(const DeviceSlot& slot, cudaStream_t stream, const void* N, int64_t n, int64_t n_rows, int64_t ld,
           const double* Ms, const double* m, double* Hd, char* err, int64_t cap) {
  constexpr int W = VecOf<T>::W;
  const int64_t npad = (n + 127) / 128 * 128;
  T* M = reinterpret_cast<T*>(slot.scratch);
  double* partial = reinterpret_cast<double*>(slot.scratch + kStageBytes);

  FieldArgs<T> a;
  a.N = (const T*)N;
  a.n = n;
  a.n_rows = n_rows;
  a.ld = ld;
  a.plane = n_rows * ld;
  a.M = M;
  a.npad = npad;
  // split the columns when the rows alone cannot fill the machine twice over (as demag.cu), within what
  // the partial-sum region holds
  const int64_t ctas = (n_rows + kWarps - 1) / kWarps;
  const int64_t want = 2LL * slot.num_sms;
  const int64_t nvec = n / W;
  int64_t nsplit = 1;
  if (ctas < want) {
    nsplit = (want + ctas - 1) / ctas;
    const int64_t max_split = (nvec + 255) / 256;  // keep >= 256 vectors per split
    if (nsplit > max_split) nsplit = max_split > 0 ? max_split : 1;
    if (nsplit > 64) nsplit = 64;
    if (nsplit > kMaxSplitRows / n_rows) nsplit = kMaxSplitRows / n_rows;
  }
  int64_t vps = (nvec + nsplit - 1) / nsplit;
  vps = (vps + 31) / 32 * 32;
  if (vps == 0) vps = 32;
  nsplit = (nvec + vps - 1) / vps;
  if (nsplit < 1) nsplit = 1;
  if (nsplit * n_rows > kMaxSplitRows)  // cannot happen for sizes within the limit; never write past the array
    return fail(err, cap, MT_ERR_INVALID_ARG, "partial sums (%lld splits x %lld rows) exceed the static scratch",
                (long long)nsplit, (long long)n_rows);
  a.vec_per_split = vps;
  a.nsplit = (int)nsplit;
  a.partial = partial;

  na_stage_kernel<T><<<dim3((unsigned)((npad + 255) / 256), 3), 256, 0, stream>>>(Ms, m, n, npad, M);
  cudaError_t rc = cudaGetLastError();
  if (rc == cudaSuccess) {
    na_field_kernel<T><<<dim3((unsigned)ctas, (unsigned)nsplit), kWarps * 32, 0, stream>>>(a);
    rc = cudaGetLastError();
  }
  if (rc == cudaSuccess) {
    na_reduce_kernel<<<(unsigned)((3 * n_rows + 255) / 256), 256, 0, stream>>>(partial, (int)nsplit, n_rows, Hd);
    rc = cudaGetLastError();
  }
  if (rc != cudaSuccess) return fail(err, cap, MT_ERR_CUDA, "kernel launch: %s", cudaGetErrorString(rc));
  return MT_OK;
}

}  // namespace

extern "C" int mt_demag_field_noalloc(int device, void* cuda_stream, const void* N, int dtype, int64_t n,
                                      int64_t n_rows, int64_t ld, const double* Ms, const double* m, double* Hd,
                                      char* err, int64_t err_cap) {
  if (err && err_cap > 0) err[0] = '\0';
  if (dtype != MT_F32 && dtype != MT_F64) return fail(err, err_cap, MT_ERR_INVALID_ARG, "unknown dtype %d", dtype);
  if (n <= 0 || n_rows <= 0) return fail(err, err_cap, MT_ERR_INVALID_ARG, "n and n_rows must be positive");
  if (n > MT_NOALLOC_MAX_N || n_rows > MT_NOALLOC_MAX_N)
    return fail(err, err_cap, MT_ERR_INVALID_ARG,
                "n = %lld, n_rows = %lld: mt_demag_field_noalloc holds its scratch in a static array sized for at "
                "most MT_NOALLOC_MAX_N = %d tiles and rows (use mt_demag_field beyond that)",
                (long long)n, (long long)n_rows, MT_NOALLOC_MAX_N);
  if (ld < n) return fail(err, err_cap, MT_ERR_INVALID_ARG, "ld (%lld) < n (%lld)", (long long)ld, (long long)n);
  const int64_t vec = dtype == MT_F32 ? 4 : 2;
  if (ld % vec) return fail(err, err_cap, MT_ERR_INVALID_ARG, "ld must be a multiple of %lld elements", (long long)vec);
  if (!N || ((uintptr_t)N & 15))
    return fail(err, err_cap, MT_ERR_INVALID_ARG, "tensor pointer null or not 16-byte aligned");
  if (!Ms || !m || !Hd || (((uintptr_t)Ms | (uintptr_t)m | (uintptr_t)Hd) & 7))
    return fail(err, err_cap, MT_ERR_INVALID_ARG, "Ms, m and Hd must be non-NULL and 8-byte aligned");
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count || device >= kMaxDevices)
    return fail(err, err_cap, MT_ERR_INVALID_ARG, "device %d out of range (%d visible)", device, count);
  DeviceGuard guard;
  cudaError_t rc = guard.enter(device);
  if (rc != cudaSuccess) return fail(err, err_cap, MT_ERR_CUDA, "cudaSetDevice(%d): %s", device, cudaGetErrorString(rc));
  DeviceSlot slot;
  int st = scratch_of(device, &slot, err, err_cap);
  if (st) return st;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  if (dtype == MT_F32) return launch<float>(slot, stream, N, n, n_rows, ld, Ms, m, Hd, err, err_cap);
  return launch<double>(slot, stream, N, n, n_rows, ld, Ms, m, Hd, err, err_cap);
}
