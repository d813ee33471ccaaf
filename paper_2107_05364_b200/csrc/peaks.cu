// peaks.cu — microbenchmarks of the roofline denominators (mt_measure_peak).
//
// north_star asks for "assembly tile-pairs/s against FP64/FP32 pipe peak" and "GEMV achieved HBM
// GB/s against B200 peak".  The HBM denominator of the headline line is the driver's measured copy
// bandwidth (MEASURED_PEAKS.json); the kernels here measure, on the device the benchmark runs on
// and in the same process, what the arithmetic pipes and a pure READ stream sustain, so that the
// assembly fraction and the read-only fraction are quoted against measured ceilings instead of
// figures derived from unit counts.  None of this is on the product's compute path.
#include "mt_internal.cuh"

namespace {

constexpr int kChains = 8;     // independent dependency chains per thread
constexpr int kUnroll = 4;     // FMAs per chain per loop iteration
constexpr int kAluThreads = 256;
constexpr int kAluBlocksPerSm = 8;  // 2,048 threads per SM: every scheduler has 16 warps to pick from

template <int KIND>
__global__ void __launch_bounds__(kAluThreads) alu_peak_kernel(int iters, double* sink, double seed) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x;
  if constexpr (KIND == MT_PEAK_DFMA) {
    double a[kChains];
    const double x = 1.0 + 1e-9 * seed, y = 1e-9 * (double)(tid & 7);
#pragma unroll
    for (int j = 0; j < kChains; ++j) a[j] = seed + j;
    for (int it = 0; it < iters; ++it)
#pragma unroll
      for (int u = 0; u < kUnroll; ++u)
#pragma unroll
        for (int j = 0; j < kChains; ++j) a[j] = fma(a[j], x, y);
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < kChains; ++j) s += a[j];
    if (s == 12345.678) sink[tid] = s;  // never true: keeps the chains live
  } else if constexpr (KIND == MT_PEAK_FFMA) {
    float a[kChains];
    const float x = 1.0f + 1e-6f * (float)seed, y = 1e-6f * (float)(tid & 7);
#pragma unroll
    for (int j = 0; j < kChains; ++j) a[j] = (float)seed + j;
    for (int it = 0; it < iters; ++it)
#pragma unroll
      for (int u = 0; u < kUnroll; ++u)
#pragma unroll
        for (int j = 0; j < kChains; ++j) a[j] = fmaf(a[j], x, y);
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < kChains; ++j) s += a[j];
    if (s == 12345.678f) sink[tid] = s;
  } else if constexpr (KIND == MT_PEAK_FFMA2) {
    unsigned long long a[kChains];
    unsigned long long x, y;
    {
      const float xf = 1.0f + 1e-6f * (float)seed, yf = 1e-6f * (float)(tid & 7);
      asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "f"(xf), "f"(xf));
      asm("mov.b64 %0, {%1, %2};" : "=l"(y) : "f"(yf), "f"(yf));
    }
#pragma unroll
    for (int j = 0; j < kChains; ++j) {
      const float v = (float)seed + j;
      asm("mov.b64 %0, {%1, %2};" : "=l"(a[j]) : "f"(v), "f"(v));
    }
    for (int it = 0; it < iters; ++it)
#pragma unroll
      for (int u = 0; u < kUnroll; ++u)
#pragma unroll
        for (int j = 0; j < kChains; ++j) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[j]) : "l"(x), "l"(y));
    unsigned long long s = 0;
#pragma unroll
    for (int j = 0; j < kChains; ++j) s ^= a[j];
    if (s == 0x123456789abcdefull) sink[tid] = (double)s;
  } else {  // MT_PEAK_MMA_TF32: warp-level mma.sync m16n8k8, tf32 operands, fp32 accumulate
    float d[kChains][4];
    const unsigned a0 = __float_as_uint(1.0f + (float)(tid & 3)), b0 = __float_as_uint(0.5f + (float)seed);
#pragma unroll
    for (int j = 0; j < kChains; ++j) d[j][0] = d[j][1] = d[j][2] = d[j][3] = (float)j;
    for (int it = 0; it < iters; ++it)
#pragma unroll
      for (int u = 0; u < kUnroll; ++u)
#pragma unroll
        for (int j = 0; j < kChains; ++j)
          asm volatile(
              "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
              : "+f"(d[j][0]), "+f"(d[j][1]), "+f"(d[j][2]), "+f"(d[j][3])
              : "r"(a0), "r"(a0), "r"(a0), "r"(a0), "r"(b0), "r"(b0));
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < kChains; ++j) s += d[j][0] + d[j][1] + d[j][2] + d[j][3];
    if (s == 12345.678f) sink[tid] = s;
  }
}

// ---- read-only HBM stream: one thread per CTA keeps a ring of 1-D bulk copies (TMA) in flight ----
constexpr int kRdStages = 6;
constexpr uint32_t kRdChunk = 32 * 1024;

__device__ __forceinline__ uint32_t s32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__global__ void __launch_bounds__(32, 1) hbm_read_kernel(const unsigned char* src, int64_t chunks) {
  extern __shared__ __align__(128) unsigned char ring[];
  __shared__ __align__(8) uint64_t bars[kRdStages];
  if (threadIdx.x != 0) return;
  for (int s = 0; s < kRdStages; ++s)
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(s32(&bars[s])) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  const int64_t P = gridDim.x, c = blockIdx.x;
  const int64_t c0 = chunks * c / P, c1 = chunks * (c + 1) / P;
  auto wait = [&](int s, uint32_t parity) {
    uint32_t ok;
    do {
      asm volatile(
          "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
          : "=r"(ok)
          : "r"(s32(&bars[s])), "r"(parity)
          : "memory");
    } while (!ok);
  };
  int64_t issued = 0;
  for (int64_t i = c0; i < c1; ++i, ++issued) {
    const int s = (int)(issued % kRdStages);
    if (issued >= kRdStages) wait(s, (uint32_t)((issued / kRdStages - 1) & 1));
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s32(&bars[s])), "r"(kRdChunk) : "memory");
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            s32(ring + (size_t)s * kRdChunk)),
        "l"(src + i * (int64_t)kRdChunk), "r"(kRdChunk), "r"(s32(&bars[s])), "l"(pol)
        : "memory");
  }
  // drain: the last min(issued, stages) copies
  const int64_t first = issued > kRdStages ? issued - kRdStages : 0;
  for (int64_t j = first; j < issued; ++j) wait((int)(j % kRdStages), (uint32_t)((j / kRdStages) & 1));
}

}  // namespace

extern "C" int mt_measure_peak(mt_ctx* ctx, int kind, const void* buf, int64_t bytes, double* out_host) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!out_host) return mt_fail(ctx, MT_ERR_INVALID_ARG, "out_host is NULL");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
  cudaEvent_t e0, e1;
  MT_CUDA_OK(ctx, cudaEventCreate(&e0));
  MT_CUDA_OK(ctx, cudaEventCreate(&e1));
  double best_ms = 1e300, work = 0.0;
  int rc = MT_OK;
  auto fail = [&](cudaError_t ce) { rc = mt_fail(ctx, MT_ERR_CUDA, "mt_measure_peak: %s", cudaGetErrorString(ce)); };
  for (int rep = 0; rep < 4 && rc == MT_OK; ++rep) {  // first repetition = warm-up, best of the other three
    cudaEventRecord(e0, st);
    if (kind == MT_PEAK_HBM_READ) {
      if (!buf || bytes < (int64_t)kRdChunk * ctx->num_sms || ((uintptr_t)buf & 15)) {
        rc = mt_fail(ctx, MT_ERR_INVALID_ARG, "MT_PEAK_HBM_READ needs a 16-byte aligned device buffer of >= %lld bytes",
                     (long long)kRdChunk * ctx->num_sms);
        break;
      }
      static unsigned char attr_set[64] = {};
      if (!attr_set[ctx->device & 63]) {
        cudaError_t ce = cudaFuncSetAttribute(hbm_read_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              (int)(kRdStages * kRdChunk));
        if (ce != cudaSuccess) { fail(ce); break; }
        attr_set[ctx->device & 63] = 1;
      }
      const int64_t chunks = bytes / kRdChunk;
      hbm_read_kernel<<<ctx->num_sms, 32, kRdStages * kRdChunk, st>>>((const unsigned char*)buf, chunks);
      work = (double)chunks * kRdChunk;
    } else {
      const int iters = (kind == MT_PEAK_DFMA || kind == MT_PEAK_MMA_TF32) ? 4096 : 16384;
      const int blocks = ctx->num_sms * kAluBlocksPerSm;
      const double seed = 1.0;
      double* sink = (double*)ctx->dscal;  // never written (the guard is never true)
      switch (kind) {
        case MT_PEAK_DFMA: alu_peak_kernel<MT_PEAK_DFMA><<<blocks, kAluThreads, 0, st>>>(iters, sink, seed); break;
        case MT_PEAK_FFMA: alu_peak_kernel<MT_PEAK_FFMA><<<blocks, kAluThreads, 0, st>>>(iters, sink, seed); break;
        case MT_PEAK_FFMA2: alu_peak_kernel<MT_PEAK_FFMA2><<<blocks, kAluThreads, 0, st>>>(iters, sink, seed); break;
        case MT_PEAK_MMA_TF32: alu_peak_kernel<MT_PEAK_MMA_TF32><<<blocks, kAluThreads, 0, st>>>(iters, sink, seed); break;
        default: rc = mt_fail(ctx, MT_ERR_INVALID_ARG, "unknown peak kind %d", kind); break;
      }
      if (rc) break;
      const double per_thread = (double)iters * kUnroll * kChains;
      const double threads = (double)blocks * kAluThreads;
      // thread-instructions (an f32x2 instruction counts as one; a warp-level mma as 1024 MACs)
      work = kind == MT_PEAK_MMA_TF32 ? per_thread * (threads / 32.0) * 1024.0 : per_thread * threads;
    }
    ctx->launches++;
    cudaError_t ce = cudaGetLastError();
    if (ce != cudaSuccess) { fail(ce); break; }
    cudaEventRecord(e1, st);
    ce = cudaEventSynchronize(e1);
    if (ce != cudaSuccess) { fail(ce); break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best_ms) best_ms = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (rc) return rc;
  out_host[0] = work / (best_ms * 1e-3);
  out_host[1] = best_ms;
  return MT_OK;
}
