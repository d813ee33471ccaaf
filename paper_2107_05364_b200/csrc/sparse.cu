// sparse.cu — F1: thresholded ("sparse") demagnetisation tensor, PAPER.md:235-243 (§4.3.1).
//
// "the demagnetization tensor can be reduced in size by removing all elements of the
// tensor smaller than a given threshold value ... This also allows the demagnetization tensor, which
// normally is a dense matrix, to be allocated as a sparse matrix, thus saving memory, which is
// especially important when doing CUDA calculations."  PAPER.md:239 defines the threshold as a
// fraction of the non-zero elements sorted by absolute value (reading DESIGN.md Q20).
//
// Three pieces:
//  1. threshold selection: the k-th smallest |v| among the non-zero elements, by an MSB-first radix
//     select over the bit patterns of |v| (which order like unsigned integers): one streaming pass of
//     the dense tensor per 11-bit digit, integer histogram in shared memory -> exact and reproducible.
//  2. compression to BITMAP ROWS: per (plane, row) a bit per column (1 = kept) and the kept values
//     packed in column order.  Unlike CSR (4-byte column index per 4-byte value: no saving until more
//     than half of the entries are gone — the slowdown at small thresholds PAPER.md:241 reports) the
//     index costs 1/32 of a dense fp32 row, so HBM bytes per evaluation fall as (1 - X) + 3 %.
//  3. the field kernel on that layout (A4-A7 semantics, same fused epilogue): one warp per target row;
//     a 32-column chunk is one mask word per plane (uniform load), lane l owns column 32 c + l and
//     fetches its value at offset popc(mask & lanes-below) of the chunk's packed run.
#include "epilogue.cuh"

namespace {

constexpr int kDigitBits = 11;
constexpr int kBins = 1 << kDigitBits;

template <typename T> struct KeyOf;
template <> struct KeyOf<float> {
  typedef uint32_t type;
  static constexpr int bits = 32;
  __device__ static __forceinline__ uint32_t key(float v) { return __float_as_uint(v) & 0x7fffffffu; }
};
template <> struct KeyOf<double> {
  typedef unsigned long long type;
  static constexpr int bits = 64;
  __device__ static __forceinline__ unsigned long long key(double v) {
    return (unsigned long long)__double_as_longlong(v) & 0x7fffffffffffffffull;
  }
};

template <typename T> struct Vec16;  // 16 bytes of the row: rows are 16-byte aligned (include/mt.h)
template <> struct Vec16<float> { typedef float4 type; static constexpr int n = 4; };
template <> struct Vec16<double> { typedef double2 type; static constexpr int n = 2; };
__device__ __forceinline__ void unpack16(const float4& q, float (&x)[4]) { x[0] = q.x; x[1] = q.y; x[2] = q.z; x[3] = q.w; }
__device__ __forceinline__ void unpack16(const double2& q, double (&x)[2]) { x[0] = q.x; x[1] = q.y; }

// hist[d] += multiplicity of every non-zero element whose key has the given prefix above `shift+width`
// and digit d at `shift`; planes xy, xz, yz (1, 2, 4) count twice (Q20).
template <typename T>
__global__ void __launch_bounds__(512) select_hist_kernel(const T* __restrict__ N, int64_t n, int64_t n_rows,
                                                          int64_t ld, typename KeyOf<T>::type prefix,
                                                          int prefix_shift, int shift, int width,
                                                          unsigned long long* __restrict__ hist) {
  typedef typename KeyOf<T>::type K;
  typedef typename Vec16<T>::type V;
  constexpr int kV = Vec16<T>::n;
  // 32-bit shared counters (a block sees far fewer than 2^31 elements: the launcher bounds the rows
  // per block), flushed into the 64-bit global histogram.  A lane reads 16 bytes (kV neighbouring
  // columns), two such loads in flight.  Neighbouring columns hold values of similar magnitude, i.e.
  // the same bin: per vector component a warp aggregates RUNS of equal bins over its lanes (one shuffle
  // + one ballot) and issues one shared atomic per run instead of up to 32 serialised ones.  In the
  // passes below the first almost no element carries the prefix: a warp whose elements are all
  // uncounted skips the aggregation (one vote).
  __shared__ unsigned int sh[kBins];
  for (int k = threadIdx.x; k < kBins; k += blockDim.x) sh[k] = 0u;
  __syncthreads();
  const int64_t rows_total = 6 * n_rows;
  const K dmask = (K)((1u << width) - 1u);
  const int lane = threadIdx.x & 31;
  const uint32_t above = ~((2u << lane) - 1u);  // lanes above this one
  // (key & pmask) == pval  <=>  the bits above prefix_shift equal the prefix (first pass: no bits)
  const bool has_prefix = prefix_shift < KeyOf<T>::bits;
  const K pmask = has_prefix ? ~(((K)1 << prefix_shift) - (K)1) : (K)0;
  const K pval = has_prefix ? (K)(prefix << prefix_shift) : (K)0;
  const int step = (int)blockDim.x * kV;
  const int n_up = (int)((n + 32 * kV - 1) / (32 * kV)) * (32 * kV);  // whole warps stay converged
  for (int64_t r = blockIdx.x; r < rows_total; r += gridDim.x) {
    const int plane = (int)(r / n_rows);
    const unsigned int w = (plane == 1 || plane == 2 || plane == 4) ? 2u : 1u;
    const T* row = N + r * ld;
    for (int j0 = (int)threadIdx.x * kV; j0 < n_up; j0 += 2 * step) {
      T x[2][kV];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int j = j0 + u * step;
        if (j < ld) {
          unpack16(__ldg(reinterpret_cast<const V*>(row + j)), x[u]);
          if (j + kV > n) {  // the row's last vector: columns >= n are padding
#pragma unroll
            for (int c = 0; c < kV; ++c)
              if (j + c >= n) x[u][c] = T(0);
          }
        } else {
#pragma unroll
          for (int c = 0; c < kV; ++c) x[u][c] = T(0);
        }
      }
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int j = j0 + u * step;
        if (j - lane * kV >= n_up) break;  // warp-uniform
        K key[kV];
        bool counted[kV], any = false;
#pragma unroll
        for (int c = 0; c < kV; ++c) {
          key[c] = KeyOf<T>::key(x[u][c]);
          counted[c] = key[c] != 0 && (key[c] & pmask) == pval;
          any |= counted[c];
        }
        if (!__any_sync(0xffffffffu, any)) continue;
#pragma unroll
        for (int c = 0; c < kV; ++c) {
          const unsigned bin = counted[c] ? (unsigned)((key[c] >> shift) & dmask) : (unsigned)kBins;  // "none"
          const unsigned prev = __shfl_up_sync(0xffffffffu, bin, 1);
          const bool head = lane == 0 || bin != prev;
          const uint32_t heads = __ballot_sync(0xffffffffu, head);
          if (head && counted[c]) {
            const uint32_t next = heads & above;
            const int len = (next ? __ffs(next) - 1 : 32) - lane;
            atomicAdd(&sh[bin], w * (unsigned)len);
          }
        }
      }
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < kBins; k += blockDim.x)
    if (sh[k]) atomicAdd(&hist[k], (unsigned long long)sh[k]);
}

// Wide digit (up to 20 bits) for the passes after the first: only the elements that carry the prefix
// fixed so far are counted — a few percent of the tensor after the first 11 bits, almost none later —
// so their bins are added straight to the global histogram (64-bit atomics in L2, spread over up to 2^20
// bins: no contention to speak of).  One pass of this kind replaces two 11-bit passes.
template <typename T>
__global__ void __launch_bounds__(512) select_hist_wide_kernel(const T* __restrict__ N, int64_t n, int64_t n_rows,
                                                               int64_t ld, typename KeyOf<T>::type prefix,
                                                               int prefix_shift, int shift, int width,
                                                               unsigned long long* __restrict__ hist) {
  typedef typename KeyOf<T>::type K;
  typedef typename Vec16<T>::type V;
  constexpr int kV = Vec16<T>::n;
  const int64_t rows_total = 6 * n_rows;
  const K dmask = (K)(((K)1 << width) - (K)1);
  const K pmask = ~(((K)1 << prefix_shift) - (K)1);
  const K pval = (K)(prefix << prefix_shift);
  const int step = (int)blockDim.x * kV;
  for (int64_t r = blockIdx.x; r < rows_total; r += gridDim.x) {
    const int plane = (int)(r / n_rows);
    const unsigned long long w = (plane == 1 || plane == 2 || plane == 4) ? 2ull : 1ull;
    const T* row = N + r * ld;
    for (int j0 = (int)threadIdx.x * kV; j0 < n; j0 += 2 * step) {
      T x[2][kV];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int j = j0 + u * step;
#pragma unroll
        for (int c = 0; c < kV; ++c) x[u][c] = T(0);
        if (j < n) {
          unpack16(__ldg(reinterpret_cast<const V*>(row + j)), x[u]);
#pragma unroll
          for (int c = 0; c < kV; ++c)
            if (j + c >= n) x[u][c] = T(0);  // padding of the row's last vector
        }
      }
#pragma unroll
      for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int c = 0; c < kV; ++c) {
          const K key = KeyOf<T>::key(x[u][c]);
          if (key != 0 && (key & pmask) == pval) atomicAdd(&hist[(size_t)((key >> shift) & dmask)], w);
        }
    }
  }
}

// One block: total = sum of the bins; first pass: k = floor(fraction * total); the bin that holds rank k
// and the rank inside it.  out[0] = total, out[1] = bin, out[2] = k - (sum of the bins below), out[3] = k
// as used.  Integer arithmetic on the bins, fixed order: exact.
__global__ void __launch_bounds__(1024) select_find_kernel(const unsigned long long* __restrict__ hist, int nbins,
                                                           unsigned long long k_in, int first_pass, double fraction,
                                                           unsigned long long* __restrict__ out) {
  __shared__ unsigned long long part[1024];
  __shared__ unsigned long long k_sh;
  const int per = nbins > 1024 ? nbins / 1024 : 1;
  const int b0 = (int)threadIdx.x * per;
  unsigned long long s = 0;
  for (int b = b0; b < b0 + per && b < nbins; ++b) s += hist[b];
  part[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long run = 0;
    for (int t = 0; t < 1024; ++t) { const unsigned long long v = part[t]; part[t] = run; run += v; }  // exclusive
    out[0] = run;
    unsigned long long k = k_in;
    if (first_pass) k = (unsigned long long)floor(fraction * (double)run);
    k_sh = k;
    out[3] = k;
    if (k >= run) { out[1] = (unsigned long long)(nbins - 1); out[2] = k; }  // caller: everything removed / last bin
  }
  __syncthreads();
  const unsigned long long k = k_sh, below = part[threadIdx.x];
  if (k >= below && k < below + s) {
    unsigned long long rem = k - below;
    int b = b0;
    while (b < b0 + per - 1 && b < nbins - 1 && rem >= hist[b]) { rem -= hist[b]; ++b; }
    out[1] = (unsigned long long)b;
    out[2] = rem;
  }
}

template <typename T> __device__ __forceinline__ bool kept(T v, T tau) { return v != T(0) && !(fabs(v) < tau); }

// N holds rows [row0, row0 + n_rows) of a tensor of n_total rows (the whole tensor: row0 = 0, n_total =
// n_rows): counts[plane * n_total + row0 + i] = kept entries of band row i of the plane; one warp per
// (plane, band row)
template <typename T>
__global__ void __launch_bounds__(256) sparse_count_kernel(const T* __restrict__ N, int64_t n, int64_t n_rows,
                                                           int64_t ld, T tau, int64_t row0, int64_t n_total,
                                                           int64_t* __restrict__ counts) {
  const int64_t r = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (r >= 6 * n_rows) return;
  const int64_t R = (r / n_rows) * n_total + row0 + r % n_rows;
  const T* row = N + r * ld;
  typedef typename Vec16<T>::type V;
  constexpr int kV = Vec16<T>::n;
  int c = 0;
  for (int64_t j = (int64_t)lane * kV; j < n; j += 32 * kV) {  // 16-byte loads (rows are 16-byte aligned)
    T x[kV];
    unpack16(__ldg(reinterpret_cast<const V*>(row + j)), x);
#pragma unroll
    for (int q = 0; q < kV; ++q) c += (j + q < n && kept(x[q], tau)) ? 1 : 0;
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) c += __shfl_xor_sync(0xffffffffu, c, off);
  if (lane == 0) counts[R] = c;
}

// in-place exclusive scan of len+1 int64 (slot len receives the total); one block, sequential chunks
__global__ void __launch_bounds__(1024) scan_kernel(int64_t* __restrict__ a, int64_t len) {
  __shared__ int64_t sh[1024];
  __shared__ int64_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int64_t base = 0; base < len; base += 1024) {
    const int64_t i = base + threadIdx.x;
    const int64_t v = i < len ? a[i] : 0;
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
      const int64_t t = (int)threadIdx.x >= off ? sh[threadIdx.x - off] : 0;
      __syncthreads();
      sh[threadIdx.x] += t;
      __syncthreads();
    }
    if (i < len) a[i] = carry + sh[threadIdx.x] - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry += sh[1023];
    __syncthreads();
  }
  if (threadIdx.x == 0) a[len] = carry;
}

// mask[(plane * n_rows + i) * nw + c] bit l = entry (i, 32 c + l) kept; kept values packed from
// vals[row_ptr[plane * n_rows + i]] in column order.  One warp per (plane, row).  Optionally (cols
// non-NULL) the index rows are written in the same pass — 16-bit column of every packed value and the
// panel offsets, exactly what sparse_index_kernel derives from the bitmap — and the bitmap itself may
// then be left out (mask NULL).
template <typename T>
__global__ void __launch_bounds__(256) sparse_fill_kernel(const T* __restrict__ N, int64_t n, int64_t n_rows,
                                                          int64_t ld, T tau, int64_t row0, int64_t n_total,
                                                          const int64_t* __restrict__ row_ptr, int64_t nw,
                                                          uint32_t* __restrict__ mask, T* __restrict__ vals,
                                                          uint16_t* __restrict__ cols,
                                                          int64_t* __restrict__ panel_ptr, int npanels) {
  const int64_t r = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (r >= 6 * n_rows) return;
  const int64_t R = (r / n_rows) * n_total + row0 + r % n_rows;  // row of the whole tensor (see count)
  const T* row = N + r * ld;
  uint32_t* mrow = mask ? mask + R * nw : nullptr;
  const int64_t base = row_ptr[R];
  T* out = vals + base;
  uint16_t* cout = cols ? cols + base : nullptr;
  int64_t off = 0;
  for (int64_t c0 = 0; c0 < nw; c0 += 4) {  // nw is a multiple of 4; four chunks loaded before any is packed
    if (cout && c0 && (c0 & 2047) == 0 && lane == 0) panel_ptr[R * (npanels - 1) + (c0 >> 11) - 1] = base + off;
    T v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t j = (c0 + u) * 32 + lane;
      v[u] = j < n ? __ldg(row + j) : T(0);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const bool k = kept(v[u], tau);
      const uint32_t word = __ballot_sync(0xffffffffu, k);
      if (k) {
        const int64_t at = off + __popc(word & ((1u << lane) - 1u));
        out[at] = v[u];
        if (cout) cout[at] = (uint16_t)((c0 + u) * 32 + lane);
      }
      if (mrow && lane == 0) mrow[c0 + u] = word;
      off += __popc(word);
    }
  }
}

// ---- field kernel on bitmap rows (A4-A7 on the thresholded tensor) ---------------------------------
// fp32: products and a run of at most 32 chunks x 3 terms in fp32, then fp64 (Q19);
// fp64: DFMA throughout.  Lanes are combined by a fixed xor butterfly: bitwise reproducible.
constexpr int kGroupChunks = 32;

struct SparseArgs {
  int64_t n, n_rows, nw, npad;
  const int64_t* row_ptr;
  const uint32_t* mask;
  const void* vals;
  const void* Mst;
  const int64_t* panel_ptr;  // index rows with n > 65536: [6 * n_rows][npanels - 1] offsets into vals
  int npanels;               // column panels of 65,536 (16-bit columns are relative to their panel)
};

// One group = 32 chunks (1,024 columns): lane l loads the mask word of chunk c0 + l of every plane
// (six coalesced 128-byte loads), a warp scan of the popcounts gives every chunk's offset into the
// packed values, and a ballot gives the chunks that hold anything at all — the others are skipped,
// which is where a thresholded tensor (near-field runs, "a more or less spherical region")
// saves time as well as bytes.  Two non-empty chunks are processed per iteration so that their value
// loads are in flight together.
template <typename T, int B>
__device__ __forceinline__ void bitmap_chunk(const uint32_t (&mw)[6], const uint32_t (&ex)[3], int c, bool valid, int lane,
                                             uint32_t lt, const T* const (&vrow)[6], const int (&base)[6],
                                             T (&v)[6]) {
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    const uint32_t e2 = __shfl_sync(0xffffffffu, ex[q], c);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int p = 2 * q + h;
      const uint32_t word = valid ? __shfl_sync(0xffffffffu, mw[p], c) : 0u;
      const int st = (int)((e2 >> (16 * h)) & 0xffffu);
      v[p] = ((word >> lane) & 1u) ? __ldg(vrow[p] + base[p] + st + __popc(word & lt)) : T(0);
    }
  }
}

template <typename T, int B>
__global__ void __launch_bounds__(256) demag_bitmap_kernel(SparseArgs a, EpiArgs e) {
  const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (row >= a.n_rows) return;
  const uint32_t lt = (1u << lane) - 1u;
  const uint32_t* mrow[6];
  const T* vrow[6];
  int base[6];
#pragma unroll
  for (int p = 0; p < 6; ++p) {
    const int64_t r = (int64_t)p * a.n_rows + row;
    mrow[p] = a.mask + r * a.nw;
    vrow[p] = (const T*)a.vals + a.row_ptr[r];
    base[p] = 0;
  }
  const T* M = (const T*)a.Mst;
  double acc[B][3];
#pragma unroll
  for (int b = 0; b < B; ++b) acc[b][0] = acc[b][1] = acc[b][2] = 0.0;
  for (int64_t c0 = 0; c0 < a.nw; c0 += kGroupChunks) {
    uint32_t mw[6], ex[3], any = 0u;
#pragma unroll
    for (int p = 0; p < 6; ++p) {
      mw[p] = (c0 + lane < a.nw) ? __ldg(mrow[p] + c0 + lane) : 0u;
      any |= mw[p];
    }
    // inclusive scan of the popcounts, two planes per register (16-bit fields; a group holds <= 1,024)
    uint32_t inc[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const uint32_t own = (uint32_t)__popc(mw[2 * q]) | ((uint32_t)__popc(mw[2 * q + 1]) << 16);
      uint32_t x = own;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += t;
      }
      inc[q] = x;
      ex[q] = x - own;
    }
    uint32_t nz = __ballot_sync(0xffffffffu, any != 0u);
    T run[B][3];
#pragma unroll
    for (int b = 0; b < B; ++b) run[b][0] = run[b][1] = run[b][2] = T(0);
    while (nz) {
      const int ca = __ffs(nz) - 1;
      nz &= nz - 1u;
      const bool two = nz != 0u;
      const int cb = two ? __ffs(nz) - 1 : ca;
      nz &= nz - 1u;  // no-op when nz == 0
      T va[6], vb[6];
      bitmap_chunk<T, B>(mw, ex, ca, true, lane, lt, vrow, base, va);
      bitmap_chunk<T, B>(mw, ex, cb, two, lane, lt, vrow, base, vb);
      const int64_t cola = (c0 + ca) * 32 + lane, colb = (c0 + cb) * 32 + lane;  // < npad
#pragma unroll
      for (int b = 0; b < B; ++b) {
        const T* Mb = M + (int64_t)b * 3 * a.npad;
        const T ax = Mb[cola], ay = Mb[a.npad + cola], az = Mb[2 * a.npad + cola];
        const T bx = Mb[colb], by = Mb[a.npad + colb], bz = Mb[2 * a.npad + colb];
        run[b][0] = fma(va[0], ax, fma(va[1], ay, fma(va[2], az, run[b][0])));
        run[b][1] = fma(va[1], ax, fma(va[3], ay, fma(va[4], az, run[b][1])));
        run[b][2] = fma(va[2], ax, fma(va[4], ay, fma(va[5], az, run[b][2])));
        run[b][0] = fma(vb[0], bx, fma(vb[1], by, fma(vb[2], bz, run[b][0])));
        run[b][1] = fma(vb[1], bx, fma(vb[3], by, fma(vb[4], bz, run[b][1])));
        run[b][2] = fma(vb[2], bx, fma(vb[4], by, fma(vb[5], bz, run[b][2])));
      }
    }
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const uint32_t tot = __shfl_sync(0xffffffffu, inc[q], 31);
      base[2 * q] += (int)(tot & 0xffffu);
      base[2 * q + 1] += (int)(tot >> 16);
    }
#pragma unroll
    for (int b = 0; b < B; ++b) {
      acc[b][0] += (double)run[b][0];
      acc[b][1] += (double)run[b][1];
      acc[b][2] += (double)run[b][2];
    }
  }
#pragma unroll
  for (int b = 0; b < B; ++b)
#pragma unroll
    for (int cc = 0; cc < 3; ++cc)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[b][cc] += __shfl_xor_sync(0xffffffffu, acc[b][cc], o);
  double s[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int b = 0; b < B; ++b)
    if (lane == b) { s[0] = acc[b][0]; s[1] = acc[b][1]; s[2] = acc[b][2]; }
  if (lane < B) {
    const double hd[3] = {-s[0], -s[1], -s[2]};
    row_epilogue(e, row, lane, hd);
  }
}

template <typename T, int B>
int launch_bitmap_B(mt_ctx* ctx, const SparseArgs& a, const EpiArgs& e) {
  demag_bitmap_kernel<T, B><<<(unsigned)((a.n_rows + 7) / 8), 256, 0, ctx->stream>>>(a, e);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

template <typename T>
int launch_bitmap(mt_ctx* ctx, const SparseArgs& a, const EpiArgs& e) {
  switch (e.batch) {
    case 1: return launch_bitmap_B<T, 1>(ctx, a, e);
    case 2: return launch_bitmap_B<T, 2>(ctx, a, e);
    case 3: return launch_bitmap_B<T, 3>(ctx, a, e);
    case 4: return launch_bitmap_B<T, 4>(ctx, a, e);
    case 5: return launch_bitmap_B<T, 5>(ctx, a, e);
    case 6: return launch_bitmap_B<T, 6>(ctx, a, e);
    case 7: return launch_bitmap_B<T, 7>(ctx, a, e);
    case 8: return launch_bitmap_B<T, 8>(ctx, a, e);
  }
  return mt_fail(ctx, MT_ERR_INVALID_ARG, "batch must be in [1, %d]", MT_MAX_BATCH);
}

// ---- index rows: the second index of the thresholded tensor ----------------------------------------
// cols[row_ptr[r] + k] = column of the k-th set bit of bitmap row r; one warp per (plane, row).
__global__ void __launch_bounds__(256) sparse_index_kernel(const uint32_t* __restrict__ mask,
                                                           const int64_t* __restrict__ row_ptr, int64_t n_rows,
                                                           int64_t nw, uint16_t* __restrict__ cols,
                                                           int64_t* __restrict__ panel_ptr, int npanels) {
  const int64_t r = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (r >= 6 * n_rows) return;
  const uint32_t* mrow = mask + r * nw;
  uint16_t* out = cols + row_ptr[r];
  const uint32_t lt = (1u << lane) - 1u;
  int64_t off = 0;
  for (int64_t c0 = 0; c0 < nw; c0 += 32) {
    // a panel of 65,536 columns = 2,048 mask words: the packed offset at which panel q >= 1 starts
    if (c0 && (c0 & 2047) == 0 && lane == 0) panel_ptr[r * (npanels - 1) + (c0 >> 11) - 1] = row_ptr[r] + off;
    const uint32_t mine = c0 + lane < nw ? __ldg(mrow + c0 + lane) : 0u;
    uint32_t nz = __ballot_sync(0xffffffffu, mine != 0u);
    while (nz) {
      const int c = __ffs(nz) - 1;
      nz &= nz - 1u;
      const uint32_t word = __shfl_sync(0xffffffffu, mine, c);
      if ((word >> lane) & 1u) out[off + __popc(word & lt)] = (uint16_t)((c0 + c) * 32 + lane);
      off += __popc(word);
    }
  }
}

// Field kernel on index rows: one warp per target row walks the packed values of each of its six
// plane rows in order (lane l takes entries l, l + 32, ...): one coalesced value load and one coalesced
// 16-bit column load per 32 entries, M gathered at the columns (near-field runs are contiguous, so the
// gathers fall in one or two 128-byte lines; M is L1/L2-resident), and only the products the plane
// contributes: one for a diagonal plane, two for an off-diagonal one.  ~12 instructions per 32 kept
// entries against ~150 per visited chunk of the bitmap decode.  fp32: a lane's run of kUnroll * kFlush
// entries per plane is summed in fp32, then added to fp64 (Q19); fp64: DFMA throughout.
// Fixed order (lane-strided walk, xor butterfly): bitwise reproducible.
constexpr int kIdxUnroll = 8;
constexpr int kIdxFlush = 8;

template <int P> struct PlaneRC;  // plane -> (row component, column component) of the 3x3 block
template <> struct PlaneRC<0> { static constexpr int r = 0, c = 0; };
template <> struct PlaneRC<1> { static constexpr int r = 0, c = 1; };
template <> struct PlaneRC<2> { static constexpr int r = 0, c = 2; };
template <> struct PlaneRC<3> { static constexpr int r = 1, c = 1; };
template <> struct PlaneRC<4> { static constexpr int r = 1, c = 2; };
template <> struct PlaneRC<5> { static constexpr int r = 2, c = 2; };

// The value and column streams are read once: they bypass L1 so that the gathered M stays there.
__device__ __forceinline__ float ld_stream(const float* p) {
  float v;
  asm volatile("ld.global.nc.L1::no_allocate.L2::256B.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ double ld_stream(const double* p) {
  double v;
  asm volatile("ld.global.nc.L1::no_allocate.L2::256B.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ int ld_stream(const uint16_t* p) {
  unsigned short v;
  asm volatile("ld.global.nc.L1::no_allocate.L2::256B.u16 %0, [%1];" : "=h"(v) : "l"(p));
  return (int)v;
}

template <typename T>
__device__ __forceinline__ void index_load(const T* __restrict__ vals, const uint16_t* __restrict__ cols, int64_t k,
                                           int64_t end, T (&v)[kIdxUnroll], int (&col)[kIdxUnroll]) {
#pragma unroll
  for (int u = 0; u < kIdxUnroll; ++u) {
    const int64_t ku = k + 32 * u;
    const bool ok = ku < end;
    v[u] = ok ? ld_stream(vals + ku) : T(0);
    col[u] = ok ? ld_stream(cols + ku) : 0;
  }
}

// beg/end: the plane row's range in vals/cols (read by the caller for all six planes up front).  The
// next block's values and columns are requested before the current block's gathers are issued, so a
// warp keeps two blocks of kIdxUnroll * 32 entries (2 x 1.5 KB) in flight towards HBM.
// BP = 0: M is the plain staged layout [B][3][npad] (one gather per state and component: fine for 1-2 states).
// BP = 4 / 8: M is interleaved [3][npad][BP] (interleave_stage_kernel), so that ONE gather of BP values serves
// all states of a batch: the per-entry cost of a batch of 8 is two 32-byte loads instead of sixteen scalar ones.
template <typename T, int BP> struct StateVec;
template <> struct StateVec<float, 4> { float4 v[1]; };
template <> struct StateVec<float, 8> { float4 v[2]; };
template <> struct StateVec<double, 4> { double2 v[2]; };
template <> struct StateVec<double, 8> { double2 v[4]; };

template <typename T, int B, int P, int BP>
__device__ __forceinline__ void index_panel(const SparseArgs& a, const uint16_t* __restrict__ cols, int64_t beg,
                                            int64_t end, int64_t col0, int lane, double (&acc)[B][3]) {
  constexpr int R = PlaneRC<P>::r, Cc = PlaneRC<P>::c;
  const T* __restrict__ vals = (const T*)a.vals;
  const T* __restrict__ M = (const T*)a.Mst + (BP ? col0 * BP : col0);
  T vn[kIdxUnroll];
  int cn[kIdxUnroll];
  int64_t kb = beg;  // warp-uniform block start
  index_load<T>(vals, cols, kb + lane, end, vn, cn);
  while (kb < end) {
    T runR[B], runC[B];
#pragma unroll
    for (int b = 0; b < B; ++b) runR[b] = runC[b] = T(0);
    for (int f = 0; f < kIdxFlush && kb < end; ++f) {
      T v[kIdxUnroll];
      int col[kIdxUnroll];
#pragma unroll
      for (int u = 0; u < kIdxUnroll; ++u) { v[u] = vn[u]; col[u] = cn[u]; }
      kb += 32 * kIdxUnroll;
      index_load<T>(vals, cols, kb + lane, end, vn, cn);
      if constexpr (BP == 0) {
#pragma unroll
        for (int b = 0; b < B; ++b) {
          const T* Mb = M + (int64_t)b * 3 * a.npad;
#pragma unroll
          for (int u = 0; u < kIdxUnroll; ++u) {
            runR[b] = fma(v[u], __ldg(Mb + (int64_t)Cc * a.npad + col[u]), runR[b]);
            if (R != Cc) runC[b] = fma(v[u], __ldg(Mb + (int64_t)R * a.npad + col[u]), runC[b]);
          }
        }
      } else {
        typedef StateVec<T, BP> SV;
#pragma unroll
        for (int u = 0; u < kIdxUnroll; ++u) {
          const SV mc = *reinterpret_cast<const SV*>(M + ((int64_t)Cc * a.npad + col[u]) * BP);
          const T* pc = reinterpret_cast<const T*>(&mc);
#pragma unroll
          for (int b = 0; b < B; ++b) runR[b] = fma(v[u], pc[b], runR[b]);
          if (R != Cc) {
            const SV mr = *reinterpret_cast<const SV*>(M + ((int64_t)R * a.npad + col[u]) * BP);
            const T* pr = reinterpret_cast<const T*>(&mr);
#pragma unroll
            for (int b = 0; b < B; ++b) runC[b] = fma(v[u], pr[b], runC[b]);
          }
        }
      }
    }
#pragma unroll
    for (int b = 0; b < B; ++b) {
      acc[b][R] += (double)runR[b];
      if (R != Cc) acc[b][Cc] += (double)runC[b];
    }
  }
}

// A plane row = its column panels in turn (PANELS = false, n <= 65,536: the one panel, nothing extra).
template <typename T, int B, int P, bool PANELS, int BP>
__device__ __forceinline__ void index_plane(const SparseArgs& a, const uint16_t* __restrict__ cols, int64_t row,
                                            int64_t beg, int64_t end, int lane, double (&acc)[B][3]) {
  if (!PANELS) {
    index_panel<T, B, P, BP>(a, cols, beg, end, 0, lane, acc);
    return;
  }
  const int64_t* pp = a.panel_ptr + ((int64_t)P * a.n_rows + row) * (a.npanels - 1);
  int64_t b = beg;
  for (int q = 0; q < a.npanels; ++q) {
    const int64_t e = q + 1 < a.npanels ? __ldg(pp + q) : end;
    index_panel<T, B, P, BP>(a, cols, b, e, (int64_t)q << 16, lane, acc);
    b = e;
  }
}

// M[b][c][j] (plain staged layout, MT_MAX_BATCH states) -> Mi[c][j][b], b < BP
template <typename T, int BP>
__global__ void __launch_bounds__(256) interleave_stage_kernel(const T* __restrict__ M, int64_t npad, T* __restrict__ Mi) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // (c, j)
  if (idx >= 3 * npad) return;
  const int64_t c = idx / npad, j = idx % npad;
#pragma unroll
  for (int b = 0; b < BP; ++b) Mi[idx * BP + b] = M[((int64_t)b * 3 + c) * npad + j];
}

template <typename T, int B, bool PANELS, int BP = 0>
__global__ void __launch_bounds__(256, (B <= 2 ? 4 : 2)) demag_index_kernel(SparseArgs a, const uint16_t* __restrict__ cols, EpiArgs e) {
  const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (row >= a.n_rows) return;
  double acc[B][3];
#pragma unroll
  for (int b = 0; b < B; ++b) acc[b][0] = acc[b][1] = acc[b][2] = 0.0;
  // the range of plane p + 1 is requested before plane p is walked
  const int64_t* rp = a.row_ptr + row;
  int64_t beg = __ldg(rp), end = __ldg(rp + 1), nbeg = 0, nend = 0;
#define MT_INDEX_PLANE(P)                                      \
  if (P < 5) {                                                 \
    nbeg = __ldg(rp + (int64_t)(P + 1) * a.n_rows);            \
    nend = __ldg(rp + (int64_t)(P + 1) * a.n_rows + 1);        \
  }                                                            \
  index_plane<T, B, P, PANELS, BP>(a, cols, row, beg, end, lane, acc); \
  beg = nbeg;                                                  \
  end = nend;
  MT_INDEX_PLANE(0)
  MT_INDEX_PLANE(1)
  MT_INDEX_PLANE(2)
  MT_INDEX_PLANE(3)
  MT_INDEX_PLANE(4)
  MT_INDEX_PLANE(5)
#undef MT_INDEX_PLANE
#pragma unroll
  for (int b = 0; b < B; ++b)
#pragma unroll
    for (int cc = 0; cc < 3; ++cc)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[b][cc] += __shfl_xor_sync(0xffffffffu, acc[b][cc], o);
  double s[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int b = 0; b < B; ++b)
    if (lane == b) { s[0] = acc[b][0]; s[1] = acc[b][1]; s[2] = acc[b][2]; }
  if (lane < B) {
    const double hd[3] = {-s[0], -s[1], -s[2]};
    row_epilogue(e, row, lane, hd);
  }
}

template <typename T, int B>
int launch_index_B(mt_ctx* ctx, const SparseArgs& a0, const uint16_t* cols, const EpiArgs& e) {
  constexpr int BP = B <= 2 ? 0 : B <= 4 ? 4 : 8;
  SparseArgs a = a0;
  if constexpr (BP != 0) {
    // batches of 3..8: the staged M re-laid out with the states innermost, once per evaluation
    const size_t need = (size_t)3 * a.npad * BP * sizeof(T);
    int rc = mt_ensure_ws(ctx, &ctx->Mq, &ctx->Mq_bytes, need);
    if (rc) return rc;
    const int64_t tot = 3 * a.npad;
    interleave_stage_kernel<T, BP><<<(unsigned)((tot + 255) / 256), 256, 0, ctx->stream>>>((const T*)a.Mst, a.npad, (T*)ctx->Mq);
    ctx->launches++;
    MT_CUDA_OK(ctx, cudaGetLastError());
    a.Mst = ctx->Mq;
  }
  if (a.npanels > 1)
    demag_index_kernel<T, B, true, BP><<<(unsigned)((a.n_rows + 7) / 8), 256, 0, ctx->stream>>>(a, cols, e);
  else
    demag_index_kernel<T, B, false, BP><<<(unsigned)((a.n_rows + 7) / 8), 256, 0, ctx->stream>>>(a, cols, e);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

template <typename T>
int launch_index(mt_ctx* ctx, const SparseArgs& a, const uint16_t* cols, const EpiArgs& e) {
  switch (e.batch) {
    case 1: return launch_index_B<T, 1>(ctx, a, cols, e);
    case 2: return launch_index_B<T, 2>(ctx, a, cols, e);
    case 3: return launch_index_B<T, 3>(ctx, a, cols, e);
    case 4: return launch_index_B<T, 4>(ctx, a, cols, e);
    case 5: return launch_index_B<T, 5>(ctx, a, cols, e);
    case 6: return launch_index_B<T, 6>(ctx, a, cols, e);
    case 7: return launch_index_B<T, 7>(ctx, a, cols, e);
    case 8: return launch_index_B<T, 8>(ctx, a, cols, e);
  }
  return mt_fail(ctx, MT_ERR_INVALID_ARG, "batch must be in [1, %d]", MT_MAX_BATCH);
}

}  // namespace

int mt_launch_select_hist(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                          unsigned long long prefix, int prefix_shift, int shift, int width,
                          unsigned long long* hist) {
  // enough blocks that none sees 2^30 elements (32-bit shared counters with multiplicity 2)
  int64_t blocks = (int64_t)ctx->num_sms * 4;
  const int64_t need = (6 * n_rows * n + (1LL << 30) - 1) >> 30;
  if (blocks < need) blocks = need;
  const unsigned grid = (unsigned)min(blocks, 6 * n_rows);
  if (width > kDigitBits) {  // wide digit: global histogram, prefix-matching elements only
    if (dtype == MT_F32)
      select_hist_wide_kernel<float><<<grid, 512, 0, ctx->stream>>>((const float*)N, n, n_rows, ld, (uint32_t)prefix,
                                                                    prefix_shift, shift, width, hist);
    else
      select_hist_wide_kernel<double><<<grid, 512, 0, ctx->stream>>>((const double*)N, n, n_rows, ld, prefix,
                                                                     prefix_shift, shift, width, hist);
    ctx->launches++;
    MT_CUDA_OK(ctx, cudaGetLastError());
    return MT_OK;
  }
  if (dtype == MT_F32)
    select_hist_kernel<float><<<grid, 512, 0, ctx->stream>>>((const float*)N, n, n_rows, ld, (uint32_t)prefix,
                                                             prefix_shift, shift, width, hist);
  else
    select_hist_kernel<double><<<grid, 512, 0, ctx->stream>>>((const double*)N, n, n_rows, ld, prefix, prefix_shift,
                                                              shift, width, hist);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_select_find(mt_ctx* ctx, const unsigned long long* hist, int nbins, unsigned long long k, int first_pass,
                          double fraction, unsigned long long* out4) {
  select_find_kernel<<<1, 1024, 0, ctx->stream>>>(hist, nbins, k, first_pass, fraction, out4);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_sparse_count(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                           int64_t row0, int64_t n_total, int64_t* counts) {
  const unsigned grid = (unsigned)((6 * n_rows + 7) / 8);
  if (dtype == MT_F32)
    sparse_count_kernel<float><<<grid, 256, 0, ctx->stream>>>((const float*)N, n, n_rows, ld, (float)tau, row0,
                                                              n_total, counts);
  else
    sparse_count_kernel<double><<<grid, 256, 0, ctx->stream>>>((const double*)N, n, n_rows, ld, tau, row0, n_total,
                                                               counts);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_sparse_scan(mt_ctx* ctx, int64_t* row_ptr, int64_t n_total) {
  scan_kernel<<<1, 1024, 0, ctx->stream>>>(row_ptr, 6 * n_total);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_sparse_fill(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                          int64_t row0, int64_t n_total, const int64_t* row_ptr, int64_t nw, uint32_t* mask,
                          void* vals, uint16_t* cols16, int64_t* panel_ptr) {
  const unsigned grid = (unsigned)((6 * n_rows + 7) / 8);
  const int npanels = (int)((n + 65535) >> 16);
  if (dtype == MT_F32)
    sparse_fill_kernel<float><<<grid, 256, 0, ctx->stream>>>((const float*)N, n, n_rows, ld, (float)tau, row0, n_total,
                                                             row_ptr, nw, mask, (float*)vals, cols16, panel_ptr, npanels);
  else
    sparse_fill_kernel<double><<<grid, 256, 0, ctx->stream>>>((const double*)N, n, n_rows, ld, tau, row0, n_total,
                                                              row_ptr, nw, mask, (double*)vals, cols16, panel_ptr,
                                                              npanels);
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_sparse_index(mt_ctx* ctx, const mt_sparse_tensor* s, uint16_t* cols16, int64_t* panel_ptr) {
  sparse_index_kernel<<<(unsigned)((6 * s->n_rows + 7) / 8), 256, 0, ctx->stream>>>(
      s->mask, s->row_ptr, s->n_rows, s->nw, cols16, panel_ptr, (int)((s->n + 65535) >> 16));
  ctx->launches++;
  MT_CUDA_OK(ctx, cudaGetLastError());
  return MT_OK;
}

int mt_launch_demag_sparse(mt_ctx* ctx, const mt_sparse_tensor* s, const void* Mst, int64_t npad, const EpiArgs& e) {
  SparseArgs a;
  a.n = s->n;
  a.n_rows = s->n_rows;
  a.nw = s->nw;
  a.npad = npad;
  a.row_ptr = s->row_ptr;
  a.mask = s->mask;
  a.vals = s->vals;
  a.Mst = Mst;
  a.panel_ptr = s->panel_ptr;
  a.npanels = (int)((s->n + 65535) >> 16);
  const bool prof = ctx->prof_on && ctx->prof_ev && ctx->prof_count < MT_PROF_CAP;
  if (prof) MT_CUDA_OK(ctx, cudaEventRecord(ctx->prof_ev[2 * ctx->prof_count], ctx->stream));
  int rc;
  if (s->cols16)
    rc = s->dtype == MT_F32 ? launch_index<float>(ctx, a, s->cols16, e) : launch_index<double>(ctx, a, s->cols16, e);
  else
    rc = s->dtype == MT_F32 ? launch_bitmap<float>(ctx, a, e) : launch_bitmap<double>(ctx, a, e);
  if (prof) {
    MT_CUDA_OK(ctx, cudaEventRecord(ctx->prof_ev[2 * ctx->prof_count + 1], ctx->stream));
    ctx->prof_count++;
  }
  return rc;
}
