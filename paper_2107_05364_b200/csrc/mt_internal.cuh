// mt_internal.cuh — shared declarations of libmagtile's translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "mt.h"

#define MT_MAX_BATCH 8
#define MT_MAX_STAGES 7
#define MT_COL_CHUNK 256 /* staged-M padding granule (elements) */

struct mt_ctx {
  int device;
  cudaStream_t stream;
  cudaStream_t cap_stream;  // private stream for CUDA-graph capture
  int num_sms;
  int variant;  // 0 auto, 1 LDG, 2 TMA, 3 TMA with the packed-FFMA2 kernel for batches of 5..8
  int assembly_mode;  // 0 closed form everywhere (the paper's method), 1 far-field-stable (F2)
  int64_t launches;
  char err[512];
  // grow-only workspaces
  void* Mst[2];
  size_t Mst_bytes;
  double* partial;
  size_t partial_bytes;
  void* Mq;  // staged M re-laid out for the tensor-core kernel's B fragments (demag_tma.cu)
  size_t Mq_bytes;
  double* rk;  // integrator stages + scratch states
  size_t rk_bytes;
  void* sym_ws;   // rowpart + colpart of the symmetric-half field kernel (F3)
  size_t sym_ws_bytes;
  double* edens;  // [B][4][n] energy densities (mt_energy)
  size_t edens_bytes;
  unsigned long long* dscal;  // device scalars: [0] err bits, [1] torque bits
  unsigned long long* hscal;  // pinned host mirror
  double* stage_io;           // device staging for the *_host entry points
  size_t stage_io_bytes;
  double* pinned_io;
  size_t pinned_io_bytes;
  // TMA descriptor cache (variant 2)
  const void* tm_base;
  int tm_dtype;
  int64_t tm_n, tm_rows, tm_ld;
  alignas(64) unsigned char tm_desc[128];
  int tm_valid;
  // per-kernel timing of the demag field kernel (mt_profile_begin / mt_profile_end)
  int prof_on;
  int prof_count;
  cudaEvent_t* prof_ev;  // MT_PROF_CAP pairs, created lazily
};
#define MT_PROF_CAP 1024

int mt_fail(mt_ctx* ctx, int code, const char* fmt, ...);
#define MT_CUDA_OK(ctx, expr)                                                                  \
  do {                                                                                         \
    cudaError_t _e = (expr);                                                                   \
    if (_e != cudaSuccess)                                                                     \
      return mt_fail((ctx), MT_ERR_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), \
                     __FILE__, __LINE__);                                                      \
  } while (0)

// ---- fused epilogue descriptor (A5, A6, Runge-Kutta stage combine, DP45 error) -----------------
struct EpiArgs {
  int mode;        // 0: store H_d only; 1: effective field + LL right-hand side (+ optional stages)
  int batch;
  int64_t n;       // tiles per state (stride of SoA vectors)
  int64_t n_rows;  // rows of the launch (== n for mode 1 unless the problem is row-sharded)
  int64_t row0;    // mode 1: global index of the launch's first row (row-sharded problems; else 0)
  double* Hd;      // mode 0 output [B][3][n_rows]
  // mode 1 inputs
  const double* y;  // state the right-hand side is evaluated at [B][3][n]
  const double* Ms;
  const int32_t* nbr;
  double inv_d2[3];
  const double* c_ex;
  double c_ex_s;
  const double* c_an;
  double c_an_s;
  const double* easy;
  double easy_c[3];
  const double* H_a;
  double H_a_c[3];
  double gamma, alpha;
  double* k_out;     // dm/dt [B][3][n]
  double* heff_out;  // optional
  double* e_dens;    // optional [B][4][n]: per-tile energy of the demag, exchange, anisotropy, Zeeman terms
  const double* vol; // tile volumes for e_dens (NULL: 1)
  unsigned long long* torque_bits;  // optional: atomicMax of |y x H_eff| (bits of a non-negative double)
  // stage combine: y_out = base + h * sum_j coef[j] * kptr[j]; optional renormalisation; optional
  // staging of Ms*y_out in the tensor's dtype for the next field evaluation
  int do_comb;
  int ncomb;
  const double* kptr[MT_MAX_STAGES];
  double coef[MT_MAX_STAGES];
  const double* base;
  double h;
  double* y_out;
  int64_t y_ld;    // y_out is [B][3][y_ld] holding rows y_row0 .. (0, 0: [B][3][n] from row 0): a rank's
  int64_t y_row0;  // block of the all-gather buffer when the problem is row-sharded
  int renorm;
  void* M_out;
  int M_dtype;
  int64_t npad;
  // DP45 error estimate: e = h * sum_j ecoef[j] * eptr[j]; err = |e| / (atol + rtol max(|ebase|, |y|))
  int nerr;
  const double* eptr[MT_MAX_STAGES];
  double ecoef[MT_MAX_STAGES];
  const double* ebase;
  double atol, rtol;
  unsigned long long* err_bits;
};

// launchers (demag.cu)
int mt_launch_stage_M(mt_ctx* ctx, int dtype, const double* Ms, const double* m, int batch, int64_t n,
                      int64_t npad, void* M_out);
int mt_launch_demag(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                    const void* Mst, int64_t npad, const EpiArgs& epi);
int mt_launch_local_only(mt_ctx* ctx, const EpiArgs& epi);  // N == NULL: H_d = 0
int mt_launch_combine(mt_ctx* ctx, const EpiArgs& epi);     // stage combine without a field evaluation
// row-sharded problems: blocks [world][B][3][pad] of the gathered stage state -> full state y[B][3][n]
// and (M_out non-NULL) the staged Ms*y in the tensor's dtype
int mt_launch_unpack(mt_ctx* ctx, const double* pack, int world, int64_t pad, int batch, int64_t n, int64_t npad,
                     const double* Ms, double* y, void* M_out, int M_dtype);
int mt_launch_mean(mt_ctx* ctx, const double* m, const double* vol, int batch, int64_t n, double t,
                   double* sample_row);
int mt_ensure_ws(mt_ctx* ctx, void** p, size_t* cur, size_t need);
// E_out[b][5] = fixed-order sums over tiles of e_dens[b][0..3][n], then their total
int mt_launch_energy_reduce(mt_ctx* ctx, const double* e_dens, int batch, int64_t n, double* E_out);

// launchers (assemble.cu)
int mt_launch_assemble(mt_ctx* ctx, const mt_tiles* t, int dtype, int64_t r0, int64_t r1, void* out,
                       int64_t ld, int32_t* status);
// TMA variant (demag_tma.cu)
int mt_launch_demag_tma(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                        const void* Mst, int64_t npad, const EpiArgs& epi);
// thresholded tensor (sparse.cu)
int mt_launch_select_hist(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                          unsigned long long prefix, int prefix_shift, int shift, int width,
                          unsigned long long* hist);
int mt_launch_sparse_count(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                           int64_t row0, int64_t n_total, int64_t* counts);
int mt_launch_sparse_scan(mt_ctx* ctx, int64_t* row_ptr, int64_t n_total);
int mt_launch_sparse_fill(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                          int64_t row0, int64_t n_total, const int64_t* row_ptr, int64_t nw, uint32_t* mask,
                          void* vals, uint16_t* cols16, int64_t* panel_ptr);
int mt_launch_sparse_index(mt_ctx* ctx, const mt_sparse_tensor* s, uint16_t* cols16, int64_t* panel_ptr);
int mt_launch_demag_sparse(mt_ctx* ctx, const mt_sparse_tensor* s, const void* Mst, int64_t npad, const EpiArgs& epi);
// pair-symmetric half (assemble.cu, sym.cu)
int mt_launch_assemble_sym(mt_ctx* ctx, const mt_tiles* t, int dtype, void* out, int32_t* status);
int mt_launch_demag_sym(mt_ctx* ctx, const mt_sym_tensor* S, const void* Mst, int64_t npad, const EpiArgs& epi);
