// mt_internal.cuh — shared declarations of libmagtile's translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "mt.h"

#define MT_MAX_BATCH 8
#define MT_MAX_STAGES 7
#define MT_COL_CHUNK 256 /* staged-M padding granule (elements) */

struct DpState;
struct mt_ctx {
  int device;
  cudaStream_t stream;
  cudaStream_t cap_stream;  // private stream for CUDA-graph capture
  int num_sms;
  int step_control;  // DP45 controller: 0 auto (device for small problems), 1 host, 2 device
  int resident_mode; // RK4 with the tensor resident in shared memory (resident.cu): 0 auto (when it fits), 1 never, 2 required
  DpState* dp_dev;   // device copy of the controller state (lazily allocated)
  DpState* dp_host;  // pinned mirror
  int variant;  // 0 auto, 1 LDG, 2 TMA, 3 TMA with the packed-FFMA2 kernel for batches of 5..8
  int assembly_mode;  // 0 closed form everywhere (the paper's method), 1 far-field-stable (F2)
  int64_t launches;
  char err[512];
  // grow-only workspaces
  void* Mst[2];
  size_t Mst_bytes;
  double* partial;
  size_t partial_bytes;
  int* split_count;  // demag_tma.cu: chunks summed so far per split row group (zero between launches)
  size_t split_count_bytes;
  void* Mq;  // staged M re-laid out for the tensor-core kernel's B fragments (demag_tma.cu)
  size_t Mq_bytes;
  double* rk;  // integrator stages + scratch states
  size_t rk_bytes;
  unsigned long long* sel_hist;  // MT_SELECT_HIST_WORDS counters of mt_threshold_value / mt_sparse_stream_count (lazy)
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
  // TMA descriptor cache (demag_tma.cu): a tensor map depends only on the base address and the
  // geometry, so it is encoded once per (tensor, box shape) and ctx instead of once per launch
  struct TmEntry {
    const void* base;
    int dtype, rank, swizzle, valid;
    uint64_t dims[3], strides[2];
    uint32_t box[3];
    alignas(64) unsigned char map[128];
  } tm_cache[8];
  int tm_next;
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
  const double* h_dev;    // non-NULL: the step h is read from the device (device-resident DP45 controller)
  const int* active_dev;  // non-NULL and *active_dev == 0: the launch's epilogue / combine does nothing
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

// ---- device-resident DP45 step controller (api.cu, demag.cu) --------------------------------------
// The state of the controller of A9 when it runs on the device: one attempted step is then a fixed
// sequence of launches (replayed from a CUDA graph) with no host round trip; the host reads this
// struct every few attempted steps.  Same rules as the host controller (Q11/Q11b).
struct DpState {
  double t, dt, h, t_target, t_end, t0, sample_dt, sample_t;
  double rtol, atol, torque_tol, max_torque, dt_last;
  unsigned long long err_bits, tq_bits;
  long long accepted, rejected, rhs_calls, n_samples, sample_cap, next_sample, max_steps, sample_row;
  int status;       // MT_DP_* below
  int active;       // this attempt integrates (stage kernels do their work)
  int accept;       // this attempt was accepted (commit copies the candidate and k7)
  int sample_flag;  // a sample row is due at the end of this attempt
  int clipped, hit_sample, has_samples, pad_;
};
#define MT_DP_RUN 0
#define MT_DP_T_END 1
#define MT_DP_TORQUE 2
#define MT_DP_UNDERFLOW 3
#define MT_DP_NONFINITE 4
#define MT_DP_MAX_STEPS 5
int mt_launch_dp_begin(mt_ctx* ctx, DpState* st);
int mt_launch_dp_decide(mt_ctx* ctx, DpState* st);
int mt_launch_dp_commit(mt_ctx* ctx, const DpState* st, double* m, const double* mc, double* k1, const double* k7,
                        int64_t count);
int mt_launch_mean_cond(mt_ctx* ctx, const DpState* st, const double* m, const double* vol, int batch, int64_t n,
                        double* samples, int64_t stride);

// launchers (demag.cu)
int mt_launch_stage_M(mt_ctx* ctx, int dtype, const double* Ms, const double* m, int batch, int64_t n,
                      int64_t npad, void* M_out);
// Ms_fuse / y_fuse non-NULL (only after mt_demag_can_fuse said yes): Mst is not read, the kernel forms Ms*y itself
int mt_launch_demag(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                    const void* Mst, int64_t npad, const EpiArgs& epi, const double* Ms_fuse = nullptr,
                    const double* y_fuse = nullptr);
bool mt_demag_can_fuse(mt_ctx* ctx, int dtype, int64_t n, int64_t n_rows, const double* Ms, const double* y);
bool mt_demag_tma_takes(mt_ctx* ctx, int dtype, int64_t n, int64_t n_rows);  // demag_tma.cu: the default choice by shape
int mt_launch_local_only(mt_ctx* ctx, const EpiArgs& epi);  // N == NULL: H_d = 0
// resident.cu: a chunk of RK4 steps in one cooperative launch, the dense tensor held in shared memory
#define MT_RES_NONE 0
#define MT_RES_SMEM 1 /* tensor resident in shared memory */
#define MT_RES_L2 2   /* tensor read from L2 at every stage by the same persistent kernel */
int mt_resident_fits(mt_ctx* ctx, int dtype, int64_t n, int64_t ld, int batch, int method);
int mt_launch_rk4_resident(mt_ctx* ctx, int mode, const void* N, int dtype, int64_t n, int64_t ld, const EpiArgs& prob,
                           double* m, double* ya, double* yb, double dt, int renorm,
                           unsigned long long* tq_slots, unsigned int* bar, int64_t count);
int mt_launch_dp45_resident(mt_ctx* ctx, int mode, const void* N, int dtype, int64_t n, int64_t ld, const EpiArgs& prob,
                            DpState* S, double* m, double* k1, double* ya, double* yb, int renorm,
                            double* samples, int64_t stride, const double* vol, unsigned long long* words,
                            unsigned int* bar, int attempts);
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
int mt_launch_select_find(mt_ctx* ctx, const unsigned long long* hist, int nbins, unsigned long long k, int first_pass,
                          double fraction, unsigned long long* out4);
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
