// api.cu — the extern "C" boundary declared in include/mt.h: argument validation, workspace
// management and the host-side drivers of the integrators (A8 RK4 with CUDA graphs, A9 DP45).
#include <math.h>
#include <string.h>

#include <new>

#include "mt_internal.cuh"
#include "sym_layout.cuh"

namespace {

inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
inline size_t elem_size(int dtype) { return dtype == MT_F32 ? 4 : 8; }

int check_tensor_args(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld) {
  if (dtype != MT_F32 && dtype != MT_F64) return mt_fail(ctx, MT_ERR_INVALID_ARG, "unknown dtype %d", dtype);
  if (n <= 0 || n_rows <= 0) return mt_fail(ctx, MT_ERR_INVALID_ARG, "n and n_rows must be positive");
  if (ld < n) return mt_fail(ctx, MT_ERR_INVALID_ARG, "ld (%lld) < n (%lld)", (long long)ld, (long long)n);
  const int64_t vec = dtype == MT_F32 ? 4 : 2;
  if (ld % vec) return mt_fail(ctx, MT_ERR_INVALID_ARG, "ld must be a multiple of %lld elements", (long long)vec);
  if (!N || ((uintptr_t)N & 15)) return mt_fail(ctx, MT_ERR_INVALID_ARG, "tensor pointer null or not 16-byte aligned");
  return MT_OK;
}

// The two staged-M buffers always have room for MT_MAX_BATCH states (the batched kernels' TMA boxes
// may cover rows beyond 3*batch; what they read there is never used) and start out zeroed.
int ensure_Mst(mt_ctx* ctx, int dtype, int batch, int64_t npad) {
  (void)batch;
  const size_t need = (size_t)MT_MAX_BATCH * 3 * npad * elem_size(dtype);
  if (ctx->Mst_bytes >= need && ctx->Mst[0]) return MT_OK;
  for (int k = 0; k < 2; ++k) {
    size_t cur = ctx->Mst[k] ? ctx->Mst_bytes : 0;
    int rc = mt_ensure_ws(ctx, &ctx->Mst[k], &cur, need);
    if (rc) return rc;
    MT_CUDA_OK(ctx, cudaMemsetAsync(ctx->Mst[k], 0, need, ctx->stream));
  }
  ctx->Mst_bytes = need;
  return MT_OK;
}

inline bool has_demag(const mt_problem* p) { return p->N != nullptr || p->N_sparse != nullptr || p->N_sym != nullptr; }
inline int demag_dtype(const mt_problem* p) {
  return p->N_sparse ? p->N_sparse->dtype : p->N_sym ? p->N_sym->dtype : p->dtype;
}

int check_sym(mt_ctx* ctx, const mt_sym_tensor* s) {
  if (!s) return mt_fail(ctx, MT_ERR_INVALID_ARG, "symmetric tensor is NULL");
  if (s->dtype != MT_F32 && s->dtype != MT_F64) return mt_fail(ctx, MT_ERR_INVALID_ARG, "unknown dtype %d", s->dtype);
  if (s->n <= 0) return mt_fail(ctx, MT_ERR_INVALID_ARG, "n must be positive");
  if (!s->data || ((uintptr_t)s->data & 15)) return mt_fail(ctx, MT_ERR_INVALID_ARG, "data null or not 16-byte aligned");
  return MT_OK;
}

int check_sparse(mt_ctx* ctx, const mt_sparse_tensor* s) {
  if (!s) return mt_fail(ctx, MT_ERR_INVALID_ARG, "sparse tensor is NULL");
  if (s->dtype != MT_F32 && s->dtype != MT_F64) return mt_fail(ctx, MT_ERR_INVALID_ARG, "unknown dtype %d", s->dtype);
  if (s->n <= 0 || s->n_rows <= 0) return mt_fail(ctx, MT_ERR_INVALID_ARG, "n and n_rows must be positive");
  if (s->nw != mt_sparse_mask_words(s->n)) return mt_fail(ctx, MT_ERR_INVALID_ARG, "nw must be mt_sparse_mask_words(n)");
  if (!s->row_ptr || (!s->mask && !s->cols16))
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "row_ptr and one of mask / cols16 must be non-NULL");
  if (s->cols16 && s->n > 65536 && !s->panel_ptr)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "cols16 with n > 65536 needs panel_ptr");
  return MT_OK;
}

// rows [r0, r1) of the right-hand side this rank evaluates: all of them, or the rank's band of a
// row-sharded problem (mt.h section 8(e): begin(g) = g n / world)
inline int64_t band_begin(const mt_problem* p) {
  return p->shard ? (int64_t)(((unsigned __int128)p->shard->rank * (unsigned __int128)p->n) / (unsigned)p->shard->world) : 0;
}
inline int64_t band_end(const mt_problem* p) {
  return p->shard ? (int64_t)(((unsigned __int128)(p->shard->rank + 1) * (unsigned __int128)p->n) / (unsigned)p->shard->world) : p->n;
}

void fill_problem(EpiArgs& e, const mt_problem* p, int batch) {
  memset(&e, 0, sizeof(e));
  e.mode = 1;
  e.batch = batch;
  e.n = p->n;
  e.n_rows = band_end(p) - band_begin(p);
  e.row0 = band_begin(p);
  e.Ms = p->Ms;
  e.nbr = p->nbr;
  for (int a = 0; a < 3; ++a) {
    e.inv_d2[a] = p->inv_d2[a];
    e.easy_c[a] = p->easy_const[a];
    e.H_a_c[a] = p->H_a_const[a];
  }
  e.c_ex = p->c_ex;
  e.c_ex_s = p->c_ex_scalar;
  e.c_an = p->c_an;
  e.c_an_s = p->c_an_scalar;
  e.easy = p->easy;
  e.H_a = p->H_a;
  e.gamma = p->gamma;
  e.alpha = p->alpha_ll;
  e.M_dtype = demag_dtype(p);
}

int check_problem(mt_ctx* ctx, const mt_problem* p, int batch) {
  if (!p) return mt_fail(ctx, MT_ERR_INVALID_ARG, "problem is NULL");
  if (p->n <= 0 || !p->Ms) return mt_fail(ctx, MT_ERR_INVALID_ARG, "problem needs n > 0 and Ms");
  if (batch < 1 || batch > MT_MAX_BATCH) return mt_fail(ctx, MT_ERR_INVALID_ARG, "batch must be in [1, %d]", MT_MAX_BATCH);
  if (const mt_shard* sh = p->shard) {
    if (sh->world < 1 || sh->rank < 0 || sh->rank >= sh->world)
      return mt_fail(ctx, MT_ERR_INVALID_ARG, "shard: need 0 <= rank < world");
    if (sh->world > p->n) return mt_fail(ctx, MT_ERR_INVALID_ARG, "shard: more ranks than tiles");
    if (!sh->pack || !sh->scal || !sh->exchange)
      return mt_fail(ctx, MT_ERR_INVALID_ARG, "shard: pack, scal and exchange must be non-NULL");
    if (sh->slice_pad < (p->n + sh->world - 1) / sh->world)
      return mt_fail(ctx, MT_ERR_INVALID_ARG, "shard: slice_pad is shorter than the longest band");
    if (p->N_sym) return mt_fail(ctx, MT_ERR_INVALID_ARG, "the pair-symmetric half cannot be row-sharded");
  }
  const int64_t rows = band_end(p) - band_begin(p);
  if (p->N_sparse) {
    int rc = check_sparse(ctx, p->N_sparse);
    if (rc) return rc;
    if (p->N_sparse->n != p->n || p->N_sparse->n_rows != rows)
      return mt_fail(ctx, MT_ERR_INVALID_ARG, "sparse tensor must be n x n (sharded: the rank's band x n)");
    return MT_OK;
  }
  if (p->N_sym) {
    int rc = check_sym(ctx, p->N_sym);
    if (rc) return rc;
    if (p->N_sym->n != p->n) return mt_fail(ctx, MT_ERR_INVALID_ARG, "symmetric tensor must have n tiles");
    return MT_OK;
  }
  if (p->N) return check_tensor_args(ctx, p->N, p->dtype, p->n, rows, p->ld);
  return MT_OK;
}

// one evaluation of the fused right-hand side: field of the staged M (ctx->Mst[src]) + epilogue
int eval_rhs(mt_ctx* ctx, const mt_problem* p, int64_t npad, int src, const EpiArgs& e) {
  if (p->N_sparse) return mt_launch_demag_sparse(ctx, p->N_sparse, ctx->Mst[src], npad, e);
  if (p->N_sym) return mt_launch_demag_sym(ctx, p->N_sym, ctx->Mst[src], npad, e);
  if (p->N) return mt_launch_demag(ctx, p->N, p->dtype, p->n, e.n_rows, p->ld, ctx->Mst[src], npad, e);
  return mt_launch_local_only(ctx, e);
}

const double DP_A[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5, 0, 0, 0, 0, 0},
    {3.0 / 40, 9.0 / 40, 0, 0, 0, 0},
    {44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0},
    {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0},
    {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0},
    {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}};
const double DP_E[7] = {35.0 / 384 - 5179.0 / 57600,       0.0,
                        500.0 / 1113 - 7571.0 / 16695,     125.0 / 192 - 393.0 / 640,
                        -2187.0 / 6784 + 92097.0 / 339200, 11.0 / 84 - 187.0 / 2100,
                        -1.0 / 40};

inline double bits_to_double(unsigned long long b) {
  double d;
  memcpy(&d, &b, 8);
  return d;
}

}  // namespace

extern "C" {

const char* mt_version(void) { return "magtile-b200 0.1 (sm_100a)"; }

int mt_create(mt_ctx** out, int device, void* cuda_stream) {
  if (!out) return MT_ERR_INVALID_ARG;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return MT_ERR_CUDA;
  if (cudaSetDevice(device) != cudaSuccess) return MT_ERR_CUDA;
  mt_ctx* c = new (std::nothrow) mt_ctx;
  if (!c) return MT_ERR_CUDA;
  memset(c, 0, sizeof(*c));
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) {
    delete c;
    return MT_ERR_CUDA;
  }
  c->num_sms = prop.multiProcessorCount;
  // device scalars: [0] err bits, [1] torque bits, [2..5] the selection's bin search, [6] the resident RK4
  // kernel's grid-barrier counter, [8 ..] 256 per-step
  // torque words of an RK4 chunk; the pinned mirror holds the two words, the search result or the chunk's torques
  if (cudaMalloc((void**)&c->dscal, (8 + 256) * sizeof(unsigned long long)) != cudaSuccess ||
      cudaMallocHost((void**)&c->hscal, 2048 * sizeof(unsigned long long)) != cudaSuccess) {
    cudaFree(c->dscal);
    delete c;
    return MT_ERR_CUDA;
  }
  *out = c;
  return MT_OK;
}

int mt_destroy(mt_ctx* c) {
  if (!c) return MT_OK;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  cudaFree(c->Mst[0]);
  cudaFree(c->Mst[1]);
  cudaFree(c->partial);
  cudaFree(c->split_count);
  cudaFree(c->Mq);
  cudaFree(c->rk);
  cudaFree(c->edens);
  cudaFree(c->sym_ws);
  cudaFree(c->dscal);
  cudaFree(c->stage_io);
  cudaFree(c->dp_dev);
  cudaFree(c->sel_hist);
  cudaFreeHost(c->dp_host);
  cudaFreeHost(c->hscal);
  cudaFreeHost(c->pinned_io);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  if (c->prof_ev) {
    for (int k = 0; k < 2 * MT_PROF_CAP; ++k) cudaEventDestroy(c->prof_ev[k]);
    delete[] c->prof_ev;
  }
  delete c;
  return MT_OK;
}

const char* mt_last_error(const mt_ctx* c) { return c ? c->err : "mt_ctx is NULL"; }

int64_t mt_launch_count(const mt_ctx* c) { return c ? c->launches : 0; }

int mt_profile_begin(mt_ctx* c) {
  if (!c) return MT_ERR_INVALID_ARG;
  MT_CUDA_OK(c, cudaSetDevice(c->device));
  if (!c->prof_ev) {
    c->prof_ev = new (std::nothrow) cudaEvent_t[2 * MT_PROF_CAP];
    if (!c->prof_ev) return mt_fail(c, MT_ERR_CUDA, "out of host memory");
    for (int k = 0; k < 2 * MT_PROF_CAP; ++k) MT_CUDA_OK(c, cudaEventCreate(&c->prof_ev[k]));
  }
  c->prof_count = 0;
  c->prof_on = 1;
  return MT_OK;
}

int mt_profile_end(mt_ctx* c, double* total_ms, int64_t* launches) {
  if (!c || !total_ms || !launches) return MT_ERR_INVALID_ARG;
  *total_ms = 0.0;
  *launches = 0;
  if (!c->prof_on) return mt_fail(c, MT_ERR_INVALID_ARG, "mt_profile_end without mt_profile_begin");
  c->prof_on = 0;
  MT_CUDA_OK(c, cudaStreamSynchronize(c->stream));
  for (int k = 0; k < c->prof_count; ++k) {
    float ms = 0.f;
    MT_CUDA_OK(c, cudaEventElapsedTime(&ms, c->prof_ev[2 * k], c->prof_ev[2 * k + 1]));
    *total_ms += ms;
  }
  *launches = c->prof_count;
  return MT_OK;
}

int mt_set_demag_variant(mt_ctx* c, int variant) {
  if (!c || variant < 0 || variant > 3) return MT_ERR_INVALID_ARG;
  c->variant = variant;
  return MT_OK;
}

int mt_set_resident_mode(mt_ctx* c, int mode) {
  if (!c || mode < 0 || mode > 2) return MT_ERR_INVALID_ARG;
  c->resident_mode = mode;
  return MT_OK;
}

int mt_set_step_control(mt_ctx* c, int mode) {
  if (!c || mode < 0 || mode > 2) return MT_ERR_INVALID_ARG;
  c->step_control = mode;
  return MT_OK;
}

int mt_set_assembly_mode(mt_ctx* c, int mode) {
  if (!c || mode < 0 || mode > 1) return MT_ERR_INVALID_ARG;
  c->assembly_mode = mode;
  return MT_OK;
}

int mt_assemble_tensor(mt_ctx* ctx, const mt_tiles* t, int dtype, int64_t row_begin, int64_t row_end,
                       void* out, int64_t ld, int32_t* status_flag) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!t || !t->type || !t->center || !t->size) return mt_fail(ctx, MT_ERR_INVALID_ARG, "tiles incomplete");
  if (row_begin < 0 || row_end < row_begin || row_end > t->n)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "row band [%lld, %lld) outside [0, %lld)", (long long)row_begin,
                   (long long)row_end, (long long)t->n);
  if (row_end == row_begin) return MT_OK;
  int rc = check_tensor_args(ctx, out, dtype, t->n, row_end - row_begin, ld);
  if (rc) return rc;
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  return mt_launch_assemble(ctx, t, dtype, row_begin, row_end, out, ld, status_flag);
}

int mt_check_status(mt_ctx* ctx, const int32_t* status_flag) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!status_flag) return mt_fail(ctx, MT_ERR_INVALID_ARG, "status_flag must be non-NULL");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  MT_CUDA_OK(ctx, cudaMemcpyAsync(ctx->hscal, status_flag, sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
  MT_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  const int32_t f = *(const int32_t*)ctx->hscal;
  if (f & 1) return mt_fail(ctx, MT_ERR_SINGULAR_GEOMETRY, "assembly produced a non-finite block: a target centre lies on a source face or edge");
  if (f & 2) return mt_fail(ctx, MT_ERR_INVALID_ARG, "the pair-symmetric half needs a mesh of congruent axis-aligned cuboids");
  return MT_OK;
}

int mt_demag_field(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                   const double* Ms, const double* m, int batch, double* Hd) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_tensor_args(ctx, N, dtype, n, n_rows, ld);
  if (rc) return rc;
  if (!Ms || !m || !Hd) return mt_fail(ctx, MT_ERR_INVALID_ARG, "Ms, m and Hd must be non-NULL");
  if (batch < 1 || batch > MT_MAX_BATCH) return mt_fail(ctx, MT_ERR_INVALID_ARG, "batch must be in [1, %d]", MT_MAX_BATCH);
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int64_t npad = round_up(n, MT_COL_CHUNK);
  EpiArgs e;
  memset(&e, 0, sizeof(e));
  e.mode = 0;
  e.batch = batch;
  e.n = n;
  e.n_rows = n_rows;
  e.Hd = Hd;
  // small problems: one launch, the field kernel forms Ms*m itself (same bits as the staged M)
  if (mt_demag_can_fuse(ctx, dtype, n, n_rows, Ms, m))
    return mt_launch_demag(ctx, N, dtype, n, n_rows, ld, nullptr, npad, e, Ms, m);
  rc = ensure_Mst(ctx, dtype, batch, npad);
  if (rc) return rc;
  rc = mt_launch_stage_M(ctx, dtype, Ms, m, batch, n, npad, ctx->Mst[0]);
  if (rc) return rc;
  return mt_launch_demag(ctx, N, dtype, n, n_rows, ld, ctx->Mst[0], npad, e);
}

int mt_demag_field_host(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                        const double* Ms, const double* m_host, int batch, double* Hd_host) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!m_host || !Hd_host) return mt_fail(ctx, MT_ERR_INVALID_ARG, "host vectors must be non-NULL");
  if (batch < 1 || batch > MT_MAX_BATCH || n <= 0 || n_rows <= 0)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "bad batch / n / n_rows");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const size_t in_b = (size_t)batch * 3 * n * sizeof(double), out_b = (size_t)batch * 3 * n_rows * sizeof(double);
  int rc = mt_ensure_ws(ctx, (void**)&ctx->stage_io, &ctx->stage_io_bytes, in_b + out_b);
  if (rc) return rc;
  double* d_m = ctx->stage_io;
  double* d_h = ctx->stage_io + (size_t)batch * 3 * n;
  MT_CUDA_OK(ctx, cudaMemcpyAsync(d_m, m_host, in_b, cudaMemcpyHostToDevice, ctx->stream));
  rc = mt_demag_field(ctx, N, dtype, n, n_rows, ld, Ms, d_m, batch, d_h);
  if (rc) return rc;
  MT_CUDA_OK(ctx, cudaMemcpyAsync(Hd_host, d_h, out_b, cudaMemcpyDeviceToHost, ctx->stream));
  MT_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  return MT_OK;
}

int mt_llg_rhs(mt_ctx* ctx, const mt_problem* p, const double* m, int batch, double* dmdt, double* Heff) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_problem(ctx, p, batch);
  if (rc) return rc;
  if (!m || !dmdt) return mt_fail(ctx, MT_ERR_INVALID_ARG, "m and dmdt must be non-NULL");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int64_t npad = round_up(p->n, MT_COL_CHUNK);
  EpiArgs e;
  fill_problem(e, p, batch);
  e.y = m;
  e.k_out = dmdt;
  e.heff_out = Heff;
  // small dense problems: one launch, the field kernel forms Ms*m itself (same bits as the staged M)
  if (p->N && !p->N_sparse && !p->N_sym && mt_demag_can_fuse(ctx, p->dtype, p->n, e.n_rows, p->Ms, m))
    return mt_launch_demag(ctx, p->N, p->dtype, p->n, e.n_rows, p->ld, nullptr, npad, e, p->Ms, m);
  if (has_demag(p)) {
    rc = ensure_Mst(ctx, demag_dtype(p), batch, npad);
    if (rc) return rc;
    rc = mt_launch_stage_M(ctx, demag_dtype(p), p->Ms, m, batch, p->n, npad, ctx->Mst[0]);
    if (rc) return rc;
  }
  return eval_rhs(ctx, p, npad, 0, e);
}

int64_t mt_sym_tensor_elems(int64_t n, int dtype) {
  if (n <= 0 || (dtype != MT_F32 && dtype != MT_F64)) return 0;
  const int tw = dtype == MT_F32 ? SymCfg<float>::TW : SymCfg<double>::TW;
  return sym_total_tiles(n, tw) * (int64_t)6 * 32 * tw;
}

int mt_assemble_tensor_sym(mt_ctx* ctx, const mt_tiles* t, int dtype, void* out, int32_t* status_flag) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!t || !t->type || !t->center || !t->size || t->n <= 0) return mt_fail(ctx, MT_ERR_INVALID_ARG, "tiles incomplete");
  if (dtype != MT_F32 && dtype != MT_F64) return mt_fail(ctx, MT_ERR_INVALID_ARG, "unknown dtype %d", dtype);
  if (!out || ((uintptr_t)out & 15)) return mt_fail(ctx, MT_ERR_INVALID_ARG, "out null or not 16-byte aligned");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  return mt_launch_assemble_sym(ctx, t, dtype, out, status_flag);
}

int mt_demag_field_sym(mt_ctx* ctx, const mt_sym_tensor* S, const double* Ms, const double* m, int batch, double* Hd) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_sym(ctx, S);
  if (rc) return rc;
  if (!Ms || !m || !Hd) return mt_fail(ctx, MT_ERR_INVALID_ARG, "Ms, m and Hd must be non-NULL");
  if (batch < 1 || batch > MT_MAX_BATCH) return mt_fail(ctx, MT_ERR_INVALID_ARG, "batch must be in [1, %d]", MT_MAX_BATCH);
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int64_t npad = round_up(S->n, MT_COL_CHUNK);
  if ((rc = ensure_Mst(ctx, S->dtype, batch, npad))) return rc;
  if ((rc = mt_launch_stage_M(ctx, S->dtype, Ms, m, batch, S->n, npad, ctx->Mst[0]))) return rc;
  EpiArgs e;
  memset(&e, 0, sizeof(e));
  e.mode = 0;
  e.batch = batch;
  e.n = S->n;
  e.n_rows = S->n;
  e.Hd = Hd;
  return mt_launch_demag_sym(ctx, S, ctx->Mst[0], npad, e);
}

int64_t mt_sparse_mask_words(int64_t n) { return n <= 0 ? 0 : round_up((n + 31) / 32, 4); }

// ---- threshold selection, one radix digit per pass; the passes may be fed band by band ---------------
// Digits: the first pass fixes the top 11 bits of the 31 / 63-bit key (every element is binned: shared-
// memory histogram with warp-aggregated runs), every later pass up to 20 bits (only the few elements that
// carry the prefix are binned, straight into the global histogram): 2 passes for fp32, 4 for fp64
// (r03: 3 and 6 passes of 11 bits).
namespace {
constexpr int kSelFirst = 11, kSelWide = 20;
constexpr int64_t kSelHistWords = MT_SELECT_HIST_WORDS;
static_assert(kSelHistWords == (1 << kSelWide), "histogram size = widest digit");
inline int sel_bits(int dtype) { return dtype == MT_F32 ? 31 : 63; }  // the sign bit is cleared
inline int sel_width(const mt_select_state* st) {
  const int w = st->hi == sel_bits(st->dtype) ? kSelFirst : kSelWide;
  return st->hi >= w ? w : st->hi;
}
int ensure_sel_hist(mt_ctx* ctx) {
  if (ctx->sel_hist) return MT_OK;
  MT_CUDA_OK(ctx, cudaMalloc((void**)&ctx->sel_hist, (size_t)kSelHistWords * sizeof(unsigned long long)));
  return MT_OK;
}
}  // namespace

int mt_select_begin(mt_ctx* ctx, mt_select_state* st, int dtype, double fraction, unsigned long long* hist) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!st || !hist) return mt_fail(ctx, MT_ERR_INVALID_ARG, "state and hist must be non-NULL");
  if (dtype != MT_F32 && dtype != MT_F64) return mt_fail(ctx, MT_ERR_INVALID_ARG, "unknown dtype %d", dtype);
  if (!(fraction >= 0.0 && fraction <= 1.0)) return mt_fail(ctx, MT_ERR_INVALID_ARG, "fraction must be in [0, 1]");
  memset(st, 0, sizeof(*st));
  st->dtype = dtype;
  st->fraction = fraction;
  st->hi = sel_bits(dtype);
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  MT_CUDA_OK(ctx, cudaMemsetAsync(hist, 0, (size_t)kSelHistWords * sizeof(unsigned long long), ctx->stream));
  return MT_OK;
}

int mt_select_accumulate(mt_ctx* ctx, const mt_select_state* st, const void* N, int64_t n, int64_t n_rows, int64_t ld,
                         unsigned long long* hist) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!st || !hist) return mt_fail(ctx, MT_ERR_INVALID_ARG, "state and hist must be non-NULL");
  if (st->done) return mt_fail(ctx, MT_ERR_INVALID_ARG, "selection already finished");
  int rc = check_tensor_args(ctx, N, st->dtype, n, n_rows, ld);
  if (rc) return rc;
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int width = sel_width(st);
  // the kernels test (key & ~((1 << hi) - 1)) == prefix << hi: in the first pass hi = 31 / 63 and the
  // prefix is empty (the cleared sign bit)
  return mt_launch_select_hist(ctx, N, st->dtype, n, n_rows, ld, st->prefix, st->hi, st->hi - width, width, hist);
}

int mt_select_advance(mt_ctx* ctx, mt_select_state* st, unsigned long long* hist) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!st || !hist) return mt_fail(ctx, MT_ERR_INVALID_ARG, "state and hist must be non-NULL");
  if (st->done) return MT_OK;
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int bits = sel_bits(st->dtype);
  const int width = sel_width(st);
  const bool first = st->hi == bits;
  // the bin that holds rank k is found on the device (one block over the histogram): 32 bytes come back
  unsigned long long* d_out = ctx->dscal + 2;
  int rc = mt_launch_select_find(ctx, hist, 1 << width, st->k, first ? 1 : 0, st->fraction, d_out);
  if (rc) return rc;
  MT_CUDA_OK(ctx, cudaMemcpyAsync(ctx->hscal, d_out, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream));
  MT_CUDA_OK(ctx, cudaMemsetAsync(hist, 0, (size_t)kSelHistWords * sizeof(unsigned long long), ctx->stream));
  MT_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  const unsigned long long total = ctx->hscal[0], bin = ctx->hscal[1], rem = ctx->hscal[2];
  if (first) {  // total number of non-zero elements, and the rank to find
    st->count = total;
    st->k = ctx->hscal[3];
    if (st->k >= st->count) {  // everything removed (also: nothing to rank)
      st->done = 1;
      st->tau = INFINITY;
      return MT_OK;
    }
  }
  st->k = rem;
  st->prefix = (st->prefix << width) | bin;
  st->hi -= width;
  if (st->hi == 0) {
    st->done = 1;
    if (st->dtype == MT_F32) {
      const uint32_t u = (uint32_t)st->prefix;
      float f;
      memcpy(&f, &u, 4);
      st->tau = (double)f;
    } else {
      st->tau = bits_to_double(st->prefix);
    }
  }
  return MT_OK;
}

int mt_threshold_value(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                       double fraction, double* tau_host, int64_t* count_host) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_tensor_args(ctx, N, dtype, n, n_rows, ld);
  if (rc) return rc;
  if (!tau_host || !(fraction >= 0.0 && fraction <= 1.0))
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "fraction must be in [0, 1] and tau_host non-NULL");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  // MSB-first radix select over the bit pattern of |v| (31 / 63 significant bits); each pass is one
  // stream of the tensor; the histogram is ctx-owned (no allocation per call after the first)
  if ((rc = ensure_sel_hist(ctx))) return rc;
  unsigned long long* d_hist = ctx->sel_hist;
  mt_select_state st;
  rc = mt_select_begin(ctx, &st, dtype, fraction, d_hist);
  while (!rc && !st.done) {
    if ((rc = mt_select_accumulate(ctx, &st, N, n, n_rows, ld, d_hist))) break;
    rc = mt_select_advance(ctx, &st, d_hist);
  }
  if (rc) return rc;
  if (count_host) *count_host = (int64_t)st.count;
  *tau_host = st.tau;
  return MT_OK;
}

int mt_sparse_count_band(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                         int64_t row0, int64_t n_total, int64_t* counts) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_tensor_args(ctx, N, dtype, n, n_rows, ld);
  if (rc) return rc;
  if (!counts) return mt_fail(ctx, MT_ERR_INVALID_ARG, "counts must be non-NULL");
  if (row0 < 0 || row0 + n_rows > n_total) return mt_fail(ctx, MT_ERR_INVALID_ARG, "band outside [0, n_total)");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  return mt_launch_sparse_count(ctx, N, dtype, n, n_rows, ld, tau, row0, n_total, counts);
}

int mt_sparse_scan(mt_ctx* ctx, int64_t* row_ptr, int64_t n_total, int64_t* nnz_host) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!row_ptr || !nnz_host || n_total <= 0)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "row_ptr and nnz_host must be non-NULL, n_total positive");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  int rc = mt_launch_sparse_scan(ctx, row_ptr, n_total);
  if (rc) return rc;
  MT_CUDA_OK(ctx, cudaMemcpyAsync(ctx->hscal, row_ptr + 6 * n_total, 8, cudaMemcpyDeviceToHost, ctx->stream));
  MT_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  *nnz_host = (int64_t)ctx->hscal[0];
  return MT_OK;
}

int mt_sparse_fill_index_band(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                              int64_t row0, int64_t n_total, const int64_t* row_ptr, uint32_t* mask, void* vals,
                              uint16_t* cols16, int64_t* panel_ptr) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_tensor_args(ctx, N, dtype, n, n_rows, ld);
  if (rc) return rc;
  if (!row_ptr || (!mask && !cols16)) return mt_fail(ctx, MT_ERR_INVALID_ARG, "row_ptr and one of mask / cols16 must be non-NULL");
  if (cols16 && n > 65536 && !panel_ptr)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "n > 65536: panel_ptr must be non-NULL with cols16");
  if (row0 < 0 || row0 + n_rows > n_total) return mt_fail(ctx, MT_ERR_INVALID_ARG, "band outside [0, n_total)");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  return mt_launch_sparse_fill(ctx, N, dtype, n, n_rows, ld, tau, row0, n_total, row_ptr, mt_sparse_mask_words(n), mask,
                               vals, cols16, panel_ptr);
}

int mt_sparse_fill_band(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                        int64_t row0, int64_t n_total, const int64_t* row_ptr, uint32_t* mask, void* vals) {
  if (ctx && !mask) return mt_fail(ctx, MT_ERR_INVALID_ARG, "row_ptr and mask must be non-NULL");
  return mt_sparse_fill_index_band(ctx, N, dtype, n, n_rows, ld, tau, row0, n_total, row_ptr, mask, vals, nullptr,
                                   nullptr);
}

int mt_sparse_count(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                    int64_t* row_ptr, int64_t* nnz_host) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!row_ptr || !nnz_host) return mt_fail(ctx, MT_ERR_INVALID_ARG, "row_ptr and nnz_host must be non-NULL");
  int rc = mt_sparse_count_band(ctx, N, dtype, n, n_rows, ld, tau, 0, n_rows, row_ptr);
  if (rc) return rc;
  return mt_sparse_scan(ctx, row_ptr, n_rows, nnz_host);
}

int mt_sparse_fill(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld, double tau,
                   const int64_t* row_ptr, uint32_t* mask, void* vals) {
  return mt_sparse_fill_band(ctx, N, dtype, n, n_rows, ld, tau, 0, n_rows, row_ptr, mask, vals);
}

namespace {
int check_stream_args(mt_ctx* ctx, const mt_tiles* t, int dtype, int64_t row_begin, int64_t row_end, const void* band,
                      int64_t band_rows, int64_t ld) {
  if (!t || !t->type || !t->center || !t->size || t->n <= 0) return mt_fail(ctx, MT_ERR_INVALID_ARG, "tiles incomplete");
  if (row_begin < 0 || row_end <= row_begin || row_end > t->n)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "row band [%lld, %lld) outside [0, %lld)", (long long)row_begin,
                   (long long)row_end, (long long)t->n);
  if (band_rows <= 0) return mt_fail(ctx, MT_ERR_INVALID_ARG, "band_rows must be positive");
  return check_tensor_args(ctx, band, dtype, t->n, band_rows, ld);
}
}  // namespace

int mt_sparse_stream_count(mt_ctx* ctx, const mt_tiles* t, int dtype, double fraction, int64_t row_begin,
                           int64_t row_end, void* band, int64_t band_rows, int64_t ld, int64_t* row_ptr,
                           unsigned long long* hist, mt_allreduce_fn allreduce, void* user, int32_t* status_flag,
                           double* tau_host, int64_t* nnz_host) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_stream_args(ctx, t, dtype, row_begin, row_end, band, band_rows, ld);
  if (rc) return rc;
  if (!row_ptr || !tau_host || !nnz_host) return mt_fail(ctx, MT_ERR_INVALID_ARG, "row_ptr, tau_host and nnz_host must be non-NULL");
  if (fraction > 1.0) return mt_fail(ctx, MT_ERR_INVALID_ARG, "fraction must be in [0, 1] (or negative: tau given)");
  if (allreduce && !hist) return mt_fail(ctx, MT_ERR_INVALID_ARG, "allreduce needs a caller-owned hist");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int64_t n_loc = row_end - row_begin;
  if (fraction >= 0.0) {
    if (!hist && (rc = ensure_sel_hist(ctx))) return rc;
    unsigned long long* h = hist ? hist : ctx->sel_hist;
    mt_select_state st;
    if ((rc = mt_select_begin(ctx, &st, dtype, fraction, h))) return rc;
    while (!st.done) {
      for (int64_t r0 = row_begin; r0 < row_end; r0 += band_rows) {
        const int64_t r1 = r0 + band_rows < row_end ? r0 + band_rows : row_end;
        if ((rc = mt_launch_assemble(ctx, t, dtype, r0, r1, band, ld, status_flag))) return rc;
        if ((rc = mt_select_accumulate(ctx, &st, band, t->n, r1 - r0, ld, h))) return rc;
      }
      if (allreduce && allreduce(user, h, (void*)ctx->stream) != 0)
        return mt_fail(ctx, MT_ERR_CUDA, "histogram all-reduce callback failed");
      if ((rc = mt_select_advance(ctx, &st, h))) return rc;
    }
    *tau_host = st.tau;
  }
  for (int64_t r0 = row_begin; r0 < row_end; r0 += band_rows) {
    const int64_t r1 = r0 + band_rows < row_end ? r0 + band_rows : row_end;
    if ((rc = mt_launch_assemble(ctx, t, dtype, r0, r1, band, ld, status_flag))) return rc;
    if ((rc = mt_launch_sparse_count(ctx, band, dtype, t->n, r1 - r0, ld, *tau_host, r0 - row_begin, n_loc, row_ptr))) return rc;
  }
  return mt_sparse_scan(ctx, row_ptr, n_loc, nnz_host);
}

int mt_sparse_stream_fill(mt_ctx* ctx, const mt_tiles* t, int dtype, double tau, int64_t row_begin, int64_t row_end,
                          void* band, int64_t band_rows, int64_t ld, const int64_t* row_ptr, uint32_t* mask, void* vals,
                          uint16_t* cols16, int64_t* panel_ptr, int32_t* status_flag) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_stream_args(ctx, t, dtype, row_begin, row_end, band, band_rows, ld);
  if (rc) return rc;
  if (!row_ptr || !vals || (!mask && !cols16))
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "row_ptr, vals and one of mask / cols16 must be non-NULL");
  if (cols16 && t->n > 65536 && !panel_ptr)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "n > 65536: panel_ptr must be non-NULL with cols16");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int64_t n_loc = row_end - row_begin;
  for (int64_t r0 = row_begin; r0 < row_end; r0 += band_rows) {
    const int64_t r1 = r0 + band_rows < row_end ? r0 + band_rows : row_end;
    if ((rc = mt_launch_assemble(ctx, t, dtype, r0, r1, band, ld, status_flag))) return rc;
    if ((rc = mt_launch_sparse_fill(ctx, band, dtype, t->n, r1 - r0, ld, tau, r0 - row_begin, n_loc, row_ptr,
                                    mt_sparse_mask_words(t->n), mask, vals, cols16, panel_ptr)))
      return rc;
  }
  MT_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  return MT_OK;
}

int mt_sparse_index(mt_ctx* ctx, const mt_sparse_tensor* S, uint16_t* cols16, int64_t* panel_ptr) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  if (!S) return mt_fail(ctx, MT_ERR_INVALID_ARG, "sparse tensor is NULL");
  mt_sparse_tensor t = *S;
  t.cols16 = nullptr;  // ignored here (it may be the array being written)
  t.panel_ptr = nullptr;
  int rc = check_sparse(ctx, &t);
  if (rc) return rc;
  if (!cols16 || !S->mask) return mt_fail(ctx, MT_ERR_INVALID_ARG, "cols16 and S->mask must be non-NULL");
  if (S->n > 65536 && !panel_ptr)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "n > 65536: panel_ptr ([6*n_rows][ceil(n/65536)-1]) must be non-NULL");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  return mt_launch_sparse_index(ctx, S, cols16, panel_ptr);
}

int mt_demag_field_sparse(mt_ctx* ctx, const mt_sparse_tensor* S, const double* Ms, const double* m, int batch,
                          double* Hd) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_sparse(ctx, S);
  if (rc) return rc;
  if (!Ms || !m || !Hd) return mt_fail(ctx, MT_ERR_INVALID_ARG, "Ms, m and Hd must be non-NULL");
  if (batch < 1 || batch > MT_MAX_BATCH) return mt_fail(ctx, MT_ERR_INVALID_ARG, "batch must be in [1, %d]", MT_MAX_BATCH);
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int64_t npad = round_up(S->n, MT_COL_CHUNK);
  if ((rc = ensure_Mst(ctx, S->dtype, batch, npad))) return rc;
  if ((rc = mt_launch_stage_M(ctx, S->dtype, Ms, m, batch, S->n, npad, ctx->Mst[0]))) return rc;
  EpiArgs e;
  memset(&e, 0, sizeof(e));
  e.mode = 0;
  e.batch = batch;
  e.n = S->n;
  e.n_rows = S->n_rows;
  e.Hd = Hd;
  return mt_launch_demag_sparse(ctx, S, ctx->Mst[0], npad, e);
}

int mt_energy(mt_ctx* ctx, const mt_problem* p, const double* m, int batch, double* E_out) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_problem(ctx, p, batch);
  if (rc) return rc;
  if (!m || !E_out) return mt_fail(ctx, MT_ERR_INVALID_ARG, "m and E_out must be non-NULL");
  if (p->shard) return mt_fail(ctx, MT_ERR_INVALID_ARG, "mt_energy does not take a row-sharded problem");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  const int64_t npad = round_up(p->n, MT_COL_CHUNK);
  rc = mt_ensure_ws(ctx, (void**)&ctx->edens, &ctx->edens_bytes, (size_t)batch * 4 * p->n * sizeof(double));
  if (rc) return rc;
  if (has_demag(p)) {
    if ((rc = ensure_Mst(ctx, demag_dtype(p), batch, npad))) return rc;
    if ((rc = mt_launch_stage_M(ctx, demag_dtype(p), p->Ms, m, batch, p->n, npad, ctx->Mst[0]))) return rc;
  }
  EpiArgs e;
  fill_problem(e, p, batch);
  e.y = m;
  e.e_dens = ctx->edens;
  e.vol = p->vol;
  if ((rc = eval_rhs(ctx, p, npad, 0, e))) return rc;
  return mt_launch_energy_reduce(ctx, ctx->edens, batch, p->n, E_out);
}

int mt_field_sweep(mt_ctx* ctx, const mt_problem* p, const mt_integrator_opts* o, const double* fields_host,
                   int64_t n_fields, double* m, int batch, double* rows, mt_integrator_result* res_host) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_problem(ctx, p, batch);
  if (rc) return rc;
  if (!o || !fields_host || n_fields < 0 || !m || !rows)
    return mt_fail(ctx, MT_ERR_INVALID_ARG, "opts, fields, m and rows must be non-NULL");
  if (p->H_a) return mt_fail(ctx, MT_ERR_INVALID_ARG, "mt_field_sweep sets the uniform applied field: H_a must be NULL");
  if (p->shard) return mt_fail(ctx, MT_ERR_INVALID_ARG, "mt_field_sweep does not take a row-sharded problem");
  const int64_t stride = 8 * (int64_t)batch;
  mt_problem pk = *p;
  mt_integrator_result total;
  memset(&total, 0, sizeof(total));
  for (int64_t f = 0; f < n_fields; ++f) {
    for (int a = 0; a < 3; ++a) pk.H_a_const[a] = fields_host[3 * f + a];
    double t = 0.0;
    mt_integrator_result r = {};
    rc = mt_integrate(ctx, &pk, o, m, batch, &t, nullptr, 0, &r);
    total.accepted += r.accepted; total.rejected += r.rejected; total.rhs_calls += r.rhs_calls;
    total.t += r.t; total.dt_last = r.dt_last; total.max_torque = r.max_torque;
    if (rc && rc != MT_ERR_MAX_STEPS) break;
    // row f: per state <m_x>, <m_y>, <m_z> (A10) then E_demag, E_exch, E_anis, E_zeeman, E_total.  The
    // mean kernel writes t into its slot 0, so it gets a scratch row of 1 + 3 B doubles and the means
    // are copied behind it; the energies are written in place.
    double* row = rows + f * stride;
    if ((rc = mt_ensure_ws(ctx, (void**)&ctx->stage_io, &ctx->stage_io_bytes, (size_t)(1 + 8 * batch) * sizeof(double)))) break;
    double* scratch = ctx->stage_io;
    if ((rc = mt_launch_mean(ctx, m, p->vol, batch, p->n, t, scratch))) break;
    if ((rc = mt_energy(ctx, &pk, m, batch, scratch + 1 + 3 * batch))) break;
    for (int b = 0; b < batch && !rc; ++b) {
      if (cudaMemcpyAsync(row + 8 * b, scratch + 1 + 3 * b, 3 * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream) != cudaSuccess ||
          cudaMemcpyAsync(row + 8 * b + 3, scratch + 1 + 3 * batch + 5 * b, 5 * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream) != cudaSuccess)
        rc = mt_fail(ctx, MT_ERR_CUDA, "cudaMemcpyAsync failed in mt_field_sweep");
    }
    if (rc) break;
    // the scratch row is reused by the next field: order is kept by the stream
  }
  if (cudaStreamSynchronize(ctx->stream) != cudaSuccess && !rc) rc = mt_fail(ctx, MT_ERR_CUDA, "stream synchronise failed");
  if (res_host) *res_host = total;
  return rc;
}

int mt_integrate(mt_ctx* ctx, const mt_problem* p, const mt_integrator_opts* o, double* m, int batch,
                 double* t_inout, double* samples, int64_t sample_cap, mt_integrator_result* res) {
  if (!ctx) return MT_ERR_INVALID_ARG;
  int rc = check_problem(ctx, p, batch);
  if (rc) return rc;
  if (!o || !m || !t_inout || !res) return mt_fail(ctx, MT_ERR_INVALID_ARG, "opts, m, t and result must be non-NULL");
  if (o->method != MT_RK4 && o->method != MT_DP45) return mt_fail(ctx, MT_ERR_INVALID_ARG, "unknown method %d", o->method);
  if (o->method == MT_RK4 && !(o->dt > 0)) return mt_fail(ctx, MT_ERR_INVALID_ARG, "RK4 needs dt > 0");
  MT_CUDA_OK(ctx, cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
  const int64_t n = p->n, sv = (int64_t)batch * 3 * n;  // doubles per state vector
  const int64_t npad = round_up(n, MT_COL_CHUNK);
  const int64_t stride = 1 + 3 * (int64_t)batch;
  memset(res, 0, sizeof(*res));
  // workspace: k1..k7, two scratch states, candidate state, chunk-start backup (RK4 stop test)
  rc = mt_ensure_ws(ctx, (void**)&ctx->rk, &ctx->rk_bytes, (size_t)(7 + 4) * sv * sizeof(double));
  if (rc) return rc;
  double* k[7];
  for (int s = 0; s < 7; ++s) k[s] = ctx->rk + (int64_t)s * sv;
  double* ya = ctx->rk + 7 * sv;
  double* yb = ctx->rk + 8 * sv;
  double* mc = ctx->rk + 9 * sv;
  double* mb = ctx->rk + 10 * sv;
  if (has_demag(p)) {
    rc = ensure_Mst(ctx, demag_dtype(p), batch, npad);
    if (rc) return rc;
    rc = mt_launch_stage_M(ctx, demag_dtype(p), p->Ms, m, batch, n, npad, ctx->Mst[0]);
    if (rc) return rc;
    // the second buffer is only ever written by the fused epilogue (rows < n): give its padding
    // defined (zero) contents for this n as well, whatever an earlier problem left there
    rc = mt_launch_stage_M(ctx, demag_dtype(p), p->Ms, m, batch, n, npad, ctx->Mst[1]);
    if (rc) return rc;
  }
  // Row-sharded problem (mt.h section 8(e)): every stage's combine writes this rank's rows into its
  // block of the all-gather buffer; `finish` then gathers the blocks and scatters them into the full
  // stage state (and the staged M).  The error / torque maxima live in the caller's `scal` and are
  // max-reduced over the ranks before the host reads them.
  const mt_shard* sh = p->shard;
  unsigned long long* d_err = sh ? sh->scal : ctx->dscal;
  unsigned long long* d_tq = d_err + 1;
  auto xchg = [&](int what) -> int {
    if (sh->exchange(sh->user, what, (void*)st) != 0)
      return mt_fail(ctx, MT_ERR_CUDA, "shard exchange callback failed (what = %d)", what);
    return MT_OK;
  };
  auto route = [&](EpiArgs& e, double* y_dst, void* M_dst) {
    if (!sh) { e.y_out = y_dst; e.M_out = M_dst; return; }
    e.y_out = sh->pack + (int64_t)sh->rank * batch * 3 * sh->slice_pad;
    e.y_ld = sh->slice_pad;
    e.y_row0 = band_begin(p);
    e.M_out = nullptr;
  };
  auto finish = [&](double* y_dst, void* M_dst) -> int {
    if (!sh) return MT_OK;
    int r = xchg(MT_XCHG_GATHER_STATE);
    if (r) return r;
    return mt_launch_unpack(ctx, sh->pack, sh->world, sh->slice_pad, batch, n, npad, p->Ms, y_dst, M_dst, demag_dtype(p));
  };
  auto read_scalars = [&](int count) -> int {  // d_err[0 .. count) -> ctx->hscal, after the ranks' maxima are combined
    if (sh) { int r = xchg(MT_XCHG_MAX_SCALARS); if (r) return r; }
    MT_CUDA_OK(ctx, cudaMemcpyAsync(ctx->hscal, d_err + (2 - count), 8 * count, cudaMemcpyDeviceToHost, st));
    MT_CUDA_OK(ctx, cudaStreamSynchronize(st));
    return MT_OK;
  };
  double t = *t_inout;
  const double t0 = t;
  int status = MT_OK;
  EpiArgs base;
  fill_problem(base, p, batch);
  base.M_out = nullptr;
  base.npad = npad;

  if (o->method == MT_RK4) {
    // ---- A8: classical RK4; the four fused launches of a step are replayed from a CUDA graph ----
    const double dt = o->dt;
    int64_t nsteps = (int64_t)llround((o->t_end - t) / dt);
    if (nsteps < 0) nsteps = 0;
    bool hit_max = false;
    if (o->max_steps > 0 && nsteps > o->max_steps) { nsteps = o->max_steps; hit_max = true; }
    const bool want_tq = o->torque_tol > 0;
    // the four stages of a step as epilogue descriptors (stage s reads the staged M of buffer src[s]):
    //   1: k1 = f(m),  ya = m + dt/2 k1      2: k2 = f(ya), yb = m + dt/2 k2
    //   3: k3 = f(yb), ya = m + dt k3        4: k4 = f(ya), m <- m + dt/6 (k1 + 2 k2 + 2 k3 + k4), renormalised
    void* const Mbuf[2] = {has_demag(p) ? ctx->Mst[0] : nullptr, has_demag(p) ? ctx->Mst[1] : nullptr};
    double* const y_in[4] = {m, ya, yb, ya};
    double* const y_to[4] = {ya, yb, ya, m};
    const int src_of[4] = {0, 1, 0, 1};
    auto make_stage = [&](int s, unsigned long long* tq) -> EpiArgs {
      EpiArgs e = base;
      e.y = y_in[s]; e.k_out = k[s]; e.torque_bits = s == 0 ? tq : nullptr;
      e.do_comb = 1; e.base = m;
      if (s < 3) {
        e.ncomb = 1; e.kptr[0] = k[s]; e.coef[0] = 1.0; e.h = s < 2 ? 0.5 * dt : dt;
      } else {
        e.ncomb = 4;
        for (int j = 0; j < 4; ++j) e.kptr[j] = k[j];
        e.coef[0] = 1.0; e.coef[1] = 2.0; e.coef[2] = 2.0; e.coef[3] = 1.0;
        e.h = dt / 6.0; e.renorm = o->renormalize;
      }
      route(e, y_to[s], Mbuf[src_of[s] ^ 1]);
      return e;
    };
    auto run_stage = [&](int s, unsigned long long* tq) -> int {
      const EpiArgs e = make_stage(s, tq);
      int r = eval_rhs(ctx, p, npad, src_of[s], e);
      return r ? r : finish(y_to[s], Mbuf[src_of[s] ^ 1]);
    };
    auto stage1 = [&](unsigned long long* tq) -> int { return run_stage(0, tq); };
    auto stages234 = [&]() -> int {
      int r;
      if ((r = run_stage(1, nullptr)) || (r = run_stage(2, nullptr))) return r;
      return run_stage(3, nullptr);
    };
    // Tensor resident in shared memory (resident.cu): dense, unsharded problems small enough for the SMs
    // to hold the tensor between them run a whole chunk of steps in ONE cooperative launch.
    const int res_mode = (p->N && !p->N_sparse && !p->N_sym && !sh && round_up(n, p->dtype == MT_F32 ? 4 : 2) <= p->ld)
                             ? mt_resident_fits(ctx, p->dtype, n, p->ld, batch, MT_RK4) : MT_RES_NONE;
    const bool res_ok = res_mode != MT_RES_NONE;
    if (ctx->resident_mode == 2 && !res_ok)
      return mt_fail(ctx, MT_ERR_INVALID_ARG, "resident RK4 required (mt_set_resident_mode 2) but the problem does not qualify "
                     "(dense unsharded tensor that fits in the SMs' shared memory)");
    const bool resident = res_ok && ctx->resident_mode != 1;
    auto sample_if_due = [&](int64_t done) -> int {
      if (o->sample_every > 0 && done % o->sample_every == 0 && samples && res->n_samples < sample_cap) {
        int r = mt_launch_mean(ctx, m, p->vol, batch, n, t0 + (double)done * dt, samples + res->n_samples * stride);
        if (r) return r;
        res->n_samples++;
      }
      return MT_OK;
    };
    int64_t done = 0;
    if (want_tq && sh) {
      // row-sharded: the stop test (Eq. 2) needs the ranks' maxima combined, one exchange
      // and one host read per step; a satisfied test leaves m untouched
      while (done < nsteps) {
        MT_CUDA_OK(ctx, cudaMemsetAsync(d_err, 0, 16, st));
        if ((rc = stage1(d_tq))) return rc;
        if ((rc = read_scalars(1))) return rc;
        res->max_torque = bits_to_double(ctx->hscal[0]);
        if (res->max_torque <= o->torque_tol) break;
        if ((rc = stages234())) return rc;
        done++;
        if ((rc = sample_if_due(done))) return rc;
      }
    } else {
      // Steps run in chunks; a whole chunk is captured once into a CUDA graph and replayed (every buffer
      // is back in its role after a step).  The first chunk runs eagerly: it sizes the workspaces, which
      // must not be allocated under capture.  With the stop test (Eq. 2) every step of a chunk
      // leaves the torque of the state it started from in its own device word; the host reads the chunk's
      // words once (one synchronisation per chunk instead of per step) and, when a step's test was
      // satisfied, goes back to the chunk's first state and repeats the steps before it: the state
      // returned is the one the per-step test would have stopped at, bit for bit.
      int64_t chunk = o->sample_every > 0 ? o->sample_every : 64;
      if (chunk > 256) chunk = 256;
      while (o->sample_every > 0 && o->sample_every % chunk) chunk--;  // chunk divides sample_every
      unsigned long long* slots = ctx->dscal + 8;
      cudaGraph_t graph = nullptr;
      cudaGraphExec_t exec = nullptr;
      int64_t graph_launches = 0;
      bool stopped = false;
      auto run_steps = [&](int64_t count, bool with_tq) -> int {
        if (resident)
          return mt_launch_rk4_resident(ctx, res_mode, p->N, p->dtype, n, p->ld, base, m, ya, yb, dt, o->renormalize,
                                        with_tq ? slots : nullptr, (unsigned int*)(ctx->dscal + 6), count);
        int r = MT_OK;
        for (int64_t s = 0; s < count && !r; ++s) {
          r = stage1(with_tq ? slots + s : nullptr);
          if (!r) r = stages234();
        }
        return r;
      };
      while (done < nsteps && !rc && !stopped) {
        // (exchange callbacks are host calls; a resident chunk already is a single launch)
        const bool use_graph = !sh && !resident && done >= chunk && done % chunk == 0 && nsteps - done >= chunk;
        int64_t kk = chunk - done % chunk;
        if (kk > nsteps - done) kk = nsteps - done;
        if (want_tq) {
          MT_CUDA_OK(ctx, cudaMemcpyAsync(mb, m, (size_t)sv * sizeof(double), cudaMemcpyDeviceToDevice, st));
          MT_CUDA_OK(ctx, cudaMemsetAsync(slots, 0, 8 * (size_t)kk, st));
        }
        if (use_graph) {
          if (!exec) {
            // capture on a private stream (the caller's may be the legacy default stream, which cannot
            // be captured); the instantiated graph is then launched on the caller's stream
            if (!ctx->cap_stream) MT_CUDA_OK(ctx, cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
            const int64_t l0 = ctx->launches;
            MT_CUDA_OK(ctx, cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
            ctx->stream = ctx->cap_stream;
            const int prof_saved = ctx->prof_on;
            ctx->prof_on = 0;  // timing events must not become graph nodes
            const int r = run_steps(chunk, want_tq);
            ctx->stream = st;
            ctx->prof_on = prof_saved;
            cudaError_t ce = cudaStreamEndCapture(ctx->cap_stream, &graph);
            graph_launches = ctx->launches - l0;
            ctx->launches = l0;  // captured, not yet launched
            if (r) { if (graph) cudaGraphDestroy(graph); return r; }
            MT_CUDA_OK(ctx, ce);
            MT_CUDA_OK(ctx, cudaGraphInstantiate(&exec, graph, 0));
          }
          cudaError_t ce = cudaGraphLaunch(exec, st);
          if (ce != cudaSuccess) { rc = mt_fail(ctx, MT_ERR_CUDA, "cudaGraphLaunch: %s", cudaGetErrorString(ce)); break; }
          ctx->launches += graph_launches;
        } else if ((rc = run_steps(kk, want_tq))) {
          break;
        }
        if (want_tq) {
          cudaError_t ce = cudaMemcpyAsync(ctx->hscal, slots, 8 * (size_t)kk, cudaMemcpyDeviceToHost, st);
          if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
          if (ce != cudaSuccess) { rc = mt_fail(ctx, MT_ERR_CUDA, "reading the chunk's torques: %s", cudaGetErrorString(ce)); break; }
          int64_t hit = -1;
          for (int64_t s = 0; s < kk && hit < 0; ++s)
            if (bits_to_double(ctx->hscal[s]) <= o->torque_tol) hit = s;
          if (hit < 0) {
            res->max_torque = bits_to_double(ctx->hscal[kk - 1]);
            done += kk;
          } else {
            // step `hit` of the chunk would not have been taken: rebuild the state it started from
            cudaError_t c2 = cudaMemcpyAsync(m, mb, (size_t)sv * sizeof(double), cudaMemcpyDeviceToDevice, st);
            if (c2 != cudaSuccess) { rc = mt_fail(ctx, MT_ERR_CUDA, "restoring the chunk's first state: %s", cudaGetErrorString(c2)); break; }
            if (has_demag(p) && (rc = mt_launch_stage_M(ctx, demag_dtype(p), p->Ms, m, batch, n, npad, ctx->Mst[0]))) break;
            if ((rc = run_steps(hit, false))) break;
            res->max_torque = bits_to_double(ctx->hscal[hit]);
            done += hit;
            stopped = true;
          }
        } else {
          done += kk;
        }
        if (!stopped) rc = sample_if_due(done);
      }
      if (exec) cudaGraphExecDestroy(exec);
      if (graph) cudaGraphDestroy(graph);
      if (rc) return rc;
    }
    res->rhs_calls = 4 * done;
    res->accepted = done;
    res->dt_last = dt;
    t = t0 + (double)done * dt;
    if (hit_max && done == nsteps) status = MT_ERR_MAX_STEPS;
  } else {
    // ---- A9: Dormand-Prince 5(4) with FSAL; the controller runs on the host, one 16-byte read per
    // attempted step (at the sizes where the step is milliseconds this is noise) ----------
    double dt = o->dt > 0 ? o->dt : 1e-3;
    int64_t next_sample = 1;
    // k1 = f(m)
    {
      MT_CUDA_OK(ctx, cudaMemsetAsync(d_err, 0, 16, st));
      EpiArgs e = base;
      e.y = m; e.k_out = k[0]; e.torque_bits = d_tq;
      if ((rc = eval_rhs(ctx, p, npad, 0, e))) return rc;
      if ((rc = read_scalars(1))) return rc;
      res->max_torque = bits_to_double(ctx->hscal[0]);
      res->rhs_calls = 1;
    }
    // Small problems: an attempted step costs tens of microseconds, of which the host round trip of the
    // controller (16-byte read + synchronisation + relaunch) is a large part.  The controller then runs on
    // the device (DpState, demag.cu): one attempted step is a fixed sequence of launches replayed from a
    // CUDA graph, and the host looks at the state every kLook attempts.  Attempts replayed after the run
    // has ended do nothing (their kernels see active == 0), but still stream the tensor: hence small n only.
    // Tensor resident in shared memory (resident.cu): the whole attempt loop, controller included, runs in
    // a cooperative kernel, kResAttempts attempted steps per launch (the kernel returns early when the run ends).
    const int res_mode = (p->N && !p->N_sparse && !p->N_sym && !sh && round_up(n, p->dtype == MT_F32 ? 4 : 2) <= p->ld)
                             ? mt_resident_fits(ctx, p->dtype, n, p->ld, batch, MT_DP45) : MT_RES_NONE;
    const bool res_ok = res_mode != MT_RES_NONE;
    if (ctx->resident_mode == 2 && !res_ok)
      return mt_fail(ctx, MT_ERR_INVALID_ARG, "resident DP45 required (mt_set_resident_mode 2) but the problem does not qualify "
                     "(dense unsharded tensor that fits in the SMs' shared memory)");
    const bool use_res = res_ok && ctx->resident_mode != 1 && ctx->step_control != 1;
    const bool use_dev = use_res || (!sh && (ctx->step_control == 2 || (ctx->step_control == 0 && n <= 8192)));
    if (use_dev) {
      if (!ctx->dp_dev) {
        MT_CUDA_OK(ctx, cudaMalloc((void**)&ctx->dp_dev, sizeof(DpState)));
        MT_CUDA_OK(ctx, cudaMallocHost((void**)&ctx->dp_host, sizeof(DpState)));
      }
      DpState* S = ctx->dp_dev;
      DpState* Hs = ctx->dp_host;
      memset(Hs, 0, sizeof(*Hs));
      Hs->t = t; Hs->dt = dt; Hs->t_end = o->t_end; Hs->t0 = t0; Hs->sample_dt = o->sample_dt;
      Hs->rtol = o->rtol; Hs->atol = o->atol; Hs->torque_tol = o->torque_tol; Hs->max_torque = res->max_torque;
      Hs->max_steps = o->max_steps; Hs->sample_cap = sample_cap; Hs->has_samples = samples != nullptr;
      Hs->next_sample = 1; Hs->rhs_calls = 1; Hs->status = MT_DP_RUN;
      MT_CUDA_OK(ctx, cudaMemcpyAsync(S, Hs, sizeof(DpState), cudaMemcpyHostToDevice, st));
      auto attempt = [&]() -> int {
        int r;
        if ((r = mt_launch_dp_begin(ctx, S))) return r;
        EpiArgs e = base;  // y2 = m + h a21 k1
        e.do_comb = 1; e.ncomb = 1; e.kptr[0] = k[0]; e.coef[0] = DP_A[1][0]; e.base = m;
        e.h_dev = &S->h; e.active_dev = &S->active; e.y_out = ya;
        e.M_out = has_demag(p) ? ctx->Mst[1] : nullptr;
        if ((r = mt_launch_combine(ctx, e))) return r;
        int src = 1;
        double* yin = ya;
        double* yout = yb;
        for (int sg = 1; sg <= 5; ++sg) {
          e = base;
          e.y = yin; e.k_out = k[sg];
          e.do_comb = 1; e.ncomb = sg + 1;
          for (int j = 0; j <= sg; ++j) { e.kptr[j] = k[j]; e.coef[j] = DP_A[sg + 1][j]; }
          e.base = m; e.h_dev = &S->h; e.active_dev = &S->active; e.y_out = yout;
          e.M_out = has_demag(p) ? ctx->Mst[src ^ 1] : nullptr;
          if ((r = eval_rhs(ctx, p, npad, src, e))) return r;
          src ^= 1;
          double* tmp = yin; yin = yout; yout = tmp;
        }
        e = base;  // k7 = f(y7), error estimate, torque, (renormalised) candidate
        e.y = yin; e.k_out = k[6]; e.torque_bits = &S->tq_bits;
        e.nerr = 7;
        for (int j = 0; j < 7; ++j) { e.eptr[j] = k[j]; e.ecoef[j] = DP_E[j]; }
        e.ebase = m; e.atol = o->atol; e.rtol = o->rtol; e.err_bits = &S->err_bits;
        e.h_dev = &S->h; e.active_dev = &S->active;
        e.do_comb = 1; e.ncomb = 0; e.base = yin; e.y_out = mc; e.renorm = o->renormalize;
        if ((r = eval_rhs(ctx, p, npad, src, e))) return r;
        if ((r = mt_launch_dp_decide(ctx, S))) return r;
        if ((r = mt_launch_dp_commit(ctx, S, m, mc, k[0], k[6], sv))) return r;
        if (samples && (r = mt_launch_mean_cond(ctx, S, m, p->vol, batch, n, samples, stride))) return r;
        return MT_OK;
      };
      auto look = [&]() -> int {  // mirror the state; true stop tests of the loop head evaluated here as well
        MT_CUDA_OK(ctx, cudaMemcpyAsync(Hs, S, sizeof(DpState), cudaMemcpyDeviceToHost, st));
        MT_CUDA_OK(ctx, cudaStreamSynchronize(st));
        return MT_OK;
      };
      auto finished = [&]() -> bool {
        if (Hs->status != MT_DP_RUN) return true;
        if (!(Hs->t < Hs->t_end)) return true;
        if (o->torque_tol > 0 && Hs->max_torque <= o->torque_tol) return true;
        if (o->max_steps > 0 && Hs->accepted + Hs->rejected >= o->max_steps) { Hs->status = MT_DP_MAX_STEPS; return true; }
        return false;
      };
      const int kLook = n <= 2048 ? 16 : 8;
      const int kResAttempts = 64;
      cudaGraph_t graph = nullptr;
      cudaGraphExec_t exec = nullptr;
      int64_t graph_launches = 0;
      bool first = true;
      while (use_res && !rc && !finished()) {
        rc = mt_launch_dp45_resident(ctx, res_mode, p->N, p->dtype, n, p->ld, base, S, m, k[0], ya, yb, o->renormalize, samples,
                                     stride, p->vol, ctx->dscal + 8, (unsigned int*)(ctx->dscal + 6), kResAttempts);
        if (!rc) rc = look();
      }
      while (!use_res && !rc && !finished()) {
        if (first) {  // eagerly: sizes the workspaces, which must not be allocated under capture
          first = false;
          if ((rc = attempt())) break;
        } else {
          if (!exec) {
            if (!ctx->cap_stream) MT_CUDA_OK(ctx, cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
            const int64_t l0 = ctx->launches;
            MT_CUDA_OK(ctx, cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
            ctx->stream = ctx->cap_stream;
            const int prof_saved = ctx->prof_on;
            ctx->prof_on = 0;
            const int r = attempt();
            ctx->stream = st;
            ctx->prof_on = prof_saved;
            cudaError_t ce = cudaStreamEndCapture(ctx->cap_stream, &graph);
            graph_launches = ctx->launches - l0;
            ctx->launches = l0;
            if (r) { if (graph) cudaGraphDestroy(graph); return r; }
            MT_CUDA_OK(ctx, ce);
            MT_CUDA_OK(ctx, cudaGraphInstantiate(&exec, graph, 0));
          }
          // near t_end look sooner: replays past the end of the run are wasted launches
          int q_max = kLook;
          const double rem = (Hs->t_end - Hs->t) / Hs->dt;
          if (rem < (double)q_max) q_max = rem > 1.0 ? (int)ceil(rem) : 1;
          for (int q = 0; q < q_max && !rc; ++q) {
            cudaError_t ce = cudaGraphLaunch(exec, st);
            if (ce != cudaSuccess) rc = mt_fail(ctx, MT_ERR_CUDA, "cudaGraphLaunch: %s", cudaGetErrorString(ce));
            ctx->launches += graph_launches;
          }
        }
        if (!rc) rc = look();
      }
      if (exec) cudaGraphExecDestroy(exec);
      if (graph) cudaGraphDestroy(graph);
      if (rc) return rc;
      t = Hs->t;
      res->accepted = Hs->accepted; res->rejected = Hs->rejected; res->rhs_calls = Hs->rhs_calls;
      res->n_samples = Hs->n_samples; res->max_torque = Hs->max_torque; res->dt_last = Hs->dt_last;
      if (Hs->status == MT_DP_MAX_STEPS) status = MT_ERR_MAX_STEPS;
      if (Hs->status == MT_DP_UNDERFLOW) status = MT_ERR_STEP_UNDERFLOW;
      if (Hs->status == MT_DP_NONFINITE) {
        status = MT_ERR_STEP_UNDERFLOW;
        mt_fail(ctx, status, "non-finite error estimate at t = %g", t);
      }
    }
    while (!use_dev && t < o->t_end) {
      if (o->torque_tol > 0 && res->max_torque <= o->torque_tol) break;
      if (o->max_steps > 0 && res->accepted + res->rejected >= o->max_steps) { status = MT_ERR_MAX_STEPS; break; }
      double t_target = o->t_end;
      bool hit_sample = false;
      if (o->sample_dt > 0) {
        const double ts = t0 + (double)next_sample * o->sample_dt;
        if (ts <= t_target) { t_target = ts; hit_sample = true; }
      }
      double h = dt;
      bool clipped = false;
      if (t + h >= t_target) { h = t_target - t; clipped = true; }
      const double h_min = 16.0 * 2.220446049250313e-16 * fmax(fabs(t), fabs(o->t_end));
      if (h <= h_min) {
        if (clipped) {
          t = t_target;
          if (hit_sample) {
            if (samples && res->n_samples < sample_cap) {
              if ((rc = mt_launch_mean(ctx, m, p->vol, batch, n, t, samples + res->n_samples * stride))) return rc;
              res->n_samples++;
            }
            next_sample++;
          }
          continue;
        }
        status = MT_ERR_STEP_UNDERFLOW;
        break;
      }
      // y2 = m + h a21 k1 (k1 is known: no field evaluation to fuse with).  The staged-M buffers
      // alternate: every evaluation reads Mst[src] and stages its successor state into the other one.
      // Ms*m itself is only needed for the very first k1: FSAL supplies k1 afterwards.
      int src = 0;
      {
        EpiArgs e = base;
        e.do_comb = 1; e.ncomb = 1; e.kptr[0] = k[0]; e.coef[0] = DP_A[1][0]; e.base = m; e.h = h;
        void* Md = has_demag(p) ? ctx->Mst[src ^ 1] : nullptr;
        route(e, ya, Md);
        if ((rc = mt_launch_combine(ctx, e)) || (rc = finish(ya, Md))) return rc;
        src ^= 1;
      }
      double* yin = ya;
      double* yout = yb;
      for (int s = 1; s <= 5; ++s) {  // evaluation of k_{s+1} at y_{s+1}, then y_{s+2}
        EpiArgs e = base;
        e.y = yin; e.k_out = k[s];
        e.do_comb = 1; e.ncomb = s + 1;
        for (int j = 0; j <= s; ++j) { e.kptr[j] = k[j]; e.coef[j] = DP_A[s + 1][j]; }
        e.base = m; e.h = h;
        void* Md = has_demag(p) ? ctx->Mst[src ^ 1] : nullptr;
        route(e, yout, Md);
        if ((rc = eval_rhs(ctx, p, npad, src, e)) || (rc = finish(yout, Md))) return rc;
        src ^= 1;
        double* tmp = yin; yin = yout; yout = tmp;
      }
      // yin now holds y7 = the 5th-order solution; k7 = f(y7) with error estimate, torque and the
      // (renormalised) candidate state + its staged M
      MT_CUDA_OK(ctx, cudaMemsetAsync(d_err, 0, 16, st));
      {
        EpiArgs e = base;
        e.y = yin; e.k_out = k[6]; e.torque_bits = d_tq;
        e.nerr = 7;
        for (int j = 0; j < 7; ++j) { e.eptr[j] = k[j]; e.ecoef[j] = DP_E[j]; }
        e.ebase = m; e.atol = o->atol; e.rtol = o->rtol; e.err_bits = d_err; e.h = h;
        e.do_comb = 1; e.ncomb = 0; e.base = yin; e.renorm = o->renormalize;
        route(e, mc, nullptr);  // sharded: the candidate's rows wait in the gather buffer for the verdict
        if ((rc = eval_rhs(ctx, p, npad, src, e))) return rc;
      }
      if ((rc = read_scalars(2))) return rc;
      res->rhs_calls += 6;
      const double err = bits_to_double(ctx->hscal[0]);
      const double tq7 = bits_to_double(ctx->hscal[1]);
      if (!(err == err) || err > 1.79e308) {  // NaN/inf state or slope: no step size can repair it (Q11b)
        res->rejected++;
        status = MT_ERR_STEP_UNDERFLOW;
        mt_fail(ctx, status, "non-finite error estimate at t = %g", t);
        break;
      }
      double fac = err > 0 ? 0.9 * pow(err, -0.2) : 5.0;
      fac = fmin(5.0, fmax(0.2, fac));
      if (err <= 1.0) {
        t = clipped ? t_target : t + h;
        if (sh) { if ((rc = finish(m, nullptr))) return rc; }
        else MT_CUDA_OK(ctx, cudaMemcpyAsync(m, mc, (size_t)sv * sizeof(double), cudaMemcpyDeviceToDevice, st));
        double* tmp = k[0]; k[0] = k[6]; k[6] = tmp;  // FSAL
        res->max_torque = tq7;
        res->accepted++;
        res->dt_last = h;
        if (clipped && hit_sample) {
          if (samples && res->n_samples < sample_cap) {
            if ((rc = mt_launch_mean(ctx, m, p->vol, batch, n, t, samples + res->n_samples * stride))) return rc;
            res->n_samples++;
          }
          next_sample++;
        }
        dt = clipped ? fmax(dt, h * fac) : h * fac;
      } else {
        res->rejected++;
        dt = h * fmin(1.0, fac);
      }
    }
  }
  MT_CUDA_OK(ctx, cudaStreamSynchronize(st));
  res->t = t;
  *t_inout = t;
  if (status == MT_ERR_MAX_STEPS) mt_fail(ctx, status, "max_steps reached at t = %g", t);
  if (status == MT_ERR_STEP_UNDERFLOW && !ctx->err[0]) mt_fail(ctx, status, "step size underflow at t = %g", t);
  return status;
}

}  // extern "C"
