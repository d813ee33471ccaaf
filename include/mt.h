/*
 * mt.h — C-ABI of libmagtile: the data-parallel hot path of MagTense (arxiv 2107.05364) on B200.
 *
 * Citations are `/root/reference/PAPER.md` line numbers + section / equation; formulas the paper
 * only cites (Smith 2010, Nielsen 2019, refs PAPER.md:286-287) are those derived in
 * SURVEY.md Appendix A and restated in DESIGN.md.
 *
 * Conventions (all entry points)
 *  - Return value: 0 (MT_OK) or a negative MT_ERR_* code.  Nothing throws or aborts across the
 *    ABI.  `mt_last_error(ctx)` returns a ctx-owned, NUL-terminated description of the last
 *    failure (valid until the next failing call on that ctx).
 *  - Unless a parameter is documented as HOST, every array pointer is a DEVICE pointer owned by
 *    the caller (e.g. a torch tensor's data_ptr()); the library never frees or retains it beyond
 *    the call.  The library owns only small workspaces inside `mt_ctx` (staged magnetisation,
 *    Runge-Kutta stages, reduction scratch), released by mt_destroy.
 *  - All work is enqueued on the ctx's stream (a `cudaStream_t` passed as void*, e.g.
 *    torch.cuda.current_stream().cuda_stream; NULL = legacy default stream).  Calls are
 *    ASYNCHRONOUS with respect to the host except mt_integrate and the *_host variants, which
 *    synchronise the stream before returning.
 *  - Layouts.  Vectors are structure-of-arrays fp64 `[B][3][n]` (B = batch of independent
 *    magnetisation states, component-major, tile index fastest).  The tensor is six planes
 *    `[6][n_rows][ld]` of MT_F32 or MT_F64 elements in component order xx, xy, xz, yy, yz, zz;
 *    row i = TARGET tile (field point = its centre), column j = SOURCE tile;
 *    ld >= n is the row pitch in elements and must make rows 16-byte aligned (ld % 4 == 0 for
 *    MT_F32, ld % 2 == 0 for MT_F64); the base pointer must be 16-byte aligned.  Index arithmetic
 *    is 64-bit throughout (a plane of n = 65,536 has 2^32 elements).
 *  - There is no CPU fallback: every entry point fails with MT_ERR_CUDA when no device is usable.
 */
#ifndef MT_H_
#define MT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes ------------------------------------------------------------------------------ */
#define MT_OK 0
#define MT_ERR_INVALID_ARG (-1)       /* null / misaligned pointer, ld < n, n <= 0, bad dtype, batch < 1 */
#define MT_ERR_CUDA (-2)              /* launch / allocation failure; text in mt_last_error            */
#define MT_ERR_SINGULAR_GEOMETRY (-3) /* mt_check_status: an assembled block was non-finite (see assembly) */
#define MT_ERR_STEP_UNDERFLOW (-4)    /* DP45 step size fell below 16 ulp of t                          */
#define MT_ERR_MAX_STEPS (-5)         /* integrator hit max_steps before t_end                          */
#define MT_ERR_UNIMPLEMENTED (-6)

/* ---- element types of the stored tensor ("stored as a float (4 byte)") ---------- */
#define MT_F32 0
#define MT_F64 1

/* ---- integrator methods ------------------------------------------------------------------------ */
#define MT_RK4 0  /* classical fixed-step Runge-Kutta (BASELINE.json config 2)                          */
#define MT_DP45 1 /* Dormand-Prince 5(4): "explicit Runge-Kutta (4,5)" PAPER.md:143, "ODE45" :181       */

typedef struct mt_ctx mt_ctx;

/* Create a context bound to CUDA device `device` and stream `cuda_stream` (HOST call).
 * *out receives the handle.  Errors: MT_ERR_INVALID_ARG (out == NULL), MT_ERR_CUDA.              */
int mt_create(mt_ctx** out, int device, void* cuda_stream);

/* Synchronise the stream, free all workspaces and the context.  NULL is accepted.                */
int mt_destroy(mt_ctx* ctx);

/* Description of the last error on this ctx ("" if none).  NULL ctx returns a static string.     */
const char* mt_last_error(const mt_ctx* ctx);

/* Library version string and the SM architecture the kernels were compiled for ("sm_100a").      */
const char* mt_version(void);

/* ---- A0. Tile-geometry buffer ("subdivides the region into N tiles"; PAPER.md:126
 * cuboid or tetrahedron; PAPER.md:27 space-dependent Ms).  DEVICE pointers, caller-owned.         */
typedef struct {
  int64_t n;             /* number of tiles                                                        */
  const int32_t* type;   /* [n]     0 = axis-aligned cuboid, 1 = tetrahedron                       */
  const double* center;  /* [n][3]  evaluation point: cuboid centre / tetrahedron centroid         */
  const double* size;    /* [n][3]  full edge lengths (cuboids; ignored for tetrahedra)            */
  const double* verts;   /* [n][4][3] tetrahedron vertices, any orientation (ignored for cuboids);
                            may be NULL when no tile has type 1                                    */
  const double* Ms;      /* [n]     saturation magnetisation per tile (not used by assembly)       */
} mt_tiles;

/* ---- A1-A3. Analytic assembly of the demagnetisation tensor (Eq. 9 PAPER.md:78;
 * "computed only once, at the beginning of the simulation" PAPER.md:143).
 * Writes rows [row_begin, row_end) : out[c][i - row_begin][j] = N^{c}_{ij}, the field at the
 * centre of tile i of tile j carrying unit uniform magnetisation, H = -N.M, evaluated from the
 * closed forms in fp64 for EVERY pair (no translation-invariance shortcut) and rounded to nearest
 * when dtype == MT_F32.  The band form is the multi-GPU shard unit and lets n = 65,536 be checked
 * in slices.  `out` is [6][row_end-row_begin][ld].
 * status_flag (DEVICE int32, may be NULL): OR-ed with 1 if any block came out non-finite — a
 * target centre lying on a source face or edge segment (genuine singularity, Q8); the
 * caller zeroes it before and reads it after synchronising.
 * Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA.                                                        */
int mt_assemble_tensor(mt_ctx* ctx, const mt_tiles* tiles, int dtype, int64_t row_begin,
                       int64_t row_end, void* out, int64_t ld, int32_t* status_flag);

/* Reads a status flag written by the assembly calls (they are asynchronous and only OR bits into it):
 * synchronises the stream and returns MT_OK when *status_flag (DEVICE int32) is 0,
 * MT_ERR_SINGULAR_GEOMETRY when bit 0 is set (a target centre on a source face or edge: the tensor
 * holds non-finite blocks and must not be used), MT_ERR_INVALID_ARG when only bit 1 is set
 * (mt_assemble_tensor_sym on a mesh that is not one of congruent cuboids).                          */
int mt_check_status(mt_ctx* ctx, const int32_t* status_flag);

/* ---- F2. Far-field-stable assembly (the analytic form's "error at large distances
 * being of the same magnitude as the elements of the tensor itself"; "different
 * approximations for the demagnetization tensor depending on the distance").
 * mode 0 (default): the closed form for every pair — the paper's method; its fp64 relative error per
 *   block grows as ~5e-16 (r/edge)^3 (1e-10 at ~60 edges).
 * mode 1: cuboid sources further than 16 of their longest edges from the target are evaluated as the
 *   Gauss-Legendre quadrature (4^3 points, 3^3 beyond 48 edges) of the point-dipole kernel over the
 *   source volume; per-block relative error <= 1e-11 at every distance.  Tetrahedron sources switch
 *   at 8 of their longest edges to the same integral in collapsed coordinates (5^3 points, 4^3 beyond
 *   24 edges).  Applies to the following mt_assemble_tensor and mt_assemble_tensor_sym calls
 *   of this ctx.
 * Returns MT_OK or MT_ERR_INVALID_ARG.                                                              */
int mt_set_assembly_mode(mt_ctx* ctx, int mode);

/* ---- A4 / A7. Demagnetising field (Eq. 9 PAPER.md:78 with the sign and Ms reading DESIGN.md Q1;
 * "the most time consuming part" PAPER.md:17,122,138; moved to CUDA PAPER.md:145,223):
 *     Hd[b][a][i] = - sum_j sum_c N^{ac}_{ij} Ms[j] m[b][c][j],   i in [0, n_rows)
 * N is [6][n_rows][ld] (n_rows == n for the full tensor; a row band gives the band's field),
 * Ms [n], m [batch][3][n], Hd [batch][3][n_rows], 1 <= batch <= 8.  For MT_F32 the product
 * Ms*m is rounded to fp32 once, products are fp32 and accumulation is fp32 over at most 128
 * consecutive terms per lane then fp64 (Q19); batches of 5..8 states on an MT_F32 tensor run
 * as an error-compensated 3xTF32 tensor-core contraction (operands split hi + lo, three products, fp32
 * accumulation over one tile then fp64: ~2e-7 relative); for MT_F64 everything is fp64.  The
 * reduction order is fixed: results are bitwise reproducible run to run.
 * Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA.                                                        */
int mt_demag_field(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                   const double* Ms, const double* m, int batch, double* Hd);

/* Same operation with HOST vectors: m_host -> device, field, Hd -> Hd_host, stream synchronised
 * before returning (the end-to-end path bench.py times).  N and Ms stay DEVICE pointers (the
 * tensor is assembled on the device and never leaves it).  Pinned host memory recommended.       */
int mt_demag_field_host(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows,
                        int64_t ld, const double* Ms, const double* m_host, int batch,
                        double* Hd_host);

/* ---- F1. Thresholded tensor (section 4.3.1) -------------------------------------
 * "removing all elements of the tensor smaller than a given threshold value ... allows the
 * demagnetization tensor ... to be allocated as a sparse matrix".  Layout ("bitmap
 * rows"): for plane c and target row i, mask[(c*n_rows + i)*nw + w] holds one bit per source column
 * (bit l of word w = column 32 w + l, 1 = kept) and the kept values are packed in column order from
 * vals[row_ptr[c*n_rows + i]].  nw = mt_sparse_mask_words(n) (a multiple of 4; padding words zero).
 * All arrays are DEVICE memory owned by the caller.
 * Optional second index ("index rows"): cols16[k] = source column of vals[k] modulo 65536, written by
 * mt_sparse_index from the bitmap; for n > 65536 the columns fall in panels of 65,536 and
 * panel_ptr[(c*n_rows + i)*(P-1) + q-1] (P = ceil(n/65536)) is the offset into vals at which panel
 * q >= 1 of plane row (c, i) starts (a row's entries are in column order, so a panel is one run).
 * When cols16 is non-NULL the field kernel walks the packed values (coalesced value + 16-bit column
 * loads, gathered M) instead of decoding the bitmap column by column, and mask may be NULL:
 * 6 bytes per kept fp32 entry instead of 4 + 1/8 per DENSE entry, i.e. smaller than the bitmap from
 * X ~ 0.94 and a far cheaper decode at any X.                                 */
typedef struct {
  int64_t n, n_rows;
  int dtype;               /* MT_F32 | MT_F64: element type of vals                                  */
  int64_t nw;              /* mask words per (plane, row)                                            */
  const int64_t* row_ptr;  /* [6*n_rows + 1] offsets into vals (elements); last = number kept        */
  const uint32_t* mask;    /* [6][n_rows][nw]                                                        */
  const void* vals;        /* [row_ptr[6*n_rows]]                                                    */
  const uint16_t* cols16;  /* NULL, or [row_ptr[6*n_rows]] column (mod 65536) of every packed value  */
  const int64_t* panel_ptr; /* n > 65536 with cols16: [6*n_rows][ceil(n/65536) - 1], else NULL         */
} mt_sparse_tensor;

int64_t mt_sparse_mask_words(int64_t n);

/* Threshold value for a fraction X in [0, 1] ("for a threshold of 20% the absolute
 * smallest fifth of the elements larger than zero in the tensor is truncated to zero"): with the
 * non-zero elements of the dense 3n x 3n matrix sorted by absolute value (off-diagonal components,
 * stored once, count twice: DESIGN.md Q20), *tau_host = the element of rank floor(X*count), i.e.
 * the smallest value kept; entries with |v| < tau are the ones removed (ties with tau are kept);
 * +inf when X*count >= count.  *count_host (may be NULL) = number of non-zero elements counted.
 * N is the dense DEVICE tensor [6][n_rows][ld].  Exact (integer radix select on the bit patterns);
 * synchronises the stream.  Errors: MT_ERR_INVALID_ARG (fraction outside [0,1], ...), MT_ERR_CUDA. */
int mt_threshold_value(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                       double fraction, double* tau_host, int64_t* count_host);

/* The same selection fed BAND BY BAND, for a tensor that is never resident as a whole (the memory
 * saving PAPER.md:237 is after: only one row band of the dense tensor and the compressed result are
 * ever held).  One radix digit (11 bits) is fixed per pass; a pass = mt_select_accumulate on every
 * row band of the tensor (any order, any band height: each band is assembled again per pass with
 * mt_assemble_tensor), then one mt_select_advance.  Repeat until st->done; st->tau, st->count then
 * equal what mt_threshold_value returns for the whole tensor (integer histograms: exact).  The first pass
 * fixes 11 bits (every element binned), each later pass up to 20 bits (only the elements carrying the
 * prefix are binned): 2 passes for MT_F32, 4 for MT_F64.
 * hist: DEVICE array of MT_SELECT_HIST_WORDS unsigned 64-bit counters owned by the caller (row-sharded
 * over several GPUs: sum it over the ranks before mt_select_advance).  mt_select_begin and mt_select_accumulate
 * are asynchronous; mt_select_advance synchronises the stream.  Errors: MT_ERR_INVALID_ARG (NULL
 * state / hist, fraction outside [0, 1], bad tensor arguments, accumulate after done), MT_ERR_CUDA. */
#define MT_SELECT_HIST_WORDS (1 << 20)
typedef struct {
  int dtype;
  double fraction;
  int hi;                          /* key bits [hi, 31|63) are fixed to prefix                     */
  unsigned long long prefix, k, count;
  int done;
  double tau;                      /* valid once done (+inf: everything removed)                   */
} mt_select_state;
int mt_select_begin(mt_ctx* ctx, mt_select_state* st, int dtype, double fraction, unsigned long long* hist);
int mt_select_accumulate(mt_ctx* ctx, const mt_select_state* st, const void* N, int64_t n, int64_t n_rows,
                         int64_t ld, unsigned long long* hist);
int mt_select_advance(mt_ctx* ctx, mt_select_state* st, unsigned long long* hist);

/* Compression band by band into ONE n_total-row thresholded tensor: N holds rows [row0, row0+n_rows)
 * of the dense tensor ([6][n_rows][ld]).  mt_sparse_count_band writes the band's kept-entry counts
 * into counts[c*n_total + row0 + i] (DEVICE, [6*n_total + 1]; asynchronous); after every band,
 * mt_sparse_scan turns the counts into row_ptr in place and returns the number of kept entries
 * (synchronises); mt_sparse_fill_band writes the band's bitmap rows and packed values at their
 * places in the whole tensor's mask / vals (asynchronous).  mt_sparse_count / mt_sparse_fill are the
 * single-band case (row0 = 0, n_total = n_rows).  Errors: MT_ERR_INVALID_ARG (NULL pointers, band
 * outside [0, n_total), bad tensor arguments), MT_ERR_CUDA.                                         */
int mt_sparse_count_band(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                         double tau, int64_t row0, int64_t n_total, int64_t* counts);
int mt_sparse_scan(mt_ctx* ctx, int64_t* row_ptr, int64_t n_total, int64_t* nnz_host);
int mt_sparse_fill_band(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                        double tau, int64_t row0, int64_t n_total, const int64_t* row_ptr,
                        uint32_t* mask, void* vals);

/* mt_sparse_fill_band that also (cols16 non-NULL) writes the index rows in the same pass — cols16 and
 * panel_ptr exactly as mt_sparse_index would derive them from the bitmap — and may then leave the
 * bitmap out (mask NULL): the thresholded tensor is held as values + 16-bit columns only.            */
int mt_sparse_fill_index_band(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows,
                              int64_t ld, double tau, int64_t row0, int64_t n_total,
                              const int64_t* row_ptr, uint32_t* mask, void* vals, uint16_t* cols16,
                              int64_t* panel_ptr);

/* The streamed build as two library calls (the band loop and the passes run inside the library; only
 * the allocation of the result, whose size the first call returns, stays with the caller).  Rows
 * [row_begin, row_end) of the tensor of `tiles` (the whole tensor, or a rank's band) are assembled band by
 * band into `band` (DEVICE, [6][band_rows][ld], ld as for mt_assemble_tensor) once per pass.
 *  mt_sparse_stream_count: fraction in [0, 1]: runs the selection passes (one assembly of every band per
 *    radix digit) and writes the threshold to *tau_host; fraction < 0: *tau_host is taken as given.  Then
 *    one more pass counts the kept entries: row_ptr (DEVICE, [6*(row_end-row_begin) + 1]) and *nnz_host.
 *    Row-sharded: the threshold is a property of the WHOLE tensor, so `allreduce` (may be NULL on a
 *    single rank) is called once per selection pass and must sum `hist` (DEVICE, MT_SELECT_HIST_WORDS
 *    64-bit counters, caller-owned; may be NULL when allreduce is NULL) over the ranks in place, enqueued
 *    on cuda_stream.
 *  mt_sparse_stream_fill: one more pass writes mask (may be NULL with cols16), vals, and, when cols16 is
 *    non-NULL, the index rows (cols16, panel_ptr) at their places, as mt_sparse_fill_index_band does.
 * status_flag as in mt_assemble_tensor.  Both synchronise the stream before returning.
 * Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA (also: a non-zero return of allreduce).                    */
typedef int (*mt_allreduce_fn)(void* user, unsigned long long* hist, void* cuda_stream);
int mt_sparse_stream_count(mt_ctx* ctx, const mt_tiles* tiles, int dtype, double fraction, int64_t row_begin,
                           int64_t row_end, void* band, int64_t band_rows, int64_t ld, int64_t* row_ptr,
                           unsigned long long* hist, mt_allreduce_fn allreduce, void* user,
                           int32_t* status_flag, double* tau_host, int64_t* nnz_host);
int mt_sparse_stream_fill(mt_ctx* ctx, const mt_tiles* tiles, int dtype, double tau, int64_t row_begin,
                          int64_t row_end, void* band, int64_t band_rows, int64_t ld, const int64_t* row_ptr,
                          uint32_t* mask, void* vals, uint16_t* cols16, int64_t* panel_ptr,
                          int32_t* status_flag);

/* Compression, two calls: mt_sparse_count fills row_ptr (DEVICE, [6*n_rows+1]) for threshold tau and
 * returns the number of kept entries in *nnz_host (synchronises); the caller allocates mask
 * ([6*n_rows*nw] uint32) and vals ([nnz] of dtype), then mt_sparse_fill writes them (asynchronous).
 * An entry is kept iff it is non-zero and not |v| < tau.                                            */
int mt_sparse_count(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                    double tau, int64_t* row_ptr, int64_t* nnz_host);
int mt_sparse_fill(mt_ctx* ctx, const void* N, int dtype, int64_t n, int64_t n_rows, int64_t ld,
                   double tau, const int64_t* row_ptr, uint32_t* mask, void* vals);

/* Index rows: cols16[row_ptr[c*n_rows+i] + k] = column (mod 65536) of the k-th set bit of the bitmap
 * row (c, i); panel_ptr as described above (may be NULL when n <= 65536).  S->mask and S->row_ptr
 * must be filled (mt_sparse_fill); S->cols16 / S->panel_ptr are ignored; cols16 is a DEVICE array of
 * row_ptr[6*n_rows] uint16, panel_ptr of 6*n_rows*(ceil(n/65536)-1) int64.  Asynchronous.          */
int mt_sparse_index(mt_ctx* ctx, const mt_sparse_tensor* S, uint16_t* cols16, int64_t* panel_ptr);

/* mt_demag_field on the thresholded tensor: Hd[b][a][i] = - sum over kept entries; same arithmetic
 * rules (fp32 runs of at most 96 terms per lane, 64 on index rows, then fp64), fixed reduction order. */
int mt_demag_field_sparse(mt_ctx* ctx, const mt_sparse_tensor* S, const double* Ms, const double* m,
                          int batch, double* Hd);

/* ---- F3. Pair-symmetric half storage ("MagTense utilizes the fact that the tensor is
 * symmetric ... reducing the scaling to ... almost N^2/2").  On a mesh of CONGRUENT axis-aligned
 * cuboids N_ij = N_ji (the block depends on c_i - c_j only and is even in it), so only blocks with
 * j >= i are kept, at tile granularity, and each serves two rows of the product: half the bytes per
 * evaluation.  `data` is a DEVICE array of mt_sym_tensor_elems(n, dtype) elements in the tiled layout
 * described in csrc/sym_layout.cuh (row blocks of 32, column tiles of 128 fp32 / 64 fp64, order of
 * the kernel's loads), written by mt_assemble_tensor_sym only.                                     */
typedef struct {
  int64_t n;
  int dtype;         /* MT_F32 | MT_F64 */
  const void* data;
} mt_sym_tensor;

int64_t mt_sym_tensor_elems(int64_t n, int dtype);

/* Assembles the kept half (every kept pair's closed form, fp64 arithmetic, rounded for MT_F32).
 * status_flag (DEVICE int32, may be NULL) is OR-ed with 1 for a non-finite block and with 2 if any
 * tile is not a cuboid (type 0) of the same size as tile 0 — the result must then not be used.
 * Asynchronous.  Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA.                                          */
int mt_assemble_tensor_sym(mt_ctx* ctx, const mt_tiles* tiles, int dtype, void* out,
                           int32_t* status_flag);

/* mt_demag_field from the half: Hd[b][a][i] for all n rows; same arithmetic rules (fp32 runs of at
 * most 96 terms, then fp64), fixed reduction order.  States of a batch are evaluated one after the
 * other (each streams the half once).                                                              */
int mt_demag_field_sym(mt_ctx* ctx, const mt_sym_tensor* S, const double* Ms, const double* m,
                       int batch, double* Hd);

/* ---- 8(e). Row sharding over several GPUs (one process and one mt_ctx per GPU) --------------------
 * The tensor shards by TARGET rows (every pair is independent): rank g of `world`
 * assembles and keeps rows [g n / world, (g+1) n / world) (integer division) — the row band of
 * mt_assemble_tensor — and evaluates the right-hand side of those rows.  Every evaluation needs the
 * whole state on every rank ("RHS -> dense product -> LL"), so each Runge-Kutta
 * stage ends with ONE exchange: the all-gather of the ranks' slices of the next stage state; DP45's
 * error norm and the torque test add one max-reduction of two scalars per step.  The library does not
 * link a communication layer: the caller supplies `exchange`, called on the host between kernels,
 * which must ENQUEUE the collective on `cuda_stream` (the ctx's stream) and return 0, or non-zero on
 * failure (-> MT_ERR_CUDA):
 *   what == MT_XCHG_GATHER_STATE: all-gather `pack` IN PLACE over the ranks.  pack is
 *     [world][batch][3][slice_pad] doubles; the fused epilogue has written rank `rank`'s block (its
 *     rows' components of the next state, rows beyond the band's length unspecified); on completion
 *     every rank holds every block (ncclAllGather / all_gather_into_tensor with the rank's block as
 *     the send buffer).  The library then scatters the blocks into the full state and the staged M.
 *   what == MT_XCHG_MAX_SCALARS: element-wise MAX over the ranks of the two 64-bit words of `scal`
 *     (bit patterns of non-negative doubles or the canonical quiet NaN 0x7ff8000000000000: they order
 *     like signed or unsigned 64-bit integers), result on every rank.
 * All ranks must make the same calls with the same arguments (the host-side step controller then
 * takes the same decisions everywhere).  pack, scal: DEVICE memory owned by the caller, at least
 * world*batch*3*slice_pad doubles and 2 words; slice_pad >= the longest band, equal on all ranks.   */
#define MT_XCHG_GATHER_STATE 0
#define MT_XCHG_MAX_SCALARS 1
typedef int (*mt_exchange_fn)(void* user, int what, void* cuda_stream);
typedef struct {
  int rank, world;
  int64_t slice_pad;
  double* pack;
  unsigned long long* scal;
  mt_exchange_fn exchange;
  void* user;
} mt_shard;

/* ---- A5 / A6. Effective field and Landau-Lifshitz right-hand side ------------------------------
 * H_eff = H_d + H_exch + H_anis + H_a                                   (Eq. 17)
 *   H_exch,i = c_ex,i * sum_{dir} (m_{i+} - 2 m_i + m_{i-}) * inv_d2[dir]   (Eq. 12 PAPER.md:94;
 *              3-point stencil PAPER.md:181; a missing neighbour (-1) is replaced by m_i:
 *              Neumann, Eq. 3)
 *   H_anis,i = c_an,i (m_i . e_i) e_i                                    (Eq. 16)
 *   H_a                                                                   (Eq. 7,  PAPER.md:70)
 * dm/dt = -gamma m x H_eff - alpha_ll m x (m x H_eff)                    (Eq. 1,  PAPER.md:33)
 * gamma and alpha_ll are the two prefactors exactly as written in Eq. 1 (Q5).
 * A NULL array pointer selects the scalar / constant beside it; nbr == NULL disables exchange;
 * N == NULL disables the demagnetising term.  The tensor must be square here (n rows) unless
 * `shard` is set: N (or N_sparse) then holds the rank's row band only, m and every per-tile array stay
 * full-size on every rank, mt_llg_rhs writes the band's rows of dmdt / Heff (at their global
 * positions; other rows untouched) and mt_integrate advances the whole state with one exchange per
 * stage.  mt_energy, mt_field_sweep and N_sym do not take a sharded problem (MT_ERR_INVALID_ARG).  */
typedef struct {
  int64_t n;
  const void* N;         /* [6][n][ld] or NULL                                                     */
  int dtype;             /* MT_F32 | MT_F64                                                        */
  int64_t ld;
  const double* Ms;      /* [n]                                                                    */
  const int32_t* nbr;    /* [n][6]  -x,+x,-y,+y,-z,+z neighbour index or -1; NULL = no exchange    */
  double inv_d2[3];      /* 1/dx^2, 1/dy^2, 1/dz^2                                                 */
  const double* c_ex;    /* [n] 2A/(mu0 Ms) per tile, or NULL -> c_ex_scalar                       */
  double c_ex_scalar;
  const double* c_an;    /* [n] 2K/(mu0 Ms) per tile, or NULL -> c_an_scalar                       */
  double c_an_scalar;
  const double* easy;    /* [n][3] unit easy axes, or NULL -> easy_const                           */
  double easy_const[3];
  const double* H_a;     /* [n][3] applied field, or NULL -> H_a_const                             */
  double H_a_const[3];
  double gamma, alpha_ll;
  const double* vol;     /* [n] tile volumes: weights of <m> (A10); NULL = plain mean              */
  const mt_sparse_tensor* N_sparse; /* HOST pointer or NULL: when set, the demagnetising term uses this
                            thresholded tensor (F1) instead of N (N may then be NULL)  */
  const mt_sym_tensor* N_sym; /* HOST pointer or NULL: demagnetising term from the pair-symmetric half
                            (F3); takes precedence over N, after N_sparse                            */
  const mt_shard* shard; /* HOST pointer or NULL: row-sharded problem (section 8(e) above)           */
} mt_problem;

/* dmdt[b][3][n] (required) and Heff[b][3][n] (optional, NULL to skip) for m[b][3][n].
 * Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA.                                                        */
int mt_llg_rhs(mt_ctx* ctx, const mt_problem* prob, const double* m, int batch, double* dmdt,
               double* Heff_or_null);

/* ---- A8-A10. Time integration ("explicit Runge-Kutta (4,5)" PAPER.md:143; RK4 per BASELINE
 * config 2; observables <m>(t) as plotted in Fig. 6).                               */
typedef struct {
  int method;            /* MT_RK4 | MT_DP45                                                       */
  double dt;             /* RK4: the step; DP45: initial step (<= 0: 1e-3)                         */
  double t_end;
  int64_t max_steps;     /* <= 0: unlimited                                                        */
  double rtol, atol;     /* DP45: err = max |e| / (atol + rtol max(|m|, |m_new|)), accept if <= 1  */
  double torque_tol;     /* stop when max_i |m_i x H_eff,i| <= torque_tol (Eq. 2);
                            <= 0: off                                                              */
  int renormalize;       /* 1: m_i <- m_i/|m_i| after every (accepted) step (Q10)        */
  int64_t sample_every;  /* RK4: write a sample every k steps (0: never)                           */
  double sample_dt;      /* DP45: land exactly on t0 + k*sample_dt and sample there (0: never)     */
} mt_integrator_opts;

typedef struct {
  int64_t accepted, rejected, rhs_calls, n_samples;
  double t, dt_last;
  double max_torque;     /* max_i |m_i x H_eff,i| of the last evaluation that measured it.  RK4 with
                            torque_tol > 0: at the state the last examined step STARTED from (the
                            stop test runs before a step is taken; the state returned at t_end has
                            not been tested); RK4 with torque_tol <= 0: 0 (not measured).  DP45: at
                            the stage-7 state of the last accepted step, before its renormalisation
                            (Q10b)                                                        */
} mt_integrator_result;

/* Advance m_inout[batch][3][n] (DEVICE) from *t_inout (HOST) towards opts->t_end.  All states of
 * the batch share the step sequence.  samples (DEVICE, may be NULL) is [sample_cap][1+3*batch]:
 * t, then <m_x>,<m_y>,<m_z> per state.  host_out (HOST) receives the counters.  Synchronises the
 * stream before returning.  Resumable: (m, t, dt_last) is the whole state.
 * Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA, MT_ERR_STEP_UNDERFLOW (DP45: the step fell below
 * 16 eps max(|t|, |t_end|), or the error estimate is not finite — a NaN/inf in the state or in the
 * tensor reaches it, Q11b), MT_ERR_MAX_STEPS (the state reached so far is still written
 * back).  A tile with m_i = 0 stays at zero under renormalisation (Q10c).                */
int mt_integrate(mt_ctx* ctx, const mt_problem* prob, const mt_integrator_opts* opts,
                 double* m_inout, int batch, double* t_inout, double* samples, int64_t sample_cap,
                 mt_integrator_result* host_out);

/* ---- F4. Energy terms and the field-sweep (hysteresis) loop -------------------------------------
 * Free energy of Eq. 4 split into its terms, each evaluated through the field it
 * generates, for state b (Ms_i V_i weights; V = prob->vol, NULL: 1):
 *   E_out[b][0] = -(1/2) sum_i Ms_i V_i m_i . H_d,i      demagnetisation, Eq. 8
 *   E_out[b][1] = -(1/2) sum_i Ms_i V_i m_i . H_exch,i   exchange,        Eq. 11
 *   E_out[b][2] = -(1/2) sum_i Ms_i V_i m_i . H_anis,i   anisotropy,      Eq. 15 (up to its
 *                                                         m-independent constant)
 *   E_out[b][3] = -      sum_i Ms_i V_i m_i . H_a,i      Zeeman,          Eq. 6
 *   E_out[b][4] = their sum.
 * In units of mu0 x (field unit)^2 x (length unit)^3.  One pass of the fused field kernel (same
 * arithmetic as mt_llg_rhs) and a fixed-order reduction: bitwise reproducible.  E_out is a DEVICE
 * array [batch][5]; asynchronous.  Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA.                        */
int mt_energy(mt_ctx* ctx, const mt_problem* prob, const double* m, int batch, double* E_out);

/* The loop of the paper's hysteresis experiment (mumag standard problem 2: "the
 * applied field is changed in steps" and the system relaxed at each): for f = 0 .. n_fields-1 the
 * uniform applied field is set to fields_host[f][0..2] (HOST array; prob->H_a must be NULL),
 * m_inout is integrated with `opts` from t = 0 to opts->t_end (or to opts->torque_tol) starting
 * from the previous field's end state, and row f of `rows` (DEVICE, [n_fields][batch][8]) receives
 * <m_x>, <m_y>, <m_z>, E_demag, E_exch, E_anis, E_zeeman, E_total of every state.  res_host (HOST,
 * may be NULL) receives the counters summed over the sweep (t = total simulated time).
 * Synchronises the stream before returning.  MT_ERR_MAX_STEPS from a field step is not fatal (the
 * sweep continues, as the paper relaxes a fixed time per field) and is returned at the end only if
 * it was the last step's status.  Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA, MT_ERR_STEP_UNDERFLOW.  */
int mt_field_sweep(mt_ctx* ctx, const mt_problem* prob, const mt_integrator_opts* opts,
                   const double* fields_host, int64_t n_fields, double* m_inout, int batch,
                   double* rows, mt_integrator_result* res_host);

/* ---- instrumentation --------------------------------------------------------------------------- */
/* Number of kernels this ctx has launched since creation (bench.py's gpu_launches).              */
int64_t mt_launch_count(const mt_ctx* ctx);

/* Per-kernel timing for the roofline (bench.py): between mt_profile_begin and mt_profile_end every
 * launch of the demag field kernel (the dominant kernel of A4-A7; for small n its fixed-order second
 * pass is included) is bracketed by CUDA events recorded on the ctx's stream, at most 1024 launches
 * (later ones are not timed).  mt_profile_end synchronises the stream and returns the summed device
 * time in milliseconds and the number of launches timed (HOST pointers).  Not for use while a CUDA
 * graph is being replayed by mt_integrate (captured launches are not bracketed).
 * Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA.                                                         */
int mt_profile_begin(mt_ctx* ctx);
int mt_profile_end(mt_ctx* ctx, double* total_ms, int64_t* launches);

/* Roofline denominators measured in place (bench.py; north_star: "assembly tile-pairs/s against
 * FP64/FP32 pipe peak", "achieved HBM GB/s against B200 peak").  Runs a microbenchmark kernel on the
 * ctx's stream four times (first = warm-up) and returns the best of the other three:
 *   out_host[0] = rate, out_host[1] = the kernel's duration in ms (HOST array of 2 doubles).
 *   MT_PEAK_DFMA      FP64 fused multiply-adds, thread-instructions per second, all SMs
 *   MT_PEAK_FFMA      FP32 fused multiply-adds (three-register FFMA), thread-instructions per second
 *   MT_PEAK_FFMA2     packed fma.rn.f32x2, thread-instructions per second (each = 2 FMAs)
 *   MT_PEAK_MMA_TF32  warp-level mma.sync m16n8k8 tf32 (fp32 accumulate), multiply-adds per second
 *   MT_PEAK_HBM_READ  read-only stream of buf[0..bytes) (DEVICE, 16-byte aligned, >= 32 KB per SM,
 *                     should exceed the L2 several times) by 1-D bulk copies into shared memory,
 *                     bytes per second; buf/bytes are ignored by the other kinds.
 * Synchronous.  Not part of the compute path.  Errors: MT_ERR_INVALID_ARG, MT_ERR_CUDA.            */
#define MT_PEAK_DFMA 0
#define MT_PEAK_FFMA 1
#define MT_PEAK_FFMA2 2
#define MT_PEAK_MMA_TF32 3
#define MT_PEAK_HBM_READ 4
int mt_measure_peak(mt_ctx* ctx, int kind, const void* buf, int64_t bytes, double* out_host);

/* Where the DP45 step controller runs (A9).  0 (default): on the device for problems of at most 8,192
 * tiles that are not row-sharded — an attempted step is then a fixed launch sequence replayed from a CUDA
 * graph, the accept / reject decision, the next step size, the clipping to sample times and the stop
 * tests are taken by a one-thread kernel, and the host reads the controller state every 8 or 16 attempts
 * (attempts replayed after the end of the run do nothing) — and on the host otherwise (one 16-byte read
 * per attempted step: invisible once a step takes milliseconds).  1: always on the host.  2: always on
 * the device (not for row-sharded problems, which stay on the host).  Both follow the same rules
 * (Q11/Q11b); the device evaluates err^(-1/5) with CUDA's pow, the host with the C library's,
 * so the two step sequences can differ in the last bit of dt.
 * Returns MT_OK or MT_ERR_INVALID_ARG.                                                              */
int mt_set_step_control(mt_ctx* ctx, int mode);

/* RK4 (A8) and DP45 (A9) with the tensor resident in shared memory.  A dense, unsharded problem whose
 * n x n x 6 tensor fits in the shared memory of the device's SMs together (one CTA per SM holding
 * ceil(n / SMs) <= 8 rows of the six planes, plus the stage states: N <= ~740 tiles fp64, ~1,020 fp32 on a
 * B200 — the sizes the paper runs) is integrated by a COOPERATIVE kernel: a chunk of RK4
 * steps, or up to 64 attempted DP45 steps, per launch.  The tensor is read once per launch; every stage
 * reads the stage state of all tiles from L2, multiplies the resident rows with Ms*m, adds
 * exchange, anisotropy and the applied field and forms the Landau-Lifshitz right-hand side and the next
 * stage state with the row's constants, the step's start state and the slopes in
 * registers, and ends at a grid barrier; no launch between right-hand sides.  DP45: the step controller
 * (the rules of mt_set_step_control's device controller) runs inside the kernel as well — every CTA takes
 * the same decision from the grid-wide error / torque maxima — and the host reads the controller state
 * once per launch.
 * A tensor too large for that but of at most 100 MB (it stays in the 126 MB L2 between right-hand sides: up to
 * ~2,000 tiles fp32, ~1,450 fp64) runs the same persistent kernels with the CTA's rows (at most 32) read from
 * L2 at every stage instead of from shared memory; everything else — stage state, epilogue, barrier,
 * controller — is unchanged.
 * mode 0 (default): used whenever the problem qualifies (DP45: unless mt_set_step_control(ctx, 1) keeps
 * the controller on the host); 1: never (per-stage launches, replayed from a CUDA graph); 2: required —
 * mt_integrate fails with MT_ERR_INVALID_ARG when the problem does not qualify.  Same arithmetic per term
 * as the streaming kernels (fp32 tensors: fp32 products and partial sums, then fp64), another summation
 * order: RK4 trajectories agree to rounding (1e-11 on fp64 tensors), DP45 takes the same accept / reject
 * sequence with step sizes equal to ~1e-10; deterministic.  Sampling, the stop tests and the result
 * counters behave as in the other paths.  Returns MT_OK or MT_ERR_INVALID_ARG.                         */
int mt_set_resident_mode(mt_ctx* ctx, int mode);

/* Tuning / A-B testing hook: selects the demag kernel variant (0 = default choice by shape,
 * 1 = register-streaming LDG kernel, 2 = TMA bulk-tensor pipeline, 3 = as 2 but batches of 5..8
 * states on fp32 tensors use the packed-FFMA2 kernel instead of the tensor-core one).  Returns MT_OK or
 * MT_ERR_INVALID_ARG.  Results of all variants agree to rounding; each is deterministic.          */
int mt_set_demag_variant(mt_ctx* ctx, int variant);

/* ---- Demagnetising field without any allocation (for callers that cannot call cudaMalloc: code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it).  Same operation as mt_demag_field
 * for ONE state (Eq. 9, sign and Ms reading DESIGN.md Q1; the arithmetic of DESIGN.md Q19):
 *     Hd[a][i] = - sum_j sum_c N^{ac}_{ij} Ms[j] m[c][j],   i in [0, n_rows)
 * N [6][n_rows][ld], Ms [n], m [3][n], Hd [3][n_rows]: DEVICE memory of `device`, owned by the caller;
 * `cuda_stream` is a cudaStream_t of that device (NULL = legacy default stream); the call only enqueues
 * work on it and does not synchronise.  No mt_ctx is involved (mt_create allocates), and the call makes no
 * cudaMalloc / cudaFree / allocating library call: the staged vector Ms*m (tensor dtype) and the partial
 * row sums of the column splits live in a file-scope __device__ array of MT_NOALLOC_SCRATCH_BYTES that every
 * GPU which loads the library holds until the process exits.  Limits: n <= MT_NOALLOC_MAX_N and
 * n_rows <= MT_NOALLOC_MAX_N; anything larger is rejected with MT_ERR_INVALID_ARG (use mt_demag_field).
 * The scratch array is SHARED by every call on a device and keeps the last call's contents: each call
 * rewrites every word it later reads (the staging kernel also zeroes the padding of the staged vector),
 * so calls in stream order are independent of one another, but two calls that overlap on the GPU (different
 * streams without an ordering between them, or two host threads) RACE on it — serialise them.
 * The first call on a device looks the array's device address up (cudaGetSymbolAddress, once per device;
 * this loads the module): make one call outside a graph capture first.  The current device of the calling
 * thread is left as it was.  The reduction order is fixed (bitwise reproducible for a given shape).
 * `err` (may be NULL) is a caller-provided HOST buffer of err_cap bytes that receives the error text.
 * Returns MT_OK, MT_ERR_INVALID_ARG (null / misaligned pointer, ld < n, size over the limit, bad dtype or
 * device) or MT_ERR_CUDA.                                                                          */
#define MT_NOALLOC_MAX_N 65536
#define MT_NOALLOC_SCRATCH_BYTES (4718592) /* 4.5 MiB: 1.5 MiB staged vector + 3 MiB partial sums */
int mt_demag_field_noalloc(int device, void* cuda_stream, const void* N, int dtype, int64_t n, int64_t n_rows,
                           int64_t ld, const double* Ms, const double* m, double* Hd, char* err,
                           int64_t err_cap);

#ifdef __cplusplus
}
#endif
#endif /* MT_H_ */
