/*
 * ttdft.h -- C ABI of the B200-native Chebyshev filter of ChFSI (TTDFT, arXiv 2110.15853).
 *
 * The library implements ONE thing: step 1 of Algorithm 1, the degree-m scaled
 * three-term Chebyshev recurrence whose every step multiplies the sparse symmetric Kohn-Sham
 * Hamiltonian H (M x M, localized Tucker tensor basis) by a dense block of
 * wavefunctions X (M x N_orb), plus the bare product it is made of.
 *
 * Conventions (all calls):
 *   - All matrices are fp64.  X, Y, ... are ROW-MAJOR M x ncols with a leading dimension (in
 *     elements) ld >= ncols.  Indices are 0-based int32.
 *   - Unless a parameter is documented as HOST, every data pointer is a DEVICE pointer owned by the
 *     caller.  The library allocates no device memory: the converted H lives in the caller's
 *     `dev_storage`, scratch panels in the caller's `work`.
 *   - `stream` is a CUDA stream handle (cudaStream_t / CUstream) passed as void*; NULL = the legacy
 *     default stream.  Work is enqueued on it and the call returns without synchronising, except
 *     where stated.
 *   - Every call returns a ttdft_status.  On a non-OK status no output has been modified, and
 *     ttdft_last_error() returns a thread-local message.  Nothing throws or aborts.
 *   - H is used AS STORED (both triangles present); symmetry is a promise that is only checked on
 *     request, and results are defined for a non-symmetric H too.
 *   - "X must not overlap Y" means the two views share no element.  Column views of one wide row-major
 *     buffer (X = B[:, :n], Y = B[:, n:2n], same leading dimension) do not overlap.
 *
 * Environment variables (every switch the library reads; none is needed for normal use).  They are read
 * at two points only: by ttdft_h_build, into the handle (which is immutable afterwards), and at the entry
 * of the handle-less calls ttdft_gram / ttdft_rotate / ttdft_orthonormalize (and ttdft_project's Gram
 * product).  Do not change them from another thread while such a call runs (getenv is not safe against
 * a concurrent setenv).
 *   TTDFT_MATH        0..3: initial math mode of a handle (TTDFT_MATH_*); default 0 = AUTO.
 *   TTDFT_K3_CLUSTER  1, 2, 4 or 8: force the CTA-cluster size of the int8 step kernel; default: chosen per launch.
 *   TTDFT_K3_L2HINTS  0, 1 or 2: L2 eviction hints of the int8 step kernel's TMA loads (0 none, 1 evict-first
 *                     H planes + evict-last Y digit tiles, 2 only the latter); default: chosen per launch.
 *   TTDFT_K3_T        0 or 1: int8 step on kernel K3 (rows of the tile on the MMA's M axis) or K3T (transposed: columns of Y on
 *                     M, no padding rows for tiles narrower than 128); default: K3T for 64- and 96-wide tiles, K3 for 128.
 *   TTDFT_K4_CLUSTER  1 or 2: CTA-cluster size of the int8 Gram kernel; default 2.
 *   TTDFT_K3_PREDICT_BIAS  test hook, -64..8, default 0: added to every predicted column exponent of the filter's int8
 *                     path (negative: predictions fail and the fallback extraction runs; positive: digits lose that many bits).
 *                     Unlike the others this one changes results in the last bits (always inside the documented error bound).
 *   TTDFT_DEBUG       non-zero: print launch decisions to stderr.
 * All others select between code paths that give bit-identical results.
 */
#ifndef TTDFT_H
#define TTDFT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ttdft_h_s* ttdft_h_t; /* opaque handle, host object owned by the library */

typedef enum {
  TTDFT_OK = 0,
  TTDFT_ERR_INVALID_ARG = 1,
  TTDFT_ERR_UNSUPPORTED = 2,
  TTDFT_ERR_WORKSPACE_TOO_SMALL = 3,
  TTDFT_ERR_NOT_SYMMETRIC = 4,
  TTDFT_ERR_CUDA = 5,
  TTDFT_ERR_BREAKDOWN = 6 /* ttdft_orthonormalize: X^T X not positive definite (dependent columns) */
} ttdft_status;

typedef enum { TTDFT_FMT_CSR = 0, TTDFT_FMT_BSR = 1, TTDFT_FMT_HYBRID = 2 } ttdft_format;

/* flags for ttdft_h_desc.flags */
#define TTDFT_CHECK_SORTED 1u   /* verify indices in range, ascending and unique per row (synchronises) */
#define TTDFT_CHECK_SYMMETRY 2u /* verify H == H^T bit for bit (synchronises; needs sorted columns)      */
#define TTDFT_FORCE_GENERIC 4u  /* keep the input format and use the generic row-per-warp kernel          */
#define TTDFT_NO_I8 8u          /* do not build the int8 digit planes (saves 0.875x of the tile bytes)    */
#define TTDFT_PACKED 32u        /* also build the PACKED copy of the tiles (per 16-column slab: row offsets, bit masks, non-zero
                                 * values: 0.65x of the dense tile bytes at 40 % zeros); products with ncols <= 16 then stream it
                                 * instead of the dense tiles.  A storage variant for memory-tight handles, NOT a speed-up on
                                 * B200: the fp64 tensor pipe multiplies the expanded zeros either way and bounds a 16-column
                                 * product at 0.66 ms for config 3, so the dense tiles (0.79 ms) are not far above the bound and
                                 * the decode costs more shared-memory bandwidth than the bytes save (1.04 ms). */
#define TTDFT_OWNED_ROWS_ONLY 16u /* row-partitioned H: this handle holds only the block rows (CSR: rows)
                                   * one rank owns; rows without any entry belong to another rank, and ttdft_spmm / ttdft_cheb_step
                                   * (and their _ws forms) leave those rows of the output UNTOUCHED instead of writing the result
                                   * for an all-zero row.  Meant for single steps between exchanges (paper_2110_15853_b200/rows.py);
                                   * ttdft_cheb_filter on such a handle never updates the rows it does not own. */

/*
 * Arithmetic of the block-sparse product (every mode returns fp64 results inside north_star's
 * tolerance; DESIGN.md "Kernel K3" has the error bound):
 *   TTDFT_MATH_FP64  fp64 tensor-core MMA (DMMA), fp64 accumulation.
 *   TTDFT_MATH_I8X7  each fp64 operand is split exactly into 7 balanced base-256 digit planes (55 bits
 *                    below the maximum of its H row / Y column; the diagonal of H stays fp64), the
 *                    plane products of significance >= 2^-55 (28 of 49) run on the int8 tensor cores
 *                    with exact int32 accumulation, and the epilogue recombines them in fp64: the
 *                    product's error bound is below that of an fp64 dot product.  Needs scratch for the
 *                    digit planes of one iterate, so it is used by the calls that take `work`.
 *   TTDFT_MATH_I8    the same with the leading 6 planes (47 bits, 21 plane products): ~1.3x faster,
 *                    error ~1e-14 per product, still 100x inside north_star's 1e-12.
 *   TTDFT_MATH_AUTO  I8X7 where it is faster than FP64 (tile size >= 64 and digit planes built), else FP64.
 */
#define TTDFT_MATH_AUTO 0
#define TTDFT_MATH_FP64 1
#define TTDFT_MATH_I8 2
#define TTDFT_MATH_I8X7 3

/*
 * Description of the input Hamiltonian (PAPER.md:L199-205 H^L; L250-252 block structure: "the
 * diagonal blocks are much denser compared to the off-diagonal blocks").
 *   CSR: row_ptr[M+1], col_idx[nnz] ascending and unique per row, values[nnz]; explicit zeros are
 *        allowed and treated as values.  nnz < 2^31.
 *   BSR: row_ptr[M/block+1], col_idx[nblocks] block columns ascending per block row,
 *        values[nblocks*block*block], each block a row-major block x block tile.  M % block == 0.
 *   subdomain_of_row (CSR only, optional, may be NULL): subdomain label of every row.  If every subdomain
 *        owns the same number b of rows, b in {32, 64, 96, 128}, the builder groups each localized
 *        subdomain's basis functions into b x b tiles (block-sparse storage).  Three label layouts qualify:
 *        (1) rows already grouped: labels strictly increasing from group to group (any integers);
 *        (2) rows in ANY order: labels are the subdomain indices 0 .. M/b-1.  The builder then REORDERS:
 *            reordered row L*b + r is the r-th row (in input order) labelled L, H is stored as the tiles of
 *            P H P^T, and the handle keeps the row map.  The caller never sees the reordering: X and Y stay
 *            in the caller's row order; ttdft_cheb_filter gathers each X panel into tile order once, runs
 *            all m steps there, and scatters the result (two extra passes per panel, no extra scratch).
 *            Single steps on such a handle: ttdft_*_ws gather/scatter through scratch; the calls without
 *            scratch run the generic kernel through the row map.
 *        (3) subdomains of UNEQUAL size (the real TTDFT basis: ranks differ per subdomain): labels are the
 *            subdomain indices 0 .. nb-1 without gaps, rows in any order, every subdomain with 1 .. 128 rows.  Every subdomain is
 *            padded with zero rows and columns to one tile size b (the smallest of 32/64/96/128 that holds the largest one)
 *            unless that more than doubles the rows; the handle then works in a tile-order space of nb*b rows behind the
 *            same row map as (2) (ttdft_cheb_filter needs a second scratch panel: ask ttdft_cheb_filter_work_bytes).
 *        Otherwise the CSR is kept as is.
 *   HYBRID: the paper's own layout (Sec. 4.1, Fig. 3: "the diagonal blocks and the off-diagonal blocks of the
 *        Hamiltonian matrix are stored as dense and sparse matrices"): diag_values holds the dense diagonal blocks H^(D) -- block k
 *        covers rows and columns [k*diag_block, min((k+1)*diag_block, M)), row-major with leading dimension diag_block at offset
 *        k*diag_block^2 (ceil(M/diag_block) blocks; what lies beyond M in the last one is ignored) -- and row_ptr / col_idx /
 *        values a CSR (as above) of H^(OD), the entries OUTSIDE those blocks.  subdomain_of_row applies as for CSR.  The library
 *        does not keep the two-part layout: zeros of the dense blocks are dropped, and the union goes into the tile format
 *        (labels usable; tiles only where an entry is non-zero) or into one CSR (otherwise), so every product is one kernel over
 *        one structure instead of the paper's dense + sparse library calls per step (L286).  nnz(H^(OD)) + the non-zeros of the
 *        dense blocks < 2^31.
 * All arrays are DEVICE pointers; the struct itself is a HOST object.
 */
typedef struct {
  ttdft_format fmt;
  int64_t M;
  int32_t block;
  const int32_t* row_ptr;
  const int32_t* col_idx;
  const double* values;
  const int32_t* subdomain_of_row;
  uint32_t flags;
  const double* diag_values; /* HYBRID only (ignored otherwise): the dense diagonal blocks */
  int64_t diag_block;        /* HYBRID only: rows of one diagonal block, 1 .. M          */
} ttdft_h_desc;

/* read-back description of a built handle (all HOST values) */
typedef struct {
  int64_t M;
  int64_t nnz_stored;     /* stored scalar entries incl. explicit zeros (BSR: nblocks*b*b) */
  int32_t block;          /* tile size of the device format, 0 if CSR                       */
  int32_t kernel;         /* 1 = block-sparse tile kernels (fp64 / int8 tensor cores), 0 = generic */
  int64_t nblocks;
  size_t storage_bytes;
  int32_t i8_planes;      /* digit planes per operand of H stored for the I8 modes (0: not built) */
  int32_t math;           /* TTDFT_MATH_FP64, _I8 or _I8X7: what calls that take `work` use */
  int32_t reordered;      /* 1: rows were regrouped by subdomain label (the handle keeps the row map) */
  int32_t padded;         /* 1: the subdomains differ in size and were padded with zero rows/columns to the tile size */
  int64_t packed_bytes;   /* bytes of the packed copy of the tiles (per 16-column slab: row offsets, bit masks, non-zero values),
                             the storage variant the products with ncols <= 16 stream instead of the dense tiles; 0: not built */
} ttdft_h_info_t;

/* A0 -- storage builder (north_star "BSR/CSR storage builder"). */

/* Bytes of device storage ttdft_h_build needs for this description.  The call has no stream: it reads
 * row_ptr's last entry and, for a CSR with labels, analyses the labels and counts the tiles with kernels
 * on the legacy default stream and blocking copies -- arrays produced on a non-blocking stream must be
 * complete before the call.  For that analysis (labelled CSR only) it takes a transient device allocation
 * of 16 bytes per row, freed before it returns: the one place besides ttdft_probe_fp64_peak's 64-byte sink
 * where the library allocates device memory.  Indices are range-guarded: an invalid CSR gives a meaningless
 * size, never a fault. */
ttdft_status ttdft_h_storage_bytes(const ttdft_h_desc* desc, size_t* bytes);

/* Validate and convert H into the device format inside dev_storage (>= the bytes reported above,
 * 1024-byte aligned).  The input arrays may be freed once `stream` has passed this call; the handle
 * only points into dev_storage, is immutable afterwards, and may be used from several streams.
 * Everything runs on `stream` (the label analysis and tile count use dev_storage as scratch: no device
 * allocation); the call synchronises `stream` to read sizes back.
 * With a CHECK flag the indices are verified BEFORE any other kernel reads them, and the call reports
 * TTDFT_ERR_INVALID_ARG (unsorted / duplicate / out-of-range indices, row_ptr not ascending from 0) or
 * TTDFT_ERR_NOT_SYMMETRIC.  Without the flag invalid indices are skipped by the conversion (never a
 * fault); the result is then undefined. */
ttdft_status ttdft_h_build(const ttdft_h_desc* desc, void* dev_storage, size_t bytes, void* stream,
                           ttdft_h_t* out);
ttdft_status ttdft_h_info(ttdft_h_t h, ttdft_h_info_t* info);
ttdft_status ttdft_h_destroy(ttdft_h_t h);

/* Select the arithmetic for the calls that take `work` (ttdft_cheb_filter*, ttdft_*_ws); the default
 * is TTDFT_MATH_AUTO (or the value of the environment variable TTDFT_MATH at build time).  Changes the
 * handle: do not call it while another thread is using the handle; query the work sizes again
 * afterwards.  TTDFT_ERR_UNSUPPORTED if an I8 mode is asked of a handle without digit planes. */
ttdft_status ttdft_h_set_math_mode(ttdft_h_t h, int32_t mode);

/*
 * Y = alpha * H * X + beta * Y         (the kernel of every filter step)
 * X, Y: M x ncols, ncols >= 1.  X must not overlap Y.  beta == 0 does not read Y (NaN-safe);
 * alpha == 0 does not read H or X.
 */
ttdft_status ttdft_spmm(ttdft_h_t h, double alpha, const double* X, int64_t ldx, double beta, double* Y,
                        int64_t ldy, int64_t ncols, void* stream);

/*
 * One fused recurrence step:
 *     Yout = alpha * (H * Yk - c * Yk) + beta * Ykm1
 * in ONE pass over H, Yk and Ykm1 (scale, shift and axpby live in the product's epilogue).
 * Ykm1 == NULL means the beta term is absent (the first step).  Ykm1 may be the
 * same matrix as Yout (it is only read at the output position); Yk must not overlap Yout.
 */
ttdft_status ttdft_cheb_step(ttdft_h_t h, double alpha, double c, double beta, const double* Yk, int64_t ldk,
                             const double* Ykm1, int64_t ldm, double* Yout, int64_t ldo, int64_t ncols,
                             void* stream);

/*
 * The same two operations with caller-provided scratch, which lets them run in the handle's math mode
 * (TTDFT_MATH_I8 needs room for the digit planes of X / Yk): `work` is a 16-byte aligned DEVICE
 * buffer of at least ttdft_step_work_bytes(h, ncols) bytes (0 in TTDFT_MATH_FP64 on a handle that was not
 * reordered: work may be NULL; a reordered handle adds two M x ncols panels in tile order).
 */
ttdft_status ttdft_step_work_bytes(ttdft_h_t h, int64_t ncols, size_t* bytes);
ttdft_status ttdft_spmm_ws(ttdft_h_t h, double alpha, const double* X, int64_t ldx, double beta, double* Y,
                           int64_t ldy, int64_t ncols, void* work, size_t work_bytes, void* stream);
ttdft_status ttdft_cheb_step_ws(ttdft_h_t h, double alpha, double c, double beta, const double* Yk, int64_t ldk,
                                const double* Ykm1, int64_t ldm, double* Yout, int64_t ldo, int64_t ncols,
                                void* work, size_t work_bytes, void* stream);

/*
 * ttdft_cheb_step_ws for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): the same fused step in the handle's math mode, with the scratch taken from a
 * static device array INSIDE the library instead of from the caller.  Arguments and overlap rules as ttdft_cheb_step_ws.
 *   - The array holds TTDFT_STATIC_SCRATCH_BYTES (32 MiB); every GPU that loads the library keeps it until the process exits.
 *     A step whose ttdft_step_work_bytes(h, ncols) exceeds it is rejected with TTDFT_ERR_WORKSPACE_TOO_SMALL (nothing is
 *     launched): use ttdft_cheb_step_ws there.  32 MiB covers about M x ncols <= 4.5e6 in the int8 modes (e.g. M = 8,192 with
 *     512 columns); TTDFT_MATH_FP64 steps on a handle that was not reordered need no scratch at all.
 *   - The call allocates and frees no device memory: no cudaMalloc / cudaFree, no allocating library routine.  The first call
 *     on a device looks the array's device address up (cudaGetSymbolAddress, with that device current) and keeps it.
 *   - ALL calls on one device share the array, and it keeps the last call's contents (the step clears what it needs zeroed).
 *     Calls that overlap on the GPU -- different streams, or graphs replayed concurrently -- RACE on it: keep such calls on one
 *     stream, or order them with events.  Calls on one stream, and calls mixed with ttdft_*_ws on caller scratch, are safe.
 */
#define TTDFT_STATIC_SCRATCH_BYTES (32u << 20)
ttdft_status ttdft_cheb_step_static(ttdft_h_t h, double alpha, double c, double beta, const double* Yk, int64_t ldk,
                                    const double* Ykm1, int64_t ldm, double* Yout, int64_t ldo, int64_t ncols, void* stream);

/*
 * A1 -- the scalars of Algorithm 1, HOST arrays of length m:
 *   e = (b-a)/2, c = (b+a)/2, sigma_1 = e/(a0-c), gamma = 2/sigma_1, sigma_{k+1} = 1/(gamma-sigma_k)
 *   alpha[0] = sigma_1/e, beta[0] = 0;   alpha[k] = 2*sigma_{k+1}/e, beta[k] = -sigma_k*sigma_{k+1}
 * so that step k (0-based) is  Y_{k+1} = alpha[k]*(H*Y_k - c*Y_k) + beta[k]*Y_{k-1},  Y_0 = X.
 * a = eps_ub^w, b = eps_ub^uw, a0 = eps_0.  Requires m >= 0, a0 < a < b.
 */
ttdft_status ttdft_cheb_scalars(int32_t m, double a, double b, double a0, double* c_out, double* alpha,
                                double* beta);

/* Bytes of scratch ttdft_cheb_filter needs: one compact M x panel panel (panel_cols == 0: the
 * library's default panel width for this ncols), plus, in the int8 modes, the digit planes of
 * two iterates (6 or 7 bytes per element each: one being read while the step's epilogue writes the
 * next) and a few per-column arrays (maxima, exponents, flags). */
ttdft_status ttdft_cheb_filter_work_bytes(ttdft_h_t h, int64_t ncols, int64_t panel_cols, size_t* bytes);

/*
 * Y = p_m(H) X,  p_m(t) = T_m((t-c)/e) / T_m((a0-c)/e)      (Algorithm 1, step 1)
 * computed as m fused steps per column panel of width panel_cols (0 = default), the iterates
 * rotating between the X panel, the Y panel and one scratch panel on `stream`.  m == 0 copies X
 * to Y.  Y may be X exactly (in place) but must not partially overlap it.  The result of every
 * column is independent of panel_cols.  Requires ncols >= 1, m >= 0, a0 < a < b.
 */
ttdft_status ttdft_cheb_filter(ttdft_h_t h, const double* X, int64_t ldx, double* Y, int64_t ldy, int64_t ncols,
                               int32_t m, double a, double b, double a0, int64_t panel_cols, void* work,
                               size_t work_bytes, void* stream);

/*
 * The same filter with X and Y in HOST memory (pinned for full speed): column panels are copied
 * host->device, filtered, and copied device->host, the copies of neighbouring panels overlapping
 * the arithmetic.  `work` is DEVICE scratch of at least ttdft_cheb_filter_host_work_bytes.  The call
 * returns after the last panel has reached Y (it synchronises).
 * panel_cols > 0: every panel has that width (the last one what is left).  panel_cols == 0: a ramp of panel widths, 256, 768, then
 * up to 2,048 columns, mirrored at the end (4,096 columns: 256 | 768 | 2,048 | 768 | 256) -- the copy of the first panel in and of
 * the last panel out are the only transfers no arithmetic can hide, so those panels are narrow, and each panel's arithmetic
 * covers the copy of the wider next one.  The scratch is sized for the widest panel (ask ttdft_cheb_filter_host_work_bytes with
 * the same panel_cols).  The result of every column is independent of the panel schedule (bit for bit).
 */
ttdft_status ttdft_cheb_filter_host_work_bytes(ttdft_h_t h, int64_t ncols, int64_t panel_cols, size_t* bytes);
ttdft_status ttdft_cheb_filter_host(ttdft_h_t h, const double* X_host, int64_t ldx, double* Y_host, int64_t ldy,
                                    int64_t ncols, int32_t m, double a, double b, double a0, int64_t panel_cols,
                                    void* work, size_t work_bytes, void* stream);

/*
 * NEXT-1 -- subspace projection, Algorithm 1 step 3 (Sec. 4.3):
 *     H_F = X_F^T (H X_F)
 * "The evaluation of H_F includes a matrix-matrix multiplication between H and X_F ... this matrix is ...
 * left-multiplied with X^T" (the paper does the second product on the host with PETSc; here both run on the GPU).
 *
 * ttdft_gram:     G = X^T W, X and W row-major M x ncols (M >= 0), G row-major ncols x ncols with ldg >= ncols.
 *                 Computed exactly from 7 int8 digit planes per operand (55 bits below each column's maximum) on the
 *                 tensor cores with int32 accumulation over chunks of <= 128*128 rows, the chunks then summed in
 *                 ascending order in fp64: deterministic, error below an fp64 dot product's bound (K4).
 *                 X and W may be the same matrix; G must not overlap them.  ncols <= 65535.
 * ttdft_project:  G = X^T (H X): one ttdft_spmm_ws into scratch, then ttdft_gram.  G is symmetric up to rounding
 *                 when H is.  If the handle was built with TTDFT_CHECK_SYMMETRY (H == H^T verified), only the upper
 *                 triangle is computed and mirrored (G exactly symmetric, ~1/4 less time); otherwise every entry is
 *                 computed as it stands and G is NOT symmetrised.
 * `work`: 1024-byte aligned DEVICE scratch of at least the bytes the matching *_work_bytes call reports.
 */
ttdft_status ttdft_gram_work_bytes(int64_t M, int64_t ncols, size_t* bytes);
ttdft_status ttdft_gram(int64_t M, const double* X, int64_t ldx, const double* W, int64_t ldw, int64_t ncols, double* G,
                        int64_t ldg, void* work, size_t work_bytes, void* stream);
ttdft_status ttdft_project_work_bytes(ttdft_h_t h, int64_t ncols, size_t* bytes);
ttdft_status ttdft_project(ttdft_h_t h, const double* X, int64_t ldx, int64_t ncols, double* G, int64_t ldg, void* work,
                           size_t work_bytes, void* stream);

/*
 * Algorithm 1 step 5 ("Rotate the basis Psi = X Q") and the product every
 * orthonormalisation of step 2 ends with (X R^-1):
 *     Y = X * Q          X: M x k row-major (ldx >= k), Q: k x n row-major (ldq >= n), Y: M x n row-major (ldy >= n)
 * computed by the int8 tensor-core step kernel: X is cut into 128 x 128 tiles of 7 digit planes scaled per ROW of X,
 * Q into digit tiles scaled per COLUMN of Q, all accumulation exact in int32 (k <= 18560), recombined in fp64:
 * error below an fp64 dot product's bound.  Y must not overlap X or Q.  M >= 0, k >= 1, n >= 1.
 * `work`: 1024-byte aligned DEVICE scratch of at least ttdft_rotate_work_bytes (about 7/8 of the bytes of X).
 */
ttdft_status ttdft_rotate_work_bytes(int64_t M, int64_t k, int64_t n, size_t* bytes);
ttdft_status ttdft_rotate(int64_t M, const double* X, int64_t ldx, int64_t k, const double* Q, int64_t ldq, int64_t n, double* Y,
                          int64_t ldy, void* work, size_t work_bytes, void* stream);

/*
 * NEXT-2 -- Algorithm 1 step 2 ("Orthonormalize the Chebyshev filtered basis functions,
 * X_F = Orth(X)", L230 "Gram-Schmidt orthogonalization procedure"; the paper leaves it on the CPU and names it the
 * bottleneck after GPU offload, L378):
 *     Y = X R^-1,  X^T X = R^T R,  R upper triangular with positive diagonal      (Cholesky-QR)
 * which for full-rank X is exactly the Q of Gram-Schmidt.  One pass = ttdft_gram(X, X), an n x n Cholesky factorisation
 * and triangular inverse (plain fp64 kernels), ttdft_rotate(X, R^-1).  passes = 2 (Cholesky-QR2, recommended) repeats it
 * on the result and restores orthogonality to rounding level for cond(X) up to ~1e7; passes = 1 loses orthogonality as
 * cond(X)^2 * 1e-16.  X: M x n row-major, M >= n; Y: M x n row-major, must not overlap X.
 * Returns TTDFT_ERR_BREAKDOWN (Y undefined) if X^T X is not positive definite to working precision.
 * The call SYNCHRONISES `stream` once per pass (it reads the factorisation's breakdown flag).
 * `work`: 1024-byte aligned DEVICE scratch of at least ttdft_orthonormalize_work_bytes.
 */
ttdft_status ttdft_orthonormalize_work_bytes(int64_t M, int64_t n, int32_t passes, size_t* bytes);
ttdft_status ttdft_orthonormalize(int64_t M, const double* X, int64_t ldx, int64_t n, double* Y, int64_t ldy, int32_t passes, void* work,
                                  size_t work_bytes, void* stream);
/*
 * The same without any synchronisation (so that it can be captured into a CUDA graph together with the filter and the projection):
 * the breakdown flag stays on the device.  dev_status: DEVICE array of `passes` int32; entry p becomes 0, or 1 + the index of the
 * first non-positive pivot of pass p + 1.  The call always runs to the end: after a breakdown Y is meaningless (the factorisation
 * goes on with unit pivots; nothing is read or written outside the buffers), and it is the caller who looks at dev_status.
 */
ttdft_status ttdft_orthonormalize_async(int64_t M, const double* X, int64_t ldx, int64_t n, double* Y, int64_t ldy, int32_t passes,
                                        void* work, size_t work_bytes, int32_t* dev_status, void* stream);

/*
 * Spectral bounds by a k-step Lanczos.  Algorithm 1 takes eps_0 and eps_ub^uw as inputs and refers to
 * [30, 31] for them; reading #5: k steps of plain Lanczos (no reorthogonalisation) from the
 * start vector v0, eigenpairs (theta, z) of the k x k tridiagonal, and the residual-corrected Ritz bounds
 *     b = theta_max + |beta_k z_max[k]|  >= lambda_max(H),      a0 = theta_min - |beta_k z_min[k]|  <= lambda_min(H) (nearly always)
 * v0: DEVICE vector of length M (stride 1), not modified.  1 <= k <= 64.  a0_out, b_out: HOST.  theta_out: HOST array of k
 * Ritz values in ascending order, or NULL.  steps_out: HOST, the number of steps actually taken (< k if an invariant subspace
 * was found), or NULL.  The call synchronises `stream`.  `work`: 1024-byte aligned DEVICE scratch of ttdft_lanczos_work_bytes.
 */
ttdft_status ttdft_lanczos_work_bytes(ttdft_h_t h, size_t* bytes);
ttdft_status ttdft_lanczos_bounds(ttdft_h_t h, int32_t k, const double* v0, void* work, size_t work_bytes, void* stream, double* a0_out,
                                  double* b_out, double* theta_out, int32_t* steps_out);

/*
 * A0 without labels: recover the subdomain of every row of a CSR from its sparsity pattern (SURVEY.md 8(a) A0 "group rows so each
 * subdomain's basis functions are contiguous", 8(f)-4 "locality recovery for unhinted CSR").  The paper states the structure that
 * makes it possible -- functions of a subdomain overlap each other (dense diagonal blocks) and the neighbouring subdomains'
 * -- but no algorithm; the rule is DESIGN.md reading #18: rows whose column sets have a Jaccard
 * similarity within 80 % of the row's best match are candidates, a pair is kept if the two candidate sets agree on at least half
 * of the larger one, groups are the sets reachable along kept pairs, numbered by their smallest row.  Exact integer arithmetic.
 * desc: a CSR description (DEVICE arrays; values and subdomain_of_row are not read; columns ascending and unique per row).
 * labels: DEVICE int32[M], written only when *n_groups > 0: the group 0..n_groups-1 of every row -- pass it as subdomain_of_row to
 * ttdft_h_build, which regroups the rows into tiles if every group has the same size b in {32, 64, 96, 128} and otherwise keeps
 * the generic format.  n_groups: HOST; 0 means "no recoverable structure" (some row has more than 192 candidates).
 * Returns TTDFT_ERR_UNSUPPORTED if M bits plus two ints per entry of the longest row exceed 200 KB of shared memory.
 * The call synchronises `stream`.  `work`: 1024-byte aligned DEVICE scratch of ttdft_recover_subdomains_work_bytes (804 B per row).
 */
ttdft_status ttdft_recover_subdomains_work_bytes(int64_t M, size_t* bytes);
ttdft_status ttdft_recover_subdomains(const ttdft_h_desc* desc, int32_t* labels, void* work, size_t work_bytes, void* stream,
                                      int32_t* n_groups);

/* Measured fp64 rate of this GPU: kind 0 = scalar DFMA loop, 1 = DMMA (mma.sync m8n8k4.f64) loop;
 * runs for about `millis` ms on `stream`, synchronises, returns TFLOP/s in *tflops. */
ttdft_status ttdft_probe_fp64_peak(int32_t kind, int32_t millis, void* stream, double* tflops);

/*
 * Device timing of the library's own kernels.  While enabled, every launch of the kernels below is
 * bracketed by a CUDA event pair on the launching stream; ttdft_timing_read waits for the events of
 * one kernel, returns the sum of their durations and their count, and clears them.
 *   kernel_id: 1 = block-sparse fp64 DMMA step, 2 = generic CSR/BSR step, 3 = block-sparse int8
 *   tensor-core step, 4 = digit planes of an iterate (full extraction: a filter's first step, single steps, Gram operands),
 *   5 = column maxima of a panel, 6 = int8 tensor-core Gram product (ttdft_gram / ttdft_project), 7 = the digit bookkeeping
 *   between two steps of a filter (exponents; digits only of the column tiles whose predicted exponent was outgrown).
 */
ttdft_status ttdft_timing_enable(int32_t on);
ttdft_status ttdft_timing_read(int32_t kernel_id, double* total_ms, int64_t* launches);

/* Number of kernels this library has launched since load (all threads). */
int64_t ttdft_launch_count(void);

/* Thread-local message describing the last non-OK status returned on this thread ("" if none). */
const char* ttdft_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TTDFT_H */
