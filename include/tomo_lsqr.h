/* tomo_lsqr.h — C ABI of the B200-native damped sparse LSQR library (libtomolsqr.so).
 *
 * The operation (Eq. 6; solver family P:142, ref. P:268): solve the sparse,
 * over-determined, regularised least-squares problem of direct surface-wave tomography
 *
 *        min_x  || A x - b ||^2  +  damp^2 || x ||^2 ,          A  m x n  in CSR on the device,
 *
 * by LSQR (Golub-Kahan bidiagonalisation, Paige & Saunders 1982) with x_0 = 0.  A stacks the
 * traveltime-sensitivity rows (Eq. 1, Eq. 5, unknowns depth-fastest Eq. 7) on top
 * of smoothing rows; the library itself accepts any canonical CSR matrix, or the sensitivity block in the factored
 * form of Eq. 5 (ray footprint x depth kernel: tomo_lsqr_create_factored, tomo_lsqr_set_nodal_kernels,
 * tomo_lsqr_update_kernels, tomo_lsqr_assemble_csr).  The step-by-step algorithm, the stopping rules and every reading
 * taken where the paper is silent are in DESIGN.md.
 *
 * Everything runs in hand-written CUDA kernels for sm_100a (no cuSPARSE/cuBLAS, no CPU fallback):
 * a device-side stable CSR->CSC transpose at create, fused SpMV+axpy+norm kernels for A v and A^T u,
 * device-resident LSQR scalars, CUDA-graph replay of `check_every` iterations per host poll.
 *
 * Conventions
 *   d_*  : DEVICE pointer on the current CUDA device (cudaMalloc / torch allocation).  A host pointer is
 *          rejected with TOMO_ERR_NOT_DEVICE_PTR.  h_* and `res`, `out`: HOST pointers.
 *   CSR  : rowptr int64[m+1] (rowptr[0]=0, rowptr[m]=nnz, non-decreasing), colind int32[nnz] with
 *          0 <= col < n STRICTLY INCREASING inside each row (sorted, no duplicates), vals fp64[nnz] or
 *          fp32[nnz], all finite.  1 <= m, n < 2^31, 0 <= nnz < 2^40.  colind and vals must be 16-byte
 *          aligned.  Violations -> TOMO_ERR_BAD_CSR / TOMO_ERR_INVALID_ARG.
 *   Ownership: the three CSR arrays are BORROWED: the caller keeps them alive and unmodified until
 *          tomo_lsqr_destroy.  The handle owns the CSC copy, the work vectors, the scalars, the graphs.
 *          Output arrays (d_x, d_out, d_X) are caller-allocated and fully overwritten.
 *   Errors: status codes only; no exceptions, no abort.  On error *out is NULL; argument errors (INVALID_ARG,
 *          NOT_DEVICE_PTR, RANGE, BAD_CSR, UNSUPPORTED_ARCH) are detected before any work is enqueued, so the
 *          output arrays are untouched; after TOMO_ERR_CUDA / TOMO_ERR_OOM their contents are unspecified.
 *   Streams: `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All work is
 *          enqueued on it; solve* return after their last host poll, i.e. results are valid on return.
 *   Threads: one handle runs one call at a time; different handles are independent.
 *   Device: compute capability 10.x only (TOMO_ERR_UNSUPPORTED_ARCH otherwise; no fallback).  A handle belongs
 *          to the device that was current at create; calling it with another current device -> INVALID_ARG.
 */
#ifndef TOMO_LSQR_H_
#define TOMO_LSQR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tomo_lsqr_s* tomo_lsqr_t; /* opaque handle */

typedef enum {
  TOMO_OK = 0,
  TOMO_ERR_INVALID_ARG = 1,
  TOMO_ERR_BAD_CSR = 2,
  TOMO_ERR_NOT_DEVICE_PTR = 3,
  TOMO_ERR_OOM = 4,
  TOMO_ERR_CUDA = 5,
  TOMO_ERR_UNSUPPORTED_ARCH = 6,
  TOMO_ERR_RANGE = 7,
  TOMO_ERR_NOALLOC_LIMIT = 8   /* tomo_lsqr_spmv_noalloc: the matrix or the device is beyond the static scratch array */
} tomo_status_t;

typedef enum { TOMO_VAL_F64 = 0, TOMO_VAL_F32 = 1 } tomo_valtype_t;

/* Filled by the solve calls (host memory).  istop: 0 = x=0 is the exact solution (b=0 or A^T b=0);
 * 1 = ||r|| <= btol*||b|| + atol*||A||*||x||;  2 = ||A^T r|| / (||A|| ||r||) <= atol;  3 unused (no
 * condition limit);  4,5,6 = the same three tests at machine precision;  7 = max_iters reached. */
typedef struct {
  int32_t itn;    /* iterations performed */
  int32_t istop;  /* reason for stopping, see above */
  double r1norm;  /* ||b - A x||  (from r2norm and xnorm, reading F3) */
  double r2norm;  /* sqrt(||b - A x||^2 + damp^2 ||x||^2): the quantity LSQR decreases monotonically */
  double arnorm;  /* ||A^T r - damp^2 x||  estimate */
  double anorm;   /* Frobenius-type estimate of ||[A; damp I]|| */
  double acond;   /* estimate of cond([A; damp I]) */
  double xnorm;   /* ||x|| estimate */
} tomo_lsqr_result_t;

/* a0 (DESIGN.md §6.3 "create"): validate the CSR arrays on the device, build the stable CSC transpose
 * (rows ascending inside each column) and the cost-balanced element split points of the persistent CTAs.  One-off per matrix.
 * vt selects the storage type of d_vals (arithmetic is fp64 either way). */
tomo_status_t tomo_lsqr_create(tomo_lsqr_t* out, int64_t m, int64_t n, int64_t nnz, const int64_t* d_rowptr,
                               const int32_t* d_colind, const void* d_vals, tomo_valtype_t vt, void* cuda_stream);

/* NEXT-2, factored form (Eq. 5, unknown ordering Eq. 7): the same solver on
 *      A = [ A_data ; A_extra ],   A_data[q * nper + p, k * nz + j] = fl( W[q, k] * g_p[j - j0_p] ),  j0_p <= j < j0_p + klen,
 * without ever storing A_data per nonzero.  q = station pair (ray), p = period, k = lateral node, j = layer:
 *   W      npairs x nnodes, canonical CSR on the device: d_lptr int64[npairs + 1], d_lnode int32[E] strictly increasing
 *          inside a pair, d_lw fp64[E] finite (the lateral footprint of the ray; pairs without entries are allowed);
 *   g      d_kern fp64[nper * klen] (row p = the depth kernel of period p on its window), d_kj0 int32[nper] the first
 *          layer of each window, 0 <= j0_p and j0_p + klen <= nz;  1 <= nper <= 32, 1 <= klen <= min(nz, 32) (RANGE);
 *   A_extra  ms x (nnodes * nz) canonical CSR block appended below A_data (the smoothing rows; ms = 0: none):
 *          d_sptr int64[ms + 1], d_sidx int32[snnz], d_svals fp64[snnz].  Its rows are walked one lane per row.
 * m = npairs * nper + ms < 2^31, n = nnodes * nz < 2^31.  BORROWED until destroy: d_lptr, d_lnode, d_lw, d_sptr, d_sidx,
 * d_svals; d_kj0 and d_kern are copied.  The handle owns W by node (CSC), A_extra by column, the static work split.
 * A lateral entry (12 bytes) stands for nper * klen nonzeros of the CSR form, so the products are bound by fp64
 * arithmetic instead of HBM (get_info "operator_bytes").  With default options every dd product uses the ROUNDED value
 * fl(W g), the number the CSR form stores: with "accumulate" = 1 all results (tomo_lsqr_spmv, the solves) are bit for bit those of a
 * tomo_lsqr_create handle on the expanded matrix; with "accumulate" = 0 they agree to rounding (other summation order and,
 * with option "two_stage" = 1, the unrounded entries W g).
 * Supported on such a handle: tomo_lsqr_solve / tomo_lsmr_solve, *_solve_host, *_solve_multi (the sides run one after
 * the other), tomo_lsqr_spmv, the options "check_every", "accumulate", "graph", "profile", "pdl", "two_stage", and get_info.
 * Not supported (INVALID_ARG): tomo_lsqr_update_values (nothing is stored per nonzero: tomo_lsqr_update_kernels
 * replaces the depth kernels), tomo_lsqr_get_csc, "compress" = 1, tomo_lsqr_solve_sharded.
 * Errors: INVALID_ARG, RANGE, NOT_DEVICE_PTR, BAD_CSR (W, A_extra or the kernel table malformed / non-finite),
 * UNSUPPORTED_ARCH, OOM, CUDA; *out is NULL on error. */
tomo_status_t tomo_lsqr_create_factored(tomo_lsqr_t* out, int64_t npairs, int32_t nper, int64_t nnodes, int32_t nz,
                                        const int64_t* d_lptr, const int32_t* d_lnode, const double* d_lw, int32_t klen,
                                        const int32_t* d_kj0, const double* d_kern, int64_t ms, int64_t snnz,
                                        const int64_t* d_sptr, const int32_t* d_sidx, const double* d_svals,
                                        void* cuda_stream);

/* NEXT-4 ("on-device assembly of G from ray paths and depth kernels"; Eq. 5, Eq. 7):
 * multiply the factored description (arguments as tomo_lsqr_create_factored) out into the canonical CSR arrays the general
 * path takes, on the device: d_rowptr int64[m + 1], d_colind int32[nnz], d_vals fp64[nnz], caller-allocated DEVICE arrays,
 * fully overwritten; nnz must equal d_lptr[npairs] * nper * klen + snnz (INVALID_ARG otherwise, nothing written).
 * Row q * nper + p holds, for the pair's lateral entries in order, value fl(W[q, k] * g_p[t]) at column k * nz + j0_p + t
 * (t = 0 .. klen - 1); the extra block follows unchanged.  The inputs are NOT validated here (tomo_lsqr_create on the
 * result validates the matrix).  nodal = 1: d_kj0 / d_kern hold a table per lateral node (int32[nnodes * nper],
 * fp64[nnodes * nper * klen], as tomo_lsqr_set_nodal_kernels takes them; the paper's Theta_k); 0: one table for all
 * nodes.  One HBM-bound pass: 12 bytes written per nonzero.  The outer Gauss-Newton loop
 * re-evaluates the depth kernels every iteration: this call (or tomo_lsqr_create_factored, which needs no assembly at all)
 * replaces the host-side assembly.  Errors: INVALID_ARG, RANGE, NOT_DEVICE_PTR, UNSUPPORTED_ARCH, CUDA. */
tomo_status_t tomo_lsqr_assemble_csr(int64_t npairs, int32_t nper, int64_t nnodes, int32_t nz, const int64_t* d_lptr,
                                     const int32_t* d_lnode, const double* d_lw, int32_t klen, const int32_t* d_kj0,
                                     const double* d_kern, int64_t ms, int64_t snnz, const int64_t* d_sptr, const int32_t* d_sidx,
                                     const double* d_svals, int64_t nnz, int64_t* d_rowptr, int32_t* d_colind, double* d_vals,
                                     int32_t nodal, void* cuda_stream);

/* NEXT-4 for a factored handle: new depth kernels on the same rays.  The outer Gauss-Newton loop
 * re-evaluates the depth kernels of the updated model and solves again; W (the rays' lateral footprints), its transpose
 * and the work splits stay.  d_kj0 int32[nper], d_kern fp64[nper * klen] (same nper, klen, nz as at create; DEVICE arrays;
 * copied into the handle: the caller's arrays are not kept).  Costs two small copies.  Results of later solves are
 * bitwise those of a handle created from scratch with the new table.
 * Errors: INVALID_ARG (not a factored handle, NULL), NOT_DEVICE_PTR, BAD_CSR (a window outside [0, nz) or a non-finite
 * value; the handle is unchanged), CUDA. */
tomo_status_t tomo_lsqr_update_kernels(tomo_lsqr_t h, const int32_t* d_kj0, const double* d_kern, void* cuda_stream);

/* Depth kernels that depend on the lateral node (the paper's Theta_k, Eq. 5; BASELINE.json's configs use
 * one table for all nodes): d_kj0 int32[nnodes * nper] (window start of node k, period p at k * nper + p),
 * d_kern fp64[nnodes * nper * klen]; same klen as at create; DEVICE arrays, copied into the handle.  From then on
 *      A_data[q * nper + p, k * nz + j] = W[q, k] * g_{k,p}[j - j0_{k,p}]
 * and the handle applies it through the depth-contraction kernels in BOTH accumulation modes, whatever "two_stage" says
 * (a table per node costs the contraction nothing, a per-entry product a table look-up per ray entry): "accumulate" = 1
 * is then the order-independent iterate on the exact entries (reading F-fac3; bit for bit the dd oracle on two-word
 * entries), "accumulate" = 0 plain fp64 sums.  May be called again to refresh the tables (the outer loop);
 * tomo_lsqr_update_kernels is INVALID_ARG afterwards.
 * Errors: INVALID_ARG (not a factored handle, NULL), NOT_DEVICE_PTR, BAD_CSR (window outside [0, nz), non-finite value;
 * the handle is unchanged), OOM, CUDA. */
tomo_status_t tomo_lsqr_set_nodal_kernels(tomo_lsqr_t h, const int32_t* d_kj0, const double* d_kern, void* cuda_stream);

/* NEXT-4: value-only refresh.  The outer Gauss-Newton loop of the inversion
 * re-evaluates G on the same rays and solves again: the sparsity pattern, hence the CSC permutation, the split
 * points and the compressed index, stay; only the values change.  d_vals: device array [nnz] of the handle's value
 * type, in CSR order of the pattern given at create, finite, 16-byte aligned; it may be the array given at create
 * (overwritten in place by the caller) or another one, which then REPLACES it as the borrowed value array (same
 * lifetime rule).  The first call records the CSR -> CSC permutation (one replay of the transpose passes, 4 bytes
 * per nonzero, 8 if nnz >= 2^32); every call then costs one pass over the values ("update_ms" in get_info).
 * Results of later solves are bitwise those of a handle created from scratch on the new values.
 * Errors: TOMO_ERR_BAD_CSR (a non-finite value; the handle is unchanged), INVALID_ARG, NOT_DEVICE_PTR, OOM, CUDA. */
tomo_status_t tomo_lsqr_update_values(tomo_lsqr_t h, const void* d_vals, void* cuda_stream);

/* a1-a7: LSQR on (A, b, damp) from x_0 = 0 until a stopping test fires or max_iters iterations.
 * d_b fp64[m], d_x fp64[n].  damp, atol, btol >= 0 and finite; max_iters >= 0 (0: x = 0, istop = 7).
 * h_r2norm_hist / h_arnorm_hist: NULL or host fp64[max_iters]; entry k-1 = r2norm / arnorm after
 * iteration k, for k = 1..res->itn. */
tomo_status_t tomo_lsqr_solve(tomo_lsqr_t h, const double* d_b, double damp, double atol, double btol,
                              int32_t max_iters, double* d_x, tomo_lsqr_result_t* res, double* h_r2norm_hist,
                              double* h_arnorm_hist, void* cuda_stream);

/* NEXT-1: the same problem by LSMR (Fong & Saunders 2011), the solver the paper itself uses
 * (ref. P:249): identical bidiagonalisation kernels (A v, A^T u with fused norms), other scalar
 * recurrences and a three-vector update (hbar, x, h), under which ||A^T r - damp^2 x|| decreases monotonically.
 * Arguments as tomo_lsqr_solve.  Result fields: r2norm = sqrt(||b - A x||^2 + damp^2 ||x||^2) (estimate),
 * arnorm = ||A^T r - damp^2 x|| (estimate), anorm, acond (estimates), xnorm = ||x|| (computed), r1norm from r2norm
 * and xnorm; istop as above.  h_normr_hist / h_normar_hist: NULL or host fp64[max_iters]. */
tomo_status_t tomo_lsmr_solve(tomo_lsqr_t h, const double* d_b, double damp, double atol, double btol,
                              int32_t max_iters, double* d_x, tomo_lsqr_result_t* res, double* h_normr_hist,
                              double* h_normar_hist, void* cuda_stream);

/* The same solves with HOST buffers: h_b fp64[m] is copied to the device, h_x fp64[n] is copied back
 * (the end-to-end entries bench.py times; the matrix stays resident in the handle).  tomo_lsmr_solve_host is
 * the LSMR counterpart (the paper's solver). */
tomo_status_t tomo_lsqr_solve_host(tomo_lsqr_t h, const double* h_b, double damp, double atol, double btol,
                                   int32_t max_iters, double* h_x, tomo_lsqr_result_t* res, void* cuda_stream);
tomo_status_t tomo_lsmr_solve_host(tomo_lsqr_t h, const double* h_b, double damp, double atol, double btol,
                                   int32_t max_iters, double* h_x, tomo_lsqr_result_t* res, void* cuda_stream);

/* a8: nrhs (1..8) independent LSQR recurrences sharing each pass over A / A^T (BASELINE configs[3]): one SpMM
 * per product on row-major len x 8 blocks (fewer sides are padded with zero columns).
 * d_B fp64[m x nrhs] row-major, d_X fp64[n x nrhs] row-major, res[nrhs].  Every right-hand side stops
 * on its own tests; iterates of a stopped side are frozen. */
tomo_status_t tomo_lsqr_solve_multi(tomo_lsqr_t h, int32_t nrhs, const double* d_B, double damp, double atol,
                                    double btol, int32_t max_iters, double* d_X, tomo_lsqr_result_t* res,
                                    void* cuda_stream);
/* The same block solve by LSMR: per-side LSMR scalars, the three-vector update on len x 8 blocks. */
tomo_status_t tomo_lsmr_solve_multi(tomo_lsqr_t h, int32_t nrhs, const double* d_B, double damp, double atol,
                                    double btol, int32_t max_iters, double* d_X, tomo_lsqr_result_t* res,
                                    void* cuda_stream);

/* NEXT-3: row-sharded LSQR.  A = [A_1; ...; A_P] by row blocks in the global order "rank 0's
 * blocks, rank 1's blocks, ..."; every block is an ordinary handle created on its own rows (m_p x n, all with the
 * same n and value type, on this rank's device); b is split the same way (d_b[l] fp64[m_l]).  u and b are local to a
 * block, v, w, x and the scalars are replicated: d_x fp64[n] is written in full on every rank.  Per iteration every
 * block computes u^_p = A_p v - alpha u_p and the UNROUNDED (hi, lo) pairs of ||u^_p||^2 and of A_p^T u_p per column;
 * two exchanges (16 bytes and 16 n bytes per block) gather them in block order and the sums are closed in that fixed
 * order and rounded once: in double-double mode the iterates are bit for bit those of tomo_lsqr_solve on the whole
 * matrix, in fast mode a deterministic sum in block order.  Options ("accumulate", "check_every") are taken from
 * shards[0]; runs on the int32 index without CUDA graph.
 * allgather (may be NULL iff nranks == 1): device all-gather supplied by the caller (e.g. NCCL through
 * torch.distributed): every rank contributes `bytes` bytes at d_send, on return d_recv holds nranks * bytes with rank
 * r's contribution at offset r * bytes; it must be ordered with `cuda_stream`; returns 0 on success.  The buffers
 * belong to shards[0]. */
typedef int (*tomo_allgather_fn)(void* ctx, const void* d_send, void* d_recv, size_t bytes, void* cuda_stream);
tomo_status_t tomo_lsqr_solve_sharded(const tomo_lsqr_t* shards, int32_t nlocal, int32_t rank, int32_t nranks,
                                      tomo_allgather_fn allgather, void* ctx, const double* const* d_b, double damp,
                                      double atol, double btol, int32_t max_iters, double* d_x, tomo_lsqr_result_t* res,
                                      void* cuda_stream);

/* y = A x (transpose = 0: d_in fp64[n], d_out fp64[m]) or y = A^T x (transpose = 1: d_in fp64[m],
 * d_out fp64[n]) with the kernels the solver uses (the A^T product gathers over the CSC copy). */
tomo_status_t tomo_lsqr_spmv(tomo_lsqr_t h, int transpose, const double* d_in, double* d_out, void* cuda_stream);

/* Copy the CSC arrays built at create to caller device buffers (colptr int64[n+1], rowind int32[nnz],
 * cvals of the handle's value type [nnz]); any pointer may be NULL to skip it.  Test/inspection hook. */
tomo_status_t tomo_lsqr_get_csc(tomo_lsqr_t h, int64_t* d_colptr, int32_t* d_rowind, void* d_cvals, void* cuda_stream);

/* Options (set between solves):
 *   "check_every" k >= 1   iterations per graph replay / host poll (default 10); never changes results
 *   "accumulate"  0 | 1    0 = fast: fp64 FMA sums; 1 = dd: double-double sums rounded once (default 1,
 *                          the order-independent iterate that parity at fixed k is claimed for)
 *   "graph"       0 | 1    replay a CUDA graph (default 1) or launch kernel by kernel
 *   "profile"     0 | 1    1: kernel-by-kernel launches bracketed by CUDA events (see tomo_lsqr_get_info)
 *   "multi_shared" 0 | 1   tomo_lsqr_solve_multi: 1 (default) the sides share every pass over A and A^T (SpMM on
 *                          len x 8 blocks); 0 runs them one after the other (same results)
 *   "compress"    0 | 1    NEXT-2, the structure-exploiting operator: 1 builds (once, on the NULL stream)
 *                          run-compressed copies of the column indices of the CSR and of the row indices of the CSC
 *                          copy (one bit per element + one int32 per run of consecutive indices; the depth-fastest
 *                          ordering of PAPER.md Eq. 7 P:79 makes every lateral node of a ray a run of consecutive
 *                          columns, Eq. 5) and streams those instead of the int32 arrays.  Same elements,
 *                          same order: results are bitwise those of "compress" = 0.  Default 0.
 *   "two_stage"   0 | 1 | 2  factored handles (default 1: in fast mode only): apply A_data as W after the depth contraction
 *                          S[k, p] = sum_t g_p[t] x[k nz + j0_p + t] (and A_data^T as the contraction of T[k, p] = sum_q W[q, k]
 *                          u[q nper + p]): klen times fewer products.  The operator applied has the UNROUNDED entries W g
 *                          (one rounding per entry away from the CSR form's fl(W g)); results stay within the fast-mode
 *                          bar (SpMV 1e-12, x_k as any other summation order).  0: per-entry products of the rounded values.
 *                          With 0 and 1, "accumulate" = 1 works on the rounded entries and its results are bit for bit
 *                          those of the CSR form.  2: the contraction in dd mode too.  S and T are kept as unrounded
 *                          (hi, lo) pairs, every product of both words is exact and each result is rounded ONCE: the
 *                          order-independent iterate of the operator with EXACT entries W g (Eq. 5 in real
 *                          arithmetic; reading F-fac3), bit for bit the dd oracle on two-word entries
 *                          (oracle/factored.py expand_exact) and ~1e-13 away from the CSR form's x_k.
 *   "pdl"         0 | 1    chain the kernels of an iteration with programmatic dependent launch (default 1): the
 *                          prologue of a kernel (barrier set-up, split points, first bulk copies) overlaps the
 *                          tail of the previous one; never changes results
 *   "row_cost"    c >= 0   weight of a row, in elements, in the cost-balanced element split of the
 *                          warp ranges (default 320: a row end costs about as much as 320 streamed elements, measured on B200); changes the summation order only */
tomo_status_t tomo_lsqr_set_option(tomo_lsqr_t h, const char* key, int64_t value);

/* Read-outs (host double): "create_ms" (whole create call, CUDA events), "transpose_ms" (its transpose section
 * including the allocation of the CSC arrays and scratch), "transpose_kernels_ms" (the transpose kernels alone),
 * "update_ms" (the last tomo_lsqr_update_values pass), "csc_bytes", "scratch_bytes", "blocks_rows",
 * "blocks_cols", "compress_bytes_rows" / "compress_bytes_cols" (bytes of the run-compressed index of each direction,
 * 0 before "compress" was set), and after a solve with "profile"=1: "k1_ms", "k2_ms", "k4_ms" (summed CUDA-event time of
 * the A v, A^T u and vector kernels over the iterations that ran) and "k_launches" (launches of each);
 * "kernels_enqueued": cumulative number of kernel launches this handle has issued in solves (nodes of
 * replayed graphs included); "cta_busy_min" / "cta_busy_mean" / "cta_busy_max": busy cycles of the persistent
 * CTAs in the most recent sparse-product launch (load balance of the static split).  Every handle: "factored" (0 | 1),
 * "operator_bytes" (what one product reads of the operator itself).  Factored handles only: "lateral_entries",
 * "cut_nodes_pieces" (pieces of the nodes the A^T x split cuts, current accumulation mode's split counted last),
 * "warp_busy_min" / "_mean" / "_max" / "_argmax" and "warp_busy@<i>" (busy cycles of the warps in the most recent
 * product launch); "csc_bytes", "compress_bytes_*" and "cta_busy_*" are INVALID_ARG on a factored handle. */
tomo_status_t tomo_lsqr_get_info(tomo_lsqr_t h, const char* key, double* out);

/* The sparse product for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): d_y <- A d_x over the caller's CSR with the streaming kernel of the solver
 * (k_wstream, the "sparse matrix-vector multiplications" PAPER.md P:144 offloads), WITHOUT a handle and without
 * any cudaMalloc / cudaFree / allocating library call.  Everything tomo_lsqr_create would allocate for this
 * product (the warp split points, the per-CTA records and tickets of the kernel, and, when the matrix has rows
 * without entries, the compacted row pointers and the row lists) lives in ONE file-scope static __device__ array
 * of TOMO_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds until the process exits.
 *   m, n, nnz, d_rowptr int64[m+1], d_colind int32[nnz], d_vals (fp64 or fp32 per vt): DEVICE arrays as for
 *     tomo_lsqr_create (same alignment rules).  They are NOT validated here: pass arrays tomo_lsqr_create accepts.
 *   accumulate: 0 = fp64 FMA sums, 1 = double-double sums rounded once (as option "accumulate").
 *   d_x fp64[n] in, d_y fp64[m] out (every entry is written), both DEVICE, caller-owned.
 * Limits: m <= TOMO_NOALLOC_MAX_ROWS and a device with at most TOMO_NOALLOC_MAX_SMS multiprocessors, otherwise
 *   TOMO_ERR_NOALLOC_LIMIT and nothing is launched; m, n, nnz ranges as for create (TOMO_ERR_RANGE).
 * Results: the same kernel, split points and summation order as tomo_lsqr_spmv(h, 0, ...) on a handle with
 *   default options, so the output is bitwise that of the handle path in both accumulation modes.
 * Sharing: every call on a device uses the same array, which keeps the previous call's contents; the call clears
 *   what must start at zero (the ticket words and the empty-row counter) itself.  Calls that overlap on the GPU
 *   (two streams, two host threads) RACE on the array: serialise them.  The call synchronises `cuda_stream` twice
 *   (it reads the number of rows without entries back to the host, and waits for the product before returning).
 * Errors: INVALID_ARG, NOT_DEVICE_PTR, RANGE, NOALLOC_LIMIT, UNSUPPORTED_ARCH, CUDA. */
#define TOMO_NOALLOC_MAX_ROWS 524288
#define TOMO_NOALLOC_MAX_SMS 256
#define TOMO_NOALLOC_SCRATCH_BYTES (24 * (TOMO_NOALLOC_MAX_ROWS + 64) + 131072)   /* 12.1 MiB */
tomo_status_t tomo_lsqr_spmv_noalloc(int64_t m, int64_t n, int64_t nnz, const int64_t* d_rowptr, const int32_t* d_colind,
                                const void* d_vals, tomo_valtype_t vt, int accumulate, const double* d_x, double* d_y,
                                void* cuda_stream);

void tomo_lsqr_destroy(tomo_lsqr_t h);

/* Static string for a status; for TOMO_ERR_CUDA the text of the last CUDA error seen by this thread. */
const char* tomo_status_string(tomo_status_t s);

#ifdef __cplusplus
}
#endif
#endif /* TOMO_LSQR_H_ */
