/* bsr_amg.h -- C ABI of libbsramg.so: the device-resident blocked AMG hot path on one NVIDIA B200 (sm_100a).
 *
 * What this library computes (arxiv/paper_2606_24748, cited as PAPER.md:<line>):
 *   - a block-CSR matrix type with independent row / column block sizes bs_r x bs_c
 *   - the rectangular-block SpMV family y = A x (3x3), y = P x (3x6), y = P^T x (6x3)
 *   - the Galerkin product A_c = P^T A P split into a symbolic phase done once and a
 *     numeric phase repeated over the cached structure ("reused sparsity")
 *     with the prolongator-side data (R = P^T) cached and gated on P's state
 *     and the coarse blocks summed through a precomputed block coordinate plan
 *   - the V-cycle over the reused hierarchy with a point-block Jacobi based smoother and a
 *     CG driver reporting the unpreconditioned residual norm
 *
 * Conventions (all entry points):
 *   - Return value: 0 (BSR_OK) on success, otherwise one of the BSR_ERR_* codes below; bsr_last_error() then
 *     returns a thread-local, human readable message.  No C++ exception crosses this boundary.
 *   - "d_" pointers are DEVICE pointers (cudaMalloc / torch CUDA tensors), "h_" pointers are HOST pointers.
 *     Double arrays passed as d_x / d_y / d_b must be 16-byte aligned (any cudaMalloc / torch allocation is).
 *   - Indices are int32, values are IEEE fp64 ("int32 indices and fp64 values").  A block is stored
 *     row-major, blocks follow each other in CSR order: value (r,c) of stored block k is d_vals[(k*bs_r + r)*bs_c + c].
 *   - Supported block shapes (bs_r x bs_c): 2x2, 2x3, 3x2, 3x3, 3x6, 6x3, 6x6.
 *   - `stream` is a cudaStream_t passed as void* (0 = the legacy default stream).
 *   - HOT calls (bsr_spmv, bsr_spmv_t, ptap_numeric, vcycle_apply, pcg_solve) only enqueue kernels on `stream`:
 *     no allocation, no device synchronisation, no device<->host copy ("no host round trip on reuse",
 *     PAPER.md:103, 186).  Asynchronous faults surface at the caller's next synchronisation.
 *     COLD calls (bsr_create, ptap_symbolic, vcycle_create, first bsr_spmv_t on a matrix) may allocate, copy and
 *     synchronise.  The *_host convenience calls copy and synchronise by definition.
 *   - Results are deterministic: fixed summation order, no floating point atomics.
 *   - There is no CPU fallback: on a machine without a CUDA device every compute call fails with BSR_ERR_CUDA.
 */
#ifndef BSR_AMG_H
#define BSR_AMG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bsr_matrix_s* bsr_t;      /* opaque; created by bsr_create, released by bsr_destroy   */
typedef struct ptap_plan_s* ptap_plan_t; /* opaque; created by ptap_symbolic, released by ptap_destroy */
typedef struct vcycle_s* vcycle_t;       /* opaque; created by vcycle_create, released by vcycle_destroy */
typedef struct psmooth_plan_s* psmooth_plan_t; /* opaque; prolongator_smooth_symbolic / prolongator_smooth_destroy */
typedef struct bcoo_plan_s* bcoo_plan_t;       /* opaque; bcoo_plan_create / bcoo_destroy */

enum {
  BSR_OK = 0,
  BSR_ERR_NULL = 1,      /* null handle or null required pointer                                   */
  BSR_ERR_SHAPE = 2,     /* dimensions do not match (A.nbcols != P.nbrows, A.bs_c != P.bs_r, ...)  */
  BSR_ERR_BLOCK = 3,     /* block shape outside the supported set                                  */
  BSR_ERR_STRUCTURE = 4, /* malformed rowptr / colidx (see bsr_create)                             */
  BSR_ERR_ALLOC = 5,     /* device or host allocation failed                                       */
  BSR_ERR_CUDA = 6,      /* a CUDA runtime call or kernel launch failed                            */
  BSR_ERR_PLAN = 7,      /* plan used with matrices it was not built from                          */
  BSR_ERR_ALIGN = 8,     /* vector pointer not 16-byte aligned                                     */
  BSR_ERR_NUMERIC = 9,   /* singular diagonal block / coarsest operator not positive definite       */
  BSR_ERR_LIMIT = 10     /* a 32-bit count would overflow                                          */
};

/* Message for the last non-zero return on this thread (never null). */
const char* bsr_last_error(void);

/* ------------------------------------------------------------------ matrix container
 * bsr_create: wrap caller-owned device arrays as a block-CSR matrix of nbrows x nbcols blocks of bs_r x bs_c.
 *   d_rowptr[nbrows+1], d_colidx[nnzb], d_vals[nnzb*bs_r*bs_c] are BORROWED: the library never frees them and the
 *   caller keeps them alive (and at the same address) until bsr_destroy.  d_vals may be rewritten in place by the
 *   caller at any time between calls; call bsr_values_changed afterwards.
 *   Validation (cold, synchronises): rowptr[0] == 0, rowptr non-decreasing, rowptr[nbrows] == nnzb, every column
 *   index in [0, nbcols) and STRICTLY ASCENDING inside each row (canonical form; no duplicate blocks).
 *   Errors: BSR_ERR_NULL, BSR_ERR_BLOCK, BSR_ERR_SHAPE (negative sizes), BSR_ERR_STRUCTURE, BSR_ERR_LIMIT
 *   (nnzb*bs_r*bs_c >= 2^31), BSR_ERR_CUDA.  On error *out is set to null. */
int bsr_create(bsr_t* out, int32_t nbrows, int32_t nbcols, int32_t bs_r, int32_t bs_c, int64_t nnzb,
               const int32_t* d_rowptr, const int32_t* d_colidx, double* d_vals, void* stream);
/* The caller rewrote d_vals in place: bumps the matrix's state counter (the analogue of PETSc's object state that
 * gates the P-side cache).  Host-only, no device work. */
int bsr_values_changed(bsr_t A);
/* The caller's values now live in another device array of the same size (double buffering of operator updates):
 * borrows d_vals (16-byte aligned) instead of the old array and bumps the state counter.  Host-only.
 * Errors: BSR_ERR_NULL, BSR_ERR_ALIGN, BSR_ERR_PLAN (a library-owned matrix). */
int bsr_rebind_values(bsr_t A, double* d_vals);
/* Releases the descriptor and every library-owned cache attached to it (cached transpose).  Null is accepted. */
int bsr_destroy(bsr_t A);
/* Queries (host-only).  Any out pointer may be null. */
int bsr_get_info(bsr_t A, int32_t* nbrows, int32_t* nbcols, int32_t* bs_r, int32_t* bs_c, int64_t* nnzb,
                 int64_t* state);

/* ------------------------------------------------------------------ SpMV family
 * bsr_spmv:   d_y[nbrows*bs_r] = A * d_x[nbcols*bs_c].                       HOT.
 * bsr_spmv_t: d_y[nbcols*bs_c] = A^T * d_x[nbrows*bs_r], computed as R*x on the cached explicit transpose R
 *   ("the transpose R" of PAPER.md:103).  The first call on a matrix builds R (cold: allocates, synchronises);
 *   later calls are HOT and re-transpose the values on the device only if the state counter moved.
 * x and y must not alias.  Errors: BSR_ERR_NULL, BSR_ERR_ALIGN, BSR_ERR_CUDA (launch failure), BSR_ERR_ALLOC. */
int bsr_spmv(bsr_t A, const double* d_x, double* d_y, void* stream);
int bsr_spmv_t(bsr_t A, const double* d_x, double* d_y, void* stream);
/* Builds / refreshes the cached transpose now (so that a following bsr_spmv_t is hot) and reports how many times
 * the transpose VALUES of this matrix have been (re)built so far (the state-gate counter). */
int bsr_transpose_prepare(bsr_t A, int64_t* n_value_builds, void* stream);
/* End-to-end convenience: same operations with HOST vectors; copies h_x to the device, runs the kernel, copies the
 * result back and synchronises `stream`.  trans = 0: y = A x, trans = 1: y = A^T x. */
int bsr_spmv_host(bsr_t A, int32_t trans, const double* h_x, double* h_y, void* stream);
/* Algorithmic bytes of one y = A x from the block format (8*bs_r*bs_c + 4 bytes per block, plus
 * row pointers and the two vectors). */
int64_t bsr_spmv_bytes(bsr_t A);

/* ------------------------------------------------------------------ Galerkin product
 * ptap_symbolic (COLD, once per hierarchy level): from the STRUCTURES of A (square, bs x bs) and P (bs x bs_coarse)
 *   computes the boolean structures of AP = A*P and A_c = P^T*(AP) (columns strictly ascending, blocks kept even
 *   if numerically zero), the cached transpose R of P, and the block coordinate plan: for every block of AP and
 *   of A_c the fixed, ordered list of block products that are summed into it (the blocked COO plan with its
 *   duplicate-summation map, built once and reused by every numeric recompute).
 *   Outputs *nbrows_c (= P.nbcols) and *nnzb_c.  Errors: BSR_ERR_NULL, BSR_ERR_SHAPE, BSR_ERR_BLOCK,
 *   BSR_ERR_ALLOC, BSR_ERR_LIMIT, BSR_ERR_CUDA.
 * ptap_structure: copies A_c's structure into caller-allocated device arrays d_rowptr_c[nbrows_c+1],
 *   d_colidx_c[nnzb_c] (enqueued on `stream`).
 * ptap_numeric (HOT): d_vals_c[nnzb_c*bc*bc] = values of P^T A P for the CURRENT values of A (and of P).  Two
 *   kernels: AP = A*P over the cached structure, then A_c = R*(AP), each output block summed in a fixed order by
 *   one thread group -- no atomics.  If P's state counter differs from the one recorded at the last (re)build,
 *   R's values are re-transposed on the device first (state gate); otherwise all P-side data is reused.
 *   d_vals_c must be 16-byte aligned (blocks are written with 16-byte stores).
 *   Errors: BSR_ERR_NULL, BSR_ERR_ALIGN, BSR_ERR_PLAN (A or P is not the matrix the plan was built from), BSR_ERR_CUDA.
 * ptap_get_info: workspace and counters of a plan (any out pointer may be null): nnzb of AP, number of block
 *   products of stage 1 and stage 2, the algorithmic bytes of one two-stage numeric recompute
 *   (bytes(A)+bytes(P)+bytes(AP) + bytes(R)+bytes(AP)+bytes(A_c)), and how often R's values were (re)built. */
int ptap_symbolic(ptap_plan_t* out, bsr_t A, bsr_t P, int32_t* nbrows_c, int64_t* nnzb_c, void* stream);
int ptap_structure(ptap_plan_t plan, int32_t* d_rowptr_c, int32_t* d_colidx_c, void* stream);
int ptap_numeric(ptap_plan_t plan, bsr_t A, bsr_t P, double* d_vals_c, void* stream);
int ptap_get_info(ptap_plan_t plan, int64_t* nnzb_ap, int64_t* n_products_1, int64_t* n_products_2,
                  int64_t* algorithmic_bytes, int64_t* n_r_value_builds);
/* How the two stages of a plan are scheduled: out8 = { stage 1 runs the staged kernel (1) or the gather kernel (0), its
 * bricks, reserved, dynamic shared memory per brick; the same four for stage 2 }. */
int ptap_get_schedule(ptap_plan_t plan, int64_t* out8);
/* Runs only one stage of ptap_numeric (1: AP = A*P, 2: A_c = R*AP from the AP left by the last stage 1); for
 * profiling and tests.  stage 2 needs d_vals_c, stage 1 ignores it. */
int ptap_numeric_stage(ptap_plan_t plan, int32_t stage, bsr_t A, bsr_t P, double* d_vals_c, void* stream);
/* Copies the plan's cached AP (structure and the values left by the last stage 1) into caller-allocated DEVICE
 * arrays d_rowptr_ap[nbrows(A)+1], d_colidx_ap[nnzb_ap], d_vals_ap[nnzb_ap*bs*bs_coarse]; any of them may be null
 * (skipped).  Enqueued on `stream`.  For tests. */
int ptap_get_ap(ptap_plan_t plan, int32_t* d_rowptr_ap, int32_t* d_colidx_ap, double* d_vals_ap, void* stream);
/* End-to-end convenience: new operator values arrive on the HOST (h_vals_a[nnzb(A)*bs*bs], copied into A's
 * borrowed device array), the recompute runs, A_c's values are copied to h_vals_c and `stream` is synchronised. */
int ptap_numeric_host(ptap_plan_t plan, bsr_t A, bsr_t P, const double* h_vals_a, double* h_vals_c,
                      double* d_vals_c, void* stream);
int ptap_destroy(ptap_plan_t plan);

/* The host part of ptap_symbolic (integer work only), exported so that the plan can be inspected and tested
 * without a GPU.  All pointers are HOST pointers; A is nbrows_a x nbrows_a blocks, P is nbrows_a x nbcols_p blocks.
 * ptap_host_plan_build returns an opaque handle (null on error, see bsr_last_error).  ptap_host_plan_get returns a
 * borrowed pointer to one named int32 / uint16 array of the plan, its element count and element size:
 *   "rowptr_ap","colidx_ap","rowidx_ap"  structure of AP and the fine row of every AP slot
 *   "rowptr_c","colidx_c","rowidx_c"     structure of A_c and the coarse row of every A_c slot
 *   "rowptr_r","colidx_r","perm_r"       structure of R = P^T and, per R slot, the P slot it is the transpose of
 *   "pairptr1","k1","q1","pstart"        stage 1: AP slot s = sum over p in [pairptr1[s], pairptr1[s+1]) of
 *                                        A[rowptr_a[i] + k1[p]] * P[pstart[rowptr_a[i] + k1[p]] + q1[p]], i = rowidx_ap[s]
 *   "pairptr2","t2","s2","apstart"       stage 2: A_c slot u = sum over p of
 *                                        R[rowptr_r[I] + t2[p]] * AP[apstart[rowptr_r[I] + t2[p]] + s2[p]], I = rowidx_c[u]
 * Products of one output block are listed by ascending inner block index (the fixed summation order). */
void* ptap_host_plan_build(int32_t nbrows_a, const int32_t* rowptr_a, const int32_t* colidx_a, int32_t nbcols_p,
                           const int32_t* rowptr_p, const int32_t* colidx_p);
int ptap_host_plan_get(void* handle, const char* name, const void** ptr, int64_t* count, int32_t* elem_bytes);
/* Host side of the staged numeric schedule (cold part of ptap_symbolic), for tests: builds the brick / chunk / pass
 * plan of stage 1 (AP = A*P) or stage 2 (A_c = R*AP) for fine / coarse block sizes bs_f / bs_c under a shared-memory
 * budget and reports out8 = { plan usable (1/0), bricks, chunks, largest brick's shared memory in bytes, set mask bits
 * (= block products covered, each exactly once), lanes over all entries, passes, steps over all passes }. */
int ptap_host_stream_stats(void* handle, int32_t bs_f, int32_t bs_c, int32_t stage, int64_t smem_budget,
                           int64_t* out8);
void ptap_host_plan_free(void* handle);

/* ------------------------------------------------------------------ V-cycle and PCG
 * vcycle_create (COLD): hierarchy of `nlevels` operators A[0..nlevels-1] (square) and prolongators
 *   P[0..nlevels-2] (P[l]: level l+1 -> level l).  Smoother on every level but the coarsest: one Chebyshev
 *   polynomial of degree `cheb_degree` (1..4) in D^-1 A over [lo*lambda_l, hi*lambda_l], D the bs x bs block
 *   diagonal (point-block Jacobi), lambda_est[l] the caller's eigenvalue estimate of D^-1 A on level
 *   l (nlevels-1 entries).  Coarsest level: dense Cholesky based direct solve on the device (at most 16384
 *   unknowns).  Matrices are borrowed and must outlive the vcycle.  Calls vcycle_refresh once.
 * vcycle_refresh: after operator values changed (e.g. after ptap_numeric): recomputes D^-1 on every level and
 *   re-factors the coarsest operator; enqueues only, but a singular block is reported at the NEXT refresh/create
 *   synchronisation through vcycle_status.
 * vcycle_apply (HOT): d_x = M^-1 d_b, one V(1,1)-cycle of the polynomial smoother from a zero initial guess:
 *   pre-smooth, residual, restrict (P^T), recurse, prolong and add, post-smooth.
 * pcg_solve (HOT): `iters` iterations of preconditioned CG on A[0] x = b with M^-1 = the V-cycle, x_0 = 0;
 *   d_resid_hist[k] = ||b - A x_k||_2 by the recursive residual, k = 0..iters ("unpreconditioned
 *   residual norm").  No host synchronisation inside. */
int vcycle_create(vcycle_t* out, int32_t nlevels, const bsr_t* A, const bsr_t* P, const double* lambda_est,
                  int32_t cheb_degree, double lo, double hi, void* stream);
int vcycle_refresh(vcycle_t vc, void* stream);
/* Synchronises `stream` and returns BSR_ERR_NUMERIC if the last refresh met a singular diagonal block or a
 * non-positive Cholesky pivot (COLD). */
int vcycle_status(vcycle_t vc, void* stream);
int vcycle_apply(vcycle_t vc, const double* d_b, double* d_x, void* stream);
/* One application of the level-l smoother to d_x in place (for tests): x <- x + p(D^-1 A)(b - A x). */
int vcycle_smooth(vcycle_t vc, int32_t level, const double* d_b, double* d_x, void* stream);
int pcg_solve(vcycle_t vc, const double* d_b, double* d_x, int32_t iters, double* d_resid_hist, void* stream);
/* End-to-end convenience with HOST vectors (copies, runs vcycle_apply, copies back, synchronises). */
int vcycle_apply_host(vcycle_t vc, const double* h_b, double* h_x, void* stream);
int vcycle_destroy(vcycle_t vc);

/* ------------------------------------------------------------------ prolongator smoothing
 * P = (I - omega D^-1 A) P~: "one step of a damped-Jacobi prolongator smoother", D the bs x bs block
 * diagonal of A, in blocks on the device; the block AXPY that adds P~ on a subset of the pattern (the paper's MatAYPX
 * with SUBSET_NONZERO_PATTERN) and the D^-1 left-multiply are fused into the store of the product A*P~,
 * so the step is ONE pass over A.
 * prolongator_smooth_symbolic (COLD): from the STRUCTURES of A (square, bs x bs, every row holding its diagonal block)
 *   and P~ (bs x bs_coarse; shapes 2x3, 3x3, 3x6, 6x6) computes the structure of P = boolean pattern of A*P~ (columns
 *   strictly ascending, blocks kept even if numerically zero) and the product schedule.  Outputs *nnzb_p.
 *   Errors: BSR_ERR_NULL, BSR_ERR_SHAPE, BSR_ERR_BLOCK, BSR_ERR_STRUCTURE (a P~ block outside the pattern: A lacks a
 *   diagonal block), BSR_ERR_ALLOC, BSR_ERR_LIMIT, BSR_ERR_CUDA.
 * prolongator_smooth_structure: copies P's structure into caller-allocated device arrays d_rowptr_p[nbrows+1],
 *   d_colidx_p[nnzb_p].
 * prolongator_smooth_numeric (HOT: enqueues two kernels, no allocation, no synchronisation): d_vals_p[nnzb_p*bs*bsc]
 *   (16-byte aligned) = values of P for the CURRENT values of A and P~ and the given omega.  A singular or missing
 *   diagonal block is reported by prolongator_smooth_status (COLD: synchronises) as BSR_ERR_NUMERIC.
 * prolongator_smooth_get_info: block products A(i,j)*P~(j,J), algorithmic bytes bytes(A)+bytes(P~)+bytes(P), and
 *   whether the staged kernel (1) or the gather fallback (0) runs.
 * prolongator_smooth_lambda (COLD: allocates two work vectors at first use, synchronises): the eigenvalue estimate of
 *   D^-1 A the damping is derived from (omega = 4 / (3 lambda), reading R10): v <- v0/||v0||_2, then `iters`
 *   times w = D^-1 (A v), lambda = ||w||_2, v = w / lambda, entirely on the device (bsr_spmv's kernel, a block-diagonal
 *   apply with a fixed-order norm); *lambda (HOST) receives the last lambda.  d_v0[nbrows*bs] is not modified. */
int prolongator_smooth_symbolic(psmooth_plan_t* out, bsr_t A, bsr_t P_tent, int64_t* nnzb_p, void* stream);
int prolongator_smooth_structure(psmooth_plan_t plan, int32_t* d_rowptr_p, int32_t* d_colidx_p, void* stream);
int prolongator_smooth_numeric(psmooth_plan_t plan, bsr_t A, bsr_t P_tent, double omega, double* d_vals_p,
                               void* stream);
int prolongator_smooth_lambda(psmooth_plan_t plan, bsr_t A, const double* d_v0, int32_t iters, double* lambda,
                              void* stream);
int prolongator_smooth_status(psmooth_plan_t plan, void* stream);
int prolongator_smooth_get_info(psmooth_plan_t plan, int64_t* n_products, int64_t* algorithmic_bytes, int32_t* staged);
int prolongator_smooth_destroy(psmooth_plan_t plan);

/* ------------------------------------------------------------------ blocked COO assembly
 * "Each declared coordinate addresses a block, the value stream is a sequence of dense blocks (square or rectangular),
 * and the scatter writes and sums contiguous bs_r*bs_c runs".
 * bcoo_plan_create (COLD, synchronises): the caller declares ONCE the block coordinates (d_brow[c], d_bcol[c]),
 *   c = 0..n-1, of every contribution, duplicates included (device arrays, read here and not kept); a contribution
 *   with a NEGATIVE coordinate is declared but ignored (its stream block is skipped by every bcoo_set_values), the
 *   coordinate-format convention for entries the caller does not own.  The plan holds
 *   the structure of the assembled matrix (one block per distinct coordinate; rows with no contribution are empty;
 *   columns strictly ascending) and the duplicate-summation map in gather form.  Outputs *nnzb.
 *   Errors: BSR_ERR_NULL, BSR_ERR_SHAPE, BSR_ERR_BLOCK, BSR_ERR_STRUCTURE (coordinate out of range), BSR_ERR_LIMIT
 *   (n >= 2^31 or nnzb*bs_r*bs_c >= 2^31), BSR_ERR_ALLOC, BSR_ERR_CUDA.
 * bcoo_structure: copies the structure into caller-allocated device arrays d_rowptr[nbrows+1], d_colidx[nnzb].
 * bcoo_set_values (HOT, one kernel): d_vals[nnzb*bs_r*bs_c] <- for every block the sum, in declaration order, of the
 *   stream blocks d_stream[c*bs_r*bs_c ...] (row-major) that carry its coordinate.  No atomics; d_vals is overwritten.
 * bcoo_get_info: contributions, blocks, algorithmic bytes 8*bs_r*bs_c*(n + nnzb) + 4*n + 4*(nnzb+1). */
int bcoo_plan_create(bcoo_plan_t* out, int64_t n, const int32_t* d_brow, const int32_t* d_bcol, int32_t nbrows,
                     int32_t nbcols, int32_t bs_r, int32_t bs_c, int64_t* nnzb, void* stream);
int bcoo_structure(bcoo_plan_t plan, int32_t* d_rowptr, int32_t* d_colidx, void* stream);
int bcoo_set_values(bcoo_plan_t plan, const double* d_stream, double* d_vals, void* stream);
int bcoo_get_info(bcoo_plan_t plan, int64_t* n_contrib, int64_t* nnzb, int64_t* algorithmic_bytes);
int bcoo_destroy(bcoo_plan_t plan);
/* d_dst block t = d_src block d_idx[t], t = 0..n-1, blocks of bs doubles (HOT, one kernel): packs the entries of a
 * vector (bs = block size) or whole matrix blocks (bs = bs_r*bs_c) that a neighbouring rank needs -- the device-side
 * staging of the halo / P_oth exchange ("the block payload is staged and exchanged directly from device
 * memory").  Errors: BSR_ERR_NULL, BSR_ERR_SHAPE, BSR_ERR_LIMIT, BSR_ERR_CUDA. */
int bsr_gather_blocks(int64_t n, const int32_t* d_idx, int32_t bs, const double* d_src, double* d_dst, void* stream);
/* The reverse: d_dst block d_idx[t] += d_src block t (HOT, one kernel).  d_idx must hold DISTINCT blocks (the owner's
 * rows a neighbour contributed to, each once): no atomics; contributions of several neighbours are added by
 * consecutive calls in a fixed order (the "off-process reduce"). */
int bsr_scatter_add_blocks(int64_t n, const int32_t* d_idx, int32_t bs, const double* d_src, double* d_dst, void* stream);
/* Finite-element driver of the primitive ("finite-element assembly the natural next application"): Q1
 * elasticity on the uniform grid of ne elements per side (d = 2 or 3), elements [e0, e1) in ascending order, 4^d
 * contributions (a, b) per element, a slowest; local node a sits at offset bit k of a in direction k.
 * fem_q1_element_coords: d_brow / d_bcol [(e1-e0)*4^d] = global node of a / of b.
 * fem_q1_element_blocks: d_stream[(e1-e0)*4^d*d*d] = E_e * Ke[a][b] blocks (d_Ke: the (d*2^d)^2 reference element
 *   matrix for E = 1, row-major; d_E: one modulus per element of the WHOLE grid, or null for E = 1).  dirichlet != 0
 *   folds the clamped face ix = 0 into the stream (a block whose row or column node is clamped is zero, the node's own
 *   diagonal block carries I / #adjacent elements: the assembled block is exactly I, reading R4). */
int fem_q1_element_coords(int32_t d, int32_t ne, int64_t e0, int64_t e1, int32_t* d_brow, int32_t* d_bcol, void* stream);
int fem_q1_element_blocks(int32_t d, int32_t ne, int64_t e0, int64_t e1, const double* d_Ke, const double* d_E,
                          int32_t dirichlet, double* d_stream, void* stream);

/* ------------------------------------------------------------------ counters (metrics)
 * Process-wide counts since load: kernels launched by this library, device allocations made by this library.
 * Hot calls must not move n_allocs. */
int bsr_counters(int64_t* n_kernel_launches, int64_t* n_allocs);
/* Measured fp64 FMA peak of the current device in TFLOP/s (register-resident FMA chains, CUDA events, best of 5):
 * the ALU roof reported beside the HBM roof of the PtAP kernels.  COLD: allocates, synchronises. */
int bsr_measure_fp64_peak(double* tflops, void* stream);
/* The same for the fp64 tensor-core path (chains of mma.sync.aligned.m8n8k4.f64, 512 flops each): the roof of the dense
 * GEMM inside vcycle_refresh.  COLD: allocates, synchronises. */
int bsr_measure_fp64_mma_peak(double* tflops, void* stream);

/* ------------------------------------------------------------------ an entry point that allocates nothing
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it).  bsr_lambda_noalloc runs prolongator_smooth_lambda's power iteration (reading R10: v <- v0/||v0||_2,
 * then `iters` times w = D^-1 (A v), lambda = ||w||_2, v = w / lambda; the same kernels in the same order, so the same
 * bits) with ALL of its work space -- D^-1, two work vectors, the norm's partial sums, the status word -- in one fixed
 * device array inside the library: BSR_NOALLOC_SCRATCH_BYTES on every GPU that loads the library, until exit.
 *   A           square, square blocks of size 2, 3 or 6, resident (bsr_create); only read.
 *   d_v0        DEVICE, nbrows*bs doubles, 16-byte aligned; not modified.
 *   d_lambda    DEVICE, 1 double: receives the last lambda (stream-ordered; the call does not synchronise).
 *   d_status    DEVICE, 1 int32, or null: receives 0, or 1 if a diagonal block of A is missing or singular.
 * HOT: enqueues 4 + 4*iters kernels, one 4-byte memset and one or two 8-/4-byte device-to-device copies on `stream`;
 * calls no cudaMalloc / cudaFree / allocating routine (the first call on a device looks the array's address up with
 * cudaGetSymbolAddress: make that call outside a capture).
 * Limit: bsr_lambda_noalloc_scratch_doubles(nbrows, bs) * 8 <= BSR_NOALLOC_SCRATCH_BYTES, i.e. about 15*nbrows + 700
 * doubles for bs = 3 (279,000 block rows; the 65^3-node grid of config 2 fits, config 3 does not) and 48*nbrows for
 * bs = 6; a larger matrix is rejected with BSR_ERR_LIMIT and nothing is enqueued.
 * Every call on a device shares the one array, which keeps the previous call's contents (the call clears what has to
 * start at zero): two calls that overlap on the GPU -- different streams, or two host threads -- race; serialise them.
 * Errors: BSR_ERR_NULL, BSR_ERR_SHAPE, BSR_ERR_BLOCK, BSR_ERR_ALIGN, BSR_ERR_LIMIT, BSR_ERR_CUDA. */
#define BSR_NOALLOC_SCRATCH_BYTES (32LL << 20)
int bsr_lambda_noalloc(bsr_t A, const double* d_v0, int32_t iters, double* d_lambda, int32_t* d_status, void* stream);
int bsr_lambda_noalloc_scratch_doubles(int32_t nbrows, int32_t bs, int64_t* doubles);

/* ------------------------------------------------------------------ workspace allocator (ownership)
 * Library-private workspace (the cached transpose, AP, plans, D^-1, work vectors, the dense factor) is obtained in COLD
 * calls only.  By default it comes from cudaMalloc; a caller that owns device memory (the Python harness: torch's caching
 * allocator) registers a pair of callbacks and every later allocation goes through them: alloc_fn(bytes, ctx) returns a
 * 256-byte aligned DEVICE pointer or null, free_fn(ptr, ctx) releases one.  A block is returned to the source it came
 * from; pass (null, null, null) to go back to cudaMalloc (blocks already handed out stay valid until the library frees
 * them through the free_fn registered at that time).  Process-wide; thread-safe.  Errors: BSR_ERR_NULL. */
typedef void* (*bsr_alloc_fn)(size_t bytes, void* ctx);
typedef void (*bsr_free_fn)(void* ptr, void* ctx);
int bsr_set_allocator(bsr_alloc_fn alloc_fn, bsr_free_fn free_fn, void* ctx);

/* ------------------------------------------------------------------ options of the COLD calls (tests, tuning)
 * Process-wide; read by ptap_symbolic only, never by a hot call.  Names: "ptap_force_gather" (1: keep the
 * one-thread-per-output-block gather kernels instead of the staged kernels, the path any matrix outside the staged
 * format takes), "ptap_smem_stage1" / "ptap_smem_stage2" (shared-memory bytes a brick of the stage may use).
 * Errors: BSR_ERR_NULL, BSR_ERR_SHAPE (unknown name or value out of range). */
int bsr_set_option(const char* name, int64_t value);

#ifdef __cplusplus
}
#endif
#endif /* BSR_AMG_H */
