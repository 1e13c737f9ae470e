/*
 * apd.h -- C ABI of libapd_b200: anisotropic power diagrams (APDs) by semi-discrete optimal
 * transport on one NVIDIA B200 (sm_100a).  Hot path of arxiv 2403.03571:
 *
 *   apd_assign : Algorithm 1 "pixel method" fused with the discrete dual
 *                and its gradient, eq. (2.7)-(2.8), and the discrete
 *                centroid of Algorithm 3.
 *   apd_solve  : Algorithm 2: L-BFGS ascent on the weights until every
 *                cell volume is within tolerance, eq. (2.5).
 *
 * Notation (SURVEY.md / DESIGN.md): M grains (seeds), N voxels, n voxels per axis, d = dim.
 * All arithmetic of the path runs in the library's CUDA kernels; there is no CPU fallback
 * and no other architecture.  Plain pointers and sizes only; every array pointer says whether
 * it is DEVICE or HOST memory.  The caller owns every array; the library owns only the
 * apd_ctx workspace and keeps no caller pointer after a call returns.
 *
 * Errors never cross the ABI as exceptions/aborts: every call returns an apd_status.
 */
#ifndef APD_B200_H
#define APD_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  APD_OK            = 0,   /* success (apd_solve: tolerance met)                                  */
  APD_NOT_CONVERGED = 1,   /* apd_solve only: limits hit / line search failed; outputs hold the
                              evaluated iterate with the smallest max relative volume error;
                              the caller may refine the grid (Alg. 2 step 4)        */
  APD_E_ARG         = -1,  /* bad argument (see each call); nothing was launched                   */
  APD_E_CUDA        = -2,  /* CUDA runtime failure; text via apd_last_error                        */
  APD_E_ARCH        = -3   /* the device is not compute capability 10.x                            */
} apd_status;

/* Regular discretisation of a box (eq. 2.6).  Voxel (ix,iy,iz) is the box
 * P(y,s) centred at y_k = lo_k + (i_k + 1/2) s_k with s_k = (hi_k - lo_k)/n_k; |P| = prod s_k.
 * Linear index j = (iz*ny + iy)*nx + ix (x fastest).  The voxel list is never stored: the
 * kernels generate y from the thread index.  n[2], lo[2], hi[2] are ignored when dim == 2. */
typedef struct {
  int32_t dim;           /* 2 or 3 */
  int32_t n[3];          /* voxels per axis, each >= 1; N = prod n_k must be < 2^31 */
  double  lo[3], hi[3];  /* hi_k > lo_k */
} apd_grid;

/* Which implementation of the voxel x seed reduction runs (all give labels by the same rule:
 * fp32 cost, lowest seed index among equal fp32 costs). */
enum {
  APD_KERNEL_AUTO   = 0,   /* the fastest one for the call: brute force APD_KERNEL_TENSOR (2D and 3D); with
                              opts.cull APD_KERNEL_ROWPOLY.  Grids with n[0] < 8 (3D also n[1] < 8 or n[2] < 4) take
                              APD_KERNEL_DIRECT (and ignore opts.cull): the row kernels expand the cost about the
                              midpoint of a row / tile, which there lies up to 8/n domain widths L outside the
                              domain: a cost then carries a few fp32 ulp of a ((1 + 8/n) L)^2 instead of a few ulp
                              of itself                                                             */
  APD_KERNEL_DIRECT = 1,   /* un-hoisted direct form: 12 (3D) / 7 (2D) FP32 instr. per pair;
                              the reference kernel the FP32-pipe fraction is quoted on             */
  APD_KERNEL_ROWPOLY = 2,  /* quadratic in the offset from the row's midpoint (1.5 FMA per pair) with
                              coefficients polynomial in the row's offset from the tile's midpoint,
                              packed f32x2, deferred argmin                                        */
  APD_KERNEL_TENSOR = 3    /* brute force only (no opts.cull): the cost lifted to a 10-monomial (2D: 6)
                              polynomial in the integer voxel offset from a tile's reference voxel,
                              coefficients split three ways into bf16, contracted on the tensor
                              cores (tcgen05.mma, fp32 accumulators in TMEM); argmin epilogue on
                              the CUDA cores.  Costs carry fp32 rounding                           */
};

/* opts.cull = 1: exact culling (not in the paper).  Per block of voxels the library keeps only
 * the seeds that can be an argmin somewhere in the block (bounds from the triangle inequality in the A_i-norm, taken
 * conservatively in fp32), nested super-tile -> tile -> 16x4x8-voxel brick, and evaluates those.  The labels are those
 * of the brute-force reduction with the same fp32 arithmetic: identical bit for bit to APD_KERNEL_ROWPOLY without culling
 * whenever that runs its short rows (grids below ~10^3 long-row tiles); against the long-row or the TENSOR brute-force
 * kernels (what AUTO picks on large grids / many seeds) the labels can differ on fp32 near-ties only.
 * Requires kernel AUTO or ROWPOLY and positive definite A_i (not checked).  Workspace grows by
 * O(number of bricks): 1 KiB per 512 voxels for the brick lists plus 3 KiB per 2048 voxels for the tile lists apd_solve
 * keeps between its evaluations (3.5 bytes per voxel in all).  pairs_evaluated reports the pairs actually evaluated. */
typedef struct {
  int32_t kernel;          /* APD_KERNEL_*                                   default AUTO         */
  int32_t cull;            /* 0 brute force, 1 exact conservative culling      default 0          */
  int32_t lbfgs_history;   /* m of L-BFGS                                     default 10          */
  int32_t max_iters;       /* apd_solve iteration limit                       default 1000        */
  int32_t max_evals;       /* apd_solve evaluation limit; 0 = 20*max_iters    default 0           */
  int32_t reserved[3];     /* must be 0                                                           */
} apd_opts;

/* Fills *o with the defaults above. */
void apd_default_opts(apd_opts* o);

typedef struct apd_ctx apd_ctx;

/* Creates a context on CUDA device `device` able to handle up to max_seeds grains in `dim`
 * dimensions.  Allocates the workspace (packed seed table, integer histograms, dual partials,
 * L-BFGS state: O(max_seeds) bytes; nothing proportional to the voxel count).
 * Returns APD_E_ARCH if the device is not sm_100-class, APD_E_ARG on dim not in {2,3} or
 * max_seeds < 1, APD_E_CUDA on allocation failure (*out is then NULL). */
int  apd_create(apd_ctx** out, int32_t dim, int32_t max_seeds, int32_t device);
void apd_destroy(apd_ctx* ctx);                 /* NULL is allowed */
/* Text of the last error of this context ("" if none); with ctx == NULL, of the last failed
 * apd_create on this thread.  The pointer stays valid until the next call on the context. */
const char* apd_last_error(const apd_ctx* ctx);

/* One evaluation: Algorithm 1 + eq. (2.7)-(2.8) at the given weights.
 *   X          [M,dim]      DEVICE fp32 row-major, seed positions x_i
 *   A          [M,dim,dim]  DEVICE fp32 row-major, anisotropy matrices; the quadratic form of
 *                           the matrix as given is used, i.e. that of (A+A^T)/2 (reading S13)
 *   w          [M]          DEVICE fp32 weights
 *   target_vol [M]          DEVICE fp32 or NULL.  NULL: `dual` is |P| sum_j min_i C_ij, the
 *                           v-independent part of eq. (2.7) (reading S6)
 *   labels     [N]          DEVICE int32 out or NULL (store skipped).  labels[j] = 0-based
 *                           index of a seed minimising C_ij = |y_j - x_i|^2_{A_i} - w_i
 *                           evaluated in fp32; among equal fp32 costs the lowest index (S1)
 *   vol        [M]          DEVICE fp64 out, required: (voxels labelled i) * |P|   (eq. 2.8)
 *   dual       [1]          DEVICE fp64 out, required: g~(W) of eq. (2.7)
 *   max_rel_err[1]          DEVICE fp64 out or NULL: max_i |vol_i - v_i| / v_i (eq. 2.5);
 *                           written only when target_vol != NULL
 *   centroids  [M,dim]      DEVICE fp64 out or NULL: discrete centroid of each cell
 *                           (PAPER.md:178); an empty cell returns its seed x_i (S5)
 *   pairs_evaluated [1]     DEVICE uint64 out or NULL: voxel-seed pairs whose cost was
 *                           evaluated (= N*M without culling)
 * Asynchronous on `cuda_stream` (a cudaStream_t; NULL = the legacy default stream): returns
 * after enqueueing; outputs are valid once the stream reaches this point.  The one exception: the FIRST call on a
 * grid with more tiles than any before it (or the first with opts.cull / APD_KERNEL_TENSOR) grows the context's
 * workspace, which synchronises `cuda_stream` and calls cudaMalloc -- not allowed under stream capture.  apd_reserve
 * does that growth ahead of time; after it, calls on that grid (or a smaller one) never allocate or synchronise.
 * A context serialises on ONE stream at a time: every call uses the context's single workspace, so two calls in
 * flight on different streams race; the caller orders them (events), or uses one context per stream.
 * `labels` needs only int32 alignment; a 16-byte aligned pointer gets vectorised stores.
 * APD_E_ARG: NULL ctx/grid/required pointer, grid.dim != ctx dim, n_k < 1, hi <= lo,
 * N >= 2^31, M < 1 or M > max_seeds, unknown opts value.  opts == NULL means defaults. */
int apd_assign(apd_ctx* ctx, const apd_grid* grid, int32_t M,
               const float* X, const float* A, const float* w, const float* target_vol,
               int32_t* labels, double* vol, double* dual, double* max_rel_err,
               double* centroids, uint64_t* pairs_evaluated,
               const apd_opts* opts, void* cuda_stream);

/* Algorithm 2: maximise g~ over W from W0 = w_init (0 when NULL, Alg. 2 step 2) by L-BFGS
 * until max_i |vol_i - v_i|/v_i <= tol (eq. 2.5; "<=" is reading S7).  The optimiser is
 * DESIGN.md's specification S9, identical to oracle/apd_oracle.py: fp64 state on the device,
 * every evaluation at fl32(w), weak-Wolfe bracketing line search, stopping test after every
 * evaluation.  The loop runs on the device; the host reads one mapped status word per
 * evaluation and nothing else.
 *   X, A, target_vol, w_init   DEVICE fp32 in (as apd_assign); every target_vol_i > 0 and
 *                              sum target_vol = |Omega| to 1e-6 relative, else APD_E_ARG.  This one
 *                              check runs on the device with the first evaluation: APD_E_ARG from it is returned
 *                              after that evaluation ran (outputs untouched)
 *   w          [M]  DEVICE fp32 out, required: exactly the weights the final evaluation used
 *   labels     [N]  DEVICE int32 out or NULL: Algorithm 1 at the returned w
 *   vol        [M]  DEVICE fp64 out or NULL: cell volumes at the returned w
 *   w64        [M]  DEVICE fp64 out or NULL: the optimiser's fp64 iterate (w = fl32(w64))
 *   iters, evals, max_rel_err, dual   HOST out, each may be NULL
 * max_iters / max_evals are tested after each line-search evaluation (as the oracle's specification S9 does): unless
 * the start already meets the tolerance at least two evaluations run.
 * Blocks until the solve has finished (synchronises `cuda_stream`).  Workspace growth as for apd_assign (apd_reserve).
 * Returns APD_OK, APD_NOT_CONVERGED, or a negative error. */
int apd_solve(apd_ctx* ctx, const apd_grid* grid, int32_t M,
              const float* X, const float* A, const float* target_vol, double tol,
              const float* w_init, float* w, int32_t* labels, double* vol, double* w64,
              int32_t* iters, int32_t* evals, double* max_rel_err, double* dual,
              const apd_opts* opts, void* cuda_stream);

/* Convergence history of the most recent apd_solve on this context: (dual g~, max relative volume error) of every
 * evaluation in order (at most the first 8192).  dual_hist, err_hist: HOST out, [cap] each.  Returns the number of
 * entries written (>= 0), or a negative apd_status.  Synchronous. */
int apd_solve_history(apd_ctx* ctx, double* dual_hist, double* err_hist, int32_t cap);

/* Algorithm 1 + eq. (2.7)-(2.8) on a USER-SUPPLIED discretisation: points y_j with volumes |P_j|,
 * e.g. element centroids and volumes of a triangulation, a masked or locally refined domain.
 *   Y     [N,dim]  DEVICE fp32 row-major, sample points        pvol [N]  DEVICE fp32, their volumes |P_j| >= 0
 *   X, A, w, target_vol, labels, dual, max_rel_err, centroids: as apd_assign (dim = the context's dim)
 *   vol   [M]      DEVICE fp64 out: sum of |P_j| over the points labelled i
 *   dual           g~ = sum_i v_i w_i + sum_j |P_j| min_i C_ij;  centroids: sum |P_j| y_j / vol_i (empty cell: x_i)
 * Volumes are real numbers here, accumulated with fp64 atomics: results are reproducible up to summation order, and
 * there is no culling (brute force, DIRECT arithmetic).  Asynchronous on cuda_stream.  1 <= N < 2^40. */
int apd_assign_points(apd_ctx* ctx, int64_t N, const float* Y, const float* pvol, int32_t M, const float* X,
                      const float* A, const float* w, const float* target_vol, int32_t* labels, double* vol,
                      double* dual, double* max_rel_err, double* centroids, void* cuda_stream);

/* Algorithm 2 on a user-supplied discretisation: the L-BFGS of apd_solve (same specification S9) with every evaluation
 * done by the point kernel of apd_assign_points.  total_volume = sum_j |P_j| (HOST; it replaces |Omega|: sum
 * target_vol must equal it to 1e-6 relative, else APD_E_ARG).  Y, pvol, X, A, target_vol, w_init, w, labels [N],
 * vol [M]: DEVICE as above; iters, evals, max_rel_err: HOST out.  No culling (opts.cull must be 0).  Because cell
 * volumes are fp64 sums accumulated in no fixed order, two runs can differ in the last bits and, rarely, in a
 * line-search decision.  Blocks until finished; returns APD_OK, APD_NOT_CONVERGED or a negative error. */
int apd_solve_points(apd_ctx* ctx, int64_t N, const float* Y, const float* pvol, double total_volume, int32_t M,
                     const float* X, const float* A, const float* target_vol, double tol, const float* w_init,
                     float* w, int32_t* labels, double* vol, int32_t* iters, int32_t* evals, double* max_rel_err,
                     const apd_opts* opts, void* cuda_stream);

/* Algorithm 3 (generalised Lloyd) on a user-supplied discretisation: apd_lloyd (below) with every
 * Algorithm 2 done by apd_solve_points and the centroid of a cell taken over its points, sum |P_j| y_j / sum |P_j|
 * (an empty cell keeps its seed).  X [M,dim] DEVICE fp32 IN/OUT (X^0 on entry, X^K on return); the other arguments as
 * apd_solve_points; iters / evals: totals over the K + 1 solves.  Blocks until finished.  Returns the status of the
 * final Algorithm 2 (APD_OK / APD_NOT_CONVERGED) or a negative error. */
int apd_lloyd_points(apd_ctx* ctx, int64_t N, const float* Y, const float* pvol, double total_volume, int32_t M,
                     float* X, const float* A, const float* target_vol, double tol, int32_t K, const float* w_init,
                     float* w, int32_t* labels, double* vol, int32_t* iters, int32_t* evals, double* max_rel_err,
                     const apd_opts* opts, void* cuda_stream);

/* Counters of the most recent apd_solve on this context (HOST out, each may be NULL): evaluations recorded by
 * apd_solve_history, and how many evaluations of the loop rebuilt the culling candidate lists (with opts.cull the
 * lists are built with a slack on the bounds and reused while the weights stay within it; 0 without culling). */
int apd_solve_stats(const apd_ctx* ctx, int32_t* evals_recorded, int32_t* cull_rebuilds);

/* Algorithm 3, generalised Lloyd: K rounds of { Algorithm 2 from the previous weights; seeds <-
 * discrete centroids of the cells (an empty cell keeps its seed) }, then a final Algorithm 2.
 *   X  [M,dim] DEVICE fp32 IN/OUT: X^0 on entry, X^K on return (each round's centroids rounded to fp32)
 *   A, target_vol, w_init, w, labels, vol: as apd_solve (w_init is W_0^0; NULL = 0); labels/vol describe the final APD
 *   iters, evals: HOST out, totals over all K+1 solves; max_rel_err: HOST out, of the final solve
 * A round that ends APD_NOT_CONVERGED continues from its best iterate; the return value is the final solve's status
 * (or a negative error).  K = 0 is apd_solve.  Blocks until finished. */
int apd_lloyd(apd_ctx* ctx, const apd_grid* grid, int32_t M, float* X, const float* A, const float* target_vol,
              double tol, int32_t K, const float* w_init, float* w, int32_t* labels, double* vol,
              int32_t* iters, int32_t* evals, double* max_rel_err, const apd_opts* opts, void* cuda_stream);

/* Algorithm 2 with its step 4 ("if it is not possible to hit the desired tolerance, increase J and
 * restart"): apd_solve on `grid`; while it returns APD_NOT_CONVERGED and fewer than max_refinements refinements were
 * made, every n_k is doubled (the paper gives no rule; reading S18) and apd_solve restarts from the best weights found
 * so far.  grid: HOST in/out, n[] holds the final resolution on return.  w, vol, w_init: DEVICE as apd_solve (no
 * labels: their size changes; call apd_assign on the returned grid).  refinements, iters, evals (totals),
 * max_rel_err (of the last solve): HOST out, may be NULL.  Returns the status of the last solve. */
int apd_solve_refine(apd_ctx* ctx, apd_grid* grid, int32_t M, const float* X, const float* A,
                     const float* target_vol, double tol, int32_t max_refinements, const float* w_init, float* w,
                     double* vol, int32_t* refinements, int32_t* iters, int32_t* evals, double* max_rel_err,
                     const apd_opts* opts, void* cuda_stream);

/* Coarse-to-fine continuation (an extension of Alg. 2 step 4, PAPER.md:157 -- not in the paper): the
 * weights do not depend on the resolution, so Algorithm 2 is run on `grid` coarsened by 2^levels, ..., 2, 1 per axis
 * (n_k -> ceil(n_k / 2^l); a level with some n_k < 16 is skipped), each level started from the weights of the one
 * before (a level that ends APD_NOT_CONVERGED hands on its best iterate).  A coarse level is asked only for what its
 * voxels can resolve, eq. (2.10) read backwards: tol_l = max(tol, 2^D |P_l| / min_i target_vol_i) (the call reads
 * target_vol back to the host once for this).  The last level is apd_solve on `grid` itself with tol:
 * same post-condition, w, labels, vol; the return value is its status.  levels = 0 is apd_solve.
 *   iters, evals   HOST out [levels + 1], coarsest level first (0 for a skipped level); each may be NULL
 *   max_rel_err    HOST out, of the last level.   Everything else as apd_solve.  Blocks until finished. */
int apd_solve_continuation(apd_ctx* ctx, const apd_grid* grid, int32_t levels, int32_t M, const float* X, const float* A,
                           const float* target_vol, double tol, const float* w_init, float* w, int32_t* labels,
                           double* vol, int32_t* iters, int32_t* evals, double* max_rel_err, const apd_opts* opts,
                           void* cuda_stream);

/* Resolution rules of PAPER.md:182-197 for a cubic grid of M voxels per axis on a domain of volume |Omega|:
 * |Omega| / M^D < factor * v_min with factor = eps (necessary: one misassigned voxel is already the tolerance; eq. 2.9
 * when v_min = |Omega|/N) or eps / 2^D (practical, eq. 2.10).  apd_resolution_bound returns the real number M must
 * EXCEED (Table 1 of the paper prints it rounded to the nearest integer); apd_choose_resolution the smallest integer M
 * that satisfies the strict inequality.  Host-only, no device work.  Negative on bad arguments. */
double  apd_resolution_bound(int32_t dim, double domain_volume, double v_min, double eps, int32_t practical);
int32_t apd_choose_resolution(int32_t dim, double domain_volume, double v_min, double eps, int32_t practical);

/* Same two calls with HOST arrays: the library copies in, runs the device call above and copies
 * the results out.  The device buffers belong to the context (grow-only, reused by the next host
 * call, freed by apd_destroy).  Every pointer is HOST memory (pinned memory makes the copies
 * faster); NULL is allowed where the device call allows it.  Synchronous.  apd_assign_host: when
 * `labels` lies in pinned (page-locked) memory, 16-byte aligned, the kernel stores the labels
 * straight into it during the evaluation (no device buffer, no copy afterwards); the array is
 * complete when the call returns, as on the copy path. */
int apd_assign_host(apd_ctx* ctx, const apd_grid* grid, int32_t M,
                    const float* X, const float* A, const float* w, const float* target_vol,
                    int32_t* labels, double* vol, double* dual, double* max_rel_err,
                    double* centroids, uint64_t* pairs_evaluated, const apd_opts* opts);
int apd_solve_host(apd_ctx* ctx, const apd_grid* grid, int32_t M,
                   const float* X, const float* A, const float* target_vol, double tol,
                   const float* w_init, float* w, int32_t* labels, double* vol, double* w64,
                   int32_t* iters, int32_t* evals, double* max_rel_err, double* dual,
                   const apd_opts* opts);

/* ---- voxel-slab sharding ---------------------------------------------------------------
 * Voxels are independent and the only cross-voxel coupling of the method is the sum of per-cell counters (eq. 2.8,
 * PAPER.md:138-140) and of the minima (eq. 2.7).  A rank that owns planes [lo, lo + n) of the grid's LAST axis (z in
 * 3D, y in 2D) evaluates them with the same arithmetic as the whole-grid call (voxel centres are formed from the
 * GLOBAL index) and leaves RAW counters; adding the counter blocks of all slabs of a partition word by word, as
 * unsigned 64-bit integers, gives exactly the counters of the whole grid:
 *     counters = [ count u64 x M | (with_idxsum) index sums u64 x 3M | layer sums of min-costs, fp64 bit patterns ]
 * (a layer = apd_slab_align(dim) planes; each layer sum is written by the one slab that owns the layer, every other
 * slab leaves 0 there, so the integer addition reproduces the fp64 bits and the dual is identical, bit for bit, to the
 * whole-grid call's whatever the number of slabs).  slab.lo must be a multiple of apd_slab_align(dim), and slab.n too
 * unless the slab ends at the grid's last plane.  The seeds (<= 1 MB) and the L-BFGS state are replicated. */
typedef struct { int32_t lo, n; } apd_slab;
int32_t apd_slab_align(int32_t dim);                                   /* 8 planes (3D), 64 rows (2D)            */
int64_t apd_counter_words(const apd_grid* grid, int32_t M, int32_t with_idxsum);   /* u64 words of a counter block */

/* apd_assign on a slab, stopping before the finalize: labels [slab voxels] DEVICE int32 or NULL (x fastest, the
 * slab's own planes only), counters DEVICE out [apd_counter_words].  Asynchronous on cuda_stream. */
int apd_assign_slab(apd_ctx* ctx, const apd_grid* grid, const apd_slab* slab, int32_t M, const float* X, const float* A,
                    const float* w, int32_t* labels, uint64_t* counters, int32_t with_idxsum, const apd_opts* opts,
                    void* cuda_stream);
/* The finalize of apd_assign from REDUCED counters (the word-wise sum over all slabs): vol, dual, max_rel_err,
 * centroids (needs with_idxsum) exactly as apd_assign returns them.  All pointers DEVICE.  Asynchronous. */
int apd_finalize_counters(apd_ctx* ctx, const apd_grid* grid, int32_t M, const uint64_t* counters, int32_t with_idxsum,
                          const float* X, const float* w, const float* target_vol, double* vol, double* dual,
                          double* max_rel_err, double* centroids, void* cuda_stream);
/* apd_solve on a slab.  After every evaluation the library packs this slab's counters into `counters` (DEVICE,
 * caller-owned, apd_counter_words(grid, M, 0) words) and calls reduce(user, cuda_stream), which must replace the block,
 * in stream order, by its word-wise unsigned 64-bit sum over all ranks (one allreduce of 8 (M + layers) bytes: NCCL
 * ncclAllReduce(ncclUint64, ncclSum) on that stream, or any equivalent) and return 0.  Every rank then runs the same
 * optimiser step on the same reduced counters, so the replicated L-BFGS states stay identical and the trajectory is
 * that of the whole-grid apd_solve bit for bit.  labels: this slab's [slab voxels]; vol [M]: of the whole grid.
 * reduce == NULL: a single slab covering the grid (then this is apd_solve). */
typedef int (*apd_reduce_fn)(void* user, void* cuda_stream);
int apd_solve_slab(apd_ctx* ctx, const apd_grid* grid, const apd_slab* slab, int32_t M, const float* X, const float* A,
                   const float* target_vol, double tol, const float* w_init, float* w, int32_t* labels, double* vol,
                   uint64_t* counters, apd_reduce_fn reduce, void* user, int32_t* iters, int32_t* evals,
                   double* max_rel_err, double* dual, const apd_opts* opts, void* cuda_stream);

/* The input checks the hot path does NOT make (a debug call).  PAPER.md:51-54 assumes every A_i
 * symmetric positive definite -- apd_assign evaluates the quadratic form of whatever matrix it is given (reading S13),
 * but the culling bounds of opts.cull hold only for positive definite A_i -- and PAPER.md:65-69 target volumes
 * v_i > 0 that sum to |Omega|.
 *   X [M,dim], A [M,dim,dim]   DEVICE fp32 in, required
 *   w [M], target_vol [M]      DEVICE fp32 in or NULL (not checked when NULL); target_vol needs `grid` (for |Omega|)
 *   problems                   HOST out, required: 0 if every check passed, else the OR of APD_BAD_*
 * One small kernel on `cuda_stream`; allocates 16 bytes and synchronises the stream (not for stream capture).
 * Returns APD_OK whenever the checks ran (whatever they found); APD_E_ARG / APD_E_CUDA otherwise. */
enum {
  APD_BAD_X_NONFINITE             = 1,    /* a seed coordinate is NaN or +-inf                                   */
  APD_BAD_A_NONFINITE             = 2,    /* an entry of some A_i is NaN or +-inf                                */
  APD_BAD_A_NOT_SYMMETRIC         = 4,    /* |A_kl - A_lk| > 1e-6 max|A_i| for some i                            */
  APD_BAD_A_NOT_POSITIVE_DEFINITE = 8,    /* a leading principal minor of (A_i + A_i^T)/2 is <= 0                */
  APD_BAD_W_NONFINITE             = 16,   /* a weight is NaN or +-inf                                            */
  APD_BAD_TARGET_VOL_NOT_POSITIVE = 32,   /* some v_i <= 0 or not finite                        */
  APD_BAD_TARGET_VOL_SUM          = 64    /* |sum_i v_i - |Omega|| > 1e-6 |Omega|: apd_solve would
                                             return APD_E_ARG                                                    */
};
int apd_validate(apd_ctx* ctx, const apd_grid* grid, int32_t M, const float* X, const float* A, const float* w,
                 const float* target_vol, uint32_t* problems, void* cuda_stream);

/* Grows the context's workspace to what apd_assign / apd_solve / apd_lloyd need on `grid` with `opts` (dual partials:
 * 8 bytes per tile; with opts.cull the candidate lists, 3.5 bytes per voxel; L-BFGS state for opts.lbfgs_history),
 * so that those calls, on this grid or any grid with no more tiles, neither allocate nor synchronise.  Synchronous
 * (cudaMalloc).  APD_E_ARG as apd_assign; APD_E_CUDA on allocation failure. */
int apd_reserve(apd_ctx* ctx, const apd_grid* grid, const apd_opts* opts);

/* What the most recent evaluation on this context launched (HOST out, each may be NULL): the kernel after AUTO was
 * resolved (APD_KERNEL_*), whether the ROWPOLY kernel ran its long-row geometry (rows of 32 voxels per thread; 0 =
 * rows of 16), whether culling ran, the number of CTA tiles, and the device time in ms of the voxel x seed kernel
 * alone (CUDA events on the launching stream around that one launch; the call waits for the second event; -1 inside
 * apd_solve's loop, which is not timed).  APD_E_ARG if no evaluation has run. */
int apd_assign_stats(apd_ctx* ctx, int32_t* kernel, int32_t* row_long, int32_t* cull, int32_t* n_tiles,
                     double* kernel_ms);

/* ---- an evaluation that allocates nothing --------------------------------------------------------------------------
 * apd_assign_static: apd_assign (Algorithm 1, with eqs. 2.7-2.8) for callers that
 * cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid it.  It takes no
 * context: its scratch (packed seeds, per-cell counts, per-tile partial sums of the dual) is a file-scope __device__
 * array of apd_static_scratch_bytes() = 344 KiB that every GPU which loads the library holds until the process exits.
 * It calls no cudaMalloc / cudaFree and no allocating library routine, and does not synchronise.
 *   Runs on the CURRENT device (the one the pointers belong to), asynchronously on cuda_stream.
 *   Kernels: those of apd_assign with opts.kernel = APD_KERNEL_ROWPOLY, opts.cull = 0, in the same order: labels, vol,
 *   dual and max_rel_err are the same bits.  All pointers DEVICE: X [M,dim], A [M,dim,dim], w [M], target_vol [M] or
 *   NULL, labels [N] or NULL, vol [M] out, dual [1] out, max_rel_err [1] out or NULL (needs target_vol).
 *   Limits: M <= APD_STATIC_MAX_SEEDS; the grid may need at most APD_STATIC_MAX_TILES CTA tiles of 32 x 16 x 8 voxels
 *   (3D) / 64 x 64 pixels (2D) -- about 64 M voxels, 400^3 fits -- and at most 1024 layers of 8 planes (3D) / 64 rows
 *   (2D) along its last axis.  Beyond them: APD_E_ARG with a text that names the limit (use apd_assign there).
 *   Every call on a device shares the one array, which keeps the last call's contents (the call itself clears the
 *   counts it adds into).  Calls that may OVERLAP on the GPU -- different streams, or threads, without an ordering
 *   between them -- race on it and give wrong results; calls on one stream are ordered and safe.
 *   Errors: APD_E_ARG, APD_E_ARCH (not sm_100), APD_E_CUDA; the text is in apd_static_last_error() (thread-local). */
#define APD_STATIC_MAX_SEEDS 4096
#define APD_STATIC_MAX_TILES 16384
int apd_assign_static(const apd_grid* grid, int32_t M, const float* X, const float* A, const float* w,
                      const float* target_vol, int32_t* labels, double* vol, double* dual, double* max_rel_err,
                      void* cuda_stream);
int64_t apd_static_scratch_bytes(void);
const char* apd_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* APD_B200_H */
