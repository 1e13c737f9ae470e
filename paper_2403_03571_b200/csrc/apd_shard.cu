// apd_shard.cu -- row f4 of DESIGN.md's scope table: voxel-slab sharding.  Voxels are independent;
// the method's only cross-voxel coupling is the sum of the per-cell counters (eq. 2.8) and of the
// minima (eq. 2.7).  A slab = planes [lo, lo + n) of the grid's last axis is evaluated by the
// ordinary kernels (GridDev::off_y / off_z: centres from the GLOBAL index), and this file packs what the evaluation
// left in the workspace into the u64 counter block the ranks sum word by word:
//     [ count u64 x M | (with_idxsum) idxsum u64 x 3M | layer sums of the dual partials, fp64 bit patterns ]
// Every layer (SLAB_ALIGN planes) is owned by exactly one slab -- the others write 0 there -- so the integer sum
// reproduces the owner's fp64 bits, and the sum of minima = the layer sums in ascending order is, bit for bit, what the
// whole-grid call computes (apd_finalize.cu, lbfgs_step_kernel use the same two-level order).
#include "apd_internal.cuh"
#include "apd_device.cuh"

namespace apd {

constexpr int PK_THREADS = 256;

__global__ void __launch_bounds__(PK_THREADS) pack_counters_kernel(
    int M, LayerMap lm, int first_layer, int n_layers_full, const unsigned int* __restrict__ count,
    const unsigned long long* __restrict__ idxsum, const double* __restrict__ dual_partial,
    unsigned long long* __restrict__ counters, const int* __restrict__ done_flag) {
  if (done_flag && *done_flag) return;
  const int tid = blockIdx.x * PK_THREADS + threadIdx.x;
  const int n_count_blocks = (M + PK_THREADS - 1) / PK_THREADS;
  if ((int)blockIdx.x < n_count_blocks) {
    if (tid < M) {
      counters[tid] = (unsigned long long)count[tid];
      if (idxsum) {
        counters[M + 3 * (size_t)tid + 0] = idxsum[3 * (size_t)tid + 0];
        counters[M + 3 * (size_t)tid + 1] = idxsum[3 * (size_t)tid + 1];
        counters[M + 3 * (size_t)tid + 2] = idxsum[3 * (size_t)tid + 2];
      }
    }
    return;
  }
  // one warp per layer of the WHOLE grid: the slab's own layers get their sum, the others 0
  unsigned long long* layers = counters + (idxsum ? 4 * (size_t)M : (size_t)M);
  const int L = ((int)blockIdx.x - n_count_blocks) * (PK_THREADS / 32) + (threadIdx.x >> 5);
  if (L >= n_layers_full) return;
  const int l = L - first_layer;
  double ls = 0.0;
  if (l >= 0 && l < lm.n_layers) {
    const int first = l * lm.per_layer, cnt = min(lm.per_layer, lm.n_partials - first);
    ls = warp_ordered_sum(dual_partial + first, cnt);
  }
  if ((threadIdx.x & 31) == 0) layers[L] = (l >= 0 && l < lm.n_layers) ? (unsigned long long)__double_as_longlong(ls) : 0ull;
}

cudaError_t launch_pack_counters(const GridDev& g, int M, LayerMap lm, int n_layers_full, const unsigned int* count,
                                 const unsigned long long* idxsum, const double* dual_partial, uint64_t* counters,
                                 const int* done_flag, cudaStream_t st) {
  const int first_layer = (g.dim == 3 ? g.off_z : g.off_y) / slab_align(g.dim);
  const int nb = (M + PK_THREADS - 1) / PK_THREADS + (n_layers_full + PK_THREADS / 32 - 1) / (PK_THREADS / 32);
  pack_counters_kernel<<<nb, PK_THREADS, 0, st>>>(M, lm, first_layer, n_layers_full, count, idxsum, dual_partial,
                                                  reinterpret_cast<unsigned long long*>(counters), done_flag);
  return cudaGetLastError();
}

}  // namespace apd

using namespace apd;

#define SH_TRY(call)                                                                \
  do {                                                                              \
    cudaError_t e__ = (call);                                                       \
    if (e__ != cudaSuccess) {                                                       \
      ctx->err = std::string(#call) + ": " + cudaGetErrorString(e__);               \
      return APD_E_CUDA;                                                            \
    }                                                                               \
  } while (0)

extern "C" int32_t apd_slab_align(int32_t dim) { return (dim == 2 || dim == 3) ? slab_align(dim) : -1; }

extern "C" int64_t apd_counter_words(const apd_grid* grid, int32_t M, int32_t with_idxsum) {
  if (!grid || (grid->dim != 2 && grid->dim != 3) || M < 1) return -1;
  const int n_last = grid->n[grid->dim - 1];
  if (n_last < 1) return -1;
  const int al = slab_align(grid->dim);
  return (int64_t)M * (with_idxsum ? 4 : 1) + (n_last + al - 1) / al;
}

extern "C" int apd_assign_slab(apd_ctx* ctx, const apd_grid* grid, const apd_slab* slab, int32_t M, const float* X,
                               const float* A, const float* w, int32_t* labels, uint64_t* counters, int32_t with_idxsum,
                               const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  std::string e;
  bool cull = false;
  const int kernel = resolve_kernel(ctx, opts, grid, M, &cull, &e);
  if (kernel < 0) { ctx->err = "apd_assign_slab: " + e; return APD_E_ARG; }
  if (M < 1 || M > ctx->ws.max_seeds) { ctx->err = "apd_assign_slab: M out of range [1, max_seeds]"; return APD_E_ARG; }
  if (!X || !A || !w || !counters || !slab) { ctx->err = "apd_assign_slab: slab, X, A, w and counters are required"; return APD_E_ARG; }
  GridDev g, gfull;
  e = make_grid(ctx, grid, kernel, cull, &g, slab);
  if (!e.empty()) { ctx->err = "apd_assign_slab: " + e; return APD_E_ARG; }
  e = make_grid(ctx, grid, kernel, cull, &gfull, nullptr);
  if (!e.empty()) { ctx->err = "apd_assign_slab: " + e; return APD_E_ARG; }
  SH_TRY(cudaSetDevice(ctx->ws.device));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  Workspace& ws = ctx->ws;
  // raw evaluation (no finalize): vol == nullptr; the index sums are accumulated when `centroids` is non-null
  double* want_idx = with_idxsum ? reinterpret_cast<double*>(ws.idxsum) : nullptr;     // only tested against nullptr
  const int rc = enqueue_evaluation(ctx, g, kernel, M, X, A, w, nullptr, labels, nullptr, nullptr, nullptr, want_idx,
                                    nullptr, true, cull, nullptr, st);
  if (rc != APD_OK) return rc;
  SH_TRY(launch_pack_counters(g, M, layer_map(g, cull), layer_map(gfull, cull).n_layers, ws.count,
                              with_idxsum ? ws.idxsum : nullptr, ws.dual_partial, counters, nullptr, st));
  return APD_OK;
}

extern "C" int apd_finalize_counters(apd_ctx* ctx, const apd_grid* grid, int32_t M, const uint64_t* counters,
                                     int32_t with_idxsum, const float* X, const float* w, const float* target_vol,
                                     double* vol, double* dual, double* max_rel_err, double* centroids,
                                     void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (M < 1 || M > ctx->ws.max_seeds) { ctx->err = "apd_finalize_counters: M out of range [1, max_seeds]"; return APD_E_ARG; }
  if (!counters || !X || !w || !vol || !dual) { ctx->err = "apd_finalize_counters: counters, X, w, vol and dual are required"; return APD_E_ARG; }
  if (centroids && !with_idxsum) { ctx->err = "apd_finalize_counters: centroids need with_idxsum"; return APD_E_ARG; }
  GridDev g;
  const std::string e = make_grid(ctx, grid, APD_KERNEL_DIRECT, false, &g, nullptr);
  if (!e.empty()) { ctx->err = "apd_finalize_counters: " + e; return APD_E_ARG; }
  SH_TRY(cudaSetDevice(ctx->ws.device));
  const unsigned long long* c64 = reinterpret_cast<const unsigned long long*>(counters);
  LayerMap lm;
  lm.n_layers = (int)(apd_counter_words(grid, M, with_idxsum) - (int64_t)M * (with_idxsum ? 4 : 1));
  lm.per_layer = 0; lm.n_partials = 0;
  double* layers = reinterpret_cast<double*>(const_cast<unsigned long long*>(c64 + (size_t)M * (with_idxsum ? 4 : 1)));
  SH_TRY(launch_finalize(g, M, lm, layers, nullptr, c64, with_idxsum ? c64 + M : nullptr, nullptr, X, w, target_vol, vol,
                         dual, max_rel_err, centroids, nullptr, nullptr, nullptr, static_cast<cudaStream_t>(cuda_stream)));
  return APD_OK;
}

extern "C" int apd_solve_slab(apd_ctx* ctx, const apd_grid* grid, const apd_slab* slab, int32_t M, const float* X,
                              const float* A, const float* target_vol, double tol, const float* w_init, float* w,
                              int32_t* labels, double* vol, uint64_t* counters, apd_reduce_fn reduce, void* user,
                              int32_t* iters, int32_t* evals, double* max_rel_err, double* dual, const apd_opts* opts,
                              void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  if (!slab) { ctx->err = "apd_solve_slab: slab is required"; return APD_E_ARG; }
  return solve_grid(ctx, "apd_solve_slab", grid, slab, M, X, A, target_vol, tol, w_init, w, labels, vol, nullptr, counters,
                    reduce, user, iters, evals, max_rel_err, dual, opts, cuda_stream);
}
