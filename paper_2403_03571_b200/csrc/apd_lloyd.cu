// apd_lloyd.cu -- NEXT rows f1 and f2 of DESIGN.md: Algorithm 3 (generalised Lloyd) as a host loop
// over apd_solve + the discrete centroids of the same pass, and the resolution rules of PAPER.md:182-197.
#include "apd_internal.cuh"
#include <cmath>
#include <vector>

namespace apd {

// x_i^{k+1} = fl32(discrete centroid of cell i)  (an empty cell keeps its seed, reading S5 --
// the finalize kernel already wrote x_i into `centroids` for it)
__global__ void centroids_to_seeds_kernel(int n, const double* __restrict__ centroids, float* __restrict__ X) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) X[i] = (float)centroids[i];
}

}  // namespace apd

using namespace apd;

#define LL_TRY(call)                                                                \
  do {                                                                              \
    cudaError_t e__ = (call);                                                       \
    if (e__ != cudaSuccess) {                                                       \
      ctx->err = std::string(#call) + ": " + cudaGetErrorString(e__);               \
      rc = APD_E_CUDA;                                                              \
      goto done;                                                                    \
    }                                                                               \
  } while (0)

extern "C" int apd_lloyd(apd_ctx* ctx, const apd_grid* grid, int32_t M, float* X, const float* A,
                         const float* target_vol, double tol, int32_t K, const float* w_init, float* w,
                         int32_t* labels, double* vol, int32_t* iters, int32_t* evals, double* max_rel_err,
                         const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (K < 0) { ctx->err = "apd_lloyd: K must be >= 0"; return APD_E_ARG; }
  if (!grid || !X || !A || !target_vol || !w || M < 1) { ctx->err = "apd_lloyd: grid, X, A, target_vol and w are required"; return APD_E_ARG; }
  const int d = grid->dim;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double *cen = nullptr, *v64 = nullptr, *scal = nullptr;
  int rc = APD_OK, it_sum = 0, ev_sum = 0;
  double err = 0.0;
  if (cudaSetDevice(ctx->ws.device) != cudaSuccess) { ctx->err = "apd_lloyd: cudaSetDevice failed"; return APD_E_CUDA; }
  {
    // scratch of the centroid evaluation: owned by the context, allocated once (apd_reserve does it ahead of time)
    Workspace& ws = ctx->ws;
    if (!ws.lloyd_buf) LL_TRY(cudaMalloc(&ws.lloyd_buf, ((size_t)ws.max_seeds * (ws.dim + 1) + 2) * sizeof(double)));
    cen = ws.lloyd_buf; v64 = cen + (size_t)ws.max_seeds * ws.dim; scal = v64 + ws.max_seeds;
  }
  for (int k = 0; k <= K; ++k) {
    // Alg. 3 step 4 / 8: Algorithm 2 from W_0^k (W_0^0 = w_init or 0, then W_0^{k+1} = W^k)
    int it = 0, ev = 0;
    const bool last = (k == K);
    rc = apd_solve(ctx, grid, M, X, A, target_vol, tol, k == 0 ? w_init : w, w, last ? labels : nullptr,
                   last ? vol : nullptr, nullptr, &it, &ev, &err, nullptr, opts, cuda_stream);
    it_sum += it; ev_sum += ev;
    if (rc < 0) goto done;
    if (last) break;
    // Alg. 3 step 5: seeds <- discrete centroids of the APD just found (one more evaluation, with index sums)
    rc = apd_assign(ctx, grid, M, X, A, w, target_vol, nullptr, v64, scal, scal + 1, cen, nullptr, opts, cuda_stream);
    if (rc < 0) goto done;
    centroids_to_seeds_kernel<<<(M * d + 255) / 256, 256, 0, st>>>(M * d, cen, X);
    LL_TRY(cudaGetLastError());
  }
  LL_TRY(cudaStreamSynchronize(st));
done:
  if (iters) *iters = it_sum;
  if (evals) *evals = ev_sum;
  if (max_rel_err) *max_rel_err = err;
  return rc;
}

// Algorithm 3 on a user-supplied discretisation (points y_j with volumes |P_j|): the same loop with
// apd_solve_points / apd_assign_points; the centroid of a cell is sum |P_j| y_j / sum |P_j| over its points.
extern "C" int apd_lloyd_points(apd_ctx* ctx, int64_t N, const float* Y, const float* pvol, double total_volume, int32_t M,
                                float* X, const float* A, const float* target_vol, double tol, int32_t K,
                                const float* w_init, float* w, int32_t* labels, double* vol, int32_t* iters,
                                int32_t* evals, double* max_rel_err, const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (K < 0) { ctx->err = "apd_lloyd_points: K must be >= 0"; return APD_E_ARG; }
  if (!Y || !pvol || !X || !A || !target_vol || !w || M < 1 || N < 1) { ctx->err = "apd_lloyd_points: Y, pvol, X, A, target_vol and w are required"; return APD_E_ARG; }
  const int d = ctx->ws.dim;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double *cen = nullptr, *v64 = nullptr, *scal = nullptr;
  int rc = APD_OK, it_sum = 0, ev_sum = 0;
  double err = 0.0;
  if (cudaSetDevice(ctx->ws.device) != cudaSuccess) { ctx->err = "apd_lloyd_points: cudaSetDevice failed"; return APD_E_CUDA; }
  {
    Workspace& ws = ctx->ws;
    if (!ws.lloyd_buf) LL_TRY(cudaMalloc(&ws.lloyd_buf, ((size_t)ws.max_seeds * (ws.dim + 1) + 2) * sizeof(double)));
    cen = ws.lloyd_buf; v64 = cen + (size_t)ws.max_seeds * ws.dim; scal = v64 + ws.max_seeds;
  }
  for (int k = 0; k <= K; ++k) {
    int it = 0, ev = 0;
    const bool last = (k == K);
    rc = apd_solve_points(ctx, N, Y, pvol, total_volume, M, X, A, target_vol, tol, k == 0 ? w_init : w, w,
                          last ? labels : nullptr, last ? vol : nullptr, &it, &ev, &err, opts, cuda_stream);
    it_sum += it; ev_sum += ev;
    if (rc < 0) goto done;
    if (last) break;
    rc = apd_assign_points(ctx, N, Y, pvol, M, X, A, w, target_vol, nullptr, v64, scal, scal + 1, cen, cuda_stream);
    if (rc < 0) goto done;
    centroids_to_seeds_kernel<<<(M * d + 255) / 256, 256, 0, st>>>(M * d, cen, X);
    LL_TRY(cudaGetLastError());
  }
  LL_TRY(cudaStreamSynchronize(st));
done:
  if (iters) *iters = it_sum;
  if (evals) *evals = ev_sum;
  if (max_rel_err) *max_rel_err = err;
  return rc;
}

// PAPER.md:182-197.  Smallest integer M (voxels per axis of a cubic grid on a domain of volume |Omega|) with
//   |Omega| / M^D < factor * v_min,   factor = eps (necessary, eq. 2.9 for general v) or eps / 2^D (practical, eq. 2.10).
extern "C" double apd_resolution_bound(int32_t dim, double domain_volume, double v_min, double eps, int32_t practical) {
  if ((dim != 2 && dim != 3) || !(domain_volume > 0.0) || !(v_min > 0.0) || !(eps > 0.0)) return -1.0;
  const double factor = practical ? eps / std::pow(2.0, (double)dim) : eps;
  return std::pow(domain_volume / (factor * v_min), 1.0 / (double)dim);   // M must be GREATER than this
}

extern "C" int32_t apd_choose_resolution(int32_t dim, double domain_volume, double v_min, double eps, int32_t practical) {
  const double b = apd_resolution_bound(dim, domain_volume, v_min, eps, practical);
  if (!(b >= 0.0) || b > 2.0e9) return -1;
  long long m = (long long)std::floor(b) + 1;                              // first integer strictly above the bound
  // guard the strict inequality against the rounding of pow()
  const double factor = practical ? eps / std::pow(2.0, (double)dim) : eps;
  while (m > 1 && domain_volume / std::pow((double)(m - 1), (double)dim) < factor * v_min) --m;
  while (!(domain_volume / std::pow((double)m, (double)dim) < factor * v_min)) ++m;
  return (int32_t)m;
}

// Algorithm 2 step 4: "if it is not possible to hit the desired tolerance, increase J and restart".
// The paper gives no rule for the increase (reading S18): every refinement doubles the voxels per axis and
// restarts Algorithm 2 from the best weights found so far (the weights do not depend on the resolution).
extern "C" int apd_solve_refine(apd_ctx* ctx, apd_grid* grid, int32_t M, const float* X, const float* A,
                                const float* target_vol, double tol, int32_t max_refinements, const float* w_init,
                                float* w, double* vol, int32_t* refinements, int32_t* iters, int32_t* evals,
                                double* max_rel_err, const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (!grid || max_refinements < 0 || !w) { ctx->err = "apd_solve_refine: grid, w required, max_refinements >= 0"; return APD_E_ARG; }
  int it_sum = 0, ev_sum = 0, r = 0, rc = APD_OK;
  double err = 0.0;
  for (;; ++r) {
    int it = 0, ev = 0;
    rc = apd_solve(ctx, grid, M, X, A, target_vol, tol, r == 0 ? w_init : w, w, nullptr, vol, nullptr, &it, &ev, &err,
                   nullptr, opts, cuda_stream);
    it_sum += it; ev_sum += ev;
    if (rc != APD_NOT_CONVERGED || r == max_refinements) break;
    long long nvox = 1;
    for (int k = 0; k < grid->dim; ++k) nvox *= 2ll * grid->n[k];
    if (nvox >= (1ll << 31)) break;                       // the next grid would exceed the index range
    for (int k = 0; k < grid->dim; ++k) grid->n[k] *= 2;
  }
  if (refinements) *refinements = r;
  if (iters) *iters = it_sum;
  if (evals) *evals = ev_sum;
  if (max_rel_err) *max_rel_err = err;
  return rc;
}

// Coarse-to-fine continuation ("natural extension" of Alg. 2 step 4): the weights do
// not depend on the resolution, so Algorithm 2 is run on the grid coarsened by 2^levels, ..., 2, 1 per axis, each level
// started from the weights of the one before; only the last level runs on `grid` itself, and it starts almost converged.
extern "C" int apd_solve_continuation(apd_ctx* ctx, const apd_grid* grid, int32_t levels, int32_t M, const float* X,
                                      const float* A, const float* target_vol, double tol, const float* w_init, float* w,
                                      int32_t* labels, double* vol, int32_t* iters, int32_t* evals, double* max_rel_err,
                                      const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (!grid || !w || levels < 0 || levels > 8) { ctx->err = "apd_solve_continuation: grid, w required, 0 <= levels <= 8"; return APD_E_ARG; }
  if (grid->dim != 2 && grid->dim != 3) { ctx->err = "apd_solve_continuation: grid.dim must be 2 or 3"; return APD_E_ARG; }
  if (!target_vol || M < 1 || M > ctx->ws.max_seeds) { ctx->err = "apd_solve_continuation: target_vol required, 1 <= M <= max_seeds"; return APD_E_ARG; }
  int rc = APD_OK;
  double err = 0.0;
  bool started = false;
  // smallest target volume (host copy of the M floats): a coarse level is only asked for the tolerance its voxels can
  // resolve, the paper's practical rule eq. (2.10) read backwards: eps_l = max(tol, 2^D |P_l| / v_min)
  double v_min = 0.0;
  if (levels > 0) {
    std::vector<float> hv((size_t)M);
    if (cudaSetDevice(ctx->ws.device) != cudaSuccess ||
        cudaStreamSynchronize(static_cast<cudaStream_t>(cuda_stream)) != cudaSuccess ||
        cudaMemcpy(hv.data(), target_vol, sizeof(float) * (size_t)M, cudaMemcpyDeviceToHost) != cudaSuccess) {
      ctx->err = "apd_solve_continuation: could not read target_vol";
      return APD_E_CUDA;
    }
    v_min = (double)hv[0];
    for (int i = 1; i < M; ++i) v_min = std::fmin(v_min, (double)hv[i]);
    if (!(v_min > 0.0)) { ctx->err = "apd_solve_continuation: target_vol must be > 0"; return APD_E_ARG; }
  }
  for (int l = levels; l >= 0; --l) {
    apd_grid g = *grid;
    bool too_coarse = false;
    double P = 1.0;
    for (int k = 0; k < grid->dim; ++k) {
      g.n[k] = (grid->n[k] + (1 << l) - 1) >> l;
      if (l > 0 && g.n[k] < 16) too_coarse = true;          // a level this coarse says nothing about the cells
      P *= (grid->hi[k] - grid->lo[k]) / (double)g.n[k];
    }
    int it = 0, ev = 0;
    if (!too_coarse) {
      const bool last = (l == 0);
      const double tol_l = last ? tol : std::fmax(tol, std::pow(2.0, (double)grid->dim) * P / v_min);
      rc = apd_solve(ctx, &g, M, X, A, target_vol, tol_l, started ? w : w_init, w, last ? labels : nullptr,
                     last ? vol : nullptr, nullptr, &it, &ev, &err, nullptr, opts, cuda_stream);
      if (rc < 0) return rc;
      started = true;
    }
    if (iters) iters[levels - l] = it;
    if (evals) evals[levels - l] = ev;
  }
  if (max_rel_err) *max_rel_err = err;
  return rc;
}
