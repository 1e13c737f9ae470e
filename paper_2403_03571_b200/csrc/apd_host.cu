// apd_host.cu -- apd_assign_host / apd_solve_host: the same calls with HOST arrays.  The library
// copies in (cudaMemcpyAsync, one per array), runs the device call, copies out (apd_assign_host writes the labels
// in place when they live in pinned host memory).  The device
// buffers belong to the context: grow-only, reused by the next host call, freed by apd_destroy
// (a 64 MiB cudaMalloc + cudaFree per call cost more than the label copy).  Used for the
// end-to-end ("e2e") measurement and by callers without a device allocator of their own.
#include "apd_internal.cuh"
#include <cstdint>

namespace {

// hands out the context's scratch slots in call order
struct DevBufs {
  apd::Workspace& ws;
  int next = 0;
  explicit DevBufs(apd::Workspace& w) : ws(w) {}
  template <typename T>
  cudaError_t alloc(T** out, size_t count) {
    if (next >= apd::Workspace::HOST_SLOTS) return cudaErrorMemoryAllocation;
    const int k = next++;                       // count == 0 (an optional array not asked for) still takes its slot
    const size_t bytes = count * sizeof(T);
    if (bytes == 0) { *out = nullptr; return cudaSuccess; }
    if (ws.host_cap[k] < bytes) {
      cudaFree(ws.host_buf[k]);
      ws.host_buf[k] = nullptr; ws.host_cap[k] = 0;
      cudaError_t e = cudaMalloc(&ws.host_buf[k], bytes);
      if (e != cudaSuccess) return e;
      ws.host_cap[k] = bytes;
    }
    *out = static_cast<T*>(ws.host_buf[k]);
    return cudaSuccess;
  }
};

#define HOST_TRY(call)                                                              \
  do {                                                                              \
    cudaError_t e__ = (call);                                                       \
    if (e__ != cudaSuccess) {                                                       \
      ctx->err = std::string(#call) + ": " + cudaGetErrorString(e__);               \
      return APD_E_CUDA;                                                            \
    }                                                                               \
  } while (0)

long long grid_voxels(const apd_grid* g) {
  long long N = 1;
  for (int k = 0; k < g->dim && k < 3; ++k) N *= (g->n[k] > 0 ? g->n[k] : 0);
  return N;
}

}  // namespace

extern "C" int apd_assign_host(apd_ctx* ctx, const apd_grid* grid, int32_t M, const float* X, const float* A,
                               const float* w, const float* target_vol, int32_t* labels, double* vol,
                               double* dual, double* max_rel_err, double* centroids,
                               uint64_t* pairs_evaluated, const apd_opts* opts) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (!grid || (grid->dim != 2 && grid->dim != 3) || M < 1 || !X || !A || !w || !vol || !dual) {
    ctx->err = "apd_assign_host: bad arguments";
    return APD_E_ARG;
  }
  const int d = grid->dim;
  const long long N = grid_voxels(grid);
  if (N < 1 || N >= (1ll << 31)) { ctx->err = "apd_assign_host: bad grid"; return APD_E_ARG; }
  HOST_TRY(cudaSetDevice(ctx->ws.device));
  DevBufs b(ctx->ws);
  float *dX, *dA, *dw, *dv = nullptr;
  int32_t* dl = nullptr;
  double *dvol, *dscal, *dcen = nullptr;
  uint64_t* dpairs;
  HOST_TRY(b.alloc(&dX, (size_t)M * d));
  HOST_TRY(b.alloc(&dA, (size_t)M * d * d));
  HOST_TRY(b.alloc(&dw, (size_t)M));
  HOST_TRY(b.alloc(&dv, target_vol ? (size_t)M : 0));
  // labels in page-locked (pinned) host memory are device-accessible: the kernel then stores them straight there
  // (posted writes over the host link, overlapped with the evaluation) instead of into a device buffer that is copied
  // out afterwards -- the 4N bytes cross the link either way, but not after the kernel
  int32_t* dl_direct = nullptr;
  if (labels) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, labels) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer &&
        (reinterpret_cast<uintptr_t>(at.devicePointer) & 15) == 0)
      dl_direct = static_cast<int32_t*>(at.devicePointer);
    else
      cudaGetLastError();          // pageable memory: not an error, take the copy path
  }
  HOST_TRY(b.alloc(&dl, labels && !dl_direct ? (size_t)N : 0));
  HOST_TRY(b.alloc(&dvol, (size_t)M));
  HOST_TRY(b.alloc(&dscal, 2));
  HOST_TRY(b.alloc(&dcen, centroids ? (size_t)M * d : 0));
  HOST_TRY(b.alloc(&dpairs, 1));
  cudaStream_t st = nullptr;
  HOST_TRY(cudaMemcpyAsync(dX, X, sizeof(float) * M * d, cudaMemcpyHostToDevice, st));
  HOST_TRY(cudaMemcpyAsync(dA, A, sizeof(float) * M * d * d, cudaMemcpyHostToDevice, st));
  HOST_TRY(cudaMemcpyAsync(dw, w, sizeof(float) * M, cudaMemcpyHostToDevice, st));
  if (target_vol) HOST_TRY(cudaMemcpyAsync(dv, target_vol, sizeof(float) * M, cudaMemcpyHostToDevice, st));
  HOST_TRY(cudaMemsetAsync(dscal, 0, 2 * sizeof(double), st));
  const int rc = apd_assign(ctx, grid, M, dX, dA, dw, dv, dl_direct ? dl_direct : dl, dvol, dscal, dscal + 1, dcen, dpairs, opts, st);
  if (rc != APD_OK) return rc;
  if (labels && !dl_direct) HOST_TRY(cudaMemcpyAsync(labels, dl, sizeof(int32_t) * N, cudaMemcpyDeviceToHost, st));
  HOST_TRY(cudaMemcpyAsync(vol, dvol, sizeof(double) * M, cudaMemcpyDeviceToHost, st));
  double scal[2] = {0, 0};
  HOST_TRY(cudaMemcpyAsync(scal, dscal, sizeof(scal), cudaMemcpyDeviceToHost, st));
  if (centroids) HOST_TRY(cudaMemcpyAsync(centroids, dcen, sizeof(double) * M * d, cudaMemcpyDeviceToHost, st));
  uint64_t pairs = 0;
  HOST_TRY(cudaMemcpyAsync(&pairs, dpairs, sizeof(pairs), cudaMemcpyDeviceToHost, st));
  HOST_TRY(cudaStreamSynchronize(st));
  *dual = scal[0];
  if (max_rel_err && target_vol) *max_rel_err = scal[1];
  if (pairs_evaluated) *pairs_evaluated = pairs;
  return APD_OK;
}

extern "C" int apd_solve_host(apd_ctx* ctx, const apd_grid* grid, int32_t M, const float* X, const float* A,
                              const float* target_vol, double tol, const float* w_init, float* w,
                              int32_t* labels, double* vol, double* w64, int32_t* iters, int32_t* evals,
                              double* max_rel_err, double* dual, const apd_opts* opts) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (!grid || (grid->dim != 2 && grid->dim != 3) || M < 1 || !X || !A || !target_vol || !w) {
    ctx->err = "apd_solve_host: bad arguments";
    return APD_E_ARG;
  }
  const int d = grid->dim;
  const long long N = grid_voxels(grid);
  if (N < 1 || N >= (1ll << 31)) { ctx->err = "apd_solve_host: bad grid"; return APD_E_ARG; }
  HOST_TRY(cudaSetDevice(ctx->ws.device));
  DevBufs b(ctx->ws);
  float *dX, *dA, *dv, *dwi = nullptr, *dw;
  int32_t* dl = nullptr;
  double *dvol = nullptr, *dw64 = nullptr;
  HOST_TRY(b.alloc(&dX, (size_t)M * d));
  HOST_TRY(b.alloc(&dA, (size_t)M * d * d));
  HOST_TRY(b.alloc(&dv, (size_t)M));
  HOST_TRY(b.alloc(&dwi, w_init ? (size_t)M : 0));
  HOST_TRY(b.alloc(&dw, (size_t)M));
  HOST_TRY(b.alloc(&dl, labels ? (size_t)N : 0));
  HOST_TRY(b.alloc(&dvol, vol ? (size_t)M : 0));
  HOST_TRY(b.alloc(&dw64, w64 ? (size_t)M : 0));
  cudaStream_t st = nullptr;
  HOST_TRY(cudaMemcpyAsync(dX, X, sizeof(float) * M * d, cudaMemcpyHostToDevice, st));
  HOST_TRY(cudaMemcpyAsync(dA, A, sizeof(float) * M * d * d, cudaMemcpyHostToDevice, st));
  HOST_TRY(cudaMemcpyAsync(dv, target_vol, sizeof(float) * M, cudaMemcpyHostToDevice, st));
  if (w_init) HOST_TRY(cudaMemcpyAsync(dwi, w_init, sizeof(float) * M, cudaMemcpyHostToDevice, st));
  const int rc = apd_solve(ctx, grid, M, dX, dA, dv, tol, dwi, dw, dl, dvol, dw64, iters, evals, max_rel_err,
                           dual, opts, st);
  if (rc < 0) return rc;
  HOST_TRY(cudaMemcpyAsync(w, dw, sizeof(float) * M, cudaMemcpyDeviceToHost, st));
  if (labels) HOST_TRY(cudaMemcpyAsync(labels, dl, sizeof(int32_t) * N, cudaMemcpyDeviceToHost, st));
  if (vol) HOST_TRY(cudaMemcpyAsync(vol, dvol, sizeof(double) * M, cudaMemcpyDeviceToHost, st));
  if (w64) HOST_TRY(cudaMemcpyAsync(w64, dw64, sizeof(double) * M, cudaMemcpyDeviceToHost, st));
  HOST_TRY(cudaStreamSynchronize(st));
  return rc;
}
