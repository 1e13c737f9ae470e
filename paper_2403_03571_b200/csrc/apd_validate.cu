// apd_validate.cu -- apd_validate: the input checks the hot path does NOT make (finiteness of X / A / w,
// symmetry and positive definiteness of A -- the paper's standing assumption, on which the culling
// bound rests -- and the target volumes of PAPER.md:65-69).  A debug call: one small kernel, one flag word back.
#include "apd_internal.cuh"
#include <cmath>
#include <math_constants.h>

#define APD_CUDA_TRY(ctx, call)                                                              \
  do {                                                                                       \
    cudaError_t e__ = (call);                                                                \
    if (e__ != cudaSuccess) {                                                                \
      (ctx)->err = std::string("apd_validate: ") + #call + ": " + cudaGetErrorString(e__);   \
      return APD_E_CUDA;                                                                     \
    }                                                                                        \
  } while (0)

namespace apd {

template <int DIM>
__global__ void validate_kernel(int M, const float* __restrict__ X, const float* __restrict__ A,
                                const float* __restrict__ w, const float* __restrict__ v, unsigned int* __restrict__ flags,
                                double* __restrict__ vsum) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int f = 0u;
  double vi = 0.0;
  if (i < M) {
    for (int k = 0; k < DIM; ++k) if (!isfinite(X[i * DIM + k])) f |= APD_BAD_X_NONFINITE;
    const float* a = A + (size_t)i * DIM * DIM;
    float amax = 0.0f;
    bool fin = true;
    for (int k = 0; k < DIM * DIM; ++k) { fin = fin && isfinite(a[k]); amax = fmaxf(amax, fabsf(a[k])); }
    if (!fin) f |= APD_BAD_A_NONFINITE;
    else {
      // symmetry: |A_kl - A_lk| <= 1e-6 max|A| (fp32 inputs)
      bool sym = true;
      for (int k = 0; k < DIM; ++k)
        for (int l = k + 1; l < DIM; ++l) sym = sym && (fabsf(a[k * DIM + l] - a[l * DIM + k]) <= 1e-6f * amax);
      if (!sym) f |= APD_BAD_A_NOT_SYMMETRIC;
      // positive definiteness of the symmetric part (the quadratic form only sees it): leading principal minors in fp64
      const double s11 = a[0], s12 = 0.5 * ((double)a[1] + (double)a[DIM]), s22 = a[DIM + 1];
      bool pd = s11 > 0.0 && s11 * s22 - s12 * s12 > 0.0;
      if (DIM == 3 && pd) {
        const double s13 = 0.5 * ((double)a[2] + (double)a[6]), s23 = 0.5 * ((double)a[5] + (double)a[7]), s33 = a[8];
        const double det = s11 * (s22 * s33 - s23 * s23) - s12 * (s12 * s33 - s23 * s13) + s13 * (s12 * s23 - s22 * s13);
        pd = det > 0.0;
      }
      if (!pd) f |= APD_BAD_A_NOT_POSITIVE_DEFINITE;
    }
    if (w && !isfinite(w[i])) f |= APD_BAD_W_NONFINITE;
    if (v) {
      vi = (double)v[i];
      if (!(vi > 0.0) || !isfinite(vi)) { f |= APD_BAD_TARGET_VOL_NOT_POSITIVE; vi = 0.0; }
    }
  }
  // one atomic per warp for the flags and the volume sum (a debug call: the order of the fp64 additions is not fixed,
  // the sum is only held to 1e-6 relative)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { f |= __shfl_xor_sync(0xffffffffu, f, o); vi += __shfl_xor_sync(0xffffffffu, vi, o); }
  if ((threadIdx.x & 31) == 0) {
    if (f) atomicOr(flags, f);
    if (v) atomicAdd(vsum, vi);
  }
}

}  // namespace apd

using namespace apd;

extern "C" int apd_validate(apd_ctx* ctx, const apd_grid* grid, int32_t M, const float* X, const float* A, const float* w,
                            const float* target_vol, uint32_t* problems, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (!problems || !X || !A) { ctx->err = "apd_validate: X, A and problems are required"; return APD_E_ARG; }
  if (M < 1 || M > ctx->ws.max_seeds) { ctx->err = "apd_validate: M out of range [1, max_seeds]"; return APD_E_ARG; }
  if (target_vol && !grid) { ctx->err = "apd_validate: grid is required with target_vol (the volumes must sum to |Omega|)"; return APD_E_ARG; }
  double domain = 1.0;
  if (grid) {
    if (grid->dim != ctx->ws.dim) { ctx->err = "apd_validate: grid.dim differs from the context's dim"; return APD_E_ARG; }
    for (int k = 0; k < grid->dim; ++k) {
      if (!(grid->hi[k] > grid->lo[k]) || !std::isfinite(grid->hi[k]) || !std::isfinite(grid->lo[k])) {
        ctx->err = "apd_validate: grid needs finite hi[k] > lo[k]";
        return APD_E_ARG;
      }
      domain *= grid->hi[k] - grid->lo[k];
    }
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  APD_CUDA_TRY(ctx, cudaSetDevice(ctx->ws.device));
  struct Out { unsigned int flags; unsigned int pad; double vsum; } h = {0u, 0u, 0.0};
  Out* d = nullptr;
  APD_CUDA_TRY(ctx, cudaMalloc(&d, sizeof(Out)));
  cudaError_t e = cudaMemsetAsync(d, 0, sizeof(Out), st);
  if (e == cudaSuccess) {
    const int nb = (M + 127) / 128;
    if (ctx->ws.dim == 3) validate_kernel<3><<<nb, 128, 0, st>>>(M, X, A, w, target_vol, &d->flags, &d->vsum);
    else                  validate_kernel<2><<<nb, 128, 0, st>>>(M, X, A, w, target_vol, &d->flags, &d->vsum);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, d, sizeof(Out), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d);
  APD_CUDA_TRY(ctx, e);
  uint32_t f = h.flags;
  if (target_vol && !(std::fabs(h.vsum - domain) <= 1e-6 * domain)) f |= APD_BAD_TARGET_VOL_SUM;
  *problems = f;
  return APD_OK;
}
