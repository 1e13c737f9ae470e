// apd_points.cu -- NEXT row f3 of DESIGN.md: Algorithm 1 and the reductions of eq. (2.7)-(2.8) on a USER-SUPPLIED
// discretisation, i.e. points y_j with volumes |P_j| ("a triangulation ... with |P_j| the volume of
// the j-th element and y_j its centroid"; masked or locally refined domains work the same way).
//   labels[j] = argmin_i |y_j - x_i|^2_{A_i} - w_i                      (lowest index among equal fp32 costs)
//   vol_i     = sum_{H_j = i} |P_j|            dual = sum_i v_i w_i + sum_j |P_j| min_i C_ij   (identity I1)
//   centroid_i = sum_{H_j = i} |P_j| y_j / vol_i                        (PAPER.md:178 with element volumes)
// Coordinates and volumes stream from HBM (16 B per point and evaluation in 3D -- still far below the ridge for
// M >~ 100 seeds); the per-pair arithmetic is the DIRECT form (no row structure to hoist).  Volumes and centroid
// numerators are fp64 atomics: exact integer counts are gone, results are reproducible to summation order only.
#include "apd_internal.cuh"
#include "apd_device.cuh"
#include <math_constants.h>
#include <cmath>

namespace apd {

constexpr int PT_THREADS = 256;
constexpr int PT_V = 4;                        // points per thread (strided by PT_THREADS: coalesced loads)
constexpr int PT_TILE = PT_THREADS * PT_V;

struct PointArgs {
  int dim;
  long long N;
  int M, M_pad;
  const float* Y;          // [N, dim]
  const float* pvol;       // [N]
  const float* seeds;      // [M_pad, REC] (pack_seeds_kernel)
  int32_t* labels;         // [N] or nullptr
  double* vol;             // [M]   zeroed before the launch
  double* csum;            // [M,3] zeroed before the launch, or nullptr
  double* dual_partial;    // [n_tiles]
  const int* done_flag;    // solve loop only
};

// zeroes the fp64 accumulators of one evaluation (a kernel, so that it can honour done_flag like the rest)
__global__ void points_zero_kernel(int n, double* acc, const int* done_flag) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (done_flag && *done_flag) return;
  if (i < n) acc[i] = 0.0;
}

template <int DIM>
__global__ void __launch_bounds__(PT_THREADS) assign_points_kernel(const PointArgs a) {
  constexpr int REC = (DIM == 3) ? REC3 : REC2;
  constexpr uint32_t CHUNK_BYTES = SEED_CHUNK * REC * sizeof(float);
  __shared__ __align__(128) float s_seeds[SEED_STAGES][SEED_CHUNK * REC];
  __shared__ __align__(8) uint64_t s_full[SEED_STAGES];
  __shared__ double s_red[PT_THREADS / 32];
  if (a.done_flag && *a.done_flag) return;
  const int tid = threadIdx.x;
  const long long j0 = (long long)blockIdx.x * PT_TILE + tid;
  const int nchunks = a.M_pad / SEED_CHUNK;
  if (tid == 0) {
    for (int s = 0; s < SEED_STAGES; ++s) mbar_init(&s_full[s], 1);
    mbar_fence_init();
    for (int s = 0; s < SEED_STAGES && s < nchunks; ++s) {
      mbar_arrive_expect_tx(&s_full[s], CHUNK_BYTES);
      tma_bulk_g2s(s_seeds[s], a.seeds + (size_t)s * SEED_CHUNK * REC, CHUNK_BYTES, &s_full[s]);
    }
  }
  __syncthreads();

  float yx[PT_V], yy[PT_V], yz[PT_V], pv[PT_V], best[PT_V];
  int lab[PT_V];
#pragma unroll
  for (int k = 0; k < PT_V; ++k) {
    const long long j = j0 + (long long)k * PT_THREADS;
    const bool ok = j < a.N;
    yx[k] = ok ? a.Y[j * DIM + 0] : 0.0f;
    yy[k] = ok ? a.Y[j * DIM + 1] : 0.0f;
    yz[k] = (ok && DIM == 3) ? a.Y[j * DIM + 2] : 0.0f;
    pv[k] = ok ? a.pvol[j] : 0.0f;
    best[k] = CUDART_INF_F; lab[k] = 0;
  }

  for (int c = 0; c < nchunks; ++c) {
    const int stage = c % SEED_STAGES;
    mbar_wait(&s_full[stage], (uint32_t)((c / SEED_STAGES) & 1));
    const float4* sp = reinterpret_cast<const float4*>(s_seeds[stage]);
    const int ibase = c * SEED_CHUNK;
#pragma unroll 2
    for (int i = 0; i < SEED_CHUNK; ++i) {
      if (DIM == 3) {
        const float4 p0 = sp[i * 3 + 0], p1 = sp[i * 3 + 1], p2 = sp[i * 3 + 2];
#pragma unroll
        for (int k = 0; k < PT_V; ++k) {
          const float dx = yx[k] - p0.x, dy = yy[k] - p0.y, dz = yz[k] - p0.z;
          const float u = fmaf(p1.y, dz, fmaf(p1.x, dy, p0.w * dx));
          const float v = fmaf(p1.w, dz, p1.z * dy);
          float cst = fmaf(dx, u, p2.y);
          cst = fmaf(dy, v, cst);
          cst = fmaf(dz, p2.x * dz, cst);
          if (cst < best[k]) { best[k] = cst; lab[k] = ibase + i; }
        }
      } else {
        const float4 p0 = sp[i * 2 + 0], p1 = sp[i * 2 + 1];
#pragma unroll
        for (int k = 0; k < PT_V; ++k) {
          const float dx = yx[k] - p0.x, dy = yy[k] - p0.y;
          float cst = fmaf(dx, fmaf(p0.w, dy, p0.z * dx), p1.y);
          cst = fmaf(dy, p1.x * dy, cst);
          if (cst < best[k]) { best[k] = cst; lab[k] = ibase + i; }
        }
      }
    }
    __syncthreads();
    if (tid == 0 && c + SEED_STAGES < nchunks) {
      mbar_arrive_expect_tx(&s_full[stage], CHUNK_BYTES);
      tma_bulk_g2s(s_seeds[stage], a.seeds + (size_t)(c + SEED_STAGES) * SEED_CHUNK * REC, CHUNK_BYTES, &s_full[stage]);
    }
  }

  double dsum = 0.0;
#pragma unroll
  for (int k = 0; k < PT_V; ++k) {
    const long long j = j0 + (long long)k * PT_THREADS;
    if (j < a.N) {
      if (a.labels) a.labels[j] = lab[k];
      const double pj = (double)pv[k];
      dsum += pj * (double)best[k];
      atomicAdd(a.vol + lab[k], pj);
      if (a.csum) {
        atomicAdd(a.csum + (size_t)lab[k] * 3 + 0, pj * (double)yx[k]);
        atomicAdd(a.csum + (size_t)lab[k] * 3 + 1, pj * (double)yy[k]);
        if (DIM == 3) atomicAdd(a.csum + (size_t)lab[k] * 3 + 2, pj * (double)yz[k]);
      }
    }
  }
  const double tot = block_sum_double<PT_THREADS>(dsum, s_red);
  if (tid == 0) a.dual_partial[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) finalize_points_kernel(
    int dim, int M, int n_partials, const double* __restrict__ vol_acc, const double* __restrict__ csum,
    const double* __restrict__ dual_partial, const float* __restrict__ X, const float* __restrict__ w,
    const float* __restrict__ target_vol, double* __restrict__ vol, double* __restrict__ dual,
    double* __restrict__ max_rel_err, double* __restrict__ centroids) {
  __shared__ double scratch[1024 / 32];
  __shared__ double s_out[3];
  const int tid = threadIdx.x;
  double vw = 0.0, err = 0.0, smin = 0.0;
  for (int i = tid; i < M; i += 1024) {
    const double vi = vol_acc[i];
    vol[i] = vi;
    if (target_vol) {
      const double tv = (double)target_vol[i];
      vw += tv * (double)w[i];
      err = fmax(err, fabs(vi - tv) / tv);
    }
    if (centroids) {
      for (int k = 0; k < dim; ++k)
        centroids[(size_t)i * dim + k] = (vi > 0.0) ? csum[(size_t)i * 3 + k] / vi : (double)X[(size_t)i * dim + k];
    }
  }
  for (int t = tid; t < n_partials; t += 1024) smin += dual_partial[t];
  const double a0 = block_sum_double<1024>(vw, scratch);
  if (tid == 0) s_out[0] = a0;
  __syncthreads();
  const double a1 = block_sum_double<1024>(smin, scratch);
  if (tid == 0) s_out[1] = a1;
  __syncthreads();
  // max: reuse the sum helper's scratch with a shuffle max
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) err = fmax(err, __shfl_down_sync(0xffffffffu, err, o));
  if ((tid & 31) == 0) scratch[tid >> 5] = err;
  __syncthreads();
  if (tid == 0) {
    double e = 0.0;
    for (int i = 0; i < 1024 / 32; ++i) e = fmax(e, scratch[i]);
    *dual = s_out[0] + s_out[1];
    if (max_rel_err && target_vol) *max_rel_err = e;
  }
}

}  // namespace apd

using namespace apd;

#define PT_TRY(call)                                                                \
  do {                                                                              \
    cudaError_t e__ = (call);                                                       \
    if (e__ != cudaSuccess) {                                                       \
      ctx->err = std::string(#call) + ": " + cudaGetErrorString(e__);               \
      return APD_E_CUDA;                                                            \
    }                                                                               \
  } while (0)

namespace apd {

int points_prepare(apd_ctx* ctx, long long N, int* n_partials, cudaStream_t st) {
  Workspace& ws = ctx->ws;
  const long long n_tiles_ll = (N + PT_TILE - 1) / PT_TILE;
  if (n_tiles_ll > 0x7fffffffll) { ctx->err = "apd points: too many points"; return APD_E_ARG; }
  const int n_tiles = (int)n_tiles_ll;
  if ((size_t)n_tiles > ws.partial_cap) {
    PT_TRY(cudaStreamSynchronize(st));
    PT_TRY(cudaFree(ws.dual_partial));
    ws.dual_partial = nullptr;
    ws.partial_cap = (size_t)n_tiles;
    PT_TRY(cudaMalloc(&ws.dual_partial, ws.partial_cap * sizeof(double)));
  }
  if (!ws.pt_acc) PT_TRY(cudaMalloc(&ws.pt_acc, (size_t)ws.max_seeds * 4 * sizeof(double)));   // vol[M] | csum[M,3]
  const size_t n_layers = (size_t)points_layer_map(n_tiles).n_layers;          // lbfgs_step_kernel's two-level sum
  if (n_layers > ws.layer_cap) {
    PT_TRY(cudaStreamSynchronize(st));
    cudaFree(ws.layer_buf);
    ws.layer_buf = nullptr; ws.layer_cap = 0;
    PT_TRY(cudaMalloc(&ws.layer_buf, n_layers * sizeof(double)));
    ws.layer_cap = n_layers;
  }
  *n_partials = n_tiles;
  return APD_OK;
}

int enqueue_points(apd_ctx* ctx, long long N, const float* Y, const float* pvol, int M, const float* X, const float* A,
                   const float* w, const float* target_vol, int32_t* labels, double* vol, double* dual,
                   double* max_rel_err, double* centroids, const int* done_flag, int* n_partials, cudaStream_t st) {
  Workspace& ws = ctx->ws;
  int rc = points_prepare(ctx, N, n_partials, st);
  if (rc != APD_OK) return rc;
  const int d = ws.dim, n_tiles = *n_partials;
  const int M_pad = (M + SEED_CHUNK - 1) / SEED_CHUNK * SEED_CHUNK;
  const int n_acc = ws.max_seeds * 4;
  points_zero_kernel<<<(n_acc + 255) / 256, 256, 0, st>>>(n_acc, ws.pt_acc, done_flag);
  PT_TRY(cudaGetLastError());
  PT_TRY(launch_pack_seeds(d, M, M_pad, X, A, w, ws.seeds, ws.count, nullptr, done_flag, st));
  PointArgs a;
  a.dim = d; a.N = N; a.M = M; a.M_pad = M_pad; a.Y = Y; a.pvol = pvol; a.seeds = ws.seeds; a.labels = labels;
  a.vol = ws.pt_acc; a.csum = centroids ? ws.pt_acc + ws.max_seeds : nullptr; a.dual_partial = ws.dual_partial;
  a.done_flag = done_flag;
  if (d == 3) assign_points_kernel<3><<<n_tiles, PT_THREADS, 0, st>>>(a);
  else        assign_points_kernel<2><<<n_tiles, PT_THREADS, 0, st>>>(a);
  PT_TRY(cudaGetLastError());
  if (vol) {
    finalize_points_kernel<<<1, 1024, 0, st>>>(d, M, n_tiles, ws.pt_acc, a.csum, ws.dual_partial, X, w, target_vol, vol,
                                               dual, max_rel_err, centroids);
    PT_TRY(cudaGetLastError());
  }
  return APD_OK;
}

}  // namespace apd

extern "C" int apd_assign_points(apd_ctx* ctx, int64_t N, const float* Y, const float* pvol, int32_t M, const float* X,
                                 const float* A, const float* w, const float* target_vol, int32_t* labels,
                                 double* vol, double* dual, double* max_rel_err, double* centroids,
                                 void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  Workspace& ws = ctx->ws;
  if (N < 1 || N >= (1ll << 40)) { ctx->err = "apd_assign_points: N out of range"; return APD_E_ARG; }
  if (M < 1 || M > ws.max_seeds) { ctx->err = "apd_assign_points: M out of range [1, max_seeds]"; return APD_E_ARG; }
  if (!Y || !pvol || !X || !A || !w || !vol || !dual) { ctx->err = "apd_assign_points: Y, pvol, X, A, w, vol and dual are required"; return APD_E_ARG; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  PT_TRY(cudaSetDevice(ws.device));
  int n_partials = 0;
  return enqueue_points(ctx, N, Y, pvol, M, X, A, w, target_vol, labels, vol, dual, max_rel_err, centroids, nullptr,
                        &n_partials, st);
}
