// apd_kernels.cu -- seed packing, the DIRECT voxel x seed kernel, and the finalize reduction.
//
// Path rows (SURVEY.md 8(a) / DESIGN.md): a1 voxel coordinates from the thread index, a2 seed
// pack + TMA staging, a3 cost C_ij = |y_j - x_i|^2_{A_i} - w_i (eq. 2.1 at
// PAPER.md:58-61), a4 argmin, a5 label store, a6 per-cell counts / index sums /
// sum of min-costs, a9 finalize: vol, dual (eq. 2.7-2.8), eq. (2.5) error,
// centroids.
#include "apd_internal.cuh"
#include "apd_device.cuh"
#include "apd_epilogue.cuh"
#include <math_constants.h>

namespace apd {

// ------------------------------------------------------------------------------------------
// a2: pack seeds.  One thread per (padded) seed.  Also zeroes the integer accumulators.
// ------------------------------------------------------------------------------------------
template <int DIM>
__global__ void pack_seeds_kernel(int M, int M_pad, const float* __restrict__ X,
                                  const float* __restrict__ A, const float* __restrict__ w,
                                  float* __restrict__ seeds, unsigned int* __restrict__ count,
                                  unsigned long long* __restrict__ idxsum, const int* __restrict__ done_flag) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M_pad) return;
  if (done_flag && *done_flag) return;
  constexpr int REC = (DIM == 3) ? REC3 : REC2;
  float r[REC];
#pragma unroll
  for (int k = 0; k < REC; ++k) r[k] = 0.0f;
  if (i < M) {
    if (DIM == 3) {
      const float* a = A + (size_t)i * 9;
      r[0] = X[i * 3 + 0]; r[1] = X[i * 3 + 1]; r[2] = X[i * 3 + 2];
      r[3] = a[0];                 // a11
      r[4] = a[1] + a[3];          // a12' = A01 + A10
      r[5] = a[2] + a[6];          // a13'
      r[6] = a[4];                 // a22
      r[7] = a[5] + a[7];          // a23'
      r[8] = a[8];                 // a33
      r[9] = -w[i];                // nw
    } else {
      const float* a = A + (size_t)i * 4;
      r[0] = X[i * 2 + 0]; r[1] = X[i * 2 + 1];
      r[2] = a[0];                 // a11
      r[3] = a[1] + a[2];          // a12'
      r[4] = a[3];                 // a22
      r[5] = -w[i];                // nw
    }
    count[i] = 0u;
    if (idxsum) { idxsum[i * 3 + 0] = 0ull; idxsum[i * 3 + 1] = 0ull; idxsum[i * 3 + 2] = 0ull; }
  } else {
    r[(DIM == 3) ? 9 : 5] = CUDART_INF_F;   // padding record: cost +inf, never wins
  }
  float4* dst = reinterpret_cast<float4*>(seeds + (size_t)i * REC);
#pragma unroll
  for (int k = 0; k < REC / 4; ++k) dst[k] = make_float4(r[4 * k], r[4 * k + 1], r[4 * k + 2], r[4 * k + 3]);
}

cudaError_t launch_pack_seeds(int dim, int M, int M_pad, const float* X, const float* A, const float* w,
                              float* seeds, unsigned int* count, unsigned long long* idxsum,
                              const int* done_flag, cudaStream_t st) {
  const int nb = (M_pad + 127) / 128;
  if (dim == 3) pack_seeds_kernel<3><<<nb, 128, 0, st>>>(M, M_pad, X, A, w, seeds, count, idxsum, done_flag);
  else          pack_seeds_kernel<2><<<nb, 128, 0, st>>>(M, M_pad, X, A, w, seeds, count, idxsum, done_flag);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Tile geometry of the DIRECT kernel: 256 threads, each owns V = 8 voxels contiguous in x.
//   3D: 4 x 8 x 8 threads -> tile 32 x 8 x 8 voxels;  2D: 8 x 32 threads -> tile 64 x 32 pixels.
// ------------------------------------------------------------------------------------------
template <int DIM> struct DirectGeom;
template <> struct DirectGeom<3> { static constexpr int V = 8, TXT = 4, TYT = 8, TZT = 8; };
template <> struct DirectGeom<2> { static constexpr int V = 8, TXT = 8, TYT = 32, TZT = 1; };

// fp32 voxel centre: the fp64 definition lo + (i + 1/2) s rounded once to fp32.
__device__ __forceinline__ float centre_f32(double lo, double s, int i) {
  return (float)(lo + ((double)i + 0.5) * s);
}

// ------------------------------------------------------------------------------------------
// DIRECT kernel: every pair evaluates the full quadratic form in delta = y - x_i
// (3 FADD + 3 FMUL + 6 FFMA in 3D), running (min, argmin) with strict '<' over ascending i.
// ------------------------------------------------------------------------------------------
template <int DIM>
__global__ void __launch_bounds__(256) assign_direct_kernel(const AssignArgs a) {
  using G = DirectGeom<DIM>;
  constexpr int V = G::V;
  constexpr int REC = (DIM == 3) ? REC3 : REC2;
  constexpr uint32_t CHUNK_BYTES = SEED_CHUNK * REC * sizeof(float);
  __shared__ __align__(128) float s_seeds[SEED_STAGES][SEED_CHUNK * REC];
  __shared__ __align__(8) uint64_t s_full[SEED_STAGES];
  __shared__ double s_red[256 / 32];

  if (a.done_flag && *a.done_flag) return;   // uniform over the grid: the solve loop has finished
  const int tid = threadIdx.x;
  const int tx = tid % G::TXT, ty = (tid / G::TXT) % G::TYT, tz = tid / (G::TXT * G::TYT);
  const int b = blockIdx.x;
  const int bx = b % a.g.tiles_x, by = (b / a.g.tiles_x) % a.g.tiles_y, bz = b / (a.g.tiles_x * a.g.tiles_y);
  const int ix0 = (bx * G::TXT + tx) * V, iy = by * G::TYT + ty, iz = bz * G::TZT + tz;
  const bool row_valid = (ix0 < a.g.nx) && (iy < a.g.ny) && (iz < a.g.nz);

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

  float yx[V];
#pragma unroll
  for (int k = 0; k < V; ++k) yx[k] = centre_f32(a.g.lo[0], a.g.s[0], ix0 + k);
  const float yy = centre_f32(a.g.lo[1], a.g.s[1], iy);
  const float yz = (DIM == 3) ? centre_f32(a.g.lo[2], a.g.s[2], iz) : 0.0f;

  float best[V];
  int lab[V];
#pragma unroll
  for (int k = 0; k < V; ++k) { best[k] = CUDART_INF_F; lab[k] = 0; }

  for (int c = 0; c < nchunks; ++c) {
    const int stage = c % SEED_STAGES;
    mbar_wait(&s_full[stage], (uint32_t)((c / SEED_STAGES) & 1));
    const float4* sp = reinterpret_cast<const float4*>(s_seeds[stage]);
    const int ibase = c * SEED_CHUNK;
#pragma unroll 2
    for (int i = 0; i < SEED_CHUNK; ++i) {
      if (DIM == 3) {
        const float4 p0 = sp[i * 3 + 0], p1 = sp[i * 3 + 1], p2 = sp[i * 3 + 2];
        const float dy = yy - p0.y, dz = yz - p0.z;
#pragma unroll
        for (int k = 0; k < V; ++k) {
          const float dx = yx[k] - p0.x;
          const float u = fmaf(p1.y, dz, fmaf(p1.x, dy, p0.w * dx));   // a11 dx + a12' dy + a13' dz
          const float v = fmaf(p1.w, dz, p1.z * dy);                   // a22 dy + a23' dz
          const float s = p2.x * dz;                                   // a33 dz
          float cst = fmaf(dx, u, p2.y);                               // ... - w
          cst = fmaf(dy, v, cst);
          cst = fmaf(dz, s, cst);
          if (cst < best[k]) { best[k] = cst; lab[k] = ibase + i; }
        }
      } else {
        const float4 p0 = sp[i * 2 + 0], p1 = sp[i * 2 + 1];
        const float dy = yy - p0.y;
#pragma unroll
        for (int k = 0; k < V; ++k) {
          const float dx = yx[k] - p0.x;
          const float u = fmaf(p0.w, dy, p0.z * dx);                   // a11 dx + a12' dy
          const float v = p1.x * dy;                                   // a22 dy
          float cst = fmaf(dx, u, p1.y);
          cst = fmaf(dy, v, cst);
          if (cst < best[k]) { best[k] = cst; lab[k] = ibase + i; }
        }
      }
    }
    __syncthreads();   // every thread is done with this stage
    if (tid == 0 && c + SEED_STAGES < nchunks) {
      mbar_arrive_expect_tx(&s_full[stage], CHUNK_BYTES);
      tma_bulk_g2s(s_seeds[stage], a.seeds + (size_t)(c + SEED_STAGES) * SEED_CHUNK * REC, CHUNK_BYTES,
                   &s_full[stage]);
    }
  }

  const double dsum = row_epilogue<V>(a, row_valid, ix0, iy, iz, best, lab);
  const double tot = block_sum_double<256>(dsum, s_red);
  if (tid == 0) a.dual_partial[b] = tot;
}

static inline int cdiv(int a, int b) { return (a + b - 1) / b; }

// Returns the ROWPOLY row-length choice (0 for the DIRECT kernel).
int assign_tile_counts(int kernel, int dim, int nx, int ny, int nz, int sm_count, bool cull, int* tx, int* ty, int* tz) {
  if (kernel == APD_KERNEL_ROWPOLY) return rowpoly_tile_counts(dim, nx, ny, nz, sm_count, cull, tx, ty, tz);
  if (kernel == APD_KERNEL_TENSOR) { tensor_tile_counts(nx, ny, nz, tx, ty, tz); return 0; }
  if (dim == 3) {
    using G = DirectGeom<3>;
    *tx = cdiv(nx, G::TXT * G::V); *ty = cdiv(ny, G::TYT); *tz = cdiv(nz, G::TZT);
  } else {
    using G = DirectGeom<2>;
    *tx = cdiv(nx, G::TXT * G::V); *ty = cdiv(ny, G::TYT); *tz = 1;
  }
  return 0;
}

cudaError_t launch_assign(int kernel, const AssignArgs& a, cudaStream_t st) {
  if (kernel == APD_KERNEL_ROWPOLY) return launch_assign_rowpoly(a, st);
  if (kernel == APD_KERNEL_TENSOR) return launch_assign_tensor(a, st);
  const int n_tiles = a.g.tiles_x * a.g.tiles_y * a.g.tiles_z;
  if (a.g.dim == 3) assign_direct_kernel<3><<<n_tiles, 256, 0, st>>>(a);
  else              assign_direct_kernel<2><<<n_tiles, 256, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace apd
