// apd_cull.cu -- row a7 of DESIGN.md's path table: exact, conservative culling of seeds per voxel tile.
//
// Not in the paper (its Algorithm 1 is brute force; adaptivity is future work); asked for
// by BASELINE.json's north_star.  For a voxel tile T whose voxel CENTRES lie in the box y0 +- h, and a seed i with
// s_i = |y0 - x_i|_{A_i} (the A_i-norm) and rho_i = max_{corners} |(+-h)|_{A_i}, the triangle
// inequality in the A_i-norm gives for every centre y of the tile
//        max(0, s_i - rho_i)^2 - w_i  <=  C_i(y) = |y - x_i|^2_{A_i} - w_i  <=  (s_i + rho_i)^2 - w_i .
// With U_T = min_k (s_k + rho_k)^2 - w_k, a seed whose lower bound exceeds U_T is beaten at EVERY voxel of the tile by
// the seed attaining U_T, so it is never an argmin and can be skipped: the labels are those of brute force.
// All bounds are taken in fp32 with a relative slack of 2^-16 on every term, three orders above the rounding of the
// fp32 cost evaluation, so rounding can never prune a winner (test: labels with culling == labels without, bit-exact).
// A must be positive definite for the bound to hold (PAPER.md:51-54 assumes it; the library does not check).
#include "apd_internal.cuh"
#include "apd_device.cuh"
#include <math_constants.h>

namespace apd {

constexpr float CULL_EPS = 1.0f / 65536.0f;
constexpr int CULL_THREADS = 256;

// Per-seed record table in the DIRECT layout (apd_internal.cuh) plus rho_i in the first spare slot.
template <int DIM>
__global__ void cull_pack_kernel(int M, int M_pad, const float* __restrict__ X, const float* __restrict__ A,
                                 const float* __restrict__ w, float hx, float hy, float hz, float* __restrict__ rec,
                                 unsigned long long* __restrict__ pairs_ctr, const int* __restrict__ done_flag) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (done_flag && *done_flag) return;
  if (i == 0) *pairs_ctr = 0ull;
  if (i >= M_pad) return;
  constexpr int REC = (DIM == 3) ? REC3 : REC2;
  float r[REC];
#pragma unroll
  for (int k = 0; k < REC; ++k) r[k] = 0.0f;
  if (i < M) {
    if (DIM == 3) {
      const float* a = A + (size_t)i * 9;
      r[0] = X[i * 3 + 0]; r[1] = X[i * 3 + 1]; r[2] = X[i * 3 + 2];
      r[3] = a[0]; r[4] = a[1] + a[3]; r[5] = a[2] + a[6]; r[6] = a[4]; r[7] = a[5] + a[7]; r[8] = a[8];
      r[9] = -w[i];
      // max over the box corners (+-hx, +-hy, +-hz) of h^T A h: the diagonal part plus the largest of the four
      // sign patterns of the off-diagonal part
      const float dg = r[3] * hx * hx + r[6] * hy * hy + r[8] * hz * hz;
      const float p12 = r[4] * hx * hy, p13 = r[5] * hx * hz, p23 = r[7] * hy * hz;
      const float off = fmaxf(fmaxf(p12 + p13 + p23, p12 - p13 - p23), fmaxf(-p12 + p13 - p23, -p12 - p13 + p23));
      r[10] = sqrtf(fmaxf(dg + off, 0.0f)) * (1.0f + 4.0f * CULL_EPS);
    } else {
      const float* a = A + (size_t)i * 4;
      r[0] = X[i * 2 + 0]; r[1] = X[i * 2 + 1];
      r[2] = a[0]; r[3] = a[1] + a[2]; r[4] = a[3];
      r[5] = -w[i];
      const float dg = r[2] * hx * hx + r[4] * hy * hy;
      r[6] = sqrtf(fmaxf(dg + fabsf(r[3] * hx * hy), 0.0f)) * (1.0f + 4.0f * CULL_EPS);
    }
  } else {
    r[(DIM == 3) ? 9 : 5] = CUDART_INF_F;
  }
  float4* dst = reinterpret_cast<float4*>(rec + (size_t)i * REC);
#pragma unroll
  for (int k = 0; k < REC / 4; ++k) dst[k] = make_float4(r[4 * k], r[4 * k + 1], r[4 * k + 2], r[4 * k + 3]);
}

struct CullArgs {
  GridDev g;
  int ex, ey, ez;        // tile extents in voxels
  int M;
  const float* rec;
  int* list;             // [n_tiles, cap]
  int* count;            // [n_tiles]
  int cap;
  const int* done_flag;
};

// s_i = |y0 - x_i|_{A_i}, rho_i and -w_i of one seed
template <int DIM>
__device__ __forceinline__ void seed_bounds(const float* __restrict__ rec, int i, float y0x, float y0y, float y0z,
                                            float* s, float* rho, float* nw) {
  if (DIM == 3) {
    const float4* p = reinterpret_cast<const float4*>(rec + (size_t)i * REC3);
    const float4 p0 = __ldg(p), p1 = __ldg(p + 1), p2 = __ldg(p + 2);
    const float dx = y0x - p0.x, dy = y0y - p0.y, dz = y0z - p0.z;
    float q = dx * fmaf(p1.y, dz, fmaf(p1.x, dy, p0.w * dx));
    q = fmaf(dy, fmaf(p1.w, dz, p1.z * dy), q);
    q = fmaf(dz, p2.x * dz, q);
    *s = sqrtf(fmaxf(q, 0.0f)); *rho = p2.z; *nw = p2.y;
  } else {
    const float4* p = reinterpret_cast<const float4*>(rec + (size_t)i * REC2);
    const float4 p0 = __ldg(p), p1 = __ldg(p + 1);
    const float dx = y0x - p0.x, dy = y0y - p0.y;
    float q = dx * fmaf(p0.w, dy, p0.z * dx);
    q = fmaf(dy, p1.x * dy, q);
    *s = sqrtf(fmaxf(q, 0.0f)); *rho = p1.z; *nw = p1.y;
  }
}

__device__ __forceinline__ float upper_bound(float s, float rho, float nw) {
  const float r = s * (1.0f + CULL_EPS) + rho;
  return r * r * (1.0f + CULL_EPS) + nw + CULL_EPS * fabsf(nw);
}
__device__ __forceinline__ float lower_bound(float s, float rho, float nw) {
  const float r = fmaxf(s * (1.0f - CULL_EPS) - rho, 0.0f);
  return r * r * (1.0f - CULL_EPS) + nw - CULL_EPS * fabsf(nw);
}

// One CTA per tile: pass 1 U_T = min_k upper bound, pass 2 ordered compaction of {i : lower bound_i <= U_T}.
template <int DIM>
__global__ void __launch_bounds__(CULL_THREADS) cull_tiles_kernel(const CullArgs c) {
  __shared__ float s_min[CULL_THREADS / 32];
  __shared__ int s_wsum[CULL_THREADS / 32];
  __shared__ float s_U;
  if (c.done_flag && *c.done_flag) return;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int b = blockIdx.x;
  const int bx = b % c.g.tiles_x, by = (b / c.g.tiles_x) % c.g.tiles_y, bz = b / (c.g.tiles_x * c.g.tiles_y);
  // centre of the box spanned by the tile's voxel centres
  const float y0x = (float)(c.g.lo[0] + ((double)(bx * c.ex) + 0.5 * (double)(c.ex - 1) + 0.5) * c.g.s[0]);
  const float y0y = (float)(c.g.lo[1] + ((double)(by * c.ey) + 0.5 * (double)(c.ey - 1) + 0.5) * c.g.s[1]);
  const float y0z = (DIM == 3) ? (float)(c.g.lo[2] + ((double)(bz * c.ez) + 0.5 * (double)(c.ez - 1) + 0.5) * c.g.s[2]) : 0.0f;

  float umin = CUDART_INF_F;
  for (int i = tid; i < c.M; i += CULL_THREADS) {
    float s, rho, nw;
    seed_bounds<DIM>(c.rec, i, y0x, y0y, y0z, &s, &rho, &nw);
    umin = fminf(umin, upper_bound(s, rho, nw));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) umin = fminf(umin, __shfl_xor_sync(0xffffffffu, umin, o));
  if (lane == 0) s_min[wid] = umin;
  __syncthreads();
  if (tid == 0) {
    float u = s_min[0];
#pragma unroll
    for (int k = 1; k < CULL_THREADS / 32; ++k) u = fminf(u, s_min[k]);
    s_U = u;
  }
  __syncthreads();
  const float U = s_U;

  int* list = c.list + (size_t)b * c.cap;
  int base = 0;
  for (int i0 = 0; i0 < c.M; i0 += CULL_THREADS) {
    const int i = i0 + tid;
    bool keep = false;
    if (i < c.M) {
      float s, rho, nw;
      seed_bounds<DIM>(c.rec, i, y0x, y0y, y0z, &s, &rho, &nw);
      keep = !(lower_bound(s, rho, nw) > U);       // NaN keeps the seed
    }
    const unsigned int bal = __ballot_sync(0xffffffffu, keep);
    if (lane == 0) s_wsum[wid] = __popc(bal);
    __syncthreads();
    int off = base, tot = 0;
#pragma unroll
    for (int k = 0; k < CULL_THREADS / 32; ++k) { const int n = s_wsum[k]; if (k < wid) off += n; tot += n; }
    if (keep) {
      const int pos = off + __popc(bal & ((1u << lane) - 1u));
      if (pos < c.cap) list[pos] = i;
    }
    base += tot;
    __syncthreads();
  }
  if (tid == 0) c.count[b] = (base <= c.cap) ? base : -1;
}

cudaError_t launch_cull(const GridDev& g, int M, int M_pad, const float* X, const float* A, const float* w, float* rec,
                        int* list, int* count, int cap, unsigned long long* pairs_ctr, const int* done_flag,
                        cudaStream_t st) {
  int ex, ey, ez;
  rowpoly_tile_extent(g.dim, g.row_long, &ex, &ey, &ez);
  const float hx = (float)(0.5 * (double)(ex - 1) * g.s[0]), hy = (float)(0.5 * (double)(ey - 1) * g.s[1]),
              hz = (g.dim == 3) ? (float)(0.5 * (double)(ez - 1) * g.s[2]) : 0.0f;
  const int nb = (M_pad + 127) / 128;
  if (g.dim == 3) cull_pack_kernel<3><<<nb, 128, 0, st>>>(M, M_pad, X, A, w, hx, hy, hz, rec, pairs_ctr, done_flag);
  else            cull_pack_kernel<2><<<nb, 128, 0, st>>>(M, M_pad, X, A, w, hx, hy, hz, rec, pairs_ctr, done_flag);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  CullArgs c;
  c.g = g; c.ex = ex; c.ey = ey; c.ez = ez; c.M = M; c.rec = rec; c.list = list; c.count = count; c.cap = cap;
  c.done_flag = done_flag;
  const int n_tiles = g.tiles_x * g.tiles_y * g.tiles_z;
  if (g.dim == 3) cull_tiles_kernel<3><<<n_tiles, CULL_THREADS, 0, st>>>(c);
  else            cull_tiles_kernel<2><<<n_tiles, CULL_THREADS, 0, st>>>(c);
  return cudaGetLastError();
}

}  // namespace apd
