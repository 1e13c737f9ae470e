// apd_cull.cu -- row a7 of DESIGN.md's path table: exact, conservative culling of seeds per voxel tile.
//
// Not in the paper (its Algorithm 1 is brute force; adaptivity is future work); asked for
// by BASELINE.json's north_star.  For a voxel tile T whose voxel CENTRES lie in the box y0 +- h, and a seed i with
// s_i = |y0 - x_i|_{A_i} (the A_i-norm) and rho_i = max_{corners} |(+-h)|_{A_i}, the triangle
// inequality in the A_i-norm gives for every centre y of the tile
//        max(0, s_i - rho_i)^2 - w_i  <=  C_i(y) = |y - x_i|^2_{A_i} - w_i  <=  (s_i + rho_i)^2 - w_i .
// With U_T = min_k (s_k + rho_k)^2 - w_k, a seed whose lower bound exceeds U_T is beaten at EVERY voxel of the tile by
// the seed attaining U_T, so it is never an argmin and can be skipped: the labels are those of brute force.
// The kernels use two sharper forms of the same bounds (lower_bound(): support function of the box along the
// A-gradient; exact_upper(): exact corner maximum of the best seed's cost) and, at brick level, a pairwise bound on
// C_i - C_k* over the box (RefSeed::pair_min()) -- derivations at the functions.
// All bounds are taken in fp32 with a relative slack of 2^-16 on every term, three orders above the rounding of the
// fp32 cost evaluation, so rounding can never prune a winner (test: labels with culling == labels without, bit-exact).
// A must be positive definite for the bound to hold (PAPER.md:51-54 assumes it; the library does not check).
// Two levels keep the bound pass O(M) per SUPER-TILE instead of per tile: level 1 builds a parent list for every
// super-tile (64 x 32 x 32 voxels) from all seeds; level 2 builds the list of every BRICK (the 16 x 4 x 8 voxels one
// warp of the culled kernel owns) from its parent's list.  A pruned seed loses everywhere in its box, and a brick lies
// inside its super-tile, so a seed missing from the parent list cannot win in the brick either.
#include "apd_internal.cuh"
#include "apd_device.cuh"
#include <math_constants.h>

namespace apd {

constexpr float CULL_EPS = 1.0f / 65536.0f;
constexpr int CULL_THREADS = 256;

// max over the corners (+-hx, +-hy[, +-hz]) of |h|_A: the diagonal part plus the largest of the sign patterns of
// the off-diagonal part (r = packed record: a_kl' are the doubled off-diagonals)
template <int DIM>
__device__ __forceinline__ float box_radius(const float* r, float hx, float hy, float hz) {
  float q;
  if (DIM == 3) {
    const float dg = r[3] * hx * hx + r[6] * hy * hy + r[8] * hz * hz;
    const float p12 = r[4] * hx * hy, p13 = r[5] * hx * hz, p23 = r[7] * hy * hz;
    q = dg + fmaxf(fmaxf(p12 + p13 + p23, p12 - p13 - p23), fmaxf(-p12 + p13 - p23, -p12 - p13 + p23));
  } else {
    q = r[2] * hx * hx + r[4] * hy * hy + fabsf(r[3] * hx * hy);
  }
  return sqrtf(fmaxf(q, 0.0f)) * (1.0f + 4.0f * CULL_EPS);
}

// sqrt(q) by the hardware reciprocal square root (2 ulp, against the 2^-16 slack every bound carries), 0 for q <= 0;
// the bound passes are instruction-bound and IEEE sqrt / division are ~10 instructions each
__device__ __forceinline__ float norm_of(float q) { return q > 0.0f ? q * rsqrtf(q) : 0.0f; }

// Per-seed record table in the DIRECT layout (apd_internal.cuh) plus rho_i of a brick and of a super-tile in the
// two spare slots.  hb = half-extents of the box of voxel centres of a brick, hs = of a super-tile.
template <int DIM>
__global__ void cull_pack_kernel(int M, int M_pad, const float* __restrict__ X, const float* __restrict__ A,
                                 const float* __restrict__ w, float3 hb, float3 hs, float* __restrict__ rec,
                                 unsigned long long* __restrict__ pairs_ctr, unsigned int* __restrict__ count,
                                 unsigned long long* __restrict__ idxsum, const int* __restrict__ done_flag) {
  pdl_enter();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (done_flag && *done_flag) return;
  if (i == 0) *pairs_ctr = 0ull;
  if (i >= M_pad) return;
  if (i < M) {      // the integer accumulators of the evaluation (the culled path runs no other pack kernel)
    count[i] = 0u;
    if (idxsum) { idxsum[i * 3 + 0] = 0ull; idxsum[i * 3 + 1] = 0ull; idxsum[i * 3 + 2] = 0ull; }
  }
  constexpr int REC = (DIM == 3) ? REC3 : REC2;
  constexpr int NP = (DIM == 3) ? 10 : 6;
  float r[REC];
#pragma unroll
  for (int k = 0; k < REC; ++k) r[k] = 0.0f;
  if (i < M) {
    if (DIM == 3) {
      const float* a = A + (size_t)i * 9;
      r[0] = X[i * 3 + 0]; r[1] = X[i * 3 + 1]; r[2] = X[i * 3 + 2];
      r[3] = a[0]; r[4] = a[1] + a[3]; r[5] = a[2] + a[6]; r[6] = a[4]; r[7] = a[5] + a[7]; r[8] = a[8];
      r[9] = -w[i];
    } else {
      const float* a = A + (size_t)i * 4;
      r[0] = X[i * 2 + 0]; r[1] = X[i * 2 + 1];
      r[2] = a[0]; r[3] = a[1] + a[2]; r[4] = a[3];
      r[5] = -w[i];
    }
    r[NP] = box_radius<DIM>(r, hb.x, hb.y, hb.z);
    r[NP + 1] = box_radius<DIM>(r, hs.x, hs.y, hs.z);
  } else {
    r[NP - 1] = CUDART_INF_F;
  }
  float4* dst = reinterpret_cast<float4*>(rec + (size_t)i * REC);
#pragma unroll
  for (int k = 0; k < REC / 4; ++k) dst[k] = make_float4(r[4 * k], r[4 * k + 1], r[4 * k + 2], r[4 * k + 3]);
}

struct CullArgs {
  GridDev g;               // tiles_* = CTA tiles of the culled kernel
  int M;
  const float* rec;
  int* super_list;         // [n_super, SUPER_CAP]
  int* super_count;        // [n_super]
  int nsx, nsy, nsz;       // super-tiles per axis
  int* brick_list;         // [n_tiles * 4, BRICK_CAP]
  int* brick_count;        // [n_tiles * 4]
  float3 hb, ht, hs;       // half-extents of the boxes of voxel centres of a brick, a CTA tile, a super-tile
  const int* done_flag;
  // list reuse inside apd_solve: the brick lists are rebuilt only when *rebuild != 0, with the slack *delta on both
  // bounds, which keeps them valid for every w' with max_i |w'_i - w_i| <= delta.  nullptr: always rebuild, delta 0.
  // The super-tile lists have their own flag and (larger) slack: the step kernel rebuilds them only when the ball
  // the brick lists must cover is no longer inside theirs (apd_lbfgs.cu).
  const int* rebuild;
  const float* delta;
  const int* rebuild_s;
  const float* delta_s;
  // the CTA-tile lists (the middle level) are kept in global memory between the evaluations of a solve, with a
  // slack of their own between the two: a brick rebuild then starts from its tile's stored list
  int* tile_list;          // [n_tiles, TILE_CAP] or nullptr (single evaluations: the tile lists live in shared memory only)
  int* tile_count;         // [n_tiles]
  const int* rebuild_t;
  const float* delta_t;
};

// For one seed and a box y0 +- h:  s_i = |y0 - x_i|_{A_i};  rho_i = max_corners |(+-h)|_{A_i} (SLOT 0 = brick,
// 1 = super-tile: stored in the record; 2 = computed);  supp_i = max_{|t_k| <= h_k} t^T A_i (y0 - x_i)
// = sum_k |(A_i (y0 - x_i))_k| h_k, the support function of the box along the A-gradient at the centre;  -w_i.
template <int DIM, int SLOT>
__device__ __forceinline__ void seed_bounds(const float* __restrict__ rec, int i, float y0x, float y0y, float y0z,
                                            float3 h, float* s, float* rho, float* supp, float* nw) {
  if (DIM == 3) {
    const float4* p = reinterpret_cast<const float4*>(rec + (size_t)i * REC3);
    const float4 p0 = __ldg(p), p1 = __ldg(p + 1), p2 = __ldg(p + 2);
    const float dx = y0x - p0.x, dy = y0y - p0.y, dz = y0z - p0.z;
    // g = A d with the symmetric matrix (the record holds doubled off-diagonals)
    const float gx = fmaf(0.5f * p1.y, dz, fmaf(0.5f * p1.x, dy, p0.w * dx));
    const float gy = fmaf(0.5f * p1.w, dz, fmaf(p1.z, dy, 0.5f * p1.x * dx));
    const float gz = fmaf(p2.x, dz, fmaf(0.5f * p1.w, dy, 0.5f * p1.y * dx));
    const float q = fmaf(dz, gz, fmaf(dy, gy, dx * gx));
    *s = norm_of(q); *nw = p2.y;
    *supp = fmaf(fabsf(gz), h.z, fmaf(fabsf(gy), h.y, fabsf(gx) * h.x));
    if (SLOT == 2) {
      const float r[9] = {0.f, 0.f, 0.f, p0.w, p1.x, p1.y, p1.z, p1.w, p2.x};
      *rho = box_radius<3>(r, h.x, h.y, h.z);
    } else {
      *rho = SLOT ? p2.w : p2.z;
    }
  } else {
    const float4* p = reinterpret_cast<const float4*>(rec + (size_t)i * REC2);
    const float4 p0 = __ldg(p), p1 = __ldg(p + 1);
    const float dx = y0x - p0.x, dy = y0y - p0.y;
    const float gx = fmaf(0.5f * p0.w, dy, p0.z * dx);
    const float gy = fmaf(p1.x, dy, 0.5f * p0.w * dx);
    const float q = fmaf(dy, gy, dx * gx);
    *s = norm_of(q); *nw = p1.y;
    *supp = fmaf(fabsf(gy), h.y, fabsf(gx) * h.x);
    if (SLOT == 2) {
      const float r[5] = {0.f, 0.f, p0.z, p0.w, p1.x};
      *rho = box_radius<2>(r, h.x, h.y, 0.0f);
    } else {
      *rho = SLOT ? p1.w : p1.z;
    }
  }
}

__device__ __forceinline__ float upper_bound(float s, float rho, float nw) {
  const float r = s * (1.0f + CULL_EPS) + rho;
  return r * r * (1.0f + CULL_EPS) + nw + CULL_EPS * fabsf(nw);
}
// Cauchy-Schwarz in the A-inner product: |d0 + t|_A >= <d0 + t, d0>_A / |d0|_A = s + t^T A d0 / s >= s - supp / s
// (this dominates the ball bound s - rho, since supp <= rho s).  s = 0 gives 0 (fmaxf drops the NaN of 0/0).
__device__ __forceinline__ float lower_bound(float s, float supp, float nw) {
  const float r = fmaxf(s * (1.0f - CULL_EPS) - __fdividef(supp * (1.0f + 4.0f * CULL_EPS), s), 0.0f);
  return r * r * (1.0f - CULL_EPS) + nw - CULL_EPS * fabsf(nw);
}

// EXACT maximum over the box y0 +- h of C_k = |y - x_k|^2_{A_k} - w_k (plus rounding slack): the cost is convex, so
// the maximum sits at a corner; with d = y0 - x_k, g = A d:  C_k(y0 + t) = d.g + 2 g.t + t^T A t - w_k.
// Used for the ONE seed that attains the smallest ball bound of a box: its true worst case is a valid, tighter U.
template <int DIM>
__device__ __forceinline__ float exact_upper(const float* __restrict__ rec, int k, float y0x, float y0y, float y0z,
                                             float3 h) {
  if (DIM == 3) {
    const float4* p = reinterpret_cast<const float4*>(rec + (size_t)k * REC3);
    const float4 p0 = __ldg(p), p1 = __ldg(p + 1), p2 = __ldg(p + 2);
    const float dx = y0x - p0.x, dy = y0y - p0.y, dz = y0z - p0.z;
    const float gx = fmaf(0.5f * p1.y, dz, fmaf(0.5f * p1.x, dy, p0.w * dx));
    const float gy = fmaf(0.5f * p1.w, dz, fmaf(p1.z, dy, 0.5f * p1.x * dx));
    const float gz = fmaf(p2.x, dz, fmaf(0.5f * p1.w, dy, 0.5f * p1.y * dx));
    const float q = fmaxf(fmaf(dz, gz, fmaf(dy, gy, dx * gx)), 0.0f);
    const float lx = 2.0f * gx * h.x, ly = 2.0f * gy * h.y, lz = 2.0f * gz * h.z;
    const float dg = p0.w * h.x * h.x + p1.z * h.y * h.y + p2.x * h.z * h.z;
    const float p12 = p1.x * h.x * h.y, p13 = p1.y * h.x * h.z, p23 = p1.w * h.y * h.z;
    float m = -CUDART_INF_F;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      const float sx = (c & 1) ? -1.f : 1.f, sy = (c & 2) ? -1.f : 1.f, sz = (c & 4) ? -1.f : 1.f;
      m = fmaxf(m, sx * lx + sy * ly + sz * lz + sx * sy * p12 + sx * sz * p13 + sy * sz * p23);
    }
    const float mag = q + fabsf(lx) + fabsf(ly) + fabsf(lz) + dg + fabsf(p12) + fabsf(p13) + fabsf(p23);
    return q + dg + m + 8.0f * CULL_EPS * mag + p2.y + CULL_EPS * fabsf(p2.y);
  } else {
    const float4* p = reinterpret_cast<const float4*>(rec + (size_t)k * REC2);
    const float4 p0 = __ldg(p), p1 = __ldg(p + 1);
    const float dx = y0x - p0.x, dy = y0y - p0.y;
    const float gx = fmaf(0.5f * p0.w, dy, p0.z * dx);
    const float gy = fmaf(p1.x, dy, 0.5f * p0.w * dx);
    const float q = fmaxf(fmaf(dy, gy, dx * gx), 0.0f);
    const float lx = 2.0f * gx * h.x, ly = 2.0f * gy * h.y;
    const float dg = p0.z * h.x * h.x + p1.x * h.y * h.y;
    const float p12 = p0.w * h.x * h.y;
    const float m = fmaxf(fmaxf(lx + ly + p12, -lx - ly + p12), fmaxf(lx - ly - p12, -lx + ly - p12));
    const float mag = q + fabsf(lx) + fabsf(ly) + dg + fabsf(p12);
    return q + dg + m + 8.0f * CULL_EPS * mag + p1.y + CULL_EPS * fabsf(p1.y);
  }
}

// (value, index) minimum over a warp; ties to the lower index
__device__ __forceinline__ void warp_argmin(float& v, int& i) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, v, o);
    const int oi = __shfl_xor_sync(0xffffffffu, i, o);
    if (ov < v || (ov == v && oi < i)) { v = ov; i = oi; }
  }
}

// centre, along one axis, of the box spanned by the centres of voxels i0 .. i0+e-1
__device__ __forceinline__ float box_centre(double lo, double s, int i0, int e) {
  return (float)(lo + ((double)i0 + 0.5 * (double)(e - 1) + 0.5) * s);
}

// LEVEL 1 -- one CTA per super-tile over ALL seeds: pass 1 U = min_k upper bound, pass 2 ordered compaction of
// {i : lower bound_i <= U} into the super-tile's parent list.
template <int DIM>
__global__ void __launch_bounds__(CULL_THREADS) cull_super_kernel(const CullArgs c) {
  pdl_enter();
  __shared__ float s_min[CULL_THREADS / 32];
  __shared__ int s_imin[CULL_THREADS / 32];
  __shared__ int s_wsum[CULL_THREADS / 32];
  __shared__ float s_U;
  if (c.done_flag && *c.done_flag) return;
  if (c.rebuild_s && !*c.rebuild_s) return;
  const float delta = c.delta_s ? *c.delta_s : 0.0f;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int b = blockIdx.x;
  const int sx = b % c.nsx, sy = (b / c.nsx) % c.nsy, sz = b / (c.nsx * c.nsy);
  constexpr int EX = (DIM == 3) ? SUPER3_TX * CULL_TILE3_X : SUPER2_TX * CULL_TILE2_X;
  constexpr int EY = (DIM == 3) ? SUPER3_TY * CULL_TILE3_Y : SUPER2_TY * CULL_TILE2_Y;
  constexpr int EZ = (DIM == 3) ? SUPER3_TZ * CULL_TILE3_Z : 1;
  const float y0x = box_centre(c.g.lo[0], c.g.s[0], sx * EX, EX);
  const float y0y = box_centre(c.g.lo[1], c.g.s[1], sy * EY + c.g.off_y, EY);
  const float y0z = (DIM == 3) ? box_centre(c.g.lo[2], c.g.s[2], sz * EZ + c.g.off_z, EZ) : 0.0f;

  float umin = CUDART_INF_F;
  int imin = 0;
  for (int i = tid; i < c.M; i += CULL_THREADS) {
    float s, rho, supp, nw;
    seed_bounds<DIM, 1>(c.rec, i, y0x, y0y, y0z, c.hs, &s, &rho, &supp, &nw);
    const float u = upper_bound(s, rho, nw);
    if (u < umin) { umin = u; imin = i; }
  }
  warp_argmin(umin, imin);
  if (lane == 0) { s_min[wid] = umin; s_imin[wid] = imin; }
  __syncthreads();
  if (tid == 0) {
    float u = s_min[0];
    int k = s_imin[0];
#pragma unroll
    for (int j = 1; j < CULL_THREADS / 32; ++j) if (s_min[j] < u) { u = s_min[j]; k = s_imin[j]; }
    s_U = fminf(u, exact_upper<DIM>(c.rec, k, y0x, y0y, y0z, c.hs));
  }
  __syncthreads();
  const float U = s_U + 2.0f * delta * (1.0f + CULL_EPS);

  int* list = c.super_list + (size_t)b * SUPER_CAP;
  int base = 0;
  for (int i0 = 0; i0 < c.M; i0 += CULL_THREADS) {
    const int i = i0 + tid;
    bool keep = false;
    if (i < c.M) {
      float s, rho, supp, nw;
      seed_bounds<DIM, 1>(c.rec, i, y0x, y0y, y0z, c.hs, &s, &rho, &supp, &nw);
      keep = !(lower_bound(s, supp, nw) > U);      // NaN keeps the seed
    }
    const unsigned int bal = __ballot_sync(0xffffffffu, keep);
    if (lane == 0) s_wsum[wid] = __popc(bal);
    __syncthreads();
    int off = base, tot = 0;
#pragma unroll
    for (int k = 0; k < CULL_THREADS / 32; ++k) { const int n = s_wsum[k]; if (k < wid) off += n; tot += n; }
    if (keep) {
      const int pos = off + __popc(bal & ((1u << lane) - 1u));
      if (pos < SUPER_CAP) list[pos] = i;
    }
    base += tot;
    __syncthreads();
  }
  if (tid == 0) c.super_count[b] = (base <= SUPER_CAP) ? base : -1;
}

// One seed's record in registers: position, matrix (doubled off-diagonals), -w.
template <int DIM>
struct SeedRec {
  float x, y, z, a11, a12, a13, a22, a23, a33, nw;
  __device__ __forceinline__ void load(const float* __restrict__ rec, int i) {
    if (DIM == 3) {
      const float4* p = reinterpret_cast<const float4*>(rec + (size_t)i * REC3);
      const float4 p0 = __ldg(p), p1 = __ldg(p + 1), p2 = __ldg(p + 2);
      x = p0.x; y = p0.y; z = p0.z; a11 = p0.w; a12 = p1.x; a13 = p1.y; a22 = p1.z; a23 = p1.w; a33 = p2.x; nw = p2.y;
    } else {
      const float4* p = reinterpret_cast<const float4*>(rec + (size_t)i * REC2);
      const float4 p0 = __ldg(p), p1 = __ldg(p + 1);
      x = p0.x; y = p0.y; z = 0.0f; a11 = p0.z; a12 = p0.w; a13 = 0.0f; a22 = p1.x; a23 = 0.0f; a33 = 0.0f; nw = p1.y;
    }
  }
  // rho of a box with half-extents h (does not depend on where the box is)
  __device__ __forceinline__ float radius(float3 h) const {
    if (DIM == 3) {
      const float r[9] = {0.f, 0.f, 0.f, a11, a12, a13, a22, a23, a33};
      return box_radius<3>(r, h.x, h.y, h.z);
    } else {
      const float r[5] = {0.f, 0.f, a11, a12, a22};
      return box_radius<2>(r, h.x, h.y, 0.0f);
    }
  }
  // g = A (y0 - x) and q = |y0 - x|^2_A -- the same expressions in the same order as seed_bounds()
  __device__ __forceinline__ void grad_at(float y0x, float y0y, float y0z, float* gx, float* gy, float* gz, float* q) const {
    if (DIM == 3) {
      const float dx = y0x - x, dy = y0y - y, dz = y0z - z;
      *gx = fmaf(0.5f * a13, dz, fmaf(0.5f * a12, dy, a11 * dx));
      *gy = fmaf(0.5f * a23, dz, fmaf(a22, dy, 0.5f * a12 * dx));
      *gz = fmaf(a33, dz, fmaf(0.5f * a23, dy, 0.5f * a13 * dx));
      *q = fmaf(dz, *gz, fmaf(dy, *gy, dx * *gx));
    } else {
      const float dx = y0x - x, dy = y0y - y;
      *gx = fmaf(0.5f * a12, dy, a11 * dx);
      *gy = fmaf(a22, dy, 0.5f * a12 * dx);
      *gz = 0.0f;
      *q = fmaf(dy, *gy, dx * *gx);
    }
  }
  // s and supp of seed_bounds() for the box y0 +- h
  __device__ __forceinline__ void at(float y0x, float y0y, float y0z, float3 h, float* s, float* supp) const {
    float gx, gy, gz, q;
    grad_at(y0x, y0y, y0z, &gx, &gy, &gz, &q);
    *s = norm_of(q);
    *supp = (DIM == 3) ? fmaf(fabsf(gz), h.z, fmaf(fabsf(gy), h.y, fabsf(gx) * h.x)) : fmaf(fabsf(gy), h.y, fabsf(gx) * h.x);
  }
};

// PAIRWISE test against one reference seed k of a box y0 +- h (the seed that attains the smallest upper bound):
// D(y) = C_i(y) - C_k(y) is a quadratic whose large common part cancels; with t = y - y0, |t_m| <= h_m,
//     D(y0 + t) = D(y0) + 2 (g_i - g_k).t + t^T (A_i - A_k) t
//              >= D(y0) - 2 sum_m |g_i - g_k|_m h_m + sum_m min(0, dA_mm) h_m^2 - sum_{m<n} |dA'_mn| h_m h_n
// (dA' = doubled off-diagonals, as stored).  If that is positive, seed k beats seed i at EVERY voxel of the box, so
// i is never an argmin there.  For equal matrices this is the exact half-space test of the power diagram; it is much
// sharper than comparing i's lower bound with k's upper bound, whose common variation over the box does not cancel.
// Returns the bound minus a rounding slack of 8 * 2^-16 of the magnitudes involved.
template <int DIM>
struct RefSeed {
  SeedRec<DIM> r;
  float gx, gy, gz, q;
  __device__ __forceinline__ void init(const float* __restrict__ rec, int k, float y0x, float y0y, float y0z) {
    r.load(rec, k);
    r.grad_at(y0x, y0y, y0z, &gx, &gy, &gz, &q);
  }
  __device__ __forceinline__ float pair_min(const SeedRec<DIM>& ri, float y0x, float y0y, float y0z, float3 h) const {
    float ix, iy, iz, iq;
    ri.grad_at(y0x, y0y, y0z, &ix, &iy, &iz, &iq);
    const float d0 = (iq + ri.nw) - (q + r.nw);
    float lin = 2.0f * (fabsf(ix - gx) * h.x + fabsf(iy - gy) * h.y);
    float quad = fminf(ri.a11 - r.a11, 0.0f) * h.x * h.x + fminf(ri.a22 - r.a22, 0.0f) * h.y * h.y -
                 fabsf(ri.a12 - r.a12) * h.x * h.y;
    if (DIM == 3) {
      lin += 2.0f * fabsf(iz - gz) * h.z;
      quad += fminf(ri.a33 - r.a33, 0.0f) * h.z * h.z - fabsf(ri.a13 - r.a13) * h.x * h.z -
              fabsf(ri.a23 - r.a23) * h.y * h.z;
    }
    const float mag = fabsf(iq) + fabsf(q) + fabsf(ri.nw) + fabsf(r.nw) + lin - quad;
    return d0 - lin + quad - 8.0f * CULL_EPS * mag;
  }
};

// LEVEL 2 -- one CTA per run of CULL_G CTA tiles adjacent in x (the tiles of one super-tile row, so they share the
// parent list).  (a) The 4 warps together cut the super-tile's parent list (all seeds if that overflowed) down, for
// each of the CULL_G tiles, to the seeds that can win somewhere in that CTA TILE, kept in shared memory: every parent
// record is gathered ONCE per pass and tested against the CULL_G boxes, which is what this kernel is bound by;
// (b) for each tile in turn, each warp cuts the tile's list down to its own brick.  Same two passes (U = min upper
// bound, ordered compaction of lower bound <= U) at both steps.
constexpr int CULL_G = 4;
static_assert(CULL_G == SUPER3_TX && CULL_G == SUPER2_TX, "a CTA of cull_bricks_kernel covers one super-tile row");
template <int DIM>
__global__ void __launch_bounds__(128) cull_bricks_kernel(const CullArgs c) {
  pdl_enter();
  __shared__ int s_tile[CULL_G][TILE_CAP];
  __shared__ float s_min[CULL_G][4];
  __shared__ int s_imin[CULL_G][4];
  __shared__ int s_wsum[4][CULL_G];
  __shared__ RefSeed<DIM> s_ref[4][4];     // (b): per warp (tile), the reference seed of each of its four bricks
  if (c.done_flag && *c.done_flag) return;
  if (c.rebuild && !*c.rebuild) return;
  const float delta = c.delta ? *c.delta : 0.0f;
  const bool rebuild_t = !c.tile_list || !c.rebuild_t || *c.rebuild_t;
  const float delta_t = (c.tile_list && c.delta_t) ? *c.delta_t : delta;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int b = blockIdx.x;
  const int qx = b % c.nsx, by = (b / c.nsx) % c.g.tiles_y, bz = b / (c.nsx * c.g.tiles_y);
  constexpr int TX = (DIM == 3) ? CULL_TILE3_X : CULL_TILE2_X, TY = (DIM == 3) ? CULL_TILE3_Y : CULL_TILE2_Y,
                TZ = (DIM == 3) ? CULL_TILE3_Z : 1;
  constexpr int STY = (DIM == 3) ? SUPER3_TY : SUPER2_TY, STZ = (DIM == 3) ? SUPER3_TZ : 1;
  const int sup = ((bz / STZ) * c.nsy + by / STY) * c.nsx + qx;
  const int ng = min(CULL_G, c.g.tiles_x - qx * CULL_G);      // tiles of this run inside the grid
  int n_par = c.super_count[sup];
  const int* par = c.super_list + (size_t)sup * SUPER_CAP;
  if (n_par < 0) { n_par = c.M; par = nullptr; }

  // (a) CTA-tile lists: built from the parent list, or (inside a solve, while the weights stayed within the slack
  // they were built with) read back from global memory
  int n_tile[CULL_G];
  const size_t tile0 = ((size_t)bz * c.g.tiles_y + by) * c.g.tiles_x + (size_t)qx * CULL_G;
  if (!rebuild_t) {
#pragma unroll
    for (int g = 0; g < CULL_G; ++g) {
      n_tile[g] = (g < ng) ? c.tile_count[tile0 + g] : 0;
      const int* src = c.tile_list + (tile0 + g) * TILE_CAP;
      for (int q = tid; q < n_tile[g]; q += 128) s_tile[g][q] = src[q];
    }
    __syncthreads();
  } else {
    float t0x[CULL_G];
#pragma unroll
    for (int g = 0; g < CULL_G; ++g) t0x[g] = box_centre(c.g.lo[0], c.g.s[0], (qx * CULL_G + g) * TX, TX);
    const float t0y = box_centre(c.g.lo[1], c.g.s[1], by * TY + c.g.off_y, TY);
    const float t0z = (DIM == 3) ? box_centre(c.g.lo[2], c.g.s[2], bz * TZ + c.g.off_z, TZ) : 0.0f;
    float umin[CULL_G];
    int imin[CULL_G];
#pragma unroll
    for (int g = 0; g < CULL_G; ++g) { umin[g] = CUDART_INF_F; imin[g] = 0; }
    for (int pos = tid; pos < n_par; pos += 128) {
      const int i = par ? __ldg(par + pos) : pos;
      SeedRec<DIM> r;
      r.load(c.rec, i);
      const float rho = r.radius(c.ht);
#pragma unroll
      for (int g = 0; g < CULL_G; ++g) {
        float s, supp;
        r.at(t0x[g], t0y, t0z, c.ht, &s, &supp);
        const float u = upper_bound(s, rho, r.nw);
        if (u < umin[g]) { umin[g] = u; imin[g] = i; }
      }
    }
#pragma unroll
    for (int g = 0; g < CULL_G; ++g) {
      warp_argmin(umin[g], imin[g]);
      if (lane == 0) { s_min[g][w] = umin[g]; s_imin[g][w] = imin[g]; }
    }
    __syncthreads();
    float U[CULL_G];
#pragma unroll
    for (int g = 0; g < CULL_G; ++g) {
      float u = s_min[g][0];
      int kbest = s_imin[g][0];
#pragma unroll
      for (int j = 1; j < 4; ++j) if (s_min[g][j] < u) { u = s_min[g][j]; kbest = s_imin[g][j]; }
      if (n_par > 0) u = fminf(u, exact_upper<DIM>(c.rec, kbest, t0x[g], t0y, t0z, c.ht));
      U[g] = u + 2.0f * delta_t * (1.0f + CULL_EPS);
    }
    int base[CULL_G];
#pragma unroll
    for (int g = 0; g < CULL_G; ++g) base[g] = 0;
    for (int p0 = 0; p0 < n_par; p0 += 128) {
      const int pos = p0 + tid;
      bool keep[CULL_G];
#pragma unroll
      for (int g = 0; g < CULL_G; ++g) keep[g] = false;
      int i = 0;
      if (pos < n_par) {
        i = par ? __ldg(par + pos) : pos;
        SeedRec<DIM> r;
        r.load(c.rec, i);
#pragma unroll
        for (int g = 0; g < CULL_G; ++g) {
          float s, supp;
          r.at(t0x[g], t0y, t0z, c.ht, &s, &supp);
          keep[g] = !(lower_bound(s, supp, r.nw) > U[g]);      // NaN keeps the seed
        }
      }
      unsigned int bal[CULL_G];
#pragma unroll
      for (int g = 0; g < CULL_G; ++g) bal[g] = __ballot_sync(0xffffffffu, keep[g]);
      __syncthreads();                       // s_wsum of the previous round has been read
      if (lane < CULL_G) {
        unsigned int m = bal[0];
#pragma unroll
        for (int g = 1; g < CULL_G; ++g) if (lane == g) m = bal[g];
        s_wsum[w][lane] = __popc(m);
      }
      __syncthreads();
#pragma unroll
      for (int g = 0; g < CULL_G; ++g) {
        int off = base[g], tot = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) { const int m = s_wsum[k][g]; if (k < w) off += m; tot += m; }
        if (keep[g]) {
          const int q = off + __popc(bal[g] & ((1u << lane) - 1u));
          if (q < TILE_CAP) s_tile[g][q] = i;
        }
        base[g] += tot;
      }
    }
    __syncthreads();
#pragma unroll
    for (int g = 0; g < CULL_G; ++g) n_tile[g] = (base[g] <= TILE_CAP) ? base[g] : -1;   // -1: bricks cut the parent list
    if (c.tile_list) {
#pragma unroll
      for (int g = 0; g < CULL_G; ++g) {
        if (g >= ng) break;
        int* dst = c.tile_list + (tile0 + g) * TILE_CAP;
        for (int q = tid; q < n_tile[g]; q += 128) dst[q] = s_tile[g][q];
        if (tid == 0) c.tile_count[tile0 + g] = n_tile[g];
      }
    }
  }

  // (b) brick lists: warp g of the CTA cuts tile g's list down to each of the tile's FOUR bricks.  Every candidate's
  // record is gathered once per pass and tested against the four brick boxes (before: each warp walked all four tiles
  // for its own brick, i.e. every record was gathered by four warps -- and this step waits for its 48-byte gathers at
  // random indices: ncu long-scoreboard 5.7 per issue).  Same bounds, same order, same lists.
  if (w < ng) {
    const int g = w;
    const int bx = qx * CULL_G + g;
    const bool from_smem = n_tile[g] >= 0;
    const int n = from_smem ? n_tile[g] : n_par;
    const int* tl = s_tile[g];
    auto cand = [&](int pos) { return from_smem ? tl[pos] : (par ? __ldg(par + pos) : pos); };
    constexpr int REC = (DIM == 3) ? REC3 : REC2;
    constexpr int NB = 4;                      // bricks per tile
    float b0x[NB], b0y[NB], b0z[NB];           // centres of the bricks' boxes of voxel centres
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      int ox, oy, oz, ex, ey, ez;
      brick_box(DIM, j, &ox, &oy, &oz, &ex, &ey, &ez);
      b0x[j] = box_centre(c.g.lo[0], c.g.s[0], bx * TX + ox, ex);
      b0y[j] = box_centre(c.g.lo[1], c.g.s[1], by * TY + oy + c.g.off_y, ey);
      b0z[j] = (DIM == 3) ? box_centre(c.g.lo[2], c.g.s[2], bz * TZ + oz + c.g.off_z, ez) : 0.0f;
    }
    // a candidate's record and its brick radius (slot NP of the record)
    auto load = [&](int i, SeedRec<DIM>& r, float& rho) {
      r.load(c.rec, i);
      rho = __ldg(c.rec + (size_t)i * REC + ((DIM == 3) ? 10 : 6));
    };
    // pass 1: per brick, the seed with the smallest upper bound (by position: the lists ascend in index)
    float umin[NB];
    int pmin[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) { umin[j] = CUDART_INF_F; pmin[j] = 0; }
    for (int pos = lane; pos < n; pos += 32) {
      SeedRec<DIM> r;
      float rho;
      load(cand(pos), r, rho);
#pragma unroll
      for (int j = 0; j < NB; ++j) {
        float sj, supp;
        r.at(b0x[j], b0y[j], b0z[j], c.hb, &sj, &supp);
        const float u = upper_bound(sj, rho, r.nw);
        if (u < umin[j]) { umin[j] = u; pmin[j] = pos; }
      }
    }
    const float slack2 = 2.0f * delta * (1.0f + CULL_EPS);
    float U[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      warp_argmin(umin[j], pmin[j]);
      const int kmin = n > 0 ? cand(pmin[j]) : 0;
      if (n > 0) umin[j] = fminf(umin[j], exact_upper<DIM>(c.rec, kmin, b0x[j], b0y[j], b0z[j], c.hb));
      U[j] = umin[j] + slack2;
      if (lane == j && n > 0) s_ref[w][j].init(c.rec, kmin, b0x[j], b0y[j], b0z[j]);     // the reference seed of brick j
    }
    __syncwarp();
    // pass 2: ordered compaction of the survivors into the four brick lists
    const size_t tile = ((size_t)bz * c.g.tiles_y + by) * c.g.tiles_x + bx;
    int base[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) base[j] = 0;
    for (int p0 = 0; p0 < n; p0 += 32) {
      const int pos = p0 + lane;
      bool keep[NB];
#pragma unroll
      for (int j = 0; j < NB; ++j) keep[j] = false;
      int i = 0;
      if (pos < n) {
        i = cand(pos);
        SeedRec<DIM> r;
        r.load(c.rec, i);
#pragma unroll
        for (int j = 0; j < NB; ++j) {
          float sj, supp;
          r.at(b0x[j], b0y[j], b0z[j], c.hb, &sj, &supp);
          keep[j] = !(lower_bound(sj, supp, r.nw) > U[j]);
          if (keep[j]) keep[j] = !(s_ref[w][j].pair_min(r, b0x[j], b0y[j], b0z[j], c.hb) > slack2);   // NaN keeps the seed
        }
      }
#pragma unroll
      for (int j = 0; j < NB; ++j) {
        const unsigned int bal = __ballot_sync(0xffffffffu, keep[j]);
        if (keep[j]) {
          const int q = base[j] + __popc(bal & ((1u << lane) - 1u));
          if (q < BRICK_CAP) c.brick_list[(tile * 4 + j) * BRICK_CAP + q] = i;
        }
        base[j] += __popc(bal);
      }
    }
    if (lane < NB) {
      int bj = base[0];
#pragma unroll
      for (int j = 1; j < NB; ++j) if (lane == j) bj = base[j];
      c.brick_count[tile * 4 + lane] = (bj <= BRICK_CAP) ? bj : -1;
    }
  }
}

void cull_super_counts(const GridDev& g, int* nsx, int* nsy, int* nsz) {
  if (g.dim == 3) {
    *nsx = (g.tiles_x + SUPER3_TX - 1) / SUPER3_TX; *nsy = (g.tiles_y + SUPER3_TY - 1) / SUPER3_TY;
    *nsz = (g.tiles_z + SUPER3_TZ - 1) / SUPER3_TZ;
  } else {
    *nsx = (g.tiles_x + SUPER2_TX - 1) / SUPER2_TX; *nsy = (g.tiles_y + SUPER2_TY - 1) / SUPER2_TY; *nsz = 1;
  }
}

cudaError_t launch_cull(const GridDev& g, int M, int M_pad, const float* X, const float* A, const float* w,
                        const CullBuffers& cb, int nsx, int nsy, int nsz, unsigned int* count,
                        unsigned long long* idxsum, const int* done_flag, const int* rebuild, const float* delta,
                        const int* rebuild_s, const float* delta_s, const int* rebuild_t, const float* delta_t,
                        bool skip_pack, cudaStream_t st) {
  // half-extents of the boxes of voxel CENTRES of a brick and of a super-tile
  int ox, oy, oz, ex, ey, ez;
  brick_box(g.dim, 0, &ox, &oy, &oz, &ex, &ey, &ez);
  const int sex = (g.dim == 3) ? SUPER3_TX * CULL_TILE3_X : SUPER2_TX * CULL_TILE2_X;
  const int sey = (g.dim == 3) ? SUPER3_TY * CULL_TILE3_Y : SUPER2_TY * CULL_TILE2_Y;
  const int sez = (g.dim == 3) ? SUPER3_TZ * CULL_TILE3_Z : 1;
  auto half = [&](int e, int k) { return (float)(0.5 * (double)(e - 1) * g.s[k]); };
  const float3 hb = make_float3(half(ex, 0), half(ey, 1), g.dim == 3 ? half(ez, 2) : 0.0f);
  const float3 hs = make_float3(half(sex, 0), half(sey, 1), g.dim == 3 ? half(sez, 2) : 0.0f);
  const int nb = (M_pad + 127) / 128;
  cudaError_t e = cudaSuccess;
  // skip_pack: inside a solve, after its first evaluation, the step kernel has already written -w into the records and
  // zeroed the counts (apd_lbfgs.cu: StepArgs::rec_nw); everything else in a record is constant over the solve
  if (!skip_pack) {
    if (g.dim == 3) e = launch_pdl(cull_pack_kernel<3>, nb, 128, 0, st, M, M_pad, X, A, w, hb, hs, cb.rec, cb.pairs_ctr, count, idxsum, done_flag);
    else            e = launch_pdl(cull_pack_kernel<2>, nb, 128, 0, st, M, M_pad, X, A, w, hb, hs, cb.rec, cb.pairs_ctr, count, idxsum, done_flag);
    if (e != cudaSuccess) return e;
  }
  CullArgs c;
  c.g = g; c.M = M; c.rec = cb.rec; c.super_list = cb.super_list; c.super_count = cb.super_count;
  c.nsx = nsx; c.nsy = nsy; c.nsz = nsz; c.brick_list = cb.brick_list; c.brick_count = cb.brick_count;
  c.done_flag = done_flag; c.rebuild = rebuild; c.delta = delta; c.rebuild_s = rebuild_s; c.delta_s = delta_s;
  // the tile lists are kept only inside a solve (rebuild flags given): a single evaluation builds them in shared memory
  c.tile_list = rebuild ? cb.tile_list : nullptr; c.tile_count = cb.tile_count; c.rebuild_t = rebuild_t; c.delta_t = delta_t;
  c.hb = hb; c.hs = hs;
  c.ht = make_float3(half(g.dim == 3 ? CULL_TILE3_X : CULL_TILE2_X, 0), half(g.dim == 3 ? CULL_TILE3_Y : CULL_TILE2_Y, 1),
                     g.dim == 3 ? half(CULL_TILE3_Z, 2) : 0.0f);
  const int n_super = nsx * nsy * nsz;
  const int n_runs = nsx * g.tiles_y * g.tiles_z;      // runs of CULL_G tiles along x
  if (g.dim == 3) e = launch_pdl(cull_super_kernel<3>, n_super, CULL_THREADS, 0, st, c);
  else            e = launch_pdl(cull_super_kernel<2>, n_super, CULL_THREADS, 0, st, c);
  if (e != cudaSuccess) return e;
  if (g.dim == 3) return launch_pdl(cull_bricks_kernel<3>, n_runs, 128, 0, st, c);
  return launch_pdl(cull_bricks_kernel<2>, n_runs, 128, 0, st, c);
}

}  // namespace apd
