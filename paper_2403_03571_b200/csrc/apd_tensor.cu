// apd_tensor.cu -- row a8 of the path: the cost matrix of Algorithm 1 step 1 (PAPER.md:131,
// eq. 2.1 at PAPER.md:58-61) lifted to a bf16 tensor-core contraction, the argmin of step 2 as the
// epilogue.  3D, and 2D as the special case without z (tile 32 x 16 pixels; 6 of the 10 monomials are non-zero).
//
// For a voxel at INTEGER offset t = (i, j, k) from the reference voxel y0 of its tile and a seed x with matrix A,
//     C(t) = sum_{m<=n} a'_mn s_m s_n t_m t_n  +  sum_m (g_m s_m) t_m  +  r0,
//     g = (A + A^T)(y0 - x),   r0 = (y0 - x)^T A (y0 - x) - w,   s = voxel sides,
// a polynomial with 10 monomials.  Phi[voxel][.] holds the monomials -- integers of magnitude <= 225, exact in bf16 --
// and Theta[seed][.] the 10 fp32 coefficients split three ways into bf16 (hi + mid + lo carries 24 bits), each
// monomial repeated under its three parts: K = 30, padded to 32.  Every product is exact in fp32 and the tensor core
// accumulates in fp32, so the cost carries fp32 rounding only.
//
// One CTA = one tile of 16 x 8 x 4 voxels = 4 UMMA M-tiles of 128 rows (one z-plane each; voxel <-> TMEM lane <->
// thread) against chunks of 128 seeds: per chunk 4 x 2 tcgen05.mma (M 128, N 128, K 16, kind::f16, A and B K-major in
// shared memory without swizzle), one accumulator region of 128 TMEM columns per M-tile (4 x 128 = 512 columns): the
// tensor core works on the other three M-tiles while one is drained.  Warp roles, coupled
// by mbarriers only (no CTA barrier inside the seed loop):
//   warp 21 (one lane): cp.async.bulk (TMA 1-D) of raw seed chunks into a 4-stage ring
//   warp 20:            issues the MMAs of (chunk c, M-tile mt) when Theta[c] is built and the region of mt is drained
//                       (one elected lane); tcgen05.commit signals both consumers
//   warps 16-19:        expand the coefficients of a chunk about this tile's y0 (one seed per thread) into the Theta
//                       ring
//   warps 0-15:         drain chunk c from TMEM (tcgen05.ld 32x32b), release the buffer, 3-input min; the argmin is
//                       found by a rescan of the registers only when some voxel's minimum dropped.
#include "apd_internal.cuh"
#include "apd_device.cuh"
#include <cuda_bf16.h>
#include <math_constants.h>

namespace apd {

// voxel tile: 512 voxels = 4 M-tiles of 128 (thread tid <-> voxel: x fastest, then y, then z).  |offset from the
// reference voxel| <= 16, 8, 4: every monomial <= 256 in magnitude, exact in bf16
template <int DIM> struct TcGeom;
template <> struct TcGeom<3> { static constexpr int TX = 16, TY = 8, TZ = 4; };
template <> struct TcGeom<2> { static constexpr int TX = 32, TY = 16, TZ = 1; };
constexpr int TC_N = 128;                             // seeds per chunk = N of one tcgen05.mma (N >= 128: below that an
                                                      // MMA costs ~45 cycles whatever its N -- measured)
constexpr int TC_EPI_THREADS = 512;                   // one per voxel of the tile
static_assert(TcGeom<3>::TX * TcGeom<3>::TY * TcGeom<3>::TZ == TC_EPI_THREADS && TcGeom<2>::TX * TcGeom<2>::TY == TC_EPI_THREADS, "tile");
constexpr int TC_BUILD_WARPS = 4;                     // 128 threads: one seed of every chunk each
constexpr int TC_THREADS = TC_EPI_THREADS + 32 * TC_BUILD_WARPS + 64;   // + the MMA-issuing warp + the TMA warp
constexpr int TC_QFIX = 24;                           // bf16 per seed in the tile-independent part (18 used)
constexpr int TC_REC = 24;                            // words per seed in the TENSOR seed table: 12 fp32 + 12 x 2 bf16
constexpr int TC_RAW_STAGES = 4, TC_TH_STAGES = 4;
constexpr uint32_t TC_RAW_BYTES = TC_N * TC_REC * 4;  // 12288 per chunk
constexpr uint32_t TC_TH_BYTES = TC_N * 64;           // 8192 per chunk
constexpr uint32_t TC_A_BYTES = 4 * 128 * 64;         // 32768
constexpr uint32_t TC_SMEM = TC_A_BYTES + TC_TH_STAGES * TC_TH_BYTES + TC_RAW_STAGES * TC_RAW_BYTES;

// ---- tcgen05 wrappers ----------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_alloc512(uint32_t* slot) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(slot)) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tc_free512(uint32_t addr) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_mma_bf16(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                            uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ uint32_t tc_elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "elect.sync _|p, 0xffffffff;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(pred));
  return pred;
}
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}
// K-major operand without swizzle: core matrix = 8 rows x 16 bytes, rows 16 bytes apart; the two core matrices of one
// K = 16 step are LBO bytes apart, 8-row groups SBO bytes apart.
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;                        // descriptor version of sm_100
  return d;                                      // base offset 0, layout type 0 = no swizzle
}
#define TC_LD32(addr, v)                                                                                              \
  asm volatile(                                                                                                       \
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "                                                                       \
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,"   \
      "%29,%30,%31}, [%32];"                                                                                          \
      : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]), "=f"(v[8]),   \
        "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15]), "=f"(v[16]),        \
        "=f"(v[17]), "=f"(v[18]), "=f"(v[19]), "=f"(v[20]), "=f"(v[21]), "=f"(v[22]), "=f"(v[23]), "=f"(v[24]),       \
        "=f"(v[25]), "=f"(v[26]), "=f"(v[27]), "=f"(v[28]), "=f"(v[29]), "=f"(v[30]), "=f"(v[31])                     \
      : "r"(addr))
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// min(m, v[0..31]) with four independent chains of 3-input minima (16 instructions, depth 6)
__device__ __forceinline__ float tc_min32(float m, const float (&v)[32]) {
  float t0 = min3f(v[0], v[1], v[2]), t1 = min3f(v[3], v[4], v[5]), t2 = min3f(v[6], v[7], v[8]), t3 = min3f(v[9], v[10], v[11]);
  t0 = min3f(t0, v[12], v[13]); t1 = min3f(t1, v[14], v[15]); t2 = min3f(t2, v[16], v[17]); t3 = min3f(t3, v[18], v[19]);
  t0 = min3f(t0, v[20], v[21]); t1 = min3f(t1, v[22], v[23]); t2 = min3f(t2, v[24], v[25]); t3 = min3f(t3, v[26], v[27]);
  t0 = min3f(t0, v[28], v[29]); t1 = min3f(t1, v[30], v[31]);
  return min3f(min3f(m, t0, t1), t2, t3);
}

// a4 for 32 consecutive seeds of one voxel: running minimum; the argmin is searched (first seed attaining the new
// minimum: lowest index on ties) only when some voxel of the warp improved
__device__ __forceinline__ void tc_take_half(const float (&v)[32], int base, float& best, int& lab) {
  const float m = tc_min32(best, v);
  if (__any_sync(0xffffffffu, m < best)) {
    if (m < best) {
      int idx = 0;
#pragma unroll
      for (int j = 31; j >= 0; --j) idx = (v[j] == m) ? j : idx;
      lab = base + idx;
      best = m;
    }
  }
}
__device__ __forceinline__ void mbar_wait_a(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive_a(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// fp32 -> three bf16 whose sum carries 24 bits of v (each remainder is exact in fp32)
__device__ __forceinline__ void split3(float v, unsigned short& h, unsigned short& m, unsigned short& l) {
  const __nv_bfloat16 bh = __float2bfloat16_rn(v);
  const float r1 = v - __bfloat162float(bh);
  const __nv_bfloat16 bm = __float2bfloat16_rn(r1);
  const float r2 = r1 - __bfloat162float(bm);
  const __nv_bfloat16 bl = __float2bfloat16_rn(r2);
  h = __bfloat16_as_ushort(bh); m = __bfloat16_as_ushort(bm); l = __bfloat16_as_ushort(bl);
}
__device__ __forceinline__ uint32_t pk(unsigned short lo, unsigned short hi) { return (uint32_t)lo | ((uint32_t)hi << 16); }
// two fp32 -> packed bf16x2 {lo = a, hi = b} in one conversion, and the fp32 values of the two halves
__device__ __forceinline__ uint32_t split_pair(float a, float b) {
  const __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<const uint32_t*>(&v);
}
__device__ __forceinline__ float bf_lo(uint32_t v) { return __uint_as_float(v << 16); }
__device__ __forceinline__ float bf_hi(uint32_t v) { return __uint_as_float(v & 0xffff0000u); }

// ---- TENSOR seed table: the DIRECT record (12 fp32) followed by the tile-independent part of Theta, the six
//      quadratic coefficients in voxel units split three ways (18 bf16, padded to 24) --------------------------------
__global__ void pack_qfix_kernel(int dim, int M_pad, const float* __restrict__ rec, double sx, double sy, double sz,
                                 uint4* __restrict__ tcs, const int* __restrict__ done_flag) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M_pad) return;
  if (done_flag && *done_flag) return;
  // 2D: the record (x, y, a11, a12', a22, -w) becomes the 3D one with z = 0 and no z-terms
  __align__(16) float r[REC3];
  if (dim == 3) {
#pragma unroll
    for (int k = 0; k < REC3; ++k) r[k] = rec[(size_t)i * REC3 + k];
  } else {
    const float* p = rec + (size_t)i * REC2;
#pragma unroll
    for (int k = 0; k < REC3; ++k) r[k] = 0.0f;
    r[0] = p[0]; r[1] = p[1]; r[3] = p[2]; r[4] = p[3]; r[6] = p[4]; r[9] = p[5];
  }
  const float q[6] = {(float)((double)r[3] * sx * sx), (float)((double)r[6] * sy * sy), (float)((double)r[8] * sz * sz),
                      (float)((double)r[4] * sx * sy), (float)((double)r[5] * sx * sz), (float)((double)r[7] * sy * sz)};
  unsigned short b[TC_QFIX];
#pragma unroll
  for (int k = 0; k < TC_QFIX; ++k) b[k] = 0;
#pragma unroll
  for (int k = 0; k < 6; ++k) split3(q[k], b[3 * k], b[3 * k + 1], b[3 * k + 2]);
  uint4* dst = tcs + (size_t)i * 6;
  const uint4* src = reinterpret_cast<const uint4*>(r);
#pragma unroll
  for (int k = 0; k < 3; ++k) dst[k] = src[k];
#pragma unroll
  for (int k = 0; k < 3; ++k)
    dst[3 + k] = make_uint4(pk(b[8 * k], b[8 * k + 1]), pk(b[8 * k + 2], b[8 * k + 3]), pk(b[8 * k + 4], b[8 * k + 5]),
                            pk(b[8 * k + 6], b[8 * k + 7]));
}

struct TcSeedRegs { float4 p0, p1, p2; uint4 q0, q1, q2; };

// Theta row of one seed about the tile's reference point -> rows of the K-major B tile (4 pieces of 16 bytes)
__device__ __forceinline__ void tc_build_seed(const TcSeedRegs& s, bool real, float y0x, float y0y, float y0z, float sx,
                                              float sy, float sz, unsigned char* btile, int row) {
  uint4 k0 = s.q0, k1 = s.q1, k2, k3;
  if (real) {
    const float dx = y0x - s.p0.x, dy = y0y - s.p0.y, dz = y0z - s.p0.z;
    const float a11 = s.p0.w, a12 = s.p1.x, a13 = s.p1.y, a22 = s.p1.z, a23 = s.p1.w, a33 = s.p2.x, nw = s.p2.y;
    const float u = fmaf(a13, dz, fmaf(a12, dy, a11 * dx));
    const float v = fmaf(a23, dz, a22 * dy);
    const float t = a33 * dz;
    float r0 = fmaf(dx, u, nw);
    r0 = fmaf(dy, v, r0);
    r0 = fmaf(dz, t, r0);
    const float gx = fmaf(a13, dz, fmaf(a12, dy, 2.0f * a11 * dx)) * sx;
    const float gy = fmaf(a23, dz, fmaf(a12, dx, 2.0f * a22 * dy)) * sy;
    const float gz = fmaf(a23, dy, fmaf(a13, dx, 2.0f * a33 * dz)) * sz;
    // three-way bf16 split of (gx, gy) and (gz, r0), two values per packed conversion; K order of the 12 parts:
    // [hx hy | hz hr | mx my | mz mr | lx ly | lz lr] (Phi carries [i j | k 1] under each)
    const uint32_t h0 = split_pair(gx, gy), h1 = split_pair(gz, r0);
    const float ex = gx - bf_lo(h0), ey = gy - bf_hi(h0), ez = gz - bf_lo(h1), er = r0 - bf_hi(h1);
    const uint32_t m0 = split_pair(ex, ey), m1 = split_pair(ez, er);
    const uint32_t l0 = split_pair(ex - bf_lo(m0), ey - bf_hi(m0)), l1 = split_pair(ez - bf_lo(m1), er - bf_hi(m1));
    k2 = make_uint4(s.q2.x, h0, h1, m0);
    k3 = make_uint4(m1, l0, l1, 0u);
  } else {   // padding seed: constant cost 2^100, never the minimum of a chunk that holds a real seed
    k0 = k1 = make_uint4(0u, 0u, 0u, 0u);
    k2 = make_uint4(0u, 0u, 0u, 0u);
    k3 = make_uint4(0u, 0u, 0u, 0u);
    k2.z = 0x71800000u;                          // K = 21 (high part of r0): bf16 0x7180 = 2^100
  }
  unsigned char* p = btile + (row >> 3) * 512 + (row & 7) * 16;
  *reinterpret_cast<uint4*>(p) = k0;
  *reinterpret_cast<uint4*>(p + 128) = k1;
  *reinterpret_cast<uint4*>(p + 256) = k2;
  *reinterpret_cast<uint4*>(p + 384) = k3;
}

// Writes the Phi rows (A operand) of the CTA's 512 voxels for a tile whose reference voxel is (rx, ry, rz).
template <int DIM>
__device__ __forceinline__ void tc_write_phi(unsigned char* s_A, int tid, int rx, int ry, int rz) {
  using TG = TcGeom<DIM>;
  // Phi row of this thread's voxel: monomials of the integer offsets, each under its three coefficient parts
  const int ti = (tid % TG::TX) - rx, tj = ((tid / TG::TX) % TG::TY) - ry, tk = (tid / (TG::TX * TG::TY)) - rz;
  const float mono[10] = {(float)(ti * ti), (float)(tj * tj), (float)(tk * tk), (float)(ti * tj), (float)(ti * tk),
                          (float)(tj * tk), (float)ti, (float)tj, (float)tk, 1.0f};
  unsigned short e[32];
#pragma unroll
  for (int m = 0; m < 6; ++m) {            // quadratic monomials: [hi mid lo] per monomial
    const unsigned short h = __bfloat16_as_ushort(__float2bfloat16_rn(mono[m]));
    e[3 * m] = h; e[3 * m + 1] = h; e[3 * m + 2] = h;
  }
#pragma unroll
  for (int r = 0; r < 3; ++r)              // linear and constant: [i j k 1] under the hi, mid and lo parts
#pragma unroll
    for (int m = 0; m < 4; ++m) e[18 + 4 * r + m] = __bfloat16_as_ushort(__float2bfloat16_rn(mono[6 + m]));
  e[30] = 0; e[31] = 0;
  const int mt = tid >> 7, row = tid & 127;
  unsigned char* p = s_A + mt * 8192 + (row >> 3) * 512 + (row & 7) * 16;
#pragma unroll
  for (int kc = 0; kc < 4; ++kc)
    *reinterpret_cast<uint4*>(p + kc * 128) = make_uint4(pk(e[8 * kc], e[8 * kc + 1]), pk(e[8 * kc + 2], e[8 * kc + 3]),
                                                         pk(e[8 * kc + 4], e[8 * kc + 5]), pk(e[8 * kc + 6], e[8 * kc + 7]));
  fence_proxy_async_smem();
}

// The MMAs of chunk G (Theta stage U = G & 3) for the four M-tiles: the whole issuing warp walks this (uniform control
// flow), one elected lane issues.  D fp32, A and B bf16, both K-major, N = 128, M = 128.
template <int U>
__device__ __forceinline__ void tc_issue_chunk(int G, uint32_t tmem, uint64_t ad0, uint64_t bd0, uint64_t* s_th_full,
                                               uint64_t* s_th_empty, uint64_t* s_acc_full, uint64_t* s_acc_empty) {
  constexpr uint32_t IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TC_N >> 3) << 17) | ((128u >> 4) << 24);
  mbar_wait(&s_th_full[U], (uint32_t)((G >> 2) & 1));
#pragma unroll
  for (int mt = 0; mt < 4; ++mt) {        // M-tile mt accumulates into its own region of 128 columns
    if (G > 0) mbar_wait(&s_acc_empty[mt], (uint32_t)((G - 1) & 1));
    tc_fence_after();
    if (tc_elect_one()) {
#pragma unroll
      for (int ks = 0; ks < 2; ++ks)
        tc_mma_bf16(tmem + (uint32_t)(mt * TC_N), ad0 + (uint64_t)((mt * 8192 + ks * 256) >> 4),
                    bd0 + (uint64_t)((U * (int)TC_TH_BYTES + ks * 256) >> 4), IDESC, (uint32_t)ks);
      if (mt == 3) tc_commit(&s_th_empty[U]);
      tc_commit(&s_acc_full[mt]);
    }
    __syncwarp();
  }
}

// PERSISTENT: one CTA per SM walks the tiles b = blockIdx.x, blockIdx.x + gridDim.x, ...  TMEM, the barriers and -- as
// long as the tile's reference voxel keeps its place in the tile, i.e. for every tile not cut by the grid's boundary --
// Phi are set up once; the TMA, builder and MMA warps simply keep streaming chunks across the tile boundary (the
// mbarrier phases run on the CTA's global chunk count G), so the next tile's first accumulators are ready while the
// epilogue warps still store the labels of the current one: no pipeline fill / drain per tile (it was ~3 of a tile's
// 79 chunks at cfg 4, ~3 of 8 at cfg 3).  A tile whose reference voxel differs (ragged edge) drains the pipeline with
// two CTA barriers and rewrites Phi.
template <int DIM>
__global__ void __launch_bounds__(TC_THREADS, 1) assign_tensor_kernel(const AssignArgs a) {
  constexpr int TC_TX = TcGeom<DIM>::TX, TC_TY = TcGeom<DIM>::TY, TC_TZ = TcGeom<DIM>::TZ;
  extern __shared__ __align__(128) unsigned char tc_smem[];
  unsigned char* s_A = tc_smem;                                    // Phi: 4 M-tiles x 128 rows x 32 bf16
  unsigned char* s_th = tc_smem + TC_A_BYTES;                      // Theta ring: stages x 128 rows x 32 bf16
  unsigned char* s_raw = s_th + TC_TH_STAGES * TC_TH_BYTES;        // raw seed ring: stages x 128 seeds x 96 bytes
  __shared__ __align__(8) uint64_t s_raw_full[TC_RAW_STAGES], s_raw_empty[TC_RAW_STAGES];
  __shared__ __align__(8) uint64_t s_th_full[TC_TH_STAGES], s_th_empty[TC_TH_STAGES];
  __shared__ __align__(8) uint64_t s_acc_full[4], s_acc_empty[4];      // one accumulator region per M-tile
  __shared__ uint32_t s_tmem;
  __shared__ double s_red[2][TC_EPI_THREADS / 32];

  if (a.done_flag && *a.done_flag) return;
  const int tid = threadIdx.x, lane = tid & 31;
  // the warp index read through a shuffle is PROVABLY warp-uniform: the role branches below become uniform branches
  // and the barrier / TMEM addresses of each role live in uniform registers (measured: 11.58 -> 10.33 ms on cfg 4)
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int n_tiles = a.g.tiles_x * a.g.tiles_y * a.g.tiles_z;
  const int nch = a.M_pad / TC_N;

  if (tid == 0) {
    for (int s = 0; s < TC_RAW_STAGES; ++s) { mbar_init(&s_raw_full[s], 1); mbar_init(&s_raw_empty[s], TC_BUILD_WARPS); }
    for (int s = 0; s < TC_TH_STAGES; ++s) { mbar_init(&s_th_full[s], TC_BUILD_WARPS); mbar_init(&s_th_empty[s], 1); }
    for (int s = 0; s < 4; ++s) { mbar_init(&s_acc_full[s], 1); mbar_init(&s_acc_empty[s], 4); }
    mbar_fence_init();
  }
  if (warp == 0) tc_alloc512(&s_tmem);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;

  // role constants
  const uint64_t ad0 = tc_smem_desc(smem_u32(s_A), 128, 512), bd0 = tc_smem_desc(smem_u32(s_th), 128, 512);
  const float sx = (float)a.g.s[0], sy = (float)a.g.s[1], sz = (float)a.g.s[2];
  const int mt_e = (warp >> 2) & 3;
  uint32_t lane_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(mt_e * TC_N);
  uint32_t full = smem_u32(&s_acc_full[mt_e]), empty = smem_u32(&s_acc_empty[mt_e]);
  asm volatile("" : "+r"(lane_addr), "+r"(full), "+r"(empty));     // keep them in registers (measured: without this 10.30 instead of 10.13 ms)

  // every role walks the same tile sequence; TILE_BEGIN gives the tile's indices and, when its reference voxel differs
  // from the previous tile's (uniform over the CTA), drains the pipeline with two CTA barriers and rewrites Phi
#define TC_TILE_LOOP                                                                                                   \
  int sig_cur = -1, G0 = 0;                                                                                            \
  for (int b = blockIdx.x, it = 0; b < n_tiles; b += gridDim.x, ++it, G0 += nch)
#define TC_TILE_BEGIN                                                                                                  \
  const int bx = b % a.g.tiles_x, by = (b / a.g.tiles_x) % a.g.tiles_y, bz = b / (a.g.tiles_x * a.g.tiles_y);         \
  const int rx = min(TC_TX, a.g.nx - bx * TC_TX) / 2, ry = min(TC_TY, a.g.ny - by * TC_TY) / 2,                       \
            rz = min(TC_TZ, a.g.nz - bz * TC_TZ) / 2;                                                                  \
  const int sig = rx | (ry << 8) | (rz << 16);                                                                         \
  if (sig != sig_cur) {                                                                                                \
    __syncthreads();                                                                                                   \
    if (tid < TC_EPI_THREADS) tc_write_phi<DIM>(s_A, tid, rx, ry, rz);                                                 \
    tc_fence_before();                                                                                                 \
    __syncthreads();                                                                                                   \
    tc_fence_after();                                                                                                  \
    sig_cur = sig;                                                                                                     \
  }                                                                                                                    \
  (void)bx; (void)by; (void)bz; (void)it;

  if (warp == 21) {
    // ===== TMA producer: one lane keeps the raw seed ring full =====
    const unsigned char* src = reinterpret_cast<const unsigned char*>(a.qfix);
    TC_TILE_LOOP {
      TC_TILE_BEGIN
      if (lane == 0) {
        for (int c = 0; c < nch; ++c) {
          const int G = G0 + c, rs = G % TC_RAW_STAGES;
          if (G >= TC_RAW_STAGES) mbar_wait(&s_raw_empty[rs], (uint32_t)(((G / TC_RAW_STAGES) - 1) & 1));
          mbar_arrive_expect_tx(&s_raw_full[rs], TC_RAW_BYTES);
          tma_bulk_g2s(s_raw + rs * TC_RAW_BYTES, src + (size_t)c * TC_RAW_BYTES, TC_RAW_BYTES, &s_raw_full[rs]);
        }
      }
      __syncwarp();
    }
  } else if (warp == 20) {
    // ===== MMA issuer =====
    static_assert(TC_TH_STAGES == 4, "Theta stage = chunk count & 3");
    TC_TILE_LOOP {
      TC_TILE_BEGIN
      for (int c = 0; c < nch; ++c) {
        const int G = G0 + c;
        switch (G & 3) {        // the Theta stage as a compile-time constant: every descriptor is base + constant
          case 0: tc_issue_chunk<0>(G, tmem, ad0, bd0, s_th_full, s_th_empty, s_acc_full, s_acc_empty); break;
          case 1: tc_issue_chunk<1>(G, tmem, ad0, bd0, s_th_full, s_th_empty, s_acc_full, s_acc_empty); break;
          case 2: tc_issue_chunk<2>(G, tmem, ad0, bd0, s_th_full, s_th_empty, s_acc_full, s_acc_empty); break;
          default: tc_issue_chunk<3>(G, tmem, ad0, bd0, s_th_full, s_th_empty, s_acc_full, s_acc_empty); break;
        }
      }
    }
  } else if (warp >= 16) {
    // ===== Theta builders: one seed of the chunk per thread =====
    const int sid = tid - TC_EPI_THREADS;
    TC_TILE_LOOP {
      TC_TILE_BEGIN
      // reference voxel of the tile
      const float y0x = (float)(a.g.lo[0] + ((double)(bx * TC_TX + rx) + 0.5) * a.g.s[0]);
      const float y0y = (float)(a.g.lo[1] + ((double)(by * TC_TY + ry + a.g.off_y) + 0.5) * a.g.s[1]);
      const float y0z = (DIM == 3) ? (float)(a.g.lo[2] + ((double)(bz * TC_TZ + rz + a.g.off_z) + 0.5) * a.g.s[2]) : 0.0f;
      for (int c = 0; c < nch; ++c) {
        const int G = G0 + c, rs = G % TC_RAW_STAGES, ts = G % TC_TH_STAGES;
        mbar_wait(&s_raw_full[rs], (uint32_t)((G / TC_RAW_STAGES) & 1));
        const uint4* rp = reinterpret_cast<const uint4*>(s_raw + rs * TC_RAW_BYTES) + sid * 6;
        TcSeedRegs sr;
        const uint4 u0 = rp[0], u1 = rp[1], u2 = rp[2];
        sr.p0 = make_float4(__uint_as_float(u0.x), __uint_as_float(u0.y), __uint_as_float(u0.z), __uint_as_float(u0.w));
        sr.p1 = make_float4(__uint_as_float(u1.x), __uint_as_float(u1.y), __uint_as_float(u1.z), __uint_as_float(u1.w));
        sr.p2 = make_float4(__uint_as_float(u2.x), __uint_as_float(u2.y), __uint_as_float(u2.z), __uint_as_float(u2.w));
        sr.q0 = rp[3]; sr.q1 = rp[4]; sr.q2 = rp[5];
        if (G >= TC_TH_STAGES) mbar_wait(&s_th_empty[ts], (uint32_t)(((G / TC_TH_STAGES) - 1) & 1));
        tc_build_seed(sr, c * TC_N + sid < a.M, y0x, y0y, y0z, sx, sy, sz, s_th + ts * TC_TH_BYTES, sid);
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) { mbar_arrive(&s_th_full[ts]); mbar_arrive(&s_raw_empty[rs]); }
      }
    }
  } else {
    // ===== epilogue: warps 0-15 =====
    TC_TILE_LOOP {
      TC_TILE_BEGIN
      float best = CUDART_INF_F;
      int lab = 0;
      float ra[32], rb[32];
      for (int c = 0; c < nch; ++c) {
        mbar_wait_a(full, (uint32_t)((G0 + c) & 1));
        tc_fence_after();
        TC_LD32(lane_addr, ra);
        tc_wait_ld();
        TC_LD32(lane_addr + 32, rb);
        tc_take_half(ra, c * TC_N, best, lab);
        tc_wait_ld();
        TC_LD32(lane_addr + 64, ra);
        tc_take_half(rb, c * TC_N + 32, best, lab);
        tc_wait_ld();
        TC_LD32(lane_addr + 96, rb);
        tc_take_half(ra, c * TC_N + 64, best, lab);
        tc_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (tc_elect_one()) mbar_arrive_a(empty);                       // the region is in registers: release it
        tc_take_half(rb, c * TC_N + 96, best, lab);
      }

      // a5 + a6: label store, warp-aggregated counts, index sums, fp64 sum of the minima
      double dsum = 0.0;
      const int ix = bx * TC_TX + (tid % TC_TX), iy = by * TC_TY + ((tid / TC_TX) % TC_TY), iz = bz * TC_TZ + tid / (TC_TX * TC_TY);
      const bool valid = ix < a.g.nx && iy < a.g.ny && iz < a.g.nz;
      const unsigned vmask = __ballot_sync(0xffffffffu, valid);
      // a voxel whose real costs are all NaN / +inf / >= 2^100 would keep a padding seed (cost 2^100) as its minimum:
      // it takes label 0 like the other kernels, and never indexes count[] beyond M
      if (lab >= a.M) lab = 0;
      if (valid) {
        if (a.labels) a.labels[((long long)iz * a.g.ny + iy) * a.g.nx + ix] = lab;
        dsum = (double)best;
        const unsigned peers = __match_any_sync(vmask, lab);
        if (lane == __ffs(peers) - 1) atomicAdd(a.count + lab, (unsigned int)__popc(peers));
        if (a.idxsum) {
          atomicAdd(a.idxsum + (size_t)lab * 3 + 0, (unsigned long long)ix);
          atomicAdd(a.idxsum + (size_t)lab * 3 + 1, (unsigned long long)(iy + a.g.off_y));
          atomicAdd(a.idxsum + (size_t)lab * 3 + 2, (unsigned long long)(iz + a.g.off_z));
        }
      }
      // the tile's sum of minima: lanes by shuffle tree, the 16 epilogue warps in order (a named barrier of the 512
      // epilogue threads only: the producer warps are already streaming the next tile); s_red is double-buffered
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) dsum += __shfl_down_sync(0xffffffffu, dsum, o);
      if (lane == 0) s_red[it & 1][warp] = dsum;
      asm volatile("bar.sync 1, %0;" ::"n"(TC_EPI_THREADS) : "memory");
      if (tid == 0) {
        double tot = 0.0;
#pragma unroll
        for (int i = 0; i < TC_EPI_THREADS / 32; ++i) tot += s_red[it & 1][i];
        a.dual_partial[b] = tot;
      }
    }
  }
#undef TC_TILE_LOOP
#undef TC_TILE_BEGIN
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tc_free512(tmem);
}


void tensor_tile_counts(int dim, int nx, int ny, int nz, int* tx, int* ty, int* tz) {
  if (dim == 3) {
    *tx = (nx + TcGeom<3>::TX - 1) / TcGeom<3>::TX; *ty = (ny + TcGeom<3>::TY - 1) / TcGeom<3>::TY; *tz = (nz + TcGeom<3>::TZ - 1) / TcGeom<3>::TZ;
  } else {
    *tx = (nx + TcGeom<2>::TX - 1) / TcGeom<2>::TX; *ty = (ny + TcGeom<2>::TY - 1) / TcGeom<2>::TY; *tz = 1;
  }
}

cudaError_t launch_pack_qfix(const GridDev& g, int M_pad, const float* rec, uint4* qfix, const int* done_flag,
                             cudaStream_t st) {
  pack_qfix_kernel<<<(M_pad + 127) / 128, 128, 0, st>>>(g.dim, M_pad, rec, g.s[0], g.s[1], g.dim == 3 ? g.s[2] : 0.0, qfix, done_flag);
  return cudaGetLastError();
}

template <int DIM>
static cudaError_t launch_assign_tensor_t(const AssignArgs& a, cudaStream_t st) {
  // per device and cheap: set on every launch (a process may drive several devices through several contexts)
  cudaError_t e = cudaFuncSetAttribute(assign_tensor_kernel<DIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM);
  if (e != cudaSuccess) return e;
  int dev = 0, sms = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
  const int n_tiles = a.g.tiles_x * a.g.tiles_y * a.g.tiles_z;
  const int n_ctas = n_tiles < sms ? n_tiles : sms;                 // persistent: one CTA per SM (112 KB smem, all of TMEM)
  assign_tensor_kernel<DIM><<<n_ctas, TC_THREADS, TC_SMEM, st>>>(a);
  return cudaGetLastError();
}
cudaError_t launch_assign_tensor(const AssignArgs& a, cudaStream_t st) {
  return a.g.dim == 3 ? launch_assign_tensor_t<3>(a, st) : launch_assign_tensor_t<2>(a, st);
}

}  // namespace apd
