// apd_rowpoly.cu -- the ROWPOLY voxel x seed kernel (rows a1-a6 of DESIGN.md's path table).
//
// Same definition as the DIRECT kernel -- C_ij = |y_j - x_i|^2_{A_i} - w_i (eq. 2.1),
// H_j = argmin_i C_ij with the lowest index among equal fp32 costs (reading S1) --
// re-associated for the machine:
//   * a thread owns a ROW of V voxels contiguous in x.  With dc = x_c - x_i, x_c the MIDPOINT of the row, the cost
//     along the row is the quadratic  c(tau) = a11 tau^2 + B' tau + R',
//        B' = 2 a11 dc + (a12' dy + a13' dz),   R' = cost at the midpoint,
//     and the voxels sit at tau = +-tau_j, tau_j = (j + 1/2) s_x, j < V/2.  The even part is shared by the two:
//        e_j = fma(a11, tau_j^2, R'),   c(+tau_j) = fma(B', tau_j, e_j),   c(-tau_j) = fma(-B', tau_j, e_j),
//     so a pair costs 1.5 FMA after a per-(row, seed) set-up of 15 operations;
//   * all arithmetic is packed f32x2 (FFMA2) over PAIRS OF SEEDS (the seed table is stored
//     pair-interleaved), one 3-input min folds both lanes into the running minimum;
//   * the inner loop keeps only the minimum.  After every GROUP seeds the minima are compared with
//     their values before the group; a voxel whose minimum dropped has its argmin inside that
//     group, and the (rare) rescan recomputes the group with the same instructions and takes the
//     first seed whose cost equals the new minimum.
#include "apd_internal.cuh"
#include "apd_device.cuh"
#include "apd_epilogue.cuh"
#include <math_constants.h>

namespace apd {

constexpr int ROW_BATCH = 8;                          // voxels of a row whose FMA chains are interleaved

// pair-interleaved seed table: PREC floats per PAIR of seeds
//   3D (20): X0 X1 Y0 Y1 | Z0 Z1 a11 a11 | a12' a12' a13' a13' | a22 a22 a23' a23' | a33 a33 nw nw
//   2D (12): X0 X1 Y0 Y1 | a11 a11 a12' a12' | a22 a22 nw nw
constexpr int PREC3 = 20;
constexpr int PREC2 = 12;

template <int DIM>
__global__ void pack_pairs_kernel(int M, int M_pad, const float* __restrict__ X, const float* __restrict__ A,
                                  const float* __restrict__ w, float* __restrict__ seeds,
                                  unsigned int* __restrict__ count, unsigned long long* __restrict__ idxsum,
                                  const int* __restrict__ done_flag) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M_pad) return;
  if (done_flag && *done_flag) return;
  constexpr int NP = (DIM == 3) ? 10 : 6;
  constexpr int PREC = (DIM == 3) ? PREC3 : PREC2;
  float r[NP];
#pragma unroll
  for (int k = 0; k < NP; ++k) r[k] = 0.0f;
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
    count[i] = 0u;
    if (idxsum) { idxsum[i * 3 + 0] = 0ull; idxsum[i * 3 + 1] = 0ull; idxsum[i * 3 + 2] = 0ull; }
  } else {
    r[NP - 1] = CUDART_INF_F;   // padding seed: cost +inf
  }
  float* dst = seeds + (size_t)(i >> 1) * PREC + (i & 1);
#pragma unroll
  for (int k = 0; k < NP; ++k) dst[2 * k] = r[k];
}

cudaError_t launch_pack_pairs(int dim, int M, int M_pad, const float* X, const float* A, const float* w,
                              float* seeds, unsigned int* count, unsigned long long* idxsum,
                              const int* done_flag, cudaStream_t st) {
  const int nb = (M_pad + 127) / 128;
  if (dim == 3) pack_pairs_kernel<3><<<nb, 128, 0, st>>>(M, M_pad, X, A, w, seeds, count, idxsum, done_flag);
  else          pack_pairs_kernel<2><<<nb, 128, 0, st>>>(M, M_pad, X, A, w, seeds, count, idxsum, done_flag);
  return cudaGetLastError();
}

// Per-(row, seed pair) coefficients of the row quadratic.
struct RowCoef { f2 a11, Bp, nBp, Rp; };      // nBp = -Bp

// 3D: B' and R' are themselves polynomials in the row's offset (Y, Z) from the TILE's reference point
// (x_c, y_0, z_0) = (row midpoint in x, tile midpoint in y and z):
//      B' = b0 + a12' Y + a13' Z,      R' = r0 + r1 Y + r2 Z + a22 Y^2 + a23' Y Z + a33 Z^2,
// with d = (x_c, y_0, z_0) - x_i:  b0 = 2 a11 dx + a12' dy + a13' dz (the x-derivative of the cost at the reference
// point), r1 = a12' dx + 2 a22 dy + a23' dz, r2 = a13' dx + a23' dy + 2 a33 dz (its y- and z-derivatives) and
// r0 = the cost there.  cook3() turns a seed's (x, y, z, -w) into (b0, r1, r2, r0) ONCE per (tile, seed) -- in the
// brute-force kernel thread t of the CTA does it in place for seed t of every staged chunk, in the culled kernel
// the lane that gathers a candidate -- and the per-(row, seed) set-up shrinks from 14 to 7 FMA.  Both kernels call
// this one function with explicit roundings, so their costs agree bit for bit.
struct Cooked3 { float b0, r1, r2, r0; };
__device__ __forceinline__ Cooked3 cook3(float X, float Y, float Z, float a11, float a12, float a13, float a22,
                                         float a23, float a33, float nw, float xc, float y0, float z0) {
  const float dx = __fsub_rn(xc, X), dy = __fsub_rn(y0, Y), dz = __fsub_rn(z0, Z);
  const float E0 = fmaf(a12, dy, __fmul_rn(a13, dz));                      // a12' dy + a13' dz
  const float u0 = fmaf(a23, dz, __fmul_rn(a22, dy));                      // a22 dy + a23' dz
  float R0 = fmaf(dy, u0, nw);                                             // ... - w
  R0 = fmaf(dz, __fmul_rn(a33, dz), R0);                                   // + a33 dz^2
  Cooked3 o;
  o.b0 = fmaf(__fadd_rn(a11, a11), dx, E0);
  o.r0 = fmaf(dx, fmaf(a11, dx, E0), R0);
  o.r1 = fmaf(a12, dx, fmaf(__fadd_rn(a22, a22), dy, __fmul_rn(a23, dz)));
  o.r2 = fmaf(a13, dx, fmaf(a23, dy, __fmul_rn(__fadd_rn(a33, a33), dz)));
  return o;
}

// Per-thread constants of the set-up.  2D: the row's midpoint x and its y.  3D: the row's offset (Y, Z) from the
// tile's reference point and its monomials.
template <int DIM> struct RowRef;
template <> struct RowRef<2> { f2 x0, yy; };
template <> struct RowRef<3> { f2 Y, Z, YY, YZ, ZZ; };

// sp = one pair record in smem; 3D: cooked, i.e. the slots of (X, Y, Z, nw) hold (b0, r1, r2, r0)
template <int DIM>
__device__ __forceinline__ RowCoef row_setup(const float* __restrict__ sp, const RowRef<DIM>& rr) {
  RowCoef o;
  if constexpr (DIM == 3) {
    const ulonglong2 q0 = *reinterpret_cast<const ulonglong2*>(sp);        // b0, r1
    const ulonglong2 q1 = *reinterpret_cast<const ulonglong2*>(sp + 4);    // r2, a11
    const ulonglong2 q2 = *reinterpret_cast<const ulonglong2*>(sp + 8);    // a12', a13'
    const ulonglong2 q3 = *reinterpret_cast<const ulonglong2*>(sp + 12);   // a22, a23'
    const ulonglong2 q4 = *reinterpret_cast<const ulonglong2*>(sp + 16);   // a33, r0
    o.a11 = q1.y;
    o.Bp = f2_fma(q2.y, rr.Z, f2_fma(q2.x, rr.Y, q0.x));
    f2 R = f2_fma(q0.y, rr.Y, q4.y);
    R = f2_fma(q1.x, rr.Z, R);
    R = f2_fma(q3.x, rr.YY, R);
    R = f2_fma(q3.y, rr.YZ, R);
    o.Rp = f2_fma(q4.x, rr.ZZ, R);
  } else {
    const ulonglong2 q0 = *reinterpret_cast<const ulonglong2*>(sp);        // X, Y
    const ulonglong2 q1 = *reinterpret_cast<const ulonglong2*>(sp + 4);    // a11, a12'
    const ulonglong2 q2 = *reinterpret_cast<const ulonglong2*>(sp + 8);    // a22, nw
    const f2 d0 = f2_sub(rr.x0, q0.x), dy = f2_sub(rr.yy, q0.y);
    const f2 a11 = q1.x;
    const f2 E = f2_mul(q1.y, dy);                                         // a12' dy
    const f2 R = f2_fma(dy, f2_mul(q2.x, dy), q2.y);                       // a22 dy^2 - w
    o.a11 = a11;
    o.Bp = f2_fma(f2_add(a11, a11), d0, E);                                // 2 a11 dc + E
    o.Rp = f2_fma(d0, f2_fma(a11, d0, E), R);                              // cost at the row's midpoint
  }
  o.nBp = o.Bp ^ 0x8000000080000000ull;                                    // both sign bits (integer pipe)
  return o;
}

// In-row offsets of a thread: tt[j] = tau_j, tsq[j] = fl32(tau_j^2), j < V/2 (kernel parameters: uniform registers).
// Voxel V/2 + j of the row sits at +tau_j, voxel V/2 - 1 - j at -tau_j.
template <int V>
struct RowTau { f2 tt[V / 2], tsq[V / 2]; };

// cost of voxel k of the row, for both seeds of the pair -- the same instructions as the main loop
template <int V>
__device__ __forceinline__ f2 row_cost(const RowCoef& c, const RowTau<V>& t, int k) {
  const int j = (k >= V / 2) ? k - V / 2 : V / 2 - 1 - k;
  return f2_fma((k >= V / 2) ? c.Bp : c.nBp, t.tt[j], f2_fma(c.a11, t.tsq[j], c.Rp));
}

// The main loop of one (row, seed pair): 3 FFMA2 + 2 three-input minima per 2 voxels x 2 seeds.  F(k, lo, hi) takes
// the two costs of voxel k.
template <int V, class F>
__device__ __forceinline__ void row_sweep(const RowCoef& rc, const RowTau<V>& t, F&& f) {
  constexpr int HB = ROW_BATCH / 2;
  static_assert((V / 2) % HB == 0, "batch");
#pragma unroll
  for (int j0 = 0; j0 < V / 2; j0 += HB) {
    f2 e[HB], cp[HB], cm[HB];
#pragma unroll
    for (int j = 0; j < HB; ++j) e[j] = f2_fma(rc.a11, t.tsq[j0 + j], rc.Rp);
#pragma unroll
    for (int j = 0; j < HB; ++j) { cp[j] = f2_fma(rc.Bp, t.tt[j0 + j], e[j]); cm[j] = f2_fma(rc.nBp, t.tt[j0 + j], e[j]); }
#pragma unroll
    for (int j = 0; j < HB; ++j) {
      float lo, hi;
      f2_unpack(cp[j], lo, hi);
      f(V / 2 + j0 + j, lo, hi);
      f2_unpack(cm[j], lo, hi);
      f(V / 2 - 1 - (j0 + j), lo, hi);
    }
  }
}

// Tile geometry: THREADS = TXT*TYT*TZT threads, each owns a row of V voxels contiguous in x, so the tile is
// (TXT*V) x TYT x TZT voxels.  MINB = CTAs per SM the register allocation is held to.
// GROUP = seeds between two argmin checks (long rows on big problems: 16; short rows / few seeds: 8, where label
// changes are denser and a rescan should be short).
template <int DIM, int V_, int TXT_, int TYT_, int TZT_, int MINB_, int GROUP_>
struct RowGeom {
  static constexpr int V = V_, TXT = TXT_, TYT = TYT_, TZT = TZT_, THREADS = TXT_ * TYT_ * TZT_, MINB = MINB_,
                       GROUP = GROUP_;
};
constexpr int ROW_MINB = 3;                           // CTAs per SM (measured: 2, 3 and 4 within 0.3%)
// Two row lengths are built.  LONG rows (V = 32) amortise the per-(row, seed) set-up best and are used once the
// grid gives every SM at least ROW_LONG_MIN_WAVES waves of long-row tiles; smaller grids take SHORT rows (V = 16),
// whose tiles are half as big, so that all SMs have work.
using RowGeom3L = RowGeom<3, 32, 1, 16, 8, ROW_MINB, 16>;    // tile 32 x 16 x 8 voxels, 128 threads
using RowGeom3S = RowGeom<3, 16, 1, 16, 8, ROW_MINB, 8>;    // tile 16 x 16 x 8 voxels
using RowGeom2L = RowGeom<2, 32, 2, 64, 1, ROW_MINB, 16>;    // tile 64 x 64 pixels
using RowGeom2S = RowGeom<2, 16, 2, 64, 1, ROW_MINB, 8>;    // tile 32 x 64 pixels
constexpr int ROW_LONG_MIN_WAVES = 2;

constexpr int ROW_STAGES = 4;                         // smem ring of seed chunks

// Dynamic shared memory of one CTA:
//   seeds [ROW_STAGES][CHUNK_PAIRS*PREC] f32 | prev [V][THREADS] f32 | lab [V][THREADS] i32 |
//   full[ROW_STAGES], empty[ROW_STAGES] mbarriers | red [THREADS/32] f64
// prev[k][tid] = the minimum of voxel k as of its last label update (== best[k] except inside the group that
// lowers it); prev and lab live in shared memory because they are touched once per ROW_GROUP seeds, which
// leaves the registers to the V running minima and to the interleaved FMA chains.
template <int DIM, class G>
struct RowSmem {
  static constexpr int PREC = (DIM == 3) ? PREC3 : PREC2;
  static constexpr int CHUNK_PAIRS = SEED_CHUNK / 2;
  static constexpr size_t SEED_BYTES = (size_t)ROW_STAGES * CHUNK_PAIRS * PREC * sizeof(float);
  static constexpr size_t PREV_OFF = SEED_BYTES;
  static constexpr size_t LAB_OFF = PREV_OFF + (size_t)G::V * G::THREADS * sizeof(float);
  static constexpr size_t BAR_OFF = LAB_OFF + (size_t)G::V * G::THREADS * sizeof(int);
  static constexpr size_t RED_OFF = BAR_OFF + 2 * ROW_STAGES * sizeof(uint64_t);
  static constexpr size_t BYTES = RED_OFF + (G::THREADS / 32) * sizeof(double);
};

// One staged chunk of SEED_CHUNK seeds ibase .. ibase+SEED_CHUNK-1 (pair-interleaved records at `sp`) against the
// thread's row: rows a3 + a4 of the brute-force kernel.
template <int DIM, int V, int T, int ROW_GROUP>
__device__ __forceinline__ void row_process_chunk(const float* __restrict__ sp, int ibase, const RowRef<DIM>& rr,
                                                  const RowTau<V>& tt, float (&best)[V], float4* __restrict__ s_prev4,
                                                  int* __restrict__ s_lab, int tid) {
  constexpr int PREC = (DIM == 3) ? PREC3 : PREC2;
  constexpr int GROUP_PAIRS = ROW_GROUP / 2;
  for (int gidx = 0; gidx < SEED_CHUNK / ROW_GROUP; ++gidx) {
    const float* gp = sp + gidx * GROUP_PAIRS * PREC;
#pragma unroll 1
    for (int p = 0; p < GROUP_PAIRS; ++p) {
      const RowCoef rc = row_setup<DIM>(gp + p * PREC, rr);
      row_sweep<V>(rc, tt, [&](int k, float lo, float hi) { best[k] = min3f(best[k], lo, hi); });
    }
    asm volatile("" ::: "memory");   // keep the prev[] loads below the group loop (they would cost V registers)
    // fast path: did ANY of the row's minima drop in this group?  (V/4 LDS.128 + V compares)
    bool any = false;
#pragma unroll
    for (int k4 = 0; k4 < V / 4; ++k4) {
      const float4 pv = s_prev4[k4 * T + tid];
      any |= (best[4 * k4] < pv.x) | (best[4 * k4 + 1] < pv.y) | (best[4 * k4 + 2] < pv.z) | (best[4 * k4 + 3] < pv.w);
    }
    if (any) {
      // a4, deferred: the new minimum of every flagged voxel lies in this group; recompute the group with the same
      // instructions and take the first seed that attains it.  Events are rare (a few per cent of the groups) and
      // the early ones flag most of the row: one predicated pass over all V voxels measured fastest.
      unsigned int mask = 0u;
#pragma unroll
      for (int k4 = 0; k4 < V / 4; ++k4) {
        float4 pv = s_prev4[k4 * T + tid];
        if (best[4 * k4] < pv.x) { mask |= 1u << (4 * k4); pv.x = best[4 * k4]; }
        if (best[4 * k4 + 1] < pv.y) { mask |= 2u << (4 * k4); pv.y = best[4 * k4 + 1]; }
        if (best[4 * k4 + 2] < pv.z) { mask |= 4u << (4 * k4); pv.z = best[4 * k4 + 2]; }
        if (best[4 * k4 + 3] < pv.w) { mask |= 8u << (4 * k4); pv.w = best[4 * k4 + 3]; }
        s_prev4[k4 * T + tid] = pv;
      }
      for (int p = 0; p < GROUP_PAIRS && mask; ++p) {
        const RowCoef rc = row_setup<DIM>(gp + p * PREC, rr);
        const int i0 = ibase + gidx * ROW_GROUP + 2 * p;
        // a new seed takes over an interval of the row, and neighbouring rows (the other lanes) similar ones: test
        // the row in blocks of 8 voxels so that the untouched blocks cost one branch
#pragma unroll
        for (int k8 = 0; k8 < V; k8 += 8) {
          if (mask & (0xffu << k8)) {
#pragma unroll
            for (int k = k8; k < k8 + 8; ++k) {
              if (mask & (1u << k)) {
                float lo, hi;
                f2_unpack(row_cost<V>(rc, tt, k), lo, hi);
                if (lo == best[k]) { s_lab[k * T + tid] = i0; mask &= ~(1u << k); }
                else if (hi == best[k]) { s_lab[k * T + tid] = i0 + 1; mask &= ~(1u << k); }
              }
            }
          }
        }
      }
    }
  }
}

// Per-thread row set-up shared by the brute-force and the culled kernel (a1).
template <int DIM, class G>
struct RowThread {
  int ix0, iy, iz;
  bool row_valid;
  RowRef<DIM> rr;
  float xc, y0, z0;        // 3D: the tile's reference point (cook3)
  __device__ __forceinline__ void init(const AssignArgs& a, int b, int tid) {
    const int tx = tid % G::TXT, ty = (tid / G::TXT) % G::TYT, tz = tid / (G::TXT * G::TYT);
    const int bx = b % a.g.tiles_x, by = (b / a.g.tiles_x) % a.g.tiles_y, bz = b / (a.g.tiles_x * a.g.tiles_y);
    init_at(a, bx, by, bz, tx, ty, tz);
  }
  __device__ __forceinline__ void init_at(const AssignArgs& a, int bx, int by, int bz, int tx, int ty, int tz) {
    ix0 = (bx * G::TXT + tx) * G::V; iy = by * G::TYT + ty; iz = bz * G::TZT + tz;
    row_valid = (ix0 < a.g.nx) && (iy < a.g.ny) && (iz < a.g.nz);
    // coordinates from the indices (fp64 definitions rounded once to fp32); in x the row's midpoint
    xc = (float)(a.g.lo[0] + ((double)ix0 + 0.5 * (double)G::V) * a.g.s[0]);
    if constexpr (DIM == 3) {
      static_assert(G::TXT == 1, "3D: one reference point per tile");
      y0 = (float)(a.g.lo[1] + ((double)(by * G::TYT + a.g.off_y) + 0.5 * (double)G::TYT) * a.g.s[1]);
      z0 = (float)(a.g.lo[2] + ((double)(bz * G::TZT + a.g.off_z) + 0.5 * (double)G::TZT) * a.g.s[2]);
      const float Yf = (float)(((double)ty + 0.5 - 0.5 * (double)G::TYT) * a.g.s[1]);
      const float Zf = (float)(((double)tz + 0.5 - 0.5 * (double)G::TZT) * a.g.s[2]);
      const float YY = __fmul_rn(Yf, Yf), YZ = __fmul_rn(Yf, Zf), ZZ = __fmul_rn(Zf, Zf);
      rr.Y = f2_pack(Yf, Yf); rr.Z = f2_pack(Zf, Zf);
      rr.YY = f2_pack(YY, YY); rr.YZ = f2_pack(YZ, YZ); rr.ZZ = f2_pack(ZZ, ZZ);
    } else {
      y0 = 0.0f; z0 = 0.0f;
      const float yyf = (float)(a.g.lo[1] + ((double)(iy + a.g.off_y) + 0.5) * a.g.s[1]);
      rr.x0 = f2_pack(xc, xc); rr.yy = f2_pack(yyf, yyf);
    }
  }
  // in-row offsets from the midpoint (kernel parameters: uniform)
  __device__ __forceinline__ void tau(const AssignArgs& a, RowTau<G::V>& t) const {
#pragma unroll
    for (int j = 0; j < G::V / 2; ++j) { t.tt[j] = f2_pack(a.tt[j], a.tt[j]); t.tsq[j] = f2_pack(a.tt[16 + j], a.tt[16 + j]); }
  }
};

template <int DIM, class G>
__global__ void __launch_bounds__(G::THREADS, G::MINB) assign_rowpoly_kernel(const AssignArgs a) {
  constexpr int V = G::V, T = G::THREADS;
  using S = RowSmem<DIM, G>;
  constexpr int PREC = S::PREC;
  constexpr int CHUNK_PAIRS = S::CHUNK_PAIRS;
  constexpr uint32_t CHUNK_BYTES = CHUNK_PAIRS * PREC * sizeof(float);
  static_assert(V <= 32 && V % 4 == 0, "row mask is 32 bits; a.tt holds 16 + 16 offsets");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* s_seeds = reinterpret_cast<float*>(smem_raw);
  float4* s_prev4 = reinterpret_cast<float4*>(smem_raw + S::PREV_OFF);   // [V/4][T]
  int* s_lab = reinterpret_cast<int*>(smem_raw + S::LAB_OFF);
  uint64_t* s_full = reinterpret_cast<uint64_t*>(smem_raw + S::BAR_OFF);
  uint64_t* s_empty = s_full + ROW_STAGES;
  double* s_red = reinterpret_cast<double*>(smem_raw + S::RED_OFF);

  if (a.done_flag && *a.done_flag) return;
  const int tid = threadIdx.x;
  const int b = blockIdx.x;
  RowThread<DIM, G> rt;
  rt.init(a, b, tid);

  const int nchunks = a.M_pad / SEED_CHUNK;
  if (tid == 0) {
    for (int s = 0; s < ROW_STAGES; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], T / 32); }
    mbar_fence_init();
    for (int s = 0; s < ROW_STAGES && s < nchunks; ++s) {
      mbar_arrive_expect_tx(&s_full[s], CHUNK_BYTES);
      tma_bulk_g2s(s_seeds + (size_t)s * CHUNK_PAIRS * PREC, a.seeds + (size_t)s * CHUNK_PAIRS * PREC, CHUNK_BYTES,
                   &s_full[s]);
    }
  }

  RowTau<V> tt;
  rt.tau(a, tt);
  float best[V];
#pragma unroll
  for (int k = 0; k < V; ++k) {
    best[k] = CUDART_INF_F;
    s_lab[k * T + tid] = 0;
  }
#pragma unroll
  for (int k4 = 0; k4 < V / 4; ++k4)
    s_prev4[k4 * T + tid] = make_float4(CUDART_INF_F, CUDART_INF_F, CUDART_INF_F, CUDART_INF_F);
  __syncthreads();   // barrier initialisation visible to every thread

  for (int c = 0; c < nchunks; ++c) {
    const int stage = c % ROW_STAGES;
    if (tid == 0 && c >= 1 && c + ROW_STAGES - 1 < nchunks) {
      // refill the stage every warp left at iteration c-1 with chunk c + ROW_STAGES - 1
      const int s2 = (c - 1) % ROW_STAGES;
      mbar_wait(&s_empty[s2], (uint32_t)(((c - 1) / ROW_STAGES) & 1));
      mbar_arrive_expect_tx(&s_full[s2], CHUNK_BYTES);
      tma_bulk_g2s(s_seeds + (size_t)s2 * CHUNK_PAIRS * PREC,
                   a.seeds + (size_t)(c + ROW_STAGES - 1) * CHUNK_PAIRS * PREC, CHUNK_BYTES, &s_full[s2]);
    }
    mbar_wait(&s_full[stage], (uint32_t)((c / ROW_STAGES) & 1));
    float* chunk = s_seeds + (size_t)stage * CHUNK_PAIRS * PREC;
    if constexpr (DIM == 3) {
      // re-expand the chunk's seeds about this tile's reference point, in place (cook3): one seed per thread
      for (int sd = tid; sd < SEED_CHUNK; sd += T) {
        float* p = chunk + (sd >> 1) * PREC + (sd & 1);
        const Cooked3 ck = cook3(p[0], p[2], p[4], p[6], p[8], p[10], p[12], p[14], p[16], p[18], rt.xc, rt.y0, rt.z0);
        p[0] = ck.b0; p[2] = ck.r1; p[4] = ck.r2; p[18] = ck.r0;
      }
      fence_proxy_async_smem();      // these generic-proxy writes precede the TMA refill of the stage
      __syncthreads();
    }
    row_process_chunk<DIM, V, T, G::GROUP>(chunk, c * SEED_CHUNK, rt.rr, tt, best, s_prev4, s_lab, tid);
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(&s_empty[stage]);
  }

  int lab[V];
#pragma unroll
  for (int k = 0; k < V; ++k) lab[k] = s_lab[k * T + tid];
  const double dsum = row_epilogue<V>(a, rt.row_valid, rt.ix0, rt.iy, rt.iz, best, lab);
  const double tot = block_sum_double<T>(dsum, s_red);
  if (tid == 0) a.dual_partial[b] = tot;
}

// ------------------------------------------------------------------------------------------------------------
// a7: the same reduction over CANDIDATE LISTS (apd_cull.cu) instead of all seeds.  Every warp owns one brick of
// 32 rows x 16 voxels and walks ITS OWN list (a few dozen seeds) in chunks of 32 candidates: the lanes gather one
// candidate each from the per-seed record table into the warp's pair-interleaved staging buffer, __syncwarp, then the
// same row polynomial.  With lists this short every seed is a likely winner, so the argmin is tracked INLINE
// (min3, one compare for "dropped", one for "which lane") instead of by deferred rescans; labels stay in registers.
// Lists are ascending in seed index and the compare is strict, so ties still go to the lowest index (reading S1).
// The four warps of a CTA never synchronise: each writes its own dual partial.
// smem: per warp 2 stages x (16 pair records + 32 indices)
// ------------------------------------------------------------------------------------------------------------
constexpr int WCHUNK = 32;                      // candidates per warp-chunk
template <int DIM> struct CullGeom;
template <> struct CullGeom<3> { static constexpr int V = 16, TXT = 1, TYT = CULL_TILE3_Y, TZT = CULL_TILE3_Z, THREADS = 128; };
template <> struct CullGeom<2> { static constexpr int V = 16, TXT = 2, TYT = CULL_TILE2_Y, TZT = 1, THREADS = 128; };
static_assert(CullGeom<3>::TXT * CullGeom<3>::V == CULL_TILE3_X && CullGeom<2>::TXT * CullGeom<2>::V == CULL_TILE2_X, "tile");

template <int DIM>
__global__ void __launch_bounds__(128, 6) assign_rowpoly_culled_kernel(const AssignArgs a) {
  using G = CullGeom<DIM>;
  constexpr int V = G::V;
  constexpr int PREC = (DIM == 3) ? PREC3 : PREC2;
  constexpr int REC = (DIM == 3) ? REC3 : REC2;
  constexpr int NP = (DIM == 3) ? 10 : 6;       // parameters per seed in a record
  constexpr int STAGE_FLOATS = (WCHUNK / 2) * PREC;
  __shared__ __align__(16) float s_seeds[4][2][STAGE_FLOATS];
  __shared__ int s_idx[4][2][WCHUNK];

  pdl_enter();
  if (a.done_flag && *a.done_flag) return;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  // one CTA per tile, launched as a 3D grid: the tile's indices cost no integer divisions (three of them were ~65 of
  // the ~1500 instructions a warp spends on a brick)
  const int bx = blockIdx.x, by = blockIdx.y, bz = blockIdx.z;
  const int b = (bz * a.g.tiles_y + by) * a.g.tiles_x + bx;

  // a1: this thread's row inside its warp's brick (apd_internal.cuh: brick_box)
  int tx, ty, tz;
  if (DIM == 3) { tx = 0; ty = 4 * w + (lane & 3); tz = lane >> 2; }
  else          { tx = w & 1; ty = 32 * (w >> 1) + lane; tz = 0; }
  RowThread<DIM, G> rt;
  rt.init_at(a, bx, by, bz, tx, ty, tz);

  // the brick's candidate list; an overflowed list falls back to the super-tile's, then to all seeds
  const size_t brick = (size_t)b * 4 + w;
  const int* const blist = a.brick_list + brick * BRICK_CAP;
  // The first chunk's index and record are loaded SPECULATIVELY, before the count is known: count -> index -> record
  // is a chain of three dependent global loads in front of every brick, and this takes one link out of it.  Slot
  // `lane` of the list always exists (capacity 256); past the list's end it holds anything, so the index is clamped
  // into the record table and the loaded record is simply not used.
  const int idx_spec = __ldg(blist + lane);
  int cnt = a.brick_count[brick];
  float4 rec_spec[REC / 4];
  {
    const int ic = min(max(idx_spec, 0), a.M_pad - 1);
    const float4* src = reinterpret_cast<const float4*>(a.rec + (size_t)ic * REC);
#pragma unroll
    for (int q = 0; q < REC / 4; ++q) rec_spec[q] = __ldg(src + q);
  }
  const int* list = blist;
  if (cnt < 0) {
    constexpr int STX = (DIM == 3) ? SUPER3_TX : SUPER2_TX, STY = (DIM == 3) ? SUPER3_TY : SUPER2_TY,
                  STZ = (DIM == 3) ? SUPER3_TZ : 1;
    const int sup = ((bz / STZ) * a.super_y + by / STY) * a.super_x + bx / STX;
    cnt = a.super_count[sup];
    list = a.super_list + (size_t)sup * SUPER_CAP;
    if (cnt < 0) { cnt = a.M; list = nullptr; }
  }
  // at least one chunk and, below, at least one pair: an empty list (it cannot occur: the seed that attains the
  // smallest upper bound always survives) would evaluate one padding pair of cost +inf and keep label 0.  Without the
  // guarantee the compiler builds a second, specialised exit for the zero-trip case (~45 instructions of constant
  // set-up in front of the loop, executed by every warp).
  const int nchunks = max(1, (cnt + WCHUNK - 1) / WCHUNK);

  auto gather = [&](int c) {
    const int stage = c & 1;
    const int pos = c * WCHUNK + lane;
    float r[REC];
    int idx = 0;
    if (pos < cnt) {
      if (c == 0 && list == blist) {       // the speculative loads above
        idx = idx_spec;
#pragma unroll
        for (int q = 0; q < REC / 4; ++q) {
          r[4 * q] = rec_spec[q].x; r[4 * q + 1] = rec_spec[q].y; r[4 * q + 2] = rec_spec[q].z; r[4 * q + 3] = rec_spec[q].w;
        }
      } else {
        idx = list ? __ldg(list + pos) : pos;
        const float4* src = reinterpret_cast<const float4*>(a.rec + (size_t)idx * REC);
#pragma unroll
        for (int q = 0; q < REC / 4; ++q) {
          const float4 v4 = __ldg(src + q);
          r[4 * q] = v4.x; r[4 * q + 1] = v4.y; r[4 * q + 2] = v4.z; r[4 * q + 3] = v4.w;
        }
      }
    } else {
#pragma unroll
      for (int q = 0; q < REC; ++q) r[q] = 0.0f;
      r[NP - 1] = CUDART_INF_F;      // padding candidate: cost +inf, never wins the strict '<'
    }
    if constexpr (DIM == 3) {        // re-expand about the CTA tile's reference point, as the brute-force kernel does
      const Cooked3 ck = cook3(r[0], r[1], r[2], r[3], r[4], r[5], r[6], r[7], r[8], r[9], rt.xc, rt.y0, rt.z0);
      r[0] = ck.b0; r[1] = ck.r1; r[2] = ck.r2; r[9] = ck.r0;
    }
    float* dst = &s_seeds[w][stage][(lane >> 1) * PREC + (lane & 1)];
#pragma unroll
    for (int q = 0; q < NP; ++q) dst[2 * q] = r[q];
    s_idx[w][stage][lane] = idx;
  };
  gather(0);        // issued first: its latency overlaps the row set-up below

  RowTau<V> tt;
  rt.tau(a, tt);
  float best[V];
  int lab[V];
#pragma unroll
  for (int k = 0; k < V; ++k) { best[k] = CUDART_INF_F; lab[k] = 0; }
  __syncwarp();

  int c = 0;
  do {
    if (c + 1 < nchunks) gather(c + 1);     // the other stage: the warp left it before the last __syncwarp
    const float* sp = s_seeds[w][c & 1];
    const int* ip = s_idx[w][c & 1];
    const int npairs = max(1, min(WCHUNK / 2, (cnt - c * WCHUNK + 1) / 2));     // pairs that hold a real candidate
    int p = 0;
#pragma unroll 2
    do {
      const RowCoef rc = row_setup<DIM>(sp + p * PREC, rt.rr);
      const int i0 = ip[2 * p], i1 = ip[2 * p + 1];
      row_sweep<V>(rc, tt, [&](int k, float lo, float hi) {
        const float m = min3f(best[k], lo, hi);
        if (m < best[k]) lab[k] = (lo == m) ? i0 : i1;    // lo == hi == m: the lower index
        best[k] = m;
      });
    } while (++p < npairs);
    __syncwarp();
  } while (++c < nchunks);

  double dsum = row_epilogue<V>(a, rt.row_valid, rt.ix0, rt.iy, rt.iz, best, lab);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dsum += __shfl_down_sync(0xffffffffu, dsum, o);     // fixed order
  if (lane == 0) {
    a.dual_partial[brick] = dsum;
    if (!a.pairs_ctr) return;          // the evaluations inside a solve do not count pairs
    // voxel-seed pairs whose cost this brick evaluated (valid voxels only)
    int ox, oy, oz, ex, ey, ez;
    brick_box(DIM, w, &ox, &oy, &oz, &ex, &ey, &ez);
    const long long vx = max(0, min(ex, a.g.nx - (bx * G::TXT * V + ox))), vy = max(0, min(ey, a.g.ny - (by * G::TYT + oy))),
                    vz = max(0, min(ez, a.g.nz - (bz * G::TZT + oz)));
    if (vx * vy * vz > 0) atomicAdd(a.pairs_ctr, (unsigned long long)(vx * vy * vz) * (unsigned long long)cnt);
  }
}

static inline int cdiv_i(int x, int y) { return (x + y - 1) / y; }

template <class G>
static void tiles_of(int nx, int ny, int nz, int* tx, int* ty, int* tz) {
  *tx = cdiv_i(nx, G::TXT * G::V); *ty = cdiv_i(ny, G::TYT); *tz = cdiv_i(nz, G::TZT);
}

// Picks the row length (returned: 0 = SHORT, 1 = LONG) and the tile counts for a grid.  The culled kernel always
// runs the CullGeom tile (short rows).
int rowpoly_tile_counts(int dim, int nx, int ny, int nz, int sm_count, bool cull, int* tx, int* ty, int* tz) {
  if (cull) {
    if (dim == 3) { *tx = cdiv_i(nx, CULL_TILE3_X); *ty = cdiv_i(ny, CULL_TILE3_Y); *tz = cdiv_i(nz, CULL_TILE3_Z); }
    else          { *tx = cdiv_i(nx, CULL_TILE2_X); *ty = cdiv_i(ny, CULL_TILE2_Y); *tz = 1; }
    return 0;
  }
  if (dim == 3) tiles_of<RowGeom3L>(nx, ny, nz, tx, ty, tz); else tiles_of<RowGeom2L>(nx, ny, 1, tx, ty, tz);
  if ((long long)(*tx) * (*ty) * (*tz) >= (long long)ROW_LONG_MIN_WAVES * ROW_MINB * sm_count) return 1;
  if (dim == 3) tiles_of<RowGeom3S>(nx, ny, nz, tx, ty, tz); else tiles_of<RowGeom2S>(nx, ny, 1, tx, ty, tz);
  return 0;
}

template <int DIM, class G>
static cudaError_t launch_rowpoly_t(const AssignArgs& a, int n_tiles, cudaStream_t st) {
  // opt in to > 48 KB of dynamic shared memory (per device; a host-side attribute write, no launch)
  constexpr size_t bytes = RowSmem<DIM, G>::BYTES;
  cudaError_t e = cudaFuncSetAttribute(assign_rowpoly_kernel<DIM, G>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)bytes);
  if (e != cudaSuccess) return e;
  assign_rowpoly_kernel<DIM, G><<<n_tiles, G::THREADS, bytes, st>>>(a);
  return cudaGetLastError();
}

template <int DIM>
static cudaError_t launch_culled_t(const AssignArgs& a, int n_tiles, cudaStream_t st) {
  (void)n_tiles;
  return launch_pdl(assign_rowpoly_culled_kernel<DIM>, dim3((unsigned)a.g.tiles_x, (unsigned)a.g.tiles_y, (unsigned)a.g.tiles_z),
                    128, 0, st, a);
}

cudaError_t launch_assign_rowpoly(const AssignArgs& a, cudaStream_t st) {
  const int n_tiles = a.g.tiles_x * a.g.tiles_y * a.g.tiles_z;
  if (a.brick_count) return a.g.dim == 3 ? launch_culled_t<3>(a, n_tiles, st) : launch_culled_t<2>(a, n_tiles, st);
  if (a.g.dim == 3)
    return a.g.row_long ? launch_rowpoly_t<3, RowGeom3L>(a, n_tiles, st) : launch_rowpoly_t<3, RowGeom3S>(a, n_tiles, st);
  return a.g.row_long ? launch_rowpoly_t<2, RowGeom2L>(a, n_tiles, st) : launch_rowpoly_t<2, RowGeom2S>(a, n_tiles, st);
}

}  // namespace apd
