// apd_lbfgs.cu -- Algorithm 2: maximise the discrete dual g~ (eq. 2.7) over the
// weights with L-BFGS until the stopping rule of eq. (2.5) holds.  The paper fixes only "W0 = 0,
// L-BFGS [70], stop when |v_i - m_i|P|| <= eps v_i"; every other detail is DESIGN.md's
// specification S9 (rows a10-a11), restated here from that specification:
//   * fp64 optimiser state; every evaluation uses fl32(w) (round to nearest even), S10
//   * f = -g~(fl32 w), grad f = vol - v                     (eq. 2.8 with the sign of f)
//   * first-direction scale gamma = l^(2-d)/d, l = (|Omega|/M)^(1/d)
//   * weak-Wolfe bracketing line search: c1 = 1e-4, c2 = 0.9, alpha0 = 1, at most 30 trials;
//     Armijo fails -> hi = alpha; curvature fails -> lo = alpha; alpha = (lo+hi)/2 or 2 alpha
//   * stopping test after EVERY evaluation
//   * curvature pair kept iff s.y > 1e-12 |s||y|; then gamma = s.y / y.y
//   * line-search failure: clear the history and retry with p = -gamma g; with an empty history
//     NOT_CONVERGED; NOT_CONVERGED returns the evaluated point with the smallest error.
// The whole state machine is ONE kernel (lbfgs_step_kernel, one cluster of 8 or 16 CTAs) that runs after each
// evaluation on the same stream; the host only reads the mapped SolveReport.done word.  The same loop serves voxel
// grids (apd_solve) and user-supplied point sets (apd_solve_points).
#include "apd_internal.cuh"
#include "apd_device.cuh"
#include <cmath>
#include <functional>
#include <cooperative_groups.h>
namespace cg = cooperative_groups;
#include <vector>

namespace apd {

constexpr int LB_THREADS = 256;
// CTAs (SMs) of the step kernel's thread-block cluster: 8 (the portable maximum), or 16 for M >= LB_CLUSTER_MAX_MIN_M
// where the device can co-schedule such a cluster (a non-portable size: B200 can; lb_cluster_size asks once per
// context).  The sweeps over the L-BFGS vectors (3.6 MB per step at M = 10^4, m = 10) go with 1 / CTAs, a cluster
// barrier costs more on 16 CTAs.  Measured step time, 8 vs 16 CTAs: M = 10^4 21.4 vs 18.7 us, M = 2 10^4 37.0 vs 27.0,
// M = 5000 13.3 vs 14.3, M = 1000 12.7 vs 13.7.
constexpr int LB_CLUSTER_MAX = 16, LB_CLUSTER_PORTABLE = 8;
constexpr int LB_CLUSTER_MAX_MIN_M = 8192;
constexpr int LB_MAX_HIST = 64;
constexpr int LB_MAX_TRIALS = 30;

struct SolveState {
  int done, phase, iters, evals, trial, hist_len, hist_start, hist_cap, max_iters, max_evals;
  double f, gp, alpha, lo, hi, gamma, eps, best_err, best_dual, domain_volume;
  double rho[LB_MAX_HIST];
  // candidate-list reuse (apd_cull.cu): the brick lists were built at wref with slack cull_delta and stay valid while
  // max_i |w32_i - wref_i| <= cull_delta; the super-tile lists they are cut from were built at wref_s with the larger
  // slack cull_delta_s and are rebuilt only when the ball the brick lists must cover leaves theirs
  int cull_rebuild, cull_rebuilds, cull_rebuild_s, cull_rebuilds_s, cull_rebuild_t, cull_rebuilds_t;
  float cull_delta, cull_cap, cull_delta_s, cull_delta_t;
};

enum { V_W = 0, V_G, V_P, V_WTRY, V_WBEST, V_GNEW, V_Q, V_HIST };   // rows of svec

struct StepArgs {
  SolveState* st;
  double* vec;         // [(V_HIST + 2 hist_cap) * stride]
  int stride;          // = max_seeds
  int M;
  const float* v;      // target volumes
  // raw outputs of the evaluation just run (the loop skips finalize_kernel and finishes eq. 2.7 / 2.8 / 2.5 here)
  const unsigned int* count;      // [M] voxels per cell (grid evaluations), or nullptr:
  const unsigned long long* count64;  // [M] the same as u64: the REDUCED counter block of a slab-sharded solve, or:
  const double* vol_in;           // [M] cell volumes already in fp64 (apd_solve_points; voxel_volume is then 1)
  const double* dual_partial;     // [lm.n_partials] sums of min-costs per tile / brick; nullptr when layer_in is given
  LayerMap lm;                    // two-level reduction of dual_partial (apd_internal.cuh)
  double* layer_buf;              // [lm.n_layers] scratch the layer sums are formed in
  const double* layer_in;         // [lm.n_layers] layer sums already reduced over the slabs (sharded solve), else nullptr
  double voxel_volume;            // |P|
  float* w32;          // next evaluation's weights
  SolveReport* report; // mapped host memory
  double* hist;        // [2 * hist_cap] (dual, max_rel_err) of every evaluation, in order
  int hist_cap;
  float* wref;         // weights the brick candidate lists were built at (culling only)
  float* wref_s;       // weights the super-tile lists were built at
  float* wref_t;       // weights the CTA-tile lists were built at
  // culled solves: the step kernel itself refreshes what cull_pack_kernel would rewrite before the next evaluation --
  // the -w slot of every seed's record and the zeroed voxel counts -- so the loop launches no pack kernel after the
  // first evaluation (X, A and the box radii of a record do not change inside a solve)
  float* rec_nw = nullptr;     // &rec[0][slot of -w], or nullptr (no culling / points)
  int rec_stride = 0;          // floats per record
  unsigned int* count_zero = nullptr;   // [M] the evaluation's voxel counts, to be zeroed for the next one
  double* gram;        // [LB_CLUSTER_MAX] copies of { (2 hist_cap + 1)^2 Gram matrix, hist_cap rho }, see GramSmem
};

constexpr double CULL_DELTA_FACTOR = 4.0;   // slack of a rebuilt list = this x the last change of the weights ...
constexpr double CULL_CAP_FACTOR = 0.5;     // ... but at most this x the mean min-cost of the first evaluation (a larger
                                            // slack would lengthen every list by more than it saves in rebuilds)
// The three list levels keep slacks of their own: a brick list is cut from its CTA tile's list, that from its
// super-tile's, and the coarser a box the looser its bounds, so a coarser list barely grows with a larger slack while
// it is rebuilt far less often.  Measured (cfg 4 / cfg 5 solve, 59 / 61 brick rebuilds in 163 / 147 evaluations), before
// programmatic dependent launch: one slack for all levels 25.0 / 107 ms; super x4 23.7 / 99.9 (27 / 28 super-tile
// rebuilds); x8 23.3 / 96.7 (12 / 11); x16 23.3 / 97.1; x64 24.5 / 106.6.  With it, super x16 and the CTA-tile lists kept
// in global memory: tile x2 22.1 / 99.3 (56 tile rebuilds), x3 21.5 / 96.1 (38), x4 21.1 / 94.7 (27), x6 21.0 / 93.0
// (17 / 14), x8 (super x24) 21.0 / 93.7, x12 (x32) 21.6 / 96.7, x24 (x64) 23.8 / 111.
constexpr double CULL_TILE_FACTOR = 6.0;    // slack of a rebuilt CTA-tile list = this x the brick lists'
constexpr double CULL_SUPER_FACTOR = 16.0;  // slack of a rebuilt super-tile list = this x the brick lists' (>= the tile factor)

// ---- reductions over the CLUSTER ------------------------------------------------------------------------------
// The step kernel is ONE thread-block cluster of nranks = 8 or 16 CTAs (one per SM): a single CTA cannot keep enough loads
// in flight to stream the L-BFGS vectors (measured: its sweeps ran at pure L2 latency), eight can.  Element i of
// every length-M vector is owned by one thread of one CTA in every sweep (i = tid + LB_THREADS (rank + nranks k)),
// so vectors need no synchronisation; scalars come from reductions that return the SAME value, bit for bit, to every
// thread of every CTA (lanes by shuffle tree, warps in order, CTAs in rank order), which keeps the control flow
// uniform over the whole cluster.  Cluster partials are exchanged through distributed shared memory; two buffers
// are used alternately so that one cluster barrier per reduction suffices.
constexpr int LB_GRAM_SLOTS = 10;                    // history slots whose inner products one pass forms at once
constexpr int LB_NPROD = 3 * 2 * LB_GRAM_SLOTS;      // (s, y, g1) x (S_j, Y_j) of LB_GRAM_SLOTS slots
constexpr int LB_NPROD_PAD = (LB_NPROD + 31) / 32 * 32;   // padded to whole warps: the products are reduced TRANSPOSED
// scalars of the evaluation sweep (the last one is a maximum, the others sums)
enum { SC_VW = 0, SC_V, SC_G1P, SC_SY, SC_SS, SC_YY, SC_G1S, SC_G1Y, SC_G1G1, SC_ERR, LB_NSCAL };
constexpr int LB_NRED = LB_NPROD_PAD + LB_NSCAL;     // most values reduced at once (eval_sweep)

struct Reducer {
  double* wbuf;        // [LB_THREADS / 32][LB_NRED]   warp partials of this CTA
  double* cbuf;        // [2][LB_NRED]                 CTA totals, read by the other CTAs of the cluster
  double* tot;         // [LB_NRED]                    cluster totals, for this CTA's threads
  int flip;
  unsigned int rank, nranks;     // this CTA's rank in the cluster, CTAs in the cluster
};

// One halving step of the TRANSPOSED warp reduction: lanes whose BIT is set keep the upper HALF of the values, the
// others the lower, and each adds what its partner sends of the half it keeps (one shuffle per PAIR of values).
template <int HALF, int BIT, int N>
__device__ __forceinline__ void warp_transpose_step(double (&v)[N], int lane) {
  const bool up = (lane & BIT) != 0;
#pragma unroll
  for (int k = 0; k < HALF; ++k) {
    const double keep = up ? v[k + HALF] : v[k];
    const double send = up ? v[k] : v[k + HALF];
    v[k] = keep + __shfl_xor_sync(0xffffffffu, send, BIT);
  }
}

// v[0 .. N-NMAX) are SUMMED, v[N-NMAX .. N) are MAXIMISED, all in one exchange (one cluster barrier).  Every value
// goes through one fixed tree: lanes, then warps in order, then CTAs in rank order.  The lane stage of the first
// NT = 32 floor((N - NMAX) / 32) sums is the transposed reduction (5 halving steps, after which each lane holds the
// totals of NT / 32 values: NT - NT/32 shuffles instead of 5 NT -- the warp shuffle unit, one instruction per clock
// per SM, was what a 70-value exchange waited for); the rest go through the xor butterfly.  A value's tree depends
// only on whether its index is below NT.  READBACK = false: the totals are left in r.tot[] only.
template <int N, int NMAX, bool READBACK = true>
__device__ __forceinline__ void cluster_all_mixed(double (&v)[N], Reducer& r) {
  cg::cluster_group cluster = cg::this_cluster();
  constexpr int NT = (N - NMAX) / 32 * 32, PER = NT / 32;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if constexpr (NT > 0) {
    warp_transpose_step<NT / 2, 16>(v, lane);
    warp_transpose_step<NT / 4, 8>(v, lane);
    warp_transpose_step<NT / 8, 4>(v, lane);
    warp_transpose_step<NT / 16, 2>(v, lane);
    warp_transpose_step<NT / 32, 1>(v, lane);
  }
#pragma unroll
  for (int n = NT; n < N; ++n) {
    const bool MAX = n >= N - NMAX;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double u = __shfl_xor_sync(0xffffffffu, v[n], o);
      v[n] = MAX ? fmax(v[n], u) : v[n] + u;
    }
  }
  __syncthreads();                                   // wbuf free (its last readers are past this point)
  if constexpr (NT > 0) {
    // lane L holds the totals of values base(L) + j, j < PER
    const int base = ((lane >> 4) & 1) * (NT / 2) + ((lane >> 3) & 1) * (NT / 4) + ((lane >> 2) & 1) * (NT / 8) +
                     ((lane >> 1) & 1) * (NT / 16) + (lane & 1) * (NT / 32);
#pragma unroll
    for (int j = 0; j < PER; ++j) r.wbuf[wid * LB_NRED + base + j] = v[j];
  }
  if (lane == 0) {
#pragma unroll
    for (int n = NT; n < N; ++n) r.wbuf[wid * LB_NRED + n] = v[n];
  }
  __syncthreads();
  r.flip ^= 1;
  double* mine = r.cbuf + r.flip * LB_NRED;
  if (threadIdx.x < N) {
    const bool MAX = (int)threadIdx.x >= N - NMAX;
    double t = r.wbuf[threadIdx.x];
#pragma unroll
    for (int k = 1; k < LB_THREADS / 32; ++k) {
      const double u = r.wbuf[k * LB_NRED + threadIdx.x];
      t = MAX ? fmax(t, u) : t + u;
    }
    mine[threadIdx.x] = t;
  }
  cluster.sync();                                    // every CTA's totals are written and visible
  // N threads fetch the other CTAs' totals (one distributed-shared-memory read each: every thread reading all of
  // them cost more than the sweeps), add them in rank order and hand the result to the CTA through shared memory
  if (threadIdx.x < N) {
    const bool MAX = (int)threadIdx.x >= N - NMAX;
    double t = cluster.map_shared_rank(mine, 0)[threadIdx.x];
    if (r.nranks == LB_CLUSTER_MAX) {         // (both sizes unrolled: the remote reads are issued together)
#pragma unroll
      for (int c = 1; c < LB_CLUSTER_MAX; ++c) {
        const double u = cluster.map_shared_rank(mine, c)[threadIdx.x];
        t = MAX ? fmax(t, u) : t + u;
      }
    } else {
#pragma unroll
      for (int c = 1; c < LB_CLUSTER_PORTABLE; ++c) {
        const double u = cluster.map_shared_rank(mine, c)[threadIdx.x];
        t = MAX ? fmax(t, u) : t + u;
      }
    }
    r.tot[threadIdx.x] = t;
  }
  __syncthreads();
  if constexpr (READBACK) {
#pragma unroll
    for (int n = 0; n < N; ++n) v[n] = r.tot[n];
  }
}
template <int N, bool MAX>
__device__ __forceinline__ void cluster_all(double (&v)[N], Reducer& r) { cluster_all_mixed<N, MAX ? N : 0>(v, r); }

__device__ __forceinline__ double cluster_allsum(double x, Reducer& r) {
  double v[1] = {x};
  cluster_all<1, false>(v, r);
  return v[0];
}
__device__ __forceinline__ double cluster_allmax(double x, Reducer& r) {
  double v[1] = {x};
  cluster_all<1, true>(v, r);
  return v[0];
}

// element loop of this thread: for (int i = LB_FIRST(r); i < M; i += LB_STEP_R)
#define LB_FIRST(r) ((int)threadIdx.x + LB_THREADS * (int)(r).rank)
#define LB_STEP_OF(r) (LB_THREADS * (int)(r).nranks)

// ---- the L-BFGS direction in "vector-free" form ---------------------------------------------------------------
// The two-loop recursion of Liu & Nocedal [70] only ever forms linear combinations of the 2m+1 basis vectors
// b = (s_0..s_{m-1}, y_0..y_{m-1}, g) and inner products with them, so it can be run on the COEFFICIENTS of q in
// that basis given the Gram matrix B = b^T b: the same algorithm, the same result up to fp64 rounding, but the 2m
// dependent passes over the length-M vectors (each a latency-bound reduction) become the Gram products, which ride on
// the evaluation sweep (eval_sweep), plus ONE combination pass (combine_and_trial): an accepted step is two passes
// over the vectors and two exchanges.  Every CTA keeps its own copy of the Gram matrix and of rho in global memory
// (all copies are identical, no cross-CTA visibility to arrange), in SLOT space (ring slots of S and Y):
//   index of S slot j = j,  of Y slot j = cap + j,  of g = 2 cap;  leading dimension ld = 2 cap + 1;
//   a copy is ld*ld doubles of Gram matrix followed by cap doubles of rho.
__device__ __forceinline__ double* gram_of(const StepArgs& a, int cap, unsigned int rank) {
  return a.gram + (size_t)rank * ((size_t)(2 * cap + 1) * (2 * cap + 1) + cap);
}

// ---- the sweep over the evaluation just run ---------------------------------------------------------------------
// ONE pass and ONE exchange for everything that depends only on that evaluation and on the state at entry:
// <v, fl32 w> and the eq. (2.5) error (a9), the gradient g1 = vol - v of f at the evaluated point (eq. 2.8), the inner
// products of the line-search tests and of the curvature pair s = alpha p, y = g1 - g, and -- GRAM, i.e. when there
// is a history -- speculatively the Gram rows an ACCEPTED step needs: (s, y, g1) . (S_j, Y_j) for the first
// LB_GRAM_SLOTS active slots (nearly every evaluation is accepted: 161 of 163 on cfg 4; a rejected trial wastes
// the products, not a pass).  Sums are accumulated per thread in element order and reduced by one tree each, so a
// value's bits do not depend on what shares the exchange.  Leaves g1 in gnew; writes nothing else.
// The cluster totals are left in r.tot[]:
//   GRAM:  [0 .. LB_NPROD) products, [(n * LB_GRAM_SLOTS + q) * 2 + (0: S, 1: Y)], n = 0: s, 1: y, 2: g1, q = position
//          of the slot in ring order (0 = oldest); [LB_NPROD_PAD + SC_*] the scalars;     !GRAM: [SC_*] the scalars.
template <bool GRAM>
__device__ void eval_sweep(const StepArgs& a, int phase, double alpha, int cap, int hist_len, int hist_start,
                           Reducer& r) {
  double out[LB_NRED];
  const int M = a.M, stride = a.stride;
  const double P = a.voxel_volume;
  const double* g = a.vec + (size_t)V_G * stride;
  const double* p = a.vec + (size_t)V_P * stride;
  double* gnew = a.vec + (size_t)V_GNEW * stride;
  const double* S = a.vec + (size_t)V_HIST * stride;
  const double* Y = S + (size_t)cap * stride;
  constexpr int NS = LB_GRAM_SLOTS;
  const int LB_STEP_R = LB_STEP_OF(r);
  size_t soff[NS];
#pragma unroll
  for (int q = 0; q < NS; ++q) soff[q] = (size_t)((hist_start + (q < hist_len ? q : 0)) % cap) * stride;   // inactive: a duplicate
#pragma unroll
  for (int n = 0; n < LB_NRED; ++n) out[n] = 0.0;
  double* sc = out + LB_NPROD_PAD;
  for (int i = LB_FIRST(r); i < M; i += LB_STEP_R) {
    const double tv = (double)a.v[i];
    const double w32 = (double)a.w32[i];
    const double vi = a.vol_in ? a.vol_in[i] : (a.count64 ? (double)a.count64[i] : (double)a.count[i]) * P;
    double pi = 0.0, go = 0.0, sv[NS], yv[NS];
    if (phase != 0) { pi = p[i]; go = g[i]; }
    if (GRAM) {
#pragma unroll
      for (int q = 0; q < NS; ++q) { sv[q] = S[soff[q] + i]; yv[q] = Y[soff[q] + i]; }
    }
    sc[SC_VW] += tv * w32;
    sc[SC_ERR] = fmax(sc[SC_ERR], fabs(vi - tv) / tv);
    const double gn = vi - tv;                                  // m_i |P| - v_i
    gnew[i] = gn;
    sc[SC_V] += tv;
    sc[SC_G1G1] += gn * gn;
    if (phase != 0) {
      const double si = __dmul_rn(alpha, pi);
      const double yi = __dsub_rn(gn, go);
      sc[SC_G1P] += gn * pi; sc[SC_SY] += si * yi; sc[SC_SS] += si * si; sc[SC_YY] += yi * yi;
      sc[SC_G1S] += gn * si; sc[SC_G1Y] += gn * yi;
      if (GRAM) {
        const double x[3] = {si, yi, gn};
#pragma unroll
        for (int q = 0; q < NS; ++q) {
#pragma unroll
          for (int n = 0; n < 3; ++n) { out[(n * NS + q) * 2] += x[n] * sv[q]; out[(n * NS + q) * 2 + 1] += x[n] * yv[q]; }
        }
      }
    }
  }
  if (GRAM) cluster_all_mixed<LB_NRED, 1, false>(out, r);
  else {
    double t[LB_NSCAL];
#pragma unroll
    for (int n = 0; n < LB_NSCAL; ++n) t[n] = sc[n];
    cluster_all_mixed<LB_NSCAL, 1, false>(t, r);
  }
}

// The same products for the active slots [t0, t0 + ns) of a history longer than LB_GRAM_SLOTS (t0 > 0): run after an
// accepted step's decision and BEFORE its vector writes (s, y, g1 are formed from alpha, p, gnew and the old g).
// The cluster totals are left in r.tot[0 .. LB_NPROD).
__device__ void gram_products(const StepArgs& a, double alpha, int cap, int hist_start, int t0, int ns, Reducer& r) {
  const int M = a.M, stride = a.stride;
  const double* g = a.vec + (size_t)V_G * stride;
  const double* p = a.vec + (size_t)V_P * stride;
  const double* gnew = a.vec + (size_t)V_GNEW * stride;
  const double* S = a.vec + (size_t)V_HIST * stride;
  const double* Y = S + (size_t)cap * stride;
  constexpr int NS = LB_GRAM_SLOTS;
  const int LB_STEP_R = LB_STEP_OF(r);
  size_t soff[NS];
#pragma unroll
  for (int q = 0; q < NS; ++q) soff[q] = (size_t)((hist_start + t0 + (q < ns ? q : 0)) % cap) * stride;
  double acc[LB_NPROD_PAD];
#pragma unroll
  for (int n = 0; n < LB_NPROD_PAD; ++n) acc[n] = 0.0;
  for (int i = LB_FIRST(r); i < M; i += LB_STEP_R) {
    const double gn = gnew[i];
    const double x[3] = {__dmul_rn(alpha, p[i]), __dsub_rn(gn, g[i]), gn};
    double sv[NS], yv[NS];
#pragma unroll
    for (int q = 0; q < NS; ++q) { sv[q] = S[soff[q] + i]; yv[q] = Y[soff[q] + i]; }
#pragma unroll
    for (int q = 0; q < NS; ++q) {
#pragma unroll
      for (int n = 0; n < 3; ++n) { acc[(n * NS + q) * 2] += x[n] * sv[q]; acc[(n * NS + q) * 2 + 1] += x[n] * yv[q]; }
    }
  }
  cluster_all_mixed<LB_NPROD_PAD, 0, false>(acc, r);
}

// The CTA's working copy of the Gram matrix lives in its dynamic shared memory for the length of a step (GramSmem):
// prefetched from the CTA's global copy at entry, patched after the decision, read by direction_coeffs; every patch
// is also written through to the global copy, which carries it to the next launch.  Layout (doubles): the matrix in
// SLOT space [ld x ld], ld = 2 cap + 1 (S slot j -> j, Y slot j -> cap + j, g -> 2 cap), rho [cap], then the
// coefficient vectors of direction_coeffs.
struct GramSmem {
  double* m;         // [ld * ld]
  double* rho;       // [cap]
  double* delta;     // [ld]
  double* al;        // [cap]
  int* slot_of;      // [cap]
  double* glob;      // this CTA's global copy: matrix, then rho
  int ld;
  __device__ void set(int r, int c, double v) const { m[(size_t)r * ld + c] = v; glob[(size_t)r * ld + c] = v; }
  __device__ void set_sym(int r, int c, double v) const { set(r, c, v); set(c, r, v); }
};
__device__ __forceinline__ GramSmem gram_smem(const StepArgs& a, int cap, unsigned int rank, double* dyn) {
  GramSmem G;
  G.ld = 2 * cap + 1;
  G.m = dyn; G.rho = G.m + (size_t)G.ld * G.ld; G.delta = G.rho + cap; G.al = G.delta + G.ld;
  G.slot_of = reinterpret_cast<int*>(G.al + cap);
  G.glob = gram_of(a, cap, rank);
  return G;
}

// Writes the products prod[] (layout of eval_sweep) of the active slots [t0, t0 + ns) -- ring positions BEFORE the
// push -- into both triangles of the Gram matrix: the row of g always; the rows of the pushed pair when
// new_slot >= 0, except against the pair it evicts (`evicts`: the ring was full, position 0 is overwritten).
__device__ void gram_writeback(const GramSmem& G, int cap, const double* prod, int hist_start, int t0, int ns,
                               int new_slot, bool evicts) {
  constexpr int NS = LB_GRAM_SLOTS;
  if ((int)threadIdx.x < 3 * ns) {
    const int n = (int)threadIdx.x / ns, k = (int)threadIdx.x % ns;
    const bool skip = (n < 2 && new_slot < 0) || (evicts && t0 + k == 0);     // (that slot now holds the new pair)
    if (!skip) {
      const int q = (n == 0) ? new_slot : (n == 1 ? cap + new_slot : 2 * cap);
      const int j = (hist_start + t0 + k) % cap;
      G.set_sym(q, j, prod[(n * NS + k) * 2]);
      G.set_sym(q, cap + j, prod[(n * NS + k) * 2 + 1]);
    }
  }
}

// The coefficients of p = -H g (H0 = gamma I) in the basis (S.., Y.., g), from the Gram matrix in shared memory
// (complete and visible to the CTA: the caller has synchronised after its last patch).
struct DirCoef {
  const double* delta;     // [2 hl + 1]: S coefficients, Y coefficients, g coefficient
  const int* slot_of;      // [hl] ring slot of pair t (0 = oldest)
  int hl;
};
__device__ DirCoef direction_coeffs(const GramSmem& G, int cap, int hist_len, int hist_start, double gamma) {
  const int ld = G.ld, hl = hist_len, n = 2 * hl + 1, tid = threadIdx.x;
  double* delta = G.delta;
  if (tid < 32 && hl <= 32) {
    // The two-loop recursion [70] on coefficients, as two TRIANGULAR substitutions with lane t owning pair t (ring
    // order, 0 = oldest).  Written out, the first loop's alpha_t = rho_t s_t.q_t with q_t = g - sum_{u>t} alpha_u y_u is
    //     alpha_t / rho_t = s_t.g - sum_{u>t} (s_t.y_u) alpha_u,
    // and the second loop's beta_t = rho_t y_t.r_t with r_t = gamma q_0 + sum_{u<t} c_u s_u, c_u = alpha_u - beta_u, is
    //     beta_t / rho_t = gamma (y_t.g - sum_u (y_t.y_u) alpha_u) + sum_{u<t} (y_t.s_u) c_u:
    // once alpha_u (c_u) is known every lane folds it into its own right-hand sides, so a step of the dependent chain
    // is one multiply, one shuffle and one FMA instead of a 5-round shuffle reduction through shared memory (9 us of
    // the step at m = 10).  The same terms as the textbook loops, summed pair by pair.
    const int lane = tid;
    const bool mine = lane < hl;
    const int my_slot = (hist_start + (mine ? lane : 0)) % cap;
    const double* rowS = G.m + (size_t)my_slot * ld;                // s_t . (S.., Y.., g), slot space
    const double* rowY = G.m + (size_t)(cap + my_slot) * ld;        // y_t . (S.., Y.., g)
    const double rho_me = mine ? G.rho[my_slot] : 0.0;
    double rhs = mine ? rowS[2 * cap] : 0.0, b = mine ? rowY[2 * cap] : 0.0, alpha_me = 0.0;
    int su = (hist_start + (hl > 0 ? hl - 1 : 0)) % cap;              // slot of pair u
    for (int u = hl - 1; u >= 0; --u) {                 // newest -> oldest
      const double au = __shfl_sync(0xffffffffu, __dmul_rn(rho_me, rhs), u);
      if (lane == u) alpha_me = au;
      if (lane < u) rhs = __fma_rn(-rowS[cap + su], au, rhs);
      if (mine) b = __fma_rn(-rowY[cap + su], au, b);    // (the second loop's alpha sum, folded in as alpha_u appears)
      su = (su == 0) ? cap - 1 : su - 1;
    }
    double acc = __dmul_rn(gamma, b), c_me = 0.0;
    su = hist_start % cap;
    for (int u = 0; u < hl; ++u) {                      // oldest -> newest
      const double cu = __shfl_sync(0xffffffffu, __dsub_rn(alpha_me, __dmul_rn(rho_me, acc)), u);
      if (lane == u) c_me = cu;
      if (mine && lane > u) acc = __fma_rn(rowY[su], cu, acc);
      su = (su + 1 == cap) ? 0 : su + 1;
    }
    if (mine) { delta[lane] = c_me; delta[hl + lane] = -__dmul_rn(gamma, alpha_me); G.slot_of[lane] = my_slot; }
    if (lane == 0) delta[2 * hl] = gamma;
  } else if (tid < 32) {
    // histories longer than a warp: the textbook loops on the coefficient vector
    const int lane = tid;
    auto gi = [&](int c) { return c < hl ? (hist_start + c) % cap : (c < 2 * hl ? cap + (hist_start + c - hl) % cap : 2 * cap); };
    for (int j = lane; j < hl; j += 32) G.slot_of[j] = (hist_start + j) % cap;
    for (int j = lane; j < n; j += 32) delta[j] = (j == n - 1) ? 1.0 : 0.0;
    __syncwarp();
    for (int t = hl - 1; t >= 0; --t) {                 // newest -> oldest: alpha_t = rho_t s_t.q ; q -= alpha_t y_t
      double part = 0.0;
      for (int j = lane; j < n; j += 32) part += delta[j] * G.m[(size_t)gi(t) * ld + gi(j)];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
      const double alv = G.rho[gi(t)] * part;
      if (lane == 0) { G.al[t] = alv; delta[hl + t] = __dsub_rn(delta[hl + t], alv); }
      __syncwarp();
    }
    for (int j = lane; j < n; j += 32) delta[j] = __dmul_rn(gamma, delta[j]);    // r = gamma q
    __syncwarp();
    for (int t = 0; t < hl; ++t) {                       // oldest -> newest: r += s_t (alpha_t - rho_t y_t.r)
      double part = 0.0;
      for (int j = lane; j < n; j += 32) part += delta[j] * G.m[(size_t)gi(hl + t) * ld + gi(j)];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
      if (lane == 0) delta[t] = __dadd_rn(delta[t], G.al[t] - G.rho[gi(t)] * part);
      __syncwarp();
    }
  }
  __syncthreads();
  return DirCoef{delta, G.slot_of, hl};
}

// The combination pass fused with the trial point and, after an accepted step whose pair is kept, with that step's
// vector writes: for every element
//     [push]  s = alpha_old p, y = g1 - g  -> ring slot push.slot;   w <- w_try;   g <- g1
//     p = -(delta_g g + sum_t delta_t s_t + delta_{m+t} y_t),   w_try = w + alpha p  (alpha = 1: a new direction),
// w32 = fl32(w_try) (S10), the best-so-far copy of the point just evaluated, and ONE exchange for g.p (sum) and the two
// maxima the candidate-list reuse needs (|change since the last evaluation|, |distance from wref|, from wref_s).  Two elements
// per thread are in flight, and the history loads of an element are issued LB_COMB_SLOTS pairs at a time before any
// of them is used (a loop of dependent load-FMA pairs ran at one L2 round trip per four pairs: 9 of the step's 36 us
// at M = 10^4).  All loads of an element precede its stores; the pushed pair is used from registers.
constexpr int LB_COMB_SLOTS = 10;
constexpr int LB_COMB_U = 2;
struct PushArgs {
  bool on;                   // this step pushes the pair (alpha_old p, g1 - g) into ring slot `slot`
  double alpha_old;
  int slot;
};
struct TrialArgs {
  bool improved;             // copy w_eval -> w_best first
  const double* w_eval;      // the point the evaluation just run was taken at
  double alpha;
};
__device__ void combine_and_trial(const StepArgs& a, int cap, const DirCoef& dc, const TrialArgs& ta,
                                  const PushArgs& pu, Reducer& r, double* gp_out, double (&mx_out)[4]) {
  const int M = a.M, stride = a.stride, hl = dc.hl;
  double* g = a.vec + (size_t)V_G * stride;
  double* p = a.vec + (size_t)V_P * stride;
  double* w = a.vec + (size_t)V_W * stride;
  double* wtry = a.vec + (size_t)V_WTRY * stride;
  double* wbest = a.vec + (size_t)V_WBEST * stride;
  const double* gnew = a.vec + (size_t)V_GNEW * stride;
  double* S = a.vec + (size_t)V_HIST * stride;
  double* Y = S + (size_t)cap * stride;
  const double dg = dc.delta[2 * hl];
  double red3[5] = {0.0, 0.0, 0.0, 0.0, 0.0}; // g.p | max |change since the last evaluation|, |distance from wref|, wref_s, wref_t
  constexpr int NC = LB_COMB_SLOTS, U = LB_COMB_U;
  const int LB_STEP_R = LB_STEP_OF(r);
  for (int i0 = LB_FIRST(r); i0 < M; i0 += U * LB_STEP_R) {
    double gi[U], wi[U], we[U], sn[U], yn[U], acc[U];
    float w32_old[U], wref[U], wref_s[U], wref_t[U];
    int idx[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = i0 + u * LB_STEP_R;
      idx[u] = i < M ? i : i0;                    // past the end: a duplicate of the first element, never stored
      const int ii = idx[u];
      we[u] = ta.improved ? ta.w_eval[ii] : 0.0;
      w32_old[u] = a.w32[ii]; wref[u] = a.wref[ii]; wref_s[u] = a.wref_s[ii]; wref_t[u] = a.wref_t[ii];
      if (pu.on) {
        const double gn = gnew[ii];
        sn[u] = __dmul_rn(pu.alpha_old, p[ii]); yn[u] = __dsub_rn(gn, g[ii]);
        gi[u] = gn; wi[u] = wtry[ii];
      } else {
        sn[u] = 0.0; yn[u] = 0.0;
        gi[u] = g[ii]; wi[u] = w[ii];
      }
      acc[u] = dg * gi[u];
    }
    for (int t0 = 0; t0 < hl; t0 += NC) {
      double sv[U][NC], yv[U][NC];
#pragma unroll
      for (int q = 0; q < NC; ++q) {
        const int sl = dc.slot_of[t0 + q < hl ? t0 + q : t0];     // past the end: a duplicate
        const size_t off = (size_t)sl * stride;
        const bool is_new = pu.on && sl == pu.slot;
#pragma unroll
        for (int u = 0; u < U; ++u) {
          sv[u][q] = S[off + idx[u]]; yv[u][q] = Y[off + idx[u]];
          if (is_new) { sv[u][q] = sn[u]; yv[u][q] = yn[u]; }     // (what the slot holds in memory is the evicted pair)
        }
      }
#pragma unroll
      for (int q = 0; q < NC; ++q) {
        if (t0 + q < hl) {
          const double ds = dc.delta[t0 + q], dy = dc.delta[hl + t0 + q];
#pragma unroll
          for (int u = 0; u < U; ++u) acc[u] = __dadd_rn(acc[u], __fma_rn(dy, yv[u][q], __dmul_rn(ds, sv[u][q])));
        }
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = i0 + u * LB_STEP_R;
      if (i < M) {
        if (pu.on) {
          S[(size_t)pu.slot * stride + i] = sn[u]; Y[(size_t)pu.slot * stride + i] = yn[u];
          w[i] = wi[u]; g[i] = gi[u];
        }
        const double pi = -acc[u];
        p[i] = pi;
        red3[0] += gi[u] * pi;
        if (ta.improved) wbest[i] = we[u];
        const double wt = __dadd_rn(wi[u], __dmul_rn(ta.alpha, pi));
        wtry[i] = wt;
        const float wn = (float)wt;
        red3[1] = fmax(red3[1], fabs((double)wn - (double)w32_old[u]));      // differences of floats: exact in fp64
        red3[2] = fmax(red3[2], fabs((double)wn - (double)wref[u]));
        red3[3] = fmax(red3[3], fabs((double)wn - (double)wref_s[u]));
        red3[4] = fmax(red3[4], fabs((double)wn - (double)wref_t[u]));
        a.w32[i] = wn;
        if (a.rec_nw) { a.rec_nw[(size_t)i * a.rec_stride] = -wn; a.count_zero[i] = 0u; }
      }
    }
  }
  cluster_all_mixed<5, 4>(red3, r);
  *gp_out = red3[0]; mx_out[0] = red3[1]; mx_out[1] = red3[2]; mx_out[2] = red3[3]; mx_out[3] = red3[4];
}

__global__ void solve_init_kernel(StepArgs a, const float* w_init, int hist_cap, int max_iters, int max_evals,
                                  double eps, double gamma0, double domain_volume) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < a.M) {
    const double w = w_init ? (double)w_init[i] : 0.0;     // Alg. 2 step 2: W0 = 0
    a.vec[(size_t)V_W * a.stride + i] = w;
    a.w32[i] = (float)w;
    a.wref[i] = (float)w;
    a.wref_s[i] = (float)w;
    a.wref_t[i] = (float)w;
  }
  if (i == 0) {
    SolveState* st = a.st;
    st->cull_rebuild = 1; st->cull_rebuilds = 1; st->cull_delta = 0.0f; st->cull_cap = 0.0f;
    st->cull_rebuild_s = 1; st->cull_rebuilds_s = 1; st->cull_delta_s = 0.0f;
    st->cull_rebuild_t = 1; st->cull_rebuilds_t = 1; st->cull_delta_t = 0.0f;
    st->done = 0; st->phase = 0; st->iters = 0; st->evals = 0; st->trial = 0;
    st->hist_len = 0; st->hist_start = 0; st->hist_cap = hist_cap;
    st->max_iters = max_iters; st->max_evals = max_evals;
    st->f = 0.0; st->gp = 0.0; st->alpha = 1.0; st->lo = 0.0; st->hi = INFINITY;
    st->gamma = gamma0; st->eps = eps; st->best_err = INFINITY; st->best_dual = 0.0;
    st->domain_volume = domain_volume;
    a.report->done = 0; a.report->status = APD_OK; a.report->iters = 0; a.report->evals = 0;
    a.report->err = 0.0; a.report->dual = 0.0; a.report->cull_rebuilds = 0; a.report->cull_rebuilds_s = 0;
  }
}

// Runs after every evaluation, as one cluster of 8 or 16 CTAs.  Control flow is uniform over the cluster: every
// decision is taken on values all threads hold identically (cluster reductions, state scalars read at entry).
// Only CTA 0 writes the state scalars, the history trace and the host report.
__global__ void __launch_bounds__(LB_THREADS) lbfgs_step_kernel(StepArgs a) {
  __shared__ double s_wbuf[(LB_THREADS / 32) * LB_NRED];
  __shared__ double s_cbuf[2 * LB_NRED];
  __shared__ double s_tot[LB_NRED];
  __shared__ double s_smin;
  __shared__ double s_prod[LB_NPROD];      // the sweep's Gram products and scalars (cluster totals)
  __shared__ double s_scal[LB_NSCAL];
  extern __shared__ double s_dyn[];        // GramSmem: Gram matrix, rho, coefficient vectors (sized by the launch)
  cg::cluster_group cluster = cg::this_cluster();
  Reducer red{s_wbuf, s_cbuf, s_tot, 0, cluster.block_rank(), cluster.num_blocks()};
  const int LB_STEP_R = LB_STEP_OF(red);
  SolveState* st = a.st;
  pdl_enter();
  if (st->done) return;                    // uniform: written by the previous launch
  const bool lead = red.rank == 0;
  const int M = a.M, stride = a.stride, tid = threadIdx.x;
  double* w = a.vec + (size_t)V_W * stride;
  double* g = a.vec + (size_t)V_G * stride;
  double* p = a.vec + (size_t)V_P * stride;
  double* wtry = a.vec + (size_t)V_WTRY * stride;
  double* wbest = a.vec + (size_t)V_WBEST * stride;
  double* gnew = a.vec + (size_t)V_GNEW * stride;

  // copy the scalars (the state is rewritten only at the very end, after several cluster barriers)
  const int phase = st->phase;
  int iters = st->iters, evals = st->evals, trial = st->trial, hist_len = st->hist_len, hist_start = st->hist_start;
  const int cap = st->hist_cap, max_iters = st->max_iters, max_evals = st->max_evals;
  double f = st->f, gp = st->gp, alpha = st->alpha, lo = st->lo, hi = st->hi, gamma = st->gamma;
  const double eps = st->eps, domain_volume = st->domain_volume;
  double best_err = st->best_err, best_dual = st->best_dual;
  float cull_cap = st->cull_cap;
  const float cull_delta_old = st->cull_delta, cull_delta_s_old = st->cull_delta_s, cull_delta_t_old = st->cull_delta_t;
  const int cull_rebuilds_old = st->cull_rebuilds, cull_rebuilds_s_old = st->cull_rebuilds_s, cull_rebuilds_t_old = st->cull_rebuilds_t;

  // the Gram matrix of the history: fetched now, stored to shared memory after the layer sums (whose loads hide the
  // latency), patched and used after the decision
  const GramSmem G = gram_smem(a, cap, red.rank, s_dyn);
  const int hl_old = hist_len, hs_old = hist_start;        // the ring as the sweep sees it (before a push)
  const bool gram = phase != 0 && hl_old > 0;
  constexpr int GPRE = 2;
  const int gram_words = G.ld * G.ld + cap;
  double gpre[GPRE] = {0.0, 0.0};
  if (gram && gram_words <= GPRE * LB_THREADS) {
#pragma unroll
    for (int k = 0; k < GPRE; ++k) if (tid + k * LB_THREADS < gram_words) gpre[k] = G.glob[tid + k * LB_THREADS];
  }

  // a9 for the loop: g~ = <v, fl32 w> + |P| sum_j min_i C_ij (identity I1), eq. (2.5) error
  const double P = a.voxel_volume;
  // sum of the minima, two-level (apd_internal.cuh): layer sums by one warp each, in a fixed order (the sweep's
  // cluster barrier publishes them to every CTA) ...
  if (!a.layer_in) {
    for (int L = (int)red.rank * (LB_THREADS / 32) + (tid >> 5); L < a.lm.n_layers; L += (int)red.nranks * (LB_THREADS / 32)) {
      const int first = L * a.lm.per_layer, cnt = min(a.lm.per_layer, a.lm.n_partials - first);
      const double ls = warp_ordered_sum(a.dual_partial + first, cnt);
      if ((tid & 31) == 0) a.layer_buf[L] = ls;
    }
  }
  if (gram) {
    if (gram_words <= GPRE * LB_THREADS) {
#pragma unroll
      for (int k = 0; k < GPRE; ++k) if (tid + k * LB_THREADS < gram_words) G.m[tid + k * LB_THREADS] = gpre[k];
    } else {
      for (int e = tid; e < gram_words; e += LB_THREADS) G.m[e] = G.glob[e];
    }
  }
  if (gram) eval_sweep<true>(a, phase, alpha, cap, hl_old, hs_old, red);
  else      eval_sweep<false>(a, phase, alpha, cap, hl_old, hs_old, red);
  // the totals sit in red.tot until the next exchange: keep the products and the scalars in shared memory of their
  // own, where the write-back can index them with run-time slot numbers
  if (gram && tid < LB_NPROD) s_prod[tid] = red.tot[tid];
  if (tid < LB_NSCAL) s_scal[tid] = gram ? red.tot[LB_NPROD_PAD + tid] : red.tot[tid];
  // ... then the layers in ascending order: the same bits in every CTA, and in a slab-sharded solve
  {
    const double* lsrc = a.layer_in ? a.layer_in : a.layer_buf;
    if (tid < 32) {
      // ascending-order sum with the loads in flight together: 32 layers per round, one per lane, then the lanes' values
      // are added in lane order (a serial loop of dependent loads cost ~0.3 us per layer)
      double t = 0.0;
      for (int L0 = 0; L0 < a.lm.n_layers; L0 += 32) {
        const double mine = (L0 + tid < a.lm.n_layers) ? __ldcg(lsrc + L0 + tid) : 0.0;
        const int cnt = min(32, a.lm.n_layers - L0);
        for (int l = 0; l < cnt; ++l) t += __shfl_sync(0xffffffffu, mine, l);
      }
      if (tid == 0) s_smin = t;
    }
    __syncthreads();
  }
  const double smin = s_smin;
  const double err1 = s_scal[SC_ERR];
  const double dual1 = s_scal[SC_VW] + P * smin, f1 = -dual1;

  evals += 1;
  if (lead && tid == 0 && evals <= a.hist_cap) { a.hist[2 * (evals - 1)] = -f1; a.hist[2 * (evals - 1) + 1] = err1; }
  const double* w_eval = (phase == 0) ? w : wtry;
  const bool improved = err1 < best_err;      // the best-so-far copy is made in the last sweep of this call
  if (improved) { best_err = err1; best_dual = -f1; }
  const double vsum = s_scal[SC_V], g1p = s_scal[SC_G1P], sy = s_scal[SC_SY], ss = s_scal[SC_SS], yy = s_scal[SC_YY];

  int finish = 0;          // 1: OK at w_eval, 2: NOT_CONVERGED at best, 3: bad target volumes
  bool need_direction = false;
  double mx[4] = {0.0, 0.0, 0.0, 0.0};   // max |change of fl32 w since the last evaluation|, |distance from wref|, wref_s, wref_t
  int new_slot = -1;       // ring slot a curvature pair is pushed into by this call, else -1
  bool evicts = false;     // ... and that slot held the oldest pair (the ring was full)
  bool accepted = false;
  const double alpha_eval = alpha;     // the step length the evaluation just run was taken with
  if (phase == 0) {
    // cost scale for the list-reuse slack: mean over the voxels of min_i C_ij = (g~ - <v, w>) / |Omega|  (identity I1)
    const double scale = fabs(P * smin) / domain_volume;
    cull_cap = isfinite(scale) ? (float)(CULL_CAP_FACTOR * scale) : 0.0f;
    // target volumes: v_i > 0 and sum v_i = |Omega| -- with sum v != |Omega| the dual
    // is unbounded along (1,..,1); fp32 inputs normalised in fp64 meet 1e-6 with two orders to spare
    double badv = 0.0;
    for (int i = LB_FIRST(red); i < M; i += LB_STEP_R) if (!((double)a.v[i] > 0.0)) badv = 1.0;
    badv = cluster_allmax(badv, red);
    if (badv != 0.0 || !(fabs(vsum - domain_volume) <= 1e-6 * domain_volume)) finish = 3;
    else if (err1 <= eps) finish = 1;
    else {
      f = f1;
      for (int i = LB_FIRST(red); i < M; i += LB_STEP_R) g[i] = gnew[i];
      need_direction = true;
    }
  } else {
    if (err1 <= eps) { finish = 1; iters += 1; }
    else {
      const double armijo_rhs = __dadd_rn(f, __dmul_rn(__dmul_rn(1e-4, alpha), gp));
      if (f1 > armijo_rhs) hi = alpha;
      else if (g1p < __dmul_rn(0.9, gp)) lo = alpha;
      else accepted = true;
      if (!accepted) {
        if (evals >= max_evals) finish = 2;
        else {
          alpha = isfinite(hi) ? __dmul_rn(0.5, __dadd_rn(lo, hi)) : __dmul_rn(2.0, alpha);
          trial += 1;
          if (trial >= LB_MAX_TRIALS) {
            if (hist_len > 0) { hist_len = 0; hist_start = 0; need_direction = true; }   // retry with p = -gamma g
            else finish = 2;
          }
        }
      } else {
        // s = alpha p, yv = g1 - g  -> curvature pair in the next ring slot; when the ring is full that slot is
        // the oldest pair, which is dropped only if the new one is kept
        const int slot = (hist_len < cap) ? (hist_start + hist_len) % cap : hist_start;
        const bool keep = sy > 1e-12 * sqrt(ss) * sqrt(yy);
        f = f1;
        iters += 1;
        if (iters >= max_iters || evals >= max_evals) finish = 2;
        else need_direction = true;
        if (keep && need_direction) {
          // the pair's vectors, w <- w_try and g <- g1 are written by the combination pass below
          if (tid == 0) { const double rh = 1.0 / sy; G.rho[slot] = rh; G.glob[(size_t)G.ld * G.ld + slot] = rh; }
          new_slot = slot;
          evicts = !(hist_len < cap);
          if (hist_len < cap) hist_len += 1; else hist_start = (hist_start + 1) % cap;
          gamma = sy / yy;
        } else {
          // (pair not kept, or the limits end the solve here: no history update is needed any more)
          for (int i = LB_FIRST(red); i < M; i += LB_STEP_R) { w[i] = wtry[i]; g[i] = gnew[i]; }
        }
      }
    }
  }

  if (need_direction) {
    if (hist_len > 0) {
      // refresh the Gram rows that changed -- those of the pushed pair (if any) and the row of the new gradient --
      // from the products the sweep formed against the ring as it was
      gram_writeback(G, cap, s_prod, hs_old, 0, min(LB_GRAM_SLOTS, hl_old), new_slot, evicts);
      for (int t0 = LB_GRAM_SLOTS; t0 < hl_old; t0 += LB_GRAM_SLOTS) {      // histories longer than one pass
        const int ns = min(LB_GRAM_SLOTS, hl_old - t0);
        gram_products(a, alpha_eval, cap, hs_old, t0, ns, red);
        gram_writeback(G, cap, red.tot, hs_old, t0, ns, new_slot, evicts);
      }
      if (tid == 0) {
        const int gq = 2 * cap;
        G.set(gq, gq, s_scal[SC_G1G1]);
        if (new_slot >= 0) {
          const int sq = new_slot, yq = cap + new_slot;
          G.set(sq, sq, ss); G.set(yq, yq, yy); G.set_sym(sq, yq, sy);
          G.set_sym(gq, sq, s_scal[SC_G1S]); G.set_sym(gq, yq, s_scal[SC_G1Y]);
        }
      }
      __syncthreads();      // the patches are visible to the warp that runs the recursion
    }
    // the new direction and, in the same pass, the first trial point along it (alpha = 1)
    alpha = 1.0; lo = 0.0; hi = INFINITY; trial = 0;
    DirCoef dc = direction_coeffs(G, cap, hist_len, hist_start, gamma);
    combine_and_trial(a, cap, dc, TrialArgs{improved, w_eval, alpha}, PushArgs{new_slot >= 0, alpha_eval, new_slot}, red,
                      &gp, mx);
    if (gp >= 0.0) {    // safeguard: not a descent direction -> steepest descent scaled by gamma
      hist_len = 0; hist_start = 0;
      const double mx0 = mx[0];
      dc = direction_coeffs(G, cap, 0, 0, gamma);
      combine_and_trial(a, cap, dc, TrialArgs{false, w_eval, alpha}, PushArgs{false, 0.0, -1}, red, &gp, mx);
      mx[0] += mx0;     // w32 was rewritten by the first pass: |change since the last evaluation| <= the sum (it only
                        // sizes the slack of a rebuilt candidate list; any value is exact)
    }
  }

  int cull_rebuild = 1, cull_rebuild_s = 1, cull_rebuild_t = 1;
  float cull_delta = 0.0f, cull_delta_s = 0.0f, cull_delta_t = 0.0f;
  if (finish == 0) {
    if (!need_direction) {
      // next trial point w + alpha p of the line search, rounded to fp32 for the evaluation (S10)
      for (int i = LB_FIRST(red); i < M; i += LB_STEP_R) {
        if (improved) wbest[i] = w_eval[i];      // best-so-far copy of the point just evaluated (before wtry is rewritten)
        const double wt = __dadd_rn(w[i], __dmul_rn(alpha, p[i]));
        wtry[i] = wt;
        const float wn = (float)wt;
        mx[0] = fmax(mx[0], fabs((double)wn - (double)a.w32[i]));     // differences of floats: exact in fp64
        mx[1] = fmax(mx[1], fabs((double)wn - (double)a.wref[i]));
        mx[2] = fmax(mx[2], fabs((double)wn - (double)a.wref_s[i]));
        mx[3] = fmax(mx[3], fabs((double)wn - (double)a.wref_t[i]));
        a.w32[i] = wn;
        if (a.rec_nw) { a.rec_nw[(size_t)i * a.rec_stride] = -wn; a.count_zero[i] = 0u; }
      }
      cluster_all<4, true>(mx, red);
    }
    cull_delta = cull_delta_old; cull_delta_s = cull_delta_s_old; cull_delta_t = cull_delta_t_old;
    cull_rebuild = !(mx[1] <= (double)cull_delta);
    cull_rebuild_s = 0; cull_rebuild_t = 0;
    if (cull_rebuild) {
      // the next evaluation rebuilds its brick lists at the new weights, valid within delta of them; they are cut from
      // the CTA-tile lists, which must hold on that whole ball: (distance from wref_t) + delta <= delta_t, else those
      // are rebuilt too, with a slack CULL_TILE_FACTOR times as large, from the super-tile lists, which must hold on
      // THAT ball, else ... (sums of floats: exact in fp64)
      cull_delta = fminf((float)(CULL_DELTA_FACTOR * mx[0]), cull_cap);
      cull_rebuild_t = !(mx[3] + (double)cull_delta <= (double)cull_delta_t);
      if (cull_rebuild_t) {
        cull_delta_t = (float)(CULL_TILE_FACTOR * (double)cull_delta);
        cull_rebuild_s = !(mx[2] + (double)cull_delta_t <= (double)cull_delta_s);
        if (cull_rebuild_s) cull_delta_s = (float)(CULL_SUPER_FACTOR * (double)cull_delta);
      }
      for (int i = LB_FIRST(red); i < M; i += LB_STEP_R) {
        const float wn = a.w32[i];
        a.wref[i] = wn;
        if (cull_rebuild_t) a.wref_t[i] = wn;
        if (cull_rebuild_s) a.wref_s[i] = wn;
      }
    }
  } else if (finish == 1) {
    if (phase != 0) for (int i = LB_FIRST(red); i < M; i += LB_STEP_R) w[i] = wtry[i];
  } else if (finish == 2) {
    for (int i = LB_FIRST(red); i < M; i += LB_STEP_R) {
      const double wb = improved ? w_eval[i] : wbest[i];
      wbest[i] = wb; w[i] = wb; a.w32[i] = (float)wb;
    }
  }
  cluster.sync();        // no CTA leaves while its shared memory may still be read; all vector writes are done
  if (lead && tid == 0) {
    st->phase = 1; st->iters = iters; st->evals = evals; st->trial = trial;
    st->hist_len = hist_len; st->hist_start = hist_start;
    st->f = f; st->gp = gp; st->alpha = alpha; st->lo = lo; st->hi = hi; st->gamma = gamma;
    st->best_err = best_err; st->best_dual = best_dual;
    st->cull_cap = cull_cap; st->cull_rebuild = cull_rebuild; st->cull_delta = cull_delta;
    st->cull_rebuild_s = cull_rebuild_s; st->cull_delta_s = cull_delta_s;
    st->cull_rebuild_t = cull_rebuild_t; st->cull_delta_t = cull_delta_t;
    st->cull_rebuilds_t = cull_rebuilds_t_old + (finish == 0 && cull_rebuild_t);
    st->cull_rebuilds = cull_rebuilds_old + (finish == 0 && cull_rebuild);
    st->cull_rebuilds_s = cull_rebuilds_s_old + (finish == 0 && cull_rebuild_s);
    if (finish) {
      st->done = 1;
      a.report->status = (finish == 1) ? APD_OK : (finish == 2 ? APD_NOT_CONVERGED : APD_E_ARG);
      a.report->iters = iters; a.report->evals = evals;
      a.report->err = (finish == 2) ? best_err : err1;
      a.report->dual = (finish == 2) ? best_dual : -f1;
      a.report->cull_rebuilds = st->cull_rebuilds; a.report->cull_rebuilds_s = st->cull_rebuilds_s; a.report->cull_rebuilds_t = st->cull_rebuilds_t;
      __threadfence_system();
      a.report->done = 1;
      __threadfence_system();
    }
  }
}

}  // namespace apd

using namespace apd;

#define LB_TRY(call)                                                                \
  do {                                                                              \
    cudaError_t e__ = (call);                                                       \
    if (e__ != cudaSuccess) {                                                       \
      ctx->err = std::string(#call) + ": " + cudaGetErrorString(e__);               \
      return APD_E_CUDA;                                                            \
    }                                                                               \
  } while (0)

int apd::ensure_solve_state(apd_ctx* ctx, int hist) {
  Workspace& ws = ctx->ws;
  const size_t ms = (size_t)ws.max_seeds;
  if (!ws.sstate) {
    LB_TRY(cudaMalloc(&ws.sstate, sizeof(SolveState)));
    LB_TRY(cudaMalloc(&ws.w32, ms * sizeof(float)));
    LB_TRY(cudaMalloc(&ws.wref, ms * sizeof(float)));
    LB_TRY(cudaMalloc(&ws.wref_s, ms * sizeof(float)));
    LB_TRY(cudaMalloc(&ws.wref_t, ms * sizeof(float)));
    LB_TRY(cudaMalloc(&ws.e_vol, ms * sizeof(double)));
    LB_TRY(cudaMalloc(&ws.e_scal, 2 * sizeof(double)));
    LB_TRY(cudaMalloc(&ws.hist, 2 * (size_t)SOLVE_HIST_CAP * sizeof(double)));
    LB_TRY(cudaHostAlloc(&ws.report, sizeof(SolveReport), cudaHostAllocMapped));
    LB_TRY(cudaEventCreateWithFlags(&ws.sev[0], cudaEventDisableTiming));
    LB_TRY(cudaEventCreateWithFlags(&ws.sev[1], cudaEventDisableTiming));
  }
  if (!ws.svec || ws.svec_hist < hist) {
    if (ws.svec) { LB_TRY(cudaDeviceSynchronize()); LB_TRY(cudaFree(ws.svec)); ws.svec = nullptr; }
    LB_TRY(cudaMalloc(&ws.svec, (size_t)(V_HIST + 2 * hist) * ms * sizeof(double)));
    cudaFree(ws.gram); ws.gram = nullptr;
    LB_TRY(cudaMalloc(&ws.gram, (size_t)LB_CLUSTER_MAX * ((size_t)(2 * hist + 1) * (2 * hist + 1) + hist) * sizeof(double)));
    ws.svec_hist = hist;
  }
  return APD_OK;
}

// The step kernel's cluster size on this context's device: LB_CLUSTER_MAX if the device can hold one such cluster of
// lbfgs_step_kernel (a non-portable size, opted into here), else LB_CLUSTER_PORTABLE.
static int lb_cluster_size(apd_ctx* ctx, size_t dyn_bytes, int* out) {
  *out = LB_CLUSTER_PORTABLE;
  if (cudaFuncSetAttribute(lbfgs_step_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
    cudaGetLastError();
    return APD_OK;
  }
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = LB_CLUSTER_MAX; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(LB_CLUSTER_MAX); cfg.blockDim = dim3(LB_THREADS); cfg.dynamicSmemBytes = dyn_bytes;
  cfg.attrs = attr; cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, lbfgs_step_kernel, &cfg) == cudaSuccess && n >= 1) *out = LB_CLUSTER_MAX;
  else cudaGetLastError();
  (void)ctx;
  return APD_OK;
}

// The device-driven optimiser loop shared by apd_solve (voxel grids) and apd_solve_points (user points).
//   loop_eval(done_flag): enqueue one evaluation at ws.w32 that leaves its RAW outputs where `sa` points
//   final_eval():         enqueue the final, labelled evaluation at ws.w32
struct SolveHooks {
  std::function<int(const int*)> loop_eval;
  std::function<int()> final_eval;
};

static int solve_common(apd_ctx* ctx, const char* who, int dim, int32_t M, const float* target_vol, double tol,
                        const float* w_init, float* w, double* w64, const apd_opts& o, double domain, StepArgs sa,
                        const SolveHooks& hooks, int32_t* iters, int32_t* evals, double* max_rel_err, double* dual,
                        cudaStream_t st) {
  Workspace& ws = ctx->ws;
  const int max_evals = o.max_evals ? o.max_evals : (o.max_iters > (1 << 26) ? (1 << 30) : 20 * o.max_iters);
  const double ell = std::pow(domain / (double)M, 1.0 / (double)dim);
  const double gamma0 = std::pow(ell, (double)(2 - dim)) / (double)dim;
  sa.st = ws.sstate; sa.vec = ws.svec; sa.stride = ws.max_seeds; sa.M = M; sa.v = target_vol; sa.w32 = ws.w32;
  sa.hist = ws.hist; sa.hist_cap = SOLVE_HIST_CAP; sa.wref = ws.wref; sa.wref_s = ws.wref_s; sa.wref_t = ws.wref_t; sa.gram = ws.gram;
  ws.hist_len = 0;
  SolveReport* dev_report = nullptr;
  LB_TRY(cudaHostGetDevicePointer((void**)&dev_report, ws.report, 0));
  sa.report = dev_report;
  ws.report->done = 0;
  solve_init_kernel<<<(M + 255) / 256, 256, 0, st>>>(sa, w_init, o.lbfgs_history, o.max_iters, max_evals, tol,
                                                    gamma0, domain);
  LB_TRY(cudaGetLastError());

  // dynamic shared memory of the step kernel: Gram matrix, rho and the coefficient vectors (GramSmem)
  const size_t nb = 2 * (size_t)o.lbfgs_history + 1;
  const size_t dyn_bytes = (nb * nb + nb + 2 * (size_t)o.lbfgs_history) * sizeof(double) + (size_t)o.lbfgs_history * sizeof(int);
  if (dyn_bytes > 32 * 1024)
    LB_TRY(cudaFuncSetAttribute(lbfgs_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_bytes));
  if (ws.lb_cluster == 0) {
    const int rc = lb_cluster_size(ctx, dyn_bytes, &ws.lb_cluster);
    if (rc != APD_OK) return rc;
  }
  cudaLaunchAttribute step_attr[2];
  step_attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;     // apd_device.cuh: pdl_enter
  step_attr[1].val.programmaticStreamSerializationAllowed = 1;
  step_attr[0].id = cudaLaunchAttributeClusterDimension;
  const unsigned n_cta = (ws.lb_cluster == LB_CLUSTER_MAX && M >= LB_CLUSTER_MAX_MIN_M) ? LB_CLUSTER_MAX : LB_CLUSTER_PORTABLE;
  step_attr[0].val.clusterDim.x = n_cta; step_attr[0].val.clusterDim.y = 1; step_attr[0].val.clusterDim.z = 1;
  cudaLaunchConfig_t step_cfg = {};
  step_cfg.gridDim = dim3(n_cta); step_cfg.blockDim = dim3(LB_THREADS);
  step_cfg.dynamicSmemBytes = dyn_bytes; step_cfg.stream = st; step_cfg.attrs = step_attr; step_cfg.numAttrs = 2;
  const int* done_flag = &ws.sstate->done;
  long long enq = 0;
  const long long hard_cap = (long long)max_evals + 64;
  for (;; ++enq) {
    int rc = hooks.loop_eval(done_flag);
    if (rc != APD_OK) return rc;
    if (!sa.layer_in) { sa.dual_partial = ws.dual_partial; sa.layer_buf = ws.layer_buf; }   // (re)allocated by the first evaluation
    LB_TRY(cudaLaunchKernelEx(&step_cfg, lbfgs_step_kernel, sa));
    LB_TRY(cudaEventRecord(ws.sev[enq & 1], st));
    if (enq >= 1) {
      // the convergence check: wait for the PREVIOUS evaluation's step while this one runs;
      // kernels enqueued after the optimiser finished see done_flag and return at once
      LB_TRY(cudaEventSynchronize(ws.sev[(enq - 1) & 1]));
      if (ws.report->done) break;
    }
    if (enq > hard_cap) { ctx->err = std::string(who) + ": optimiser did not report completion"; return APD_E_CUDA; }
  }
  LB_TRY(cudaStreamSynchronize(st));
  const int status = ws.report->status;
  if (status == APD_E_ARG) {
    ctx->err = std::string(who) + ": target_vol must be > 0 and sum to |Omega| within 1e-6 relative";
    return APD_E_ARG;
  }
  // final evaluation at the returned fp32 weights, with labels (Algorithm 1 at the solution)
  int rc = hooks.final_eval();
  if (rc != APD_OK) return rc;
  LB_TRY(cudaMemcpyAsync(w, ws.w32, sizeof(float) * M, cudaMemcpyDeviceToDevice, st));
  if (w64) LB_TRY(cudaMemcpyAsync(w64, ws.svec + (size_t)V_W * ws.max_seeds, sizeof(double) * M,
                                  cudaMemcpyDeviceToDevice, st));
  LB_TRY(cudaStreamSynchronize(st));
  ws.hist_len = ws.report->evals < SOLVE_HIST_CAP ? ws.report->evals : SOLVE_HIST_CAP;
  ws.last_rebuilds = o.cull ? ws.report->cull_rebuilds : 0;
  if (iters) *iters = ws.report->iters;
  if (evals) *evals = ws.report->evals;
  if (max_rel_err) *max_rel_err = ws.report->err;
  if (dual) *dual = ws.report->dual;
  return status;
}

static int check_solve_opts(apd_ctx* ctx, const char* who, const apd_opts* opts, double tol, apd_opts* o) {
  apd_default_opts(o);
  if (opts) *o = *opts;
  if (!(tol > 0.0) || !std::isfinite(tol)) { ctx->err = std::string(who) + ": tol must be finite and > 0"; return APD_E_ARG; }
  if (o->lbfgs_history < 1 || o->lbfgs_history > LB_MAX_HIST) { ctx->err = std::string(who) + ": lbfgs_history must be in [1,64]"; return APD_E_ARG; }
  if (o->max_iters < 1 || o->max_evals < 0) { ctx->err = std::string(who) + ": max_iters >= 1 and max_evals >= 0 required"; return APD_E_ARG; }
  return APD_OK;
}

// Algorithm 2 on a grid or on one slab of it (f4).  slab == nullptr: the whole grid, no exchange.  With a slab every
// evaluation leaves its raw counters in `counters` (apd_shard.cu: pack_counters) and reduce(user, stream) sums them over
// the ranks before the optimiser step, which then reads the REDUCED block: identical inputs on every rank.
int apd::solve_grid(apd_ctx* ctx, const char* who, const apd_grid* grid, const apd_slab* slab, int32_t M, const float* X,
                    const float* A, const float* target_vol, double tol, const float* w_init, float* w, int32_t* labels,
                    double* vol, double* w64, uint64_t* counters, apd_reduce_fn reduce, void* user, int32_t* iters,
                    int32_t* evals, double* max_rel_err, double* dual, const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  const std::string pre = std::string(who) + ": ";
  std::string e;
  bool cull = false;
  const int kernel = resolve_kernel(ctx, opts, grid, M, &cull, &e);
  if (kernel < 0) { ctx->err = pre + e; return APD_E_ARG; }
  if (M < 1 || M > ctx->ws.max_seeds) { ctx->err = pre + "M out of range [1, max_seeds]"; return APD_E_ARG; }
  if (!X || !A || !target_vol || !w) { ctx->err = pre + "X, A, target_vol and w are required"; return APD_E_ARG; }
  if (slab && !counters) { ctx->err = pre + "counters is required"; return APD_E_ARG; }
  apd_opts o;
  int rc = check_solve_opts(ctx, who, opts, tol, &o);
  if (rc != APD_OK) return rc;
  o.cull = cull ? 1 : 0;
  GridDev g, gfull;
  e = make_grid(ctx, grid, kernel, o.cull != 0, &g, slab);
  if (!e.empty()) { ctx->err = pre + e; return APD_E_ARG; }
  e = make_grid(ctx, grid, kernel, o.cull != 0, &gfull, nullptr);
  if (!e.empty()) { ctx->err = pre + e; return APD_E_ARG; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  LB_TRY(cudaSetDevice(ctx->ws.device));
  rc = ensure_solve_state(ctx, o.lbfgs_history);
  if (rc != APD_OK) return rc;
  Workspace& ws = ctx->ws;
  double domain = 1.0;
  for (int k = 0; k < g.dim; ++k) domain *= (grid->hi[k] - grid->lo[k]);
  const LayerMap lm = layer_map(g, o.cull != 0);
  const int n_layers_full = layer_map(gfull, o.cull != 0).n_layers;
  StepArgs sa;
  sa.count = ws.count; sa.count64 = nullptr; sa.vol_in = nullptr; sa.voxel_volume = g.voxel_volume;
  sa.lm = lm; sa.dual_partial = nullptr; sa.layer_buf = nullptr; sa.layer_in = nullptr;
  if (slab) {
    sa.count = nullptr; sa.count64 = reinterpret_cast<const unsigned long long*>(counters);
    sa.layer_in = reinterpret_cast<const double*>(counters + M);
    sa.lm.n_layers = n_layers_full;
  }
  auto exchange = [&](bool with_idxsum, const int* done_flag) -> int {
    // this slab's counters -> `counters`, then their sum over the ranks, in stream order
    LB_TRY(launch_pack_counters(g, M, lm, n_layers_full, ws.count, with_idxsum ? ws.idxsum : nullptr, ws.dual_partial,
                                counters, done_flag, st));
    if (reduce && reduce(user, cuda_stream) != 0) { ctx->err = pre + "the reduce callback failed"; return APD_E_CUDA; }
    return APD_OK;
  };
  if (o.cull) {
    // the record table exists before the loop starts: the step kernel writes into it (StepArgs::rec_nw)
    rc = ensure_eval_buffers(ctx, g, kernel, true, st);
    if (rc != APD_OK) return rc;
    sa.rec_nw = ws.rec + (g.dim == 3 ? 9 : 5);
    sa.rec_stride = rec_floats(g.dim);
    sa.count_zero = ws.count;
  }
  int n_loop_evals = 0;
  SolveHooks hooks;
  hooks.loop_eval = [&](const int* done_flag) -> int {
    // after the first evaluation the records' -w and the zeroed counts come from the step kernel: no pack launch
    const bool skip_pack = o.cull != 0 && n_loop_evals > 0;
    ++n_loop_evals;
    int r = enqueue_evaluation(ctx, g, kernel, M, X, A, ws.w32, target_vol, nullptr, nullptr, nullptr, nullptr, nullptr,
                               nullptr, false, o.cull != 0, done_flag, st, &ws.sstate->cull_rebuild,
                               &ws.sstate->cull_delta, &ws.sstate->cull_rebuild_s, &ws.sstate->cull_delta_s,
                               &ws.sstate->cull_rebuild_t, &ws.sstate->cull_delta_t, skip_pack);
    if (r == APD_OK && slab) r = exchange(false, done_flag);
    return r;
  };
  hooks.final_eval = [&]() -> int {
    if (!slab)
      return enqueue_evaluation(ctx, g, kernel, M, X, A, ws.w32, target_vol, labels, vol ? vol : ws.e_vol, ws.e_scal,
                                ws.e_scal + 1, nullptr, nullptr, true, o.cull != 0, nullptr, st);
    int r = enqueue_evaluation(ctx, g, kernel, M, X, A, ws.w32, target_vol, labels, nullptr, nullptr, nullptr, nullptr,
                               nullptr, true, o.cull != 0, nullptr, st);
    if (r == APD_OK) r = exchange(false, nullptr);
    if (r != APD_OK) return r;
    LayerMap lf = lm; lf.n_layers = n_layers_full;
    LB_TRY(launch_finalize(gfull, M, lf, const_cast<double*>(sa.layer_in), nullptr, sa.count64, nullptr, nullptr, X,
                           ws.w32, target_vol, vol ? vol : ws.e_vol, ws.e_scal, ws.e_scal + 1, nullptr, nullptr, nullptr,
                           nullptr, st));
    return APD_OK;
  };
  return solve_common(ctx, who, g.dim, M, target_vol, tol, w_init, w, w64, o, domain, sa, hooks, iters, evals,
                      max_rel_err, dual, st);
}

extern "C" int apd_solve(apd_ctx* ctx, const apd_grid* grid, int32_t M, const float* X, const float* A,
                         const float* target_vol, double tol, const float* w_init, float* w, int32_t* labels,
                         double* vol, double* w64, int32_t* iters, int32_t* evals, double* max_rel_err,
                         double* dual, const apd_opts* opts, void* cuda_stream) {
  return solve_grid(ctx, "apd_solve", grid, nullptr, M, X, A, target_vol, tol, w_init, w, labels, vol, w64, nullptr,
                    nullptr, nullptr, iters, evals, max_rel_err, dual, opts, cuda_stream);
}

// Algorithm 2 on a user-supplied discretisation (points with element volumes, apd_points.cu)
extern "C" int apd_solve_points(apd_ctx* ctx, int64_t N, const float* Y, const float* pvol, double total_volume,
                                int32_t M, const float* X, const float* A, const float* target_vol, double tol,
                                const float* w_init, float* w, int32_t* labels, double* vol, int32_t* iters,
                                int32_t* evals, double* max_rel_err, const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  if (M < 1 || M > ctx->ws.max_seeds) { ctx->err = "apd_solve_points: M out of range [1, max_seeds]"; return APD_E_ARG; }
  if (!Y || !pvol || !X || !A || !target_vol || !w || N < 1) { ctx->err = "apd_solve_points: Y, pvol, X, A, target_vol and w are required"; return APD_E_ARG; }
  if (!(total_volume > 0.0) || !std::isfinite(total_volume)) { ctx->err = "apd_solve_points: total_volume must be the (positive) sum of pvol"; return APD_E_ARG; }
  apd_opts o;
  int rc = check_solve_opts(ctx, "apd_solve_points", opts, tol, &o);
  if (rc != APD_OK) return rc;
  if (o.cull) { ctx->err = "apd_solve_points: opts.cull is not available on point sets"; return APD_E_ARG; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  LB_TRY(cudaSetDevice(ctx->ws.device));
  rc = ensure_solve_state(ctx, o.lbfgs_history);
  if (rc != APD_OK) return rc;
  Workspace& ws = ctx->ws;
  int n_partials = 0;
  SolveHooks hooks;
  hooks.loop_eval = [&](const int* done_flag) {
    return enqueue_points(ctx, N, Y, pvol, M, X, A, ws.w32, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
                          done_flag, &n_partials, st);
  };
  hooks.final_eval = [&]() {
    return enqueue_points(ctx, N, Y, pvol, M, X, A, ws.w32, target_vol, labels, vol ? vol : ws.e_vol, ws.e_scal,
                          ws.e_scal + 1, nullptr, nullptr, &n_partials, st);
  };
  // the first evaluation allocates the accumulators: run the sizing part now so that StepArgs can point at them
  rc = points_prepare(ctx, N, &n_partials, st);
  if (rc != APD_OK) return rc;
  StepArgs sa;
  sa.count = nullptr; sa.count64 = nullptr; sa.vol_in = ws.pt_acc; sa.voxel_volume = 1.0;
  sa.lm = points_layer_map(n_partials); sa.dual_partial = nullptr; sa.layer_buf = nullptr; sa.layer_in = nullptr;
  return solve_common(ctx, "apd_solve_points", ws.dim, M, target_vol, tol, w_init, w, nullptr, o, total_volume, sa,
                      hooks, iters, evals, max_rel_err, nullptr, st);
}

extern "C" int apd_solve_stats(const apd_ctx* ctx, int32_t* evals_recorded, int32_t* cull_rebuilds) {
  if (!ctx) return APD_E_ARG;
  if (evals_recorded) *evals_recorded = ctx->ws.hist_len;
  if (cull_rebuilds) *cull_rebuilds = ctx->ws.last_rebuilds;
  return APD_OK;
}

extern "C" int apd_solve_history(apd_ctx* ctx, double* dual_hist, double* err_hist, int32_t cap) {
  if (!ctx || cap < 0 || (cap > 0 && (!dual_hist || !err_hist))) return APD_E_ARG;
  Workspace& ws = ctx->ws;
  const int n = ws.hist_len < cap ? ws.hist_len : cap;
  if (n <= 0 || !ws.hist) return 0;
  std::vector<double> h(2 * (size_t)n);
  if (cudaSetDevice(ws.device) != cudaSuccess ||
      cudaMemcpy(h.data(), ws.hist, h.size() * sizeof(double), cudaMemcpyDeviceToHost) != cudaSuccess) {
    ctx->err = "apd_solve_history: copy failed";
    return APD_E_CUDA;
  }
  for (int k = 0; k < n; ++k) { dual_hist[k] = h[2 * k]; err_hist[k] = h[2 * k + 1]; }
  return n;
}
