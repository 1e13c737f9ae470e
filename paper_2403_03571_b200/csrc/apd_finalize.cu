// apd_finalize.cu -- a9: turn the integer histograms and the per-tile partial sums of one
// evaluation into vol (eq. 2.8), the dual g~ (eq. 2.7, via
// identity I1: g~ = sum_i v_i w_i + |P| sum_j min_i C_ij), the stopping quantity of eq. (2.5)
// and the discrete centroids.  One CTA, fixed reduction order:
// the result is bitwise reproducible run to run.
#include "apd_internal.cuh"
#include "apd_device.cuh"

namespace apd {

constexpr int FIN_THREADS = 1024;

__device__ __forceinline__ double block_max_double(double v, double* scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) scratch[wid] = v;
  __syncthreads();
  double t = 0.0;
  if (threadIdx.x == 0)
    for (int i = 0; i < FIN_THREADS / 32; ++i) t = fmax(t, scratch[i]);
  return t;
}

// count64 != nullptr: the counts come as u64 (reduced counter block of a sharded evaluation, apd_shard.cu).
// dual_partial != nullptr: the layer sums of the per-tile partials are formed here (into layer_buf); nullptr: layer_buf
// already holds them (reduced over the slabs).  Either way the dual's sum of minima = the layer sums added in ascending
// layer order -- the same two-level order in every path (apd_internal.cuh).
__global__ void __launch_bounds__(FIN_THREADS) finalize_kernel(
    GridDev g, int M, LayerMap lm, double* __restrict__ layer_buf, const unsigned int* __restrict__ count,
    const unsigned long long* __restrict__ count64, const unsigned long long* __restrict__ idxsum,
    const double* __restrict__ dual_partial, const float* __restrict__ X, const float* __restrict__ w,
    const float* __restrict__ target_vol, double* __restrict__ vol, double* __restrict__ dual,
    double* __restrict__ max_rel_err, double* __restrict__ centroids, uint64_t* __restrict__ pairs_evaluated,
    const unsigned long long* __restrict__ pairs_ctr, const int* __restrict__ done_flag) {
  __shared__ double scratch[FIN_THREADS / 32];
  __shared__ double s_smin;
  if (done_flag && *done_flag) return;
  const int tid = threadIdx.x;
  const double P = g.voxel_volume;
  double vw = 0.0, err = 0.0;
  for (int i = tid; i < M; i += FIN_THREADS) {
    const unsigned long long c = count64 ? count64[i] : (unsigned long long)count[i];
    const double vi = (double)c * P;                       // m_i |P|
    vol[i] = vi;
    if (target_vol) {
      const double tv = (double)target_vol[i];
      vw += tv * (double)w[i];
      err = fmax(err, fabs(vi - tv) / tv);                 // eq. (2.5)
    }
    if (centroids) {
      for (int k = 0; k < g.dim; ++k) {
        double ck;
        if (c > 0) ck = g.lo[k] + g.s[k] * ((double)idxsum[(size_t)i * 3 + k] / (double)c + 0.5);
        else       ck = (double)X[(size_t)i * g.dim + k];  // empty cell keeps its seed (reading S5)
        centroids[(size_t)i * g.dim + k] = ck;
      }
    }
  }
  if (dual_partial) {
    for (int L = tid >> 5; L < lm.n_layers; L += FIN_THREADS / 32) {
      const int first = L * lm.per_layer, cnt = min(lm.per_layer, lm.n_partials - first);
      const double ls = warp_ordered_sum(dual_partial + first, cnt);
      if ((tid & 31) == 0) layer_buf[L] = ls;
    }
  }
  __syncthreads();
  if (tid < 32) {        // ascending-order sum, 32 loads in flight per round (as in lbfgs_step_kernel: the same bits)
    double t = 0.0;
    for (int L0 = 0; L0 < lm.n_layers; L0 += 32) {
      const double mine = (L0 + tid < lm.n_layers) ? layer_buf[L0 + tid] : 0.0;
      const int cnt = min(32, lm.n_layers - L0);
      for (int l = 0; l < cnt; ++l) t += __shfl_sync(0xffffffffu, mine, l);
    }
    if (tid == 0) s_smin = t;
  }

  const double vw_tot = block_sum_double<FIN_THREADS>(vw, scratch);
  __syncthreads();
  const double err_tot = block_max_double(err, scratch);
  if (tid == 0) {
    *dual = vw_tot + P * s_smin;
    if (max_rel_err && target_vol) *max_rel_err = err_tot;
    if (pairs_evaluated)
      *pairs_evaluated = pairs_ctr ? (uint64_t)*pairs_ctr      // culled: what the tiles counted
                                   : (uint64_t)g.nx * (uint64_t)g.ny * (uint64_t)g.nz * (uint64_t)M;
  }
}

cudaError_t launch_finalize(const GridDev& g, int M, LayerMap lm, double* layer_buf, const unsigned int* count,
                            const unsigned long long* count64, const unsigned long long* idxsum,
                            const double* dual_partial, const float* X, const float* w, const float* target_vol,
                            double* vol, double* dual, double* max_rel_err, double* centroids,
                            uint64_t* pairs_evaluated, const unsigned long long* pairs_ctr, const int* done_flag,
                            cudaStream_t st) {
  finalize_kernel<<<1, FIN_THREADS, 0, st>>>(g, M, lm, layer_buf, count, count64, idxsum, dual_partial, X, w, target_vol,
                                             vol, dual, max_rel_err, centroids, pairs_evaluated, pairs_ctr, done_flag);
  return cudaGetLastError();
}

}  // namespace apd
