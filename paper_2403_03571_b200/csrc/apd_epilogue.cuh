// apd_epilogue.cuh -- rows a5 + a6 for one thread's row of V voxels, shared by the assign kernels.
#pragma once
#include "apd_internal.cuh"

namespace apd {

// Shared epilogue of every assign kernel (a5 + a6) for one thread's row of V voxels:
// label store, run-length aggregated integer histogram updates, fp64 sum of the min-costs.
template <int V>
__device__ __forceinline__ double row_epilogue(const AssignArgs& a, bool row_valid, int ix0, int iy, int iz,
                                               const float (&best)[V], const int (&lab)[V]) {
  double dsum = 0.0;
  const unsigned vmask = __ballot_sync(0xffffffffu, row_valid);     // (every lane of the warp calls this function)
  if (!row_valid) return dsum;
  const int nvalid = min(V, a.g.nx - ix0);
  if (!a.labels && !a.idxsum && __all_sync(vmask, nvalid == V)) {      // (uniform over the lanes of vmask: they meet again below)
    // The evaluations inside a solve (no label store, no index sums) on a full row: the same sums and the same counts,
    // written without a divergent region per voxel -- the run that ends in front of voxel k is flushed by ONE predicated
    // reduction (the branchy form below cost ~19 instructions per voxel: a quarter of the culled kernel, whose bricks
    // hold only a dozen candidates)
    unsigned int run_cnt = 1u;
    dsum += (double)best[0];
#pragma unroll
    for (int k = 1; k < V; ++k) {
      dsum += (double)best[k];
      asm volatile("{\n.reg .pred p;\nsetp.ne.s32 p, %0, %1;\n@p red.global.add.u32 [%2], %3;\n}\n"
                   :: "r"(lab[k]), "r"(lab[k - 1]), "l"(a.count + lab[k - 1]), "r"(run_cnt) : "memory");
      run_cnt = (lab[k] != lab[k - 1]) ? 1u : run_cnt + 1u;
    }
    const int run_lab = lab[V - 1];
    const unsigned peers = __match_any_sync(vmask, run_lab);
    const unsigned int tot = __reduce_add_sync(peers, run_cnt);
    if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(a.count + run_lab, tot);
    return dsum;
  }
  const long long j0 = ((long long)iz * a.g.ny + iy) * a.g.nx + ix0;
  if (a.labels) {
    if (nvalid == V && (a.g.nx & 3) == 0 && a.labels_vec) {
      int4* p = reinterpret_cast<int4*>(a.labels + j0);      // 16-byte aligned: the base is (labels_vec), and j0 % 4 == 0
                                                             // because nx % 4 == 0 and ix0 % V == 0
#pragma unroll
      for (int k = 0; k < V / 4; ++k) p[k] = make_int4(lab[4 * k], lab[4 * k + 1], lab[4 * k + 2], lab[4 * k + 3]);
    } else {
#pragma unroll
      for (int k = 0; k < V; ++k) if (k < nvalid) a.labels[j0 + k] = lab[k];
    }
  }
  // run-length aggregation: consecutive voxels of a row mostly share their label
  int run_lab = lab[0];
  unsigned int run_cnt = 0;
  unsigned long long run_sx = 0;
#pragma unroll
  for (int k = 0; k < V; ++k) {
    if (k < nvalid) {
      dsum += (double)best[k];
      if (lab[k] != run_lab) {
        atomicAdd(a.count + run_lab, run_cnt);
        if (a.idxsum) {
          atomicAdd(a.idxsum + (size_t)run_lab * 3 + 0, run_sx);
          atomicAdd(a.idxsum + (size_t)run_lab * 3 + 1, (unsigned long long)run_cnt * (iy + a.g.off_y));
          atomicAdd(a.idxsum + (size_t)run_lab * 3 + 2, (unsigned long long)run_cnt * (iz + a.g.off_z));
        }
        run_lab = lab[k]; run_cnt = 0; run_sx = 0;
      }
      run_cnt += 1;
      run_sx += (unsigned long long)(ix0 + k);
    }
  }
  // the last run of every row: the rows of a warp mostly end in the same cell, so the warp adds them up first and
  // sends ONE atomic per distinct label (the counts are integers: exact whatever the grouping)
  {
    const unsigned peers = __match_any_sync(vmask, run_lab);
    const unsigned int tot = __reduce_add_sync(peers, run_cnt);
    if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(a.count + run_lab, tot);
  }
  if (a.idxsum) {
    atomicAdd(a.idxsum + (size_t)run_lab * 3 + 0, run_sx);
    atomicAdd(a.idxsum + (size_t)run_lab * 3 + 1, (unsigned long long)run_cnt * (iy + a.g.off_y));
    atomicAdd(a.idxsum + (size_t)run_lab * 3 + 2, (unsigned long long)run_cnt * (iz + a.g.off_z));
  }
  return dsum;
}

}  // namespace apd
