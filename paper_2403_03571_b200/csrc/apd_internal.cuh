// apd_internal.cuh -- declarations shared by the translation units of libapd_b200 (sm_100a only).
// Nothing here is shared with oracle/: the oracle is an independent fp64 CPU program.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include "../../include/apd.h"

namespace apd {

// Packed seed record: REC floats per seed, 16-byte aligned so a chunk
// of seeds is one contiguous cp.async.bulk (TMA 1-D bulk copy) source.
//   3D (12 floats): x y z a11 | a12' a13' a22 a23' | a33 nw 0 0      a_kl' = A_kl + A_lk
//   2D ( 8 floats): x y a11 a12' | a22 nw 0 0                        nw = -w
// The table is padded to a multiple of SEED_CHUNK with records {0.., nw = +inf} whose cost is
// +inf and therefore never wins the strict '<' argmin.
constexpr int REC3 = 12;
constexpr int REC2 = 8;
constexpr int SEED_CHUNK = 128;                  // seeds per smem stage
constexpr int SEED_STAGES = 2;                   // double buffer

__host__ __device__ constexpr int rec_floats(int dim) { return dim == 3 ? REC3 : REC2; }

// Grid as the kernels see it.  Voxel centres are formed in fp64 exactly as the definition
// and split into fp32 hi + lo parts.
struct GridDev {
  int dim;
  int nx, ny, nz;
  double lo[3];
  double s[3];          // voxel side lengths
  double voxel_volume;  // |P|
  int tiles_x, tiles_y, tiles_z;
  int row_long;         // ROWPOLY kernel: 1 = rows of 32 voxels per thread, 0 = rows of 16
  // voxel-slab sharding (f4, apd_shard.cu): this GridDev describes planes [off, off + n) of the grid's LAST axis (z in
  // 3D, y in 2D); ny / nz above is the slab's own count, off_y / off_z the index of its first plane in the whole grid
  // (0 for a whole grid; one of the two is always 0).  Voxel centres and index sums use the GLOBAL index i + off, so a
  // slab's arithmetic is that of the whole-grid call bit for bit; label positions are local to the slab.
  int off_y, off_z;
};

// The dual's sum of minima is reduced in two levels, the same way everywhere, so that a slab-sharded evaluation
// reproduces the whole-grid one bit for bit: the per-tile (per-brick) partials of one LAYER -- SLAB_ALIGN planes of the
// last axis: a whole number of tile layers of every kernel -- are summed by one warp in a fixed order
// (warp_ordered_sum), then the layer sums are added in ascending layer order.
constexpr int SLAB_ALIGN3 = 8, SLAB_ALIGN2 = 64;
__host__ __device__ constexpr int slab_align(int dim) { return dim == 3 ? SLAB_ALIGN3 : SLAB_ALIGN2; }
struct LayerMap {
  int n_layers;           // layers of this (slab) grid
  int per_layer;          // partials per full layer
  int n_partials;         // all partials (the last layer may hold fewer)
};

struct AssignArgs {
  GridDev g;
  int M;                 // real seeds
  int M_pad;             // padded to SEED_CHUNK
  const float* seeds;    // [M_pad, REC]
  int32_t* labels;       // [N] or nullptr
  int labels_vec;        // 1: the labels pointer is 16-byte aligned, rows may leave as int4 stores; 0: scalar stores
  unsigned int* count;   // [M] voxels per cell (exact integers: eq. 2.8)
  unsigned long long* idxsum;  // [M,3] sum of voxel indices per axis, or nullptr
  double* dual_partial;  // [n_tiles] sum over the tile of min_i C_ij
  // culling (a7); all nullptr / 0 for brute force.  Two levels: SUPER-TILES (groups of CTA tiles) hold a parent
  // candidate list each; every BRICK (the voxels of one warp, 4 per CTA tile) holds its own list, a subset of its
  // parent's.  Lists are ascending in seed index.  count < 0 = the list overflowed its capacity: fall back one
  // level (brick -> parent -> all seeds).
  const float* rec;        // [M_pad, REC] per-seed records (DIRECT layout) + rho_brick, rho_super
  const int* brick_list;   // [n_tiles * 4, BRICK_CAP]
  const int* brick_count;  // [n_tiles * 4]
  const int* super_list;   // [n_super, SUPER_CAP]
  const int* super_count;  // [n_super]
  int super_x, super_y;    // super-tiles per axis (x, y); super-tile of CTA tile (bx,by,bz) = (bx/SUPER_TX, ...)
  unsigned long long* pairs_ctr;  // [1] voxel-seed pairs evaluated
  // in-row offsets from a row's midpoint, tt[j] = fl32((j + 1/2) s_x), and their squares tt[16 + j] = fl32(tau_j^2),
  // j < 16: the same for every row of every tile, so they are kernel PARAMETERS -- the compiler keeps them in
  // uniform registers / the constant bank and the FFMA2s read them from there, which frees the vector registers.
  // (Voxel V/2 + j of a row is evaluated at x_mid + tau_j, V/2 - 1 - j at x_mid - tau_j: within one ulp of its fp32
  // centre, and exactly the centre on power-of-two grids.)
  float tt[32];
  const int* done_flag;  // solve loop only: kernels return at once when *done_flag != 0; else nullptr
  const uint4* qfix;     // TENSOR kernel only: [M_pad, 6] record + tile-independent bf16 coefficient parts (apd_tensor.cu)
};

struct Workspace {
  int dim = 0, max_seeds = 0, device = 0, sm_count = 0;
  float* seeds = nullptr;              // packed table [M_pad, REC]
  unsigned int* count = nullptr;       // [max_seeds]
  unsigned long long* idxsum = nullptr;  // [max_seeds,3]
  double* dual_partial = nullptr;      // [partial_cap]
  size_t partial_cap = 0;
  double* layer_buf = nullptr;         // [layer_cap] layer sums of the dual partials (two-level reduction)
  size_t layer_cap = 0;
  // culling (apd_cull.cu), allocated on first use
  float* rec = nullptr;                // [M_pad, REC] per-seed records + rho_brick, rho_super
  int* brick_list = nullptr;           // [brick_cap_n * BRICK_CAP]
  int* brick_count = nullptr;          // [brick_cap_n]
  int* tile_list = nullptr;            // [brick_cap_n / 4 * TILE_CAP] CTA-tile lists kept between the evaluations of a solve
  int* tile_count = nullptr;           // [brick_cap_n / 4]
  size_t brick_cap_n = 0;
  int* super_list = nullptr;           // [super_cap_n * SUPER_CAP]
  int* super_count = nullptr;          // [super_cap_n]
  size_t super_cap_n = 0;
  unsigned long long* pairs_ctr = nullptr;
  uint4* qfix = nullptr;               // TENSOR kernel: [M_pad, 6] uint4, allocated on first use
  double* pt_acc = nullptr;            // apd_assign_points: fp64 accumulators vol[max_seeds] | csum[max_seeds,3]
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool timed = false;
  // what the most recent evaluation launched (apd_assign_stats)
  int last_kernel = -1, last_row_long = 0, last_cull = 0, last_tiles = 0;
  double* lloyd_buf = nullptr;         // apd_lloyd scratch: centroids [max_seeds, dim] | vol [max_seeds] | 2 scalars
  // apd_solve state (apd_lbfgs.cu), allocated on first use
  struct SolveState* sstate = nullptr;  // device scalars
  double* svec = nullptr;               // device fp64 vectors: w, g, p, w_try, w_best, g_new, q, S[m], Y[m]
  int svec_hist = 0;                    // history capacity svec was sized for
  int lb_cluster = 0;                   // CTAs of lbfgs_step_kernel's cluster on this device (0: not chosen yet)
  double* gram = nullptr;               // [(2 svec_hist + 1)^2] Gram matrix of the L-BFGS basis
  float* w32 = nullptr;                 // [max_seeds] fl32(w) the next evaluation uses
  float* wref = nullptr;                // [max_seeds] weights the current brick candidate lists were built at
  float* wref_s = nullptr;              // [max_seeds] weights the current super-tile lists were built at
  float* wref_t = nullptr;              // [max_seeds] weights the current CTA-tile lists were built at
  double* e_vol = nullptr;              // [max_seeds] evaluation outputs inside the solve loop
  double* e_scal = nullptr;             // [2] dual, max_rel_err
  double* hist = nullptr;               // [2 * SOLVE_HIST_CAP] (dual, err) per evaluation of the last solve
  int hist_len = 0;
  int last_rebuilds = 0;                // candidate-list rebuilds of the last solve (0 without culling)
  struct SolveReport* report = nullptr; // pinned, mapped host memory the step kernel writes
  // device scratch of the *_host calls (apd_host.cu): grow-only, kept between calls, freed with the context
  static constexpr int HOST_SLOTS = 10;
  void* host_buf[HOST_SLOTS] = {};
  size_t host_cap[HOST_SLOTS] = {};
  cudaEvent_t sev[2] = {nullptr, nullptr};
};

// kernels (apd_kernels.cu)
cudaError_t launch_pack_seeds(int dim, int M, int M_pad, const float* X, const float* A, const float* w,
                              float* seeds, unsigned int* count, unsigned long long* idxsum,
                              const int* done_flag, cudaStream_t st);
cudaError_t launch_assign(int kernel, const AssignArgs& a, cudaStream_t st);
// ROWPOLY kernel (apd_rowpoly.cu): its own pair-interleaved seed table
cudaError_t launch_pack_pairs(int dim, int M, int M_pad, const float* X, const float* A, const float* w,
                              float* seeds, unsigned int* count, unsigned long long* idxsum,
                              const int* done_flag, cudaStream_t st);
cudaError_t launch_assign_rowpoly(const AssignArgs& a, cudaStream_t st);
// TENSOR kernel (apd_tensor.cu, row a8): reads the DIRECT record table plus its own bf16 table
void tensor_tile_counts(int dim, int nx, int ny, int nz, int* tx, int* ty, int* tz);
cudaError_t launch_pack_qfix(const GridDev& g, int M_pad, const float* rec, uint4* qfix, const int* done_flag,
                             cudaStream_t st);
cudaError_t launch_assign_tensor(const AssignArgs& a, cudaStream_t st);
// ---- culling geometry (a7) --------------------------------------------------------------------------------
// The culled kernel always runs the SHORT-row geometry: CTA tile 16 x 16 x 8 voxels (3D) / 32 x 64 pixels (2D),
// 128 threads = 4 warps, each warp owning one BRICK of 32 rows of 16 voxels:
//   3D: brick w = x [0,16) x y [4w, 4w+4) x z [0,8)      lane -> (y = lane & 3, z = lane >> 2)
//   2D: brick w = x [16 (w&1), +16) x y [32 (w>>1), +32)   lane -> y
// A SUPER-TILE is SUPER_T{X,Y,Z} CTA tiles per axis: 64 x 32 x 32 voxels (3D) / 128 x 128 pixels (2D).
constexpr int CULL_TILE3_X = 16, CULL_TILE3_Y = 16, CULL_TILE3_Z = 8;
constexpr int CULL_TILE2_X = 32, CULL_TILE2_Y = 64;
constexpr int SUPER3_TX = 4, SUPER3_TY = 2, SUPER3_TZ = 4;
constexpr int SUPER2_TX = 4, SUPER2_TY = 2;
constexpr int BRICK_CAP = 256;         // candidate-list capacity of a brick
constexpr int SUPER_CAP = 4096;        // candidate-list capacity of a super-tile
constexpr int TILE_CAP = 768;          // candidate-list capacity of a CTA tile (shared memory; global inside a solve)
constexpr int SOLVE_HIST_CAP = 8192;   // evaluations of a solve whose (dual, err) are kept for apd_solve_history

// origin (relative to the CTA tile) and extent, in voxels, of brick w
__host__ __device__ inline void brick_box(int dim, int w, int* ox, int* oy, int* oz, int* ex, int* ey, int* ez) {
  if (dim == 3) { *ox = 0; *oy = 4 * w; *oz = 0; *ex = 16; *ey = 4; *ez = 8; }
  else          { *ox = 16 * (w & 1); *oy = 32 * (w >> 1); *oz = 0; *ex = 16; *ey = 32; *ez = 1; }
}

// Launch with programmatic stream serialization: the kernel's CTAs may be scheduled while the kernel before it in the
// stream drains; the kernel starts with pdl_enter() (apd_device.cuh), which waits for that kernel's completion.
template <class... KArgs, class... Args>
static inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, int block, size_t smem, cudaStream_t st,
                                     Args&&... args) {
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

struct CullBuffers {
  float* rec; int* brick_list; int* brick_count; int* super_list; int* super_count; int* tile_list; int* tile_count;
  unsigned long long* pairs_ctr;
};
cudaError_t launch_cull(const GridDev& g, int M, int M_pad, const float* X, const float* A, const float* w,
                        const CullBuffers& cb, int n_super_x, int n_super_y, int n_super_z, unsigned int* count,
                        unsigned long long* idxsum, const int* done_flag, const int* rebuild, const float* delta,
                        const int* rebuild_s, const float* delta_s, const int* rebuild_t, const float* delta_t,
                        bool skip_pack, cudaStream_t st);
void cull_super_counts(const GridDev& g, int* nsx, int* nsy, int* nsz);
int rowpoly_tile_counts(int dim, int nx, int ny, int nz, int sm_count, bool cull, int* tx, int* ty, int* tz);
int assign_tile_counts(int kernel, int dim, int nx, int ny, int nz, int sm_count, bool cull, int* tx, int* ty, int* tz);
cudaError_t launch_finalize(const GridDev& g, int M, LayerMap lm, double* layer_buf, const unsigned int* count,
                            const unsigned long long* count64, const unsigned long long* idxsum,
                            const double* dual_partial,
                            const float* X, const float* w, const float* target_vol,
                            double* vol, double* dual, double* max_rel_err, double* centroids,
                            uint64_t* pairs_evaluated, const unsigned long long* pairs_ctr, const int* done_flag,
                            cudaStream_t st);

// apd_points.cu: sizing / allocation of the point-set accumulators, and one evaluation on points.  vol == nullptr
// leaves the raw outputs (ws.pt_acc volumes, ws.dual_partial) for lbfgs_step_kernel and skips the finalize kernel.
int points_prepare(apd_ctx* ctx, long long N, int* n_partials, cudaStream_t st);
int enqueue_points(apd_ctx* ctx, long long N, const float* Y, const float* pvol, int M, const float* X, const float* A,
                   const float* w, const float* target_vol, int32_t* labels, double* vol, double* dual,
                   double* max_rel_err, double* centroids, const int* done_flag, int* n_partials, cudaStream_t st);

// What the device-side optimiser reports to the host (mapped pinned memory).
struct SolveReport {
  volatile int done;      // 0 running, 1 finished
  volatile int status;    // apd_status
  volatile int iters, evals;
  volatile double err, dual;
  volatile int cull_rebuilds;   // evaluations of the solve loop that rebuilt the brick candidate lists
  volatile int cull_rebuilds_s; // ... and the super-tile lists
  volatile int cull_rebuilds_t; // ... and the CTA-tile lists
};

// host helpers shared by apd_api.cu and apd_lbfgs.cu
std::string make_grid(const apd_ctx* ctx, const apd_grid* grid, int kernel, bool cull, GridDev* g,
                      const apd_slab* slab = nullptr);
LayerMap layer_map(const GridDev& g, bool cull);
int resolve_kernel(const apd_ctx* ctx, const apd_opts* o, const apd_grid* grid, int M, bool* cull, std::string* err);
// Sizes the buffers an evaluation of grid `g` needs (dual partials; with culling the candidate lists and the record
// table; for the TENSOR kernel its seed table).  Grow-only.  Growing synchronises `st` and reallocates: apd_reserve
// does this ahead of time so that apd_assign / apd_solve never do.
int ensure_eval_buffers(apd_ctx* ctx, const GridDev& g, int kernel, bool cull, cudaStream_t st);
int ensure_solve_state(apd_ctx* ctx, int hist);
// apd_lbfgs.cu: Algorithm 2 on a grid (slab == nullptr) or on one slab of it with a counter exchange (apd_shard.cu)
int solve_grid(apd_ctx* ctx, const char* who, const apd_grid* grid, const apd_slab* slab, int32_t M, const float* X,
               const float* A, const float* target_vol, double tol, const float* w_init, float* w, int32_t* labels,
               double* vol, double* w64, uint64_t* counters, apd_reduce_fn reduce, void* user, int32_t* iters,
               int32_t* evals, double* max_rel_err, double* dual, const apd_opts* opts, void* cuda_stream);
// apd_shard.cu: count[M] u32 (+ idxsum) and the layer sums of this slab's dual partials -> the u64 counter block
cudaError_t launch_pack_counters(const GridDev& g, int M, LayerMap lm, int n_layers_full, const unsigned int* count,
                                 const unsigned long long* idxsum, const double* dual_partial, uint64_t* counters,
                                 const int* done_flag, cudaStream_t st);
// user point sets (apd_points.cu) have no layers: their flat partials are grouped by 256
inline LayerMap points_layer_map(int n_partials) {
  LayerMap lm; lm.per_layer = 256; lm.n_partials = n_partials; lm.n_layers = (n_partials + 255) / 256; return lm;
}
int enqueue_evaluation(apd_ctx* ctx, const GridDev& g, int kernel, int M, const float* X, const float* A,
                       const float* w, const float* target_vol, int32_t* labels, double* vol, double* dual,
                       double* max_rel_err, double* centroids, uint64_t* pairs, bool timed, bool cull,
                       const int* done_flag, cudaStream_t st, const int* cull_rebuild = nullptr,
                       const float* cull_delta = nullptr, const int* cull_rebuild_s = nullptr,
                       const float* cull_delta_s = nullptr, const int* cull_rebuild_t = nullptr,
                       const float* cull_delta_t = nullptr, bool cull_skip_pack = false);

}  // namespace apd

struct apd_ctx {
  apd::Workspace ws;
  std::string err;
};
