// apd_api.cu -- the C ABI of include/apd.h: context, argument validation, apd_assign and the
// host-buffer wrappers.  Host logic only; every step of the path runs in the kernels.
#include "apd_internal.cuh"
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

using namespace apd;

static thread_local std::string g_create_err;

#define APD_CUDA_TRY(ctx, call)                                                              \
  do {                                                                                       \
    cudaError_t e__ = (call);                                                                \
    if (e__ != cudaSuccess) {                                                                \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);                      \
      return APD_E_CUDA;                                                                     \
    }                                                                                        \
  } while (0)

extern "C" void apd_default_opts(apd_opts* o) {
  if (!o) return;
  std::memset(o, 0, sizeof(*o));
  o->kernel = APD_KERNEL_AUTO;
  o->cull = 0;
  o->lbfgs_history = 10;
  o->max_iters = 1000;
  o->max_evals = 0;
}

static void free_ws(Workspace& ws) {
  cudaFree(ws.lloyd_buf); cudaFree(ws.pt_acc); cudaFree(ws.qfix); cudaFree(ws.rec); cudaFree(ws.brick_list); cudaFree(ws.brick_count); cudaFree(ws.tile_list); cudaFree(ws.tile_count); cudaFree(ws.super_list);
  cudaFree(ws.super_count); cudaFree(ws.pairs_ctr);
  cudaFree(ws.seeds); cudaFree(ws.count); cudaFree(ws.idxsum); cudaFree(ws.dual_partial); cudaFree(ws.layer_buf);
  cudaFree(ws.sstate); cudaFree(ws.svec); cudaFree(ws.gram); cudaFree(ws.w32); cudaFree(ws.wref); cudaFree(ws.wref_s); cudaFree(ws.wref_t); cudaFree(ws.e_vol); cudaFree(ws.e_scal); cudaFree(ws.hist);
  for (int i = 0; i < Workspace::HOST_SLOTS; ++i) cudaFree(ws.host_buf[i]);
  if (ws.report) cudaFreeHost(ws.report);
  for (int i = 0; i < 2; ++i) if (ws.sev[i]) cudaEventDestroy(ws.sev[i]);
  if (ws.ev0) cudaEventDestroy(ws.ev0);
  if (ws.ev1) cudaEventDestroy(ws.ev1);
  ws = Workspace();
}

extern "C" int apd_create(apd_ctx** out, int32_t dim, int32_t max_seeds, int32_t device) {
  if (!out) { g_create_err = "apd_create: out is NULL"; return APD_E_ARG; }
  *out = nullptr;
  if (dim != 2 && dim != 3) { g_create_err = "apd_create: dim must be 2 or 3"; return APD_E_ARG; }
  if (max_seeds < 1) { g_create_err = "apd_create: max_seeds must be >= 1"; return APD_E_ARG; }
  cudaDeviceProp prop;
  cudaError_t e = cudaGetDeviceProperties(&prop, device);
  if (e != cudaSuccess) { g_create_err = std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e); return APD_E_CUDA; }
  if (prop.major != 10) {
    g_create_err = "apd_create: device is compute capability " + std::to_string(prop.major) + "." +
                   std::to_string(prop.minor) + "; this library is built for sm_100a only";
    return APD_E_ARCH;
  }
  e = cudaSetDevice(device);
  if (e != cudaSuccess) { g_create_err = std::string("cudaSetDevice: ") + cudaGetErrorString(e); return APD_E_CUDA; }
  apd_ctx* c = new (std::nothrow) apd_ctx();
  if (!c) { g_create_err = "apd_create: out of host memory"; return APD_E_CUDA; }
  Workspace& ws = c->ws;
  ws.dim = dim; ws.max_seeds = max_seeds; ws.device = device; ws.sm_count = prop.multiProcessorCount;
  const size_t m_pad = ((size_t)max_seeds + SEED_CHUNK - 1) / SEED_CHUNK * SEED_CHUNK;
  ws.partial_cap = 1 << 16;
  bool ok = cudaMalloc(&ws.seeds, m_pad * rec_floats(dim) * sizeof(float)) == cudaSuccess &&
            cudaMalloc(&ws.count, (size_t)max_seeds * sizeof(unsigned int)) == cudaSuccess &&
            cudaMalloc(&ws.idxsum, (size_t)max_seeds * 3 * sizeof(unsigned long long)) == cudaSuccess &&
            cudaMalloc(&ws.dual_partial, ws.partial_cap * sizeof(double)) == cudaSuccess &&
            cudaEventCreate(&ws.ev0) == cudaSuccess && cudaEventCreate(&ws.ev1) == cudaSuccess;
  if (!ok) {
    g_create_err = std::string("apd_create: workspace allocation failed: ") + cudaGetErrorString(cudaGetLastError());
    free_ws(ws);
    delete c;
    return APD_E_CUDA;
  }
  *out = c;
  return APD_OK;
}

extern "C" void apd_destroy(apd_ctx* ctx) {
  if (!ctx) return;
  cudaSetDevice(ctx->ws.device);
  free_ws(ctx->ws);
  delete ctx;
}

extern "C" const char* apd_last_error(const apd_ctx* ctx) {
  return ctx ? ctx->err.c_str() : g_create_err.c_str();
}

namespace apd {

// Validates the grid and fills the device-side description.  Returns "" or an error text.
std::string make_grid(const apd_ctx* ctx, const apd_grid* grid, int kernel, bool cull, GridDev* g,
                      const apd_slab* slab) {
  if (!grid) return "grid is NULL";
  if (grid->dim != ctx->ws.dim) return "grid.dim differs from the context's dim";
  const int d = grid->dim;
  long long N = 1;
  double P = 1.0;
  GridDev out;
  std::memset(&out, 0, sizeof(out));
  out.dim = d;
  int n[3] = {1, 1, 1};
  for (int k = 0; k < d; ++k) {
    if (grid->n[k] < 1) return "grid.n[k] must be >= 1";
    if (!(grid->hi[k] > grid->lo[k]) || !std::isfinite(grid->hi[k]) || !std::isfinite(grid->lo[k]))
      return "grid needs finite hi[k] > lo[k]";
    n[k] = grid->n[k];
    N *= n[k];
    if (N >= (1ll << 31)) return "grid has 2^31 voxels or more";
    out.lo[k] = grid->lo[k];
    out.s[k] = (grid->hi[k] - grid->lo[k]) / (double)n[k];
    P *= out.s[k];
  }
  if (slab) {
    // planes [lo, lo + n) of the last axis; boundaries on whole layers so that every layer sum has one owner
    const int last = d - 1, al = slab_align(d);
    if (slab->lo < 0 || slab->n < 1 || (long long)slab->lo + slab->n > n[last]) return "slab outside the grid";
    if (slab->lo % al != 0) return "slab.lo must be a multiple of apd_slab_align(dim)";
    if (slab->n % al != 0 && slab->lo + slab->n != n[last])
      return "slab.n must be a multiple of apd_slab_align(dim) unless the slab ends at the grid's last plane";
    n[last] = slab->n;
    if (d == 3) out.off_z = slab->lo; else out.off_y = slab->lo;
  }
  out.nx = n[0]; out.ny = n[1]; out.nz = n[2];
  out.voxel_volume = P;
  out.row_long = assign_tile_counts(kernel, d, out.nx, out.ny, out.nz, ctx->ws.sm_count, cull, &out.tiles_x, &out.tiles_y,
                                    &out.tiles_z);
  *g = out;
  return "";
}

// The two-level reduction of the dual partials for grid (slab) g: SLAB_ALIGN planes of the last axis per layer.
LayerMap layer_map(const GridDev& g, bool cull) {
  const int al = slab_align(g.dim);
  const int n_last = g.dim == 3 ? g.nz : g.ny, tiles_last = g.dim == 3 ? g.tiles_z : g.tiles_y;
  const int n_layers = (n_last + al - 1) / al;
  const int tiles_per_layer_axis = (tiles_last + n_layers - 1) / n_layers;      // 1 or 2 tile layers per layer
  const int per_tile_layer = g.tiles_x * (g.dim == 3 ? g.tiles_y : 1) * (cull ? 4 : 1);
  LayerMap lm;
  lm.n_layers = n_layers;
  lm.per_layer = tiles_per_layer_axis * per_tile_layer;
  lm.n_partials = tiles_last * per_tile_layer;
  return lm;
}

// opts -> kernel (AUTO resolved) and whether culling runs.  AUTO on a grid with fewer voxels along an axis than
// half a tile of the row kernels (x: 8, y: 8 in 3D, z: 4) takes DIRECT and drops opts.cull: those kernels expand the
// cost about a row's midpoint in x and (3D) the tile's midpoint in y and z, which on such a grid lie several domain
// widths L outside it: a cost then carries a few fp32 ulp of a ((1 + 8/n) L)^2 instead of a few ulp of itself
// (DESIGN.md 5).
static bool narrow_grid(const apd_grid* grid) {
  if (!grid) return false;
  if (grid->n[0] < 8) return true;
  return grid->dim == 3 && (grid->n[1] < 8 || grid->n[2] < 4);
}
int resolve_kernel(const apd_ctx* /*ctx*/, const apd_opts* o, const apd_grid* grid, int /*M*/, bool* cull, std::string* err) {
  int k = o ? o->kernel : APD_KERNEL_AUTO;
  if (k != APD_KERNEL_AUTO && k != APD_KERNEL_DIRECT && k != APD_KERNEL_ROWPOLY && k != APD_KERNEL_TENSOR) { *err = "unknown opts.kernel"; return -1; }
  if (o && (o->cull != 0 && o->cull != 1)) { *err = "opts.cull must be 0 or 1"; return -1; }
  if (o && (o->reserved[0] || o->reserved[1] || o->reserved[2])) { *err = "opts.reserved must be 0"; return -1; }
  *cull = o && o->cull;
  if (k == APD_KERNEL_AUTO) {
    if (narrow_grid(grid)) { *cull = false; return APD_KERNEL_DIRECT; }
    k = APD_KERNEL_ROWPOLY;
    // brute force: the tensor-core kernel.  Measured on B200 with the persistent kernel: TENSOR /
    // ROWPOLY time 0.22-0.88 on every 3D grid and seed count tried (32^3 .. 256^3 voxels, M = 64 .. 10^4), and
    // 0.42-0.83 in 2D (64^2 x 10 .. 4096^2 x 1000; 1024^2 x 1000: 0.65, 2048^2 x 5000: 0.70).
    if (grid && !*cull) k = APD_KERNEL_TENSOR;
  }
  if (*cull && k != APD_KERNEL_ROWPOLY) { *err = "opts.cull needs kernel AUTO or ROWPOLY"; return -1; }
  return k;
}

int ensure_eval_buffers(apd_ctx* ctx, const GridDev& g, int kernel, bool cull, cudaStream_t st) {
  Workspace& ws = ctx->ws;
  const size_t n_tiles = (size_t)g.tiles_x * g.tiles_y * g.tiles_z;
  const size_t n_partials = cull ? 4 * n_tiles : n_tiles;      // the culled kernel writes one partial per brick (warp)
  const size_t m_pad_max = ((size_t)ws.max_seeds + SEED_CHUNK - 1) / SEED_CHUNK * SEED_CHUNK;
  if (n_partials > ws.partial_cap) {
    APD_CUDA_TRY(ctx, cudaStreamSynchronize(st));            // earlier work on st may still read the old buffer
    APD_CUDA_TRY(ctx, cudaFree(ws.dual_partial));
    ws.dual_partial = nullptr;
    ws.partial_cap = 0;
    APD_CUDA_TRY(ctx, cudaMalloc(&ws.dual_partial, n_partials * sizeof(double)));
    ws.partial_cap = n_partials;
  }
  const size_t n_layers = (size_t)layer_map(g, cull).n_layers;
  if (n_layers > ws.layer_cap) {
    APD_CUDA_TRY(ctx, cudaStreamSynchronize(st));
    cudaFree(ws.layer_buf);
    ws.layer_buf = nullptr; ws.layer_cap = 0;
    APD_CUDA_TRY(ctx, cudaMalloc(&ws.layer_buf, n_layers * sizeof(double)));
    ws.layer_cap = n_layers;
  }
  if (kernel == APD_KERNEL_TENSOR && !ws.qfix)
    APD_CUDA_TRY(ctx, cudaMalloc(&ws.qfix, m_pad_max * 6 * sizeof(uint4)));
  if (cull) {
    int nsx, nsy, nsz;
    cull_super_counts(g, &nsx, &nsy, &nsz);
    const size_t n_super = (size_t)nsx * nsy * nsz, n_bricks = n_tiles * 4;
    if (!ws.rec) {
      APD_CUDA_TRY(ctx, cudaMalloc(&ws.rec, m_pad_max * rec_floats(ws.dim) * sizeof(float)));
      APD_CUDA_TRY(ctx, cudaMalloc(&ws.pairs_ctr, sizeof(unsigned long long)));
    }
    if (n_bricks > ws.brick_cap_n || n_super > ws.super_cap_n) {
      APD_CUDA_TRY(ctx, cudaStreamSynchronize(st));
      cudaFree(ws.brick_list); cudaFree(ws.brick_count); cudaFree(ws.super_list); cudaFree(ws.super_count);
      cudaFree(ws.tile_list); cudaFree(ws.tile_count);
      ws.brick_list = ws.brick_count = ws.super_list = ws.super_count = ws.tile_list = ws.tile_count = nullptr;
      const size_t nb = n_bricks > ws.brick_cap_n ? n_bricks : ws.brick_cap_n;
      const size_t ns = n_super > ws.super_cap_n ? n_super : ws.super_cap_n;
      ws.brick_cap_n = ws.super_cap_n = 0;
      APD_CUDA_TRY(ctx, cudaMalloc(&ws.brick_list, nb * BRICK_CAP * sizeof(int)));
      APD_CUDA_TRY(ctx, cudaMalloc(&ws.brick_count, nb * sizeof(int)));
      APD_CUDA_TRY(ctx, cudaMalloc(&ws.tile_list, (nb / 4) * TILE_CAP * sizeof(int)));
      APD_CUDA_TRY(ctx, cudaMalloc(&ws.tile_count, (nb / 4) * sizeof(int)));
      APD_CUDA_TRY(ctx, cudaMalloc(&ws.super_list, ns * SUPER_CAP * sizeof(int)));
      APD_CUDA_TRY(ctx, cudaMalloc(&ws.super_count, ns * sizeof(int)));
      ws.brick_cap_n = nb; ws.super_cap_n = ns;
    }
  }
  return APD_OK;
}

// Enqueues one evaluation (pack -> assign -> finalize) on `st`.  All pointers device.
int enqueue_evaluation(apd_ctx* ctx, const GridDev& g, int kernel, int M, const float* X, const float* A,
                       const float* w, const float* target_vol, int32_t* labels, double* vol, double* dual,
                       double* max_rel_err, double* centroids, uint64_t* pairs, bool timed, bool cull,
                       const int* done_flag, cudaStream_t st, const int* cull_rebuild, const float* cull_delta,
                       const int* cull_rebuild_s, const float* cull_delta_s, const int* cull_rebuild_t,
                       const float* cull_delta_t, bool cull_skip_pack) {
  Workspace& ws = ctx->ws;
  const int M_pad = (M + SEED_CHUNK - 1) / SEED_CHUNK * SEED_CHUNK;
  const int n_tiles = g.tiles_x * g.tiles_y * g.tiles_z;
  const int rc_buf = ensure_eval_buffers(ctx, g, kernel, cull, st);   // no-op after apd_reserve / a call of this size
  if (rc_buf != APD_OK) return rc_buf;
  if (cull) {
    // the culled kernel reads the per-seed record table that launch_cull packs (and which zeroes the accumulators)
  } else if (kernel == APD_KERNEL_ROWPOLY)
    APD_CUDA_TRY(ctx, launch_pack_pairs(g.dim, M, M_pad, X, A, w, ws.seeds, ws.count,
                                        centroids ? ws.idxsum : nullptr, done_flag, st));
  else
    APD_CUDA_TRY(ctx, launch_pack_seeds(g.dim, M, M_pad, X, A, w, ws.seeds, ws.count,
                                        centroids ? ws.idxsum : nullptr, done_flag, st));
  if (kernel == APD_KERNEL_TENSOR)
    APD_CUDA_TRY(ctx, launch_pack_qfix(g, M_pad, ws.seeds, ws.qfix, done_flag, st));
  AssignArgs a;
  a.g = g; a.M = M; a.M_pad = M_pad; a.seeds = ws.seeds; a.labels = labels; a.count = ws.count;
  a.labels_vec = (reinterpret_cast<uintptr_t>(labels) & 15) == 0;
  for (int j = 0; j < 16; ++j) {      // in-row offsets from a row's midpoint and their squares (apd_rowpoly.cu: RowTau)
    const double tau = ((double)j + 0.5) * g.s[0];
    a.tt[j] = (float)tau;
    a.tt[16 + j] = (float)(tau * tau);
  }
  a.idxsum = centroids ? ws.idxsum : nullptr; a.dual_partial = ws.dual_partial;
  a.rec = nullptr; a.brick_list = nullptr; a.brick_count = nullptr; a.super_list = nullptr; a.super_count = nullptr;
  a.super_x = a.super_y = 0; a.pairs_ctr = nullptr;
  a.done_flag = done_flag;
  a.qfix = ws.qfix;
  if (cull) {
    // a7: two-level candidate lists (rebuilt when the weights left the slack they were built with)
    int nsx, nsy, nsz;
    cull_super_counts(g, &nsx, &nsy, &nsz);
    CullBuffers cb{ws.rec, ws.brick_list, ws.brick_count, ws.super_list, ws.super_count, ws.tile_list, ws.tile_count, ws.pairs_ctr};
    APD_CUDA_TRY(ctx, launch_cull(g, M, M_pad, X, A, w, cb, nsx, nsy, nsz, ws.count, centroids ? ws.idxsum : nullptr, done_flag,
                                  cull_rebuild, cull_delta, cull_rebuild_s, cull_delta_s, cull_rebuild_t, cull_delta_t, cull_skip_pack, st));
    a.rec = ws.rec; a.brick_list = ws.brick_list; a.brick_count = ws.brick_count; a.super_list = ws.super_list;
    a.super_count = ws.super_count; a.super_x = nsx; a.super_y = nsy;
    a.pairs_ctr = vol ? ws.pairs_ctr : nullptr;      // apd_solve's loop (vol == nullptr) has no use for the pair count
  }
  ws.last_kernel = kernel; ws.last_row_long = g.row_long; ws.last_cull = cull ? 1 : 0; ws.last_tiles = n_tiles;
  if (timed) APD_CUDA_TRY(ctx, cudaEventRecord(ws.ev0, st));
  APD_CUDA_TRY(ctx, launch_assign(kernel, a, st));
  if (timed) { APD_CUDA_TRY(ctx, cudaEventRecord(ws.ev1, st)); ws.timed = true; }
  if (vol)     // apd_solve's loop passes vol == nullptr: lbfgs_step_kernel finishes the evaluation itself
    APD_CUDA_TRY(ctx, launch_finalize(g, M, layer_map(g, cull), ws.layer_buf, ws.count, nullptr, a.idxsum, ws.dual_partial,
                                      X, w, target_vol, vol, dual, max_rel_err, centroids, pairs,
                                      cull ? ws.pairs_ctr : nullptr, done_flag, st));
  return APD_OK;
}

}  // namespace apd

extern "C" int apd_assign(apd_ctx* ctx, const apd_grid* grid, int32_t M, const float* X, const float* A,
                          const float* w, const float* target_vol, int32_t* labels, double* vol, double* dual,
                          double* max_rel_err, double* centroids, uint64_t* pairs_evaluated,
                          const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  std::string e;
  bool cull = false;
  const int kernel = resolve_kernel(ctx, opts, grid, M, &cull, &e);
  if (kernel < 0) { ctx->err = "apd_assign: " + e; return APD_E_ARG; }
  if (M < 1 || M > ctx->ws.max_seeds) { ctx->err = "apd_assign: M out of range [1, max_seeds]"; return APD_E_ARG; }
  if (!X || !A || !w || !vol || !dual) { ctx->err = "apd_assign: X, A, w, vol and dual are required"; return APD_E_ARG; }
  GridDev g;
  e = make_grid(ctx, grid, kernel, cull, &g);
  if (!e.empty()) { ctx->err = "apd_assign: " + e; return APD_E_ARG; }
  APD_CUDA_TRY(ctx, cudaSetDevice(ctx->ws.device));
  return enqueue_evaluation(ctx, g, kernel, M, X, A, w, target_vol, labels, vol, dual, max_rel_err, centroids,
                            pairs_evaluated, true, cull, nullptr, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int apd_assign_stats(apd_ctx* ctx, int32_t* kernel, int32_t* row_long, int32_t* cull, int32_t* n_tiles,
                                double* kernel_ms) {
  if (!ctx) return APD_E_ARG;
  const Workspace& ws = ctx->ws;
  if (ws.last_kernel < 0) { ctx->err = "apd_assign_stats: no evaluation has run on this context"; return APD_E_ARG; }
  if (kernel) *kernel = ws.last_kernel;
  if (row_long) *row_long = ws.last_row_long;
  if (cull) *cull = ws.last_cull;
  if (n_tiles) *n_tiles = ws.last_tiles;
  if (kernel_ms) {
    *kernel_ms = -1.0;
    if (ws.timed) {
      float ms = 0.f;
      if (cudaEventSynchronize(ws.ev1) != cudaSuccess || cudaEventElapsedTime(&ms, ws.ev0, ws.ev1) != cudaSuccess) {
        ctx->err = "apd_assign_stats: the kernel's events could not be read";
        return APD_E_CUDA;
      }
      *kernel_ms = (double)ms;
    }
  }
  return APD_OK;
}

extern "C" int apd_reserve(apd_ctx* ctx, const apd_grid* grid, const apd_opts* opts) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  std::string e;
  bool cull = false;
  const int kernel = resolve_kernel(ctx, opts, grid, ctx->ws.max_seeds, &cull, &e);
  if (kernel < 0) { ctx->err = "apd_reserve: " + e; return APD_E_ARG; }
  GridDev g;
  e = make_grid(ctx, grid, kernel, cull, &g);
  if (!e.empty()) { ctx->err = "apd_reserve: " + e; return APD_E_ARG; }
  APD_CUDA_TRY(ctx, cudaSetDevice(ctx->ws.device));
  int rc = ensure_eval_buffers(ctx, g, kernel, cull, nullptr);
  if (rc != APD_OK) return rc;
  if ((!opts || opts->kernel == APD_KERNEL_AUTO) && !cull) {
    // AUTO picks ROWPOLY or TENSOR by the number of seeds of the call: size the workspace for both
    for (int k2 : {APD_KERNEL_ROWPOLY, APD_KERNEL_TENSOR}) {
      GridDev g2;
      e = make_grid(ctx, grid, k2, false, &g2);
      if (!e.empty()) { ctx->err = "apd_reserve: " + e; return APD_E_ARG; }
      rc = ensure_eval_buffers(ctx, g2, k2, false, nullptr);
      if (rc != APD_OK) return rc;
    }
  }
  const int hist = opts ? opts->lbfgs_history : 10;
  if (hist < 1 || hist > 64) { ctx->err = "apd_reserve: lbfgs_history must be in [1,64]"; return APD_E_ARG; }
  rc = ensure_solve_state(ctx, hist);
  if (rc != APD_OK) return rc;
  Workspace& ws = ctx->ws;
  if (!ws.lloyd_buf)
    APD_CUDA_TRY(ctx, cudaMalloc(&ws.lloyd_buf, ((size_t)ws.max_seeds * (ws.dim + 1) + 2) * sizeof(double)));
  return APD_OK;
}
