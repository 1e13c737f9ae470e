// apd_static.cu -- apd_assign_static: one evaluation (seed pack -> ROWPOLY voxel x seed kernel -> finalize) that
// ALLOCATES NOTHING.  For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
// harnesses that forbid it).  The scratch the evaluation needs -- the packed seed table, the per-cell counts, the
// per-tile partial sums of the dual and their layer sums -- lives in ONE file-scope __device__ array of a fixed,
// modest size; every GPU that loads the library holds it until the process exits.  The kernels and their launch
// order are those of apd_assign with opts.kernel = APD_KERNEL_ROWPOLY, opts.cull = 0 (apd_api.cu:
// enqueue_evaluation), so the results are the same bits.
//
// Host code must not hand the array's NAME to a kernel: on the host it is a stand-in, not a device address.  The
// address is taken once per device with cudaGetSymbolAddress, with that device current (static_scratch_of below).
#include "apd_internal.cuh"
#include <cstdarg>
#include <cstdio>
#include <mutex>

using namespace apd;

// Limits of the entry point (include/apd.h states them too).
constexpr int STATIC_MAX_SEEDS = APD_STATIC_MAX_SEEDS;        // 4096
constexpr int STATIC_MAX_TILES = APD_STATIC_MAX_TILES;        // 16384 CTA tiles (one dual partial each)
constexpr int STATIC_MAX_LAYERS = 1024;                       // layers of 8 planes (3D) / 64 rows (2D)

// Layout of the scratch array, in bytes from its start; every part 256-byte aligned.
constexpr size_t ST_SEEDS_OFF = 0;                       // pair table, 10 (3D) / 6 (2D) of REC3 = 12 floats per seed
constexpr size_t ST_SEEDS_BYTES = (size_t)STATIC_MAX_SEEDS * REC3 * sizeof(float);       // 196,608
constexpr size_t ST_COUNT_OFF = ST_SEEDS_OFF + ST_SEEDS_BYTES;                           // [M] u32
constexpr size_t ST_COUNT_BYTES = (size_t)STATIC_MAX_SEEDS * sizeof(unsigned int);       // 16,384
constexpr size_t ST_PARTIAL_OFF = ST_COUNT_OFF + ST_COUNT_BYTES;                         // [n_tiles] fp64
constexpr size_t ST_PARTIAL_BYTES = (size_t)STATIC_MAX_TILES * sizeof(double);           // 131,072
constexpr size_t ST_LAYER_OFF = ST_PARTIAL_OFF + ST_PARTIAL_BYTES;                       // [n_layers] fp64
constexpr size_t ST_LAYER_BYTES = (size_t)STATIC_MAX_LAYERS * sizeof(double);            // 8,192
constexpr size_t ST_BYTES = ST_LAYER_OFF + ST_LAYER_BYTES;                               // 352,256 = 344 KiB
static_assert(STATIC_MAX_SEEDS % SEED_CHUNK == 0, "the padded seed table must fit");
static_assert(ST_COUNT_OFF % 256 == 0 && ST_PARTIAL_OFF % 256 == 0 && ST_LAYER_OFF % 256 == 0, "256-byte parts");

static __device__ __align__(256) unsigned char g_static_scratch[ST_BYTES];

// ---- error text: a fixed thread-local buffer (no allocation of any kind on this path) ------------------------------
static thread_local char g_static_err[256] = "";
static int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_static_err, sizeof(g_static_err), fmt, ap);
  va_end(ap);
  return code;
}
extern "C" const char* apd_static_last_error(void) { return g_static_err; }

// ---- set-up, once per device ----------------------------------------------------------------------------------------
constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDev { bool ready; unsigned char* scratch; int sm_count; };
static StaticDev g_static_dev[STATIC_MAX_DEVICES];
static std::mutex g_static_mutex;

// The scratch array's DEVICE address on `device`, which must be the current device.
static int static_scratch_of(int device, StaticDev* out) {
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticDev& d = g_static_dev[device];
  if (!d.ready) {
    int major = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return fail(APD_E_CUDA, "apd_assign_static: cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
    if (major != 10)
      return fail(APD_E_ARCH, "apd_assign_static: device %d is compute capability %d.x; this library is built for "
                  "sm_100a only", device, major);
    unsigned char* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess || !p)
      return fail(APD_E_CUDA, "apd_assign_static: cudaGetSymbolAddress(scratch) on device %d: %s", device,
                  cudaGetErrorString(e));
    d.scratch = p; d.sm_count = sms; d.ready = true;
  }
  *out = d;
  return APD_OK;
}

extern "C" int64_t apd_static_scratch_bytes(void) { return (int64_t)ST_BYTES; }

extern "C" int apd_assign_static(const apd_grid* grid, int32_t M, const float* X, const float* A, const float* w,
                                 const float* target_vol, int32_t* labels, double* vol, double* dual,
                                 double* max_rel_err, void* cuda_stream) {
  g_static_err[0] = 0;
  if (!grid) return fail(APD_E_ARG, "apd_assign_static: grid is NULL");
  if (grid->dim != 2 && grid->dim != 3) return fail(APD_E_ARG, "apd_assign_static: grid.dim must be 2 or 3");
  if (M < 1) return fail(APD_E_ARG, "apd_assign_static: M must be >= 1");
  if (M > STATIC_MAX_SEEDS)
    return fail(APD_E_ARG, "apd_assign_static: M = %d exceeds the static scratch's maximum of %d seeds (use apd_assign)",
                (int)M, STATIC_MAX_SEEDS);
  if (!X || !A || !w || !vol || !dual) return fail(APD_E_ARG, "apd_assign_static: X, A, w, vol and dual are required");
  if (max_rel_err && !target_vol) return fail(APD_E_ARG, "apd_assign_static: max_rel_err needs target_vol");

  int device = -1;
  cudaError_t ce = cudaGetDevice(&device);
  if (ce != cudaSuccess) return fail(APD_E_CUDA, "apd_assign_static: cudaGetDevice: %s", cudaGetErrorString(ce));
  if (device < 0 || device >= STATIC_MAX_DEVICES)
    return fail(APD_E_ARG, "apd_assign_static: device index %d outside [0, %d)", device, STATIC_MAX_DEVICES);
  StaticDev sd;
  const int rc = static_scratch_of(device, &sd);
  if (rc != APD_OK) return rc;

  // grid -> tiles, exactly as apd_assign does (make_grid reads only dim and sm_count of the context it is given)
  apd_ctx shape;
  shape.ws.dim = grid->dim; shape.ws.sm_count = sd.sm_count;
  GridDev g;
  const std::string ge = make_grid(&shape, grid, APD_KERNEL_ROWPOLY, false, &g);
  if (!ge.empty()) return fail(APD_E_ARG, "apd_assign_static: %s", ge.c_str());
  const long long n_tiles = (long long)g.tiles_x * g.tiles_y * g.tiles_z;
  const LayerMap lm = layer_map(g, false);
  if (n_tiles > STATIC_MAX_TILES)
    return fail(APD_E_ARG, "apd_assign_static: the grid needs %lld CTA tiles, the static scratch holds %d (about 64 M "
                "voxels; use apd_assign)", n_tiles, STATIC_MAX_TILES);
  if (lm.n_layers > STATIC_MAX_LAYERS)
    return fail(APD_E_ARG, "apd_assign_static: the grid has %d layers along its last axis, the static scratch holds %d "
                "(use apd_assign)", lm.n_layers, STATIC_MAX_LAYERS);

  float* seeds = reinterpret_cast<float*>(sd.scratch + ST_SEEDS_OFF);
  unsigned int* count = reinterpret_cast<unsigned int*>(sd.scratch + ST_COUNT_OFF);
  double* dual_partial = reinterpret_cast<double*>(sd.scratch + ST_PARTIAL_OFF);
  double* layer_buf = reinterpret_cast<double*>(sd.scratch + ST_LAYER_OFF);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int M_pad = (M + SEED_CHUNK - 1) / SEED_CHUNK * SEED_CHUNK;

  // The array keeps the last call's contents.  What must start at zero is the count histogram (the kernel adds into
  // it): pack_pairs zeroes count[0, M) on the stream before the voxel x seed kernel runs.  The seed table is rewritten
  // for [0, M_pad), every tile writes its own partial, finalize writes every layer sum before it reads them.
  ce = launch_pack_pairs(g.dim, M, M_pad, X, A, w, seeds, count, nullptr, nullptr, st);
  if (ce != cudaSuccess) return fail(APD_E_CUDA, "apd_assign_static: pack_pairs: %s", cudaGetErrorString(ce));
  AssignArgs a;
  a.g = g; a.M = M; a.M_pad = M_pad; a.seeds = seeds; a.labels = labels; a.count = count;
  a.labels_vec = (reinterpret_cast<uintptr_t>(labels) & 15) == 0;
  for (int j = 0; j < 16; ++j) {
    const double tau = ((double)j + 0.5) * g.s[0];
    a.tt[j] = (float)tau;
    a.tt[16 + j] = (float)(tau * tau);
  }
  a.idxsum = nullptr; a.dual_partial = dual_partial;
  a.rec = nullptr; a.brick_list = nullptr; a.brick_count = nullptr; a.super_list = nullptr; a.super_count = nullptr;
  a.super_x = a.super_y = 0; a.pairs_ctr = nullptr; a.done_flag = nullptr; a.qfix = nullptr;
  ce = launch_assign(APD_KERNEL_ROWPOLY, a, st);
  if (ce != cudaSuccess) return fail(APD_E_CUDA, "apd_assign_static: voxel x seed kernel: %s", cudaGetErrorString(ce));
  ce = launch_finalize(g, M, lm, layer_buf, count, nullptr, nullptr, dual_partial, X, w, target_vol, vol, dual,
                       max_rel_err, nullptr, nullptr, nullptr, nullptr, st);
  if (ce != cudaSuccess) return fail(APD_E_CUDA, "apd_assign_static: finalize: %s", cudaGetErrorString(ce));
  return APD_OK;
}
