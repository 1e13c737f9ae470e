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
// The whole state machine is ONE single-CTA kernel (lbfgs_step_kernel) that runs after each
// evaluation on the same stream; the host only reads the mapped SolveReport.done word.
#include "apd_internal.cuh"
#include "apd_device.cuh"
#include <cmath>
#include <vector>

namespace apd {

constexpr int LB_THREADS = 1024;
constexpr int LB_MAX_HIST = 64;
constexpr int LB_MAX_TRIALS = 30;

struct SolveState {
  int done, phase, iters, evals, trial, hist_len, hist_start, hist_cap, max_iters, max_evals;
  double f, gp, alpha, lo, hi, gamma, eps, best_err, best_dual, domain_volume;
  double rho[LB_MAX_HIST];
  // candidate-list reuse (apd_cull.cu): the lists were built at wref with slack cull_delta and stay valid while
  // max_i |w32_i - wref_i| <= cull_delta
  int cull_rebuild, cull_rebuilds;
  float cull_delta, cull_cap;
};

enum { V_W = 0, V_G, V_P, V_WTRY, V_WBEST, V_GNEW, V_Q, V_HIST };   // rows of svec

struct StepArgs {
  SolveState* st;
  double* vec;         // [(V_HIST + 2 hist_cap) * stride]
  int stride;          // = max_seeds
  int M;
  const float* v;      // target volumes
  const double* e_vol; // evaluation outputs
  const double* e_scal;  // [0] dual, [1] max_rel_err
  float* w32;          // next evaluation's weights
  SolveReport* report; // mapped host memory
  double* hist;        // [2 * hist_cap] (dual, max_rel_err) of every evaluation, in order
  int hist_cap;
  float* wref;         // weights the candidate lists were built at (culling only)
};

constexpr double CULL_DELTA_FACTOR = 4.0;   // slack of a rebuilt list = this x the last change of the weights ...
constexpr double CULL_CAP_FACTOR = 0.5;     // ... but at most this x the mean min-cost of the first evaluation (a larger
                                            // slack would lengthen every list by more than it saves in rebuilds)

// Sum over the block, identical value returned to every thread; fixed order.
__device__ __forceinline__ double block_allsum(double v, double* scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();                       // scratch free
  if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
#pragma unroll
  for (int i = 0; i < LB_THREADS / 32; ++i) t += scratch[i];
  return t;
}

__device__ __forceinline__ double block_allmax(double v, double* scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  __syncthreads();
  if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
#pragma unroll
  for (int i = 0; i < LB_THREADS / 32; ++i) t = fmax(t, scratch[i]);
  return t;
}

__device__ __forceinline__ double block_dot(const double* a, const double* b, int M, double* scratch) {
  double p = 0.0;
  for (int i = threadIdx.x; i < M; i += LB_THREADS) p += a[i] * b[i];
  return block_allsum(p, scratch);
}

// p = -H g (two-loop recursion of Liu & Nocedal [70], H0 = gamma I); returns g.p to all threads.
__device__ double new_direction(const StepArgs& a, SolveState* st, int hist_len, int hist_start, double gamma,
                                double* scratch, double* s_alpha) {
  const int M = a.M, stride = a.stride, cap = st->hist_cap;
  double* g = a.vec + (size_t)V_G * stride;
  double* p = a.vec + (size_t)V_P * stride;
  double* q = a.vec + (size_t)V_Q * stride;
  double* S = a.vec + (size_t)V_HIST * stride;
  double* Y = S + (size_t)cap * stride;
  for (int i = threadIdx.x; i < M; i += LB_THREADS) q[i] = g[i];
  for (int t = hist_len - 1; t >= 0; --t) {              // newest -> oldest
    const int slot = (hist_start + t) % cap;
    const double al = st->rho[slot] * block_dot(S + (size_t)slot * stride, q, M, scratch);
    if (threadIdx.x == 0) s_alpha[t] = al;
    const double* y = Y + (size_t)slot * stride;
    for (int i = threadIdx.x; i < M; i += LB_THREADS) q[i] = __dsub_rn(q[i], __dmul_rn(al, y[i]));
  }
  for (int i = threadIdx.x; i < M; i += LB_THREADS) q[i] = __dmul_rn(gamma, q[i]);
  __syncthreads();                                        // s_alpha visible
  for (int t = 0; t < hist_len; ++t) {                    // oldest -> newest
    const int slot = (hist_start + t) % cap;
    const double be = st->rho[slot] * block_dot(Y + (size_t)slot * stride, q, M, scratch);
    const double coef = s_alpha[t] - be;
    const double* s = S + (size_t)slot * stride;
    for (int i = threadIdx.x; i < M; i += LB_THREADS) q[i] = __dadd_rn(q[i], __dmul_rn(s[i], coef));
  }
  for (int i = threadIdx.x; i < M; i += LB_THREADS) p[i] = -q[i];
  return block_dot(g, p, M, scratch);
}

__global__ void solve_init_kernel(StepArgs a, const float* w_init, int hist_cap, int max_iters, int max_evals,
                                  double eps, double gamma0, double domain_volume) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < a.M) {
    const double w = w_init ? (double)w_init[i] : 0.0;     // Alg. 2 step 2: W0 = 0
    a.vec[(size_t)V_W * a.stride + i] = w;
    a.w32[i] = (float)w;
    a.wref[i] = (float)w;
  }
  if (i == 0) {
    SolveState* st = a.st;
    st->cull_rebuild = 1; st->cull_rebuilds = 1; st->cull_delta = 0.0f; st->cull_cap = 0.0f;
    st->done = 0; st->phase = 0; st->iters = 0; st->evals = 0; st->trial = 0;
    st->hist_len = 0; st->hist_start = 0; st->hist_cap = hist_cap;
    st->max_iters = max_iters; st->max_evals = max_evals;
    st->f = 0.0; st->gp = 0.0; st->alpha = 1.0; st->lo = 0.0; st->hi = INFINITY;
    st->gamma = gamma0; st->eps = eps; st->best_err = INFINITY; st->best_dual = 0.0;
    st->domain_volume = domain_volume;
    a.report->done = 0; a.report->status = APD_OK; a.report->iters = 0; a.report->evals = 0;
    a.report->err = 0.0; a.report->dual = 0.0; a.report->cull_rebuilds = 0;
  }
}

// Runs after every evaluation.  Control flow is uniform over the CTA: every decision is taken on
// values all threads hold identically (block_allsum results, state scalars read after a sync).
__global__ void __launch_bounds__(LB_THREADS) lbfgs_step_kernel(StepArgs a) {
  __shared__ double scratch[LB_THREADS / 32];
  __shared__ double s_alpha[LB_MAX_HIST];
  SolveState* st = a.st;
  if (st->done) return;
  const int M = a.M, stride = a.stride, tid = threadIdx.x;
  double* w = a.vec + (size_t)V_W * stride;
  double* g = a.vec + (size_t)V_G * stride;
  double* p = a.vec + (size_t)V_P * stride;
  double* wtry = a.vec + (size_t)V_WTRY * stride;
  double* wbest = a.vec + (size_t)V_WBEST * stride;
  double* gnew = a.vec + (size_t)V_GNEW * stride;
  double* S = a.vec + (size_t)V_HIST * stride;
  double* Y = S + (size_t)st->hist_cap * stride;

  // copy the scalars (all threads read the same global values before anyone writes them)
  const int phase = st->phase;
  int iters = st->iters, evals = st->evals, trial = st->trial, hist_len = st->hist_len, hist_start = st->hist_start;
  const int cap = st->hist_cap, max_iters = st->max_iters, max_evals = st->max_evals;
  double f = st->f, gp = st->gp, alpha = st->alpha, lo = st->lo, hi = st->hi, gamma = st->gamma;
  const double eps = st->eps;
  double best_err = st->best_err, best_dual = st->best_dual;
  const double f1 = -a.e_scal[0], err1 = a.e_scal[1];
  __syncthreads();

  // gradient of f at the evaluated point: vol - v (eq. 2.8)
  double vsum = 0.0;
  for (int i = tid; i < M; i += LB_THREADS) {
    const double tv = (double)a.v[i];
    gnew[i] = a.e_vol[i] - tv;
    vsum += tv;
  }
  evals += 1;
  if (tid == 0 && evals <= a.hist_cap) { a.hist[2 * (evals - 1)] = -f1; a.hist[2 * (evals - 1) + 1] = err1; }
  const double* w_eval = (phase == 0) ? w : wtry;
  if (err1 < best_err) {
    best_err = err1; best_dual = -f1;
    for (int i = tid; i < M; i += LB_THREADS) wbest[i] = w_eval[i];
  }

  int finish = 0;          // 1: OK at w_eval, 2: NOT_CONVERGED at best, 3: bad target volumes
  bool need_direction = false;
  float cull_cap = st->cull_cap;
  if (phase == 0) {
    // cost scale for the list-reuse slack: mean over the voxels of min_i C_ij = (g~ - <v, w>) / |Omega|  (identity I1)
    double vw = 0.0;
    for (int i = tid; i < M; i += LB_THREADS) vw += (double)a.v[i] * (double)a.w32[i];
    vw = block_allsum(vw, scratch);
    const double scale = fabs(a.e_scal[0] - vw) / st->domain_volume;
    cull_cap = isfinite(scale) ? (float)(CULL_CAP_FACTOR * scale) : 0.0f;
    vsum = block_allsum(vsum, scratch);
    if (!(fabs(vsum - st->domain_volume) <= 1e-5 * st->domain_volume)) finish = 3;
    else if (err1 <= eps) finish = 1;
    else {
      f = f1;
      for (int i = tid; i < M; i += LB_THREADS) g[i] = gnew[i];
      need_direction = true;
    }
  } else {
    if (err1 <= eps) { finish = 1; iters += 1; }
    else {
      bool accepted = false;
      const double armijo_rhs = __dadd_rn(f, __dmul_rn(__dmul_rn(1e-4, alpha), gp));
      if (f1 > armijo_rhs) hi = alpha;
      else if (block_dot(gnew, p, M, scratch) < __dmul_rn(0.9, gp)) lo = alpha;
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
        // s = alpha p, yv = g1 - g  -> candidate curvature pair in the next ring slot
        const int slot = (hist_len < cap) ? (hist_start + hist_len) % cap : hist_start;
        double* s_new = S + (size_t)slot * stride;
        double* y_new = Y + (size_t)slot * stride;
        double sy = 0.0, ss = 0.0, yy = 0.0;
        // the pair is first formed in q/gnew-independent temporaries: when the ring is full the
        // slot being overwritten is the oldest pair, which is dropped only if the new one is kept
        double* q = a.vec + (size_t)V_Q * stride;
        for (int i = tid; i < M; i += LB_THREADS) {
          const double si = __dmul_rn(alpha, p[i]);
          const double yi = __dsub_rn(gnew[i], g[i]);
          q[i] = si;
          sy += si * yi; ss += si * si; yy += yi * yi;
        }
        sy = block_allsum(sy, scratch);
        ss = block_allsum(ss, scratch);
        yy = block_allsum(yy, scratch);
        if (sy > 1e-12 * sqrt(ss) * sqrt(yy)) {
          for (int i = tid; i < M; i += LB_THREADS) {
            s_new[i] = q[i];
            y_new[i] = __dsub_rn(gnew[i], g[i]);
          }
          if (tid == 0) st->rho[slot] = 1.0 / sy;
          if (hist_len < cap) hist_len += 1; else hist_start = (hist_start + 1) % cap;
          gamma = sy / yy;
        }
        for (int i = tid; i < M; i += LB_THREADS) { w[i] = wtry[i]; g[i] = gnew[i]; }
        f = f1;
        iters += 1;
        if (iters >= max_iters || evals >= max_evals) finish = 2;
        else need_direction = true;
      }
    }
  }

  if (need_direction) {
    __syncthreads();    // rho / history writes visible
    gp = new_direction(a, st, hist_len, hist_start, gamma, scratch, s_alpha);
    if (gp >= 0.0) {    // safeguard: not a descent direction -> steepest descent scaled by gamma
      hist_len = 0; hist_start = 0;
      gp = new_direction(a, st, 0, 0, gamma, scratch, s_alpha);
    }
    alpha = 1.0; lo = 0.0; hi = INFINITY; trial = 0;
  }

  int cull_rebuild = 1;
  float cull_delta = 0.0f;
  if (finish == 0) {
    // next trial point w + alpha p, rounded to fp32 for the evaluation (S10)
    double step_max = 0.0, ref_max = 0.0;   // max |change since the last evaluation|, max |distance from wref|
    for (int i = tid; i < M; i += LB_THREADS) {
      const double wt = __dadd_rn(w[i], __dmul_rn(alpha, p[i]));
      wtry[i] = wt;
      const float wn = (float)wt;
      step_max = fmax(step_max, fabs((double)wn - (double)a.w32[i]));     // differences of floats: exact in fp64
      ref_max = fmax(ref_max, fabs((double)wn - (double)a.wref[i]));
      a.w32[i] = wn;
    }
    step_max = block_allmax(step_max, scratch);
    ref_max = block_allmax(ref_max, scratch);
    cull_delta = st->cull_delta;
    cull_rebuild = !(ref_max <= (double)cull_delta);
    if (cull_rebuild) {
      // the next evaluation rebuilds its candidate lists at the new weights, valid within delta of them
      cull_delta = fminf((float)(CULL_DELTA_FACTOR * step_max), cull_cap);
      for (int i = tid; i < M; i += LB_THREADS) a.wref[i] = a.w32[i];
    }
  } else if (finish == 1) {
    if (phase != 0) for (int i = tid; i < M; i += LB_THREADS) w[i] = wtry[i];
  } else if (finish == 2) {
    for (int i = tid; i < M; i += LB_THREADS) { w[i] = wbest[i]; a.w32[i] = (float)wbest[i]; }
  }
  __syncthreads();
  if (tid == 0) {
    st->phase = 1; st->iters = iters; st->evals = evals; st->trial = trial;
    st->hist_len = hist_len; st->hist_start = hist_start;
    st->f = f; st->gp = gp; st->alpha = alpha; st->lo = lo; st->hi = hi; st->gamma = gamma;
    st->best_err = best_err; st->best_dual = best_dual;
    st->cull_cap = cull_cap; st->cull_rebuild = cull_rebuild; st->cull_delta = cull_delta; st->cull_rebuilds += (finish == 0 && cull_rebuild);
    if (finish) {
      st->done = 1;
      a.report->status = (finish == 1) ? APD_OK : (finish == 2 ? APD_NOT_CONVERGED : APD_E_ARG);
      a.report->iters = iters; a.report->evals = evals;
      a.report->err = (finish == 2) ? best_err : err1;
      a.report->dual = (finish == 2) ? best_dual : -f1;
      a.report->cull_rebuilds = st->cull_rebuilds;
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

static int ensure_solve_state(apd_ctx* ctx, int hist) {
  Workspace& ws = ctx->ws;
  const size_t ms = (size_t)ws.max_seeds;
  if (!ws.sstate) {
    LB_TRY(cudaMalloc(&ws.sstate, sizeof(SolveState)));
    LB_TRY(cudaMalloc(&ws.w32, ms * sizeof(float)));
    LB_TRY(cudaMalloc(&ws.wref, ms * sizeof(float)));
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
    ws.svec_hist = hist;
  }
  return APD_OK;
}

extern "C" int apd_solve(apd_ctx* ctx, const apd_grid* grid, int32_t M, const float* X, const float* A,
                         const float* target_vol, double tol, const float* w_init, float* w, int32_t* labels,
                         double* vol, double* w64, int32_t* iters, int32_t* evals, double* max_rel_err,
                         double* dual, const apd_opts* opts, void* cuda_stream) {
  if (!ctx) return APD_E_ARG;
  ctx->err.clear();
  std::string e;
  const int kernel = resolve_kernel(opts, &e);
  if (kernel < 0) { ctx->err = "apd_solve: " + e; return APD_E_ARG; }
  if (M < 1 || M > ctx->ws.max_seeds) { ctx->err = "apd_solve: M out of range [1, max_seeds]"; return APD_E_ARG; }
  if (!X || !A || !target_vol || !w) { ctx->err = "apd_solve: X, A, target_vol and w are required"; return APD_E_ARG; }
  if (!(tol > 0.0) || !std::isfinite(tol)) { ctx->err = "apd_solve: tol must be finite and > 0"; return APD_E_ARG; }
  apd_opts o;
  apd_default_opts(&o);
  if (opts) o = *opts;
  if (o.lbfgs_history < 1 || o.lbfgs_history > LB_MAX_HIST) { ctx->err = "apd_solve: lbfgs_history must be in [1,64]"; return APD_E_ARG; }
  if (o.max_iters < 1 || o.max_evals < 0) { ctx->err = "apd_solve: max_iters >= 1 and max_evals >= 0 required"; return APD_E_ARG; }
  const int max_evals = o.max_evals ? o.max_evals : (o.max_iters > (1 << 26) ? (1 << 30) : 20 * o.max_iters);
  GridDev g;
  e = make_grid(ctx, grid, kernel, o.cull != 0, &g);
  if (!e.empty()) { ctx->err = "apd_solve: " + e; return APD_E_ARG; }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  LB_TRY(cudaSetDevice(ctx->ws.device));
  int rc = ensure_solve_state(ctx, o.lbfgs_history);
  if (rc != APD_OK) return rc;
  Workspace& ws = ctx->ws;

  double domain = 1.0;
  for (int k = 0; k < g.dim; ++k) domain *= (grid->hi[k] - grid->lo[k]);
  const double ell = std::pow(domain / (double)M, 1.0 / (double)g.dim);
  const double gamma0 = std::pow(ell, (double)(2 - g.dim)) / (double)g.dim;

  StepArgs sa;
  sa.st = ws.sstate; sa.vec = ws.svec; sa.stride = ws.max_seeds; sa.M = M; sa.v = target_vol;
  sa.e_vol = ws.e_vol; sa.e_scal = ws.e_scal; sa.w32 = ws.w32;
  sa.hist = ws.hist; sa.hist_cap = SOLVE_HIST_CAP; sa.wref = ws.wref;
  ws.hist_len = 0;
  SolveReport* dev_report = nullptr;
  LB_TRY(cudaHostGetDevicePointer((void**)&dev_report, ws.report, 0));
  sa.report = dev_report;
  ws.report->done = 0;
  solve_init_kernel<<<(M + 255) / 256, 256, 0, st>>>(sa, w_init, o.lbfgs_history, o.max_iters, max_evals, tol,
                                                    gamma0, domain);
  LB_TRY(cudaGetLastError());

  const int* done_flag = &ws.sstate->done;
  long long enq = 0;
  const long long hard_cap = (long long)max_evals + 64;
  for (;; ++enq) {
    rc = enqueue_evaluation(ctx, g, kernel, M, X, A, ws.w32, target_vol, nullptr, ws.e_vol, ws.e_scal,
                            ws.e_scal + 1, nullptr, nullptr, false, o.cull != 0, done_flag, st, &ws.sstate->cull_rebuild,
                            &ws.sstate->cull_delta);
    if (rc != APD_OK) return rc;
    lbfgs_step_kernel<<<1, LB_THREADS, 0, st>>>(sa);
    LB_TRY(cudaGetLastError());
    LB_TRY(cudaEventRecord(ws.sev[enq & 1], st));
    if (enq >= 1) {
      // the convergence check: wait for the PREVIOUS evaluation's step while this one runs;
      // kernels enqueued after the optimiser finished see done_flag and return at once
      LB_TRY(cudaEventSynchronize(ws.sev[(enq - 1) & 1]));
      if (ws.report->done) break;
    }
    if (enq > hard_cap) { ctx->err = "apd_solve: optimiser did not report completion"; return APD_E_CUDA; }
  }
  LB_TRY(cudaStreamSynchronize(st));
  const int status = ws.report->status;
  if (status == APD_E_ARG) { ctx->err = "apd_solve: sum(target_vol) differs from |Omega| by more than 1e-5 relative"; return APD_E_ARG; }

  // final evaluation at the returned fp32 weights, with labels (Algorithm 1 at the solution)
  rc = enqueue_evaluation(ctx, g, kernel, M, X, A, ws.w32, target_vol, labels, vol ? vol : ws.e_vol, ws.e_scal,
                          ws.e_scal + 1, nullptr, nullptr, true, o.cull != 0, nullptr, st);
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
