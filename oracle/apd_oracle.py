"""oracle/apd_oracle.py -- TEST INFRASTRUCTURE, not the product.

fp64 CPU oracle for the APD hot path, written from the paper (arxiv 2403.03571,
PAPER.md) and DESIGN.md's readings.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / ``--impl reference`` legs may import this; the product
path (paper_2403_03571_b200) never does, and this module never imports it.

  oracle_assign  -- the DEFINITION (exact brute force): Algorithm 1
                    plus the discrete dual and gradient, eq. (2.7)-(2.8)
                    and the discrete centroid of Algorithm 3.
                    The O(N*M) loop is oracle/apd_oracle.c; the reductions are here.
  oracle_solve   -- Algorithm 2 step by step; the paper only fixes
                    "W0 = 0, L-BFGS [70], stop when |v_i - m_i|P|| <= eps v_i for all i";
                    the L-BFGS details are DESIGN.md reading S9 and bind this file AND
                    the CUDA path identically.

Pins (tests/test_oracle_pins.py): P1 Voronoi brute force, P2 half-space power diagram,
P3 exact rational arithmetic, P4 concentric ellipse volume, P5 Moebius sphere, P6
tessellation, P7 dual identity, P8 super-gradient / finite differences, P9 concavity,
P10 gauge, P11 exact symmetries, P12 monotonicity, P13 trivial optimum, P14 closed-form
solved weights, P15 post-condition.
PARITY UNPINNED against the paper: L-BFGS iteration/evaluation counts and the particular w
among the valid ones (the paper prints none for a regenerable input) -- see DESIGN.md.
"""
from __future__ import annotations

import ctypes
import dataclasses
import math
import os
import subprocess
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "apd_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_apd.so")
_lib = None

OK = 0
NOT_CONVERGED = 1


def build(force: bool = False) -> str:
    """Compile the C part with gcc (-O2, fp64, OpenMP over voxels; no fast-math)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        p = ctypes.c_void_p
        lib.oracle_apd_assign.restype = ctypes.c_int
        lib.oracle_apd_assign.argtypes = [ctypes.c_int, p, p, p, ctypes.c_int64, p, p, p,
                                          ctypes.c_int64, p, p, p, p, p, p]
        lib.oracle_apd_cost_of.restype = ctypes.c_int
        lib.oracle_apd_cost_of.argtypes = [ctypes.c_int, p, p, p, ctypes.c_int64, p, p, p,
                                           ctypes.c_int64, p, p, p]
        lib.oracle_apd_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_apd_num_threads())


@dataclasses.dataclass
class Grid:
    """Regular discretisation of a box: voxel (ix,iy[,iz]) is centred at
    lo + (i + 1/2) s, s_k = (hi_k - lo_k)/n_k, |P| = prod s_k; linear index j = (iz*ny+iy)*nx+ix
    (x fastest; reading S3)."""
    dim: int
    n: Sequence[int]
    lo: Sequence[float]
    hi: Sequence[float]

    @property
    def N(self) -> int:
        return int(np.prod([int(k) for k in self.n[: self.dim]]))

    @property
    def s(self) -> np.ndarray:
        return (np.asarray(self.hi[: self.dim], dtype=np.float64)
                - np.asarray(self.lo[: self.dim], dtype=np.float64)) / np.asarray(self.n[: self.dim], dtype=np.float64)

    @property
    def voxel_volume(self) -> float:
        return float(np.prod(self.s))

    @property
    def domain_volume(self) -> float:
        return float(np.prod(np.asarray(self.hi[: self.dim], dtype=np.float64)
                             - np.asarray(self.lo[: self.dim], dtype=np.float64)))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _grid_arrays(grid: Grid):
    n = np.ones(3, dtype=np.int64)
    n[: grid.dim] = np.asarray(grid.n[: grid.dim], dtype=np.int64)
    lo = np.zeros(3, dtype=np.float64)
    hi = np.zeros(3, dtype=np.float64)
    lo[: grid.dim] = grid.lo[: grid.dim]
    hi[: grid.dim] = grid.hi[: grid.dim]
    return n, lo, hi


def _widen(X, A, w, dim):
    X = np.ascontiguousarray(np.asarray(X), dtype=np.float64).reshape(-1, dim)   # exact widening of fp32
    M = X.shape[0]
    A = np.ascontiguousarray(np.asarray(A), dtype=np.float64).reshape(M, dim, dim)
    w = np.ascontiguousarray(np.asarray(w), dtype=np.float64).reshape(M)
    return X, A, w, M


@dataclasses.dataclass
class AssignResult:
    labels: np.ndarray            # int32 [n_sel]
    best: np.ndarray              # fp64  min_i C_ij
    qbest: np.ndarray             # fp64  |y_j - x_label|^2_A
    second: Optional[np.ndarray]  # fp64  runner-up cost
    runner: Optional[np.ndarray]  # int32 runner-up index
    count: Optional[np.ndarray] = None     # int64 [M]  m_i
    vol: Optional[np.ndarray] = None       # fp64 [M]   m_i |P|
    dual: Optional[float] = None           # eq. (2.7) literally (None when v is None)
    dual_min_part: Optional[float] = None  # |P| * sum_j min_i C_ij  (= dual - <v,w>, identity I1)
    quad_part: Optional[float] = None      # |P| * sum_j |y_j - x_{H_j}|^2_A
    idxsum: Optional[np.ndarray] = None    # int64 [M, d] sum of voxel indices per cell
    centroids: Optional[np.ndarray] = None  # fp64 [M, d]
    err: Optional[float] = None            # max_i |vol_i - v_i| / v_i  (eq. 2.5)


def oracle_assign(grid: Grid, X, A, w, v=None, sel=None, diagnostics: bool = True) -> AssignResult:
    """Algorithm 1 on the voxels `sel` (all when None) and, when all voxels are evaluated,
    the reductions of eq. (2.7)-(2.8).  X, A, w: the SAME fp32 arrays the GPU gets (widened
    exactly to fp64 here)."""
    lib = _load()
    X, A, w, M = _widen(X, A, w, grid.dim)
    n, lo, hi = _grid_arrays(grid)
    if sel is None:
        n_sel = grid.N
        sel_arr = None
    else:
        sel_arr = np.ascontiguousarray(sel, dtype=np.int64)
        n_sel = sel_arr.size
    labels = np.empty(n_sel, dtype=np.int32)
    best = np.empty(n_sel, dtype=np.float64)
    qbest = np.empty(n_sel, dtype=np.float64)
    second = np.empty(n_sel, dtype=np.float64) if diagnostics else None
    runner = np.empty(n_sel, dtype=np.int32) if diagnostics else None
    rc = lib.oracle_apd_assign(grid.dim, _ptr(n), _ptr(lo), _ptr(hi), M, _ptr(X), _ptr(A), _ptr(w),
                               n_sel, _ptr(sel_arr), _ptr(labels), _ptr(best), _ptr(qbest),
                               _ptr(second), _ptr(runner))
    if rc != 0:
        raise ValueError(f"oracle_apd_assign: bad arguments (rc={rc})")
    res = AssignResult(labels=labels, best=best, qbest=qbest, second=second, runner=runner)
    if sel is not None:
        return res

    # ---- reductions over ALL voxels: eq. (2.7), (2.8), Alg. 3 centroid -----------------
    P = grid.voxel_volume
    count = np.bincount(labels, minlength=M).astype(np.int64)            # m_i
    res.count = count
    res.vol = count.astype(np.float64) * P                               # sum_{H_j=i} |P|, eq. (2.8)
    T = math.fsum(qbest.tolist()) if n_sel <= (1 << 22) else float(np.sum(qbest, dtype=np.longdouble))
    S = math.fsum(best.tolist()) if n_sel <= (1 << 22) else float(np.sum(best, dtype=np.longdouble))
    res.quad_part = P * T
    res.dual_min_part = P * S
    if v is not None:
        v64 = np.asarray(v, dtype=np.float64).reshape(M)
        # eq. (2.7), literally:  sum_i (v_i - vol_i) w_i  +  sum_j |P| |y_j - x_{H_j}|^2
        res.dual = math.fsum(((v64 - res.vol) * w).tolist()) + P * T
        res.err = float(np.max(np.abs(res.vol - v64) / v64))             # eq. (2.5)
    # centroid: x_i <- sum_{H_j=i} |P| y_j / sum_{H_j=i} |P|.  With
    # y = lo + (idx + 1/2) s this is lo + s (idxsum_i / m_i + 1/2); an empty cell keeps x_i (S5).
    d = grid.dim
    nx = int(n[0]); ny = int(n[1])
    j = np.arange(n_sel, dtype=np.int64)
    comps = [j % nx, (j // nx) % ny, j // (nx * ny)]
    idxsum = np.zeros((M, d), dtype=np.int64)
    for k in range(d):
        # integer-valued fp64 weights: every partial sum is an integer < 2^53, hence exact
        idxsum[:, k] = np.bincount(labels, weights=comps[k].astype(np.float64), minlength=M).round().astype(np.int64)
    res.idxsum = idxsum
    cen = X.copy()
    nz = count > 0
    s = grid.s
    for k in range(d):
        cen[nz, k] = lo[k] + s[k] * (idxsum[nz, k] / count[nz] + 0.5)
    res.centroids = cen
    return res


def oracle_cost_of(grid: Grid, X, A, w, sel, seed) -> np.ndarray:
    """fp64 cost C_ij of the named seed i = seed[t] at voxel j = sel[t] (parity rule 1)."""
    lib = _load()
    X, A, w, M = _widen(X, A, w, grid.dim)
    n, lo, hi = _grid_arrays(grid)
    sel = np.ascontiguousarray(sel, dtype=np.int64)
    seed = np.ascontiguousarray(seed, dtype=np.int32)
    out = np.empty(sel.size, dtype=np.float64)
    rc = lib.oracle_apd_cost_of(grid.dim, _ptr(n), _ptr(lo), _ptr(hi), M, _ptr(X), _ptr(A), _ptr(w),
                                sel.size, _ptr(sel), _ptr(seed), _ptr(out))
    if rc != 0:
        raise ValueError(f"oracle_apd_cost_of: bad arguments (rc={rc})")
    return out


# ----------------------------------------------------------------------------------------
# Algorithm 2 with the L-BFGS of DESIGN.md reading S9
# ----------------------------------------------------------------------------------------
@dataclasses.dataclass
class PointSet:
    """A user-supplied discretisation for oracle_solve: points y_j [N,d] with volumes |P_j| [N]."""
    Y: np.ndarray
    pvol: np.ndarray

    @property
    def dim(self) -> int:
        return int(np.asarray(self.Y).shape[1])

    @property
    def domain_volume(self) -> float:
        return float(np.sum(np.asarray(self.pvol, dtype=np.float64)))


@dataclasses.dataclass
class SolveResult:
    status: int                   # OK / NOT_CONVERGED
    w: np.ndarray                 # fp64 iterate
    w32: np.ndarray               # fl32(w): exactly what the final evaluation used
    labels: np.ndarray
    vol: np.ndarray
    iters: int
    evals: int
    err: float
    dual: float
    trajectory: Optional[List[dict]] = None


def _two_loop(g, S_hist, Y_hist, rho, gamma):
    """Liu-Nocedal two-loop recursion [70]: returns H*g with H0 = gamma*I.
    Pinned (tests/test_oracle_lbfgs_pins.py) against the dense BFGS inverse update
    H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T applied from gamma*I, and by finite termination on a
    strictly convex quadratic under exact line minimisation."""
    q = g.copy()
    alphas = []
    for s_i, y_i, r_i in zip(reversed(S_hist), reversed(Y_hist), reversed(rho)):
        a = r_i * float(np.dot(s_i, q))
        alphas.append(a)
        q = q - a * y_i
    r = gamma * q
    for (s_i, y_i, r_i), a in zip(zip(S_hist, Y_hist, rho), reversed(alphas)):
        b = r_i * float(np.dot(y_i, r))
        r = r + s_i * (a - b)
    return r


LS_ACCEPTED, LS_STOP, LS_BUDGET, LS_FAILED = "accepted", "stop", "budget", "failed"


def weak_wolfe_search(phi, f0: float, gp0: float, c1: float = 1e-4, c2: float = 0.9, max_trials: int = 30):
    """The line search of specification S9 on phi(alpha) = f(w + alpha p), as a function of
    its own so that it can be pinned without oracle_assign.
      phi(alpha) -> (f1, gp1, stop, out_of_budget): value, directional derivative g(w + alpha p).p, "the outer
                    stopping test holds at this point" and "no evaluation is left after this one"
      f0, gp0     : phi(0) and phi'(0) < 0
    alpha = 1, lo = 0, hi = inf; per trial: stop -> (LS_STOP, alpha); Armijo fails (f1 > f0 + c1 alpha gp0) ->
    hi = alpha; else curvature fails (gp1 < c2 gp0) -> lo = alpha; else (LS_ACCEPTED, alpha); out of budget ->
    (LS_BUDGET, alpha); next alpha = (lo + hi)/2 when hi is finite, else 2 alpha.  After max_trials: LS_FAILED.
    An accepted alpha satisfies both weak-Wolfe inequalities by construction of the two tests."""
    alpha, lo_a, hi_a = 1.0, 0.0, math.inf
    for _trial in range(max_trials):
        f1, gp1, stop, out_of_budget = phi(alpha)
        if stop:
            return LS_STOP, alpha
        if f1 > f0 + c1 * alpha * gp0:
            hi_a = alpha
        elif gp1 < c2 * gp0:
            lo_a = alpha
        else:
            return LS_ACCEPTED, alpha
        if out_of_budget:
            return LS_BUDGET, alpha
        alpha = 0.5 * (lo_a + hi_a) if math.isfinite(hi_a) else 2.0 * alpha
    return LS_FAILED, alpha


def lbfgs_s9(evaluate, w0: np.ndarray, gamma0: float, eps: float, history: int = 10, max_iters: int = 1000,
             max_evals: Optional[int] = None):
    """Specification S9 as a generic minimiser of f, driven by a callable (oracle_solve passes the APD dual).
      evaluate(w) -> (f, g, err): value, gradient and the quantity the stopping test `err <= eps` is applied to
                     (after EVERY evaluation, S9c)
    Returns (status, w, iters, evals) with status OK (stopping test met at w, the last point evaluated) or
    NOT_CONVERGED (w is then None: the caller keeps track of the best point it saw).
      * direction p = -H g by the two-loop recursion, H0 = gamma I, first gamma = gamma0, then s.y / y.y
      * g.p >= 0: clear the history and take p = -gamma g
      * weak_wolfe_search; on failure clear the history and retry once with p = -gamma g, else NOT_CONVERGED
      * curvature pair kept iff s.y > 1e-12 |s| |y|; at most `history` pairs
    """
    if max_evals is None:
        max_evals = 20 * max_iters
    c1, c2 = 1e-4, 0.9
    w = np.asarray(w0, dtype=np.float64).copy()
    f, g, err = evaluate(w)
    evals, iters = 1, 0
    if err <= eps:
        return OK, w, iters, evals
    gamma = gamma0
    S_hist: List[np.ndarray] = []
    Y_hist: List[np.ndarray] = []
    rho: List[float] = []
    while True:
        p = -_two_loop(g, S_hist, Y_hist, rho, gamma)
        gp = float(np.dot(g, p))
        if gp >= 0.0:
            S_hist, Y_hist, rho = [], [], []
            p = -gamma * g
            gp = float(np.dot(g, p))
        last = {}

        def phi(alpha):
            nonlocal evals
            w_try = w + alpha * p
            f1, g1, err1 = evaluate(w_try)
            evals += 1
            last.update(w=w_try, f=f1, g=g1)
            return f1, float(np.dot(g1, p)), err1 <= eps, evals >= max_evals

        outcome, alpha = weak_wolfe_search(phi, f, gp, c1, c2, 30)
        if outcome == LS_STOP:
            return OK, last["w"], iters + 1, evals
        if outcome == LS_BUDGET:
            return NOT_CONVERGED, None, iters, evals
        if outcome == LS_FAILED:
            if S_hist:
                S_hist, Y_hist, rho = [], [], []
                continue                                  # retry once with p = -gamma g
            return NOT_CONVERGED, None, iters, evals
        w_try, f1, g1 = last["w"], last["f"], last["g"]
        s = alpha * p
        yv = g1 - g
        sy = float(np.dot(s, yv))
        if sy > 1e-12 * math.sqrt(float(np.dot(s, s))) * math.sqrt(float(np.dot(yv, yv))):
            S_hist.append(s); Y_hist.append(yv); rho.append(1.0 / sy)
            if len(S_hist) > history:
                S_hist.pop(0); Y_hist.pop(0); rho.pop(0)
            gamma = sy / float(np.dot(yv, yv))
        w, f, g = w_try, f1, g1
        iters += 1
        if iters >= max_iters or evals >= max_evals:
            return NOT_CONVERGED, None, iters, evals


def oracle_solve(grid: Grid, X, A, v, eps: float, w_init=None, history: int = 10,
                 max_iters: int = 1000, max_evals: Optional[int] = None,
                 record: bool = False) -> SolveResult:
    """Maximise g~ (eq. 2.7) <=> minimise f = -g~ from W0 = 0 (Alg. 2 step 2) with L-BFGS,
    stop when max_i |vol_i - v_i|/v_i <= eps (Alg. 2 step 3, eq. 2.5; '<=' is reading S7).
    Specification S9 (shared with the CUDA path; the optimiser itself is lbfgs_s9 above):
      * fp64 optimiser state; every evaluation uses fl32(w) (round-to-nearest-even), S10
      * f = -g~(fl32 w), grad f = vol - v  (eq. 2.8 with the sign of f)
      * first-direction scale gamma = l^(2-d)/d, l = (|Omega|/M)^(1/d)  (S9a)
      * weak-Wolfe bracketing line search, c1 = 1e-4, c2 = 0.9, alpha0 = 1, <= 30 trials:
        Armijo fails -> hi = alpha; curvature fails -> lo = alpha; alpha = (lo+hi)/2 or 2 alpha
      * stopping test after EVERY evaluation (S9c)
      * curvature pair kept iff s.y > 1e-12 |s||y|; then gamma = s.y / y.y
      * line-search failure: clear the history and retry once with p = -gamma g; else NOT_CONVERGED
      * NOT_CONVERGED returns the evaluated point with the smallest err.
    """
    d = grid.dim
    M = np.asarray(X).reshape(-1, d).shape[0]
    v64 = np.asarray(v, dtype=np.float64).reshape(M)
    traj: Optional[List[dict]] = [] if record else None
    best = {"err": math.inf}
    last = {}

    def evaluate(wd):
        w32 = wd.astype(np.float32)                     # RNE rounding, S10
        if isinstance(grid, PointSet):                  # user-supplied discretisation
            r = oracle_assign_points(grid.Y, grid.pvol, X, A, w32, v=v64)
        else:
            r = oracle_assign(grid, X, A, w32, v=v64, diagnostics=False)
        f = -r.dual
        g = r.vol - v64
        if r.err < best["err"]:
            best.update(err=r.err, w=wd.copy(), w32=w32.copy(), labels=r.labels, vol=r.vol, dual=r.dual)
        if traj is not None:
            traj.append(dict(tag="init" if not traj else "ls", w=wd.copy(), f=f, err=r.err))
        last.update(w32=w32, r=r)
        return f, g, r.err

    w0 = np.zeros(M, dtype=np.float64) if w_init is None else np.asarray(w_init, dtype=np.float64).copy()
    ell = (grid.domain_volume / M) ** (1.0 / d)
    gamma0 = ell ** (2 - d) / d
    status, w, iters, evals = lbfgs_s9(evaluate, w0, gamma0, eps, history=history, max_iters=max_iters,
                                       max_evals=max_evals)
    if status == OK:
        r = last["r"]
        return SolveResult(status=OK, w=w, w32=last["w32"], labels=r.labels, vol=r.vol, iters=iters, evals=evals,
                           err=r.err, dual=r.dual, trajectory=traj)
    return SolveResult(status=NOT_CONVERGED, w=best["w"], w32=best["w32"], labels=best["labels"], vol=best["vol"],
                       iters=iters, evals=evals, err=best["err"], dual=best["dual"], trajectory=traj)


# ----------------------------------------------------------------------------------------
# Algorithm 3, generalised Lloyd, and the resolution rules
# ----------------------------------------------------------------------------------------
def oracle_lloyd(grid: Grid, X0, A, v, eps: float, K: int, w_init=None, **solve_kw):
    """K rounds of { Algorithm 2 from W_0^k ; x_i^{k+1} = discrete centroid of cell i ;
    W_0^{k+1} = W^k }, then a final Algorithm 2 (step 8).  Seeds are fp32 inputs of every round
    (the centroid is rounded to fp32, as the CUDA path does); an empty cell keeps its seed (reading S5); a round
    that ends NOT_CONVERGED continues from its best iterate.  Returns (X^K fp32, final SolveResult, iters, evals)."""
    d = grid.dim
    X = np.ascontiguousarray(np.asarray(X0, dtype=np.float32).reshape(-1, d)).copy()
    w0 = w_init
    iters = evals = 0
    for k in range(K + 1):
        r = oracle_solve(grid, X, A, v, eps, w_init=w0, **solve_kw)
        iters += r.iters
        evals += r.evals
        if k == K:
            return X, r, iters, evals
        if isinstance(grid, PointSet):      # user-supplied discretisation: centroid over the cell's points
            c = oracle_assign_points(grid.Y, grid.pvol, X, A, r.w32, v=v).centroids
        else:
            c = oracle_assign(grid, X, A, r.w32, v=v, diagnostics=False).centroids
        X = np.ascontiguousarray(c.astype(np.float32))
        w0 = r.w32


def resolution_bound(dim: int, domain_volume: float, v_min: float, eps: float, practical: bool) -> float:
    """The real number M must exceed: |Omega|/M^D < eps v_min (eq. 2.9 when v_min = |Omega|/N) or
    |Omega|/M^D < (eps/2^D) v_min (eq. 2.10)."""
    factor = eps / (2 ** dim) if practical else eps
    return (domain_volume / (factor * v_min)) ** (1.0 / dim)


def choose_resolution(dim: int, domain_volume: float, v_min: float, eps: float, practical: bool) -> int:
    """Smallest integer M satisfying the strict inequality, by direct search (no closed form trusted)."""
    factor = eps / (2 ** dim) if practical else eps
    m = 1
    while not (domain_volume / float(m) ** dim < factor * v_min):
        m += 1
    return m


def oracle_solve_refine(grid: Grid, X, A, v, eps: float, max_refinements: int, w_init=None, **solve_kw):
    """Algorithm 2 with its step 4: while Algorithm 2 ends NOT_CONVERGED, double the voxels per axis
    (reading S18: the paper gives no rule) and restart from the best weights found so far.
    Returns (final Grid, SolveResult of the last solve, refinements, total iters, total evals)."""
    w0 = w_init
    iters = evals = 0
    r = 0
    while True:
        res = oracle_solve(grid, X, A, v, eps, w_init=w0, **solve_kw)
        iters += res.iters
        evals += res.evals
        if res.status != NOT_CONVERGED or r == max_refinements:
            return grid, res, r, iters, evals
        if np.prod([2 * k for k in grid.n], dtype=np.float64) >= 2.0 ** 31:
            return grid, res, r, iters, evals
        grid = Grid(grid.dim, tuple(2 * k for k in grid.n), grid.lo, grid.hi)
        w0 = res.w32
        r += 1


def oracle_solve_continuation(grid: Grid, X, A, v, eps: float, levels: int, w_init=None, **solve_kw):
    """Coarse-to-fine continuation (an extension of Alg. 2 step 4; reading S18b): Algorithm 2 on
    the grid coarsened by 2^levels, ..., 2, 1 per axis (n_k -> ceil(n_k / 2^l); a level with some n_k < 16 is skipped),
    each level from the fp32 weights of the one before (a NOT_CONVERGED level hands on its best iterate); a coarse
    level's tolerance is eps_l = max(eps, 2^D |P_l| / v_min), the last level's is eps.
    Returns (SolveResult of the last level = on `grid`, [iters per level], [evals per level]), coarsest first."""
    w0 = w_init
    iters, evals, res = [], [], None
    v_min = float(np.min(np.asarray(v, dtype=np.float32).astype(np.float64)))
    for l in range(levels, -1, -1):
        n = tuple((int(k) + (1 << l) - 1) >> l for k in grid.n[: grid.dim])
        if l > 0 and min(n) < 16:
            iters.append(0); evals.append(0)
            continue
        g_l = Grid(grid.dim, n, grid.lo, grid.hi)
        # a coarse level is asked only for what its voxels can resolve: eq. (2.10) read backwards
        eps_l = eps if l == 0 else max(eps, 2.0 ** grid.dim * g_l.voxel_volume / v_min)
        res = oracle_solve(g_l, X, A, v, eps_l, w_init=w0, **solve_kw)
        iters.append(res.iters); evals.append(res.evals)
        w0 = res.w32
    return res, iters, evals


# ----------------------------------------------------------------------------------------
# user-supplied discretisation: points y_j with volumes |P_j|
# ----------------------------------------------------------------------------------------
@dataclasses.dataclass
class PointsResult:
    labels: np.ndarray        # [N] argmin, lowest index on ties
    best: np.ndarray          # [N] min_i C_ij
    second: np.ndarray        # [N] runner-up cost (inf if M == 1)
    vol: np.ndarray           # [M] sum of |P_j| over the cell
    dual: float               # eq. (2.7) with element volumes, literally
    dual_min_part: float      # sum_j |P_j| min_i C_ij
    centroids: np.ndarray     # [M,d]
    err: float


def oracle_assign_points(Y, pvol, X, A, w, v=None, chunk: int = 4096) -> PointsResult:
    """The definition with element volumes: C_ij = (y_j - x_i)^T A_i (y_j - x_i) - w_i, all d^2
    terms, fp64; H_j = lowest argmin; vol_i = sum_{H_j=i} |P_j|;
    g~ = sum_i [(v_i - vol_i) w_i + sum_{H_j=i} |P_j| |y_j - x_i|^2_{A_i}]  (eq. 2.7 with |P| -> |P_j|);
    centroid_i = sum |P_j| y_j / vol_i, the seed itself for an empty cell (reading S5)."""
    Y = np.asarray(Y, dtype=np.float64)
    N, d = Y.shape
    X = np.asarray(X, dtype=np.float64).reshape(-1, d)
    M = X.shape[0]
    A = np.asarray(A, dtype=np.float64).reshape(M, d, d)
    w = np.asarray(w, dtype=np.float64).reshape(M)
    p = np.asarray(pvol, dtype=np.float64).reshape(N)
    labels = np.empty(N, dtype=np.int64); best = np.empty(N); second = np.full(N, np.inf); qbest = np.empty(N)
    for j0 in range(0, N, chunk):
        D = Y[j0:j0 + chunk, None, :] - X[None, :, :]                        # [n, M, d]
        q = np.einsum("nmk,mkl,nml->nm", D, A, D)                            # all d^2 terms (S13)
        c = q - w[None, :]
        lab = np.argmin(c, axis=1)                                           # first minimum = lowest index (S1)
        r = np.arange(c.shape[0])
        labels[j0:j0 + chunk] = lab; best[j0:j0 + chunk] = c[r, lab]; qbest[j0:j0 + chunk] = q[r, lab]
        if M > 1:
            c2 = c.copy(); c2[r, lab] = np.inf
            second[j0:j0 + chunk] = c2.min(axis=1)
    vol = np.bincount(labels, weights=p, minlength=M)
    T = float(np.sum(p * qbest))
    v64 = np.zeros(M) if v is None else np.asarray(v, dtype=np.float64).reshape(M)
    dual = float(np.sum((v64 - vol) * w)) + T
    cen = np.empty((M, d))
    for k in range(d):
        num = np.bincount(labels, weights=p * Y[:, k], minlength=M)
        cen[:, k] = np.where(vol > 0, num / np.where(vol > 0, vol, 1.0), X[:, k])
    err = float(np.max(np.abs(vol - v64) / v64)) if v is not None else float("nan")
    return PointsResult(labels=labels, best=best, second=second, vol=vol, dual=dual,
                        dual_min_part=float(np.sum(p * best)), centroids=cen, err=err)
