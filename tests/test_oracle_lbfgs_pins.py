"""Pins for the oracle's optimiser (CPU only): the two-loop recursion, the weak-Wolfe bracketing search and the
L-BFGS driver of specification S9 ("L-BFGS [70]", ref [70] at PAPER.md:424),
checked against what the MATHEMATICS fixes -- none of these tests calls oracle_assign:

  P17  two-loop == the dense BFGS inverse update  H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T  applied from
       gamma I (numpy matrices; shares nothing with _two_loop).  A swapped loop order, a wrong sign or s/y exchanged
       fails it.
  P18  finite termination: on a strictly convex quadratic with EXACT line minimisation and full memory, BFGS
       directions are conjugate and the minimum is reached in <= n steps (Nocedal & Wright, Thm 6.4 / 5.x).
  P19  an alpha accepted by weak_wolfe_search satisfies both weak-Wolfe inequalities (c1 = 1e-4, c2 = 0.9); the
       bracketing rules (doubling while hi = inf, bisection after) are followed trial by trial.
  P20  lbfgs_s9 minimises smooth convex functions to the known minimiser, obeys the evaluation / iteration limits and
       stops at the first evaluation that meets the stopping test.
"""
import math

import numpy as np
import pytest

from oracle.apd_oracle import (_two_loop, weak_wolfe_search, lbfgs_s9, OK, NOT_CONVERGED, LS_ACCEPTED, LS_STOP,
                               LS_BUDGET, LS_FAILED)


def dense_bfgs_inverse(S, Y, gamma):
    """H_k from H_0 = gamma I by the textbook inverse update, oldest pair first."""
    n = S[0].size if S else 0
    H = gamma * np.eye(n)
    I = np.eye(n)
    for s, y in zip(S, Y):
        rho = 1.0 / float(y @ s)
        H = (I - rho * np.outer(s, y)) @ H @ (I - rho * np.outer(y, s)) + rho * np.outer(s, s)
    return H


def curvature_pairs(rng, n, m):
    """m pairs with s.y > 0: y = B s for a random SPD B plus a perturbation that keeps the curvature positive."""
    Q = rng.standard_normal((n, n))
    B = Q @ Q.T + n * np.eye(n)
    S, Y = [], []
    while len(S) < m:
        s = rng.standard_normal(n)
        y = B @ s + 0.3 * rng.standard_normal(n)
        if float(s @ y) > 1e-3:
            S.append(s); Y.append(y)
    return S, Y


# ---------------------------------------------------------------- P17
@pytest.mark.parametrize("n,m,seed", [(5, 1, 0), (7, 3, 1), (12, 10, 2), (30, 10, 3), (6, 9, 4)])
def test_P17_two_loop_equals_dense_bfgs_inverse(n, m, seed):
    rng = np.random.default_rng(1700 + seed)
    S, Y = curvature_pairs(rng, n, m)
    rho = [1.0 / float(s @ y) for s, y in zip(S, Y)]
    gamma = float(rng.uniform(0.2, 3.0))
    H = dense_bfgs_inverse(S, Y, gamma)
    for _ in range(3):
        g = rng.standard_normal(n)
        r = _two_loop(g, S, Y, rho, gamma)
        np.testing.assert_allclose(r, H @ g, rtol=1e-12, atol=1e-12 * np.abs(H @ g).max())
    # no history: H = gamma I
    np.testing.assert_array_equal(_two_loop(g, [], [], [], gamma), gamma * g)


def test_P17_mutations_of_the_recursion_are_caught():
    """The pin has teeth: the plausible mistakes (loops in the same order, s and y exchanged, the sign of the
    correction) all move the result away from H g by far more than the tolerance."""
    rng = np.random.default_rng(1717)
    n, m = 9, 4
    S, Y = curvature_pairs(rng, n, m)
    rho = [1.0 / float(s @ y) for s, y in zip(S, Y)]
    gamma, g = 0.7, rng.standard_normal(n)
    Hg = dense_bfgs_inverse(S, Y, gamma) @ g

    def rel(x):
        return float(np.abs(x - Hg).max() / np.abs(Hg).max())

    assert rel(_two_loop(g, S, Y, rho, gamma)) < 1e-12
    assert rel(_two_loop(g, S[::-1], Y[::-1], rho[::-1], gamma)) > 1e-3      # pair order reversed
    assert rel(_two_loop(g, Y, S, rho, gamma)) > 1e-3                        # s and y exchanged
    assert rel(_two_loop(g, S, Y, [-r for r in rho], gamma)) > 1e-3          # sign of rho
    assert rel(-_two_loop(-g, S, Y, rho, gamma)) < 1e-12                     # linear in g


# ---------------------------------------------------------------- P18
@pytest.mark.parametrize("n,seed", [(4, 0), (8, 1), (15, 2)])
def test_P18_finite_termination_on_a_quadratic_with_exact_line_search(n, seed):
    rng = np.random.default_rng(1800 + seed)
    Q = rng.standard_normal((n, n))
    B = Q @ Q.T + np.eye(n)
    b = rng.standard_normal(n)
    x_star = np.linalg.solve(B, b)
    x = rng.standard_normal(n)
    g = B @ x - b
    g0 = float(np.linalg.norm(g))
    S, Y, rho = [], [], []
    dirs = []
    for it in range(n):
        p = -_two_loop(g, S, Y, rho, 1.0)
        assert float(g @ p) < 0.0
        alpha = -float(g @ p) / float(p @ B @ p)           # exact minimiser of the quadratic along p
        s = alpha * p
        x = x + s
        g_new = B @ x - b
        y = g_new - g
        S.append(s); Y.append(y); rho.append(1.0 / float(s @ y))
        dirs.append(p)
        g = g_new
        if np.linalg.norm(g) <= 1e-9 * g0:
            break
    assert np.linalg.norm(g) <= 1e-8 * g0, f"not at the minimum after n = {n} exact steps"
    np.testing.assert_allclose(x, x_star, rtol=1e-7, atol=1e-9)
    # the directions are B-conjugate
    D = np.array(dirs)
    G = D @ B @ D.T
    off = G - np.diag(np.diag(G))
    assert np.abs(off).max() <= 1e-7 * np.abs(np.diag(G)).max()


# ---------------------------------------------------------------- P19
def _phi_of(f, df, w, p):
    def phi(alpha):
        x = w + alpha * p
        return float(f(x)), float(df(x) @ p), False, False
    return phi


@pytest.mark.parametrize("case", ["quadratic_long_step", "quadratic_short_step", "logsumexp", "quartic"])
def test_P19_accepted_step_satisfies_weak_wolfe(case):
    rng = np.random.default_rng(1900)
    n = 6
    if case.startswith("quadratic"):
        Q = rng.standard_normal((n, n)); B = Q @ Q.T + np.eye(n)
        f = lambda x: 0.5 * x @ B @ x
        df = lambda x: B @ x
        w = rng.standard_normal(n)
        scale = 50.0 if case == "quadratic_long_step" else 1e-4     # alpha = 1 far too long / far too short
        p = -scale * df(w)
    elif case == "logsumexp":
        Z = rng.standard_normal((20, n))
        f = lambda x: float(np.log(np.sum(np.exp(Z @ x)))) + 0.5 * float(x @ x)
        df = lambda x: Z.T @ (np.exp(Z @ x) / np.sum(np.exp(Z @ x))) + x
        w = rng.standard_normal(n); p = -3.0 * df(w)
    else:
        f = lambda x: float(np.sum(x ** 4) + 0.5 * np.sum(x ** 2))
        df = lambda x: 4 * x ** 3 + x
        w = 2.0 * rng.standard_normal(n); p = -0.01 * df(w)
    f0, gp0 = float(f(w)), float(df(w) @ p)
    assert gp0 < 0
    trace = []
    inner = _phi_of(f, df, w, p)

    def phi(alpha):
        trace.append(alpha)
        return inner(alpha)

    outcome, alpha = weak_wolfe_search(phi, f0, gp0)
    assert outcome == LS_ACCEPTED and alpha == trace[-1]
    c1, c2 = 1e-4, 0.9
    assert f(w + alpha * p) <= f0 + c1 * alpha * gp0               # sufficient decrease (Armijo)
    assert df(w + alpha * p) @ p >= c2 * gp0                        # weak curvature condition
    # the bracketing rules, replayed from the recorded trial points
    lo, hi = 0.0, math.inf
    assert trace[0] == 1.0
    for a, a_next in zip(trace[:-1], trace[1:]):
        if f(w + a * p) > f0 + c1 * a * gp0:
            hi = a
        else:
            assert df(w + a * p) @ p < c2 * gp0
            lo = a
        assert a_next == (0.5 * (lo + hi) if math.isfinite(hi) else 2.0 * a)
    if case == "quadratic_long_step":
        assert alpha < 1.0 and len(trace) > 1
    if case == "quadratic_short_step":
        assert alpha > 1.0 and len(trace) > 1


def test_P19_search_outcomes_stop_budget_failed():
    # a function that never satisfies Armijo (phi increases): 30 bisections, then LS_FAILED
    calls = []
    out, alpha = weak_wolfe_search(lambda a: (calls.append(a) or (1.0 + a, 1.0, False, False)), 1.0, -1.0)
    assert out == LS_FAILED and len(calls) == 30 and calls[1] == 0.5 and calls[2] == 0.25
    # the stopping test is looked at BEFORE the Wolfe tests (S9c)
    out, alpha = weak_wolfe_search(lambda a: (1e9, 0.0, a == 4.0, False), 0.0, -1.0)
    assert out == LS_FAILED                      # Armijo fails at 1, halving never reaches 4
    out, alpha = weak_wolfe_search(lambda a: (-1e9, -1e9, a == 4.0, False), 0.0, -1.0)
    assert (out, alpha) == (LS_STOP, 4.0)        # curvature fails at 1, 2 -> doubling reaches 4
    # budget: reported after the Wolfe tests of the last affordable evaluation
    out, alpha = weak_wolfe_search(lambda a: (-1e9, -1e9, False, a == 2.0), 0.0, -1.0)
    assert (out, alpha) == (LS_BUDGET, 2.0)
    out, alpha = weak_wolfe_search(lambda a: (-1.0, 0.0, False, True), 0.0, -1.0)
    assert (out, alpha) == (LS_ACCEPTED, 1.0)    # an acceptable point wins over the budget flag


# ---------------------------------------------------------------- P20
def test_P20_driver_minimises_convex_functions_and_respects_limits():
    rng = np.random.default_rng(2000)
    n = 25
    Q = rng.standard_normal((n, n)); B = Q @ Q.T + np.eye(n)
    b = rng.standard_normal(n)
    x_star = np.linalg.solve(B, b)
    n_eval = [0]

    def evaluate(x):
        n_eval[0] += 1
        g = B @ x - b
        return 0.5 * float(x @ B @ x) - float(b @ x), g, float(np.abs(g).max())

    # (1e-6: below ~1e-7 the Armijo test drowns in the rounding of f, as for any line search on function values)
    status, x, iters, evals = lbfgs_s9(evaluate, np.zeros(n), 1.0, 1e-6, history=10)
    assert status == OK and evals == n_eval[0] and iters <= evals
    assert float(np.abs(B @ x - b).max()) <= 1e-6            # x is the LAST point evaluated and meets the test
    np.testing.assert_allclose(x, x_star, rtol=1e-5, atol=1e-6)
    # with full memory on a quadratic the iteration count stays near n even though the search is inexact
    status, x, iters_full, _ = lbfgs_s9(evaluate, np.zeros(n), 1.0, 1e-6, history=64)
    assert status == OK and iters_full <= 3 * n
    # limits
    n_eval[0] = 0
    status, x, iters, evals = lbfgs_s9(evaluate, np.zeros(n), 1.0, 1e-300, history=10, max_iters=1000, max_evals=9)
    assert status == NOT_CONVERGED and x is None and evals == 9 and n_eval[0] == 9
    status, x, iters, evals = lbfgs_s9(evaluate, np.zeros(n), 1.0, 1e-300, history=10, max_iters=4)
    assert status == NOT_CONVERGED and iters == 4
    # already converged at the start: iters = 0, one evaluation
    status, x, iters, evals = lbfgs_s9(evaluate, x_star, 1.0, 1e-6)
    assert (status, iters, evals) == (OK, 0, 1)


def test_P20_driver_on_a_piecewise_linear_concave_dual_like_function():
    """f(w) = -sum_j min_i (c_ij - w_i) - <v, w>... the 1-D-per-point analogue of the semi-discrete dual: convex,
    piecewise linear, gradient = mass of each cell - v.  The optimiser must drive every cell's mass to its target
    within eps although the curvature pairs are often rejected (y = 0 on a linear piece)."""
    rng = np.random.default_rng(2020)
    M, N = 6, 4000
    C = rng.random((N, M))
    v = rng.dirichlet(np.full(M, 5.0))

    def evaluate(w):
        c = C - w[None, :]
        lab = np.argmin(c, axis=1)
        mass = np.bincount(lab, minlength=M) / N
        dual = float(v @ w) + float(np.mean(c[np.arange(N), lab]))
        return -dual, mass - v, float(np.max(np.abs(mass - v) / v))

    status, w, iters, evals = lbfgs_s9(evaluate, np.zeros(M), 0.1, 0.02)
    assert status == OK
    assert evaluate(w)[2] <= 0.02
