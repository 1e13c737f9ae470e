"""Pins for the fp64 oracle (CPU only).  Each test checks oracle/ against something OTHER than
its own formula: a library routine, a closed form, exact rational arithmetic, an invariant.
Numbering P1..P15 follows DESIGN.md ("What pins the oracle")."""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle.apd_oracle import Grid, oracle_assign, oracle_cost_of, oracle_solve, OK, NOT_CONVERGED


def centres(grid: Grid):
    """Voxel centres lo + (i+1/2)s in label order (x fastest) -- PAPER.md:106-119."""
    d = grid.dim
    s = grid.s
    axes = [np.asarray(grid.lo[k]) + (np.arange(grid.n[k]) + 0.5) * s[k] for k in range(d)]
    if d == 2:
        yy, xx = np.meshgrid(axes[1], axes[0], indexing="ij")
        return np.stack([xx.ravel(), yy.ravel()], axis=1)
    zz, yy, xx = np.meshgrid(axes[2], axes[1], axes[0], indexing="ij")
    return np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1)


def eye(M, d):
    return np.tile(np.eye(d, dtype=np.float32), (M, 1, 1))


def rand_spd(rng, M, d, aspect=4.0):
    Q, _ = np.linalg.qr(rng.standard_normal((M, d, d)))
    lam = rng.uniform(1.0, aspect, (M, d))
    A = np.einsum("mij,mj,mkj->mik", Q, lam, Q)
    return (0.5 * (A + A.transpose(0, 2, 1))).astype(np.float32)


# ---------------------------------------------------------------- P1 Voronoi
@pytest.mark.parametrize("d,n,M", [(2, (8, 8), 5), (2, (16, 16), 8), (3, (8, 8, 8), 7), (3, (12, 10, 9), 8)])
def test_P1_voronoi_matches_kdtree(d, n, M):
    """A=I, w=0 is the Voronoi diagram (PAPER.md:63 case (i)): nearest seed by Euclidean distance,
    found by scipy's cKDTree (independent library routine)."""
    from scipy.spatial import cKDTree
    rng = np.random.default_rng(11 + d * 100 + M)
    X = rng.random((M, d)).astype(np.float32)
    g = Grid(d, n, (0.0,) * d, (1.0,) * d)
    r = oracle_assign(g, X, eye(M, d), np.zeros(M, np.float32))
    Y = centres(g)
    dist, nn = cKDTree(X.astype(np.float64)).query(Y, k=2)
    clear = (dist[:, 1] - dist[:, 0]) > 1e-9
    assert clear.sum() > 0.9 * len(Y)
    assert np.array_equal(r.labels[clear], nn[clear, 0].astype(np.int32))
    np.testing.assert_allclose(r.best[clear], dist[clear, 0] ** 2, rtol=1e-12, atol=1e-15)
    assert np.array_equal(r.runner[clear], nn[clear, 1].astype(np.int32))


# ---------------------------------------------------------------- P2 power diagram, two seeds
@pytest.mark.parametrize("d", [2, 3])
def test_P2_power_two_seeds_halfspace(d):
    """A=I (power diagram, PAPER.md:63 case (ii)), two seeds: c1 <= c2 <=> 2(x2-x1).y <= |x2|^2-|x1|^2-(w2-w1).
    Evaluated in exact rational arithmetic; pins the SIGN of w."""
    rng = np.random.default_rng(5 + d)
    X = (rng.integers(1, 63, (2, d)) / 64.0).astype(np.float32)
    w = np.array([3 / 64.0, -5 / 128.0], dtype=np.float32)
    n = (16,) * d
    g = Grid(d, n, (0.0,) * d, (1.0,) * d)
    r = oracle_assign(g, X, eye(2, d), w)
    Y = centres(g)
    Xf = [[Fraction(float(t)) for t in row] for row in X]
    wf = [Fraction(float(t)) for t in w]
    rhs = sum(t * t for t in Xf[1]) - sum(t * t for t in Xf[0]) - (wf[1] - wf[0])
    n_first = 0
    for j, y in enumerate(Y):
        yf = [Fraction(float(t)) for t in y]
        lhs = 2 * sum((Xf[1][k] - Xf[0][k]) * yf[k] for k in range(d))
        expect = 0 if lhs <= rhs else 1          # tie -> lowest index (reading S1)
        assert r.labels[j] == expect
        n_first += expect == 0
    assert 0 < n_first < len(Y)
    # raising w_1 grows cell 1 (sign convention of eq. 2.1: cost is  |.|^2 MINUS w)
    r2 = oracle_assign(g, X, eye(2, d), w + np.array([0, 0.25], np.float32))
    assert r2.count[1] > r.count[1]


# ---------------------------------------------------------------- P3 exact rational arithmetic
def exact_assign(grid: Grid, X, A, w):
    """eq. (2.1)/Alg. 1 in Fractions: exact argmin (lowest index on ties), exact min and runner-up."""
    d = grid.dim
    lo = [Fraction(float(t)) for t in grid.lo]
    hi = [Fraction(float(t)) for t in grid.hi]
    s = [(hi[k] - lo[k]) / int(grid.n[k]) for k in range(d)]
    Xf = [[Fraction(float(t)) for t in row] for row in X]
    Af = [[[Fraction(float(A[i, k, l])) for l in range(d)] for k in range(d)] for i in range(len(X))]
    wf = [Fraction(float(t)) for t in w]
    n = list(grid.n) + [1] * (3 - d)
    labels, best, second = [], [], []
    for iz in range(n[2] if d == 3 else 1):
        for iy in range(n[1]):
            for ix in range(n[0]):
                idx = (ix, iy, iz)
                y = [lo[k] + (idx[k] + Fraction(1, 2)) * s[k] for k in range(d)]
                costs = []
                for i in range(len(X)):
                    dl = [y[k] - Xf[i][k] for k in range(d)]
                    q = sum(dl[k] * Af[i][k][l] * dl[l] for k in range(d) for l in range(d))
                    costs.append(q - wf[i])
                m = min(costs)
                i1 = costs.index(m)
                rest = [c for i, c in enumerate(costs) if i != i1]
                labels.append(i1)
                best.append(m)
                second.append(min(rest) if rest else None)
    return labels, best, second


@pytest.mark.parametrize("d,n,M,seed", [(2, (16, 16), 6, 1), (2, (12, 9), 5, 2), (3, (8, 8, 8), 6, 3), (3, (5, 6, 7), 4, 4)])
def test_P3_exact_rational(d, n, M, seed):
    """Inputs with few mantissa bits => the fp64 oracle is EXACT, so labels (incl. ties), min,
    runner-up and the dual must equal the Fraction evaluation exactly."""
    rng = np.random.default_rng(seed)
    X = (rng.integers(0, 64, (M, d)) / 64.0).astype(np.float32)
    B = rng.integers(-3, 4, (M, d, d)) / 4.0
    A = (np.einsum("mij,mkj->mik", B, B) + np.eye(d)[None] * 0.5).astype(np.float32)   # SPD, dyadic
    w = (rng.integers(-8, 9, M) / 256.0).astype(np.float32)
    lo = (0.0,) * d
    hi = tuple(float(k) / 4.0 for k in n)          # s = 1/4 exactly, also for the odd sizes
    g = Grid(d, n, lo, hi)
    r = oracle_assign(g, X, A, w)
    labels, best, second = exact_assign(g, X, A, w)
    assert r.labels.tolist() == labels
    assert [Fraction(float(t)) for t in r.best] == best
    assert [Fraction(float(t)) for t in r.second] == second
    v = np.full(M, g.domain_volume / M)
    rr = oracle_assign(g, X, A, w, v=v)
    P = Fraction(g.voxel_volume)
    cnt = [labels.count(i) for i in range(M)]
    assert rr.count.tolist() == cnt
    wf = [Fraction(float(t)) for t in w]
    dual_exact = sum((Fraction(float(v[i])) - cnt[i] * P) * wf[i] for i in range(M)) + \
        P * sum(best[j] + wf[labels[j]] for j in range(len(labels)))
    assert abs(Fraction(rr.dual) - dual_exact) <= abs(dual_exact) * Fraction(1, 10 ** 14)


def test_P3_exact_ties_lowest_index():
    """Mirror-symmetric input with voxel centres ON the bisector, and coincident seeds: ties go to
    the lowest index (reading S1)."""
    g = Grid(2, (3, 2), (0.0, 0.0), (3.0, 2.0))            # centres x = 0.5, 1.5, 2.5
    X = np.array([[2.0, 1.0], [1.0, 1.0], [2.0, 1.0]], np.float32)   # seed 2 coincides with seed 0
    r = oracle_assign(g, X, eye(3, 2), np.zeros(3, np.float32))
    lab = r.labels.reshape(2, 3)
    assert lab[:, 1].tolist() == [0, 0]      # x = 1.5 equidistant from seeds 0 and 1 -> 0
    assert lab[:, 0].tolist() == [1, 1]
    assert lab[:, 2].tolist() == [0, 0]      # seed 2 never wins
    assert r.count[2] == 0
    assert np.all(r.second[[1, 4]] == r.best[[1, 4]])


# ---------------------------------------------------------------- P4 concentric ellipse / ellipsoid
@pytest.mark.parametrize("d", [2, 3])
def test_P4_concentric_ellipsoid_volume(d):
    """Two seeds at the same point, A2 = k I with k < lambda_min(A1), w1 - w2 = rho > 0:
    cell 1 = { delta^T (A1 - kI) delta <= rho }, an ellipse of area pi rho / sqrt(det(A1-kI))
    (3D: 4/3 pi rho^{3/2} / sqrt det).  count*|P| must converge to it."""
    if d == 2:
        th = 0.7
        R = np.array([[math.cos(th), -math.sin(th)], [math.sin(th), math.cos(th)]])
        A1 = R @ np.diag([9.0, 3.0]) @ R.T
    else:
        Q, _ = np.linalg.qr(np.random.default_rng(3).standard_normal((3, 3)))
        A1 = Q @ np.diag([8.0, 5.0, 3.0]) @ Q.T
    A1 = (0.5 * (A1 + A1.T)).astype(np.float32)
    k, rho = 1.0, 0.05
    A = np.stack([A1, k * np.eye(d, dtype=np.float32)])
    X = np.full((2, d), 0.5, np.float32) + np.float32(0.013)
    w = np.array([rho, 0.0], np.float32)
    B = A1.astype(np.float64) - k * np.eye(d)
    rho64 = float(np.float32(rho))
    exact = (math.pi * rho64 if d == 2 else 4.0 / 3.0 * math.pi * rho64 ** 1.5) / math.sqrt(np.linalg.det(B))
    semi_max = math.sqrt(rho64 / np.linalg.eigvalsh(B)[0])
    assert semi_max < 0.45                       # ellipsoid inside the box
    errs = []
    for n in ([32, 64, 128, 256] if d == 2 else [16, 32, 64]):
        g = Grid(d, (n,) * d, (0.0,) * d, (1.0,) * d)
        r = oracle_assign(g, X, A, w)
        errs.append(abs(r.vol[0] - exact))
        surf = (2 * math.pi * semi_max) if d == 2 else (4 * math.pi * semi_max ** 2)
        assert errs[-1] <= surf * (1.0 / n)      # error <~ surface * h
    assert errs[-1] < 0.2 * errs[0] + 1e-12
    assert errs[-1] / exact < 5e-3


# ---------------------------------------------------------------- P5 Moebius, two seeds
@pytest.mark.parametrize("d", [2, 3])
def test_P5_moebius_sphere(d):
    """A_i = c_i I, w = 0 (PAPER.md:63 case (iv)): boundary is the sphere with centre
    (c1 x1 - c2 x2)/(c1 - c2) and radius^2 c1 c2 |x1-x2|^2/(c1-c2)^2; larger c owns the inside."""
    c1, c2 = 4.0, 1.0
    x1 = np.array([0.45, 0.5, 0.55][:d])
    x2 = np.array([0.6, 0.45, 0.5][:d])
    X = np.stack([x1, x2]).astype(np.float32)
    A = np.stack([c1 * np.eye(d), c2 * np.eye(d)]).astype(np.float32)
    x1, x2 = X[0].astype(np.float64), X[1].astype(np.float64)
    m = (c1 * x1 - c2 * x2) / (c1 - c2)
    rad = math.sqrt(c1 * c2 * np.sum((x1 - x2) ** 2)) / (c1 - c2)
    n = 96 if d == 2 else 48
    g = Grid(d, (n,) * d, (0.0,) * d, (1.0,) * d)
    r = oracle_assign(g, X, A, np.zeros(2, np.float32))
    Y = centres(g)
    dist = np.linalg.norm(Y - m, axis=1)
    clear = np.abs(dist - rad) > 1e-9
    assert np.array_equal(r.labels[clear] == 0, (dist < rad)[clear])
    exact = math.pi * rad ** 2 if d == 2 else 4.0 / 3.0 * math.pi * rad ** 3
    assert abs(r.vol[0] - exact) / exact < 0.02


# ---------------------------------------------------------------- P6..P12 invariants
def _rand_problem(d, n, M, seed, lo=None, hi=None):
    rng = np.random.default_rng(seed)
    lo = lo or (0.0,) * d
    hi = hi or (1.0,) * d
    ext = np.array(hi) - np.array(lo)
    X = (np.array(lo) + rng.random((M, d)) * ext).astype(np.float32)
    A = rand_spd(rng, M, d)
    w = (rng.standard_normal(M) * 0.02).astype(np.float32)
    v = np.exp(rng.normal(0, 0.4, M))
    v = (v / v.sum() * np.prod(ext)).astype(np.float32)
    return Grid(d, n, lo, hi), X, A, w, v


@pytest.mark.parametrize("d,n", [(2, (40, 30)), (3, (16, 12, 10))])
def test_P6_P7_tessellation_and_dual_identity(d, n):
    g, X, A, w, v = _rand_problem(d, n, 9, 21 + d, lo=(-1.0, 0.5, 2.0)[:d], hi=(1.0, 2.0, 2.75)[:d])
    r = oracle_assign(g, X, A, w, v=v)
    assert int(r.count.sum()) == g.N                                         # P6
    assert abs(r.vol.sum() - g.domain_volume) <= 1e-12 * g.domain_volume
    # P7: eq. (2.7) literally  ==  <v,w> + |P| sum_j min_i C_ij   (identity I1)
    dual2 = float(np.dot(v.astype(np.float64), w.astype(np.float64))) + r.dual_min_part
    assert abs(r.dual - dual2) <= 1e-12 * max(abs(r.dual), abs(r.quad_part))
    # best = q - w of the winner
    np.testing.assert_allclose(r.best, r.qbest - w.astype(np.float64)[r.labels], rtol=0, atol=1e-15)
    # centroids: mean of member voxel centres
    Y = centres(g)
    for i in range(len(X)):
        if r.count[i]:
            np.testing.assert_allclose(r.centroids[i], Y[r.labels == i].mean(axis=0), rtol=1e-12, atol=1e-13)
        else:
            np.testing.assert_array_equal(r.centroids[i], X[i].astype(np.float64))   # S5


@pytest.mark.parametrize("d,n", [(2, (32, 32)), (3, (12, 12, 12))])
def test_P8_supergradient_and_finite_difference(d, n):
    """g~ is concave with super-gradient v - vol (eq. 2.4/2.8): g~(w') <= g~(w) + (v-vol(w)).(w'-w);
    and for h so small that no label changes, the finite difference equals v_i - vol_i exactly
    (north_star: 'gradient entries match finite differences of the dual')."""
    g, X, A, w, v = _rand_problem(d, n, 7, 33 + d)
    r = oracle_assign(g, X, A, w, v=v)
    grad = v.astype(np.float64) - r.vol
    rng = np.random.default_rng(0)
    for _ in range(5):
        w2 = (w + rng.standard_normal(len(w)) * 0.03).astype(np.float32)
        r2 = oracle_assign(g, X, A, w2, v=v)
        lin = r.dual + float(np.dot(grad, w2.astype(np.float64) - w.astype(np.float64)))
        assert r2.dual <= lin + 1e-12 * abs(lin)
    gap_min = float(np.min(r.second - r.best))
    h = np.float32(min(gap_min * 0.25, 1e-3))
    assert h > 0
    checked = 0
    for i in range(len(w)):
        wp = w.copy()
        wp[i] = w[i] + h
        hh = float(wp[i]) - float(w[i])                      # the step actually taken in fp32
        if not (0 < hh < gap_min):
            continue
        rp = oracle_assign(g, X, A, wp, v=v)
        assert np.array_equal(rp.labels, r.labels)
        fd = (rp.dual - r.dual) / hh
        assert abs(fd - grad[i]) <= 1e-13 * max(abs(r.dual), abs(r.quad_part)) / hh + 1e-12
        checked += 1
    assert checked >= len(w) - 1


def test_P9_concavity_midpoint():
    g, X, A, w, v = _rand_problem(2, (24, 24), 6, 77)
    rng = np.random.default_rng(1)
    for _ in range(5):
        wa = (rng.standard_normal(6) * 0.05).astype(np.float32)
        wb = (rng.standard_normal(6) * 0.05).astype(np.float32)
        wm = ((wa.astype(np.float64) + wb.astype(np.float64)) / 2)
        wm32 = wm.astype(np.float32)
        if not np.array_equal(wm32.astype(np.float64), wm):
            continue
        ga = oracle_assign(g, X, A, wa, v=v).dual
        gb = oracle_assign(g, X, A, wb, v=v).dual
        gm = oracle_assign(g, X, A, wm32, v=v).dual
        assert gm >= 0.5 * (ga + gb) - 1e-13 * (abs(ga) + abs(gb))


def test_P10_gauge():
    """Adding a constant to every w_i: same labels; g~ changes by const*(sum v - |Omega|) = 0 (I3)."""
    g, X, A, w, v = _rand_problem(3, (10, 10, 10), 8, 5)
    w = (np.round(w * 1024) / 1024).astype(np.float32)
    c = np.float32(0.125)                                    # w + c exact in fp32
    r0 = oracle_assign(g, X, A, w, v=v)
    r1 = oracle_assign(g, X, A, w + c, v=v)
    assert np.array_equal(r0.labels, r1.labels)
    vsum = float(v.astype(np.float64).sum())
    assert abs((r1.dual - r0.dual) - float(c) * (vsum - g.domain_volume)) <= 1e-12


def test_P11_exact_symmetries():
    g, X, A, w, v = _rand_problem(2, (32, 16), 6, 9)
    r = oracle_assign(g, X, A, w, v=v)
    # (A, w) -> (2A, 2w): every cost doubles exactly => same labels, quad part doubles exactly
    r2 = oracle_assign(g, X, 2 * A, 2 * w, v=v)
    assert np.array_equal(r.labels, r2.labels)
    assert r2.quad_part == 2 * r.quad_part
    # seed permutation
    perm = np.array([3, 0, 5, 1, 4, 2])
    rp = oracle_assign(g, X[perm], A[perm], w[perm], v=v[perm])
    assert np.array_equal(perm[rp.labels], r.labels)
    # reflection x -> 1 - x (power-of-two grid on [0,1]: exact)
    Xr = X.copy(); Xr[:, 0] = 1 - X[:, 0]
    if np.array_equal((1 - Xr[:, 0]).astype(np.float32), X[:, 0]):
        Ar = A.copy(); Ar[:, 0, 1] *= -1; Ar[:, 1, 0] *= -1
        rr = oracle_assign(g, Xr, Ar, w, v=v)
        assert np.array_equal(rr.labels.reshape(16, 32)[:, ::-1].ravel(), r.labels)


def test_P12_monotonicity():
    """raising w_i alone never shrinks cell i nor grows another; scaling A_i by c>1
    never grows cell i."""
    g, X, A, w, v = _rand_problem(2, (40, 40), 8, 123)
    r = oracle_assign(g, X, A, w)
    for i in range(8):
        wp = w.copy(); wp[i] += np.float32(0.01)
        rp = oracle_assign(g, X, A, wp)
        assert rp.count[i] >= r.count[i]
        others = np.arange(8) != i
        assert np.all(rp.count[others] <= r.count[others])
        Ap = A.copy(); Ap[i] *= np.float32(1.5)
        ra = oracle_assign(g, X, Ap, w)
        assert ra.count[i] <= r.count[i]
    Abig = A.copy(); Abig[0] *= np.float32(1e4)
    assert oracle_assign(g, X, Abig, w).count[0] <= 1


def test_cost_of_matches_best():
    g, X, A, w, v = _rand_problem(3, (9, 8, 7), 5, 6)
    r = oracle_assign(g, X, A, w)
    sel = np.arange(g.N, dtype=np.int64)
    np.testing.assert_array_equal(oracle_cost_of(g, X, A, w, sel, r.labels), r.best)
    np.testing.assert_array_equal(oracle_cost_of(g, X, A, w, sel, r.runner), r.second)
    sub = sel[::7]
    rs = oracle_assign(g, X, A, w, sel=sub)
    np.testing.assert_array_equal(rs.labels, r.labels[::7])
    np.testing.assert_array_equal(rs.best, r.best[::7])


def test_nonsymmetric_A_uses_quadratic_form_of_given_matrix():
    """S13: the quadratic form of A as given equals that of (A+A^T)/2."""
    g, X, A, w, v = _rand_problem(3, (8, 8, 8), 5, 8)
    K = np.random.default_rng(2).integers(-4, 5, A.shape) / 8.0
    An = (A.astype(np.float64) + (K - K.transpose(0, 2, 1))).astype(np.float32)
    As = (0.5 * (An.astype(np.float64) + An.astype(np.float64).transpose(0, 2, 1)))
    r1 = oracle_assign(g, X, An, w)
    r2 = oracle_assign(g, X, As, w)
    assert np.mean(r1.labels == r2.labels) > 0.999
    np.testing.assert_allclose(r1.best, r2.best, rtol=1e-12, atol=1e-14)


# ---------------------------------------------------------------- P13..P15 the solver
def test_P13_trivial_optimum_lattice():
    """Seeds on a regular k^d lattice, A=I, equal targets, n divisible by k: W=0 is optimal,
    iters = 0, cells are exact boxes."""
    k, n = 4, 32
    c = (np.arange(k) + 0.5) / k
    X = np.stack(np.meshgrid(c, c, indexing="ij"), -1).reshape(-1, 2).astype(np.float32)
    M = k * k
    # perturb centres off the voxel-boundary symmetry so there are no ties
    X = X + np.float32(1.0 / 256)
    g = Grid(2, (n, n), (0, 0), (1, 1))
    res = oracle_solve(g, X, eye(M, 2), np.full(M, 1.0 / M, np.float32), 0.01)
    assert res.status == OK and res.iters == 0 and res.evals == 1
    assert np.all(res.w32 == 0)
    assert set(np.bincount(res.labels, minlength=M).tolist()) == {n * n // M}


@pytest.mark.parametrize("aniso", [False, True])
def test_P14_closed_form_weights(aniso):
    """2D, seeds (1/4,1/2),(3/4,1/2), targets (0.3,0.7).  A=I: boundary x = 1/2 + (w1 - w2) must sit
    at 0.3 => w2 - w1 = 0.2 (up to +-h/2).  Anisotropic variant A_i = diag(a_i,1): boundary from
    a1 (x-1/4)^2 - w1 = a2 (x-3/4)^2 - w2."""
    n = 100
    g = Grid(2, (n, 8), (0, 0), (1, 1))
    X = np.array([[0.25, 0.5], [0.75, 0.5]], np.float32)
    a1, a2 = (2.0, 0.5) if aniso else (1.0, 1.0)
    A = np.array([[[a1, 0], [0, 1]], [[a2, 0], [0, 1]]], np.float32)
    v = np.array([0.3, 0.7], np.float32)
    res = oracle_solve(g, X, A, v, 0.01)
    assert res.status == OK
    dw = float(res.w[1] - res.w[0])
    h = 1.0 / n
    lo_b, hi_b = 0.3 - h / 2, 0.3 + h / 2          # boundary may sit anywhere between two centres
    f = lambda x: a1 * (x - 0.25) ** 2 - a2 * (x - 0.75) ** 2       # = w1 - w2 at the boundary
    vals = sorted([-f(lo_b), -f(hi_b)])
    assert vals[0] - 1e-9 <= dw <= vals[1] + 1e-9
    if not aniso:
        assert abs(dw - 0.2) <= h / 2 + 1e-9
    assert abs(float(np.mean(res.w))) < 1e-9          # gauge: sum w stays 0 (I3)
    assert res.labels.reshape(8, n)[0].tolist() == [0] * 30 + [1] * 70


@pytest.mark.parametrize("d,n,M", [(2, (64, 64), 10), (3, (24, 24, 24), 12)])
def test_P15_postcondition(d, n, M):
    from paper_2403_03571_b200 import workloads
    wl = workloads.make_config(1) if d == 2 else workloads.make_config(3, n=n, M=M)
    g = Grid(wl.dim, wl.n, wl.lo, wl.hi)
    res = oracle_solve(g, wl.X, wl.A, wl.v, wl.eps, record=True)
    assert res.status == OK
    chk = oracle_assign(g, wl.X, wl.A, res.w32, v=wl.v)
    assert chk.err <= wl.eps                              # Alg. 2 output spec
    assert np.array_equal(chk.labels, res.labels)
    assert res.evals == len(res.trajectory)
    # the dual is non-decreasing along ACCEPTED iterates is not guaranteed per evaluation, but the
    # final dual must exceed the initial one (ascent on a concave function)
    assert res.dual >= -res.trajectory[0]["f"] - 1e-15


def test_solver_reports_not_converged():
    """Alg. 2 step 4: 'if it is not possible to hit the desired tolerance' -> status, best iterate."""
    g = Grid(2, (6, 6), (0, 0), (1, 1))
    rng = np.random.default_rng(4)
    X = rng.random((5, 2)).astype(np.float32)
    v = np.array([0.2, 0.2, 0.2, 0.2, 0.2], np.float32)     # 7.2 pixels each: unreachable to 0.1%
    res = oracle_solve(g, X, eye(5, 2), v, 1e-3, max_iters=50)
    assert res.status == NOT_CONVERGED
    assert res.err > 1e-3
    chk = oracle_assign(g, X, eye(5, 2), res.w32, v=v)
    assert chk.err == res.err
