"""NEXT row f3: Algorithm 1 + eq. (2.7)-(2.8) on user-supplied points with element volumes.
CPU part pins oracle_assign_points to the (already pinned) grid oracle and to invariants; GPU part is parity."""
import numpy as np
import pytest

from paper_2403_03571_b200 import workloads
from oracle.apd_oracle import Grid, oracle_assign, oracle_assign_points


def grid_points(wl):
    """Voxel centres (x fastest) and the constant voxel volume of a Workload's grid."""
    g = Grid(wl.dim, wl.n, wl.lo, wl.hi)
    ax = [np.asarray(wl.lo[k]) + (np.arange(wl.n[k]) + 0.5) * g.s[k] for k in range(wl.dim)]
    mesh = np.meshgrid(*ax[::-1], indexing="ij")                  # slowest axis first
    Y = np.stack([m.ravel() for m in mesh[::-1]], axis=1)         # columns x, y[, z]
    return Y, np.full(Y.shape[0], g.voxel_volume)


@pytest.mark.parametrize("dim,n,M", [(2, (24, 17), 9), (3, (10, 9, 7), 12)])
def test_points_oracle_reduces_to_the_grid_oracle(dim, n, M):
    """With y_j = voxel centres and |P_j| = |P| the element formulation IS the pixel method: same labels, volumes,
    dual and centroids as oracle_assign (which is pinned by P1-P15)."""
    wl = workloads.make_random(dim, n, M, 5, lo=(0.0, -1.0, 0.5)[:dim], hi=(2.0, 0.5, 1.5)[:dim], w_scale=0.2)
    Y, p = grid_points(wl)
    a = oracle_assign(Grid(dim, wl.n, wl.lo, wl.hi), wl.X, wl.A, wl.w0, v=wl.v)
    b = oracle_assign_points(Y, p, wl.X, wl.A, wl.w0, v=wl.v)
    assert np.array_equal(a.labels, b.labels)
    np.testing.assert_allclose(b.vol, a.vol, rtol=1e-13, atol=0)
    np.testing.assert_allclose(b.dual, a.dual, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(b.centroids, a.centroids, rtol=0, atol=1e-12)
    np.testing.assert_allclose(b.best, a.best, rtol=1e-12, atol=1e-15)


def test_points_oracle_invariants():
    """Permuting the points permutes the labels and leaves vol/dual; splitting an element into two halves at the same
    location changes nothing; volumes sum to sum |P_j|; dual identity I1 with element volumes."""
    rng = np.random.default_rng(3)
    wl = workloads.make_random(3, (4, 4, 4), 15, 6, w_scale=0.2)
    N = 3000
    Y = rng.random((N, 3)); p = rng.random(N) * 1e-3
    r = oracle_assign_points(Y, p, wl.X, wl.A, wl.w0, v=wl.v)
    perm = rng.permutation(N)
    r2 = oracle_assign_points(Y[perm], p[perm], wl.X, wl.A, wl.w0, v=wl.v)
    assert np.array_equal(r2.labels, r.labels[perm])
    np.testing.assert_allclose(r2.vol, r.vol, rtol=1e-12); np.testing.assert_allclose(r2.dual, r.dual, rtol=1e-12)
    r3 = oracle_assign_points(np.concatenate([Y, Y]), np.concatenate([p / 2, p / 2]), wl.X, wl.A, wl.w0, v=wl.v)
    np.testing.assert_allclose(r3.vol, r.vol, rtol=1e-12); np.testing.assert_allclose(r3.dual, r.dual, rtol=1e-12)
    np.testing.assert_allclose(r.vol.sum(), p.sum(), rtol=1e-13)
    i1 = float(np.dot(wl.v.astype(np.float64), wl.w0.astype(np.float64))) + r.dual_min_part
    np.testing.assert_allclose(r.dual, i1, rtol=1e-12)


# ------------------------------------------------------------------------------------------------ GPU
@pytest.fixture(scope="module")
def apd():
    from paper_2403_03571_b200 import binding
    binding.load_library()
    return binding


def run_points(apd, dim, Y, p, wl, w, want_centroids=True):
    import torch
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(dim, wl.M)
    t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dtype=dt)).to(dev)
    N = Y.shape[0]
    labels = torch.full((N,), -3, dtype=torch.int32, device=dev)
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev); dual = torch.zeros(1, dtype=torch.float64, device=dev)
    err = torch.zeros(1, dtype=torch.float64, device=dev)
    cen = torch.zeros(wl.M, dim, dtype=torch.float64, device=dev) if want_centroids else None
    ctx.apd_assign_points(t(Y, np.float32), t(p, np.float32), t(wl.X, np.float32), t(wl.A, np.float32), t(w, np.float32),
                          target_vol=t(wl.v, np.float32), labels=labels, vol=vol, dual=dual, max_rel_err=err, centroids=cen)
    torch.cuda.synchronize()
    return labels.cpu().numpy(), vol.cpu().numpy(), float(dual.item()), float(err.item()), \
        (cen.cpu().numpy() if want_centroids else None)


def check_points(Y32, p32, wl, w, labels, vol, dual, err, cen):
    """The parity rule of DESIGN.md section 8 with element volumes: mismatches must be near-ties and fewer than
    1e-5 N; volumes agree up to the mismatching elements (+ fp64 summation order); dual to 1e-6."""
    orc = oracle_assign_points(Y32, p32, wl.X, wl.A, w, v=wl.v)
    w64 = np.asarray(w, np.float64)
    mism = np.nonzero(labels != orc.labels)[0]
    assert labels.min() >= 0 and labels.max() < wl.M
    assert mism.size < max(1e-5 * labels.size, 1) or mism.size == 0
    if mism.size:
        Y = Y32.astype(np.float64)
        D = Y[mism] - wl.X.astype(np.float64)[labels[mism]]
        c_gpu = np.einsum("nk,nkl,nl->n", D, wl.A.astype(np.float64)[labels[mism]], D) - w64[labels[mism]]
        q1 = orc.best[mism] + w64[orc.labels[mism]]
        scale = np.maximum(np.abs(q1), np.abs(w64[orc.labels[mism]]))
        assert np.all(c_gpu - orc.best[mism] < 1e-5 * scale)
    moved = float(p32.astype(np.float64)[mism].sum())
    assert np.abs(vol - orc.vol).sum() <= 2 * moved + 1e-12 * orc.vol.sum()
    assert abs(dual - orc.dual) <= 1e-6 * max(abs(orc.dual), abs(orc.dual_min_part))
    assert abs(err - orc.err) <= 2 * moved / float(wl.v.min()) + 1e-9
    if cen is not None and mism.size == 0:
        np.testing.assert_allclose(cen, orc.centroids, rtol=0, atol=1e-9)
    return mism.size


@pytest.mark.gpu
@pytest.mark.parametrize("dim,N,M", [(3, 50000, 300), (2, 30011, 129), (3, 1, 5), (2, 1025, 1)])
def test_gpu_points_parity(apd, dim, N, M):
    rng = np.random.default_rng(100 + N)
    wl = workloads.make_random(dim, (4,) * dim, M, 8, w_scale=0.15)
    Y = rng.random((N, dim)).astype(np.float32)
    p = ((0.5 + rng.random(N)) / N).astype(np.float32)
    if N > 10:
        p[3::7] = 0.0                                                          # some empty elements
    wl.v[:] = (wl.v / wl.v.sum() * p.astype(np.float64).sum()).astype(np.float32)
    labels, vol, dual, err, cen = run_points(apd, dim, Y, p, wl, wl.w0)
    nm = check_points(Y, p, wl, wl.w0, labels, vol, dual, err, cen)
    print(f"points {dim}D N={N} M={M}: {nm} mismatches")


@pytest.mark.gpu
def test_gpu_points_on_grid_centres_match_apd_assign(apd):
    """Fed the voxel centres of a power-of-two grid (exact in fp32) with |P_j| = |P|, apd_assign_points gives the
    labels of the DIRECT grid kernel bit for bit and the same volumes."""
    import torch
    wl = workloads.make_config(3, n=(32, 32, 16), M=120)
    Y, p = grid_points(wl)
    labels, vol, dual, err, _ = run_points(apd, 3, Y.astype(np.float32), p.astype(np.float32), wl, wl.w0, want_centroids=False)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(3, wl.M)
    grid = apd.make_grid(3, wl.n, wl.lo, wl.hi)
    t = lambda a: torch.from_numpy(a).to(dev)
    lab2 = torch.empty(wl.N, dtype=torch.int32, device=dev); vol2 = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    d2 = torch.zeros(1, dtype=torch.float64, device=dev)
    ctx.apd_assign(grid, t(wl.X), t(wl.A), t(wl.w0), target_vol=t(wl.v), labels=lab2, vol=vol2, dual=d2,
                   opts=apd.make_opts(kernel=apd.KERNEL_DIRECT))
    torch.cuda.synchronize()
    assert np.array_equal(labels, lab2.cpu().numpy())
    np.testing.assert_allclose(vol, vol2.cpu().numpy(), rtol=1e-12, atol=0)
    assert abs(dual - float(d2.item())) <= 1e-12 * abs(dual)


# ------------------------------------------------------------------------------------------------ Algorithm 2 on points
def test_oracle_solve_on_points_equals_solve_on_grid():
    """oracle_solve fed the voxel centres of a grid as a PointSet walks the same trajectory as on the Grid itself."""
    from oracle.apd_oracle import PointSet, oracle_solve
    wl = workloads.make_config(1)
    Y, p = grid_points(wl)
    a = oracle_solve(Grid(2, wl.n, wl.lo, wl.hi), wl.X, wl.A, wl.v, 0.01)
    b = oracle_solve(PointSet(Y, p), wl.X, wl.A, wl.v, 0.01)
    assert (a.status, a.iters, a.evals) == (b.status, b.iters, b.evals)
    np.testing.assert_allclose(b.w, a.w, rtol=0, atol=1e-9 * np.abs(a.w).max())


@pytest.mark.gpu
def test_gpu_solve_points(apd):
    """Monte-Carlo discretisation of the unit square (random points, equal volumes): apd_solve_points reaches the
    tolerance as judged by the ORACLE at the GPU's weights; the optimisers walk closely related paths."""
    import torch
    from oracle.apd_oracle import PointSet, oracle_solve
    rng = np.random.default_rng(5)
    wl = workloads.make_config(2, n=(8, 8), M=30)
    N = 60000
    Y = rng.random((N, 2)).astype(np.float32)
    p = np.full(N, 1.0 / N, np.float32)
    tot = float(p.astype(np.float64).sum())
    wl.v[:] = (wl.v.astype(np.float64) / wl.v.astype(np.float64).sum() * tot).astype(np.float32)
    orc = oracle_solve(PointSet(Y, p), wl.X, wl.A, wl.v, 0.02)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(2, wl.M)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    w = torch.zeros(wl.M, dtype=torch.float32, device=dev)
    labels = torch.full((N,), -1, dtype=torch.int32, device=dev); vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    info = ctx.apd_solve_points(t(Y), t(p), tot, t(wl.X), t(wl.A), t(wl.v), 0.02, w=w, labels=labels, vol=vol)
    assert info.status == orc.status == 0 and info.max_rel_err <= 0.02
    chk = oracle_assign_points(Y, p, wl.X, wl.A, w.cpu().numpy(), v=wl.v)
    nm = int((labels.cpu().numpy() != chk.labels).sum())
    assert nm < max(1e-5 * N, 1) or nm == 0
    assert chk.err <= 0.02 + 2 * nm / N / float(wl.v.min())
    np.testing.assert_allclose(vol.cpu().numpy(), chk.vol, rtol=0, atol=2 * nm / N + 1e-12)
    assert abs(info.evals - orc.evals) <= max(4, orc.evals // 4)
    print(f"solve on points: gpu {info.iters}/{info.evals} err {info.max_rel_err:.4g}; oracle {orc.iters}/{orc.evals}")


# ------------------------------------------------------------------------------------------------ Algorithm 3 on points
def test_oracle_lloyd_on_points_equals_lloyd_on_grid():
    """oracle_lloyd fed the voxel centres of a grid as a PointSet is Algorithm 3 on the grid itself (whose pins are in
    tests/test_lloyd_resolution.py): same seeds after every round, same evaluation counts."""
    from oracle.apd_oracle import PointSet, oracle_lloyd
    wl = workloads.make_config(1)
    Y, p = grid_points(wl)
    Xa, ra, ia, ea = oracle_lloyd(Grid(2, wl.n, wl.lo, wl.hi), wl.X, wl.A, wl.v, 0.01, K=2)
    Xb, rb, ib, eb = oracle_lloyd(PointSet(Y, p), wl.X, wl.A, wl.v, 0.01, K=2)
    assert (ra.status, ia, ea) == (rb.status, ib, eb)
    np.testing.assert_allclose(Xb, Xa, rtol=0, atol=1e-6)
    np.testing.assert_allclose(rb.w, ra.w, rtol=0, atol=1e-7 * np.abs(ra.w).max() + 1e-12)
    assert not np.allclose(Xa, wl.X, atol=1e-4)                         # the seeds did move


@pytest.mark.gpu
def test_gpu_lloyd_points(apd):
    """K = 2 rounds of Algorithm 3 on a Monte-Carlo discretisation against oracle_lloyd(PointSet): the seeds agree to a
    small fraction of the mean point spacing, and the post-condition is judged by the oracle at the GPU's (X, w)."""
    import torch
    from oracle.apd_oracle import PointSet, oracle_lloyd
    rng = np.random.default_rng(11)
    wl = workloads.make_config(2, n=(8, 8), M=24)
    N = 50000
    Y = rng.random((N, 2)).astype(np.float32)
    p = np.full(N, 1.0 / N, np.float32)
    tot = float(p.astype(np.float64).sum())
    v = (wl.v.astype(np.float64) / wl.v.astype(np.float64).sum() * tot).astype(np.float32)
    Xo, ro, it_o, ev_o = oracle_lloyd(PointSet(Y, p), wl.X, wl.A, v, 0.02, K=2)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(2, wl.M)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    X = t(wl.X.copy()); w = torch.zeros(wl.M, dtype=torch.float32, device=dev)
    labels = torch.full((N,), -1, dtype=torch.int32, device=dev); vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    info = ctx.apd_lloyd_points(t(Y), t(p), tot, X, t(wl.A), t(v), 0.02, 2, w=w, labels=labels, vol=vol)
    ctx.close()
    assert info.status == ro.status == 0 and info.max_rel_err <= 0.02
    Xg = X.cpu().numpy()
    h = (1.0 / N) ** 0.5                                                 # mean point spacing
    assert np.abs(Xg - Xo).max() <= 0.25 * h, f"seeds differ by {np.abs(Xg - Xo).max() / h:.3f} point spacings"
    assert not np.allclose(Xg, wl.X, atol=1e-4)
    chk = oracle_assign_points(Y, p, Xg, wl.A, w.cpu().numpy(), v=v)
    nm = int((labels.cpu().numpy() != chk.labels).sum())
    assert nm < max(1e-5 * N, 1) or nm == 0
    assert chk.err <= 0.02 + 2 * nm / N / float(v.min())
    assert abs(info.evals - ev_o) <= max(6, ev_o // 3)
    print(f"lloyd on points: gpu evals {info.evals} vs oracle {ev_o}; max seed diff {np.abs(Xg - Xo).max() / h:.4f} spacings")
