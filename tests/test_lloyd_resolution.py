"""NEXT rows f1/f2: Algorithm 3 and the resolution rules.
CPU part pins the oracle (Table 1 as printed; lattice fixed point; centroid step); GPU part is parity."""
import os

import numpy as np
import pytest

from paper_2403_03571_b200 import workloads
from oracle.apd_oracle import (Grid, OK, choose_resolution, oracle_assign, oracle_lloyd, oracle_solve,
                               resolution_bound)

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_table1.txt")


def table1():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    return [(int(a), int(b), int(c)) for a, b, c in rows]


def test_P16_table1_as_printed():
    """(N/eps)^(1/D) rounded to the nearest integer reproduces all 18 printed values (eq. 2.9 with v_i = 1/N)."""
    rows = table1()
    assert len(rows) == 18
    for D, N, M in rows:
        assert int(np.floor(resolution_bound(D, 1.0, 1.0 / N, 0.01, practical=False) + 0.5)) == M


def test_choose_resolution_is_the_strict_inequality():
    for D, N, _ in table1():
        for practical in (False, True):
            m = choose_resolution(D, 1.0, 1.0 / N, 0.01, practical)
            f = 0.01 / 2 ** D if practical else 0.01
            rhs = f * (1.0 / N)      # the same double expression as the rule's right-hand side (exact ties exist:
            assert 1.0 / m ** D < rhs and not (1.0 / (m - 1) ** D < rhs)      # 1/500^2 vs 0.01/2500)
    # "choosing M equal to two times the value given by (2.9)" == eq. (2.10)  (Table 1 caption)
    assert abs(resolution_bound(3, 1.0, 1e-4, 0.01, True) - 2 * resolution_bound(3, 1.0, 1e-4, 0.01, False)) < 1e-9


def lattice(k, n, d):
    g = (np.arange(k) + 0.5) / k
    X = np.stack(np.meshgrid(*([g] * d), indexing="ij"), -1).reshape(-1, d).astype(np.float32)
    M = X.shape[0]
    A = np.tile(np.eye(d, dtype=np.float32), (M, 1, 1))
    return workloads.Workload("lattice", d, (n,) * d, (0.0,) * d, (1.0,) * d, X, A,
                              np.full(M, 1.0 / M, np.float32), np.zeros(M, np.float32))


def test_lloyd_lattice_is_a_fixed_point():
    """Seeds on a regular lattice, A = I, equal targets: every cell is a box centred at its seed, so the centroid
    step leaves X unchanged and every solve stops at iters = 0."""
    wl = lattice(4, 32, 2)
    X, r, iters, evals = oracle_lloyd(Grid(2, wl.n, wl.lo, wl.hi), wl.X, wl.A, wl.v, 0.01, K=3)
    assert np.array_equal(X, wl.X) and r.status == OK and iters == 0 and evals == 4


def test_lloyd_centroid_step_and_warm_start():
    """One round by hand: X^1 = fl32(centroids of the optimal APD of X^0), W_0^1 = W^0; Lloyd
    moves seeds towards their cells' centroids, so seed-to-centroid distances shrink from round to round."""
    wl = workloads.make_config(1)
    grid = Grid(2, wl.n, wl.lo, wl.hi)
    r0 = oracle_solve(grid, wl.X, wl.A, wl.v, 0.01)
    c0 = oracle_assign(grid, wl.X, wl.A, r0.w32, v=wl.v).centroids
    X1, r1, _, _ = oracle_lloyd(grid, wl.X, wl.A, wl.v, 0.01, K=1)
    assert np.array_equal(X1, c0.astype(np.float32))
    r1_by_hand = oracle_solve(grid, X1, wl.A, wl.v, 0.01, w_init=r0.w32)
    assert np.array_equal(r1.w32, r1_by_hand.w32) and r1.status == OK
    X4, r4, _, _ = oracle_lloyd(grid, wl.X, wl.A, wl.v, 0.01, K=4)
    c4 = oracle_assign(grid, X4, wl.A, r4.w32, v=wl.v).centroids
    assert np.abs(c4 - X4).max() < np.abs(c0 - wl.X).max()


# ------------------------------------------------------------------------------------------------ GPU
@pytest.fixture(scope="module")
def apd():
    from paper_2403_03571_b200 import binding
    binding.load_library()
    return binding


def test_resolution_helpers_match_oracle():
    """Host-only entry points of the C ABI (no device work): callable without a GPU."""
    from paper_2403_03571_b200 import binding
    for D, N, M in table1():
        b = binding.apd_resolution_bound(D, 1.0, 1.0 / N, 0.01, False)
        assert int(np.floor(b + 0.5)) == M
        for practical in (False, True):
            assert binding.apd_choose_resolution(D, 1.0, 1.0 / N, 0.01, practical) == \
                choose_resolution(D, 1.0, 1.0 / N, 0.01, practical)
    assert binding.apd_choose_resolution(4, 1.0, 0.1, 0.01, False) == -1


def run_lloyd(apd, wl, eps, K, cull=0):
    import torch
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(wl.dim, wl.M)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X.copy()).to(dev); A = torch.from_numpy(wl.A).to(dev); v = torch.from_numpy(wl.v).to(dev)
    w = torch.zeros(wl.M, dtype=torch.float32, device=dev)
    labels = torch.full((wl.N,), -1, dtype=torch.int32, device=dev)
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    info = ctx.apd_lloyd(grid, X, A, v, eps, K, w=w, labels=labels, vol=vol, opts=apd.make_opts(cull=cull))
    return info, X.cpu().numpy(), w.cpu().numpy(), labels.cpu().numpy(), vol.cpu().numpy()


@pytest.mark.gpu
def test_gpu_lloyd_lattice_fixed_point(apd):
    wl = lattice(4, 32, 3)
    info, X, w, labels, vol = run_lloyd(apd, wl, 0.01, K=2)
    assert info.status == 0 and info.iters == 0 and info.evals == 3
    assert np.array_equal(X, wl.X) and np.all(w == 0)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n,M,eps,cull", [(1, None, None, 0.01, 0), (2, (256, 256), 60, 0.01, 1),
                                              (3, (64, 64, 64), 80, 0.02, 1)])
def test_gpu_lloyd_parity(apd, cfg, n, M, eps, cull):
    """K = 2 rounds against oracle_lloyd.  The two optimisers agree to ~1e-3 in w (parity rule 5), which moves a
    handful of boundary voxels, so the seeds after two centroid steps agree to a small fraction of a voxel; the
    post-condition is judged by the oracle at the GPU's (X, w)."""
    wl = workloads.make_config(cfg, n=n, M=M)
    grid = Grid(wl.dim, wl.n, wl.lo, wl.hi)
    Xo, ro, it_o, ev_o = oracle_lloyd(grid, wl.X, wl.A, wl.v, eps, K=2)
    info, X, w, labels, vol = run_lloyd(apd, wl, eps, K=2, cull=cull)
    assert info.status == ro.status == OK
    h = 1.0 / max(wl.n)
    assert np.abs(X - Xo).max() <= 0.25 * h, f"seeds differ by {np.abs(X - Xo).max() / h:.3f} voxels"
    chk = oracle_assign(grid, X, wl.A, w, v=wl.v)
    nm = int((labels != chk.labels).sum())
    assert nm < max(1e-5 * wl.N, 1) or nm == 0
    assert chk.err <= eps + 2 * nm * grid.voxel_volume / float(wl.v.min())
    assert abs(info.evals - ev_o) <= max(6, ev_o // 3)
    print(f"cfg{cfg}: gpu evals {info.evals} vs oracle {ev_o}; max seed diff {np.abs(X - Xo).max() / h:.4f} voxels")


# ------------------------------------------------------------------------------------------------ Alg. 2 step 4
def coarse_problem():
    """40 polydisperse grains on 32 x 32 pixels: the smallest grain holds ~8 pixels, so 1% is out of reach
    (|P| > eps v_min) until the grid has been refined."""
    return workloads.make_config(2, n=(32, 32), M=40)


def test_refine_and_restart_oracle():
    from oracle.apd_oracle import oracle_solve_refine, NOT_CONVERGED
    wl = coarse_problem()
    g0 = Grid(2, wl.n, wl.lo, wl.hi)
    assert g0.voxel_volume > 0.01 * float(wl.v.min())                       # the necessary condition (2.9) fails
    assert oracle_solve(g0, wl.X, wl.A, wl.v, 0.01, max_iters=200).status == NOT_CONVERGED
    g, res, r, iters, evals = oracle_solve_refine(g0, wl.X, wl.A, wl.v, 0.01, 4, max_iters=200)
    assert res.status == OK and 1 <= r <= 4 and tuple(g.n) == (32 * 2 ** r, 32 * 2 ** r)
    chk = oracle_assign(g, wl.X, wl.A, res.w32, v=wl.v)                     # post-condition on the FINAL grid
    assert chk.err <= 0.01
    # with no refinement allowed the call is Algorithm 2 steps 1-3 alone
    g1, res1, r1, _, _ = oracle_solve_refine(g0, wl.X, wl.A, wl.v, 0.01, 0, max_iters=200)
    assert r1 == 0 and res1.status == NOT_CONVERGED and tuple(g1.n) == (32, 32)


@pytest.mark.gpu
def test_gpu_refine_and_restart(apd):
    import torch
    from oracle.apd_oracle import oracle_solve_refine
    wl = coarse_problem()
    g_or, res, r_or, _, ev_or = oracle_solve_refine(Grid(2, wl.n, wl.lo, wl.hi), wl.X, wl.A, wl.v, 0.01, 4, max_iters=200)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(2, wl.M)
    grid = apd.make_grid(2, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); v = torch.from_numpy(wl.v).to(dev)
    w = torch.zeros(wl.M, dtype=torch.float32, device=dev)
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    info, r = ctx.apd_solve_refine(grid, X, A, v, 0.01, 4, w=w, vol=vol, opts=apd.make_opts(max_iters=200))
    assert info.status == 0 and r == r_or and (grid.n[0], grid.n[1]) == tuple(g_or.n)
    chk = oracle_assign(g_or, wl.X, wl.A, w.cpu().numpy(), v=wl.v)          # judged by the oracle on the final grid
    assert chk.err <= 0.01 + 2 * g_or.voxel_volume / float(wl.v.min())
    # the coarse, non-converging solves wander (every decision sits on a few pixels): only the order of magnitude of
    # the work is comparable
    assert abs(info.evals - ev_or) <= max(10, ev_or // 2)
    print(f"refinements {r}, final grid {grid.n[0]}x{grid.n[1]}, gpu evals {info.evals} vs oracle {ev_or}")


# ---------------------------------------------------------------- coarse-to-fine continuation (f2 extension)
def test_oracle_continuation_levels0_is_solve_and_postcondition():
    from oracle.apd_oracle import oracle_solve_continuation
    wl = workloads.make_config(2, n=(128, 128), M=30)
    g = Grid(wl.dim, wl.n, wl.lo, wl.hi)
    plain = oracle_solve(g, wl.X, wl.A, wl.v, 0.01)
    r0, it0, ev0 = oracle_solve_continuation(g, wl.X, wl.A, wl.v, 0.01, 0)
    assert (r0.status, r0.iters, r0.evals) == (plain.status, plain.iters, plain.evals) and np.array_equal(r0.w, plain.w)
    assert it0 == [plain.iters] and ev0 == [plain.evals]
    r2, it2, ev2 = oracle_solve_continuation(g, wl.X, wl.A, wl.v, 0.01, 2)
    assert r2.status == OK and len(ev2) == 3
    chk = oracle_assign(g, wl.X, wl.A, r2.w32, v=wl.v)
    assert chk.err <= 0.01                                    # the last level is Algorithm 2 on the grid itself (P15)
    assert ev2[-1] < plain.evals                              # it starts almost converged
    # a level coarser than 16 voxels per axis is skipped
    r5, it5, ev5 = oracle_solve_continuation(g, wl.X, wl.A, wl.v, 0.01, 5)
    assert ev5[0] == 0 and ev5[1] == 0 and ev5[-1] > 0


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n,M,eps,cull,levels", [(2, (256, 256), 60, 0.01, 1, 2), (3, (96, 96, 96), 120, 0.02, 1, 2),
                                                     (4, (128, 128, 128), 300, 0.02, 0, 1)])
def test_gpu_continuation_parity(apd, cfg, n, M, eps, cull, levels):
    """apd_solve_continuation against oracle_solve_continuation: same level structure, the oracle's evaluation at the
    GPU's weights meets the tolerance, labels agree up to near-ties, per-level evaluation counts close (identical when
    no voxel flips: parity rule 5), and the fine level needs fewer evaluations than plain apd_solve."""
    from oracle.apd_oracle import oracle_solve_continuation
    import torch
    import apd_parity as parity
    wl = workloads.make_config(cfg, n=n, M=M)
    grid_o = Grid(wl.dim, wl.n, wl.lo, wl.hi)
    ro, it_o, ev_o = oracle_solve_continuation(grid_o, wl.X, wl.A, wl.v, eps, levels)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(wl.dim, wl.M)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); v = torch.from_numpy(wl.v).to(dev)
    w = torch.zeros(wl.M, dtype=torch.float32, device=dev); labels = torch.empty(wl.N, dtype=torch.int32, device=dev)
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    rc, it_g, ev_g, err = ctx.apd_solve_continuation(grid, levels, X, A, v, eps, w=w, labels=labels, vol=vol,
                                                     opts=apd.make_opts(cull=cull))
    plain = ctx.apd_solve(grid, X, A, v, eps, w=torch.zeros_like(w), opts=apd.make_opts(cull=cull))
    assert rc == 0 and ro.status == OK and err <= eps
    chk = oracle_assign(grid_o, wl.X, wl.A, w.cpu().numpy(), v=wl.v)
    nm = parity.check_labels(grid_o, wl.X, wl.A, w.cpu().numpy(), labels.cpu().numpy(), chk)["mismatches"]
    assert chk.err <= eps + 2 * nm * grid_o.voxel_volume / float(wl.v.min())
    assert len(ev_g) == levels + 1 and [e > 0 for e in ev_g] == [e > 0 for e in ev_o]
    for a, b in zip(ev_g, ev_o):
        assert abs(a - b) <= max(6, b // 3)
    assert ev_g[-1] < plain.evals
    print(f"continuation cfg{cfg} {n}: evals per level gpu {ev_g} oracle {ev_o}; plain apd_solve {plain.evals} evaluations")
    ctx.close()
