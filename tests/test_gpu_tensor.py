"""GPU parity of APD_KERNEL_TENSOR (row a8: the cost matrix of Algorithm 1 step 1, lifted to a bf16
tensor-core contraction with 3-way split coefficients; argmin epilogue) against the fp64 oracle, through
the C ABI.  north_star keeps the lifted path only if label agreement stays within the parity rule: these tests are that
check.  Run on the B200 box with `pytest -m gpu`."""
import numpy as np
import pytest
import torch

from paper_2403_03571_b200 import workloads
import apd_parity as parity
from test_gpu_assign import run_assign, rand_w, apd  # noqa: F401  (apd is the module fixture)

pytestmark = pytest.mark.gpu

TENSOR, DIRECT = 3, 1


@pytest.mark.parametrize("wscale", [0.0, 0.15])
def test_cfg3_full_parity(apd, wscale):
    wl = workloads.make_config(3)
    w = wl.w0 if wscale == 0.0 else rand_w(wl, wscale, 303)
    r = run_assign(apd, wl, w, v=wl.v, kernel=TENSOR, want_centroids=True)
    info = parity.check_assign(wl, w, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                               err_gpu=r["err"])
    assert r["pairs"] == wl.N * wl.M
    print(f"cfg3 tensor wscale={wscale}: {info}")


# ragged tiles on every axis, non-unit boxes (voxel centres not exact in fp32), M = 1, 2, 3, 5, M around the chunk of
# 64 seeds and around the padding unit of 128
EDGE3 = [
    dict(n=(50, 60, 70), M=130, lo=(0, 0, 0), hi=(1, 1, 1), seed=2),
    dict(n=(33, 17, 9), M=5, lo=(-1, 2, 0), hi=(1, 5, 0.5), seed=3),
    dict(n=(5, 1, 1), M=1, lo=(0, 0, 0), hi=(1, 1, 1), seed=5),
    dict(n=(16, 8, 4), M=2, lo=(0, 0, 0), hi=(1, 1, 1), seed=6),
    dict(n=(17, 9, 5), M=3, lo=(0, 0, 0), hi=(2, 1, 0.5), seed=7),
    dict(n=(64, 64, 64), M=129, lo=(0, 0, 0), hi=(1, 1, 1), seed=8),
    dict(n=(40, 40, 40), M=64, lo=(0, 0, 0), hi=(1, 1, 1), seed=9),
    dict(n=(40, 40, 40), M=65, lo=(0, 0, 0), hi=(1, 1, 1), seed=10),
    dict(n=(48, 40, 36), M=1000, lo=(0, 0, 0), hi=(1, 1, 1), seed=11),
]


@pytest.mark.parametrize("case", EDGE3, ids=lambda c: f"{'x'.join(map(str, c['n']))}_M{c['M']}")
@pytest.mark.parametrize("nonsym", [False, True])
def test_edge_cases(apd, case, nonsym):
    wl = workloads.make_random(3, case["n"], case["M"], case["seed"], lo=case["lo"], hi=case["hi"], w_scale=0.1,
                               nonsymmetric=nonsym)
    r = run_assign(apd, wl, wl.w0, v=wl.v, kernel=TENSOR, want_centroids=True)
    parity.check_assign(wl, wl.w0, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                        err_gpu=r["err"])


# ---- 2D: the same kernel on tiles of 32 x 16 pixels (6 of the 10 monomials are non-zero) ----------------------------

@pytest.mark.parametrize("cfg,wscale", [(1, 0.0), (1, 0.1), (2, 0.0), (2, 0.002)])
def test_2d_configs_full_parity(apd, cfg, wscale):
    wl = workloads.make_config(cfg)
    w = wl.w0 if wscale == 0.0 else rand_w(wl, wscale, 200 + cfg)
    r = run_assign(apd, wl, w, v=wl.v, kernel=TENSOR, want_centroids=True)
    info = parity.check_assign(wl, w, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                               err_gpu=r["err"])
    assert r["pairs"] == wl.N * wl.M
    print(f"cfg{cfg} tensor 2D wscale={wscale}: {info}")


EDGE2 = [
    dict(n=(100, 70), M=130, lo=(0, 0), hi=(1, 1), seed=42),
    dict(n=(33, 17), M=5, lo=(-1, 2), hi=(1, 5), seed=43),
    dict(n=(5, 1), M=1, lo=(0, 0), hi=(1, 1), seed=45),
    dict(n=(32, 16), M=2, lo=(0, 0), hi=(1, 1), seed=46),
    dict(n=(33, 17), M=3, lo=(0, 0), hi=(2, 1), seed=47),
    dict(n=(1, 40), M=7, lo=(0, 0), hi=(1, 3), seed=48),
    dict(n=(257, 129), M=129, lo=(0, 0), hi=(1, 1), seed=49),
    dict(n=(300, 200), M=1000, lo=(0, 0), hi=(1, 1), seed=50),
]


@pytest.mark.parametrize("case", EDGE2, ids=lambda c: f"{'x'.join(map(str, c['n']))}_M{c['M']}")
@pytest.mark.parametrize("nonsym", [False, True])
def test_2d_edge_cases(apd, case, nonsym):
    wl = workloads.make_random(2, case["n"], case["M"], case["seed"], lo=case["lo"], hi=case["hi"], w_scale=0.1,
                               nonsymmetric=nonsym)
    r = run_assign(apd, wl, wl.w0, v=wl.v, kernel=TENSOR, want_centroids=True)
    parity.check_assign(wl, wl.w0, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                        err_gpu=r["err"])


def test_2d_agrees_with_the_direct_kernel(apd):
    wl = workloads.make_config(2)
    w = rand_w(wl, 0.002, 77)
    rt = run_assign(apd, wl, w, v=wl.v, kernel=TENSOR)
    rd = run_assign(apd, wl, w, v=wl.v, kernel=DIRECT)
    assert (rt["labels"] != rd["labels"]).sum() < 2e-5 * wl.N
    assert abs(rt["dual"] - rd["dual"]) <= 1e-6 * abs(rd["dual"])


def test_no_target_volume_no_labels_and_reproducible(apd):
    wl = workloads.make_random(3, (40, 24, 16), 50, 21, w_scale=0.1)
    r = run_assign(apd, wl, wl.w0, v=None, kernel=TENSOR)
    parity.check_assign(wl, wl.w0, r["labels"], r["vol"], r["dual"], v=None)
    r2 = run_assign(apd, wl, wl.w0, v=None, kernel=TENSOR, want_labels=False)
    assert r2["dual"] == r["dual"] and np.array_equal(r2["vol"], r["vol"])     # bitwise reproducible


def test_one_huge_weight_and_coincident_seeds(apd):
    wl = workloads.make_random(3, (48, 32, 24), 40, 31, w_scale=0.05)
    w = wl.w0.copy()
    w[7] = 50.0                                  # cell 7 swallows the box
    r = run_assign(apd, wl, w, v=wl.v, kernel=TENSOR)
    parity.check_assign(wl, w, r["labels"], r["vol"], r["dual"], v=wl.v)
    assert (r["labels"] == 7).all()
    X = wl.X.copy()
    X[11] = X[3]                                 # coincident seeds with equal A and w: the lower index wins (S17)
    A = wl.A.copy()
    A[11] = A[3]
    w2 = wl.w0.copy()
    w2[11] = w2[3]
    import dataclasses
    wl2 = dataclasses.replace(wl, X=X, A=A)
    r = run_assign(apd, wl2, w2, v=wl2.v, kernel=TENSOR)
    parity.check_assign(wl2, w2, r["labels"], r["vol"], r["dual"], v=wl2.v)
    assert not (r["labels"] == 11).any()


def test_agrees_with_the_direct_kernel_up_to_near_ties(apd):
    """Same fp32 inputs, two arithmetics (tensor-core polynomial vs direct form): labels may differ on fp32 near-ties
    only; the parity rule against the oracle holds for both, so they differ on < 2e-5 N voxels."""
    wl = workloads.make_config(4, n=(96, 96, 96), M=3000)
    w = rand_w(wl, 0.1, 404)
    a = run_assign(apd, wl, w, v=wl.v, kernel=DIRECT)
    b = run_assign(apd, wl, w, v=wl.v, kernel=TENSOR)
    ndiff = int((a["labels"] != b["labels"]).sum())
    assert ndiff < 2e-5 * wl.N, ndiff
    assert abs(a["dual"] - b["dual"]) <= 1e-6 * abs(a["dual"])
    parity.check_assign(wl, w, b["labels"], b["vol"], b["dual"], v=wl.v, err_gpu=b["err"])


def test_cfg4_full_size_sampled_parity(apd):
    """BASELINE config 4 at full size (256^3 x 10^4) in the launch configuration bench.py times."""
    from oracle.apd_oracle import oracle_assign
    wl = workloads.make_config(4)
    w = rand_w(wl, 0.1, 204)
    r = run_assign(apd, wl, w, v=wl.v, kernel=TENSOR)
    assert r["pairs"] == wl.N * wl.M
    grid = parity.grid_of(wl)
    sel = workloads.voxel_sample(wl.N, 60000, 4)
    orc = oracle_assign(grid, wl.X, wl.A, w, sel=sel)
    info = parity.check_labels(grid, wl.X, wl.A, w, r["labels"][sel], orc, sel=sel)
    P = grid.voxel_volume
    cnt = np.rint(r["vol"] / P).astype(np.int64)
    assert int(cnt.sum()) == wl.N
    assert np.array_equal(cnt, np.bincount(r["labels"], minlength=wl.M))
    est = float(np.dot(wl.v.astype(np.float64), w.astype(np.float64))) + float(np.mean(orc.best))
    se = float(np.std(orc.best)) / np.sqrt(len(sel))
    assert abs(r["dual"] - est) < 6 * se + 1e-9
    print(f"cfg4 tensor sampled: {info}")


def test_rejects_culling(apd):
    wl3 = workloads.make_random(3, (32, 32, 32), 20, 5)
    with pytest.raises(Exception):
        run_assign(apd, wl3, wl3.w0, v=wl3.v, kernel=TENSOR, cull=1)
    wl2 = workloads.make_random(2, (64, 64), 20, 5)
    with pytest.raises(Exception):
        run_assign(apd, wl2, wl2.w0, v=wl2.v, kernel=TENSOR, cull=1)


def test_solve_with_the_tensor_kernel_meets_the_tolerance(apd):
    """apd_solve driven by the TENSOR evaluation: the post-condition of Algorithm 2 checked by the
    ORACLE at the returned weights."""
    from oracle.apd_oracle import Grid, oracle_assign
    dev = torch.device("cuda:0")
    wl = workloads.make_config(3, n=(64, 64, 64), M=200)
    ctx = apd.ApdContext(wl.dim, wl.M)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); v = torch.from_numpy(wl.v).to(dev)
    wS = torch.zeros(wl.M, dtype=torch.float32, device=dev)
    info = ctx.apd_solve(grid, X, A, v, 0.02, w=wS, opts=apd.make_opts(kernel=TENSOR))
    assert info.status == 0 and info.max_rel_err <= 0.02
    chk = oracle_assign(Grid(wl.dim, wl.n, wl.lo, wl.hi), wl.X, wl.A, wS.cpu().numpy(), v=wl.v)
    P = float(np.prod((np.asarray(wl.hi) - np.asarray(wl.lo)) / np.asarray(wl.n)))
    assert chk.err <= 0.02 + 4 * P / float(wl.v.min())
    ctx.close()
