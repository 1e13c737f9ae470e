"""GPU parity of apd_assign (through the C ABI via the ctypes binding) against the fp64 oracle.
Run on the B200 box with `pytest -m gpu`."""
import numpy as np
import pytest
import torch

from paper_2403_03571_b200 import workloads
import apd_parity as parity

pytestmark = pytest.mark.gpu

KERNELS = {"auto": 0, "direct": 1, "rowpoly": 2}


@pytest.fixture(scope="module")
def apd():
    from paper_2403_03571_b200 import binding
    binding.load_library()
    return binding


def run_assign(apd, wl, w, v=None, kernel=0, want_centroids=False, want_labels=True, ctx=None, cull=0):
    dev = torch.device("cuda:0")
    ctx = ctx or apd.ApdContext(wl.dim, max(wl.M, 1))
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev)
    A = torch.from_numpy(wl.A).to(dev)
    wt = torch.from_numpy(np.ascontiguousarray(w, dtype=np.float32)).to(dev)
    vt = torch.from_numpy(np.ascontiguousarray(v, dtype=np.float32)).to(dev) if v is not None else None
    labels = torch.full((wl.N,), -7, dtype=torch.int32, device=dev) if want_labels else None
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    dual = torch.zeros(1, dtype=torch.float64, device=dev)
    err = torch.zeros(1, dtype=torch.float64, device=dev)
    cen = torch.zeros(wl.M, wl.dim, dtype=torch.float64, device=dev) if want_centroids else None
    pairs = torch.zeros(1, dtype=torch.int64, device=dev)
    ctx.apd_assign(grid, X, A, wt, target_vol=vt, labels=labels, vol=vol, dual=dual, max_rel_err=err,
                   centroids=cen, pairs_evaluated=pairs, opts=apd.make_opts(kernel=kernel, cull=cull))
    torch.cuda.synchronize()
    return dict(labels=labels.cpu().numpy() if want_labels else None, vol=vol.cpu().numpy(),
                dual=float(dual.item()), err=float(err.item()),
                centroids=cen.cpu().numpy() if want_centroids else None, pairs=int(pairs.item()))


def rand_w(wl, scale, seed):
    """Weights of the size that moves boundaries by a fraction of a grain: scale * l^2."""
    rng = np.random.default_rng(seed)
    ext = np.prod(np.asarray(wl.hi) - np.asarray(wl.lo))
    ell2 = (ext / wl.M) ** (2.0 / wl.dim)
    return (rng.standard_normal(wl.M) * scale * ell2).astype(np.float32)


# ------------------------------------------------------------------ BASELINE configs 1-3, full size
@pytest.mark.parametrize("kernel", ["direct", "auto"])
@pytest.mark.parametrize("cfg", [1, 2, 3])
@pytest.mark.parametrize("wscale", [0.0, 0.15])
def test_configs_full_parity(apd, cfg, kernel, wscale):
    wl = workloads.make_config(cfg)
    w = wl.w0 if wscale == 0.0 else rand_w(wl, wscale, 100 + cfg)
    r = run_assign(apd, wl, w, v=wl.v, kernel=KERNELS[kernel], want_centroids=True)
    info = parity.check_assign(wl, w, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                               err_gpu=r["err"])
    assert r["pairs"] == wl.N * wl.M
    print(f"cfg{cfg} {kernel} wscale={wscale}: {info}")


# ------------------------------------------------------------------ configs 4-5 at full size: sampled voxels
@pytest.mark.parametrize("kernel,cull", [("auto", 0), ("auto", 1)])
@pytest.mark.parametrize("cfg,nsample", [(4, 60000), (5, 30000)])
def test_large_configs_sampled_parity(apd, cfg, nsample, kernel, cull):
    from oracle.apd_oracle import oracle_assign
    wl = workloads.make_config(cfg)
    w = rand_w(wl, 0.1, 200 + cfg)
    r = run_assign(apd, wl, w, v=wl.v, kernel=KERNELS[kernel], cull=cull)
    assert (r["pairs"] == wl.N * wl.M) if not cull else (0 < r["pairs"] < 0.02 * wl.N * wl.M)
    grid = parity.grid_of(wl)
    sel = workloads.voxel_sample(wl.N, nsample, cfg)
    orc = oracle_assign(grid, wl.X, wl.A, w, sel=sel)
    info = parity.check_labels(grid, wl.X, wl.A, w, r["labels"][sel], orc, sel=sel)
    # properties that hold at any size
    P = grid.voxel_volume
    cnt = np.rint(r["vol"] / P).astype(np.int64)
    assert int(cnt.sum()) == wl.N
    assert np.array_equal(cnt, np.bincount(r["labels"], minlength=wl.M))
    # dual = <v,w> + |P| sum_j min_i C_ij : estimate the second term from the sample (law of large numbers)
    est = float(np.dot(wl.v.astype(np.float64), w.astype(np.float64))) + float(np.mean(orc.best))
    se = float(np.std(orc.best)) / np.sqrt(len(sel))
    assert abs(r["dual"] - est) < 6 * se + 1e-9
    print(f"cfg{cfg} cull={cull} sampled: {info}; pruned fraction {1 - r['pairs'] / (wl.N * wl.M):.5f}")


# ------------------------------------------------------------------ edge cases
EDGE = [
    dict(dim=2, n=(100, 75), M=37, lo=(0.0, -1.0), hi=(2.0, 0.5), seed=1),          # non-pow2, non-unit box
    dict(dim=3, n=(50, 60, 70), M=130, lo=(0, 0, 0), hi=(1, 1, 1), seed=2),          # M not a chunk multiple
    dict(dim=3, n=(33, 17, 9), M=5, lo=(-1, 2, 0), hi=(1, 5, 0.5), seed=3),          # ragged tiles everywhere
    dict(dim=2, n=(1, 1), M=3, lo=(0, 0), hi=(1, 1), seed=4),                        # one pixel
    dict(dim=3, n=(5, 1, 1), M=1, lo=(0, 0, 0), hi=(1, 1, 1), seed=5),               # one seed
    dict(dim=2, n=(257, 3), M=2, lo=(0, 0), hi=(1, 1), seed=6),
    dict(dim=3, n=(64, 64, 64), M=129, lo=(0, 0, 0), hi=(1, 1, 1), seed=7),
    dict(dim=2, n=(130, 131), M=300, lo=(0, 0), hi=(3, 3), seed=8),
]


@pytest.mark.parametrize("kernel", ["direct", "auto"])
@pytest.mark.parametrize("case", EDGE, ids=lambda c: f"{c['dim']}d_{'x'.join(map(str, c['n']))}_M{c['M']}")
@pytest.mark.parametrize("nonsym", [False, True])
def test_edge_cases(apd, case, kernel, nonsym):
    wl = workloads.make_random(case["dim"], case["n"], case["M"], case["seed"], lo=case["lo"], hi=case["hi"],
                               w_scale=0.1, nonsymmetric=nonsym)
    r = run_assign(apd, wl, wl.w0, v=wl.v, kernel=KERNELS[kernel], want_centroids=True)
    parity.check_assign(wl, wl.w0, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                        err_gpu=r["err"])


@pytest.mark.parametrize("kernel", ["direct", "auto"])
def test_no_target_volume_and_no_labels(apd, kernel):
    wl = workloads.make_random(3, (40, 24, 16), 50, 21, w_scale=0.1)
    r = run_assign(apd, wl, wl.w0, v=None, kernel=KERNELS[kernel])
    parity.check_assign(wl, wl.w0, r["labels"], r["vol"], r["dual"], v=None)
    r2 = run_assign(apd, wl, wl.w0, v=None, kernel=KERNELS[kernel], want_labels=False)
    assert r2["dual"] == r["dual"] and np.array_equal(r2["vol"], r["vol"])     # bitwise reproducible


@pytest.mark.parametrize("kernel,cull", [("direct", 0), ("auto", 0), ("auto", 1)])
@pytest.mark.parametrize("dim", [2, 3])
def test_exact_ties_lowest_index(apd, kernel, cull, dim):
    """Mirror-symmetric seeds on a power-of-two grid: costs are exactly equal in fp32 AND fp64 on the
    mirror plane's neighbours... here seeds are duplicated, so every voxel ties: lowest index wins (S1)."""
    wl = workloads.make_random(dim, (32,) * dim, 6, 31)
    X = np.concatenate([wl.X, wl.X]); A = np.concatenate([wl.A, wl.A])
    wl2 = workloads.Workload("dup", dim, wl.n, wl.lo, wl.hi, X, A, np.full(12, 1 / 12, np.float32),
                             np.zeros(12, np.float32))
    r = run_assign(apd, wl2, wl2.w0, kernel=KERNELS[kernel], cull=cull)
    assert r["labels"].max() < 6
    parity.check_assign(wl2, wl2.w0, r["labels"], r["vol"], r["dual"])


@pytest.mark.parametrize("kernel", ["direct", "auto"])
def test_empty_cell_centroid_is_seed(apd, kernel):
    wl = workloads.make_random(2, (64, 64), 9, 41)
    w = np.zeros(9, np.float32); w[3] = -10.0          # cell 3 cannot win anywhere
    r = run_assign(apd, wl, w, v=wl.v, kernel=KERNELS[kernel], want_centroids=True)
    assert r["vol"][3] == 0.0
    np.testing.assert_array_equal(r["centroids"][3], wl.X[3].astype(np.float64))
    parity.check_assign(wl, w, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"])


@pytest.mark.parametrize("kernel,cull", [("direct", 0), ("auto", 0), ("auto", 1)])
def test_P11_exact_scaling_symmetry(apd, kernel, cull):
    """(A, w) -> (2A, 2w) doubles every fp32 cost exactly: labels identical, dual doubles exactly."""
    wl = workloads.make_config(3, n=(64, 64, 64), M=200)
    w = rand_w(wl, 0.1, 7)
    r1 = run_assign(apd, wl, w, kernel=KERNELS[kernel], cull=cull)
    wl2 = workloads.Workload("x2", wl.dim, wl.n, wl.lo, wl.hi, wl.X, (2 * wl.A).astype(np.float32), wl.v, wl.w0)
    r2 = run_assign(apd, wl2, (2 * w).astype(np.float32), kernel=KERNELS[kernel], cull=cull)
    assert np.array_equal(r1["labels"], r2["labels"])
    assert r2["dual"] == 2.0 * r1["dual"]


def test_kernels_agree_bitwise(apd):
    """DIRECT and the default kernel use different fp32 association, so they may differ on near-ties only."""
    wl = workloads.make_config(3, n=(96, 96, 96), M=700)
    w = rand_w(wl, 0.1, 9)
    a = run_assign(apd, wl, w, kernel=1)
    b = run_assign(apd, wl, w, kernel=0)
    assert np.mean(a["labels"] != b["labels"]) < 1e-5


def test_argument_errors(apd):
    ctx = apd.ApdContext(2, 16)
    wl = workloads.make_random(2, (8, 8), 4, 1)
    dev = torch.device("cuda:0")
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); w = torch.zeros(4, device=dev)
    vol = torch.zeros(4, dtype=torch.float64, device=dev); dual = torch.zeros(1, dtype=torch.float64, device=dev)
    bad = apd.make_grid(2, (8, 0), (0, 0), (1, 1))
    with pytest.raises(apd.ApdError) as e:
        ctx.apd_assign(bad, X, A, w, vol=vol, dual=dual)
    assert e.value.status == apd.APD_E_ARG
    bad = apd.make_grid(2, (8, 8), (0, 0), (1, 0))
    with pytest.raises(apd.ApdError):
        ctx.apd_assign(bad, X, A, w, vol=vol, dual=dual)
    g3 = apd.make_grid(3, (8, 8, 8), (0, 0, 0), (1, 1, 1))
    wl3 = workloads.make_random(3, (8, 8, 8), 4, 1)
    with pytest.raises(apd.ApdError):                             # dim differs from the context's
        ctx.apd_assign(g3, torch.from_numpy(wl3.X).to(dev), torch.from_numpy(wl3.A).to(dev), w, vol=vol, dual=dual)
    ok = apd.make_grid(2, (8, 8), (0, 0), (1, 1))
    with pytest.raises(apd.ApdError):
        ctx.apd_assign(ok, X, A, w, vol=vol, dual=dual, opts=apd.make_opts(kernel=99))
    big = workloads.make_random(2, (8, 8), 17, 1)
    with pytest.raises(apd.ApdError):
        ctx.apd_assign(ok, torch.from_numpy(big.X).to(dev), torch.from_numpy(big.A).to(dev),
                       torch.zeros(17, device=dev), vol=torch.zeros(17, dtype=torch.float64, device=dev), dual=dual)
    with pytest.raises(apd.ApdError):
        apd.ApdContext(4, 16)


def test_host_call_matches_device_call(apd):
    wl = workloads.make_random(3, (48, 40, 24), 77, 51, w_scale=0.1)
    r = run_assign(apd, wl, wl.w0, v=wl.v, want_centroids=True)
    ctx = apd.ApdContext(3, 77)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    labels = torch.empty(wl.N, dtype=torch.int32); vol = torch.empty(wl.M, dtype=torch.float64)
    cen = torch.empty(wl.M, 3, dtype=torch.float64)
    dual, err, pairs = ctx.apd_assign_host(grid, torch.from_numpy(wl.X), torch.from_numpy(wl.A),
                                           torch.from_numpy(wl.w0), target_vol=torch.from_numpy(wl.v),
                                           labels=labels, vol=vol, centroids=cen)
    assert np.array_equal(labels.numpy(), r["labels"]) and np.array_equal(vol.numpy(), r["vol"])
    assert dual == r["dual"] and err == r["err"] and pairs == wl.N * wl.M
    assert np.array_equal(cen.numpy(), r["centroids"])
    ctx.close()


@pytest.mark.parametrize("kernel,cull", [("direct", 0), ("auto", 0), ("auto", 1), ("tensor", 0)])
def test_host_call_with_pinned_labels_writes_them_in_place(apd, kernel, cull):
    """apd_assign_host stores the labels straight into PINNED host memory (no device buffer, no copy afterwards); the
    result is the device call's, bit for bit, on a grid with ragged tiles (scalar and vector label stores)."""
    kid = {"tensor": 3}.get(kernel, KERNELS.get(kernel, 0))
    wl = workloads.make_random(3, (52, 40, 23), 77, 52, w_scale=0.1)
    r = run_assign(apd, wl, wl.w0, v=wl.v, kernel=kid, cull=cull)
    ctx = apd.ApdContext(3, 77)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    labels = torch.full((wl.N,), -7, dtype=torch.int32).pin_memory()
    vol = torch.empty(wl.M, dtype=torch.float64).pin_memory()
    dual, err, pairs = ctx.apd_assign_host(grid, torch.from_numpy(wl.X).pin_memory(), torch.from_numpy(wl.A).pin_memory(),
                                           torch.from_numpy(wl.w0).pin_memory(), target_vol=torch.from_numpy(wl.v).pin_memory(),
                                           labels=labels, vol=vol, opts=apd.make_opts(kernel=kid, cull=cull))
    assert np.array_equal(labels.numpy(), r["labels"]) and np.array_equal(vol.numpy(), r["vol"])
    assert dual == r["dual"] and err == r["err"]
    ctx.close()


# ------------------------------------------------------------------ a7: exact tile culling
@pytest.mark.parametrize("cfg,n,M", [(1, None, None), (2, None, None), (3, None, None), (4, (160, 128, 96), 3000),
                                     (5, (128, 128, 128), 2500)])
@pytest.mark.parametrize("wscale", [0.0, 0.2])
def test_culling_is_exact(apd, cfg, n, M, wscale):
    """Labels, volumes and centroids with culling == ROWPOLY without, bit for bit (grids small enough that brute force
    runs the same short-row arithmetic as the culled kernel); the dual up to the order of the fp64 partial sums."""
    wl = workloads.make_config(cfg, n=n, M=M)
    w = wl.w0 if wscale == 0.0 else rand_w(wl, wscale, 300 + cfg)
    r0 = run_assign(apd, wl, w, v=wl.v, want_centroids=True, cull=0, kernel=KERNELS["rowpoly"])   # (AUTO would take
    r1 = run_assign(apd, wl, w, v=wl.v, want_centroids=True, cull=1, kernel=KERNELS["rowpoly"])   #  TENSOR at M >= 384)
    assert np.array_equal(r0["labels"], r1["labels"])
    assert np.array_equal(r0["vol"], r1["vol"]) and np.array_equal(r0["centroids"], r1["centroids"])
    assert abs(r1["dual"] - r0["dual"]) <= 1e-13 * abs(r0["dual"]) and r1["err"] == r0["err"]   # same fp32 minima
    assert 0 < r1["pairs"] <= wl.N * wl.M and r0["pairs"] == wl.N * wl.M
    print(f"cfg{cfg} {wl.n} M={wl.M} wscale={wscale}: pruned fraction {1 - r1['pairs'] / (wl.N * wl.M):.4f}")


@pytest.mark.parametrize("case", EDGE, ids=lambda c: f"{c['dim']}d_{'x'.join(map(str, c['n']))}_M{c['M']}")
def test_culling_edge_cases_parity(apd, case):
    wl = workloads.make_random(case["dim"], case["n"], case["M"], case["seed"], lo=case["lo"], hi=case["hi"],
                               w_scale=0.1, aspect=5.0)
    r = run_assign(apd, wl, wl.w0, v=wl.v, want_centroids=True, cull=1)
    parity.check_assign(wl, wl.w0, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                        err_gpu=r["err"])
    r0 = run_assign(apd, wl, wl.w0, v=wl.v, cull=0, kernel=KERNELS["rowpoly"])
    assert np.array_equal(r0["labels"], r["labels"])


def test_culling_extreme_weights_and_overflow(apd):
    """One seed with a huge weight owns everything; every seed coincident => every brick list overflows BRICK_CAP
    (256) and falls back to its super-tile's list, and beyond SUPER_CAP (4096) to scanning all seeds."""
    wl = workloads.make_random(3, (64, 48, 40), 300, 31, w_scale=0.1)
    w = wl.w0.copy(); w[17] = 10.0
    r = run_assign(apd, wl, w, v=wl.v, cull=1)
    assert np.all(r["labels"] == 17)
    wl2 = workloads.make_random(3, (40, 40, 40), 1500, 32)
    wl2.X[:] = wl2.X[0]; wl2.A[:] = wl2.A[0]                 # coincident, identical seeds: nothing can be pruned
    r0 = run_assign(apd, wl2, wl2.w0, v=wl2.v, cull=0)
    r1 = run_assign(apd, wl2, wl2.w0, v=wl2.v, cull=1)
    assert np.all(r0["labels"] == 0) and np.array_equal(r0["labels"], r1["labels"])
    assert r1["pairs"] == wl2.N * wl2.M
    # more coincident seeds than a super-tile list holds (4096): brick -> super-tile -> all seeds
    wl3 = workloads.make_random(3, (20, 12, 10), 4200, 33)
    wl3.X[:] = wl3.X[0]; wl3.A[:] = wl3.A[0]
    r3 = run_assign(apd, wl3, wl3.w0, v=wl3.v, cull=1)
    assert np.all(r3["labels"] == 0) and r3["pairs"] == wl3.N * wl3.M


def test_culling_rejects_direct_kernel(apd):
    wl = workloads.make_config(1)
    with pytest.raises(apd.ApdError) as e:
        run_assign(apd, wl, wl.w0, kernel=KERNELS["direct"], cull=1)
    assert e.value.status == apd.APD_E_ARG


@pytest.mark.parametrize("dim,n", [(2, (5, 200)), (3, (64, 6, 64)), (3, (64, 64, 3)), (3, (3, 40, 40))])
def test_narrow_grids_take_the_direct_kernel(apd, dim, n):
    """AUTO on a grid narrower than half a tile of the row kernels (include/apd.h) runs DIRECT and ignores opts.cull:
    bit-identical outputs, N*M pairs.  An explicit ROWPOLY is honoured and stays inside the parity rule with the dual
    bound of the expansion about a midpoint up to 8/n domain widths L outside the domain: a few fp32 ulp of
    a ((1 + 8/n) L)^2 per cost, i.e. ((1 + 8/n) L / l)^2 ulp relative to costs of the size a l^2 (l = grain size)."""
    wl = workloads.make_random(dim, n, 60, 4242, w_scale=0.1)
    rd = run_assign(apd, wl, wl.w0, v=wl.v, kernel=KERNELS["direct"])
    for cull in (0, 1):
        ra = run_assign(apd, wl, wl.w0, v=wl.v, kernel=KERNELS["auto"], cull=cull)
        assert np.array_equal(ra["labels"], rd["labels"]) and ra["dual"] == rd["dual"] and ra["pairs"] == wl.N * wl.M
    parity.check_assign(wl, wl.w0, rd["labels"], rd["vol"], rd["dual"], v=wl.v, err_gpu=rd["err"])
    rr = run_assign(apd, wl, wl.w0, v=wl.v, kernel=KERNELS["rowpoly"])
    orc = parity.oracle_assign(parity.grid_of(wl), wl.X, wl.A, wl.w0, v=wl.v)
    parity.check_labels(parity.grid_of(wl), wl.X, wl.A, wl.w0, rr["labels"], orc)
    ell = (1.0 / wl.M) ** (1.0 / dim)                       # unit box
    rel = 2.0 ** -23 * ((1.0 + 8.0 / min(n)) / ell) ** 2
    assert abs(rr["dual"] - orc.dual) <= rel * max(abs(orc.dual), abs(orc.quad_part))


def test_slab_decomposition_is_exact(apd):
    """The path shards by voxel slabs with the EXISTING call: a z-slab is an apd_grid with
    shifted lo/hi and fewer n_z.  On a power-of-two grid the slab's voxel centres are bit-identical, so labels
    concatenate and the integer counts / min-cost sums add up exactly to the single-grid evaluation."""
    wl = workloads.make_config(3, n=(64, 64, 64), M=300)
    w = rand_w(wl, 0.15, 77)
    full = run_assign(apd, wl, w, v=None)
    labs, vol, dual = [], np.zeros(wl.M), 0.0
    for z0, z1 in ((0, 16), (16, 48), (48, 64)):
        part = workloads.Workload("slab", 3, (64, 64, z1 - z0), (0.0, 0.0, z0 / 64.0), (1.0, 1.0, z1 / 64.0),
                                  wl.X, wl.A, wl.v, wl.w0)
        r = run_assign(apd, part, w, v=None)
        labs.append(r["labels"]); vol += r["vol"]; dual += r["dual"]
    assert np.array_equal(np.concatenate(labs), full["labels"])
    assert np.array_equal(vol, full["vol"])                       # integer counts x |P| (a power of two): exact
    assert abs(dual - full["dual"]) <= 1e-13 * abs(full["dual"])  # same minima, different partial-sum order
