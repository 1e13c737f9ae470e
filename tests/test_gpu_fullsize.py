"""Full-grid, element-by-element GPU <-> oracle parity for EVERY compiled instantiation of the voxel x seed kernels,
at the sizes where each is actually chosen -- above all the ones bench.py times:

  * cfg 4 at full size (256^3 x 10^4): ONE full oracle_assign (~1.7e11 fp64 pairs, about 80 s on 16 host cores) serves
    the long-row ROWPOLY kernel, the TENSOR kernel, the culled kernel and whatever AUTO resolves to: labels (rule 1),
    volumes / counts (rule 2), dual (rule 3), eq. (2.5) error.
  * large 3D grids with few seeds, exact and ragged, so that RowGeom3L (rows of 32 voxels) runs on a grid the oracle
    covers in a second; the same for the 2D long-row geometry RowGeom2L, which needs >= 3.6 M pixels.
  * cfg 5 (512^3 x 2*10^4): a contiguous full z-slab of 8 planes straddling a tile boundary (4.2e10 oracle pairs) with
    counts compared on the slab, beside the random sample of test_gpu_assign.py.
Each test asserts WHICH kernel / geometry ran (apd_assign_stats)."""
import numpy as np
import pytest
import torch

from paper_2403_03571_b200 import workloads
import apd_parity as parity
from test_gpu_assign import run_assign, rand_w

pytestmark = pytest.mark.gpu

K_AUTO, K_DIRECT, K_ROWPOLY, K_TENSOR = 0, 1, 2, 3


@pytest.fixture(scope="module")
def apd():
    from paper_2403_03571_b200 import binding
    binding.load_library()
    return binding


def run_with_stats(apd, wl, w, kernel, cull=0, v=None, want_centroids=False):
    ctx = apd.ApdContext(wl.dim, wl.M)
    r = run_assign(apd, wl, w, v=v, kernel=kernel, cull=cull, want_centroids=want_centroids, ctx=ctx)
    r["stats"] = ctx.assign_stats()
    ctx.close()
    return r


# ------------------------------------------------------------------ cfg 4, full grid, one oracle pass
@pytest.fixture(scope="module")
def cfg4_oracle():
    wl = workloads.make_config(4)
    w = rand_w(wl, 0.1, 204)
    orc = parity.oracle_assign(parity.grid_of(wl), wl.X, wl.A, w, v=wl.v)
    return wl, w, orc


@pytest.mark.parametrize("name,kernel,cull", [("rowpoly_long", K_ROWPOLY, 0), ("tensor", K_TENSOR, 0),
                                              ("culled", K_ROWPOLY, 1), ("auto", K_AUTO, 0), ("auto_culled", K_AUTO, 1)])
def test_cfg4_full_grid_every_kernel(apd, cfg4_oracle, name, kernel, cull):
    wl, w, orc = cfg4_oracle
    r = run_with_stats(apd, wl, w, kernel, cull=cull, v=wl.v, want_centroids=True)
    st = r["stats"]
    if name == "rowpoly_long":
        assert (st["kernel"], st["row_long"], st["cull"]) == (K_ROWPOLY, 1, 0)     # the long-row instantiation
    elif name == "tensor":
        assert st["kernel"] == K_TENSOR
    elif name == "culled":
        assert (st["kernel"], st["cull"]) == (K_ROWPOLY, 1)
    info = parity.check_assign(wl, w, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                               err_gpu=r["err"], orc=orc)
    assert info["mismatches"] < 1e-5 * wl.N
    print(f"cfg4 full grid {name}: ran {st}; {info}")


# ------------------------------------------------------------------ long-row geometries on grids the oracle covers fast
BIG3 = [dict(n=(192, 160, 128), M=300, seed=71), dict(n=(197, 163, 131), M=301, seed=72)]
BIG2 = [dict(n=(2048, 2048), M=200, seed=73), dict(n=(2050, 1999), M=203, seed=74)]


@pytest.mark.parametrize("case", BIG3, ids=lambda c: "x".join(map(str, c["n"])))
@pytest.mark.parametrize("kernel,cull", [(K_ROWPOLY, 0), (K_TENSOR, 0), (K_AUTO, 0), (K_ROWPOLY, 1)])
def test_long_rows_3d_full_grid(apd, case, kernel, cull):
    wl = workloads.make_random(3, case["n"], case["M"], case["seed"], lo=(0.0, -0.5, 1.0), hi=(1.5, 0.75, 2.0),
                               w_scale=0.1, aspect=4.0)
    r = run_with_stats(apd, wl, wl.w0, kernel, cull=cull, v=wl.v, want_centroids=True)
    st = r["stats"]
    if kernel == K_ROWPOLY and not cull:
        assert (st["kernel"], st["row_long"]) == (K_ROWPOLY, 1), st
    info = parity.check_assign(wl, wl.w0, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                               err_gpu=r["err"])
    print(f"3D {wl.n} kernel={kernel} cull={cull}: ran {st}; {info}")


@pytest.mark.parametrize("case", BIG2, ids=lambda c: "x".join(map(str, c["n"])))
@pytest.mark.parametrize("kernel,cull", [(K_ROWPOLY, 0), (K_AUTO, 0), (K_DIRECT, 0), (K_ROWPOLY, 1)])
def test_long_rows_2d_full_grid(apd, case, kernel, cull):
    wl = workloads.make_random(2, case["n"], case["M"], case["seed"], lo=(-1.0, 0.0), hi=(1.0, 2.5), w_scale=0.1,
                               aspect=4.0)
    r = run_with_stats(apd, wl, wl.w0, kernel, cull=cull, v=wl.v, want_centroids=True)
    st = r["stats"]
    if kernel == K_ROWPOLY and not cull:
        assert (st["kernel"], st["row_long"]) == (K_ROWPOLY, 1), st      # RowGeom2L: 64 x 64-pixel tiles
    if kernel == K_AUTO:
        assert st["kernel"] == K_TENSOR, st                              # 2D brute force: tiles of 32 x 16 pixels
    info = parity.check_assign(wl, wl.w0, r["labels"], r["vol"], r["dual"], v=wl.v, centroids_gpu=r["centroids"],
                               err_gpu=r["err"])
    print(f"2D {wl.n} kernel={kernel} cull={cull}: ran {st}; {info}")


# ------------------------------------------------------------------ cfg 5: a full z-slab at full size
@pytest.fixture(scope="module")
def cfg5_slab_oracle():
    wl = workloads.make_config(5)
    w = rand_w(wl, 0.1, 205)
    nx, ny, nz = wl.n
    z0, z1 = nz // 2 - 6, nz // 2 + 2          # 8 planes that straddle a tile boundary of every kernel (tiles of 4 / 8 in z)
    sel = np.arange(z0 * nx * ny, z1 * nx * ny, dtype=np.int64)
    orc = parity.oracle_assign(parity.grid_of(wl), wl.X, wl.A, w, sel=sel)
    return wl, w, sel, orc


@pytest.mark.parametrize("name,kernel,cull", [("rowpoly_long", K_ROWPOLY, 0), ("tensor", K_TENSOR, 0), ("culled", K_AUTO, 1)])
def test_cfg5_full_size_z_slab(apd, cfg5_slab_oracle, name, kernel, cull):
    wl, w, sel, orc = cfg5_slab_oracle
    r = run_with_stats(apd, wl, w, kernel, cull=cull, v=wl.v)
    st = r["stats"]
    if name == "rowpoly_long":
        assert (st["kernel"], st["row_long"]) == (K_ROWPOLY, 1)
    grid = parity.grid_of(wl)
    lab = r["labels"][sel]
    info = parity.check_labels(grid, wl.X, wl.A, w, lab, orc, sel=sel)
    # rule 2 on the slab: counts of the GPU's labels vs the oracle's, over the slab's voxels
    cg = np.bincount(lab, minlength=wl.M).astype(np.int64)
    co = np.bincount(orc.labels, minlength=wl.M).astype(np.int64)
    assert int(np.abs(cg - co).sum()) <= 2 * info["mismatches"]
    # whole grid: vol = integer counts of the GPU's own labels, sum = N
    P = grid.voxel_volume
    cnt = np.rint(r["vol"] / P).astype(np.int64)
    assert int(cnt.sum()) == wl.N and np.array_equal(cnt, np.bincount(r["labels"], minlength=wl.M))
    print(f"cfg5 z-slab {name}: ran {st}; {info}; pruned {1 - r['pairs'] / (wl.N * wl.M):.5f}")


# ------------------------------------------------------------------ labels pointer alignment (int4 stores)
@pytest.mark.parametrize("kernel,cull", [(K_DIRECT, 0), (K_ROWPOLY, 0), (K_ROWPOLY, 1), (K_TENSOR, 0)])
@pytest.mark.parametrize("offset", [1, 2, 3])
def test_labels_pointer_offset_by_a_few_elements(apd, kernel, cull, offset):
    """apd.h asks only int32 alignment of `labels`: a view such as buf[1:] on a grid with nx % 4 == 0 (where rows leave
    as int4 stores when the base is 16-byte aligned) must give the same labels, and touch nothing outside."""
    wl = workloads.make_random(3, (64, 24, 16), 40, 81, w_scale=0.1)
    ref = run_assign(apd, wl, wl.w0, v=wl.v, kernel=kernel, cull=cull)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(3, wl.M)
    buf = torch.full((wl.N + 8,), -7, dtype=torch.int32, device=dev)
    labels = buf[offset:offset + wl.N]
    assert labels.data_ptr() % 16 != 0
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev); dual = torch.zeros(1, dtype=torch.float64, device=dev)
    ctx.apd_assign(apd.make_grid(3, wl.n, wl.lo, wl.hi), torch.from_numpy(wl.X).to(dev), torch.from_numpy(wl.A).to(dev),
                   torch.from_numpy(wl.w0).to(dev), labels=labels, vol=vol, dual=dual,
                   opts=apd.make_opts(kernel=kernel, cull=cull))
    torch.cuda.synchronize()
    out = buf.cpu().numpy()
    assert np.array_equal(out[offset:offset + wl.N], ref["labels"])
    assert np.all(out[:offset] == -7) and np.all(out[offset + wl.N:] == -7)
    ctx.close()


def test_tensor_kernel_padding_seed_never_becomes_a_label(apd):
    """Every real cost NaN (NaN weights) with M % 128 != 0: the TENSOR kernel's padding seeds (finite cost 2^100) must
    not leak out as labels >= M nor index the histograms out of bounds; like the other kernels it returns label 0."""
    wl = workloads.make_random(3, (32, 16, 8), 5, 82)
    w = np.full(wl.M, np.nan, np.float32)
    for kernel in (K_TENSOR, K_ROWPOLY, K_DIRECT):
        r = run_assign(apd, wl, w, kernel=kernel)
        assert r["labels"].min() == 0 and r["labels"].max() == 0, kernel
        assert r["vol"][0] == pytest.approx(np.prod(np.asarray(wl.hi) - np.asarray(wl.lo)))


def test_reserve_then_no_growth(apd):
    """apd_reserve sizes the workspace ahead of time; the calls after it give the same results as without it."""
    wl = workloads.make_config(3, n=(96, 80, 72), M=400)
    ref = run_assign(apd, wl, wl.w0, v=wl.v, cull=1)
    ctx = apd.ApdContext(3, wl.M)
    grid = apd.make_grid(3, wl.n, wl.lo, wl.hi)
    ctx.reserve(grid, apd.make_opts(cull=1))
    ctx.reserve(grid, apd.make_opts(kernel=K_TENSOR))
    r = run_assign(apd, wl, wl.w0, v=wl.v, cull=1, ctx=ctx)
    assert np.array_equal(r["labels"], ref["labels"]) and r["dual"] == ref["dual"]
    with pytest.raises(apd.ApdError):
        ctx.reserve(apd.make_grid(3, (0, 1, 1), (0, 0, 0), (1, 1, 1)))
    ctx.close()
