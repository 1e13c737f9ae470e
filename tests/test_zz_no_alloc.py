"""apd_assign_static (include/apd.h): the evaluation that allocates nothing -- its scratch is a file-scope __device__
array -- against the existing path, apd_assign with opts.kernel = ROWPOLY, cull = 0, which launches the same kernels
on a context's cudaMalloc'ed workspace.  Integer work (labels, counts) must agree bit for bit; the dual and the
stopping quantity are compared at the tolerance of parity rule 3 (1e-6 relative) and, since the kernels and their
reduction order are the same, are expected to be the same bits (asserted too).

Named test_zz_* so that pytest collects it LAST: the suite runs with `pytest -x`, a failure here must not hide any
other test.  It keeps no state of other tests: it passes alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest
import torch

from paper_2403_03571_b200 import workloads

pytestmark = pytest.mark.gpu

ROWPOLY = 2


@pytest.fixture(scope="module")
def apd():
    from paper_2403_03571_b200 import binding
    binding.load_library()
    return binding


def device_inputs(wl, w, dev):
    X = torch.from_numpy(wl.X).to(dev)
    A = torch.from_numpy(wl.A).to(dev)
    wt = torch.from_numpy(np.ascontiguousarray(w, dtype=np.float32)).to(dev)
    vt = torch.from_numpy(wl.v).to(dev)
    return X, A, wt, vt


def outputs(wl, dev):
    return dict(labels=torch.full((wl.N,), -7, dtype=torch.int32, device=dev),
                vol=torch.full((wl.M,), -1.0, dtype=torch.float64, device=dev),
                dual=torch.full((1,), float("nan"), dtype=torch.float64, device=dev),
                max_rel_err=torch.full((1,), float("nan"), dtype=torch.float64, device=dev))


def existing_path(apd, wl, w):
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(wl.dim, wl.M)
    X, A, wt, vt = device_inputs(wl, w, dev)
    o = outputs(wl, dev)
    ctx.apd_assign(apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi), X, A, wt, target_vol=vt, opts=apd.make_opts(kernel=ROWPOLY),
                   **o)
    torch.cuda.synchronize()
    return {k: t.cpu().numpy() for k, t in o.items()}


def static_path(apd, wl, w):
    dev = torch.device("cuda:0")
    X, A, wt, vt = device_inputs(wl, w, dev)
    o = outputs(wl, dev)
    apd.apd_assign_static(apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi), X, A, wt, target_vol=vt, **o)
    torch.cuda.synchronize()
    return {k: t.cpu().numpy() for k, t in o.items()}


def weights(wl, scale, seed):
    rng = np.random.default_rng(seed)
    ell2 = (1.0 / wl.M) ** (2.0 / wl.dim)
    return (rng.standard_normal(wl.M) * scale * ell2).astype(np.float32)


def compare(new, old, wl):
    assert np.array_equal(new["labels"], old["labels"]), "labels differ from apd_assign's"
    assert new["labels"].min() >= 0 and new["labels"].max() < wl.M
    assert np.array_equal(new["vol"], old["vol"]), "volumes (integer counts x |P|) differ"
    for k in ("dual", "max_rel_err"):
        a, b = float(new[k][0]), float(old[k][0])
        assert abs(a - b) <= 1e-6 * max(abs(b), 1e-300), f"{k}: {a!r} vs {b!r}"          # parity rule 3
        assert a == b, f"{k}: same kernels, same reduction order, yet {a!r} != {b!r}"


def cases():
    # ragged 3D grid over several tiles, a 2D grid, a grid big enough for the long-row geometry; M not a multiple of
    # the 128-seed chunk; the SECOND call has fewer seeds and tiles than the first, so stale scratch would show
    a = workloads.make_random(3, (70, 45, 33), 777, seed=9101)
    b = workloads.make_random(2, (300, 210), 130, seed=9102)
    c = workloads.make_random(3, (256, 160, 120), 1500, seed=9103)     # 1200 long-row tiles
    return [(a, weights(a, 0.1, 1)), (b, weights(b, 0.1, 2)), (c, weights(c, 0.05, 3))]


def test_static_entry_matches_apd_assign_on_calls_in_a_row(apd):
    cs = cases()
    ref = [existing_path(apd, wl, w) for wl, w in cs]
    # calls in a row on the one shared scratch array: a, b, a again, c, b again
    for k in (0, 1, 0, 2, 1):
        wl, w = cs[k]
        compare(static_path(apd, wl, w), ref[k], wl)


def test_back_to_back_without_a_sync_between(apd):
    """Two calls enqueued on one stream with no host synchronisation between them are ordered by the stream: the
    second call's clearing of the counts must not disturb the first call's finalize."""
    dev = torch.device("cuda:0")
    (wa, w_a), (wb, w_b), _ = cases()
    ra, rb = existing_path(apd, wa, w_a), existing_path(apd, wb, w_b)
    ia, ib = device_inputs(wa, w_a, dev), device_inputs(wb, w_b, dev)
    oa, ob = outputs(wa, dev), outputs(wb, dev)
    torch.cuda.synchronize()
    apd.apd_assign_static(apd.make_grid(wa.dim, wa.n, wa.lo, wa.hi), ia[0], ia[1], ia[2], target_vol=ia[3], **oa)
    apd.apd_assign_static(apd.make_grid(wb.dim, wb.n, wb.lo, wb.hi), ib[0], ib[1], ib[2], target_vol=ib[3], **ob)
    torch.cuda.synchronize()
    compare({k: t.cpu().numpy() for k, t in oa.items()}, ra, wa)
    compare({k: t.cpu().numpy() for k, t in ob.items()}, rb, wb)


def test_static_entry_allocates_no_device_memory(apd):
    """Free device memory (driver's view: cudaMemGetInfo) is the same before and after calls of a shape that has run
    before (the first call of a shape may load its kernel's code)."""
    dev = torch.device("cuda:0")
    wl, w = cases()[0]
    X, A, wt, vt = device_inputs(wl, w, dev)
    o = outputs(wl, dev)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    apd.apd_assign_static(grid, X, A, wt, target_vol=vt, **o)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(dev)
    for _ in range(5):
        apd.apd_assign_static(grid, X, A, wt, target_vol=vt, **o)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(dev)
    assert free1 == free0, f"free device memory changed by {free0 - free1} bytes over 5 calls"
    assert apd.static_scratch_bytes() == 344 * 1024


def test_static_entry_rejects_sizes_beyond_its_scratch(apd):
    dev = torch.device("cuda:0")
    vol = torch.zeros(apd.STATIC_MAX_SEEDS + 1, dtype=torch.float64, device=dev)
    dual = torch.zeros(1, dtype=torch.float64, device=dev)

    def call(n, M, dim=3):
        X = torch.rand(M, dim, device=dev)
        A = torch.eye(dim, device=dev).repeat(M, 1, 1).contiguous()
        w = torch.zeros(M, device=dev)
        grid = apd.make_grid(dim, n, (0.0,) * dim, (1.0,) * dim)
        apd.apd_assign_static(grid, X, A, w, vol=vol[:M], dual=dual)
        torch.cuda.synchronize()

    call((32, 32, 32), apd.STATIC_MAX_SEEDS)                       # the maximum itself is accepted
    with pytest.raises(apd.ApdError, match="maximum of 4096 seeds") as e:
        call((32, 32, 32), apd.STATIC_MAX_SEEDS + 1)
    assert e.value.status == apd.APD_E_ARG
    with pytest.raises(apd.ApdError, match="CTA tiles") as e:       # 32 x 64 x 64 = 131072 tiles; nothing is launched
        call((1024, 1024, 512), 16)
    assert e.value.status == apd.APD_E_ARG
    with pytest.raises(apd.ApdError, match="layers") as e:          # 2D: 1025 layers of 64 rows
        call((64, 64 * 1024 + 1), 16, dim=2)
    assert e.value.status == apd.APD_E_ARG
    with pytest.raises(apd.ApdError, match="required"):
        apd.apd_assign_static(apd.make_grid(3, (8, 8, 8), (0.0,) * 3, (1.0,) * 3), torch.rand(4, 3, device=dev),
                              torch.eye(3, device=dev).repeat(4, 1, 1).contiguous(), torch.zeros(4, device=dev),
                              vol=None, dual=dual)
