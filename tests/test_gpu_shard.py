"""Voxel-slab sharding (row f4) on the GPU: the raw counters of the slabs of a partition, summed word
by word, give the whole-grid evaluation BIT FOR BIT (labels, volumes, dual, centroids) for every kernel; apd_solve_slab
with a counter exchange between two processes (gloo, both on cuda:0 -- their kernels never wait on one another, the
hosts meet in the allreduce) walks the whole-grid apd_solve trajectory bit for bit.  Unmeasured on multi-GPU hardware."""
import json
import os
import sys

import numpy as np
import pytest
import torch

from paper_2403_03571_b200 import workloads
from test_gpu_assign import run_assign

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def apd():
    from paper_2403_03571_b200 import binding
    binding.load_library()
    return binding


CASES = [dict(dim=3, n=(52, 40, 44), lo=(0.0, -1.0, 0.5), hi=(1.3, 0.4, 1.6), M=70, slabs=[(0, 16), (16, 24), (40, 4)]),
         dict(dim=3, n=(64, 64, 64), lo=(0, 0, 0), hi=(1, 1, 1), M=300, slabs=[(0, 8), (8, 56)]),
         dict(dim=2, n=(100, 200), lo=(0.0, 0.0), hi=(2.0, 3.0), M=45, slabs=[(0, 64), (64, 128), (192, 8)])]


@pytest.mark.parametrize("kernel,cull", [(1, 0), (2, 0), (2, 1), (3, 0), (0, 0)])
@pytest.mark.parametrize("case", CASES, ids=lambda c: "x".join(map(str, c["n"])))
def test_slab_counters_add_up_to_the_whole_grid_bit_for_bit(apd, case, kernel, cull):
    wl = workloads.make_random(case["dim"], case["n"], case["M"], 91, lo=case["lo"], hi=case["hi"], w_scale=0.1, aspect=4.0)
    ref = run_assign(apd, wl, wl.w0, v=wl.v, kernel=kernel, cull=cull, want_centroids=True)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(wl.dim, wl.M)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); w = torch.from_numpy(wl.w0).to(dev)
    v = torch.from_numpy(wl.v).to(dev)
    words = apd.counter_words(grid, wl.M, True)
    total = torch.zeros(words, dtype=torch.int64, device=dev)
    per_plane = int(np.prod(wl.n[:-1]))
    labs = []
    assert apd.slab_align(wl.dim) == (8 if wl.dim == 3 else 64)
    for lo, n in case["slabs"]:
        c = torch.full((words,), -1, dtype=torch.int64, device=dev)
        lab = torch.full((per_plane * n,), -7, dtype=torch.int32, device=dev)
        ctx.apd_assign_slab(grid, (lo, n), X, A, w, labels=lab, counters=c, with_idxsum=True,
                            opts=apd.make_opts(kernel=kernel, cull=cull))
        total += c                                        # the word-wise integer sum an allreduce would do
        labs.append(lab.cpu().numpy())
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev); dual = torch.zeros(1, dtype=torch.float64, device=dev)
    err = torch.zeros(1, dtype=torch.float64, device=dev); cen = torch.zeros(wl.M, wl.dim, dtype=torch.float64, device=dev)
    ctx.apd_finalize_counters(grid, total, X, w, target_vol=v, vol=vol, dual=dual, max_rel_err=err, centroids=cen,
                              with_idxsum=True)
    torch.cuda.synchronize()
    assert np.array_equal(np.concatenate(labs), ref["labels"])
    assert np.array_equal(vol.cpu().numpy(), ref["vol"])
    assert float(dual.item()) == ref["dual"], (float(dual.item()), ref["dual"])         # bit for bit
    assert float(err.item()) == ref["err"]
    assert np.array_equal(cen.cpu().numpy(), ref["centroids"])
    ctx.close()


def test_slab_argument_errors(apd):
    wl = workloads.make_random(3, (32, 32, 32), 10, 5)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(3, 10)
    grid = apd.make_grid(3, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); w = torch.from_numpy(wl.w0).to(dev)
    c = torch.zeros(apd.counter_words(grid, 10), dtype=torch.int64, device=dev)
    for bad in [(4, 8), (0, 12), (24, 16), (0, 0), (-8, 8)]:       # unaligned lo, unaligned n inside, past the end, empty
        with pytest.raises(apd.ApdError) as e:
            ctx.apd_assign_slab(grid, bad, X, A, w, counters=c)
        assert e.value.status == apd.APD_E_ARG
    ctx.apd_assign_slab(grid, (24, 8), X, A, w, counters=c)
    ctx.close()


def _solve_whole(apd, wl, eps, kernel, cull):
    from test_gpu_solve import run_solve
    info, w32, w64, labels, vol, hist = run_solve(apd, wl, eps, kernel=kernel, cull=cull, want_hist=True)
    return info, w32, labels, vol, hist


@pytest.mark.parametrize("kernel,cull", [(2, 0), (2, 1), (3, 0)])
def test_solve_slab_single_slab_is_apd_solve(apd, kernel, cull):
    """One slab covering the grid, no reduce: the u64 / reduced-layer path of the optimiser kernel gives apd_solve's
    trajectory bit for bit."""
    wl = workloads.make_config(4, n=(64, 48, 40), M=90)
    info0, w0, lab0, vol0, hist0 = _solve_whole(apd, wl, 0.02, kernel, cull)
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(3, wl.M)
    grid = apd.make_grid(3, wl.n, wl.lo, wl.hi)
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); v = torch.from_numpy(wl.v).to(dev)
    w = torch.zeros(wl.M, dtype=torch.float32, device=dev); lab = torch.empty(wl.N, dtype=torch.int32, device=dev)
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    c = torch.zeros(apd.counter_words(grid, wl.M), dtype=torch.int64, device=dev)
    info = ctx.apd_solve_slab(grid, (0, wl.n[2]), X, A, v, 0.02, c, reduce=None, w=w, labels=lab, vol=vol,
                              opts=apd.make_opts(kernel=kernel, cull=cull))
    hist = ctx.solve_history()
    assert (info.status, info.iters, info.evals) == (info0.status, info0.iters, info0.evals)
    assert np.array_equal(w.cpu().numpy(), w0) and np.array_equal(lab.cpu().numpy(), lab0)
    assert np.array_equal(vol.cpu().numpy(), vol0)
    assert np.array_equal(hist[0], hist0[0]) and np.array_equal(hist[1], hist0[1])      # dual and error histories
    ctx.close()


def _rank(rank, world, port, out, cfg, n, M, eps, kernel, cull):
    sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))
    import torch.distributed as dist
    from paper_2403_03571_b200 import binding as apd, workloads as W
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.make_config(cfg, n=n, M=M)
    info0, w0, lab0, vol0, hist0 = _solve_whole(apd, wl, eps, kernel, cull)           # the single-call solve, locally
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(wl.dim, wl.M)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    lo, ns = apd.slab_partition(wl.n[-1], world, apd.slab_align(wl.dim))[rank]
    per_plane = int(np.prod(wl.n[:-1]))
    X = torch.from_numpy(wl.X).to(dev); A = torch.from_numpy(wl.A).to(dev); v = torch.from_numpy(wl.v).to(dev)
    w = torch.zeros(wl.M, dtype=torch.float32, device=dev); lab = torch.empty(per_plane * ns, dtype=torch.int32, device=dev)
    vol = torch.zeros(wl.M, dtype=torch.float64, device=dev)
    c = torch.zeros(apd.counter_words(grid, wl.M), dtype=torch.int64, device=dev)
    n_reduce = [0]

    def reduce():
        n_reduce[0] += 1
        dist.all_reduce(c)              # gloo on a CUDA tensor: ordered after the work on the current stream; SUM of int64

    info = ctx.apd_solve_slab(grid, (lo, ns), X, A, v, eps, c, reduce=reduce, w=w, labels=lab, vol=vol,
                              opts=apd.make_opts(kernel=kernel, cull=cull))
    hist = ctx.solve_history()
    res = dict(rank=rank, slab=[lo, ns], status=info.status, iters=info.iters, evals=info.evals, n_reduce=n_reduce[0],
               same_counts=(info.status, info.iters, info.evals) == (info0.status, info0.iters, info0.evals),
               same_w=bool(np.array_equal(w.cpu().numpy(), w0)),
               same_labels=bool(np.array_equal(lab.cpu().numpy(), lab0[per_plane * lo: per_plane * (lo + ns)])),
               same_vol=bool(np.array_equal(vol.cpu().numpy(), vol0)),
               same_hist=bool(np.array_equal(hist[0], hist0[0]) and np.array_equal(hist[1], hist0[1])))
    allres = [None] * world
    dist.all_gather_object(allres, res)
    if rank == 0:
        json.dump(allres, open(out, "w"))
    ctx.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("cfg,n,M,eps,kernel,cull", [(4, (64, 48, 40), 90, 0.02, 2, 1), (3, (48, 48, 48), 60, 0.01, 3, 0),
                                                     (2, (192, 256), 50, 0.01, 2, 0), (5, (40, 40, 72), 80, 0.02, 2, 0)])
def test_sharded_solve_two_processes_is_the_single_call_trajectory(apd, tmp_path, cfg, n, M, eps, kernel, cull):
    import torch.multiprocessing as mp
    out = str(tmp_path / "r.json")
    port = 29500 + (os.getpid() * 13 + cfg) % 2000
    mp.spawn(_rank, args=(2, port, out, cfg, n, M, eps, kernel, cull), nprocs=2, join=True)
    res = json.load(open(out))
    assert len(res) == 2 and res[0]["slab"][0] == 0 and sum(r["slab"][1] for r in res) == n[-1]
    for r in res:
        assert r["same_counts"] and r["same_w"] and r["same_labels"] and r["same_vol"] and r["same_hist"], r
        assert r["n_reduce"] >= r["evals"] + 1             # one exchange per evaluation + the final labelled one
    assert res[0]["n_reduce"] == res[1]["n_reduce"]        # every rank calls the collective equally often
