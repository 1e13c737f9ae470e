"""include/apd.h states that apd_assign_static never allocates and that, after apd_reserve, apd_assign neither allocates
nor synchronises.  The sharpest check of both is stream capture, which forbids either: the calls are captured into a CUDA
graph (torch.cuda.graph), replayed at other weights, and must give bit for bit what the eager calls give.  The culled
path's kernels are launched with programmatic dependent launch, which capture turns into programmatic graph edges."""
import numpy as np
import pytest
import torch

from paper_2403_03571_b200 import workloads
from test_gpu_assign import apd  # noqa: F401  (module fixture)

pytestmark = pytest.mark.gpu


def _buffers(wl, dev):
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    return dict(X=t(wl.X), A=t(wl.A), v=t(wl.v), w=torch.zeros(wl.M, dtype=torch.float32, device=dev),
                labels=torch.empty(wl.N, dtype=torch.int32, device=dev),
                vol=torch.zeros(wl.M, dtype=torch.float64, device=dev),
                dual=torch.zeros(1, dtype=torch.float64, device=dev), err=torch.zeros(1, dtype=torch.float64, device=dev))


def _replay_equals_eager(wl, b, call):
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        call()                                  # warm-up on a side stream, as torch asks before a capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        call()
    for rep in range(3):
        b["w"].copy_(torch.from_numpy((0.002 * rep * np.arange(wl.M) / wl.M).astype(np.float32)))
        b["labels"].fill_(-1); b["vol"].zero_(); b["dual"].zero_(); b["err"].zero_()
        g.replay()
        torch.cuda.synchronize()
        got = [b[k].clone() for k in ("labels", "vol", "dual", "err")]
        call()
        torch.cuda.synchronize()
        for k, t in zip(("labels", "vol", "dual", "err"), got):
            assert torch.equal(t, b[k]), f"replay {rep}: {k} differs from the eager call"
        assert int(b["labels"].min()) >= 0 and abs(float(b["vol"].sum()) - 1.0) < 1e-9


@pytest.mark.parametrize("dim,n,M", [(3, (64, 64, 40), 200), (2, (300, 200), 90)])
def test_static_entry_under_stream_capture(apd, dim, n, M):
    dev = torch.device("cuda:0")
    wl = workloads.make_config(3 if dim == 3 else 2, n=n, M=M)
    b = _buffers(wl, dev)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    _replay_equals_eager(wl, b, lambda: apd.apd_assign_static(grid, b["X"], b["A"], b["w"], target_vol=b["v"],
                                                              labels=b["labels"], vol=b["vol"], dual=b["dual"],
                                                              max_rel_err=b["err"]))


@pytest.mark.parametrize("kernel,cull", [(0, 0), (2, 0), (0, 1)])
@pytest.mark.parametrize("dim,n,M", [(3, (64, 64, 40), 200), (2, (300, 200), 90)])
def test_assign_after_reserve_under_stream_capture(apd, dim, n, M, kernel, cull):
    dev = torch.device("cuda:0")
    wl = workloads.make_config(3 if dim == 3 else 2, n=n, M=M)
    b = _buffers(wl, dev)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    ctx = apd.ApdContext(wl.dim, wl.M)
    o = apd.make_opts(kernel=kernel, cull=cull)
    ctx.reserve(grid, o)
    _replay_equals_eager(wl, b, lambda: ctx.apd_assign(grid, b["X"], b["A"], b["w"], target_vol=b["v"], labels=b["labels"],
                                                       vol=b["vol"], dual=b["dual"], max_rel_err=b["err"], opts=o))
    ctx.close()
