"""apd_validate (include/apd.h): the input checks the hot path does not make (the paper's standing
assumptions PAPER.md:51-54 on A_i and PAPER.md:65-69 on the target volumes), through the C ABI on the GPU.  The expected
flags come from numpy (eigenvalues of the symmetric part, sums), not from the library."""
import numpy as np
import pytest
import torch

from paper_2403_03571_b200 import workloads
from test_gpu_assign import apd  # noqa: F401  (module fixture)

pytestmark = pytest.mark.gpu


def _run(apd, wl, X=None, A=None, w=None, v=None, with_grid=True, with_w=True, with_v=True):
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(wl.dim, wl.M)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi) if with_grid else None
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
    f = ctx.validate(grid, t(wl.X if X is None else X), t(wl.A if A is None else A),
                     t(wl.w0 if w is None else w) if with_w else None, t(wl.v if v is None else v) if with_v else None)
    ctx.close()
    return f


@pytest.mark.parametrize("dim,n,M", [(2, (64, 64), 37), (3, (32, 32, 32), 300)])
def test_clean_inputs_and_each_flag(apd, dim, n, M):
    wl = workloads.make_random(dim, n, M, 5150 + dim, w_scale=0.1)
    # the generator's matrices are symmetric positive definite (checked here, independently of the library)
    for Ai in wl.A.astype(np.float64):
        assert np.allclose(Ai, Ai.T, atol=1e-6 * np.abs(Ai).max()) and np.linalg.eigvalsh(0.5 * (Ai + Ai.T)).min() > 0
    assert _run(apd, wl) == 0
    assert _run(apd, wl, with_grid=False, with_v=False, with_w=False) == 0

    X = wl.X.copy(); X[M // 2, dim - 1] = np.nan
    assert _run(apd, wl, X=X) == apd.BAD_X_NONFINITE
    A = wl.A.copy(); A[3, 0, 1] = np.inf
    assert _run(apd, wl, A=A) == apd.BAD_A_NONFINITE
    A = wl.A.copy(); A[M - 1, 0, 1] += 0.01 * np.abs(A[M - 1]).max()         # the last seed: a partial warp
    f = _run(apd, wl, A=A)
    assert f & apd.BAD_A_NOT_SYMMETRIC and not f & ~(apd.BAD_A_NOT_SYMMETRIC | apd.BAD_A_NOT_POSITIVE_DEFINITE)
    # indefinite: flip the sign of the smallest eigenvalue of one matrix (stays symmetric)
    A = wl.A.astype(np.float64).copy()
    lam, Q = np.linalg.eigh(A[7]); lam[0] = -lam[0]
    A[7] = (Q * lam) @ Q.T
    A[7] = 0.5 * (A[7] + A[7].T)
    assert np.linalg.eigvalsh(A[7]).min() < 0
    assert _run(apd, wl, A=A) == apd.BAD_A_NOT_POSITIVE_DEFINITE
    # singular (rank deficient) counts as not positive definite
    A = wl.A.copy(); A[0] = 0.0; A[0, 0, 0] = 1.0
    assert _run(apd, wl, A=A) == apd.BAD_A_NOT_POSITIVE_DEFINITE
    w = wl.w0.copy(); w[1] = -np.inf
    assert _run(apd, wl, w=w) == apd.BAD_W_NONFINITE
    v = wl.v.copy(); v[2] = 0.0
    f = _run(apd, wl, v=v)
    assert f & apd.BAD_TARGET_VOL_NOT_POSITIVE and f & apd.BAD_TARGET_VOL_SUM
    v = (wl.v * 1.001).astype(np.float32)
    assert _run(apd, wl, v=v) == apd.BAD_TARGET_VOL_SUM
    # several at once
    X = wl.X.copy(); X[0, 0] = np.inf
    w = wl.w0.copy(); w[M - 1] = np.nan
    assert _run(apd, wl, X=X, w=w) == (apd.BAD_X_NONFINITE | apd.BAD_W_NONFINITE)


def test_target_volumes_need_the_grid(apd):
    wl = workloads.make_random(2, (32, 32), 9, 77)
    with pytest.raises(Exception):
        _run(apd, wl, with_grid=False)


def test_agrees_with_what_solve_rejects(apd):
    """BAD_TARGET_VOL_SUM is the condition under which apd_solve returns APD_E_ARG (include/apd.h)."""
    wl = workloads.make_config(1)
    v = (wl.v * 1.01).astype(np.float32)
    assert _run(apd, wl, v=v) & apd.BAD_TARGET_VOL_SUM
    dev = torch.device("cuda:0")
    ctx = apd.ApdContext(wl.dim, wl.M)
    grid = apd.make_grid(wl.dim, wl.n, wl.lo, wl.hi)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
    w = torch.zeros(wl.M, dtype=torch.float32, device=dev)
    with pytest.raises(Exception):
        ctx.apd_solve(grid, t(wl.X), t(wl.A), t(v), 0.01, w=w)
    ctx.close()
