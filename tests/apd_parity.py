"""GPU <-> oracle parity rule (from BASELINE.json north_star):

1. labels: a voxel mismatches if labels_gpu[j] != oracle label.  Every mismatch must be a near-tie:
   c_{labels_gpu[j]}(y_j) - c_1 < 1e-5 * scale_j with scale_j = max(|q_1|,|w_1|,|q_2|,|w_2|) over the
   oracle's best and runner-up (q = c + w);  #mismatches < 1e-5 * N.
2. volumes: sum_i |count_gpu - count_or| <= 2 #mismatches, sum count_gpu = N exactly.
3. dual: |dual_gpu - dual_or| <= 1e-6 * max(|dual_or|, |P| sum_j q_1(y_j)).
4. centroids: equal to 1e-6 (hi-lo) on cells no mismatching voxel touches.
"""
from __future__ import annotations

import numpy as np

from oracle.apd_oracle import Grid, oracle_assign, oracle_cost_of

NEAR_TIE = 1e-5


def grid_of(wl) -> Grid:
    return Grid(wl.dim, wl.n, wl.lo, wl.hi)


def check_labels(grid: Grid, X, A, w, labels_gpu: np.ndarray, orc, sel=None) -> dict:
    """Rule 1 on all voxels (sel None) or on the sampled voxels `sel` (orc computed on the same sel)."""
    w64 = np.asarray(w, dtype=np.float64)
    lab_or = orc.labels
    mism = np.nonzero(labels_gpu != lab_or)[0]
    n = labels_gpu.size
    scale = None
    if orc.second is not None:
        q1 = orc.best + w64[lab_or]
        run = np.where(orc.runner >= 0, orc.runner, lab_or)
        q2 = np.where(orc.runner >= 0, orc.second + w64[run], q1)
        scale = np.maximum.reduce([np.abs(q1), np.abs(w64[lab_or]), np.abs(q2), np.abs(w64[run])])
        near_pop = int(np.sum((orc.second - orc.best) < NEAR_TIE * scale))
    else:
        near_pop = -1
    out = dict(n=n, mismatches=int(mism.size), near_tie_population=near_pop)
    assert labels_gpu.min() >= 0 and labels_gpu.max() < len(w64), "label out of range"
    if mism.size:
        vox = mism if sel is None else np.asarray(sel)[mism]
        c_gpu = oracle_cost_of(grid, X, A, w, vox, labels_gpu[mism].astype(np.int32))
        excess = c_gpu - orc.best[mism]
        assert scale is not None
        bad = excess >= NEAR_TIE * scale[mism]
        assert not bad.any(), (f"{int(bad.sum())} mismatching voxels are NOT near-ties; worst excess/scale = "
                               f"{float(np.max(excess / scale[mism])):.3e}")
        out["worst_excess_over_scale"] = float(np.max(excess / scale[mism]))
    assert mism.size < max(NEAR_TIE * n, 1e-300) or mism.size == 0, \
        f"{mism.size} mismatches >= 1e-5 * {n}"
    return out


def check_assign(wl, w, labels_gpu, vol_gpu, dual_gpu, v=None, centroids_gpu=None, err_gpu=None, orc=None) -> dict:
    """Full-grid parity (rules 1-4) of one evaluation against oracle_assign on the same inputs (`orc`: that oracle
    result when the caller already has it -- one oracle pass can serve several kernels)."""
    grid = grid_of(wl)
    if orc is None:
        orc = oracle_assign(grid, wl.X, wl.A, w, v=v)
    out = check_labels(grid, wl.X, wl.A, w, labels_gpu, orc)
    nm = out["mismatches"]
    P = grid.voxel_volume
    count_gpu = np.rint(vol_gpu / P).astype(np.int64)
    np.testing.assert_allclose(count_gpu * P, vol_gpu, rtol=1e-13, atol=0)          # vol = integer count * |P|
    assert int(count_gpu.sum()) == grid.N, "sum of counts != N"
    assert np.array_equal(count_gpu, np.bincount(labels_gpu, minlength=wl.M)), "vol disagrees with the GPU's own labels"
    assert int(np.abs(count_gpu - orc.count).sum()) <= 2 * nm
    ref = orc.dual if v is not None else orc.dual_min_part
    tol = 1e-6 * max(abs(ref), abs(orc.quad_part))
    assert abs(dual_gpu - ref) <= tol, f"dual {dual_gpu!r} vs oracle {ref!r} (tol {tol:.3e})"
    out["dual_rel_diff"] = abs(dual_gpu - ref) / max(abs(ref), abs(orc.quad_part))
    if err_gpu is not None and v is not None:
        v64 = np.asarray(v, dtype=np.float64)
        assert abs(err_gpu - orc.err) <= 2.0 * nm * P / v64.min() + 1e-12
    if centroids_gpu is not None:
        touched = np.zeros(wl.M, dtype=bool)
        mism = np.nonzero(labels_gpu != orc.labels)[0]
        touched[labels_gpu[mism]] = True
        touched[orc.labels[mism]] = True
        ext = np.asarray(wl.hi, dtype=np.float64) - np.asarray(wl.lo, dtype=np.float64)
        diff = np.abs(centroids_gpu - orc.centroids) / ext
        assert float(diff[~touched].max(initial=0.0)) <= 1e-6
    return out
