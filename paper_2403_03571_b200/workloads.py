"""Seeded synthetic inputs for the APD hot path (shared by the oracle tests and the GPU harness).

This module holds NONE of the method's arithmetic (no cost, no argmin, no
volumes): it only draws seeds X, anisotropy matrices A and target volumes v with
the shapes and distributions of BASELINE.json's five configs, which stand in for
the paper's workloads (runtime tests (a)/(b); rolled-steel
EBSD statistics, PAPER.md:284-294 -- whose data are not available).  It imports
neither ``oracle/`` nor the CUDA binding.

Recipe (stated in DESIGN.md, section "Input recipe"):
  rng = numpy Generator(PCG64(240303571*10 + cfg)); draw order seeds -> shapes ->
  orientations -> volumes; everything fp64, then X, A, v cast to fp32 (A
  symmetrised before the cast, v renormalised in fp64 before the cast).
  Omega = [0,1]^d, w0 = 0, eps = 0.01.

Notation (SURVEY.md notation table): M = number of grains/seeds, N = number of
voxels, n = voxels per axis, d = dimension.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Tuple

import numpy as np

BASE_SEED = 240303571 * 10


@dataclasses.dataclass
class Workload:
    """One problem instance. Arrays are host numpy, fp32 (what both sides are fed)."""

    name: str
    dim: int
    n: Tuple[int, ...]          # voxels per axis, (nx, ny[, nz]); x fastest in the label array
    lo: Tuple[float, ...]
    hi: Tuple[float, ...]
    X: np.ndarray               # [M, d]   float32 seeds
    A: np.ndarray               # [M, d, d] float32 anisotropy matrices
    v: np.ndarray               # [M]      float32 target volumes, sum = |Omega|
    w0: np.ndarray              # [M]      float32 initial weights (zeros)
    eps: float = 0.01
    rejection_rate: float = 0.0  # of the seed exclusion rule

    @property
    def M(self) -> int:
        return int(self.X.shape[0])

    @property
    def N(self) -> int:
        return int(np.prod(self.n))

    @property
    def pairs(self) -> int:
        return self.N * self.M


# ----------------------------------------------------------------------------------------
# building blocks
# ----------------------------------------------------------------------------------------
def sample_seeds_with_exclusion(rng: np.random.Generator, M: int, d: int, C: float = 0.2):
    """Sequential uniform sampling on [0,1]^d; a draw is rejected if it is closer than
    C * M^(-1/d) to an already accepted seed (C = 2/10)."""
    r2 = (C * M ** (-1.0 / d)) ** 2
    X = np.empty((M, d), dtype=np.float64)
    k = 0
    draws = 0
    while k < M:
        # draw in small batches; order of acceptance is still sequential
        batch = rng.random((64, d))
        for p in batch:
            draws += 1
            if k == 0 or np.min(np.sum((X[:k] - p) ** 2, axis=1)) > r2:
                X[k] = p
                k += 1
                if k == M:
                    break
    return X, 1.0 - M / draws


def rot2(theta: np.ndarray) -> np.ndarray:
    c, s = np.cos(theta), np.sin(theta)
    R = np.empty(theta.shape + (2, 2))
    R[..., 0, 0] = c
    R[..., 0, 1] = -s
    R[..., 1, 0] = s
    R[..., 1, 1] = c
    return R


def aniso2(a: np.ndarray, b: np.ndarray, theta: np.ndarray) -> np.ndarray:
    """A(a,b,theta) = V diag(a^-2, b^-2) V^-1, V = rotation by theta (eq. 2.2)."""
    V = rot2(theta)
    D = np.zeros(theta.shape + (2, 2))
    D[..., 0, 0] = a ** -2.0
    D[..., 1, 1] = b ** -2.0
    return V @ D @ np.swapaxes(V, -1, -2)


def quat_to_rot(q: np.ndarray) -> np.ndarray:
    q = q / np.linalg.norm(q, axis=-1, keepdims=True)
    w, x, y, z = q[..., 0], q[..., 1], q[..., 2], q[..., 3]
    R = np.empty(q.shape[:-1] + (3, 3))
    R[..., 0, 0] = 1 - 2 * (y * y + z * z)
    R[..., 0, 1] = 2 * (x * y - z * w)
    R[..., 0, 2] = 2 * (x * z + y * w)
    R[..., 1, 0] = 2 * (x * y + z * w)
    R[..., 1, 1] = 1 - 2 * (x * x + z * z)
    R[..., 1, 2] = 2 * (y * z - x * w)
    R[..., 2, 0] = 2 * (x * z - y * w)
    R[..., 2, 1] = 2 * (y * z + x * w)
    R[..., 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def haar_rotations(rng: np.random.Generator, M: int) -> np.ndarray:
    """Uniform on SO(3): normalised 4-Gaussian quaternion."""
    return quat_to_rot(rng.standard_normal((M, 4)))


def axis_angle_rot(axis: np.ndarray, ang: np.ndarray) -> np.ndarray:
    axis = axis / np.linalg.norm(axis, axis=-1, keepdims=True)
    half = 0.5 * ang
    q = np.concatenate([np.cos(half)[..., None], np.sin(half)[..., None] * axis], axis=-1)
    return quat_to_rot(q)


def aniso3(axes: np.ndarray, R: np.ndarray) -> np.ndarray:
    """Ellipsoid with semi-axes `axes[:,k]` along the COLUMNS of R:  A = R diag(axes^-2) R^T.
    (SURVEY.md writes R^T diag R with the axes along the rows of R; for Haar-uniform R the
    two are the same distribution.)"""
    D = np.zeros(R.shape)
    for k in range(3):
        D[..., k, k] = axes[..., k] ** -2.0
    return R @ D @ np.swapaxes(R, -1, -2)


def _finish(name, dim, n, X, A, v, rej) -> Workload:
    A = 0.5 * (A + np.swapaxes(A, -1, -2))
    v = v / np.sum(v)  # |Omega| = 1
    return Workload(
        name=name, dim=dim, n=tuple(n), lo=(0.0,) * dim, hi=(1.0,) * dim,
        X=np.ascontiguousarray(X, dtype=np.float32),
        A=np.ascontiguousarray(A, dtype=np.float32),
        v=np.ascontiguousarray(v, dtype=np.float32),
        w0=np.zeros(X.shape[0], dtype=np.float32), eps=0.01, rejection_rate=rej)


# ----------------------------------------------------------------------------------------
# BASELINE.json configs 1..5
# ----------------------------------------------------------------------------------------
CONFIG_SHAPES = {
    1: dict(dim=2, n=(64, 64), M=10),
    2: dict(dim=2, n=(1024, 1024), M=1000),
    3: dict(dim=3, n=(128, 128, 128), M=1000),
    4: dict(dim=3, n=(256, 256, 256), M=10000),
    5: dict(dim=3, n=(512, 512, 512), M=20000),
}


def make_config(cfg: int, n: Optional[Tuple[int, ...]] = None, M: Optional[int] = None) -> Workload:
    """BASELINE.json `configs[cfg-1]`.  `n` / `M` override the grid / grain count (used by the
    tests to get a same-distribution problem the oracle finishes in seconds)."""
    shp = CONFIG_SHAPES[cfg]
    dim = shp["dim"]
    n = tuple(n) if n is not None else shp["n"]
    M = int(M) if M is not None else shp["M"]
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + cfg))
    X, rej = sample_seeds_with_exclusion(rng, M, dim)
    if cfg == 1:
        a = rng.uniform(1.0, 3.0, M)
        b = np.ones(M)
        theta = rng.uniform(0.0, math.pi, M)
        A = aniso2(a, b, theta)                      # NOT det-normalised (config text, literally)
        v = np.full(M, 1.0 / M)
    elif cfg == 2:
        r = np.clip(np.exp(rng.normal(0.3, 0.3, M)), 1.0, 5.0)
        theta = rng.uniform(0.0, math.pi, M)
        A = aniso2(np.sqrt(r), 1.0 / np.sqrt(r), theta)   # det A = 1
        v = np.exp(rng.normal(0.0, 0.5, M))
    elif cfg == 3:
        ratios = np.sort(rng.uniform(0.3, 1.0, (M, 2)), axis=1)[:, ::-1]   # b/a >= c/a
        axes = np.concatenate([np.ones((M, 1)), ratios], axis=1)
        axes = axes / np.cbrt(np.prod(axes, axis=1, keepdims=True))         # abc = 1
        R = haar_rotations(rng, M)
        A = aniso3(axes, R)
        v = np.exp(rng.normal(0.0, 0.4, M))
    elif cfg == 4:
        axes = np.array([3.0, 1.5, 1.0]) * (1.0 + rng.uniform(-0.2, 0.2, (M, 3)))
        axes = axes / np.cbrt(np.prod(axes, axis=1, keepdims=True))
        polar = np.abs(rng.normal(0.0, math.radians(10.0), M))
        azim = rng.uniform(0.0, 2 * math.pi, M)
        spin = rng.uniform(0.0, 2 * math.pi, M)
        # tilt: rotate e_x towards (0, cos az, sin az) by `polar`, i.e. about axis e_x x that
        tilt_axis = np.stack([np.zeros(M), -np.sin(azim), np.cos(azim)], axis=1)
        Rt = axis_angle_rot(tilt_axis, polar)
        Rs = axis_angle_rot(np.tile(np.array([1.0, 0.0, 0.0]), (M, 1)), spin)
        R = Rt @ Rs                                   # columns: major axis (tilted e_x), then spun b, c
        A = aniso3(axes, R)
        v = np.exp(rng.normal(0.0, 0.5, M))
    elif cfg == 5:
        iso = rng.random(M) < 0.5
        bi, ci = rng.uniform(0.9, 1.0, M), rng.uniform(0.9, 1.0, M)
        ac = rng.uniform(1.0, 5.0, M)
        bc = 1.0 + rng.random(M) * (ac - 1.0)         # b/c ~ U[1, a/c]
        axes = np.where(iso[:, None], np.stack([np.ones(M), bi, ci], 1), np.stack([ac, bc, np.ones(M)], 1))
        axes = axes / np.cbrt(np.prod(axes, axis=1, keepdims=True))
        R = haar_rotations(rng, M)
        A = aniso3(axes, R)
        big = rng.random(M) < 0.5
        v = np.exp(rng.normal(0.0, 0.3, M)) * np.where(big, 4.0, 1.0)
    else:
        raise ValueError(f"unknown config {cfg}")
    return _finish(f"cfg{cfg}", dim, n, X, A, v, rej)


# ----------------------------------------------------------------------------------------
# correctness-only inputs (SURVEY.md 8(d) "additional non-config inputs")
# ----------------------------------------------------------------------------------------
def make_random(dim: int, n: Tuple[int, ...], M: int, seed: int, lo=None, hi=None,
                aspect: float = 3.0, vol_sigma: float = 0.4, w_scale: float = 0.0,
                nonsymmetric: bool = False) -> Workload:
    """Generic random problem on a (possibly non-unit, non-cubic) box with random SPD A.
    `w_scale` > 0 also draws non-zero initial weights of that size relative to (box/M^(1/d))^2."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 1000 + seed))
    lo = tuple(lo) if lo is not None else (0.0,) * dim
    hi = tuple(hi) if hi is not None else (1.0,) * dim
    ext = np.array(hi) - np.array(lo)
    X = np.array(lo) + rng.random((M, dim)) * ext
    if dim == 2:
        r = rng.uniform(1.0, aspect, M)
        A = aniso2(np.sqrt(r), 1 / np.sqrt(r), rng.uniform(0, math.pi, M))
    else:
        ax = np.sort(rng.uniform(1.0, aspect, (M, 3)), axis=1)[:, ::-1]
        ax = ax / np.cbrt(np.prod(ax, axis=1, keepdims=True))
        A = aniso3(ax, haar_rotations(rng, M))
    A = 0.5 * (A + np.swapaxes(A, -1, -2))
    if nonsymmetric:  # same quadratic form, skew part added
        K = rng.standard_normal(A.shape) * 0.3
        A = A + (K - np.swapaxes(K, -1, -2))
    v = np.exp(rng.normal(0.0, vol_sigma, M))
    v = v / np.sum(v) * float(np.prod(ext))
    ell2 = (float(np.prod(ext)) / M) ** (2.0 / dim)
    w0 = (rng.standard_normal(M) * w_scale * ell2).astype(np.float32)
    return Workload(name=f"rand{dim}d_s{seed}", dim=dim, n=tuple(n), lo=lo, hi=hi,
                    X=X.astype(np.float32), A=np.ascontiguousarray(A, dtype=np.float32),
                    v=v.astype(np.float32), w0=w0)


def voxel_sample(N: int, k: int, seed: int) -> np.ndarray:
    """k distinct voxel indices in [0,N), sorted (for sampled full-size parity)."""
    rng = np.random.Generator(np.random.PCG64(BASE_SEED + 5000 + seed))
    k = min(k, N)
    idx = rng.choice(N, size=k, replace=False) if N < (1 << 62) else None
    return np.sort(idx.astype(np.int64))
