"""Host-side logic of the voxel-slab sharding (row f4) on CPU, world_size 2 over gloo: the slab
partition, and the counter-block exchange protocol -- a word-wise int64 SUM allreduce in which every fp64 layer sum has
exactly one non-zero contributor, so the integer sum reproduces its bits and the total (layers added in ascending
order) is the same on every rank and the same as without sharding.  No GPU needed."""
import json
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2403_03571_b200 import binding  # noqa: E402


@pytest.mark.parametrize("n_last,world,align", [(256, 8, 8), (256, 3, 8), (100, 2, 8), (44, 2, 8), (1024, 4, 64),
                                                (200, 3, 64), (9, 2, 8), (512, 7, 8)])
def test_slab_partition_covers_the_axis_on_aligned_boundaries(n_last, world, align):
    parts = binding.slab_partition(n_last, world, align)
    assert len(parts) == world and parts[0][0] == 0
    for (lo, n), (lo2, _) in zip(parts[:-1], parts[1:]):
        assert lo + n == lo2 and n > 0
    lo, n = parts[-1]
    assert lo + n == n_last and n > 0
    for lo, n in parts:
        assert lo % align == 0 and (n % align == 0 or lo + n == n_last)
    sizes = [n for _, n in parts]
    assert max(sizes) - min(sizes) < 2 * align         # as even as whole layers allow (the last layer may be partial)


def test_slab_partition_needs_a_layer_per_rank():
    with pytest.raises(ValueError):
        binding.slab_partition(16, 3, 8)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    M, n_last, align = 37, 44, 8
    n_layers = (n_last + align - 1) // align
    rng = np.random.default_rng(7)                                   # the same "whole grid" data on both ranks
    counts_by_layer = rng.integers(0, 1000, size=(n_layers, M))
    layer_sums = rng.standard_normal(n_layers) * 10.0 ** rng.integers(-8, 3, n_layers)
    layer_sums[2] = -0.0 * 1.0 + layer_sums[2]
    lo, n = binding.slab_partition(n_last, world, align)[rank]
    own = range(lo // align, (lo + n + align - 1) // align)
    block = np.zeros(M + n_layers, dtype=np.int64)                   # [count u64 x M | layer sums as fp64 bits]
    for L in own:
        block[:M] += counts_by_layer[L]
        block[M + L] = np.float64(layer_sums[L]).view(np.int64)
    t = torch.from_numpy(block)
    dist.all_reduce(t)                                               # word-wise integer SUM
    got_counts = t[:M].numpy()
    got_layers = t[M:].numpy().view(np.float64)
    total = 0.0
    for L in range(n_layers):
        total += got_layers[L]
    ref_total = 0.0
    for L in range(n_layers):
        ref_total += layer_sums[L]
    ok = bool(np.array_equal(got_counts, counts_by_layer.sum(axis=0)) and
              np.array_equal(got_layers.view(np.int64), layer_sums.view(np.int64)) and total == ref_total)
    flags = [None] * world
    dist.all_gather_object(flags, (ok, float(total)))
    if rank == 0:
        json.dump({"ok": [f[0] for f in flags], "totals": [f[1] for f in flags], "ref": ref_total}, open(out, "w"))
    dist.destroy_process_group()


def test_counter_block_exchange_is_exact_gloo_world2(tmp_path):
    out = str(tmp_path / "r.json")
    port = 29500 + (os.getpid() * 7) % 2000
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["ok"] == [True, True]
    assert r["totals"][0] == r["totals"][1] == r["ref"]              # bit-identical on both ranks, and to no sharding
