"""Multi-GPU host logic on CPU (gloo, world_size 2): slab arithmetic and the one all-reduce of the map.

The shooter is the CPU oracle through the `shoot_fn` hook of multi.shoot_distributed -- the code path that on
GPUs calls Field.shoot per slab and all-reduces over NCCL is the same, only the backend and shooter differ."""
import math
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2506_02114_b200 import multi  # noqa: E402


def test_slab_bounds_cover_every_row_once():
    for n in (0, 1, 7, 100, 84556):
        for world in (1, 2, 3, 8):
            seen = np.zeros(n, dtype=int)
            prev = 0
            for r in range(world):
                j0, j1 = multi.slab_bounds(n, world, r)
                assert j0 == prev and j1 >= j0
                seen[j0:j1] += 1
                prev = j1
            assert prev == n and np.all(seen == 1)
    # equal split up to one row
    sizes = [b - a for a, b in (multi.slab_bounds(1000, 8, r) for r in range(8))]
    assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        multi.slab_bounds(10, 2, 2)


def test_slab_bounds_weighted_and_aligned():
    n = 1000
    w = np.ones(n)
    w[100:110] = 500.0                                  # a star-heavy band of rows
    cost = []
    for r in range(4):
        j0, j1 = multi.slab_bounds(n, 4, r, weights=w)
        cost.append(w[j0:j1].sum())
    assert max(cost) <= 1.0 / 4 * w.sum() + 500.0       # balanced to within one heavy row
    assert max(cost) < 0.5 * w.sum()                    # an equal-rows split would put 84 % in slab 0
    cuts = [multi.slab_bounds(n, 4, r, align=31) for r in range(4)]
    assert all(a % 31 == 0 for a, _ in cuts) and cuts[-1][1] == n
    assert all(cuts[r][1] == cuts[r + 1][0] for r in range(3))
    ys = np.array([0.05, 0.051, 3.2])
    rw = multi.star_row_weights(ys, 0.0, 0.1, 40, per_star=10.0)
    assert rw[0] == 21.0 and rw[32] == 11.0 and rw.sum() == 40 + 30.0


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    n, ks, kt, gam = 40, 0.2, 0.4, 0.2
    R = math.sqrt(n / ks)
    xs, ys, ms = oracle.starfield(77, n, shape=0, a1=R)
    of = oracle.Field.make(kt, ks, gam, xs, ys, ms, R=R)
    g = oracle.geometry(kt, ks, gam, 3.0, 24, 2.0, 0)

    class _Field:                                        # what shoot_distributed needs of a Field: the grid
        def grid(self, *a, **k):
            return g

    def shoot_fn(sub):
        if sub[3] <= sub[2]:
            return np.zeros((24, 24)), None
        return oracle.shoot(of, g, 0, sub=sub), None

    w = multi.star_row_weights(ys, g.x0_2, g.h2, g.n2, per_star=50.0)
    m, (j0, j1), _ = multi.shoot_distributed(_Field(), 3.0, 24, 2.0, weights=w, shoot_fn=shoot_fn)
    np.save(os.path.join(out_dir, f"map{rank}.npy"), m.numpy())
    np.save(os.path.join(out_dir, f"slab{rank}.npy"), np.array([j0, j1, g.n2]))
    if rank == 0:
        np.save(os.path.join(out_dir, "whole.npy"), oracle.shoot(of, g, 0))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_slabs_and_allreduce(tmp_path):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    whole = np.load(tmp_path / "whole.npy")
    m0, m1 = np.load(tmp_path / "map0.npy"), np.load(tmp_path / "map1.npy")
    s0, s1 = np.load(tmp_path / "slab0.npy"), np.load(tmp_path / "slab1.npy")
    assert s0[0] == 0 and s0[1] == s1[0] and s1[1] == s1[2]             # the slabs tile the grid
    assert 0 < s0[1] < s0[2]
    assert np.array_equal(m0, m1)                                          # every rank holds the reduced map
    assert np.max(np.abs(m0 - whole)) <= 1e-12 * whole.max()              # slabs add up to the whole map
