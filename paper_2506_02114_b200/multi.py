"""One map on several GPUs (the paper names multi-GPU as its one remaining speed-up).

Rays are independent and deposition is a sum, so the global cell grid is cut into contiguous
row slabs (the `sub` range of mlens_shoot), one per rank.  Stars and tree are replicated (their set-up is
milliseconds); every rank accumulates a private full-size map and ONE exchange step follows: an
all-reduce (sum, float64) of npix1 x npix2 values over NCCL (NVLink 5 / NVSwitch) -- 8 MB for the bench
workload, 0.8 GB for the 10^4 x 10^4 production map.  There is no other communication on the path.

Host logic only: the slab arithmetic and the reduction call.  Every ray and every deposit still runs in
libmlens' kernels through Field.shoot.  The `shoot_fn` hook lets the CPU tests (gloo, world_size 2)
drive the same code with another shooter.
"""
import numpy as np


def slab_bounds(n_rows, world, rank, weights=None, align=1):
    """Rows [j0, j1) of rank `rank` out of `n_rows` cell rows split into `world` contiguous slabs.

    weights: optional per-row cost (e.g. 1 + c * stars in the row: cells next to a star map to
    triangles that cover the whole map); slabs then hold equal cost, not equal row counts.
    align: slab borders are rounded to multiples of `align` rows (the kernels' tile height).
    Every row belongs to exactly one slab; slabs may be empty when world > n_rows."""
    if world < 1 or not (0 <= rank < world) or n_rows < 0:
        raise ValueError("bad slab request")
    if weights is None:
        cuts = [(n_rows * r) // world for r in range(world + 1)]
    else:
        w = np.asarray(weights, dtype=np.float64)
        if w.shape != (n_rows,) or np.any(w < 0):
            raise ValueError("weights must be n_rows non-negative numbers")
        c = np.concatenate([[0.0], np.cumsum(w)])
        tot = c[-1]
        cuts = [0] + [int(np.searchsorted(c, tot * r / world, side="left")) for r in range(1, world)] + [n_rows]
    if align > 1:
        cuts = [0] + [min(n_rows, (c + align // 2) // align * align) for c in cuts[1:-1]] + [n_rows]
    for r in range(1, world + 1):                       # monotone whatever the rounding did
        cuts[r] = max(cuts[r], cuts[r - 1])
    return cuts[rank], cuts[rank + 1]


def star_row_weights(ys, x0_2, h2, n_rows, per_star=10.0):
    """Per-row cost model for slab_bounds: one unit per cell row plus `per_star` for every star whose
    x2 lies in the row (the cells around a star map to triangles covering thousands of pixels).  per_star = 10 rows is
    the least-squares fit of t = a rows + b stars to the times of eight equal-row slabs of BASELINE config 1 on one
    B200 (bench.py `slab_balance`: a = 0.19 us per row, b = 1.9 us per star; equal rows are off by 17 %, weighted
    rows by 11 % -- the window's edge rows hold no stars and fewer in-map triangles)."""
    w = np.ones(n_rows)
    j = np.floor((np.asarray(ys) - x0_2) / h2).astype(np.int64)
    j = j[(j >= 0) & (j < n_rows)]
    np.add.at(w, j, per_star)
    return w


def shoot_distributed(field, half_y, npix, k, *, group=None, weights=None, shoot_fn=None, device=None, **kw):
    """The whole map on every rank of `group` (default: the world group).

    Rank r shoots rows slab_bounds(n2, world, r) of the cell grid into its own map, then the maps are
    summed with one all-reduce.  Returns (map, (j0, j1), stats_of_this_rank).  With torch.distributed
    uninitialised it is a plain single-GPU shoot."""
    import torch
    import torch.distributed as dist
    world, rank = 1, 0
    if dist.is_available() and dist.is_initialized():
        world, rank = dist.get_world_size(group), dist.get_rank(group)
    g = field.grid(half_y, npix, k, **{a: b for a, b in kw.items() if a in ("map_mode", "eval_mode", "border_mode", "border_param", "center", "He")})
    n1, n2 = int(g.n1), int(g.n2)
    j0, j1 = slab_bounds(n2, world, rank, weights=weights)
    if shoot_fn is None:
        def shoot_fn(sub):
            if sub[3] <= sub[2]:
                npx = npix if isinstance(npix, (tuple, list)) else (npix, npix)
                return torch.zeros((npx[1], npx[0]), dtype=torch.float64, device=device), None
            r = field.shoot(half_y, npix, k, sub=sub, device=device, **kw)
            return r.map, r.stats
    part, stats = shoot_fn((0, n1, j0, j1))
    if not torch.is_tensor(part):
        part = torch.from_numpy(np.ascontiguousarray(part))
    if world > 1:
        if dist.get_backend(group) == "nccl" and not part.is_cuda:
            raise ValueError("shoot_distributed over NCCL needs the partial map on the GPU: pass device=torch.device('cuda', local_rank) "
                             "or a CUDA tensor as out= (a host map can only be reduced over gloo)")
        dist.all_reduce(part, op=dist.ReduceOp.SUM, group=group)      # the one exchange step of the path
    return part, (j0, j1), stats
