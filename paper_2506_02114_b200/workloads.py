"""Named GPU workloads of the hot path, for profilers and sanitizers: `python -m paper_2506_02114_b200.workloads CASE`.

Every case runs the library's own kernels through the binding on seeded synthetic inputs (synth/, BASELINE.json's
configs) and prints one line of checksums; nothing here is timed and nothing is compared (tests/ does that).  The
captures under profiles/ name the case they ran, e.g.
    ncu --set full -k regex:deflect_direct -c 1 python -m paper_2506_02114_b200.workloads direct
    compute-sanitizer --tool racecheck python -m paper_2506_02114_b200.workloads tiny

  tiny            a 300-star disc field, a rectangular field and a clustered field; IPM, IRS and F32 maps of 64^2 pixels
                  (the sanitizer target: every kernel of the path in a fraction of a second)
  direct [IDX]    mlens_deflect in DIRECT mode (the paper's "no FMM" P2P sum, eq 13) at 2^18 points, config IDX (default 1)
  create [IDX]    seeded field of config IDX (default 4): star field, Morton sort, tree, lists, P2M/M2M/M2L/L2L
  irs [IDX] [F]   IRS map of config IDX (default 4) over the central fraction F (default 0.25) of the cell rows
  ipm [IDX] [F]   IPM map, likewise
"""
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _seeded(ml, c):
    return ml.Field.seeded(c.kappa_tot, c.gamma, c.n_stars, c.seed, kappa_star=c.kappa_star,
                           mass_law=c.mass_law, mass_a=c.mass_a, mass_lo=c.mass_lo, mass_hi=c.mass_hi)


def _rows(g, frac):
    n2 = int(g.n2)
    nj = max(32, int(n2 * frac)) // 32 * 32
    j0 = max(0, (n2 - nj) // 2 // 32 * 32)
    return (0, int(g.n1), j0, min(n2, j0 + nj))


def main(argv):
    import torch
    import synth
    import paper_2506_02114_b200 as ml
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device: libmlens has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    case = argv[0] if argv else "tiny"
    idx = int(argv[1]) if len(argv) > 1 else (1 if case == "direct" else 4)
    frac = float(argv[2]) if len(argv) > 2 else 0.25
    if case == "tiny":
        sums = []
        n, ks, kt, gam = 300, 0.25, 0.45, 0.15
        f = ml.Field.seeded(kt, gam, n, 12345, kappa_star=ks)
        for kw in (dict(), dict(map_mode=ml.MAP_IRS), dict(eval_mode=ml.EVAL_FMM_F32),
                   dict(map_mode=ml.MAP_IRS, eval_mode=ml.EVAL_FMM_F32), dict(small_px=1), dict(queue_mb=1, band_fixed=True, band_cells=4096)):
            sums.append(float(f.shoot(4.0, 64, 2.0, border_mode=ml.BORDER_EQ16, device=dev, **kw).map.sum()))
        z = np.random.default_rng(0).uniform(-8, 8, (2, 4096))
        sums.append(float(np.sum(f.deflect(z[0], z[1])[0])) + float(np.sum(f.deflect(z[0], z[1], ml.EVAL_DIRECT)[0])))
        f.close()
        c1, c2 = 30.0, 12.0
        xs, ys, ms = synth.rect_stars(n, c1, c2, 11)
        f = ml.Field.from_stars(0.5, 0.1, xs, ys, ms, kappa_star=math.pi * n / (4 * c1 * c2), shape=ml.SHAPE_RECT, c1=c1, c2=c2)
        for kw in (dict(), dict(map_mode=ml.MAP_IRS)):
            sums.append(float(f.shoot(2.0, 48, 2.0, border_mode=ml.BORDER_MARGIN, border_param=0.2, device=dev, **kw).map.sum()))
        f.close()
        R = math.sqrt(2000 / 0.3)
        xs, ys, ms = synth.clustered_stars(2000, R, 5)
        f = ml.Field.from_stars(0.5, 0.2, xs, ys, ms, kappa_star=0.3, R=R)
        sums.append(float(f.shoot(3.0, 64, 2.0, border_mode=ml.BORDER_EQ16, device=dev).map.sum()))
        m = f.shoot(3.0, 64, 2.0, border_mode=ml.BORDER_EQ16, device=dev).map
        sums.append(float(ml.histogram(m, 2.0, -1.0, 1.0, 32).sum()))
        out = torch.zeros(34, dtype=torch.int64, device=dev)
        sums.append(float(ml.histogram_static(m, 2.0, -1.0, 1.0, 32, out).sum()))
        f.close()
        print("tiny ok:", " ".join(f"{v:.6g}" for v in sums))
        return
    c = synth.get_config(idx)
    f = _seeded(ml, c)
    info = f.info()
    if case == "create":
        print(f"create ok: cfg{idx} order={info['order']} nodes={info['n_nodes']} levels={info['n_levels']} spot={info['spot_check_err']:.3g}")
    elif case == "direct":
        g = f.grid(c.half_y, c.npix, c.rays_per_pixel_length, border_mode=c.border_mode, border_param=c.border_param)
        zx, zy = synth.sample_points_window(1 << 18, g.X1, g.X2, g.H1, g.H2, 1)
        zx, zy = torch.from_numpy(zx).to(dev), torch.from_numpy(zy).to(dev)
        ax, ay = f.deflect(zx, zy, ml.EVAL_DIRECT)
        torch.cuda.synchronize()
        print(f"direct ok: cfg{idx} {zx.numel()} points x {c.n_stars} stars, sum = {float(ax.sum()):.6g}")
    elif case in ("irs", "ipm"):
        kw = dict(border_mode=c.border_mode, border_param=c.border_param)
        g = f.grid(c.half_y, c.npix, c.rays_per_pixel_length, **kw)
        sub = _rows(g, frac)
        r = f.shoot(c.half_y, c.npix, c.rays_per_pixel_length, sub=sub, device=dev,
                    map_mode=ml.MAP_IRS if case == "irs" else ml.MAP_IPM, **kw)
        print(f"{case} ok: cfg{idx} rows {sub[2]}..{sub[3]} of {int(g.n2)}, rays {r.stats['n_rays']}, "
              f"shoot {r.stats['ms_shoot']:.1f} ms in {r.stats['n_shoot_launches']} launches, sum = {float(r.map.sum()):.6g}")
    else:
        raise SystemExit(__doc__)
    f.close()


if __name__ == "__main__":
    main(sys.argv[1:])
