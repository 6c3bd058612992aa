#!/usr/bin/env python
"""bench.py -- the headline measurement of the hot path (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

One STEP is one pass of the whole hot path over one synthetic workload (BASELINE.json configs[1] by
default, the configuration the metric is quoted on):

    seeded star field -> Morton sort -> quadtree + lists -> P2M/M2M -> M2L/P2L/L2L -> leaf series
    -> fused ray evaluation + IPM deposit (map 1)  -> fused ray evaluation + IRS count (map 2)

all of it in libmlens' CUDA kernels, called through the C ABI (include/mlens.h).  `value` is lens-equation
evaluations per second over the whole step (unique rays of both maps / step time), inputs resident in
HBM (the star field is generated on the device from the seed).  `e2e` repeats the step with HOST
buffers: stars handed over as pinned host arrays, maps returned into pinned host arrays, the library
doing the copies inside the timed region.

N > 1 (torchrun): the SAME map on N GPUs: stars and tree replicated, the cell grid cut
into star-weighted row slabs (paper_2506_02114_b200/multi.py), one all-reduce (sum, float64) of each
map over NCCL -- the path's only exchange step; total work is fixed, so scaling is "strong";
time = max over ranks.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload, on the host cores of this box.  It is a deliberately slow baseline, not the target.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import synth  # noqa: E402

METRIC = "lens_eq_evals_per_s"
UNIT = "evals/s"

# B200 FP64 vector peak used as the "alu" roofline denominator: 148 SMs x 64 DFMA
# lanes/SM/clk x 2 flop x 1.965 GHz (clocks.max.sm of MEASURED_PEAKS.json).  The DFMA rate measured
# by mlens_bench_dfma in the same run is reported beside it as `peak_measured_dfma`.
FP64_LANES_PER_SM = 64
# dram bytes per launch of the dominant kernel from the committed `ncu --set full` capture
# (profiles/r01e_launches.md: dram read + write of shoot_ipm_kernel, mean of the two launches of a map).
NCU_TRAFFIC_BYTES_PER_LAUNCH = 3.43e9


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (default 1)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--maps", default="", help="also time whole maps of these configs, e.g. 0,2,3,4 (create, IPM, IRS wall ms)")
    return ap.parse_args()


def workload_name(cfg):
    return (f"{cfg.name}: {cfg.n_stars} stars, kappa_tot={cfg.kappa_tot} kappa_star={cfg.kappa_star} "
            f"gamma={cfg.gamma}, {cfg.npix}x{cfg.npix} px, half={cfg.half_y}, k={cfg.rays_per_pixel_length:g}")


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                c = [v.strip() for v in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); mx.append(float(c[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, c[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


# ------------------------------------------------------------------------------------------------
def oracle_sample(cfg, patch, want_irs=True):
    """Times the CPU oracle on a patch of `patch` = (ni, nj) cells at the window centre: the whole path
    (direct sum over all stars + brute-force clipping; IRS binning).  Returns (evals, seconds, threads)."""
    import oracle
    oracle.build()
    R = cfg.R_star
    xs, ys, ms = oracle.starfield(cfg.seed, cfg.n_stars, shape=0, a1=R, mass_law=cfg.mass_law,
                                  a=cfg.mass_a, lo=cfg.mass_lo, hi=cfg.mass_hi)
    of = oracle.Field.make(cfg.kappa_tot, cfg.kappa_star, cfg.gamma, xs, ys, ms, R=R)
    g = oracle.geometry(cfg.kappa_tot, cfg.kappa_star, cfg.gamma, cfg.half_y, cfg.npix, cfg.rays_per_pixel_length,
                        cfg.border_mode, cfg.border_param, m2_over_m=cfg.m2_over_m)
    ni, nj = min(patch[0], g.n1), min(patch[1], g.n2)
    i0, j0 = (g.n1 - ni) // 2, (g.n2 - nj) // 2
    sub = (i0, i0 + ni, j0, j0 + nj)
    t0 = time.perf_counter()
    oracle.shoot(of, g, 0, sub=sub)
    evals = (ni + 1) * (nj + 1)
    if want_irs:
        oracle.shoot(of, g, 1, sub=sub)
        evals += ni * nj
    return evals, time.perf_counter() - t0, oracle.num_threads(), sub


def run_reference(args):
    """--impl reference: the oracle, as it stands, on this box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = synth.get_config(args.config)
    patch = (128, 128)
    for _ in range(args.warmup):
        oracle_sample(cfg, (32, 32))
    tot_e, tot_t, thr, sub = 0, 0.0, 1, None
    for _ in range(args.steps):
        e, t, thr, sub = oracle_sample(cfg, patch)
        tot_e += e; tot_t += t
    v = tot_e / tot_t
    sample = f"IPM + IRS on the {patch[0]}x{patch[1]}-cell patch {sub} at the window centre, all {cfg.n_stars} stars per ray"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2506_02114_b200 as ml
    from paper_2506_02114_b200 import multi

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libmlens has no CPU fallback")
    ml.lib()                                         # fail loudly if the extension is missing
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = synth.get_config(args.config)
    seed = cfg.seed                                  # N > 1: the same field on every rank, one slab of rays each
    kw = dict(border_mode=cfg.border_mode, border_param=cfg.border_param)
    half, npix, k = cfg.half_y, cfg.npix, cfg.rays_per_pixel_length
    stream = torch.cuda.current_stream()

    map_ipm = torch.zeros((npix, npix), dtype=torch.float64, device=dev)
    map_irs = torch.zeros((npix, npix), dtype=torch.float64, device=dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    state = {}

    def step_device():
        f = ml.Field.seeded(cfg.kappa_tot, cfg.gamma, cfg.n_stars, seed, kappa_star=cfg.kappa_star,
                            mass_law=cfg.mass_law, mass_a=cfg.mass_a, mass_lo=cfg.mass_lo, mass_hi=cfg.mass_hi)
        if world > 1 and "weights" not in state:     # slab cost model from the star rows (same on every rank; cached)
            g0 = f.grid(half, npix, k, **kw)
            state["weights"] = multi.star_row_weights(f.stars()[1], g0.x0_2, g0.h2, int(g0.n2))
        _, slab, s1 = multi.shoot_distributed(f, half, npix, k, weights=state.get("weights"), out=map_ipm,
                                              map_mode=ml.MAP_IPM, **kw)
        _, _, s2 = multi.shoot_distributed(f, half, npix, k, weights=state.get("weights"), out=map_irs,
                                           map_mode=ml.MAP_IRS, **kw)
        state.update(info=f.info(), ipm=s1, irs=s2, slab=slab, grid=f.grid(half, npix, k, **kw))
        if "near_mean" not in state:                 # mean near-field list of a ray's leaf (area-weighted over the window)
            t = f.tree()
            g_ = state["grid"]
            leaves = np.where(t["child0"] < 0)[0]
            half_l = t["root_half"] / 2.0 ** t["level"][leaves]
            cx = -t["root_half"] + (2 * t["ix"][leaves] + 1) * half_l
            cy = -t["root_half"] + (2 * t["iy"][leaves] + 1) * half_l
            inside = (np.abs(cx - g_.X1) < g_.H1) & (np.abs(cy - g_.X2) < g_.H2)
            wgt = (half_l ** 2) * inside
            state["near_mean"] = float(np.sum(wgt * t["near_cnt"][t["leaf_id"][leaves]]) / max(np.sum(wgt), 1e-300))
        f.close()

    # host-side buffers of the e2e leg: pinned, numpy views handed to the C ABI as HOST pointers
    R = cfg.R_star
    hx, hy, hm = (torch.empty(cfg.n_stars, dtype=torch.float64).pin_memory() for _ in range(3))
    h_ipm = torch.empty((npix, npix), dtype=torch.float64).pin_memory()
    h_irs = torch.empty((npix, npix), dtype=torch.float64).pin_memory()

    def step_host():
        f = ml.Field.from_stars(cfg.kappa_tot, cfg.gamma, hx.numpy(), hy.numpy(), hm.numpy(),
                                kappa_star=cfg.kappa_star, R=R)
        if world == 1:
            f.shoot(half, npix, k, out=h_ipm.numpy(), map_mode=ml.MAP_IPM, **kw)
            f.shoot(half, npix, k, out=h_irs.numpy(), map_mode=ml.MAP_IRS, **kw)
        else:                                        # slabs on the device, all-reduce, then the result back to the host
            multi.shoot_distributed(f, half, npix, k, weights=state.get("weights"), out=map_ipm, map_mode=ml.MAP_IPM, **kw)
            multi.shoot_distributed(f, half, npix, k, weights=state.get("weights"), out=map_irs, map_mode=ml.MAP_IRS, **kw)
            h_ipm.copy_(map_ipm, non_blocking=True); h_irs.copy_(map_irs, non_blocking=True)
            torch.cuda.current_stream().synchronize()
        f.close()
        return float(h_ipm[npix // 2, npix // 2])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        """K steps, each between its own CUDA events on the launching stream; L2 flushed between steps
        outside the event pairs.  Returns (seconds per step, max over ranks)."""
        total_ms = 0.0
        barrier()
        for _ in range(steps):
            flush.fill_(1)                           # 512 MiB > 126 MB L2
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            e1.synchronize()
            total_ms += e0.elapsed_time(e1)
            if os.environ.get("MLENS_BENCH_VERBOSE"):
                print(f"step {fn.__name__}: {e0.elapsed_time(e1):.2f} ms", file=sys.stderr)
        barrier()
        t = torch.tensor([total_ms / steps], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item()) * 1e-3

    # the sampler starts before the warm-up: nvidia-smi takes ~0.5 s to come up, and its start-up inside the timed
    # region (a few hundred ms in all) stalls the host round trips of create; it keeps sampling through the timed steps
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(max(args.warmup, 3)):
        step_device()
    l0 = ml.launch_count()
    sec = timed(step_device, args.steps)
    launches = (ml.launch_count() - l0) // args.steps
    clocks = sampler.stop() if rank == 0 else None

    g = state["grid"]
    evals_ipm = (g.n1 + 1) * (g.n2 + 1)              # unique rays of the whole map, whatever N
    evals_irs = g.n1 * g.n2
    evals = evals_ipm + evals_irs
    value = evals / sec

    e2e = None
    if not args.no_e2e:
        # the stars of the e2e leg come from the library's own generator (read back once, outside the timing)
        f0 = ml.Field.seeded(cfg.kappa_tot, cfg.gamma, cfg.n_stars, seed, kappa_star=cfg.kappa_star,
                             mass_law=cfg.mass_law, mass_a=cfg.mass_a, mass_lo=cfg.mass_lo, mass_hi=cfg.mass_hi)
        sx, sy, sm = f0.stars()
        f0.close()
        hx.numpy()[:], hy.numpy()[:], hm.numpy()[:] = sx, sy, sm
        step_host()
        sec_h = timed(step_host, args.steps)
        e2e = {"value": evals / sec_h, "unit": UNIT, "ms_per_step": sec_h * 1e3,
               "h2d_bytes_per_step": 3 * 8 * cfg.n_stars, "d2h_bytes_per_step": 2 * 8 * npix * npix}

    # ---- roofline of the dominant kernel (fused evaluate + IPM deposit), DESIGN.md s7
    # Algorithmic work per lens-equation evaluation: the leaf's near-field list summed directly
    # (10 flop per star) + the leaf's order-p Taylor series by Horner (8 flop per term) + 10 flop macro and sheet.
    # The kernel itself does less (it re-expands the series per 32x32-ray tile, order 6-15 by geometry, and folds the distant
    # near-field stars into it): `flop_executed` counts what it really issues for the evaluation.
    st = state["ipm"]
    p = state["info"]["order"]
    n_near_leaf = state["near_mean"]
    rays_k = st["n_rays"]                                        # evaluations the kernel performed
    flop_alg = rays_k * (10.0 * n_near_leaf + 8.0 * (p - 1) + 10.0)
    flop_exec = 10.0 * st["n_near_terms"] + (8.0 * st["tile_order"] + 10.0) * rays_k
    n_l = max(1, st["n_shoot_launches"])
    dur = st["ms_shoot"] * 1e-3 / n_l
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    sm_max = peaks.get("sm_max_mhz", 1965.0)
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_tf = nsm * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    achieved_tf = flop_alg / n_l / dur / 1e12 if dur > 0 else 0.0
    roofline = {"bound": "alu", "kernel": "shoot_ipm_kernel", "achieved": achieved_tf, "peak": peak_tf,
                "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
                "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH,
                "peak_source": f"{nsm} SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x {sm_max:.0f} MHz (derived, DESIGN.md s7)",
                "peak_measured_dfma": ml.bench_dfma() / 1e12,
                "flop_per_eval_algorithmic": flop_alg / rays_k, "near_stars_per_leaf_mean": n_near_leaf,
                "flop_per_launch": flop_alg / n_l, "flop_executed_per_launch": flop_exec / n_l,
                "achieved_executed": flop_exec / n_l / dur / 1e12 if dur > 0 else 0.0,
                "launch_ms": dur * 1e3, "launches_per_map": n_l,
                "share_of_step": st["ms_shoot"] * 1e-3 / sec}

    # BASELINE.json metric: fraction of the atomic roofline for deposition.  Random 64-bit atomic adds into a buffer
    # the size of config 1's accumulators (16 MB, L2-resident) and of config 4's (1.6 GB, HBM-resident), measured here,
    # against what the apportioning kernels issued per second of their own time (one add per clipped pixel, two per
    # edge step at least).
    atomics = None
    if world == 1:
        st_i = state["ipm"]
        a_l2 = ml.bench_atomics(2 * npix * npix, True)
        a_hbm = ml.bench_atomics(200_000_000, True)
        adds = st_i["n_px_clipped"] + 2 * st_i["n_edge_steps"]
        rate = adds / (st_i["ms_drain"] * 1e-3)
        atomics = {"l2_resident_adds_per_s": a_l2, "hbm_resident_adds_per_s": a_hbm, "apportioning_adds_per_s": rate,
                   "frac_of_l2_atomic_rate": rate / a_l2, "apportioning_adds_per_map": adds}

    # the single-precision evaluator on the same workload, beside the float64 numbers
    f32 = None
    if world == 1:
        ff = ml.Field.seeded(cfg.kappa_tot, cfg.gamma, cfg.n_stars, seed, kappa_star=cfg.kappa_star,
                             mass_law=cfg.mass_law, mass_a=cfg.mass_a, mass_lo=cfg.mass_lo, mass_hi=cfg.mass_hi)
        out32 = torch.zeros((npix, npix), dtype=torch.float64, device=dev)
        f32 = {}
        for name, mode in (("ipm", ml.MAP_IPM), ("irs", ml.MAP_IRS)):
            for _ in range(2):
                r32 = ff.shoot(half, npix, k, out=out32, map_mode=mode, eval_mode=ml.EVAL_FMM_F32, **kw)
            f32[name + "_map_ms"] = r32.stats["ms_total"]
            f32[name + "_shoot_ms"] = r32.stats["ms_shoot"]
            ref64 = map_ipm if mode == ml.MAP_IPM else map_irs
            sel = ref64 >= 0.1
            rel = ((out32 - ref64).abs()[sel] / ref64[sel])
            f32[name + "_pixels_beyond_1e-3_of_f64"] = float((rel > 1e-3).double().mean())
            f32[name + "_median_rel_dev_of_f64"] = float(rel.median())
        f32["f64_ipm_shoot_ms"] = state["ipm"]["ms_shoot"]; f32["f64_irs_shoot_ms"] = state["irs"]["ms_shoot"]
        ff.close()
        del out32

    # the map consumers (HBM-bound): histogram of a synthetic log-normal 8192^2 map (512 MiB > L2)
    consumers = None
    if world == 1:
        big = torch.empty((8192, 8192), dtype=torch.float64, device=dev).log_normal_(0.0, 1.0)
        ms = []
        for _ in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); hh = ml.histogram(big, 1.0, -2.0, 2.0, 64); e1.record(stream); e1.synchronize()
            ms.append(e0.elapsed_time(e1))
        gbs = big.numel() * 8 / (min(ms[1:]) * 1e-3) / 1e9
        peak_hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs") if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else None
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        lc = ml.light_curve(map_ipm, g.ylo1, g.ylo2, g.p1, g.p2, (-0.9 * half, -0.7 * half), (0.9 * half, 0.8 * half), 1 << 20,
                            interp=ml.INTERP_BILINEAR)
        e1.record(stream); e1.synchronize()
        consumers = {"histogram_ms": min(ms[1:]), "histogram_GBps": gbs, "hbm_peak_GBps": peak_hbm,
                     "histogram_frac_of_hbm": (gbs / peak_hbm) if peak_hbm else None, "histogram_total": int(hh.sum()),
                     "light_curve_1M_samples_ms": e0.elapsed_time(e1), "light_curve_mean_mu": float(lc.nanmean())}
        del big

    maps = None
    if args.maps and world == 1:
        # BASELINE.json's second metric, map wall-time, on the other configurations (one warm-up, one timed run each)
        maps = {}
        for ci in [int(c) for c in args.maps.split(",") if c != ""]:
            c2 = synth.get_config(ci)
            kw2 = dict(border_mode=c2.border_mode, border_param=c2.border_param)
            out2 = torch.zeros((c2.npix, c2.npix), dtype=torch.float64, device=dev)
            rec = {}
            for rep in range(2):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                f2 = ml.Field.seeded(c2.kappa_tot, c2.gamma, c2.n_stars, c2.seed, kappa_star=c2.kappa_star,
                                     mass_law=c2.mass_law, mass_a=c2.mass_a, mass_lo=c2.mass_lo, mass_hi=c2.mass_hi)
                e1.record(stream); e1.synchronize()
                rec["create_ms"] = e0.elapsed_time(e1)
                for name, mode in (("ipm", ml.MAP_IPM), ("irs", ml.MAP_IRS)):
                    r = f2.shoot(c2.half_y, c2.npix, c2.rays_per_pixel_length, out=out2, map_mode=mode, **kw2)
                    rec[name + "_map_ms"] = r.stats["ms_total"]
                    rec[name + "_rays"] = r.stats["n_rays"]
                    rec[name + "_evals_per_s"] = r.stats["n_rays"] / (r.stats["ms_total"] * 1e-3)
                    rec[name + "_shoot_ms"] = r.stats["ms_shoot"]
                    rec["tile_order"] = r.stats["tile_order"]
                    if mode == ml.MAP_IPM:
                        rec["ipm_drain_walk_ms"] = r.stats["ms_drain"]
                        rec["ipm_bands"] = r.stats["n_bands"]
                        rec["tri"] = {k: r.stats[k] for k in ("n_tri_single", "n_tri_strip", "n_tri_queued", "n_tri_walked",
                                                              "n_px_clipped", "n_edge_steps")}
                        rec["queue_overflow"] = r.stats["n_queue_overflow"]
                        rec["mean_mu"] = float(out2.mean())
                rec["order_p"] = f2.info()["order"]
                f2.close()
            maps[workload_name(c2)] = rec
            del out2

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        e, t, thr, sub = oracle_sample(cfg, (384, 384))
        cpu = {"value": e / t, "unit": UNIT, "cores": thr, "kind": "oracle", "seconds": t,
               "sample": f"IPM + IRS on the 384x384-cell patch {sub} at the window centre "
                         f"({e} evaluations, each a direct sum over all {cfg.n_stars} stars)"}

    if rank == 0:
        irs = state["irs"]
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "rays_ipm": evals_ipm, "rays_irs": evals_irs,
                       "stars_seed": seed, "order_p": p, "tile_order": state["ipm"]["tile_order"], "border": "eq16",
                       "l2": "flushed between steps (512 MiB fill outside the per-step events)",
                       "parallelism": (f"{world} GPUs: star-weighted row slabs of one map + all-reduce of the map "
                                       f"(rank 0 rows {state['slab']})") if world > 1 else "1 GPU"},
            "phases_ms": {"ipm_map": st["ms_total"], "ipm_shoot_kernels": st["ms_shoot"], "ipm_drain_and_walk_kernels": st["ms_drain"],
                          "irs_map": irs["ms_total"], "irs_shoot_kernels": irs["ms_shoot"],
                          "create_and_rest": sec * 1e3 - st["ms_total"] - irs["ms_total"]},
            "ipm_map_wall_ms": st["ms_total"],
            "evals_per_s_ipm_kernel": rays_k / (st["ms_shoot"] * 1e-3) if st["ms_shoot"] > 0 else None,
            "triangles": {k_: st[k_] for k_ in ("n_tri_single", "n_tri_strip", "n_tri_queued", "n_tri_walked",
                                                  "n_queue_overflow", "n_px_clipped", "n_edge_steps", "n_rays_fallback")},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "roofline": roofline, "cpu_baseline": cpu, "atomics": atomics, "f32_mode": f32, "consumers": consumers, "maps": maps,
        }))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
