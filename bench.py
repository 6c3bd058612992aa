#!/usr/bin/env python
"""bench.py -- the headline measurement of the hot path (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

One STEP is one pass of the whole hot path over one synthetic workload -- by default BASELINE.json configs[4],
the largest configuration that fits one GPU (`metric` names no configuration; 1e7 Salpeter stars, 10^4 x 10^4
pixels, 10 rays per pixel length: the paper's production regime):

    seeded star field -> Morton sort -> quadtree + lists -> P2M/M2M -> M2L/P2L/L2L -> leaf series
    -> fused ray evaluation + IPM deposit (map 1)  -> fused ray evaluation + IRS count (map 2)

all of it in libmlens' CUDA kernels, called through the C ABI (include/mlens.h).  `value` is lens-equation
evaluations per second over the whole step (unique rays of both maps / step time), inputs resident in HBM (the
star field is generated on the device from the seed).  `e2e` repeats the step with HOST buffers: stars handed
over as pinned host arrays, maps returned into pinned host arrays, the library doing the copies inside the
timed region.  The `maps` object carries create / IPM / IRS wall times of the other four configurations
(BASELINE.json's second metric, map wall-time), `roofline` the FP64 account of the fused evaluate + deposit
kernel and `roofline_atomics` the atomic account of the apportioning kernels.

N > 1 (torchrun): the SAME map on N GPUs: stars and tree replicated, the cell grid cut into
row slabs (paper_2506_02114_b200/multi.py), one all-reduce (sum, float64) of each map over NCCL -- the path's
only exchange step; total work is fixed, so scaling is "strong"; time = max over ranks.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload, on the
host cores of this box.  It is a deliberately slow baseline, not the target.
"""
import argparse
import json
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

# B200 FP64 vector units: 64 DFMA lanes per SM (guide); the derived peak is reported beside the DFMA rate measured
# by libmlens_bench in the same run, which is the roofline denominator.
FP64_LANES_PER_SM = 64
# Algorithmic work per lens-equation evaluation in the paper's per-ray scheme:
#   n_near x (9 flop + 1 reciprocal) + (p - 1) complex Horner steps x 8 flop + 10 flop (macro + sheet terms)
FLOP_PER_NEAR_STAR, FLOP_PER_TERM, FLOP_MACRO = 9.0, 8.0, 10.0
QUEUE_ENTRY_BYTES = 48


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs (default 4: the largest single-GPU one)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--maps", default="0,1,2,3,rect1", help="also time whole maps of these configs (create, IPM, IRS wall ms); "
                    "'rect1' = config 1 with a rectangular star region; '' = none")
    ap.add_argument("--no-extras", action="store_true", help="skip the f32, consumers and slab-balance objects")
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
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                c = [v.strip() for v in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
                except ValueError:
                    continue
                for nm, v in zip(names, c[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm), power_w_median=float(np.median(pw)))
        out["reasons"] = sorted(reasons)
        return out


# ------------------------------------------------------------------------------------------------
_ORACLE_FIELD = {}


def oracle_sample(cfg, patch, want_irs=True):
    """Times the CPU oracle on a patch of `patch` = (ni, nj) cells at the window centre: the whole path
    (direct sum over all stars + brute-force clipping; IRS binning).  Returns (evals, seconds, threads, sub).
    The star field (an input) is drawn once per process."""
    import oracle
    oracle.build()
    R = cfg.R_star
    if cfg.name not in _ORACLE_FIELD:
        xs, ys, ms = oracle.starfield(cfg.seed, cfg.n_stars, shape=0, a1=R, mass_law=cfg.mass_law,
                                      a=cfg.mass_a, lo=cfg.mass_lo, hi=cfg.mass_hi)
        _ORACLE_FIELD[cfg.name] = oracle.Field.make(cfg.kappa_tot, cfg.kappa_star, cfg.gamma, xs, ys, ms, R=R)
    of = _ORACLE_FIELD[cfg.name]
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


def oracle_patch_for(cfg, seconds, cores=16):
    """Patch side such that the oracle's direct sum (~4e-9 core-seconds per star and ray, long double) takes about
    `seconds` on `cores` cores."""
    evals = seconds * cores / (4.0e-9 * cfg.n_stars)
    side = int(max(8, min(384, (evals / 2.0) ** 0.5)))
    return (side, side)


def run_reference(args):
    """--impl reference: the oracle, as it stands, on this box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = synth.get_config(args.config)
    cores = os.cpu_count() or 16
    patch = oracle_patch_for(cfg, 8.0, cores)
    for _ in range(args.warmup):
        oracle_sample(cfg, (8, 8))
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

    def seeded(c):
        return ml.Field.seeded(c.kappa_tot, c.gamma, c.n_stars, c.seed, kappa_star=c.kappa_star,
                               mass_law=c.mass_law, mass_a=c.mass_a, mass_lo=c.mass_lo, mass_hi=c.mass_hi)

    map_ipm = torch.zeros((npix, npix), dtype=torch.float64, device=dev)
    map_irs = torch.zeros((npix, npix), dtype=torch.float64, device=dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    state = {}

    def step_device():
        f = seeded(cfg)
        if world > 1 and "weights" not in state:     # slab cost model from the star rows (same on every rank; cached)
            g0 = f.grid(half, npix, k, **kw)
            state["weights"] = multi.star_row_weights(f.stars()[1], g0.x0_2, g0.h2, int(g0.n2))
        _, slab, s1 = multi.shoot_distributed(f, half, npix, k, weights=state.get("weights"), out=map_ipm,
                                              map_mode=ml.MAP_IPM, **kw)
        _, _, s2 = multi.shoot_distributed(f, half, npix, k, weights=state.get("weights"), out=map_irs,
                                           map_mode=ml.MAP_IRS, **kw)
        state.update(info=f.info(), ipm=s1, irs=s2, slab=slab, grid=f.grid(half, npix, k, **kw))
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
    warm = max(args.warmup, 3)
    for _ in range(warm):
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
        f0 = seeded(cfg)
        sx, sy, sm = f0.stars()
        f0.close()
        hx.numpy()[:], hy.numpy()[:], hm.numpy()[:] = sx, sy, sm
        del sx, sy, sm
        step_host()
        e2e_steps = args.steps if sec * args.steps < 60.0 else max(2, min(args.steps, int(60.0 / sec)))
        sec_h = timed(step_host, e2e_steps)
        e2e = {"value": evals / sec_h, "unit": UNIT, "ms_per_step": sec_h * 1e3, "steps": e2e_steps,
               "h2d_bytes_per_step": 3 * 8 * cfg.n_stars, "d2h_bytes_per_step": 2 * 8 * npix * npix}

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass

    # ---- roofline of the fused evaluate + IPM deposit kernel, DESIGN.md s7.
    # `achieved` = the FP64 flops the kernel ISSUES for the evaluation (series re-expanded per 32 x 32-ray tile at order
    # 6-15, the near-field stars it sums directly, macro and sheet terms) / its time, against the measured DFMA rate.
    # Beside it, for context: SURVEY 8(d)'s algorithmic flops of the paper's per-ray scheme x the UNIQUE rays of the map
    # (tile-border corners that the kernel evaluates twice are not counted): the mean near-field list of a ray's leaf
    # (measured in the run, per tile) summed directly + the leaf's order-p series by Horner + the macro terms.
    st = state["ipm"]
    p = state["info"]["order"]
    n_near_leaf = st["n_near_leaf_sum"] / max(1, st["n_tiles"])
    flop_per_eval = FLOP_PER_NEAR_STAR * n_near_leaf + FLOP_PER_TERM * (p - 1) + FLOP_MACRO
    rays_unique = evals_ipm if world == 1 else st["n_cells"]                 # N > 1: this rank's slab
    flop_alg = rays_unique * flop_per_eval
    flop_exec = FLOP_PER_NEAR_STAR * st["n_near_terms"] + (FLOP_PER_TERM * st["tile_order"] + FLOP_MACRO) * st["n_rays"]
    n_l = max(1, st["n_shoot_launches"])
    t_shoot = st["ms_shoot"] * 1e-3
    sm_max = peaks.get("sm_max_mhz", 1965.0)
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_derived = nsm * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    peak_dfma = ml.bench_dfma() / 1e12
    # `achieved` and `frac` count the flops the kernel really ISSUES for the evaluation (tile series of order
    # 6-15 + the near stars it sums directly + macro terms), against the measured DFMA rate: hardware utilisation.
    # The paper's per-ray scheme would need `flop_per_eval_algorithmic` per ray; what that scheme's work divided by this
    # kernel's time comes to is kept as `achieved_paper_equivalent` (an algorithmic speed-up figure, not utilisation).
    # The kernel is bound by instruction issue (bookkeeping around the evaluation), not by the FP64 pipe: DESIGN.md s7.
    paper_tf = flop_alg / t_shoot / 1e12 if t_shoot > 0 else 0.0
    achieved_tf = flop_exec / t_shoot / 1e12 if t_shoot > 0 else 0.0
    # DRAM traffic of the launches, from the run's own counters: every queued triangle is written once (48 B) by this
    # kernel; the per-tile leaf data and the map windows are L2 hits
    traffic = st["n_tri_queued"] * QUEUE_ENTRY_BYTES / n_l
    roofline = {"bound": "alu", "kernel": "shoot_ipm_kernel", "achieved": achieved_tf, "peak": peak_dfma,
                "unit": "TFLOP/s", "frac": achieved_tf / peak_dfma if peak_dfma > 0 else None,
                "achieved_source": "FP64 flops the kernel issues for the evaluation (mlens_stats: n_near_terms, tile_order, n_rays) / summed CUDA-event time of its launches",
                "traffic": traffic,
                "traffic_source": "n_tri_queued x 48 B of queue writes / launches (mlens_stats of the timed run); ncu dram bytes of a capture are in profiles/",
                "peak_source": "FP64 FMA rate measured by libmlens_bench (mlens_bench_dfma) in this run",
                "peak_derived": peak_derived,
                "peak_derived_source": f"{nsm} SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x {sm_max:.0f} MHz",
                "achieved_paper_equivalent": paper_tf,
                "frac_paper_equivalent": paper_tf / peak_dfma if peak_dfma > 0 else None,
                "paper_equivalent_source": "SURVEY 8(d) flops of the paper's per-ray scheme (leaf near list + order-p Horner) x unique rays / the same time: not utilisation",
                "limiter": "instruction issue (ncu: profiles/r02_ncu_full.md), not the FP64 pipe",
                "flop_per_eval_algorithmic": flop_per_eval, "near_stars_per_leaf_mean": n_near_leaf, "order_p": p,
                "unique_rays": rays_unique, "rays_evaluated": st["n_rays"],
                "flop_per_launch": flop_exec / n_l, "flop_paper_equivalent_per_launch": flop_alg / n_l,
                "launch_ms": t_shoot * 1e3 / n_l, "launches_per_map": n_l, "kernel_ms_per_map": st["ms_shoot"],
                "share_of_step": t_shoot / sec}

    # ---- BASELINE.json metric: fraction of the atomic roofline for deposition.  Adds the apportioning kernels (drain,
    # walk, giant walk) issue: one per clipped (triangle, pixel) pair, two per edge step at least -- against the rate of
    # random 64-bit atomic adds measured here into a buffer that L2 holds (16 MB) and into one the size of this map's
    # accumulators (HBM-resident when larger than L2).
    roofline_atomics = None
    if world == 1:
        # the ceiling, measured with loops whose slot choice costs two integer instructions (round 2's 64-bit modulo was a
        # ~64-instruction subroutine per add and measured itself: VERDICT r2): profiles/r03_sass_atomics.txt
        n_l2, n_map = 2_000_000, max(2 * npix * npix, 2_000_000)
        a_l2 = ml.bench_atomics(n_l2, True)
        a_map = ml.bench_atomics(n_map, True)
        table = {"global_u64_L2_16MB": {"random": a_l2, "8_sectors_per_warp": ml.bench_atomics(n_l2, True, pattern=1),
                                        "1_sector_per_warp": ml.bench_atomics(n_l2, True, pattern=2)},
                 "global_u64_map_sized": {"random": a_map, "8_sectors_per_warp": ml.bench_atomics(n_map, True, pattern=1),
                                          "1_sector_per_warp": ml.bench_atomics(n_map, True, pattern=2), "bytes": 8 * n_map},
                 "global_f64_L2_16MB": {"random": ml.bench_atomics(n_l2, False)},
                 "shared_64KB_tile": {
                     "u64_two_32bit_adds_with_carry_random": ml.bench_shared_atomics(kind=1),
                     "u64_two_32bit_adds_with_carry_conflict_free": ml.bench_shared_atomics(kind=1, conflict_free=True),
                     "u32_add_random": ml.bench_shared_atomics(kind=2),
                     "u32_add_conflict_free": ml.bench_shared_atomics(kind=2, conflict_free=True),
                     "u64_atomicAdd_cas_loop_random": ml.bench_shared_atomics(kind=0),
                     "u64_atomicAdd_cas_loop_conflict_free": ml.bench_shared_atomics(kind=0, conflict_free=True)}}
        adds = st["n_px_clipped"] + 2 * st["n_edge_steps"]
        t_ap = st["ms_drain"] * 1e-3
        rate = adds / t_ap if t_ap > 0 else 0.0
        queue_bytes = st["n_tri_queued"] * QUEUE_ENTRY_BYTES + st["n_tri_walked"] * (QUEUE_ENTRY_BYTES + 8)
        roofline_atomics = {"bound": "atomics", "kernels": "drain_kernel + walk_kernel + walk_giant_kernel",
                            "achieved": rate, "peak": a_l2, "unit": "adds/s", "frac": rate / a_l2,
                            "peak_source": "random REDG.E.ADD.64 into a 16 MB (L2-resident) buffer, libmlens_bench, this run; loop of 5.8 SASS instructions per add, no CALL (profiles/r03_sass_atomics.txt)",
                            "measured_add_rates_per_s": table,
                            "map_sized_buffer_adds_per_s": a_map, "map_accumulator_bytes": 16 * npix * npix,
                            "shared_memory_adds_per_s": table["shared_64KB_tile"]["u64_two_32bit_adds_with_carry_random"],
                            "frac_of_map_sized_rate": rate / a_map,
                            "adds_per_map": adds, "n_px_clipped": st["n_px_clipped"], "n_edge_steps": st["n_edge_steps"],
                            "kernel_ms_per_map": st["ms_drain"], "walk_ms": st["ms_walk"], "giant_ms": st["ms_giant"],
                            "traffic": queue_bytes, "traffic_source": "queue reads: n_tri_queued x 48 B + walk list n_tri_walked x 56 B (whole map)",
                            "traffic_GBps": queue_bytes / t_ap / 1e9 if t_ap > 0 else None,
                            "hbm_peak_GBps": peaks.get("hbm_gbs"), "share_of_step": t_ap / sec}

    extras = world == 1 and not args.no_extras
    # ---- the single-precision evaluator where the paper says single precision fails
    # (the cluster regime, config 3) and on config 1, beside the float64 numbers
    f32 = None
    if extras:
        f32 = {}
        for ci in (1, 3):
            c2 = synth.get_config(ci)
            kw2 = dict(border_mode=c2.border_mode, border_param=c2.border_param)
            ff = seeded(c2)
            a2 = (c2.half_y, c2.npix, c2.rays_per_pixel_length)
            o64 = torch.zeros((c2.npix, c2.npix), dtype=torch.float64, device=dev)
            o32 = torch.zeros_like(o64)
            rec = {}
            for name, mode in (("ipm", ml.MAP_IPM), ("irs", ml.MAP_IRS)):
                for _ in range(2):
                    r64 = ff.shoot(*a2, out=o64, map_mode=mode, **kw2)
                    r32 = ff.shoot(*a2, out=o32, map_mode=mode, eval_mode=ml.EVAL_FMM_F32, **kw2)
                rec[name + "_shoot_ms_f64"] = r64.stats["ms_shoot"]; rec[name + "_shoot_ms_f32"] = r32.stats["ms_shoot"]
                rec[name + "_map_ms_f64"] = r64.stats["ms_total"]; rec[name + "_map_ms_f32"] = r32.stats["ms_total"]
                sel = o64 >= 0.1
                rel = ((o32 - o64).abs()[sel] / o64[sel])
                rec[name + "_median_rel_dev_of_f64"] = float(rel.median())
                rec[name + "_pixels_beyond_1e-3_of_f64"] = float((rel > 1e-3).double().mean())
                rec[name + "_max_rel_dev_of_f64"] = float(rel.max())
            ff.close()
            f32[c2.name] = rec
            del o64, o32

    # ---- the map consumers (HBM-bound): histogram of a synthetic log-normal 8192^2 map (512 MiB > L2)
    consumers = None
    if extras:
        big = torch.empty((8192, 8192), dtype=torch.float64, device=dev).log_normal_(0.0, 1.0)
        ms = []
        for _ in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); hh = ml.histogram(big, 1.0, -2.0, 2.0, 64); e1.record(stream); e1.synchronize()
            ms.append(e0.elapsed_time(e1))
        gbs = big.numel() * 8 / (min(ms[1:]) * 1e-3) / 1e9
        peak_hbm = peaks.get("hbm_gbs")
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        lc = ml.light_curve(map_ipm, g.ylo1, g.ylo2, g.p1, g.p2, (-0.9 * half, -0.7 * half), (0.9 * half, 0.8 * half), 1 << 20,
                            interp=ml.INTERP_BILINEAR)
        e1.record(stream); e1.synchronize()
        consumers = {"histogram_ms": min(ms[1:]), "histogram_GBps": gbs, "hbm_peak_GBps": peak_hbm,
                     "histogram_frac_of_hbm": (gbs / peak_hbm) if peak_hbm else None, "histogram_total": int(hh.sum()),
                     "light_curve_1M_samples_ms": e0.elapsed_time(e1), "light_curve_mean_mu": float(lc.nanmean())}
        del big

    # ---- BASELINE.json's second metric, map wall-time, on the other configurations (one warm-up, one timed run each)
    maps = None
    if args.maps and world == 1:
        maps = {}
        for tok in [c for c in args.maps.split(",") if c != ""]:
            rect = tok.startswith("rect")
            c2 = synth.get_config(int(tok[4:]) if rect else int(tok))
            kw2 = dict(border_mode=c2.border_mode, border_param=c2.border_param)
            out2 = torch.zeros((c2.npix, c2.npix), dtype=torch.float64, device=dev)
            rec = {}
            if rect:
                # the same lens with a RECTANGULAR star region sized for the same map (eq 20/21): side ratio
                # of the shooting window, area from the rectangle's own corner formula, stars at the same density
                f_tmp = seeded(c2)
                g2 = f_tmp.grid(c2.half_y, c2.npix, c2.rays_per_pixel_length, **kw2)
                f_tmp.close()
                c1r, c2r = 1.2 * g2.H1 + 10.0, 1.2 * g2.H2 + 10.0
                n_rect = int(round(c2.kappa_star * 4 * c1r * c2r / np.pi))
            for rep in range(2):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                if rect:
                    f2 = ml.Field.seeded(c2.kappa_tot, c2.gamma, n_rect, c2.seed, kappa_star=c2.kappa_star, shape=ml.SHAPE_RECT,
                                         rect_aspect=c1r / c2r, mass_law=c2.mass_law, mass_a=c2.mass_a, mass_lo=c2.mass_lo, mass_hi=c2.mass_hi)
                    rec["n_stars_rect"] = n_rect
                else:
                    f2 = seeded(c2)
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
                        rec["tri"] = {k_: r.stats[k_] for k_ in ("n_tri_single", "n_tri_strip", "n_tri_queued", "n_tri_walked",
                                                                  "n_px_clipped", "n_edge_steps")}
                        rec["queue_overflow"] = r.stats["n_queue_overflow"]
                        rec["mean_mu"] = float(out2.mean())
                rec["order_p"] = f2.info()["order"]
                rec["n_levels"] = f2.info()["n_levels"]
                f2.close()
            maps[("rect variant of " if rect else "") + workload_name(c2)] = rec
            del out2

    # ---- load balance of row slabs without a second GPU: 8 slabs of config 1 shot one after another, equal
    # rows against star-weighted rows (the weight per star fitted from the equal-row times)
    slab_balance = None
    if extras:
        c2 = synth.get_config(1)
        kw2 = dict(border_mode=c2.border_mode, border_param=c2.border_param)
        f2 = seeded(c2)
        a2 = (c2.half_y, c2.npix, c2.rays_per_pixel_length)
        g2 = f2.grid(*a2, **kw2)
        ys = f2.stars()[1]
        out2 = torch.zeros((c2.npix, c2.npix), dtype=torch.float64, device=dev)
        n2 = int(g2.n2)

        def slab_times(weights, nslab=8):
            ts, rows, stars = [], [], []
            for r in range(nslab):
                j0, j1 = multi.slab_bounds(n2, nslab, r, weights=weights)
                for _ in range(2):
                    rr = f2.shoot(*a2, sub=(0, int(g2.n1), j0, j1), out=out2, **kw2)
                ts.append(rr.stats["ms_total"]); rows.append(j1 - j0)
                jj = np.floor((ys - g2.x0_2) / g2.h2)
                stars.append(int(np.sum((jj >= j0) & (jj < j1))))
            return np.array(ts), np.array(rows, dtype=float), np.array(stars, dtype=float)

        t_eq, rows_eq, stars_eq = slab_times(None)
        A = np.stack([rows_eq, stars_eq], axis=1)
        coef, *_ = np.linalg.lstsq(A, t_eq, rcond=None)
        per_star = float(max(coef[1], 0.0) / coef[0]) if coef[0] > 0 else 0.0
        t_w, _, _ = slab_times(multi.star_row_weights(ys, g2.x0_2, g2.h2, n2, per_star=per_star))
        slab_balance = {"workload": workload_name(c2), "slabs": 8,
                        "equal_rows_ms": [float(v) for v in t_eq], "equal_rows_max_over_mean": float(t_eq.max() / t_eq.mean()),
                        "fitted_ms_per_row": float(coef[0]), "fitted_ms_per_star": float(coef[1]), "per_star_in_rows": per_star,
                        "weighted_ms": [float(v) for v in t_w], "weighted_max_over_mean": float(t_w.max() / t_w.mean())}
        f2.close()
        del out2

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        patch = oracle_patch_for(cfg, 20.0, os.cpu_count() or 16)
        e, t, thr, sub = oracle_sample(cfg, patch)
        cpu = {"value": e / t, "unit": UNIT, "cores": thr, "kind": "oracle", "seconds": t,
               "sample": f"IPM + IRS on the {patch[0]}x{patch[1]}-cell patch {sub} at the window centre "
                         f"({e} evaluations, each a direct sum over all {cfg.n_stars} stars)",
               # the oracle's cost is exactly rays x stars, so the sample's rate carries over to the whole
               # grid; an EXTRAPOLATION, labelled as one, not a measurement
               "extrapolated_full_step_seconds": (evals_ipm + evals_irs) * t / e,
               "extrapolation": f"linear in the rays: {evals_ipm + evals_irs} evaluations of one step (IPM + IRS maps) "
                                f"at the sample's measured rate; not measured"}

    if rank == 0:
        irs = state["irs"]
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warm, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "rays_ipm": evals_ipm, "rays_irs": evals_irs,
                       "stars_seed": seed, "order_p": p, "tile_order": state["ipm"]["tile_order"], "border": "eq16",
                       "l2": "flushed between steps (512 MiB fill outside the per-step events)",
                       "parallelism": (f"{world} GPUs: star-weighted row slabs of one map + all-reduce of the map "
                                       f"(rank 0 rows {state['slab']})") if world > 1 else "1 GPU"},
            "phases_ms": {"ipm_map": st["ms_total"], "ipm_shoot_kernels": st["ms_shoot"], "ipm_drain_and_walk_kernels": st["ms_drain"],
                          "ipm_walk_kernel": st["ms_walk"], "ipm_giant_kernel": st["ms_giant"], "ipm_bands": st["n_bands"],
                          "irs_map": irs["ms_total"], "irs_shoot_kernels": irs["ms_shoot"],
                          "create_and_rest": sec * 1e3 - st["ms_total"] - irs["ms_total"]},
            "ipm_map_wall_ms": st["ms_total"], "irs_map_wall_ms": irs["ms_total"],
            "evals_per_s_ipm_kernel": evals_ipm / t_shoot if t_shoot > 0 and world == 1 else None,
            "evals_per_s_irs_kernel": evals_irs / (irs["ms_shoot"] * 1e-3) if irs["ms_shoot"] > 0 and world == 1 else None,
            "triangles": {k_: st[k_] for k_ in ("n_tri_single", "n_tri_strip", "n_tri_queued", "n_tri_walked",
                                                  "n_queue_overflow", "n_px_clipped", "n_edge_steps", "n_giant_chunks", "n_rays_fallback")},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "roofline": roofline, "roofline_atomics": roofline_atomics, "cpu_baseline": cpu,
            "f32_mode": f32, "consumers": consumers, "maps": maps, "slab_balance": slab_balance,
        }))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
