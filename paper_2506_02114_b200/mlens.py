"""ctypes binding of libmlens (include/mlens.h): argument marshalling only.

torch supplies device memory and the stream; numpy arrays are passed as HOST pointers (the library
then does the copies itself).  Missing library or missing CUDA device => MlensError, never a fallback.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libmlens.so")
_BENCH_SO = os.path.join(_HERE, "libmlens_bench.so")
_lib = None
_bench_lib = None

SHAPE_DISC, SHAPE_RECT = 0, 1
MASS_EQUAL, MASS_POWER = 0, 1
EVAL_FMM, EVAL_DIRECT, EVAL_FMM_F32 = 0, 1, 2
MAP_IPM, MAP_IRS = 0, 1
BORDER_EQ16, BORDER_A6, BORDER_MARGIN, BORDER_EXPLICIT = 0, 1, 2, 3
PTR_DEVICE, PTR_HOST = 0, 1
MAX_ORDER, MAX_DIRECT = 47, 32

_dp = C.POINTER(C.c_double)
_u64p = C.POINTER(C.c_uint64)
_i32p = C.POINTER(C.c_int32)


class MlensError(RuntimeError):
    pass


class FieldDesc(C.Structure):
    _fields_ = [("kappa_tot", C.c_double), ("kappa_star", C.c_double), ("kappa_smooth", C.c_double),
                ("gamma", C.c_double), ("theta_star", C.c_double), ("shape", C.c_int32), ("ptr_kind", C.c_int32),
                ("R", C.c_double), ("c1", C.c_double), ("c2", C.c_double), ("n_stars", C.c_int64),
                ("x", C.c_void_p), ("y", C.c_void_p), ("m", C.c_void_p), ("eps_deflection", C.c_double),
                ("max_direct", C.c_int32), ("order", C.c_int32), ("stream", C.c_void_p)]


class SeedDesc(C.Structure):
    _fields_ = [("kappa_tot", C.c_double), ("kappa_star", C.c_double), ("kappa_smooth", C.c_double),
                ("gamma", C.c_double), ("theta_star", C.c_double), ("shape", C.c_int32), ("mass_law", C.c_int32),
                ("rect_aspect", C.c_double), ("mass_a", C.c_double), ("mass_lo", C.c_double), ("mass_hi", C.c_double),
                ("n_stars", C.c_int64), ("seed", C.c_uint64), ("eps_deflection", C.c_double),
                ("max_direct", C.c_int32), ("order", C.c_int32), ("stream", C.c_void_p)]


class FieldInfo(C.Structure):
    _fields_ = [("n_stars", C.c_int64), ("order", C.c_int32), ("n_levels", C.c_int32), ("n_nodes", C.c_int64),
                ("n_leaves", C.c_int64), ("root_half", C.c_double), ("leaf_half_min", C.c_double),
                ("kappa_star_actual", C.c_double), ("mean_m", C.c_double), ("mean_m2", C.c_double),
                ("R", C.c_double), ("c1", C.c_double), ("c2", C.c_double), ("spot_check_err", C.c_double),
                ("max_near", C.c_int32), ("max_m2l", C.c_int32), ("max_p2l", C.c_int32)]


class ShootDesc(C.Structure):
    _fields_ = [("center_y1", C.c_double), ("center_y2", C.c_double), ("half_y1", C.c_double), ("half_y2", C.c_double),
                ("npix1", C.c_int32), ("npix2", C.c_int32), ("rays_per_pixel_length", C.c_double),
                ("map_mode", C.c_int32), ("eval_mode", C.c_int32), ("border_mode", C.c_int32), ("accumulate", C.c_int32),
                ("border_param", C.c_double), ("He1", C.c_double), ("He2", C.c_double),
                ("i0", C.c_int64), ("i1", C.c_int64), ("j0", C.c_int64), ("j1", C.c_int64),
                ("ptr_kind", C.c_int32), ("sync", C.c_int32), ("dump_w1", C.c_void_p), ("dump_w2", C.c_void_p),
                ("queue_mb", C.c_int32), ("tile_order", C.c_int32), ("small_px", C.c_int32), ("band_fixed", C.c_int32),
                ("band_cells", C.c_int64), ("tile_traversal", C.c_int32), ("pad_", C.c_int32)]


class Grid(C.Structure):
    _fields_ = [("X1", C.c_double), ("X2", C.c_double), ("H1", C.c_double), ("H2", C.c_double),
                ("h1", C.c_double), ("h2", C.c_double), ("p1", C.c_double), ("p2", C.c_double),
                ("x0_1", C.c_double), ("x0_2", C.c_double), ("ylo1", C.c_double), ("ylo2", C.c_double),
                ("n1", C.c_int64), ("n2", C.c_int64), ("weight", C.c_double), ("order", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [("n_rays", C.c_int64), ("n_cells", C.c_int64), ("n_tri_single", C.c_int64), ("n_tri_strip", C.c_int64),
                ("n_tri_queued", C.c_int64), ("n_tri_walked", C.c_int64), ("n_queue_overflow", C.c_int64),
                ("n_rays_fallback", C.c_int64), ("n_bands", C.c_int32), ("gpu_launches", C.c_int32),
                ("ms_total", C.c_float), ("ms_shoot", C.c_float), ("ms_drain", C.c_float),
                ("ms_finalise", C.c_float), ("n_shoot_launches", C.c_int32), ("n_near_terms", C.c_int64),
                ("n_px_strip", C.c_int64), ("n_px_clipped", C.c_int64), ("n_edge_steps", C.c_int64), ("reserved_", C.c_int64),
                ("n_tiles_full", C.c_int64), ("tile_order", C.c_int32), ("pad_", C.c_int32),
                ("ms_walk", C.c_float), ("ms_giant", C.c_float), ("n_giant_chunks", C.c_int64),
                ("n_tiles", C.c_int64), ("n_near_leaf_sum", C.c_int64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class TreeView(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in
                ("level", "ix", "iy", "parent", "child0", "star_lo", "star_n", "leaf_id", "nbr",
                 "m2l_cnt", "m2l_list", "p2l_cnt", "p2l_list", "multipole", "local",
                 "near_cnt", "near_x", "near_y", "near_m", "sorted_x", "sorted_y", "sorted_m")]


def lib():
    """Loads libmlens.so (in-tree).  Raises MlensError if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise MlensError(f"{_SO} is missing: run `python -m paper_2506_02114_b200.build` "
                             "(there is no CPU fallback)")
        L = C.CDLL(_SO)
        L.mlens_version.restype = C.c_int
        L.mlens_last_error.restype = C.c_char_p
        L.mlens_launch_count.restype = C.c_int64
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.mlens_field_create.argtypes = [C.POINTER(FieldDesc), C.POINTER(vp)]
        L.mlens_field_create_seeded.argtypes = [C.POINTER(SeedDesc), C.POINTER(vp)]
        L.mlens_field_destroy.argtypes = [vp]
        L.mlens_field_get_info.argtypes = [vp, C.POINTER(FieldInfo)]
        L.mlens_field_get_stars.argtypes = [vp, vp, vp, vp, i32, vp]
        L.mlens_deflect.argtypes = [vp, i64, vp, vp, vp, vp, i32, i32, vp]
        L.mlens_lens_map.argtypes = [vp, i64, vp, vp, vp, vp, i32, i32, vp]
        L.mlens_grid_info.argtypes = [vp, C.POINTER(ShootDesc), C.POINTER(Grid)]
        L.mlens_shoot.argtypes = [vp, C.POINTER(ShootDesc), vp, vp, C.POINTER(Stats), vp]
        L.mlens_field_get_tree.argtypes = [vp, C.POINTER(TreeView)]
        dbl = C.c_double
        L.mlens_map_light_curve.argtypes = [vp, i32, i32, dbl, dbl, dbl, dbl, dbl, dbl, dbl, dbl, i64, i32, vp, i32, vp]
        L.mlens_map_histogram.argtypes = [vp, i64, dbl, dbl, dbl, i32, vp, i32, vp]
        L.mlens_map_histogram_static.argtypes = [vp, i64, dbl, dbl, dbl, i32, vp, vp]
        L.mlens_field_set_macro_quadratic.argtypes = [vp, dbl, dbl, dbl, dbl]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise MlensError(f"libmlens error {rc}: {lib().mlens_last_error().decode()}")


def version():
    return lib().mlens_version()


def launch_count():
    """Kernels launched by libmlens in this process so far."""
    return int(lib().mlens_launch_count())


def _is_torch(a):
    return type(a).__module__.startswith("torch")


def _ptr(a):
    """(pointer, ptr_kind) of a torch CUDA tensor or a numpy array; keeps nothing alive."""
    if a is None:
        return None, None
    if _is_torch(a):
        if not a.is_cuda:
            raise MlensError("torch tensors must live on the CUDA device (pass numpy arrays for host data)")
        if not a.is_contiguous():
            raise MlensError("tensor must be contiguous")
        return a.data_ptr(), PTR_DEVICE
    if not isinstance(a, np.ndarray) or not a.flags["C_CONTIGUOUS"]:
        raise MlensError("expected a C-contiguous numpy array or a CUDA tensor")
    return a.ctypes.data, PTR_HOST


def _stream(stream):
    if stream is None:
        try:
            import torch
            if torch.cuda.is_available():
                return torch.cuda.current_stream().cuda_stream
        except ImportError:
            pass
        return None
    return getattr(stream, "cuda_stream", stream)


def _same_kind(*arrs):
    kinds = {_ptr(a)[1] for a in arrs if a is not None}
    if len(kinds) > 1:
        raise MlensError("all arrays of one call must be either numpy (host) or CUDA tensors (device)")
    return kinds.pop() if kinds else PTR_DEVICE


class ShootResult:
    def __init__(self, map_, counts, stats, grid, dump):
        self.map, self.counts, self.stats, self.grid, self.dump = map_, counts, stats, grid, dump


class Field:
    """A lens field (mlens_field handle).  Use Field.from_stars or Field.seeded."""

    def __init__(self, handle):
        self._h = handle

    # ---- creation ------------------------------------------------------------------------------
    @classmethod
    def from_stars(cls, kappa_tot, gamma, x, y, m, *, kappa_star=float("nan"), kappa_smooth=float("nan"),
                   shape=SHAPE_DISC, R=0.0, c1=0.0, c2=0.0, theta_star=1.0, eps=1e-8, max_direct=0, order=0,
                   stream=None):
        d = FieldDesc()
        d.kappa_tot, d.kappa_star, d.kappa_smooth, d.gamma, d.theta_star = kappa_tot, kappa_star, kappa_smooth, gamma, theta_star
        d.shape, d.R, d.c1, d.c2 = shape, R, c1, c2
        if not _is_torch(x):
            x, y, m = (np.ascontiguousarray(a, dtype=np.float64) for a in (x, y, m))
        d.ptr_kind = _same_kind(x, y, m)
        d.n_stars = int(x.shape[0]) if x.ndim else 0
        d.x, d.y, d.m = _ptr(x)[0], _ptr(y)[0], _ptr(m)[0]
        d.eps_deflection, d.max_direct, d.order = eps, max_direct, order
        d.stream = _stream(stream)
        h = C.c_void_p()
        _check(lib().mlens_field_create(C.byref(d), C.byref(h)))
        return cls(h)

    @classmethod
    def seeded(cls, kappa_tot, gamma, n_stars, seed, *, kappa_star=float("nan"), kappa_smooth=float("nan"),
               shape=SHAPE_DISC, rect_aspect=1.0, mass_law=MASS_EQUAL, mass_a=2.35, mass_lo=0.08, mass_hi=1.0,
               theta_star=1.0, eps=1e-8, max_direct=0, order=0, stream=None):
        d = SeedDesc()
        d.kappa_tot, d.kappa_star, d.kappa_smooth, d.gamma, d.theta_star = kappa_tot, kappa_star, kappa_smooth, gamma, theta_star
        d.shape, d.mass_law, d.rect_aspect = shape, mass_law, rect_aspect
        d.mass_a, d.mass_lo, d.mass_hi = mass_a, mass_lo, mass_hi
        d.n_stars, d.seed = n_stars, seed
        d.eps_deflection, d.max_direct, d.order = eps, max_direct, order
        d.stream = _stream(stream)
        h = C.c_void_p()
        _check(lib().mlens_field_create_seeded(C.byref(d), C.byref(h)))
        return cls(h)

    def close(self):
        if self._h:
            lib().mlens_field_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- queries -------------------------------------------------------------------------------
    def info(self):
        i = FieldInfo()
        _check(lib().mlens_field_get_info(self._h, C.byref(i)))
        return {k: getattr(i, k) for k, _ in i._fields_}

    def stars(self):
        """Host copies (numpy) of the stars in the caller's original order."""
        n = self.info()["n_stars"]
        x, y, m = np.empty(n), np.empty(n), np.empty(n)
        _check(lib().mlens_field_get_stars(self._h, x.ctypes.data, y.ctypes.data, m.ctypes.data, PTR_HOST, _stream(None)))
        return x, y, m

    def _points(self, fn, zx, zy, eval_mode, stream):
        if _is_torch(zx):
            import torch
            ox, oy = torch.empty_like(zx), torch.empty_like(zy)
        else:
            zx = np.ascontiguousarray(zx, dtype=np.float64)
            zy = np.ascontiguousarray(zy, dtype=np.float64)
            ox, oy = np.empty_like(zx), np.empty_like(zy)
        kind = _same_kind(zx, zy)
        n = int(np.prod(zx.shape))
        _check(fn(self._h, n, _ptr(zx)[0], _ptr(zy)[0], _ptr(ox)[0], _ptr(oy)[0], eval_mode, kind, _stream(stream)))
        return ox, oy

    def deflect(self, zx, zy, eval_mode=EVAL_FMM, stream=None):
        """alpha_star (eq 13) at the given points."""
        return self._points(lib().mlens_deflect, zx, zy, eval_mode, stream)

    def set_macro_quadratic(self, psi_111, psi_112, psi_122, psi_222):
        """mlens_field_set_macro_quadratic: second-order Taylor term of the macro deflection (App. D; maps next to a
        macro-caustic).  Shooting then needs border_mode=BORDER_EXPLICIT.  All zero switches it off."""
        _check(lib().mlens_field_set_macro_quadratic(self._h, C.c_double(psi_111), C.c_double(psi_112),
                                                     C.c_double(psi_122), C.c_double(psi_222)))
        return self

    def lens_map(self, zx, zy, eval_mode=EVAL_FMM, stream=None):
        """w of eq 12 at the given points."""
        return self._points(lib().mlens_lens_map, zx, zy, eval_mode, stream)

    # ---- shooting ------------------------------------------------------------------------------
    @staticmethod
    def _desc(half_y, npix, k, *, map_mode=MAP_IPM, eval_mode=EVAL_FMM, border_mode=BORDER_A6, border_param=1e-3,
              center=(0.0, 0.0), He=(0.0, 0.0), sub=None, accumulate=False, sync=True,
              queue_mb=0, tile_order=0, small_px=0, band_fixed=False, band_cells=0, tile_traversal=0):
        d = ShootDesc()
        hy = half_y if isinstance(half_y, (tuple, list)) else (half_y, half_y)
        npx = npix if isinstance(npix, (tuple, list)) else (npix, npix)
        d.center_y1, d.center_y2 = center
        d.half_y1, d.half_y2 = hy
        d.npix1, d.npix2 = npx
        d.rays_per_pixel_length = k
        d.map_mode, d.eval_mode, d.border_mode, d.border_param = map_mode, eval_mode, border_mode, border_param
        d.He1, d.He2 = He
        d.accumulate, d.sync = int(accumulate), int(sync)
        d.queue_mb, d.tile_order, d.small_px, d.band_fixed = queue_mb, tile_order, small_px, int(band_fixed)
        d.band_cells, d.tile_traversal = band_cells, tile_traversal
        if sub is not None:
            d.i0, d.i1, d.j0, d.j1 = sub
        return d

    def grid(self, half_y, npix, k, **kw):
        d = self._desc(half_y, npix, k, **kw)
        g = Grid()
        _check(lib().mlens_grid_info(self._h, C.byref(d), C.byref(g)))
        return g

    def shoot(self, half_y, npix, k, *, out=None, counts=None, device=None, dump=False, want_counts=False,
              stream=None, **kw):
        """Builds the map.  Host (numpy) result by default; device=torch.device(...) or a CUDA tensor
        in `out` keeps everything in HBM.  Returns ShootResult(map, counts, stats, grid, dump)."""
        d = self._desc(half_y, npix, k, **kw)
        g = Grid()
        _check(lib().mlens_grid_info(self._h, C.byref(d), C.byref(g)))
        npx2, npx1 = d.npix2, d.npix1
        on_device = device is not None or (out is not None and _is_torch(out))
        irs = d.map_mode == MAP_IRS
        i0, i1, j0, j1 = (d.i0, d.i1, d.j0, d.j1) if (d.i1 > 0 and d.j1 > 0) else (0, g.n1, 0, g.n2)
        dshape = (j1 - j0, i1 - i0) if irs else (j1 - j0 + 1, i1 - i0 + 1)
        if on_device:
            import torch
            dev = device if device is not None else out.device
            if out is None:
                out = torch.zeros((npx2, npx1), dtype=torch.float64, device=dev)
            if irs and want_counts and counts is None:
                counts = torch.zeros((npx2, npx1), dtype=torch.int64, device=dev)   # same bits as uint64
            dw = (torch.empty(dshape, dtype=torch.float64, device=dev), torch.empty(dshape, dtype=torch.float64, device=dev)) if dump else None
        else:
            if out is None:
                out = np.zeros((npx2, npx1))
            if irs and want_counts and counts is None:
                counts = np.zeros((npx2, npx1), dtype=np.uint64)
            dw = (np.empty(dshape), np.empty(dshape)) if dump else None
        d.ptr_kind = _same_kind(out, counts, *(dw or ()))
        if dw:
            d.dump_w1, d.dump_w2 = _ptr(dw[0])[0], _ptr(dw[1])[0]
        st = Stats()
        _check(lib().mlens_shoot(self._h, C.byref(d), _ptr(out)[0], _ptr(counts)[0] if counts is not None else None,
                                 C.byref(st), _stream(stream)))
        return ShootResult(out, counts, st.as_dict(), g, dw)

    # ---- introspection -------------------------------------------------------------------------
    def tree(self):
        """Host copies of the tree arrays (tests)."""
        inf = self.info()
        nn, nl, p1, ns = inf["n_nodes"], inf["n_leaves"], inf["order"] + 1, inf["n_stars"]
        a = {}
        for name in ("level", "ix", "iy", "parent", "child0", "star_lo", "star_n", "leaf_id", "m2l_cnt", "p2l_cnt"):
            a[name] = np.empty(nn, dtype=np.int32)
        a["nbr"] = np.empty((nn, 8), dtype=np.int32)
        a["m2l_list"] = np.empty((nn, 27), dtype=np.int32)
        a["p2l_list"] = np.empty((nn, 8), dtype=np.int32)
        a["multipole"] = np.empty((nn, p1, 2))
        a["local"] = np.empty((nn, p1, 2))
        a["near_cnt"] = np.empty(nl, dtype=np.int32)
        for name in ("near_x", "near_y", "near_m"):
            a[name] = np.empty((nl, MAX_DIRECT))
        for name in ("sorted_x", "sorted_y", "sorted_m"):
            a[name] = np.empty(ns)
        v = TreeView()
        for name, _ in v._fields_:
            setattr(v, name, a[name].ctypes.data)
        _check(lib().mlens_field_get_tree(self._h, C.byref(v)))
        a["multipole"] = a["multipole"][..., 0] + 1j * a["multipole"][..., 1]
        a["local"] = a["local"][..., 0] + 1j * a["local"][..., 1]
        a.update(root_half=inf["root_half"], order=inf["order"])
        return a


def bench_lib():
    """Loads libmlens_bench.so (include/mlens_bench.h): the roofline micro-benchmarks, a library of their own."""
    global _bench_lib
    if _bench_lib is None:
        if not os.path.exists(_BENCH_SO):
            raise MlensError(f"{_BENCH_SO} is missing: run `python -m paper_2506_02114_b200.build`")
        L = C.CDLL(_BENCH_SO)
        L.mlens_bench_dfma.argtypes = [_dp, C.c_void_p]
        L.mlens_bench_atomics.argtypes = [C.c_int64, C.c_int32, _dp, C.c_void_p]
        L.mlens_bench_shared_atomics.argtypes = [_dp, C.c_void_p]
        L.mlens_bench_atomics_pattern.argtypes = [C.c_int64, C.c_int32, C.c_int32, _dp, C.c_void_p]
        L.mlens_bench_shared_atomics_kind.argtypes = [C.c_int32, C.c_int32, _dp, C.c_void_p]
        _bench_lib = L
    return _bench_lib


def _bench_check(rc):
    if rc != 0:
        raise MlensError(f"libmlens_bench: CUDA error {-rc}")


def bench_dfma(stream=None):
    v = C.c_double()
    _bench_check(bench_lib().mlens_bench_dfma(C.byref(v), _stream(stream)))
    return v.value


def bench_atomics(n_slots, use_u64=True, stream=None, pattern=0):
    """Global 64-bit atomic adds per second; pattern 0 random slots, 1 eight sectors per warp, 2 one sector per warp."""
    v = C.c_double()
    _bench_check(bench_lib().mlens_bench_atomics_pattern(n_slots, int(use_u64), int(pattern), C.byref(v), _stream(stream)))
    return v.value


def bench_shared_atomics(stream=None, kind=1, conflict_free=False):
    """Shared-memory atomic adds per second; kind 0 64-bit CAS loop, 1 the product's two 32-bit adds, 2 one 32-bit add."""
    v = C.c_double()
    _bench_check(bench_lib().mlens_bench_shared_atomics_kind(int(kind), int(conflict_free), C.byref(v), _stream(stream)))
    return v.value


# ---- map consumers: marshalling only --------------------------------------------------
INTERP_NEAREST, INTERP_BILINEAR = 0, 1


def light_curve(map_, ylo1, ylo2, p1, p2, ya, yb, n, interp=INTERP_NEAREST, stream=None):
    """mlens_map_light_curve: n samples of the map along the straight source track ya -> yb (numpy or CUDA tensor map)."""
    npix2, npix1 = map_.shape
    if _is_torch(map_):
        import torch
        out = torch.empty(n, dtype=torch.float64, device=map_.device)
    else:
        map_ = np.ascontiguousarray(map_, dtype=np.float64)
        out = np.empty(n)
    kind = _same_kind(map_, out)
    _check(lib().mlens_map_light_curve(_ptr(map_)[0], C.c_int32(npix1), C.c_int32(npix2), C.c_double(ylo1), C.c_double(ylo2),
                                       C.c_double(p1), C.c_double(p2), C.c_double(ya[0]), C.c_double(ya[1]),
                                       C.c_double(yb[0]), C.c_double(yb[1]), C.c_int64(n), C.c_int32(interp),
                                       _ptr(out)[0], C.c_int32(kind), _stream(stream)))
    return out


def histogram(map_, mu_ref, lo, hi, nbins, stream=None):
    """mlens_map_histogram: counts of log10(mu/mu_ref) in nbins bins of [lo, hi): [below, bins..., above]."""
    n = int(map_.numel()) if _is_torch(map_) else int(np.size(map_))
    if _is_torch(map_):
        import torch
        map_ = map_.contiguous()
        out = torch.zeros(nbins + 2, dtype=torch.int64, device=map_.device)      # same bits as uint64
    else:
        map_ = np.ascontiguousarray(map_, dtype=np.float64)
        out = np.zeros(nbins + 2, dtype=np.uint64)
    kind = _same_kind(map_, out)
    _check(lib().mlens_map_histogram(_ptr(map_)[0], C.c_int64(n), C.c_double(mu_ref), C.c_double(lo), C.c_double(hi),
                                     C.c_int32(nbins), _ptr(out)[0], C.c_int32(kind), _stream(stream)))
    return out



HIST_STATIC_MAXBINS = 4096


def histogram_static(map_, mu_ref, lo, hi, nbins, out, stream=None):
    """mlens_map_histogram_static: histogram() for callers that cannot let the library allocate device memory (a
    process whose own memory manager holds the whole GPU, or a path where an allocation's stall or failure is not
    acceptable).  The bin edges go into a fixed 32 KB table inside the library instead of a pool allocation, so:
    nbins <= HIST_STATIC_MAXBINS; `map_` and `out` are contiguous torch CUDA tensors the caller made beforehand (`out`:
    nbins + 2 int64, overwritten with [below, bins..., above]); nothing here allocates, not even the result.  Calls share
    the table: keep them on one stream or otherwise from overlapping.  The first call on a device does a one-time
    set-up and belongs before any stream capture.  Returns `out`."""
    if not (_is_torch(map_) and _is_torch(out)):
        raise MlensError("histogram_static takes torch CUDA tensors only (host arrays would need a staging allocation)")
    if not map_.is_contiguous() or int(out.numel()) != nbins + 2 or out.element_size() != 8:
        raise MlensError("histogram_static: map_ must be contiguous and out must hold nbins + 2 64-bit integers")
    _check(lib().mlens_map_histogram_static(_ptr(map_)[0], C.c_int64(int(map_.numel())), C.c_double(mu_ref), C.c_double(lo),
                                            C.c_double(hi), C.c_int32(nbins), _ptr(out)[0], _stream(stream)))
    return out
