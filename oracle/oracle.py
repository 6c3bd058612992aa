"""ctypes binding of the CPU oracle (mlens_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only; all arithmetic is in the C file.  `build()` compiles
liboracle.so with gcc (-ffp-contract=off so that "one multiply, one add" stays that).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mlens_oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")
_lib = None

_dp = C.POINTER(C.c_double)


class Field(C.Structure):
    """orc_field: lens parameters + star arrays (numpy arrays are kept alive on the object)."""
    _fields_ = [("kappa_tot", C.c_double), ("kappa_star", C.c_double), ("gamma", C.c_double),
                ("theta_star", C.c_double), ("shape", C.c_int32), ("pad_", C.c_int32),
                ("R", C.c_double), ("c1", C.c_double), ("c2", C.c_double),
                ("n_stars", C.c_int64), ("x", _dp), ("y", _dp), ("m", _dp),
                ("t111", C.c_double), ("t112", C.c_double), ("t122", C.c_double), ("t222", C.c_double)]

    @classmethod
    def make(cls, kappa_tot, kappa_star, gamma, x, y, m, *, shape=0, R=0.0, c1=0.0, c2=0.0,
             theta_star=1.0, macro_quad=(0.0, 0.0, 0.0, 0.0)):
        f = cls()
        f.t111, f.t112, f.t122, f.t222 = macro_quad      # reading G23: third derivatives of the macro potential at 0
        f.kappa_tot, f.kappa_star, f.gamma, f.theta_star = kappa_tot, kappa_star, gamma, theta_star
        f.shape, f.R, f.c1, f.c2 = shape, R, c1, c2
        f._x = np.ascontiguousarray(x, dtype=np.float64)
        f._y = np.ascontiguousarray(y, dtype=np.float64)
        f._m = np.ascontiguousarray(m, dtype=np.float64)
        assert f._x.shape == f._y.shape == f._m.shape and f._x.ndim == 1
        f.n_stars = f._x.size
        f.x, f.y, f.m = (a.ctypes.data_as(_dp) for a in (f._x, f._y, f._m))
        return f


class Geometry(C.Structure):
    """orc_geom: inputs (first block) and outputs of orc_geometry."""
    _fields_ = [("kappa_tot", C.c_double), ("kappa_star", C.c_double), ("gamma", C.c_double),
                ("theta_star", C.c_double), ("m2_over_m", C.c_double),
                ("Y1", C.c_double), ("Y2", C.c_double), ("dY1", C.c_double), ("dY2", C.c_double),
                ("npix1", C.c_int32), ("npix2", C.c_int32), ("k", C.c_double),
                ("border_mode", C.c_int32), ("pad_", C.c_int32),
                ("border_param", C.c_double), ("He1", C.c_double), ("He2", C.c_double),
                ("X1", C.c_double), ("X2", C.c_double), ("H1", C.c_double), ("H2", C.c_double),
                ("h1", C.c_double), ("h2", C.c_double), ("p1", C.c_double), ("p2", C.c_double),
                ("x0_1", C.c_double), ("x0_2", C.c_double), ("ylo1", C.c_double), ("ylo2", C.c_double),
                ("n1", C.c_int64), ("n2", C.c_int64), ("weight", C.c_double)]


def build(force=False):
    """Compile liboracle.so if missing or older than its source."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= os.path.getmtime(_SRC)):
        return _SO
    cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-o", _SO, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        fp, gp = C.POINTER(Field), C.POINTER(Geometry)
        i64, i32, dbl, u64 = C.c_int64, C.c_int32, C.c_double, C.c_uint64
        L.orc_num_threads.restype = C.c_int
        L.orc_alpha_star.argtypes = [fp, i64, _dp, _dp, _dp, _dp]
        L.orc_alpha_smooth.argtypes = [fp, i64, _dp, _dp, _dp, _dp]
        L.orc_lens_map.argtypes = [fp, i64, _dp, _dp, _dp, _dp]
        L.orc_geometry.argtypes = [gp]
        L.orc_geometry.restype = C.c_int
        L.orc_triangle_pixel_area.argtypes = [_dp, dbl, dbl]
        L.orc_triangle_pixel_area.restype = dbl
        L.orc_deposit_ipm.argtypes = [_dp, _dp, i64, i64, dbl, dbl, dbl, dbl, i32, i32, dbl, _dp]
        L.orc_bin_irs.argtypes = [_dp, _dp, i64, dbl, dbl, dbl, dbl, i32, i32, C.POINTER(u64)]
        L.orc_map_corners.argtypes = [fp, gp, i64, i64, i64, i64, _dp, _dp]
        L.orc_map_centres.argtypes = [fp, gp, i64, i64, i64, i64, _dp, _dp]
        L.orc_shoot.argtypes = [fp, gp, i64, i64, i64, i64, C.c_int, _dp, C.POINTER(u64)]
        L.orc_shoot.restype = C.c_int
        L.orc_rng_draw.argtypes = [u64, u64]
        L.orc_rng_draw.restype = u64
        L.orc_starfield.argtypes = [u64, i64, C.c_int, dbl, dbl, C.c_int, dbl, dbl, dbl, _dp, _dp, _dp]
        L.orc_multipole_def.argtypes = [i64, _dp, _dp, _dp, dbl, dbl, dbl, C.c_int, _dp]
        L.orc_local_def.argtypes = [i64, _dp, _dp, _dp, dbl, dbl, dbl, C.c_int, _dp]
        L.orc_local_eval.argtypes = [_dp, C.c_int, dbl, dbl, dbl, dbl, dbl, dbl, _dp, _dp]
        for name in ("orc_alpha_star", "orc_alpha_smooth", "orc_lens_map", "orc_deposit_ipm",
                     "orc_bin_irs", "orc_map_corners", "orc_map_centres", "orc_starfield",
                     "orc_multipole_def", "orc_local_def", "orc_local_eval"):
            getattr(L, name).restype = None
        _lib = L
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(_dp)


def num_threads():
    return int(lib().orc_num_threads())


def _pointwise(fn, f, zx, zy):
    zx, zy = _d(zx).ravel(), _d(zy).ravel()
    ox, oy = np.empty_like(zx), np.empty_like(zy)
    fn(C.byref(f), zx.size, _p(zx), _p(zy), _p(ox), _p(oy))
    return ox, oy


def alpha_star(f, zx, zy):
    """eq 13 summed over ALL stars (long double accumulation)."""
    return _pointwise(lib().orc_alpha_star, f, zx, zy)


def alpha_smooth(f, zx, zy):
    """eq 19 (disc) or eq B7 (rectangle)."""
    return _pointwise(lib().orc_alpha_smooth, f, zx, zy)


def lens_map(f, zx, zy):
    """eq 12."""
    return _pointwise(lib().orc_lens_map, f, zx, zy)


def geometry(kappa_tot, kappa_star, gamma, half_y, npix, k, border_mode, border_param=0.0, *,
             m2_over_m=1.0, theta_star=1.0, Y=(0.0, 0.0), He=(0.0, 0.0)):
    g = Geometry()
    g.kappa_tot, g.kappa_star, g.gamma, g.theta_star = kappa_tot, kappa_star, gamma, theta_star
    g.m2_over_m = m2_over_m
    g.Y1, g.Y2 = Y
    hy = half_y if isinstance(half_y, (tuple, list)) else (half_y, half_y)
    npx = npix if isinstance(npix, (tuple, list)) else (npix, npix)
    g.dY1, g.dY2 = hy
    g.npix1, g.npix2 = npx
    g.k = k
    g.border_mode, g.border_param = border_mode, border_param
    g.He1, g.He2 = He
    rc = lib().orc_geometry(C.byref(g))
    if rc != 0:
        raise ValueError("orc_geometry: invalid parameters")
    return g


def map_corners(f, g, i0, i1, j0, j1):
    """Mapped corners of cells [i0,i1)x[j0,j1): arrays of shape (j1-j0+1, i1-i0+1)."""
    shp = (j1 - j0 + 1, i1 - i0 + 1)
    wx, wy = np.empty(shp), np.empty(shp)
    lib().orc_map_corners(C.byref(f), C.byref(g), i0, i1, j0, j1, _p(wx), _p(wy))
    return wx, wy


def map_centres(f, g, i0, i1, j0, j1):
    shp = (j1 - j0, i1 - i0)
    wx, wy = np.empty(shp), np.empty(shp)
    lib().orc_map_centres(C.byref(f), C.byref(g), i0, i1, j0, j1, _p(wx), _p(wy))
    return wx, wy


def deposit_ipm(wx, wy, g, out=None):
    """Brute-force IPM deposit of a 2-D array of mapped corners (row = x2 index)."""
    wx, wy = _d(wx), _d(wy)
    nc2, nc1 = wx.shape
    if out is None:
        out = np.zeros((g.npix2, g.npix1))
    lib().orc_deposit_ipm(_p(wx), _p(wy), nc1, nc2, g.ylo1, g.ylo2, g.p1, g.p2,
                          g.npix1, g.npix2, g.weight, _p(out))
    return out


def bin_irs(wx, wy, g, out=None):
    wx, wy = _d(wx).ravel(), _d(wy).ravel()
    if out is None:
        out = np.zeros((g.npix2, g.npix1), dtype=np.uint64)
    lib().orc_bin_irs(_p(wx), _p(wy), wx.size, g.ylo1, g.ylo2, g.p1, g.p2, g.npix1, g.npix2,
                      out.ctypes.data_as(C.POINTER(C.c_uint64)))
    return out


def shoot(f, g, mode=0, sub=None, out=None):
    """Whole path on a cell sub-range (default all): mode 0 IPM -> float64 map, 1 IRS -> uint64 counts."""
    i0, i1, j0, j1 = sub if sub is not None else (0, g.n1, 0, g.n2)
    if mode == 0:
        if out is None:
            out = np.zeros((g.npix2, g.npix1))
        rc = lib().orc_shoot(C.byref(f), C.byref(g), i0, i1, j0, j1, 0, _p(out), None)
    else:
        if out is None:
            out = np.zeros((g.npix2, g.npix1), dtype=np.uint64)
        rc = lib().orc_shoot(C.byref(f), C.byref(g), i0, i1, j0, j1, 1, None,
                             out.ctypes.data_as(C.POINTER(C.c_uint64)))
    if rc != 0:
        raise ValueError(f"orc_shoot failed ({rc})")
    return out


def triangle_pixel_area(tri, px, py):
    t = _d(tri).ravel()
    assert t.size == 6
    return float(lib().orc_triangle_pixel_area(_p(t), float(px), float(py)))


def rng_draw(seed, n):
    return int(lib().orc_rng_draw(seed, n))


def starfield(seed, n, *, shape=0, a1=1.0, a2=0.0, mass_law=0, a=2.35, lo=0.08, hi=1.0):
    x, y, m = np.empty(n), np.empty(n), np.empty(n)
    lib().orc_starfield(seed, n, shape, a1, a2, mass_law, a, lo, hi, _p(x), _p(y), _p(m))
    return x, y, m


def multipole_def(x, y, m, cx, cy, L, p):
    x, y, m = _d(x), _d(y), _d(m)
    out = np.empty(2 * (p + 1))
    lib().orc_multipole_def(x.size, _p(x), _p(y), _p(m), cx, cy, L, p, _p(out))
    return out[0::2] + 1j * out[1::2]


def local_def(x, y, m, cx, cy, L, p):
    x, y, m = _d(x), _d(y), _d(m)
    out = np.empty(2 * (p + 1))
    lib().orc_local_def(x.size, _p(x), _p(y), _p(m), cx, cy, L, p, _p(out))
    return out[0::2] + 1j * out[1::2]


def local_eval(coef, cx, cy, L, zx, zy, theta=1.0):
    c = np.asarray(coef, dtype=np.complex128)
    p = c.size - 1
    buf = np.empty(2 * (p + 1))
    buf[0::2], buf[1::2] = c.real, c.imag
    ax, ay = C.c_double(), C.c_double()
    lib().orc_local_eval(_p(buf), p, cx, cy, L, theta, zx, zy, C.byref(ax), C.byref(ay))
    return ax.value, ay.value


def light_curve(map_, ylo1, ylo2, p1, p2, ya, yb, n, mode=0):
    m = _d(map_)
    npix2, npix1 = m.shape
    out = np.empty(n)
    lib().orc_light_curve(_p(m), C.c_int32(npix1), C.c_int32(npix2), C.c_double(ylo1), C.c_double(ylo2), C.c_double(p1),
                          C.c_double(p2), C.c_double(ya[0]), C.c_double(ya[1]), C.c_double(yb[0]), C.c_double(yb[1]),
                          C.c_int64(n), C.c_int32(mode), _p(out))
    return out


def histogram(map_, mu_ref, lo, hi, nbins):
    m = _d(map_).ravel()
    out = np.zeros(nbins + 2, dtype=np.uint64)
    lib().orc_histogram(_p(m), C.c_int64(m.size), C.c_double(mu_ref), C.c_double(lo), C.c_double(hi), C.c_int32(nbins),
                        out.ctypes.data_as(C.POINTER(C.c_uint64)))
    return out

