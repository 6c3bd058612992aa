// shoot.cu -- the two hot loops of the method, fused: evaluate the lens equation on a tile of the ray
// grid (eq 12/23/24) and deposit the mapped cells into the source-plane map without ever writing the
// rays to HBM.
//   IPM: cell -> 2 triangles -> exact area apportioning over the pixel grid.
//   IRS:     one ray per cell centre -> count.
//
// Evaluation.  Targets outnumber sources by 10^4..10^5, so the FMM hierarchy is continued
// on the target side: for every 32x32-ray tile the leaf's local series is shifted to the tile centre
// (eq C7 once more) and the leaf's near-field stars that are far from the tile on the tile's scale are
// added to it directly (eq C6); what is left per ray is a ~13-term Horner sum plus the few stars within
// 10 tile radii.  Both truncations are bounded per tile from the coefficients themselves; a tile whose
// bound fails evaluates the leaf's full series and full star list instead.
//
// Accumulation is integer: the map is a u64 array in units of 2^-FIXBITS of one whole triangle (IPM) or of
// one ray (IRS); integer adds commute, so maps are bit-reproducible whatever the atomic order.  Interior
// runs of large triangles are written as +c/-c into a row-difference array that finalise prefix-sums
// (exact in modular integer arithmetic), so a triangle costs its perimeter, not its area.
#include "device.cuh"
#include <math.h>
#include <stdlib.h>

namespace ml {

static const int TCX = 32;            // rays per tile row (= warp width)
static const int TCY = 32;            // ray rows per tile
static const int NWARP = 8;           // 256 threads
static const int RPT = TCY / NWARP;   // rays per thread
static const int WW = 32, WH = 32;    // shared-memory pixel window of a tile
static const int FIXBITS = 36;
static const int TQMAX = 20;          // highest order of the tile series
static const int SMALL_MAX = 16;      // triangles whose clipped bounding box has <= this many pixels stay in-thread
static const int CHUNK_ROWS = 64;     // pixel rows per queue entry
static const int QENT = 8;            // doubles per queue entry

enum { C_QUEUE = 0, C_TILE, C_SINGLE, C_SMALL, C_QUEUED, C_CHUNKS, C_OVERFLOW, C_FALLBACK, C_RAYS, C_NEAR,
       C_PX_SMALL, C_PX_INT, C_PX_EDGE, C_ROWS, C_TILES_FULL, C_NCOUNTERS };

struct ShootDev {
    LensDev L;
    double x0_1, x0_2, h1, h2;
    long long i0, i1, j0, j1;          // cell sub-range
    double ylo1, ylo2, p1, p2, inv_p1, inv_p2;
    int npix1, npix2;
    unsigned long long *acc, *diff;
    double *queue;
    unsigned long long *counters;
    long long queue_cap;
    double *dump1, *dump2;
    const double *binom;               // Pascal triangle, stride BN
    int eval_mode;
    int ntx;                           // tiles along x1
    long long tile_row0, tile_rows;    // band of tile rows handled by this launch
    int tq;                            // order of the tile series
    double eps_far, eps_star;          // truncation budgets of the tile series (absolute, units of theta)
};
static const int BN = 2 * ML_P1MAX;

__device__ __forceinline__ double corner_x(const ShootDev &S, long long i) { return __dadd_rn(S.x0_1, __dmul_rn((double)i, S.h1)); }
__device__ __forceinline__ double corner_y(const ShootDev &S, long long j) { return __dadd_rn(S.x0_2, __dmul_rn((double)j, S.h2)); }

__device__ __forceinline__ int floor_to_int(double u) {
    return (int)floor(fmin(fmax(u, -1.0e9), 1.0e9));      // NaN -> -1e9
}
// pixel coordinates packed as two int16 (values beyond the map on one side collapse: such triangles are outside)
__device__ __forceinline__ int pack_px(double u, double v) {
    int a = (int)floor(fmin(fmax(u, -30000.0), 30000.0)), b = (int)floor(fmin(fmax(v, -30000.0), 30000.0));
    if (u != u) a = -30000;
    if (v != v) b = -30000;
    return (b << 16) | (a & 0xffff);
}
__device__ __forceinline__ int px_of(int pk) { return (int)(short)(pk & 0xffff); }
__device__ __forceinline__ int py_of(int pk) { return pk >> 16; }

// 1/a to double precision from the 20-bit hardware seed: one cubic step, e^3 ~ 2^-60 (a normal, finite, > 0)
__device__ __forceinline__ double fast_rcp(double a) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double e = fma(-a, y, 1.0);
    double t = fma(e, e, e);
    return fma(y, t, y);
}

// ------------------------------------------------------------------------------------------------
// Exact area of (triangle  intersect  unit pixel) by Green's theorem: area = closed integral of
// clamp(x,0,1) over the part of the boundary with y in [0,1].  Same value as Sutherland-Hodgman
// clipping + shoelace up to rounding; no polygon arrays, no data-dependent vertex counts.
struct TriEdges {
    double px[3], py[3], dx[3], dy[3], idx[3], idy[3];
};

__device__ __forceinline__ void tri_setup(TriEdges &E, double x0, double y0, double x1, double y1, double x2, double y2) {
    E.px[0] = x0; E.py[0] = y0; E.dx[0] = x1 - x0; E.dy[0] = y1 - y0;
    E.px[1] = x1; E.py[1] = y1; E.dx[1] = x2 - x1; E.dy[1] = y2 - y1;
    E.px[2] = x2; E.py[2] = y2; E.dx[2] = x0 - x2; E.dy[2] = y0 - y2;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        E.idx[e] = (E.dx[e] != 0.0) ? 1.0 / E.dx[e] : 0.0;
        E.idy[e] = (E.dy[e] != 0.0) ? 1.0 / E.dy[e] : 0.0;
    }
}

__device__ __forceinline__ double clamp01(double v) { return fmin(fmax(v, 0.0), 1.0); }

__device__ __forceinline__ double tri_pixel_area(const TriEdges &E, double qx, double qy) {
    double s = 0.0;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        double dy = E.dy[e];
        if (dy == 0.0) continue;
        double px = E.px[e] - qx, py = E.py[e] - qy, dx = E.dx[e];
        double ta = -py * E.idy[e], tb = (1.0 - py) * E.idy[e];
        double t0 = fmax(0.0, fmin(ta, tb)), t1 = fmin(1.0, fmax(ta, tb));
        if (!(t1 > t0)) continue;
        double integ;
        if (dx == 0.0) {
            integ = (t1 - t0) * clamp01(px);
        } else {
            double sa = -px * E.idx[e], sb = (1.0 - px) * E.idx[e];
            double ua = fmax(t0, fmin(sa, sb)), ub = fmin(t1, fmax(sa, sb));
            double mid = (ub > ua) ? (ub - ua) * clamp01(fma(0.5 * (ua + ub), dx, px)) : 0.0;
            double over = (dx > 0.0) ? fmax(0.0, t1 - fmax(sb, t0)) : fmax(0.0, fmin(sb, t1) - t0);
            integ = mid + over;
        }
        s = fma(dy, integ, s);
    }
    return s;
}

// Fraction of a triangle's area on the side  coordinate < a  of an axis-parallel line, c0..c2 the vertex
// coordinates along that axis: the lone vertex cuts off a similar corner, ratio t1 t2 of its two edges.
__device__ __forceinline__ double frac_below(double c0, double c1, double c2, double a) {
    double d0 = c0 - a, d1 = c1 - a, d2 = c2 - a;
    bool n0 = d0 < 0.0, n1 = d1 < 0.0, n2 = d2 < 0.0;
    int cnt = (int)n0 + (int)n1 + (int)n2;
    if (cnt == 0) return 0.0;
    if (cnt == 3) return 1.0;
    bool lone_neg = (cnt == 1);
    double l, o1, o2;
    if (n0 == lone_neg) { l = d0; o1 = d1; o2 = d2; }
    else if (n1 == lone_neg) { l = d1; o1 = d0; o2 = d2; }
    else { l = d2; o1 = d0; o2 = d1; }
    double f = (l * l) / ((l - o1) * (l - o2));
    return lone_neg ? f : 1.0 - f;
}

// Area of  unit pixel  intersect  half-plane {f0 + gx s + gy t >= 0}, (s,t) in [0,1]^2.
__device__ __forceinline__ double halfplane_pixel_area(double f0, double gx, double gy) {
    double a = fabs(gx), b = fabs(gy);
    double v = f0 + fmax(gx, 0.0) + fmax(gy, 0.0);           // value at the innermost corner
    if (!(v > 0.0)) return 0.0;
    double lo = fmin(a, b), hi = fmax(a, b);
    if (lo <= 1e-9 * hi) return (hi > 0.0) ? fmin(v / hi, 1.0) : 1.0;
    double p0 = v * v;
    double va = fmax(v - a, 0.0), vb = fmax(v - b, 0.0), vab = fmax(v - a - b, 0.0);
    double s = (p0 - va * va) - (vb * vb - vab * vab);
    return fmin(s / (2.0 * a * b), 1.0);
}

struct Window {                       // the tile's privatised piece of the map
    unsigned long long *win;
    int ax, ay;
};

__device__ __forceinline__ void deposit_fix(const ShootDev &S, const Window &W, int px, int py, unsigned long long v) {
    if (v == 0ull) return;
    int lx = px - W.ax, ly = py - W.ay;
    if (W.win && lx >= 0 && lx < WW && ly >= 0 && ly < WH) atomicAdd(&W.win[ly * WW + lx], v);
    else atomicAdd(&S.acc[(size_t)py * S.npix1 + px], v);
}
__device__ __forceinline__ unsigned long long to_fix(double frac) {
    long long v = __double2ll_rn(frac * (double)(1ull << FIXBITS));
    return v > 0 ? (unsigned long long)v : 0ull;
}
__device__ __forceinline__ void deposit_frac(const ShootDev &S, const Window &W, int px, int py, double frac) {
    if (px < 0 || px >= S.npix1 || py < 0 || py >= S.npix2) return;
    deposit_fix(S, W, px, py, to_fix(frac));
}

struct TriBox {
    double bx, by, A;
    int lox, hix, loy, hiy;           // bounding box clipped to the map
    int wu, hu;                       // unclipped bounding box size in pixels (saturated)
    double x[3], y[3];                // local coordinates (relative to bx, by)
};

// returns 0: nothing to deposit, 1: degenerate handled, 2: box ready
__device__ __forceinline__ int tri_prepare(const ShootDev &S, const Window &W, double u0, double v0, double u1, double v1,
                                           double u2, double v2, TriBox &B) {
    double mnx = fmin(u0, fmin(u1, u2)), mxx = fmax(u0, fmax(u1, u2));
    double mny = fmin(v0, fmin(v1, v2)), mxy = fmax(v0, fmax(v1, v2));
    if (!(mxx >= 0.0) || !(mxy >= 0.0) || !(mnx < (double)S.npix1) || !(mny < (double)S.npix2)) return 0;
    if (!(mnx > -1.0e15) || !(mny > -1.0e15) || !(mxx < 1.0e15) || !(mxy < 1.0e15)) return 0;   // inf / absurd
    if (u0 != u0 || u1 != u1 || u2 != u2 || v0 != v0 || v1 != v1 || v2 != v2) return 0;
    B.bx = floor(mnx); B.by = floor(mny);
    B.x[0] = u0 - B.bx; B.y[0] = v0 - B.by; B.x[1] = u1 - B.bx; B.y[1] = v1 - B.by; B.x[2] = u2 - B.bx; B.y[2] = v2 - B.by;
    B.A = 0.5 * ((B.x[1] - B.x[0]) * (B.y[2] - B.y[0]) - (B.x[2] - B.x[0]) * (B.y[1] - B.y[0]));
    if (B.A == 0.0) {                                   // reading G12: whole weight to the pixel of vertex 0
        deposit_frac(S, W, floor_to_int(u0), floor_to_int(v0), 1.0);
        return 1;
    }
    double ex = floor(mxx), ey = floor(mxy);
    B.lox = (int)fmax(B.bx, 0.0); B.hix = (int)fmin(ex, (double)S.npix1 - 1.0);
    B.loy = (int)fmax(B.by, 0.0); B.hiy = (int)fmin(ey, (double)S.npix2 - 1.0);
    B.wu = (int)fmin(ex - B.bx + 1.0, 1.0e6); B.hu = (int)fmin(ey - B.by + 1.0, 1.0e6);
    return 2;
}

struct ThreadCounters { unsigned int single = 0, small_ = 0, queued = 0, chunks = 0, overflow = 0, fallback = 0, rays = 0, near_ = 0, px_small = 0; };

// every pixel of the clipped bounding box, one by one
__device__ __noinline__ void tri_deposit_loop(const ShootDev &S, const Window &W, const TriBox &B, ThreadCounters &tc) {
    TriEdges E;
    tri_setup(E, B.x[0], B.y[0], B.x[1], B.y[1], B.x[2], B.y[2]);
    double invA = 1.0 / B.A;
    for (int py = B.loy; py <= B.hiy; ++py)
        for (int px = B.lox; px <= B.hix; ++px) {
            double a = tri_pixel_area(E, (double)px - B.bx, (double)py - B.by);
            deposit_fix(S, W, px, py, to_fix(a * invA));
            ++tc.px_small;
        }
}

// A triangle that is not wholly inside one pixel.  Strips (one pixel row or column) are apportioned by
// differences of frac_below at the pixel lines, 2x2 boxes by inclusion-exclusion around one clipped
// pixel, other small boxes pixel by pixel; anything larger goes to the cooperative queue.
__device__ __forceinline__ void deposit_general(const ShootDev &S, const Window &W, double u0, double v0, double u1, double v1,
                                                double u2, double v2, ThreadCounters &tc) {
    TriBox B;
    int st = tri_prepare(S, W, u0, v0, u1, v1, u2, v2, B);
    if (st != 2) { if (st == 1) ++tc.small_; return; }
    long long w = (long long)B.hix - B.lox + 1, h = (long long)B.hiy - B.loy + 1;
    if (w <= 0 || h <= 0) return;
    if (B.hu == 1 && w <= SMALL_MAX) {                            // one pixel row
        ++tc.small_;
        double prev = frac_below(B.x[0], B.x[1], B.x[2], (double)B.lox - B.bx);
        for (int px = B.lox; px <= B.hix; ++px) {
            double cur = frac_below(B.x[0], B.x[1], B.x[2], (double)(px + 1) - B.bx);
            deposit_fix(S, W, px, B.loy, to_fix(cur - prev));
            prev = cur; ++tc.px_small;
        }
        return;
    }
    if (B.wu == 1 && h <= SMALL_MAX) {                            // one pixel column
        ++tc.small_;
        double prev = frac_below(B.y[0], B.y[1], B.y[2], (double)B.loy - B.by);
        for (int py = B.loy; py <= B.hiy; ++py) {
            double cur = frac_below(B.y[0], B.y[1], B.y[2], (double)(py + 1) - B.by);
            deposit_fix(S, W, B.lox, py, to_fix(cur - prev));
            prev = cur; ++tc.px_small;
        }
        return;
    }
    if (B.wu == 2 && B.hu == 2) {                                 // four pixels around one grid corner
        ++tc.small_; tc.px_small += 4;
        TriEdges E;
        tri_setup(E, B.x[0], B.y[0], B.x[1], B.y[1], B.x[2], B.y[2]);
        double f00 = tri_pixel_area(E, 0.0, 0.0) / B.A;
        double fl = frac_below(B.x[0], B.x[1], B.x[2], 1.0), fb = frac_below(B.y[0], B.y[1], B.y[2], 1.0);
        int X = (int)B.bx, Y = (int)B.by;
        deposit_frac(S, W, X, Y, f00);
        deposit_frac(S, W, X + 1, Y, fb - f00);
        deposit_frac(S, W, X, Y + 1, fl - f00);
        deposit_frac(S, W, X + 1, Y + 1, 1.0 - fl - fb + f00);
        return;
    }
    if (w * h <= SMALL_MAX) { ++tc.small_; tri_deposit_loop(S, W, B, tc); return; }
    long long nch = (h + CHUNK_ROWS - 1) / CHUNK_ROWS;
    unsigned long long old = atomicAdd(&S.counters[C_QUEUE], (unsigned long long)nch);
    if ((long long)old + nch > S.queue_cap) {
        atomicAdd(&S.counters[C_QUEUE], (unsigned long long)(-nch));
        ++tc.overflow;
        tri_deposit_loop(S, W, B, tc);
        return;
    }
    ++tc.queued; tc.chunks += (unsigned int)nch;
    for (long long c = 0; c < nch; ++c) {
        double *q = S.queue + (size_t)(old + c) * QENT;
        int r0 = B.loy + (int)(c * CHUNK_ROWS), r1 = min(B.hiy + 1, r0 + CHUNK_ROWS);
        q[0] = u0; q[1] = v0; q[2] = u1; q[3] = v1; q[4] = u2; q[5] = v2;
        q[6] = __hiloint2double(r1, r0); q[7] = 0.0;
    }
}

__device__ __forceinline__ void flush_counters(const ShootDev &S, ThreadCounters &tc) {
    // order = the C_SINGLE.. block of the counter enum, then C_PX_SMALL
    unsigned int v[9] = {tc.single, tc.small_, tc.queued, tc.chunks, tc.overflow, tc.fallback, tc.rays, tc.near_, tc.px_small};
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        unsigned int x = v[k];
        for (int o = 16; o; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) == 0 && x) atomicAdd(&S.counters[C_SINGLE + k], (unsigned long long)x);
    }
}

// ------------------------------------------------------------------------------------------------
// Tile expansion.  A tile touches at most 2x2 leaves (one per extreme ray); each distinct leaf gets a
// slot.  Slot mode: 0 = tile series + direct stars, 1 = the leaf's full series and star list (bounds
// failed), -1 = unused.
struct TileExp {
    double2 t[4][TQMAX + 1];          // conj(alpha)(u) = sum_j t_j u^j, u = (z - z_t)/r_t, theta^2 included
    double sx[4][ML_NEAR], sy[4][ML_NEAR], sm[4][ML_NEAR];   // direct stars (absolute positions, m theta^2)
    uint32_t bx0[4], bx1[4], by0[4], by1[4];
    int leaf[4], nd[4], mode[4], node[4];
    int nslots;
    double zt_x, zt_y, inv_rt;
    // scratch of the set-up
    double2 e[ML_P1MAX];              // the leaf's derivative series
    double tail[ML_P1MAX];
    bool one_leaf;                    // all four extreme rays sit in the same leaf (then so does every ray)
};

__device__ __forceinline__ void tile_find(const ShootDev &S, TileExp &T, int slot, double x, double y) {
    uint32_t qx, qy;
    T.leaf[slot] = -1; T.nd[slot] = 0; T.mode[slot] = -1; T.node[slot] = -1;
    T.bx0[slot] = T.bx1[slot] = T.by0[slot] = T.by1[slot] = 0;
    if (!quantise(S.L, x, y, qx, qy)) return;
    int node = find_leaf_node(S.L, qx, qy);
    int lev = S.L.level[node], ix = S.L.ix[node], iy = S.L.iy[node];
    int sh = ML_QBITS - lev;
    T.leaf[slot] = S.L.leaf_id[node]; T.node[slot] = node;
    T.bx0[slot] = (uint32_t)ix << sh; T.bx1[slot] = (uint32_t)(ix + 1) << sh;
    T.by0[slot] = (uint32_t)iy << sh; T.by1[slot] = (uint32_t)(iy + 1) << sh;
}

// Builds slot `s` (block-wide; contains __syncthreads).  rt = tile radius.
// `fold` = (TQMAX+1) x ML_NEAR complex scratch: per-star terms of eq C6 about the tile centre.
__device__ void tile_build_slot(const ShootDev &S, TileExp &T, int s, double rt, double2 *fold) {
    const int tid = threadIdx.x;
    const int p = S.L.p, Q = S.tq;
    const int leaf = T.leaf[s], node = T.node[s];
    const int lev = S.L.level[node];
    const double half = S.L.root_half / (double)(1 << lev);
    const double cx = -S.L.root_half + (2.0 * S.L.ix[node] + 1.0) * half;
    const double cy = -S.L.root_half + (2.0 * S.L.iy[node] + 1.0) * half;
    const int cnt = S.L.near_cnt[leaf];
    if (tid < p) T.e[tid] = S.L.ecoef[(size_t)leaf * S.L.p1 + tid];
    __syncthreads();
    const double rho = rt / half;
    double2 Tj = make_double2(0.0, 0.0);
    if (tid < p) {
        // shift of the derivative series to the tile centre: T_j = rho^j sum_m e_{j+m} C(j+m, j) zeta_t^m   (eq C7)
        const int j = tid;
        const double zr = (T.zt_x - cx) / half, zi = (T.zt_y - cy) / half;
        double ar = 0.0, ai = 0.0;
        for (int m = p - 1 - j; m >= 0; --m) {
            double bc = __ldg(&S.binom[(size_t)(j + m) * BN + j]);
            double2 c = T.e[j + m];
            double tr = fma(ar, zr, fma(-ai, zi, bc * c.x));
            double ti = fma(ar, zi, fma(ai, zr, bc * c.y));
            ar = tr; ai = ti;
        }
        double sc = 1.0;
        for (int k = 0; k < j; ++k) sc *= rho;
        Tj = make_double2(ar * sc, ai * sc);
        T.tail[j] = (j > Q) ? (fabs(Tj.x) + fabs(Tj.y)) : 0.0;
    } else if (tid >= 64 && tid < 64 + ML_NEAR) {
        // near-field stars: those far from the tile on the tile's scale join the series (eq C6), the rest stay direct
        const int k = tid - 64;
        bool have = k < cnt, direct = false;
        double x = 0, y = 0, m = 0;
        double2 term = make_double2(0.0, 0.0), w = make_double2(0.0, 0.0);
        if (have) {
            size_t o = (size_t)leaf * ML_NEAR + k;
            x = S.L.near_x[o]; y = S.L.near_y[o]; m = S.L.near_m[o] * S.L.theta2;
            double dx = x - T.zt_x, dy = y - T.zt_y;
            double d2 = dx * dx + dy * dy, d = sqrt(d2);
            double r = (d > 0.0) ? rt / d : 2.0;
            direct = true;
            if (r < 0.5) {
                double rq = r;
                for (int k2 = 0; k2 < Q; ++k2) rq *= r;                  // r^(Q+1)
                double bound = (m / d) * rq / (1.0 - r);
                if (bound <= S.eps_star) {
                    direct = false;
                    // conj(alpha_i) = m/(eta - d) = -(m/d) sum_j (eta/d)^j ; with eta = rt u: term_j = -(m/d)(rt/d)^j
                    double id2 = 1.0 / d2;
                    term = make_double2(-m * dx * id2, m * dy * id2);     // -m/d = -m conj(d)/|d|^2
                    w = make_double2(rt * dx * id2, -rt * dy * id2);      // rt/d
                }
            }
        }
        for (int j = 0; j <= Q; ++j) {
            fold[j * ML_NEAR + k] = term;
            term = cmul(term, w);
        }
        unsigned dm = __ballot_sync(0xffffffffu, direct);
        if (direct) {
            int pos = __popc(dm & ((1u << k) - 1u));
            T.sx[s][pos] = x; T.sy[s][pos] = y; T.sm[s][pos] = m;
        }
        if (k == 0) T.nd[s] = __popc(dm);
    }
    __syncthreads();
    if (tid <= Q) {
        double ar = (tid < p) ? Tj.x : 0.0, ai = (tid < p) ? Tj.y : 0.0;
#pragma unroll 4
        for (int k = 0; k < ML_NEAR; ++k) { double2 f = fold[tid * ML_NEAR + k]; ar += f.x; ai += f.y; }
        T.t[s][tid] = make_double2(ar, ai);
    }
    if (tid == 32) {
        double tl = 0.0;
        for (int j = Q + 1; j < p; ++j) tl += T.tail[j];
        T.mode[s] = (tl <= S.eps_far) ? 0 : 1;
    }
    __syncthreads();
}

// Sets up the tile: centre, radius, leaves of the four extreme rays, one slot per distinct leaf.
// off = offset of the rays from the grid corners in cells (0 for IPM, 0.5 for IRS).
__device__ void tile_setup(const ShootDev &S, TileExp &T, long long ci0, long long cj0, long long ci1, long long cj1,
                           double off, unsigned long long *full_counter, double2 *fold) {
    const int tid = threadIdx.x;
    if (S.eval_mode != MLENS_EVAL_FMM) { if (tid == 0) { T.nslots = 0; T.inv_rt = 1.0; T.one_leaf = false; } __syncthreads(); return; }
    const double rt = 0.5 * sqrt((double)((TCX - 1) * (TCX - 1)) * S.h1 * S.h1 + (double)((TCY - 1) * (TCY - 1)) * S.h2 * S.h2) * (1.0 + 1e-9);
    if (tid < 4)
        tile_find(S, T, tid, corner_x(S, (tid & 1) ? ci1 : ci0) + off * S.h1, corner_y(S, (tid & 2) ? cj1 : cj0) + off * S.h2);
    if (tid == 0) {
        T.zt_x = corner_x(S, ci0) + (0.5 * (TCX - 1) + off) * S.h1;
        T.zt_y = corner_y(S, cj0) + (0.5 * (TCY - 1) + off) * S.h2;
        T.inv_rt = 1.0 / rt;
    }
    __syncthreads();
    if (tid == 0) {
        // drop duplicate leaves; a slot is built only for the first occurrence
        int n = 0;
        T.one_leaf = T.leaf[0] >= 0 && T.leaf[1] == T.leaf[0] && T.leaf[2] == T.leaf[0] && T.leaf[3] == T.leaf[0];
        for (int a = 0; a < 4; ++a) {
            if (T.leaf[a] < 0) continue;
            bool dup = false;
            for (int b = 0; b < a; ++b) dup = dup || (T.leaf[b] == T.leaf[a]);
            if (dup) T.leaf[a] = -1; else ++n;
        }
        T.nslots = n;
    }
    __syncthreads();
    for (int s = 0; s < 4; ++s) {
        if (T.leaf[s] < 0) continue;                              // block-uniform
        tile_build_slot(S, T, s, rt, fold);
        if (tid == 0 && T.mode[s] == 1 && full_counter) atomicAdd(full_counter, 1ull);
    }
}

// w(z) of eq 12 for the RPT rays of one thread (same column, rows warp + r NWARP).
__device__ __forceinline__ void eval_rays(const ShootDev &S, const TileExp &T, const double (&x)[RPT], const double (&y)[RPT],
                                          const double (&ux)[RPT], const double (&uy)[RPT], const bool (&valid)[RPT],
                                          double (&wx)[RPT], double (&wy)[RPT], ThreadCounters &tc) {
    double ax[RPT], ay[RPT];
    if (S.eval_mode == MLENS_EVAL_DIRECT) {
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            ax[r] = ay[r] = 0.0;
            if (valid[r]) { direct_all(S.L, x[r], y[r], ax[r], ay[r]); ax[r] *= S.L.theta2; ay[r] *= S.L.theta2; ++tc.rays; }
        }
    } else {
        int slot[RPT];
        bool uniform = true;                                   // all rays of this thread in one tile-series slot
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            slot[r] = -1;
            if (!valid[r]) continue;
            ++tc.rays;
            if (T.one_leaf) {
                slot[r] = 0;
            } else {
                uint32_t qx, qy;
                if (quantise(S.L, x[r], y[r], qx, qy)) {
#pragma unroll
                    for (int s = 0; s < 4; ++s)
                        if (T.leaf[s] >= 0 && qx >= T.bx0[s] && qx < T.bx1[s] && qy >= T.by0[s] && qy < T.by1[s]) slot[r] = s;
                }
            }
            if (slot[r] >= 0 && T.mode[slot[r]] != 0) slot[r] = -1;
        }
#pragma unroll
        for (int r = 1; r < RPT; ++r) uniform = uniform && (slot[r] == slot[0]);
        uniform = uniform && (slot[0] >= 0);
#pragma unroll
        for (int r = 0; r < RPT; ++r) uniform = uniform && valid[r];
        if (uniform) {
            // the common case: RPT independent Horner chains share every coefficient load
            const int s = slot[0], Q = S.tq;
            const double2 *t = T.t[s];
            double sr[RPT], si[RPT];
            double2 c = t[Q];
#pragma unroll
            for (int r = 0; r < RPT; ++r) { sr[r] = c.x; si[r] = c.y; }
            for (int j = Q - 1; j >= 0; --j) {
                c = t[j];
#pragma unroll
                for (int r = 0; r < RPT; ++r) {
                    double tr = fma(sr[r], ux[r], fma(-si[r], uy[r], c.x));
                    double ti = fma(sr[r], uy[r], fma(si[r], ux[r], c.y));
                    sr[r] = tr; si[r] = ti;
                }
            }
            const int nd = T.nd[s];
            tc.near_ += (unsigned int)(nd * RPT);
            for (int k = 0; k < nd; ++k) {
                double X = T.sx[s][k], Y = T.sy[s][k], M = T.sm[s][k];
#pragma unroll
                for (int r = 0; r < RPT; ++r) {
                    double dx = x[r] - X, dy = y[r] - Y;
                    double r2 = fma(dx, dx, dy * dy);
                    double q = (__double2hiint(r2) >= 0x00100000) ? M * fast_rcp(r2) : 0.0;   // reading G11: skip r = 0
                    sr[r] = fma(q, dx, sr[r]);
                    si[r] = fma(-q, dy, si[r]);
                }
            }
#pragma unroll
            for (int r = 0; r < RPT; ++r) { ax[r] = sr[r]; ay[r] = -si[r]; }
        } else {
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                ax[r] = ay[r] = 0.0;
                if (!valid[r]) continue;
                const int s = slot[r];
                if (s >= 0) {
                    const int Q = S.tq;
                    double sr = T.t[s][Q].x, si = T.t[s][Q].y;
                    for (int j = Q - 1; j >= 0; --j) {
                        double2 c = T.t[s][j];
                        double tr = fma(sr, ux[r], fma(-si, uy[r], c.x));
                        double ti = fma(sr, uy[r], fma(si, ux[r], c.y));
                        sr = tr; si = ti;
                    }
                    const int nd = T.nd[s];
                    tc.near_ += (unsigned int)nd;
                    for (int k = 0; k < nd; ++k) {
                        double dx = x[r] - T.sx[s][k], dy = y[r] - T.sy[s][k];
                        double r2 = fma(dx, dx, dy * dy);
                        double q = (__double2hiint(r2) >= 0x00100000) ? T.sm[s][k] * fast_rcp(r2) : 0.0;
                        sr = fma(q, dx, sr);
                        si = fma(-q, dy, si);
                    }
                    ax[r] = sr; ay[r] = -si;
                } else {
                    ++tc.fallback;
                    alpha_fmm_global(S.L, x[r], y[r], ax[r], ay[r]);
                }
            }
        }
    }
#pragma unroll
    for (int r = 0; r < RPT; ++r)
        if (valid[r]) lens_w(S.L, x[r], y[r], ax[r], ay[r], wx[r], wy[r]);
        else { wx[r] = 0.0; wy[r] = 0.0; }
}

// Adds `cnt` to the run of equal keys among consecutive lanes with one shared-memory atomic per run.
__device__ __forceinline__ void window_add_rle(unsigned long long *win, int key, unsigned long long cnt) {
    const unsigned full = 0xffffffffu;
    int lane = threadIdx.x & 31;
    int prev = __shfl_up_sync(full, key, 1);
    bool head = (lane == 0) || (key != prev);
    unsigned heads = __ballot_sync(full, head);
    if (head && key >= 0) {
        unsigned above = (lane == 31) ? 0u : (heads & ~((2u << lane) - 1u));
        int next = above ? (__ffs(above) - 1) : 32;
        atomicAdd(&win[key], cnt * (unsigned long long)(next - lane));
    }
}

// next tile of the band, handed out dynamically (heavy tiles sit near stars)
__device__ __forceinline__ long long next_tile(const ShootDev &S, long long *slot) {
    __syncthreads();
    if (threadIdx.x == 0) *slot = (long long)atomicAdd(&S.counters[C_TILE], 1ull);
    __syncthreads();
    return *slot;
}

__global__ void __launch_bounds__(NWARP * 32) shoot_ipm_kernel(ShootDev S) {
    __shared__ double suv[2 * TCY * TCX];                 // mapped corners in pixel units; set-up scratch before that
    __shared__ int spk[TCY * TCX];
    double *const su = suv, *const sv = suv + TCY * TCX;
    static_assert((TQMAX + 1) * ML_NEAR * sizeof(double2) <= sizeof(suv), "fold scratch must fit");
    __shared__ TileExp T;
    __shared__ unsigned long long win[WH * WW];
    __shared__ unsigned short list[2 * (TCX - 1) * (TCY - 1)];
    __shared__ int list_n;
    __shared__ long long tile_slot;
    __shared__ Window W;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ThreadCounters tc;
    const long long ntiles = (long long)S.ntx * S.tile_rows;
    const long long ncx = S.i1 - S.i0 + 1;               // corners per dump row

    for (long long tile = next_tile(S, &tile_slot); tile < ntiles; tile = next_tile(S, &tile_slot)) {
        long long ty = S.tile_row0 + tile / S.ntx;
        int tx = (int)(tile % S.ntx);
        long long ci0 = S.i0 + (long long)tx * (TCX - 1), cj0 = S.j0 + ty * (TCY - 1);
        long long ci1 = min(ci0 + TCX - 1, S.i1), cj1 = min(cj0 + TCY - 1, S.j1);   // last corner of the tile

        if (threadIdx.x == 0) list_n = 0;
        for (int k = threadIdx.x; k < WH * WW; k += blockDim.x) win[k] = 0ull;
        tile_setup(S, T, ci0, cj0, ci1, cj1, 0.0, &S.counters[C_TILES_FULL], (double2 *)suv);

        // ---- hot loop A: map the corners (eq 12)
        {
            double x[RPT], y[RPT], ux[RPT], uy[RPT], wx[RPT], wy[RPT];
            bool valid[RPT];
            const long long ci = ci0 + lane;
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const int row = warp + r * NWARP;
                const long long cj = cj0 + row;
                valid[r] = (ci <= S.i1) && (cj <= S.j1);
                x[r] = corner_x(S, ci); y[r] = corner_y(S, cj);
                ux[r] = ((double)lane - 0.5 * (TCX - 1)) * S.h1 * T.inv_rt;
                uy[r] = ((double)row - 0.5 * (TCY - 1)) * S.h2 * T.inv_rt;
            }
            eval_rays(S, T, x, y, ux, uy, valid, wx, wy, tc);
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const int row = warp + r * NWARP;
                const int o = row * TCX + lane;
                if (valid[r]) {
                    if (S.dump1) {
                        size_t d = (size_t)(cj0 + row - S.j0) * ncx + (size_t)(ci - S.i0);
                        S.dump1[d] = wx[r]; S.dump2[d] = wy[r];
                    }
                    double u = (wx[r] - S.ylo1) * S.inv_p1, v = (wy[r] - S.ylo2) * S.inv_p2;
                    su[o] = u; sv[o] = v; spk[o] = pack_px(u, v);
                } else {
                    su[o] = 0.0; sv[o] = 0.0; spk[o] = 0;
                }
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int rc = (int)min((long long)(TCY / 2), cj1 - cj0), cc = (int)min((long long)(TCX / 2), ci1 - ci0);
            int pk = spk[rc * TCX + cc];
            W.win = win; W.ax = px_of(pk) - WW / 2; W.ay = py_of(pk) - WH / 2;
        }
        __syncthreads();
        const Window Wl = W;

        // ---- hot loop B, part 1: cells whose triangles sit inside one pixel are just counted
        for (int row = warp; row < TCY - 1; row += NWARP) {
            long long ci = ci0 + lane, cj = cj0 + row;
            bool valid = (lane < TCX - 1) && (ci < S.i1) && (cj < S.j1);
            int o = row * TCX + lane;
            int key = -1;
            if (valid) {
                int a = spk[o], b = spk[o + 1], c = spk[o + TCX + 1], d = spk[o + TCX];
                bool t1 = (a == b) && (a == c);
                bool t2 = (a == c) && (a == d);
                int ax = px_of(a), ay = py_of(a);
                bool inmap = ax >= 0 && ax < S.npix1 && ay >= 0 && ay < S.npix2;
                if (t1 && t2) {
                    tc.single += 2;
                    if (inmap) {
                        int lx = ax - Wl.ax, ly = ay - Wl.ay;
                        if (lx >= 0 && lx < WW && ly >= 0 && ly < WH) key = ly * WW + lx;
                        else atomicAdd(&S.acc[(size_t)ay * S.npix1 + ax], 2ull << FIXBITS);
                    }
                } else {
                    if (t1 || t2) {
                        ++tc.single;
                        if (inmap) deposit_fix(S, Wl, ax, ay, 1ull << FIXBITS);
                    }
                    int slot = atomicAdd(&list_n, (t1 || t2) ? 1 : 2);
                    unsigned short id = (unsigned short)((row * (TCX - 1) + lane) << 1);
                    if (!t1) list[slot++] = id;
                    if (!t2) list[slot] = id | 1;
                }
            }
            window_add_rle(win, key, 2ull << FIXBITS);
        }
        __syncthreads();

        // ---- part 2: the remaining triangles, densely packed over the threads
        int nl = list_n;
        for (int e = threadIdx.x; e < nl; e += blockDim.x) {
            int id = list[e];
            int cell = id >> 1, row = cell / (TCX - 1), col = cell % (TCX - 1);
            int o = row * TCX + col;
            int o1 = (id & 1) ? o + TCX + 1 : o + 1;             // T1 = a,b,c ; T2 = a,c,d  (reading G9)
            int o2 = (id & 1) ? o + TCX : o + TCX + 1;
            deposit_general(S, Wl, su[o], sv[o], su[o1], sv[o1], su[o2], sv[o2], tc);
        }
        __syncthreads();
        // ---- flush the window (it holds in-map pixels only)
        for (int k = threadIdx.x; k < WH * WW; k += blockDim.x) {
            unsigned long long c = win[k];
            if (c) {
                int px = Wl.ax + k % WW, py = Wl.ay + k / WW;
                atomicAdd(&S.acc[(size_t)py * S.npix1 + px], c);
            }
        }
    }
    flush_counters(S, tc);
}

// Cooperative apportioning of the queued large triangles: one warp per queue entry (<= CHUNK_ROWS pixel
// rows).  Lanes take one row each: span of the row, run of pixels lying wholly inside (two adds into the
// row-difference array), then the warp walks the remaining edge pixels of its 32 rows together.
__global__ void __launch_bounds__(256) drain_kernel(ShootDev S) {
    const int lane = threadIdx.x & 31;
    const unsigned full = 0xffffffffu;
    long long nq = (long long)S.counters[C_QUEUE];
    if (nq > S.queue_cap) nq = S.queue_cap;
    long long wid = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    Window W0; W0.win = nullptr; W0.ax = 0; W0.ay = 0;
    unsigned int n_int = 0, n_edge = 0, n_rows = 0;
    for (long long q = wid; q < nq; q += nw) {
        const double *e = S.queue + (size_t)q * QENT;
        TriBox B;
        if (tri_prepare(S, W0, e[0], e[1], e[2], e[3], e[4], e[5], B) != 2) continue;
        TriEdges E;
        tri_setup(E, B.x[0], B.y[0], B.x[1], B.y[1], B.x[2], B.y[2]);
        const int r0 = __double2loint(e[6]), r1 = __double2hiint(e[6]);
        const double sgn = (B.A > 0.0) ? 1.0 : -1.0, invA = 1.0 / B.A;
        const unsigned long long cfix = to_fix(fabs(invA));
        // edge functions F_k(x,y) = gx_k (x - px_k) + gy_k (y - py_k) >= 0 inside
        double gx[3], gy[3], m0[3], m1[3], igx[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            gx[k] = -sgn * E.dy[k]; gy[k] = sgn * E.dx[k];
            m0[k] = fmin(0.0, gx[k]) + fmin(0.0, gy[k]);
            m1[k] = fmax(0.0, gx[k]) + fmax(0.0, gy[k]);
            igx[k] = (gx[k] != 0.0) ? 1.0 / gx[k] : 0.0;
        }
        for (int base = r0; base < r1; base += 32) {
            const int py = base + lane;
            const bool have = py < r1;
            const double yl = (double)py - B.by;               // strip [yl, yl+1] in local coordinates
            int xs = 0, xe = -1, xa = 0, xb = -1;
            if (have) {
                double xmin = 1.0e300, xmax = -1.0e300;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    double vy = E.py[k];
                    if (vy >= yl && vy <= yl + 1.0) { xmin = fmin(xmin, E.px[k]); xmax = fmax(xmax, E.px[k]); }
                    if (E.dy[k] != 0.0) {
                        double ta = (yl - vy) * E.idy[k], tb = (yl + 1.0 - vy) * E.idy[k];
                        if (ta >= 0.0 && ta <= 1.0) { double xx = fma(ta, E.dx[k], E.px[k]); xmin = fmin(xmin, xx); xmax = fmax(xmax, xx); }
                        if (tb >= 0.0 && tb <= 1.0) { double xx = fma(tb, E.dx[k], E.px[k]); xmin = fmin(xmin, xx); xmax = fmax(xmax, xx); }
                    }
                }
                if (xmax >= xmin) {
                    xs = max(B.lox, (int)fmax(floor(xmin - 1e-9) + B.bx, -1.0e9));
                    xe = min(B.hix, (int)fmin(floor(xmax + 1e-9) + B.bx, 1.0e9));
                    // pixels wholly inside: F_k(X, yl) + m0_k >= 0 for all k, linear in X
                    double lo = -1.0e18, hi = 1.0e18;
                    bool none = false;
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        double c0 = fma(gy[k], yl - E.py[k], m0[k]) - gx[k] * E.px[k];    // F + m0 at X = 0
                        if (gx[k] > 0.0) lo = fmax(lo, -c0 * igx[k]);
                        else if (gx[k] < 0.0) hi = fmin(hi, -c0 * igx[k]);
                        else if (c0 < 0.0) none = true;
                    }
                    xa = xe + 1; xb = xe;                              // default: no interior run
                    if (!none && hi >= lo && xe >= xs) {
                        int ta = max(xs, (int)fmax(ceil(lo) + B.bx, -1.0e9));
                        int tb = min(xe, (int)fmin(floor(hi) + B.bx, 1.0e9));
                        if (tb >= ta) {
                            xa = ta; xb = tb;
                            unsigned long long *row = S.diff + (size_t)py * S.npix1;
                            atomicAdd(&row[xa], cfix);
                            if (xb + 1 < S.npix1) atomicAdd(&row[xb + 1], (unsigned long long)(-(long long)cfix));
                            n_int += (unsigned int)(xb - xa + 1);
                        }
                    }
                    ++n_rows;
                }
            }
            const int nL = (have && xe >= xs) ? max(0, xa - xs) : 0;
            const int nR = (have && xe >= xs) ? max(0, xe - xb) : 0;
            int cnt = nL + nR, inc = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(full, inc, o); if (lane >= o) inc += t; }
            const int total = __shfl_sync(full, inc, 31), off = inc - cnt;
            for (int t0 = 0; t0 < total; t0 += 32) {
                const int t = t0 + lane;
                int r = 0;
#pragma unroll
                for (int step = 16; step; step >>= 1) {
                    int cand = r + step;
                    int v = __shfl_sync(full, off, cand & 31);
                    if (cand < 32 && v <= t) r = cand;
                }
                const int o_r = __shfl_sync(full, off, r), xs_r = __shfl_sync(full, xs, r);
                const int nL_r = __shfl_sync(full, nL, r), xb_r = __shfl_sync(full, xb, r);
                if (t < total) {
                    const int kk = t - o_r;
                    const int px = (kk < nL_r) ? xs_r + kk : xb_r + 1 + (kk - nL_r);
                    const int pyr = base + r;
                    const double qx = (double)px - B.bx, qy = (double)pyr - B.by;
                    int cut = 0, which = 0;
                    bool outside = false;
                    double f0w = 0.0;
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        double f0 = fma(gx[k], qx - E.px[k], gy[k] * (qy - E.py[k]));
                        if (f0 + m1[k] < 0.0) outside = true;
                        if (f0 + m0[k] < 0.0) { ++cut; which = k; f0w = f0; }
                    }
                    if (!outside) {
                        double area;
                        if (cut == 0) area = 1.0;
                        else if (cut == 1) area = halfplane_pixel_area(f0w, gx[which], gy[which]);
                        else area = sgn * tri_pixel_area(E, qx, qy);
                        deposit_fix(S, W0, px, pyr, to_fix(area * fabs(invA)));
                        ++n_edge;
                    }
                }
            }
        }
    }
    for (int o = 16; o; o >>= 1) {
        n_int += __shfl_xor_sync(full, n_int, o); n_edge += __shfl_xor_sync(full, n_edge, o); n_rows += __shfl_xor_sync(full, n_rows, o);
    }
    if (lane == 0) {
        if (n_int) atomicAdd(&S.counters[C_PX_INT], (unsigned long long)n_int);
        if (n_edge) atomicAdd(&S.counters[C_PX_EDGE], (unsigned long long)n_edge);
        if (n_rows) atomicAdd(&S.counters[C_ROWS], (unsigned long long)n_rows);
    }
}

// ------------------------------------------------------------------------------------------------
// IRS: rays at cell centres (reading G10), floor of a true division (O5), counts.
__global__ void __launch_bounds__(NWARP * 32) shoot_irs_kernel(ShootDev S) {
    __shared__ TileExp T;
    __shared__ double2 fold[(TQMAX + 1) * ML_NEAR];
    __shared__ unsigned long long win[WH * WW];
    __shared__ int wax, way;
    __shared__ long long tile_slot;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ThreadCounters tc;
    const long long ntiles = (long long)S.ntx * S.tile_rows;
    const long long nrx = S.i1 - S.i0;

    for (long long tile = next_tile(S, &tile_slot); tile < ntiles; tile = next_tile(S, &tile_slot)) {
        long long ty = S.tile_row0 + tile / S.ntx;
        int tx = (int)(tile % S.ntx);
        long long ci0 = S.i0 + (long long)tx * TCX, cj0 = S.j0 + ty * TCY;
        long long ci1 = min(ci0 + TCX, S.i1) - 1, cj1 = min(cj0 + TCY, S.j1) - 1;      // last cell of the tile
        for (int k = threadIdx.x; k < WH * WW; k += blockDim.x) win[k] = 0ull;
        tile_setup(S, T, ci0, cj0, ci1, cj1, 0.5, &S.counters[C_TILES_FULL], fold);
        // the window is anchored on the ray in the middle of the tile's existing part
        const int arow = (int)min((long long)(TCY / 2), cj1 - cj0), acol = (int)min((long long)(TCX / 2), ci1 - ci0);

        double x[RPT], y[RPT], ux[RPT], uy[RPT], wx[RPT], wy[RPT];
        bool valid[RPT];
        int px[RPT], py[RPT];
        const long long ci = ci0 + lane;
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            const int row = warp + r * NWARP;
            const long long cj = cj0 + row;
            valid[r] = (ci < S.i1) && (cj < S.j1);
            x[r] = corner_x(S, ci) + 0.5 * S.h1; y[r] = corner_y(S, cj) + 0.5 * S.h2;
            ux[r] = ((double)lane - 0.5 * (TCX - 1)) * S.h1 * T.inv_rt;
            uy[r] = ((double)row - 0.5 * (TCY - 1)) * S.h2 * T.inv_rt;
        }
        eval_rays(S, T, x, y, ux, uy, valid, wx, wy, tc);
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            px[r] = -1; py[r] = -1;
            if (!valid[r]) continue;
            const int row = warp + r * NWARP;
            if (S.dump1) {
                size_t d = (size_t)(cj0 + row - S.j0) * nrx + (size_t)(ci - S.i0);
                S.dump1[d] = wx[r]; S.dump2[d] = wy[r];
            }
            double fx = floor((wx[r] - S.ylo1) / S.p1), fy = floor((wy[r] - S.ylo2) / S.p2);
            if (fx >= 0.0 && fx < (double)S.npix1 && fy >= 0.0 && fy < (double)S.npix2) { px[r] = (int)fx; py[r] = (int)fy; }
            if (lane == acol && row == arow) {
                wax = (int)fmin(fmax(fx, -1e9), 1e9) - WW / 2; way = (int)fmin(fmax(fy, -1e9), 1e9) - WH / 2;
            }
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            int key = -1;
            if (px[r] >= 0) {
                ++tc.single;
                int lx = px[r] - wax, ly = py[r] - way;
                if (lx >= 0 && lx < WW && ly >= 0 && ly < WH) key = ly * WW + lx;
                else atomicAdd(&S.acc[(size_t)py[r] * S.npix1 + px[r]], 1ull);
            }
            window_add_rle(win, key, 1ull);
        }
        __syncthreads();
        for (int k = threadIdx.x; k < WH * WW; k += blockDim.x) {
            unsigned long long c = win[k];
            if (c) atomicAdd(&S.acc[(size_t)(way + k / WW) * S.npix1 + (wax + k % WW)], c);
        }
    }
    flush_counters(S, tc);
}

// ------------------------------------------------------------------------------------------------
// map[i] = scale * (acc[i] + prefix sum of diff along the row); one block per pixel row.
static const int FIN_T = 256;
__global__ void __launch_bounds__(FIN_T) finalise_kernel(const unsigned long long *acc, const unsigned long long *diff,
                                                         int npix1, double scale, int accumulate,
                                                         double *map, unsigned long long *counts) {
    __shared__ unsigned long long wsum[FIN_T / 32];
    __shared__ unsigned long long carry_s;
    const size_t row = (size_t)blockIdx.x * npix1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0ull;
    __syncthreads();
    for (int base = 0; base < npix1; base += FIN_T) {
        const int i = base + threadIdx.x;
        unsigned long long d = (diff && i < npix1) ? diff[row + i] : 0ull;
        unsigned long long inc = d;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
        if (lane == 31) wsum[warp] = inc;
        __syncthreads();
        unsigned long long pre = carry_s;
        for (int w = 0; w < warp; ++w) pre += wsum[w];
        unsigned long long run = pre + inc;                  // inclusive prefix of diff up to i
        if (i < npix1) {
            unsigned long long a = acc[row + i] + run;
            if (map) { double v = (double)a * scale; map[row + i] = accumulate ? map[row + i] + v : v; }
            if (counts) counts[row + i] = accumulate ? counts[row + i] + a : a;
        }
        __syncthreads();
        if (threadIdx.x == FIN_T - 1) carry_s = run;
        __syncthreads();
    }
}

// Geometry of the shooting window and ray grid: eq 14-16, eq A6; O1/O2.
int geometry(const mlens_field *f, const mlens_shoot_desc *d, mlens_grid *g) {
    double a1 = 1.0 - f->kappa_tot + f->gamma, a2 = 1.0 - f->kappa_tot - f->gamma;
    if (a1 == 0.0 || a2 == 0.0) { set_error("macro model is singular (1-kappa+-gamma = 0)"); return MLENS_EINVAL; }
    if (d->npix1 <= 0 || d->npix2 <= 0 || !(d->rays_per_pixel_length > 0) || !(d->half_y1 > 0) || !(d->half_y2 > 0)) {
        set_error("bad map description"); return MLENS_EINVAL;
    }
    if (d->npix1 > 30000 || d->npix2 > 30000) { set_error("maps are limited to 30000 pixels per side"); return MLENS_EINVAL; }
    g->p1 = 2.0 * d->half_y1 / d->npix1;
    g->p2 = 2.0 * d->half_y2 / d->npix2;
    g->h1 = g->p1 / d->rays_per_pixel_length;
    g->h2 = g->p2 / d->rays_per_pixel_length;
    g->X1 = d->center_y1 / a1;
    g->X2 = d->center_y2 / a2;
    double b1 = 0, b2 = 0, H1, H2;
    switch (d->border_mode) {
        case MLENS_BORDER_EQ16: {
            double r = 10.0 * f->theta * sqrt(f->kappa_star);
            b1 = d->half_y1 + r; b2 = d->half_y2 + r; break; }
        case MLENS_BORDER_A6: {
            if (!(d->border_param > 0)) { set_error("eq A6 needs f > 0"); return MLENS_EINVAL; }
            double m2m = (f->mean_m > 0) ? f->mean_m2 / f->mean_m : 1.0;
            double r = f->theta * sqrt(f->kappa_star * m2m / d->border_param);
            b1 = d->half_y1 + r; b2 = d->half_y2 + r; break; }
        case MLENS_BORDER_MARGIN:
            b1 = d->half_y1 * (1.0 + d->border_param); b2 = d->half_y2 * (1.0 + d->border_param); break;
        case MLENS_BORDER_EXPLICIT:
            if (!(d->He1 > 0) || !(d->He2 > 0)) { set_error("explicit window needs He1, He2 > 0"); return MLENS_EINVAL; }
            break;
        default: set_error("unknown border mode"); return MLENS_EINVAL;
    }
    H1 = (d->border_mode == MLENS_BORDER_EXPLICIT) ? d->He1 : b1 / fabs(a1);
    H2 = (d->border_mode == MLENS_BORDER_EXPLICIT) ? d->He2 : b2 / fabs(a2);
    double n1 = ceil(2.0 * H1 / g->h1), n2 = ceil(2.0 * H2 / g->h2);
    if (!(n1 >= 1) || !(n2 >= 1) || n1 > 4.0e9 || n2 > 4.0e9) { set_error("ray grid out of range"); return MLENS_EINVAL; }
    g->n1 = (int64_t)n1; g->n2 = (int64_t)n2;
    g->H1 = 0.5 * ((double)g->n1 * g->h1);
    g->H2 = 0.5 * ((double)g->n2 * g->h2);
    g->x0_1 = g->X1 - g->H1;
    g->x0_2 = g->X2 - g->H2;
    g->ylo1 = d->center_y1 - d->half_y1;
    g->ylo2 = d->center_y2 - d->half_y2;
    g->weight = (g->h1 * g->h2) / (2.0 * (g->p1 * g->p2));
    g->order = f->order;
    return MLENS_OK;
}

static long long env_ll(const char *name, long long dflt) {
    const char *v = getenv(name);
    if (!v || !*v) return dflt;
    long long x = atoll(v);
    return x > 0 ? x : dflt;
}

int shoot(mlens_field *f, const mlens_shoot_desc *d, const mlens_grid *g, double *map,
          unsigned long long *counts, mlens_stats *st, cudaStream_t s) {
    long long i0 = d->i0, i1 = d->i1, j0 = d->j0, j1 = d->j1;
    if (i1 <= 0 || j1 <= 0) { i0 = 0; i1 = g->n1; j0 = 0; j1 = g->n2; }
    if (i0 < 0 || j0 < 0 || i1 > g->n1 || j1 > g->n2 || i1 <= i0 || j1 <= j0) { set_error("bad cell sub-range"); return MLENS_EINVAL; }
    const long long npix = (long long)d->npix1 * d->npix2;
    const bool ipm = d->map_mode == MLENS_MAP_IPM;
    ML_TRY(f->acc.reserve((size_t)npix, s, false));
    ML_TRY(f->counters.reserve(C_NCOUNTERS, s, false));
    ML_CUDA(cudaMemsetAsync(f->acc.p, 0, (size_t)npix * 8, s));
    ML_CUDA(cudaMemsetAsync(f->counters.p, 0, C_NCOUNTERS * 8, s));
    long long qcap = 0;
    if (ipm) {
        ML_TRY(f->diff.reserve((size_t)npix, s, false));
        ML_CUDA(cudaMemsetAsync(f->diff.p, 0, (size_t)npix * 8, s));
        long long qmb = env_ll("MLENS_QUEUE_MB", 1024);
        qcap = qmb * (1ll << 20) / (QENT * 8);
        ML_TRY(f->queue.reserve((size_t)qcap * QENT, s, false));
    }
    ShootDev S;
    S.L = make_lens_dev(f);
    S.x0_1 = g->x0_1; S.x0_2 = g->x0_2; S.h1 = g->h1; S.h2 = g->h2;
    S.i0 = i0; S.i1 = i1; S.j0 = j0; S.j1 = j1;
    S.ylo1 = g->ylo1; S.ylo2 = g->ylo2; S.p1 = g->p1; S.p2 = g->p2; S.inv_p1 = 1.0 / g->p1; S.inv_p2 = 1.0 / g->p2;
    S.npix1 = d->npix1; S.npix2 = d->npix2;
    S.acc = f->acc.p; S.diff = f->diff.p; S.queue = f->queue.p; S.counters = f->counters.p; S.queue_cap = qcap;
    S.dump1 = d->dump_w1; S.dump2 = d->dump_w2;
    S.binom = f->binom.p;
    if ((S.dump1 == nullptr) != (S.dump2 == nullptr)) { set_error("dump_w1 and dump_w2 go together"); return MLENS_EINVAL; }
    S.eval_mode = d->eval_mode;
    S.tq = (int)env_ll("MLENS_TILE_ORDER", 12);
    if (S.tq > TQMAX) S.tq = TQMAX;
    if (S.tq < 2) S.tq = 2;
    // truncation budget of the tile series: 5 % of the deflection accuracy the field was built for
    S.eps_far = 0.02 * f->eps * f->theta;
    S.eps_star = 0.03 * f->eps * f->theta / (double)ML_NEAR;
    const int stepx = ipm ? TCX - 1 : TCX, stepy = ipm ? TCY - 1 : TCY;
    long long ntx = (i1 - i0 + stepx - 1) / stepx, nty = (j1 - j0 + stepy - 1) / stepy;
    if (ntx > 0x7fffffffLL) { set_error("too many tiles per row"); return MLENS_EINVAL; }
    S.ntx = (int)ntx;
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    long long band_cells = env_ll("MLENS_BAND_CELLS", 1ll << 27);
    long long rows_per_band = band_cells / (ntx * stepx * stepy);
    if (rows_per_band < 1) rows_per_band = 1;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const bool timed = st && (d->sync || d->ptr_kind == MLENS_PTR_HOST);
    if (timed) { ML_CUDA(cudaEventCreate(&e0)); ML_CUDA(cudaEventCreate(&e1)); ML_CUDA(cudaEventRecord(e0, s)); }
    int launches = 0, bands = 0;
    // per-kernel device times: events between the back-to-back launches of each band (timed calls only)
    std::vector<cudaEvent_t> ev;
    auto mark = [&]() -> int {
        if (!timed) return MLENS_OK;
        cudaEvent_t e; ML_CUDA(cudaEventCreate(&e)); ML_CUDA(cudaEventRecord(e, s)); ev.push_back(e);
        return MLENS_OK;
    };
    int bps_ipm = 1, bps_irs = 1;
    ML_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps_ipm, shoot_ipm_kernel, NWARP * 32, 0));
    ML_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps_irs, shoot_irs_kernel, NWARP * 32, 0));
    for (long long r0 = 0; r0 < nty; r0 += rows_per_band, ++bands) {
        S.tile_row0 = r0;
        S.tile_rows = (nty - r0 < rows_per_band) ? (nty - r0) : rows_per_band;
        long long nt = ntx * S.tile_rows;
        const long long resident = (long long)nsm * (ipm ? bps_ipm : bps_irs);     // persistent blocks, tiles handed out dynamically
        int grid = (int)((nt < resident) ? nt : resident);
        ML_CUDA(cudaMemsetAsync(f->counters.p, 0, 16, s));         // queue fill count and tile counter
        ML_TRY(mark());
        if (ipm) {
            ML_LAUNCH(shoot_ipm_kernel, grid, NWARP * 32, 0, s, S);
            ML_TRY(mark());
            ML_LAUNCH(drain_kernel, nsm * 8, 256, 0, s, S);
            ML_TRY(mark());
            launches += 2;
        } else {
            ML_LAUNCH(shoot_irs_kernel, grid, NWARP * 32, 0, s, S);
            ML_TRY(mark());
            launches += 1;
        }
        ML_CUDA(cudaGetLastError());
    }
    double scale = ipm ? g->weight / (double)(1ull << FIXBITS)
                       : 1.0 / (d->rays_per_pixel_length * d->rays_per_pixel_length);
    ML_LAUNCH(finalise_kernel, (unsigned)d->npix2, FIN_T, 0, s, f->acc.p, ipm ? f->diff.p : nullptr, d->npix1, scale,
              d->accumulate, map, ipm ? nullptr : counts);
    ML_TRY(mark());
    ++launches;
    ML_CUDA(cudaGetLastError());
    if (timed) ML_CUDA(cudaEventRecord(e1, s));
    if (st) {
        unsigned long long h[C_NCOUNTERS];
        ML_CUDA(cudaMemcpyAsync(h, f->counters.p, sizeof(h), cudaMemcpyDeviceToHost, s));
        ML_CUDA(cudaStreamSynchronize(s));
        memset(st, 0, sizeof(*st));
        st->n_rays = (int64_t)h[C_RAYS];
        st->n_cells = (i1 - i0) * (j1 - j0);
        st->n_tri_single = (int64_t)h[C_SINGLE]; st->n_tri_small = (int64_t)h[C_SMALL];
        st->n_tri_queued = (int64_t)h[C_QUEUED]; st->n_queue_chunks = (int64_t)h[C_CHUNKS];
        st->n_queue_overflow = (int64_t)h[C_OVERFLOW]; st->n_rays_fallback = (int64_t)h[C_FALLBACK];
        st->n_near_terms = (int64_t)h[C_NEAR];
        st->n_px_small = (int64_t)h[C_PX_SMALL]; st->n_px_interior = (int64_t)h[C_PX_INT];
        st->n_px_edge = (int64_t)h[C_PX_EDGE]; st->n_rows = (int64_t)h[C_ROWS];
        st->n_tiles_full = (int64_t)h[C_TILES_FULL];
        st->tile_order = S.tq;
        st->n_bands = bands; st->gpu_launches = launches; st->n_shoot_launches = bands;
        if (timed) {
            ML_CUDA(cudaEventElapsedTime(&st->ms_total, e0, e1)); cudaEventDestroy(e0); cudaEventDestroy(e1);
            const size_t per = ipm ? 3 : 2;              // events per band
            for (int b = 0; b < bands; ++b) {
                float ms = 0;
                ML_CUDA(cudaEventElapsedTime(&ms, ev[b * per], ev[b * per + 1])); st->ms_shoot += ms;
                if (ipm) { ML_CUDA(cudaEventElapsedTime(&ms, ev[b * per + 1], ev[b * per + 2])); st->ms_drain += ms; }
            }
            float ms = 0;
            ML_CUDA(cudaEventElapsedTime(&ms, ev[ev.size() - 2], ev[ev.size() - 1])); st->ms_finalise = ms;
        }
    } else if (d->sync) {
        ML_CUDA(cudaStreamSynchronize(s));
    }
    for (cudaEvent_t e : ev) cudaEventDestroy(e);
    return MLENS_OK;
}

}  // namespace ml
