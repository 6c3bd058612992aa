// deposit.cuh -- exact area apportioning of mapped triangles (hot loop B) for warp-autonomous kernels.
//
// Accumulation is 64-bit fixed point, ONE = 2^FIXBITS per whole triangle: integer adds commute, so maps are
// bit-reproducible whatever the atomic order.  Two arrays: `acc` holds pixel sums, `diff` the ROW DIFFERENCES
// of what the large triangles add (map[y][x] = acc[y][x] + sum_{x' <= x} diff[y][x'], finalise_kernel).
//   - a triangle inside one pixel:            ONE into that pixel                       (run-length merged per warp)
//   - a triangle over two adjacent pixels:    closed-form split by the area fraction below the pixel line
//   - a triangle with a small bounding box:   every pixel of the box clipped exactly (Green's theorem form of
//     Sutherland-Hodgman + shoelace), the pixels of 32 triangles spread evenly over the warp's lanes
//   - any larger triangle (drain_kernel):     signed-area edge walk.  Every edge is cut into pieces by the
//     pixel grid lines it crosses; a piece inside pixel (i, j) that rises by dy covers dy (1 - m) of pixel i
//     and dy of every pixel to its right in row j (m = mean x of the piece within the pixel), i.e.
//     diff[j][i] += c dy (1 - m), diff[j][i+1] += c dy m  with c = -sign(A) ONE/|A|.  The three edges' covers
//     cancel to the right of the triangle; they cancel EXACTLY because c dy is computed as G(y_end) - G(y_start)
//     with G(y) = round(c y) evaluated on values shared by consecutive pieces (vertices, grid lines, and the exact
//     row line where the first or last row of the map cuts an edge).
//     Cost is proportional to the triangle's perimeter in pixels, never to its area, and the result is the same
//     area of intersection as clipping every pixel, up to rounding.  An edge is set up in a frame and direction of
//     its own, so the two triangles that share it see identical pieces and walk_kernel walks it once for both.
#pragma once
#include "tile.cuh"

namespace ml {

static const int FIXBITS = 36;
static const unsigned long long FIX_ONE = 1ull << FIXBITS;
static const int QENT = 6;                 // doubles per queue entry: the 3 vertices in pixel units
static const int QCHUNK = 256;             // queue entries a warp reserves at a time


struct Win {                           // where a warp's deposits go (uniform registers)
    unsigned int *w32;                 // the warp's shared window viewed as 32-bit halves, or nullptr
    int ax, ay;
};

// 64-bit add into shared memory from two native 32-bit atomics (a 64-bit shared atomicAdd is a CAS loop):
// the low word returns its old value, the carry it produced joins the high word.  Sums commute, so the
// word pair always ends up holding the exact 64-bit total.
__device__ __forceinline__ void shared_add64(unsigned int *w32, int idx, unsigned long long v) {
    unsigned int lo = (unsigned int)v, hi = (unsigned int)(v >> 32);
    if (lo) {
        unsigned int old = atomicAdd(&w32[2 * idx], lo);
        hi += (old + lo < old) ? 1u : 0u;
    }
    if (hi) atomicAdd(&w32[2 * idx + 1], hi);
}

// v into pixel (px, py) of the map (window if it covers the pixel, else L2); pixels outside the map receive nothing
__device__ __forceinline__ void pix_add(const ShootDev &S, const Win &W, int px, int py, unsigned long long v) {
    if ((unsigned)px >= (unsigned)S.npix1 || (unsigned)py >= (unsigned)S.npix2 || v == 0ull) return;
    unsigned int lx = (unsigned int)(px - W.ax), ly = (unsigned int)(py - W.ay);
    if (W.w32 && lx < (unsigned)WX && ly < (unsigned)WY) shared_add64(W.w32, (int)(ly * WX + lx), v);
    else atomicAdd(&S.acc[(size_t)py * S.npix1 + px], v);
}
__device__ __forceinline__ void flush_window(const ShootDev &S, const WarpShared &Ws, const Win &W) {
    const int lane = threadIdx.x & 31;
#pragma unroll 4
    for (int k = lane; k < WY * WX; k += 32) {
        unsigned long long c = Ws.win[k];
        if (c) {
            int px = W.ax + (k % WX), py = W.ay + (k / WX);            // only in-map pixels were ever added
            atomicAdd(&S.acc[(size_t)py * S.npix1 + px], c);
        }
    }
}

__device__ __forceinline__ int floor_to_int(double u) {
    return (int)floor(fmin(fmax(u, -1.0e9), 1.0e9));      // NaN -> -1e9
}
// pixel coordinates packed as two int16 (values beyond the map on one side collapse: such triangles are outside)
__device__ __forceinline__ int pack_px(double u, double v) {
    // floor by the converting instruction itself (saturates for huge values, gives 0 for NaN), then clamp in integers
    int a = max(min(__double2int_rd(u), 30000), -30000), b = max(min(__double2int_rd(v), 30000), -30000);
    if (u != u) a = -30000;
    if (v != v) b = -30000;
    return (b << 16) | (a & 0xffff);
}
// ... and the sides of the map the pixel lies beyond (Cohen-Sutherland code): a triangle whose three codes share a
// bit cannot touch the map
__device__ __forceinline__ int out_code(int pk, int npix1, int npix2) {
    const int a = (int)(short)(pk & 0xffff), b = pk >> 16;
    return (a < 0 ? 1 : 0) | (a >= npix1 ? 2 : 0) | (b < 0 ? 4 : 0) | (b >= npix2 ? 8 : 0);
}
__device__ __forceinline__ int px_of(int pk) { return (int)(short)(pk & 0xffff); }
__device__ __forceinline__ int py_of(int pk) { return pk >> 16; }

__device__ __forceinline__ unsigned long long to_fix(double frac) {
    long long v = __double2ll_rn(frac * (double)FIX_ONE);
    v = v < 0 ? 0 : v;
    return v > (long long)FIX_ONE ? FIX_ONE : (unsigned long long)v;
}

// Fraction of a triangle's area on the negative side of an axis-parallel line, d0..d2 the signed distances
// of the vertices from it: the lone vertex cuts off a similar corner, ratio t1 t2 of its two edges.
__device__ __forceinline__ double frac_below(double d0, double d1, double d2) {
    bool n0 = d0 < 0.0, n1 = d1 < 0.0, n2 = d2 < 0.0;
    int cnt = (int)n0 + (int)n1 + (int)n2;
    if (cnt == 0) return 0.0;
    if (cnt == 3) return 1.0;
    bool lone_neg = (cnt == 1);
    double l, o1, o2;
    if (n0 == lone_neg) { l = d0; o1 = d1; o2 = d2; }
    else if (n1 == lone_neg) { l = d1; o1 = d0; o2 = d2; }
    else { l = d2; o1 = d0; o2 = d1; }
    double f = (l * l) * fast_rcp((l - o1) * (l - o2));
    return lone_neg ? f : 1.0 - f;
}

// min / max by one compare and one select (fmin / fmax also order NaNs: a dozen instructions each on FP64)
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }     // operands are never NaN here
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double clamp01(double v) { return dmin(dmax(v, 0.0), 1.0); }

// ---- the edge walk ------------------------------------------------------------------------------------------
// An edge is walked along its MAJOR axis: between two consecutive grid lines of that axis it stays inside one
// row (or column) of pixels and, its slope being <= 1, crosses at most one grid line of the other axis -- so a
// step yields one or two pieces, found without any search, and the steps are independent (one per lane).
struct EdgeWalk {                     // one triangle edge, clipped to the map rows and to the columns left of the map's right border
    double x0, y0, x1, y1, dx, dy, idx, idy, ta, tb;
    double g0, sg;                    // first grid line crossed along the major axis and the step (+-1)
    int majorY;                       // 1: walk rows (|dy| >= |dx|), 0: walk columns
    int n;                            // steps = crossings of major-axis grid lines + 1, or 0
    int cf;                           // ends cut by a border row of the map: bits 0-1 the start (1: row line ry0, 2: ry1), bits 2-3 the end
    int bx, by;                       // integer origin of the edge's own frame (edge_setup_canon)
    int fwd;                          // 1: the canonical direction (smaller end first) is the direction the triangle's boundary runs in
};

// local coordinates: pixel units relative to the integer point (bx, by); rows [ry0, ry1] and columns <= cx1 are the map
__device__ __forceinline__ void edge_setup(EdgeWalk &E, double x0, double y0, double x1, double y1, double ry0, double ry1, double cx1) {
    E.x0 = x0; E.y0 = y0; E.x1 = x1; E.y1 = y1; E.dx = x1 - x0; E.dy = y1 - y0;
    E.n = 0; E.ta = 0.0; E.tb = 1.0; E.idx = 0.0; E.idy = 0.0; E.g0 = 0.0; E.sg = 1.0; E.majorY = 1; E.cf = 0;
    if (E.dy == 0.0) return;                                   // a horizontal edge covers nothing
    E.idy = 1.0 / E.dy;
    double ta = 0.0, tb = 1.0;
    const double t0 = (ry0 - y0) * E.idy, t1 = (ry1 - y0) * E.idy;
    const double tlo = fmin(t0, t1), thi = fmax(t0, t1);       // where the edge enters and leaves the rows of the map
    ta = fmax(ta, tlo); tb = fmin(tb, thi);
    if (E.dx != 0.0) {
        E.idx = 1.0 / E.dx;
        double tc = (cx1 - x0) * E.idx;
        if (E.dx > 0.0) tb = fmin(tb, tc); else ta = fmax(ta, tc);
    } else if (x0 >= cx1) return;
    if (!(tb > ta)) return;
    E.ta = ta; E.tb = tb;
    // An end cut by a border row of the map lies ON that row line: it takes the line's exact (integer) value of y,
    // as the ends on grid lines and vertices do, so that the covers G(y) of all the edges that cross the border
    // telescope there too.  A row line lies strictly between the edge's ends only if it is the map's first or last
    // one (ry0 = 0 and ry1 = the top of the bounding box never do: every vertex lies between them) -- decided on the
    // coordinates themselves, not on the parameters, whose rounding can put a vertex that sits ON such a line inside.
    int cf = 0;
    const double ylo = fmin(y0, y1), yhi = fmax(y0, y1);
    const double ls = (E.dy > 0.0) ? ry0 : ry1, le = (E.dy > 0.0) ? ry1 : ry0;     // row lines where the edge enters / leaves the map
    if (ta == tlo && ls > ylo && ls < yhi) cf |= (E.dy > 0.0) ? 1 : 2;
    if (tb == thi && le > ylo && le < yhi) cf |= (E.dy > 0.0) ? 8 : 4;
    E.cf = cf;
    E.majorY = fabs(E.dy) >= fabs(E.dx);
    const double d = E.majorY ? E.dy : E.dx, c0 = E.majorY ? y0 : x0;
    double a = fma(ta, d, c0), b = fma(tb, d, c0);             // major coordinate at the clipped ends
    if (E.majorY) {
        if (cf & 3) a = (cf & 1) ? ry0 : ry1;
        if (cf & 12) b = (cf & 4) ? ry0 : ry1;
    }
    double nc;
    if (d > 0.0) { E.sg = 1.0; E.g0 = floor(a) + 1.0; nc = ceil(b) - 1.0 - floor(a); }
    else { E.sg = -1.0; E.g0 = ceil(a) - 1.0; nc = ceil(a) - 1.0 - floor(b); }
    E.n = ((nc > 0.0) ? (int)fmin(nc, 1.0e7) : 0) + 1;
}

// An edge is set up in a frame and a direction of ITS OWN -- origin = the integer lower-left of its two end points,
// direction = smaller end first (by x, then y) -- so that the two triangles that share it compute the very same pieces,
// bit for bit, whichever of them walks it and whether it is walked once for both or once for each.  (ux0, uy0) ->
// (ux1, uy1): the end points in GLOBAL pixel units, in the order of the triangle's boundary.
__device__ __forceinline__ void edge_setup_canon(const ShootDev &S, EdgeWalk &E, double ux0, double uy0, double ux1, double uy1) {
    const bool fwd = (ux0 < ux1) || (ux0 == ux1 && uy0 <= uy1);
    const double ax = fwd ? ux0 : ux1, ay = fwd ? uy0 : uy1, cx = fwd ? ux1 : ux0, cy = fwd ? uy1 : uy0;
    const double fbx = floor(ax), fby = floor(dmin(ay, cy));          // ax <= cx
    const double hgt = dmax(ay, cy) - fby + 1.0;
    edge_setup(E, ax - fbx, ay - fby, cx - fbx, cy - fby, fmax(0.0, -fby), fmin(hgt, (double)S.npix2 - fby), (double)S.npix1 - fbx);
    E.bx = (int)fbx; E.by = (int)fby; E.fwd = fwd ? 1 : 0;
}

// One piece of an edge, from (xs, ys) to (xe, ye), inside one pixel, with the covers ta, tb it has for the (one or two)
// triangles on its sides: t = G(ye) - G(ys), G(y) = rn(c y), c = -+ONE/|A| of that triangle; (bx, by) = integer origin
// of the local coordinates.  The covers telescope exactly along each triangle's boundary because consecutive pieces
// share the value of G at the point where they meet.  The share that moves to the next column is rounded per triangle,
// so a piece walked once for two triangles deposits exactly what two walks would.
__device__ __forceinline__ void piece_deposit(const ShootDev &S, double xs, double ys, double xe, double ye, long long ta, long long tb, int bx, int by) {
    const long long tcov = ta + tb;
    if ((ta | tb) == 0) return;
    const double ym = 0.5 * (ys + ye), xm = 0.5 * (xs + xe);
    const int jr = __double2int_rd(ym) + by;                   // (coordinates are bounded by 1e9: no saturation)
    if ((unsigned)jr >= (unsigned)S.npix2) return;
    const int il = __double2int_rd(xm);
    const int ic = il + bx;
    if (ic >= S.npix1) return;
    unsigned long long *row = S.diff + (size_t)jr * S.npix1;
    long long r = tcov;                                        // left of the map: the whole cover enters at column 0
    int c0 = 0;
    if (ic >= 0) {
        const double m = clamp01(xm - (double)il);
        r = __double2ll_rn((double)ta * m);
        if (tb) r += __double2ll_rn((double)tb * m);
        c0 = ic + 1;
        if (tcov != r) atomicAdd(row + ic, (unsigned long long)(tcov - r));
    }
    if (c0 < S.npix1 && r != 0) atomicAdd(row + c0, (unsigned long long)r);
}

// An edge in (major, other) order, as the walk reads it (EREC doubles, e.g. in shared memory): c0 -> c1 along the axis
// that is walked, oc0 -> o1 along the other, id / oid the reciprocals of the two extents (0 for an extent of 0),
// [ta, tb] the clipped parameter range, g0 the first grid line; q[9] packs the step count n (high word) with the
// flags: bit 0 major axis is y, bit 1 walking towards smaller coordinates, bits 2-5 the border-row flags cf.
// q[10], q[11]: weight c1 of the triangle the edge was set up for (signed for the canonical direction) and the offset
// d1 = by_edge - by_triangle that takes the edge's local y into that triangle's frame (G is taken there, so that the
// triangle's three edges see the same numbers at the vertices they share).  q[12], q[13]: the same for a SECOND
// triangle on the other side (walk_kernel pairs the edges two triangles of a batch share), c2 = 0 if there is none.
// q[14]: the edge's frame origin (by, bx) packed.
static const int EREC = 16;
__device__ __forceinline__ void edge_record(const EdgeWalk &E, double cs_tri, int by_tri, double *q) {
    const bool my = E.majorY != 0;
    q[0] = my ? E.y0 : E.x0; q[1] = my ? E.x0 : E.y0; q[2] = my ? E.y1 : E.x1; q[3] = my ? E.x1 : E.y1;
    q[4] = my ? E.idy : E.idx; q[5] = my ? E.idx : E.idy; q[6] = E.ta; q[7] = E.tb; q[8] = E.g0;
    q[9] = __hiloint2double(E.n, E.majorY | (E.sg < 0.0 ? 2 : 0) | (E.cf << 2));
    q[10] = E.fwd ? cs_tri : -cs_tri; q[11] = (double)(E.by - by_tri);
    q[12] = 0.0; q[13] = 0.0;
    q[14] = __hiloint2double(E.by, E.bx); q[15] = 0.0;
}
__device__ __forceinline__ int edge_record_steps(const double *q) { return __double2hiint(q[9]); }
// the same geometric edge (set up from the same two end points): everything but the weights agrees bit for bit
__device__ __forceinline__ bool edge_record_same(const double *a, const double *b) {
    return a[0] == b[0] && a[1] == b[1] && a[2] == b[2] && a[3] == b[3] &&
           __double_as_longlong(a[14]) == __double_as_longlong(b[14]);
}

// Steps [m0, m1) of an edge, 0 <= m0 < m1 <= n.  Step k runs from major-axis grid line k-1 (or the clipped start) to
// grid line k (or the clipped end).  End points on a grid line take its exact value, an unclipped end the vertex
// itself, an end cut by a border row of the map that row line's value: consecutive steps and consecutive edges share
// their end points bit for bit.  A lane walks CONSECUTIVE steps: the end of a step (its coordinates and G) is carried
// into the next one, so that every point of the edge is computed once.
__device__ __forceinline__ void edge_run(const ShootDev &S, const double *q, int m0, int m1) {
    const double c0 = q[0], oc0 = q[1], c1 = q[2], o1 = q[3], id = q[4], oid = q[5], ta = q[6], tb = q[7], g0 = q[8];
    const int fl = __double2loint(q[9]), n = __double2hiint(q[9]);
    const double ca = q[10], da = q[11], cb = q[12], db = q[13];
    const int bx = __double2loint(q[14]), by = __double2hiint(q[14]);
    const bool my = (fl & 1) != 0, two = (cb != 0.0);
    const double sg = (fl & 2) ? -1.0 : 1.0;
    const int cf = fl >> 2;
    const double d = c1 - c0, od = o1 - oc0;
    double ms, os, ts;
    if (m0 == 0) {
        ts = ta; ms = (ts == 0.0) ? c0 : fma(ts, d, c0); os = (ts == 0.0) ? oc0 : fma(ts, od, oc0);
        if (cf & 3) {                                          // start on a border row of the map: exactly on it
            const double yl = (cf & 1) ? (double)(-by) : (double)(S.npix2 - by);
            if (my) ms = yl; else os = yl;
        }
    } else { ms = g0 + sg * (double)(m0 - 1); ts = dmin(dmax((ms - c0) * id, ta), tb); os = fma(ts, od, oc0); }
    long long Gas = __double2ll_rn(ca * ((my ? ms : os) + da)), Gbs = two ? __double2ll_rn(cb * ((my ? ms : os) + db)) : 0ll;
#pragma unroll 1
    for (int k = m0; k < m1; ++k) {
        double me, oe, te;
        if (k == n - 1) {
            te = tb;
            const bool vtx = (te == 1.0);
            me = vtx ? c1 : fma(te, d, c0);
            oe = vtx ? o1 : fma(te, od, oc0);
            if (cf & 12) {
                const double yl = (cf & 4) ? (double)(-by) : (double)(S.npix2 - by);
                if (my) me = yl; else oe = yl;
            }
        } else { me = g0 + sg * (double)k; te = dmin(dmax((me - c0) * id, ta), tb); oe = fma(te, od, oc0); }
        const long long Gae = __double2ll_rn(ca * ((my ? me : oe) + da)), Gbe = two ? __double2ll_rn(cb * ((my ? me : oe) + db)) : 0ll;
        // at most one grid line of the other axis lies strictly between os and oe
        const double gl = (oe > os) ? floor(os) + 1.0 : ceil(os) - 1.0;
        const bool cross = (od != 0.0) && ((oe > os) ? (gl < oe) : (gl > oe)) && (oe != os);
        double mg = me, og = oe;                               // where the first piece ends
        long long Gag = Gae, Gbg = Gbe;
        if (cross) {
            const double tg = dmin(dmax((gl - oc0) * oid, ts), te);
            mg = fma(tg, d, c0); og = gl;
            Gag = __double2ll_rn(ca * ((my ? mg : og) + da));
            if (two) Gbg = __double2ll_rn(cb * ((my ? mg : og) + db));
        }
        // the axes are swapped back before the deposit, so that one copy of it serves all lanes: the first piece,
        // then the second of those that cross
        piece_deposit(S, my ? os : ms, my ? ms : os, my ? og : mg, my ? mg : og, Gag - Gas, Gbg - Gbs, bx, by);
        if (cross) piece_deposit(S, my ? og : mg, my ? mg : og, my ? oe : me, my ? me : oe, Gae - Gag, Gbe - Gbg, bx, by);
        ms = me; os = oe; ts = te; Gas = Gae; Gbs = Gbe;
    }
}

struct TriSetup {
    double x[3], y[3];                // local coordinates
    double cs, ry0, ry1, cx1;
    int bx, by;
    int status;                       // 0: nothing to deposit, 1: walk the edges
};

// Reading G12: a triangle of zero area puts its whole weight into the pixel of vertex 0.  The same is done
// when ONE/|A| times the triangle's height would leave the 63-bit range (aspect ratio beyond ~2^26).
__device__ __forceinline__ void tri_setup(const ShootDev &S, const Win &W, const double *v, TriSetup &T) {
    T.status = 0;
    const double u0 = v[0], v0 = v[1], u1 = v[2], v1 = v[3], u2 = v[4], v2 = v[5];
    const double nan_probe = (u0 + u1 + u2) + (v0 + v1 + v2);                    // NaN if any is (or if infinities cancel)
    if (!(nan_probe == nan_probe)) return;
    const double mnx = dmin(u0, dmin(u1, u2)), mxx = dmax(u0, dmax(u1, u2));
    const double mny = dmin(v0, dmin(v1, v2)), mxy = dmax(v0, dmax(v1, v2));
    if (!(mxx >= 0.0) || !(mxy >= 0.0) || !(mnx < (double)S.npix1) || !(mny < (double)S.npix2)) return;
    if (!(mnx > -1.0e9) || !(mny > -1.0e9) || !(mxx < 1.0e9) || !(mxy < 1.0e9)) return;                     // inf / absurd
    const double fbx = floor(mnx), fby = floor(mny);
    T.bx = (int)fbx; T.by = (int)fby;
    T.x[0] = u0 - fbx; T.y[0] = v0 - fby; T.x[1] = u1 - fbx; T.y[1] = v1 - fby; T.x[2] = u2 - fbx; T.y[2] = v2 - fby;
    const double A2 = (T.x[1] - T.x[0]) * (T.y[2] - T.y[0]) - (T.x[2] - T.x[0]) * (T.y[1] - T.y[0]);
    const double hgt = mxy - fby + 1.0;
    const double c = (A2 != 0.0) ? 2.0 * (double)FIX_ONE / fabs(A2) : 0.0;
    if (A2 == 0.0 || !(c * hgt < 4.0e18)) {
        pix_add(S, W, floor_to_int(u0), floor_to_int(v0), FIX_ONE);
        return;
    }
    T.cs = (A2 > 0.0) ? -c : c;
    T.ry0 = fmax(0.0, -fby); T.ry1 = fmin(hgt, (double)S.npix2 - fby); T.cx1 = (double)S.npix1 - fbx;
    T.status = 1;
}

// Exact area of (triangle  intersect  unit pixel [qx, qx+1] x [qy, qy+1]) by Green's theorem: area = closed
// integral of clamp(x - qx, 0, 1) dy over the part of the boundary with y in the pixel's row.  Same value as
// Sutherland-Hodgman clipping + shoelace up to rounding; no polygon arrays, no data-dependent vertex
// counts.  Signed like the triangle.  (x, y)[3] = vertices, (idx, idy)[3] = reciprocal edge vectors (0 if the
// component is 0), edge k runs from vertex k to vertex k+1.
__device__ __forceinline__ double tri_pixel_area(const double (&x)[3], const double (&y)[3], const double (&idx)[3], const double (&idy)[3],
                                                 double qx, double qy) {
    double s = 0.0;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        const int e1 = (e == 2) ? 0 : e + 1;
        const double dy = y[e1] - y[e];
        if (dy == 0.0) continue;
        const double px = x[e] - qx, py = y[e] - qy, dx = x[e1] - x[e];
        const double ta = -py * idy[e], tb = (1.0 - py) * idy[e];
        const double t0 = dmax(0.0, dmin(ta, tb)), t1 = dmin(1.0, dmax(ta, tb));
        if (!(t1 > t0)) continue;
        double integ;
        if (dx == 0.0) {
            integ = (t1 - t0) * clamp01(px);
        } else {
            const double sa = -px * idx[e], sb = (1.0 - px) * idx[e];
            const double ua = dmax(t0, dmin(sa, sb)), ub = dmin(t1, dmax(sa, sb));
            const double mid = (ub > ua) ? (ub - ua) * clamp01(fma(0.5 * (ua + ub), dx, px)) : 0.0;
            const double over = (dx > 0.0) ? dmax(0.0, t1 - dmax(sb, t0)) : dmax(0.0, dmin(sb, t1) - t0);
            integ = mid + over;
        }
        s = fma(dy, integ, s);
    }
    return s;
}

// Apportions n <= 32 general triangles, entry i at ent + ((head + i) & mask) * QENT.  Lane = triangle for the
// set-up; then the pixels of all the (clipped) bounding boxes of the batch are spread evenly over the lanes,
// each clipped exactly against its triangle.  With WALK_BIG, triangles whose box holds more than S.small_px
// pixels are left out and reported in the returned lane mask (the caller walks their edges: cost ~ perimeter).
// `done` counts the pixels this lane clipped.
template <bool WALK_BIG>
__device__ __forceinline__ unsigned apportion_batch(const ShootDev &S, const Win &W, double (*rec)[10], const double *ent, int head, int mask,
                                                    int n, int &done) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    int npx = 0;
    bool big = false;
    if (lane < n) {
        const double *v = ent + (size_t)((head + lane) & mask) * QENT;
        const double u0 = v[0], v0 = v[1], u1 = v[2], v1 = v[3], u2 = v[4], v2 = v[5];
        const double nan_probe = (u0 + u1 + u2) + (v0 + v1 + v2);                // NaN if any is (or if infinities cancel)
        const double mnx = dmin(u0, dmin(u1, u2)), mxx = dmax(u0, dmax(u1, u2));
        const double mny = dmin(v0, dmin(v1, v2)), mxy = dmax(v0, dmax(v1, v2));
        const bool sane = (nan_probe == nan_probe) && (mxx >= 0.0) && (mxy >= 0.0) && (mnx < (double)S.npix1) && (mny < (double)S.npix2) &&
                          (mnx > -1.0e9) && (mny > -1.0e9) && (mxx < 1.0e9) && (mxy < 1.0e9);      // false for NaN too
        if (sane) {
            const double fbx = floor(mnx), fby = floor(mny);
            const double x0 = u0 - fbx, y0 = v0 - fby, x1 = u1 - fbx, y1 = v1 - fby, x2 = u2 - fbx, y2 = v2 - fby;
            const double A2 = (x1 - x0) * (y2 - y0) - (x2 - x0) * (y1 - y0);
            if (A2 == 0.0) {                                    // reading G12: whole weight to the pixel of vertex 0
                pix_add(S, W, floor_to_int(u0), floor_to_int(v0), FIX_ONE);
            } else {
                const int lox = max((int)fbx, 0), hix = min((int)floor(mxx), S.npix1 - 1);
                const int loy = max((int)fby, 0), hiy = min((int)floor(mxy), S.npix2 - 1);
                const long long wc = (long long)hix - lox + 1, hc = (long long)hiy - loy + 1;
                if (wc > 0 && hc > 0) {
                    big = WALK_BIG && (wc * hc > (long long)S.small_px);
                    if (!big) {
                        const double dx0 = x1 - x0, dx1 = x2 - x1, dx2 = x0 - x2, dy0 = y1 - y0, dy1 = y2 - y1, dy2 = y0 - y2;
                        const double idx[3] = {(dx0 != 0.0) ? fast_rcp(fabs(dx0)) * (dx0 < 0.0 ? -1.0 : 1.0) : 0.0,
                                               (dx1 != 0.0) ? fast_rcp(fabs(dx1)) * (dx1 < 0.0 ? -1.0 : 1.0) : 0.0,
                                               (dx2 != 0.0) ? fast_rcp(fabs(dx2)) * (dx2 < 0.0 ? -1.0 : 1.0) : 0.0};
                        const double idy[3] = {(dy0 != 0.0) ? fast_rcp(fabs(dy0)) * (dy0 < 0.0 ? -1.0 : 1.0) : 0.0,
                                               (dy1 != 0.0) ? fast_rcp(fabs(dy1)) * (dy1 < 0.0 ? -1.0 : 1.0) : 0.0,
                                               (dy2 != 0.0) ? fast_rcp(fabs(dy2)) * (dy2 < 0.0 ? -1.0 : 1.0) : 0.0};
                        if (wc == 2 && hc == 2 && mxx - fbx < 2.0 && mxy - fby < 2.0 && fbx >= 0.0 && fby >= 0.0) {
                            // the commonest general triangle, four pixels around one grid corner: one clipped pixel
                            // and the two line fractions give all four by inclusion-exclusion
                            const double xs[3] = {x0, x1, x2}, ys[3] = {y0, y1, y2};
                            const double f00 = tri_pixel_area(xs, ys, idx, idy, 0.0, 0.0) * (2.0 / A2);
                            const double fl = frac_below(x0 - 1.0, x1 - 1.0, x2 - 1.0), fb = frac_below(y0 - 1.0, y1 - 1.0, y2 - 1.0);
                            const unsigned long long a00 = to_fix(f00), a10 = to_fix(fb - f00), a01 = to_fix(fl - f00);
                            const unsigned long long rest = a00 + a10 + a01;
                            pix_add(S, W, lox, loy, a00);
                            pix_add(S, W, lox + 1, loy, a10);
                            pix_add(S, W, lox, loy + 1, a01);
                            pix_add(S, W, lox + 1, loy + 1, rest < FIX_ONE ? FIX_ONE - rest : 0ull);
                            done += 4;
                        } else {
                            npx = (int)((wc * hc < (1ll << 26)) ? wc * hc : (1ll << 26));   // (only a full queue can bring such boxes here)
                            double *rc = rec[lane];
                            rc[0] = 2.0 / A2;
                            rc[1] = __hiloint2double(loy, lox);
                            rc[2] = __hiloint2double((int)fby, (int)fbx);
                            rc[3] = __hiloint2double(0, (int)wc);
                            rc[4] = idx[0]; rc[5] = idx[1]; rc[6] = idx[2]; rc[7] = idy[0]; rc[8] = idy[1]; rc[9] = idy[2];
                        }
                    }
                }
            }
        }
    }
    int inc = npx;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(full, inc, o); if (lane >= o) inc += t; }
    const int total = __shfl_sync(full, inc, 31);
    const unsigned bigmask = __ballot_sync(full, big);
    __syncwarp();
#pragma unroll 1
    for (int k0 = 0; k0 < total; k0 += 32) {
        const int k = k0 + lane;
        int i = 0;                                              // first triangle whose inclusive prefix exceeds k
#pragma unroll
        for (int step = 16; step; step >>= 1) {
            int v = __shfl_sync(full, inc, (i + step - 1) & 31);
            if (v <= k) i += step;
        }
        i &= 31;
        const int incl = __shfl_sync(full, inc, i), cnt = __shfl_sync(full, npx, i);
        if (k < total) {
            const int m = k - (incl - cnt);
            const double *v = ent + (size_t)((head + i) & mask) * QENT;
            const double *rc = rec[i];
            const int lox = __double2loint(rc[1]), loy = __double2hiint(rc[1]);
            const int bx = __double2loint(rc[2]), by = __double2hiint(rc[2]);
            const int wc = __double2loint(rc[3]);
            const int py = loy + m / wc, px = lox + m % wc;
            const double fbx = (double)bx, fby = (double)by;
            const double x[3] = {v[0] - fbx, v[2] - fbx, v[4] - fbx}, y[3] = {v[1] - fby, v[3] - fby, v[5] - fby};
            const double idx[3] = {rc[4], rc[5], rc[6]}, idy[3] = {rc[7], rc[8], rc[9]};
            const double a = tri_pixel_area(x, y, idx, idy, (double)(px - bx), (double)(py - by));
            pix_add(S, W, px, py, to_fix(a * rc[0]));
            ++done;
        }
    }
    __syncwarp();
    return bigmask;
}

// Warp-cooperative edge walk of one large triangle (v = its 3 vertices in pixel units, same in all lanes): the cold
// copy, for the triangles that found the walk list or the queue full.  Lanes 0-2 set up one edge each into `scratch`
// (3 x EREC doubles of the warp's shared memory); then the lanes take runs of consecutive steps of each edge in turn.
static const int RUN = 4;             // consecutive steps of an edge a lane walks at a time
__device__ __forceinline__ unsigned long long walk_triangle(const ShootDev &S, const double (&v)[QENT], double *scratch) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    Win W; W.w32 = nullptr; W.ax = 0; W.ay = 0;
    TriSetup T;
    T.status = 0;
    if (lane == 0) tri_setup(S, W, v, T);                      // the degenerate case deposits: one lane only
    const int status = __shfl_sync(full, T.status, 0);
    if (status != 1) return 0ull;
    const double cs = __shfl_sync(full, T.cs, 0);
    const int by = __shfl_sync(full, T.by, 0);
    __syncwarp();
    if (lane < 3) {
        const double xa = (lane == 0) ? v[0] : (lane == 1) ? v[2] : v[4], ya = (lane == 0) ? v[1] : (lane == 1) ? v[3] : v[5];
        const double xb = (lane == 0) ? v[2] : (lane == 1) ? v[4] : v[0], yb = (lane == 0) ? v[3] : (lane == 1) ? v[5] : v[1];
        EdgeWalk E;
        edge_setup_canon(S, E, xa, ya, xb, yb);
        edge_record(E, cs, by, scratch + EREC * lane);
    }
    __syncwarp();
    unsigned long long total = 0;
#pragma unroll 1
    for (int e = 0; e < 3; ++e) {
        const double *q = scratch + EREC * e;
        const int n = edge_record_steps(q);
        total += (unsigned long long)n;
#pragma unroll 1
        for (int m0 = lane * RUN; m0 < n; m0 += 32 * RUN) edge_run(S, q, m0, min(m0 + RUN, n));
    }
    __syncwarp();
    return total;
}

// The shooting kernel's own copy, for the triangles it could not hand to the global queue (queue full).
// Out of line, cold.
static __device__ __noinline__ int tri_batch(const ShootDev *Sp, unsigned int *w32, int ax, int ay, WarpSharedIpm *Wsp, int head, int n) {
    Win W; W.w32 = w32; W.ax = ax; W.ay = ay;
    int done = 0;
    __syncwarp();
    unsigned big = apportion_batch<true>(*Sp, W, Wsp->rec(), &Wsp->ringE[0][0], head, 7, n, done);
    while (big) {
        const int i = __ffs(big) - 1;
        big &= big - 1;
        double v[QENT];
#pragma unroll
        for (int k = 0; k < QENT; ++k) v[k] = Wsp->ringE[(head + i) & 7][k];
        walk_triangle(*Sp, v, &Wsp->rec()[0][0]);
    }
    return done;
}

}  // namespace ml
