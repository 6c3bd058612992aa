// shoot.cu -- the two hot loops of the method, fused: evaluate the lens equation on a tile of the ray
// grid (near-field P2P + local Taylor series + macro + sheet, eq 12/23/24) and deposit the mapped cells
// into the source-plane map without ever writing the rays to HBM.
//   IPM: cell -> 2 triangles -> exact area apportioning over the pixel grid.
//   IRS:     one ray per cell centre -> count.
// Accumulation is integer: the map is a u64 array in units of 2^-FIXBITS of one whole triangle (IPM)
// or of one ray (IRS); integer adds commute, so maps are bit-reproducible whatever the atomic order.
#include "device.cuh"
#include <math.h>
#include <stdlib.h>

namespace ml {

static const int TCX = 32;            // corners per tile row (= warp width)
static const int TCY = 32;            // corner rows per tile
static const int NWARP = 8;           // 256 threads
static const int WW = 32, WH = 32;    // shared-memory pixel window of a tile
static const int FIXBITS = 36;
static const int SMALL_MAX = 16;      // triangles whose clipped bounding box has <= this many pixels stay in-thread
static const int CHUNK_PX = 4096;     // pixels of bounding box per queue chunk
static const int QENT = 8;            // doubles per queue entry

enum { C_QUEUE = 0, C_SINGLE, C_SMALL, C_QUEUED, C_CHUNKS, C_OVERFLOW, C_FALLBACK, C_RAYS, C_NEAR, C_NCOUNTERS };

struct ShootDev {
    LensDev L;
    double x0_1, x0_2, h1, h2;
    long long i0, i1, j0, j1;          // cell sub-range
    double ylo1, ylo2, p1, p2, inv_p1, inv_p2;
    int npix1, npix2;
    unsigned long long *acc;
    double *queue;
    unsigned long long *counters;
    long long queue_cap;
    double *dump1, *dump2;
    int eval_mode;
    int ntx;                           // tiles along x1
    long long tile_row0, tile_rows;    // band of tile rows handled by this launch
};

__device__ __forceinline__ double corner_x(const ShootDev &S, long long i) { return __dadd_rn(S.x0_1, __dmul_rn((double)i, S.h1)); }
__device__ __forceinline__ double corner_y(const ShootDev &S, long long j) { return __dadd_rn(S.x0_2, __dmul_rn((double)j, S.h2)); }

__device__ __forceinline__ int floor_to_int(double u) {
    return (int)floor(fmin(fmax(u, -1.0e9), 1.0e9));      // NaN -> -1e9
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

__device__ __forceinline__ void add_fraction(const ShootDev &S, int px, int py, double frac) {
    long long v = __double2ll_rn(frac * (double)(1ull << FIXBITS));
    if (v > 0) atomicAdd(&S.acc[(size_t)py * S.npix1 + px], (unsigned long long)v);
}

struct TriBox {
    double bx, by, A;
    int lox, hix, loy, hiy;
    TriEdges E;
};

// returns 0: nothing to deposit, 1: degenerate handled, 2: box ready
__device__ __forceinline__ int tri_prepare(const ShootDev &S, double u0, double v0, double u1, double v1,
                                           double u2, double v2, TriBox &B) {
    double mnx = fmin(u0, fmin(u1, u2)), mxx = fmax(u0, fmax(u1, u2));
    double mny = fmin(v0, fmin(v1, v2)), mxy = fmax(v0, fmax(v1, v2));
    if (!(mxx >= 0.0) || !(mxy >= 0.0) || !(mnx < (double)S.npix1) || !(mny < (double)S.npix2)) return 0;
    if (!(mnx > -1.0e15) || !(mny > -1.0e15) || !(mxx < 1.0e15) || !(mxy < 1.0e15)) return 0;   // inf / absurd
    if (u0 != u0 || u1 != u1 || u2 != u2 || v0 != v0 || v1 != v1 || v2 != v2) return 0;
    B.bx = floor(mnx); B.by = floor(mny);
    double x0 = u0 - B.bx, y0 = v0 - B.by, x1 = u1 - B.bx, y1 = v1 - B.by, x2 = u2 - B.bx, y2 = v2 - B.by;
    B.A = 0.5 * ((x1 - x0) * (y2 - y0) - (x2 - x0) * (y1 - y0));
    if (B.A == 0.0) {                                   // reading G12: whole weight to the pixel of vertex 0
        double fx = floor(u0), fy = floor(v0);
        if (fx >= 0.0 && fx < (double)S.npix1 && fy >= 0.0 && fy < (double)S.npix2)
            add_fraction(S, (int)fx, (int)fy, 1.0);
        return 1;
    }
    B.lox = (int)fmax(B.bx, 0.0); B.hix = (int)fmin(floor(mxx), (double)S.npix1 - 1.0);
    B.loy = (int)fmax(B.by, 0.0); B.hiy = (int)fmin(floor(mxy), (double)S.npix2 - 1.0);
    tri_setup(B.E, x0, y0, x1, y1, x2, y2);
    return 2;
}

// every pixel of the clipped bounding box, one by one (small triangles; queue-overflow fallback)
__device__ __noinline__ void tri_deposit_loop(const ShootDev &S, const TriBox &B) {
    double invA = 1.0 / B.A;
    for (int py = B.loy; py <= B.hiy; ++py)
        for (int px = B.lox; px <= B.hix; ++px) {
            double a = tri_pixel_area(B.E, (double)px - B.bx, (double)py - B.by);
            add_fraction(S, px, py, a * invA);
        }
}

struct ThreadCounters { unsigned int single = 0, small_ = 0, queued = 0, chunks = 0, overflow = 0, fallback = 0, rays = 0, near_ = 0; };

__device__ __forceinline__ void deposit_general(const ShootDev &S, double u0, double v0, double u1, double v1,
                                                double u2, double v2, ThreadCounters &tc) {
    TriBox B;
    int st = tri_prepare(S, u0, v0, u1, v1, u2, v2, B);
    if (st != 2) { if (st == 1) ++tc.small_; return; }
    long long w = (long long)B.hix - B.lox + 1, h = (long long)B.hiy - B.loy + 1;
    if (w <= 0 || h <= 0) return;
    if (w * h <= SMALL_MAX) { ++tc.small_; tri_deposit_loop(S, B); return; }
    long long rows_per = CHUNK_PX / w; if (rows_per < 1) rows_per = 1;
    long long nch = (h + rows_per - 1) / rows_per;
    unsigned long long old = atomicAdd(&S.counters[C_QUEUE], (unsigned long long)nch);
    if ((long long)old + nch > S.queue_cap) {
        atomicAdd(&S.counters[C_QUEUE], (unsigned long long)(-nch));
        ++tc.overflow;
        tri_deposit_loop(S, B);
        return;
    }
    ++tc.queued; tc.chunks += (unsigned int)nch;
    for (long long c = 0; c < nch; ++c) {
        double *q = S.queue + (size_t)(old + c) * QENT;
        int r0 = B.loy + (int)(c * rows_per), r1 = min(B.hiy + 1, r0 + (int)rows_per);
        q[0] = u0; q[1] = v0; q[2] = u1; q[3] = v1; q[4] = u2; q[5] = v2;
        q[6] = __hiloint2double(r1, r0); q[7] = 0.0;
    }
}

__device__ __forceinline__ void flush_counters(const ShootDev &S, ThreadCounters &tc) {
    unsigned int v[8] = {tc.single, tc.small_, tc.queued, tc.chunks, tc.overflow, tc.fallback, tc.rays, tc.near_};
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        unsigned int x = v[k];
        for (int o = 16; o; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) == 0 && x) atomicAdd(&S.counters[C_SINGLE + k], (unsigned long long)x);
    }
}

// ------------------------------------------------------------------------------------------------
// Per-tile cache of up to four leaves (a tile is smaller than a leaf, so it touches at most 2x2 of them)
struct LeafCache {
    double nx[4][ML_NEAR], ny[4][ML_NEAR], nm[4][ML_NEAR];
    double2 ec[4][ML_P1MAX];
    double cx[4], cy[4], invh[4];
    uint32_t bx0[4], bx1[4], by0[4], by1[4];
    int cnt[4], leaf[4];
};

__device__ __forceinline__ void cache_find(const ShootDev &S, LeafCache &C, int slot, double x, double y) {
    uint32_t qx, qy;
    C.leaf[slot] = -1; C.cnt[slot] = 0;
    C.bx0[slot] = C.bx1[slot] = C.by0[slot] = C.by1[slot] = 0;
    if (!quantise(S.L, x, y, qx, qy)) return;
    int node = find_leaf_node(S.L, qx, qy);
    int lev = S.L.level[node], ix = S.L.ix[node], iy = S.L.iy[node];
    int sh = ML_QBITS - lev;
    C.leaf[slot] = S.L.leaf_id[node];
    C.bx0[slot] = (uint32_t)ix << sh; C.bx1[slot] = (uint32_t)(ix + 1) << sh;
    C.by0[slot] = (uint32_t)iy << sh; C.by1[slot] = (uint32_t)(iy + 1) << sh;
    double half = S.L.root_half / (double)(1 << lev);
    C.cx[slot] = -S.L.root_half + (2.0 * ix + 1.0) * half;
    C.cy[slot] = -S.L.root_half + (2.0 * iy + 1.0) * half;
    C.invh[slot] = 1.0 / half;
    C.cnt[slot] = S.L.near_cnt[C.leaf[slot]];
}

__device__ __forceinline__ void cache_fill(const ShootDev &S, LeafCache &C) {
    int t = threadIdx.x;
    if (t < 4 * ML_NEAR) {
        int slot = t / ML_NEAR, e = t % ML_NEAR;
        int leaf = C.leaf[slot];
        bool v = leaf >= 0 && e < C.cnt[slot];
        size_t o = (size_t)(leaf < 0 ? 0 : leaf) * ML_NEAR + e;
        C.nx[slot][e] = v ? S.L.near_x[o] : 0.0;
        C.ny[slot][e] = v ? S.L.near_y[o] : 0.0;
        C.nm[slot][e] = v ? S.L.near_m[o] : 0.0;
    }
    for (int k = t; k < 4 * S.L.p1; k += blockDim.x) {
        int slot = k / S.L.p1, l = k % S.L.p1;
        int leaf = C.leaf[slot];
        C.ec[slot][l] = (leaf >= 0) ? S.L.ecoef[(size_t)leaf * S.L.p1 + l] : make_double2(0.0, 0.0);
    }
}

// w(z) of eq 12 for one ray of the tile
__device__ __forceinline__ void eval_ray(const ShootDev &S, const LeafCache &C, double x, double y,
                                         double &wx, double &wy, ThreadCounters &tc) {
    double ax, ay;
    ++tc.rays;
    if (S.eval_mode == MLENS_EVAL_DIRECT) {
        direct_all(S.L, x, y, ax, ay);
        ax *= S.L.theta2; ay *= S.L.theta2;
    } else {
        uint32_t qx, qy;
        int slot = -1;
        if (quantise(S.L, x, y, qx, qy)) {
#pragma unroll
            for (int s = 0; s < 4; ++s)
                if (C.leaf[s] >= 0 && qx >= C.bx0[s] && qx < C.bx1[s] && qy >= C.by0[s] && qy < C.by1[s]) slot = s;
        }
        if (slot >= 0) {
            double nx_, ny_, fx, fy;
            tc.near_ += (unsigned int)C.cnt[slot];
            near_sum(C.nx[slot], C.ny[slot], C.nm[slot], C.cnt[slot], x, y, nx_, ny_);
            far_horner(C.ec[slot], S.L.p, (x - C.cx[slot]) * C.invh[slot], (y - C.cy[slot]) * C.invh[slot], fx, fy);
            ax = fma(S.L.theta2, nx_, fx);
            ay = fma(S.L.theta2, ny_, fy);
        } else {
            ++tc.fallback;
            alpha_fmm_global(S.L, x, y, ax, ay);
        }
    }
    lens_w(S.L, x, y, ax, ay, wx, wy);
}

// Adds `cnt` to the run of equal keys among consecutive lanes with one shared-memory atomic per run.
__device__ __forceinline__ void window_add_rle(unsigned int *win, int key, unsigned int cnt) {
    const unsigned full = 0xffffffffu;
    int lane = threadIdx.x & 31;
    int prev = __shfl_up_sync(full, key, 1);
    bool head = (lane == 0) || (key != prev);
    unsigned heads = __ballot_sync(full, head);
    if (head && key >= 0) {
        unsigned above = (lane == 31) ? 0u : (heads & ~((2u << lane) - 1u));
        int next = above ? (__ffs(above) - 1) : 32;
        atomicAdd(&win[key], cnt * (unsigned int)(next - lane));
    }
}

__global__ void __launch_bounds__(NWARP * 32) shoot_ipm_kernel(ShootDev S) {
    __shared__ double su[TCY * TCX], sv[TCY * TCX];
    __shared__ int spx[TCY * TCX], spy[TCY * TCX];
    __shared__ LeafCache C;
    __shared__ unsigned int win[WH * WW];
    __shared__ unsigned short list[2 * (TCX - 1) * (TCY - 1)];
    __shared__ int list_n, wax, way;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ThreadCounters tc;
    const long long ntiles = (long long)S.ntx * S.tile_rows;
    const long long ncx = S.i1 - S.i0 + 1;               // corners per dump row

    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        long long ty = S.tile_row0 + tile / S.ntx;
        int tx = (int)(tile % S.ntx);
        long long ci0 = S.i0 + (long long)tx * (TCX - 1), cj0 = S.j0 + ty * (TCY - 1);
        long long ci1 = min(ci0 + TCX - 1, S.i1), cj1 = min(cj0 + TCY - 1, S.j1);   // last corner of the tile

        // ---- leaves of the four extreme corners
        if (threadIdx.x < 4 && S.eval_mode == MLENS_EVAL_FMM)
            cache_find(S, C, threadIdx.x, corner_x(S, (threadIdx.x & 1) ? ci1 : ci0), corner_y(S, (threadIdx.x & 2) ? cj1 : cj0));
        if (threadIdx.x == 0) list_n = 0;
        for (int k = threadIdx.x; k < WH * WW; k += blockDim.x) win[k] = 0u;
        __syncthreads();
        if (S.eval_mode == MLENS_EVAL_FMM) cache_fill(S, C);
        __syncthreads();

        // ---- hot loop A: map the corners (eq 12)
        for (int row = warp; row < TCY; row += NWARP) {
            long long ci = ci0 + lane, cj = cj0 + row;
            int o = row * TCX + lane;
            if (ci <= S.i1 && cj <= S.j1) {
                double wx, wy;
                eval_ray(S, C, corner_x(S, ci), corner_y(S, cj), wx, wy, tc);
                if (S.dump1) {
                    size_t d = (size_t)(cj - S.j0) * ncx + (size_t)(ci - S.i0);
                    S.dump1[d] = wx; S.dump2[d] = wy;
                }
                double u = (wx - S.ylo1) * S.inv_p1, v = (wy - S.ylo2) * S.inv_p2;
                su[o] = u; sv[o] = v;
                spx[o] = floor_to_int(u); spy[o] = floor_to_int(v);
            } else {
                su[o] = 0.0; sv[o] = 0.0; spx[o] = 0; spy[o] = 0;
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int rc = (int)min((long long)(TCY / 2), cj1 - cj0), cc = (int)min((long long)(TCX / 2), ci1 - ci0);
            wax = spx[rc * TCX + cc] - WW / 2; way = spy[rc * TCX + cc] - WH / 2;
        }
        __syncthreads();

        // ---- hot loop B, part 1: cells whose triangles sit inside one pixel are just counted
        for (int row = warp; row < TCY - 1; row += NWARP) {
            long long ci = ci0 + lane, cj = cj0 + row;
            bool valid = (lane < TCX - 1) && (ci < S.i1) && (cj < S.j1);
            int o = row * TCX + lane;
            int key = -1;
            if (valid) {
                int ax = spx[o], ay = spy[o], bx = spx[o + 1], by = spy[o + 1];
                int cx = spx[o + TCX + 1], cy = spy[o + TCX + 1], dx = spx[o + TCX], dy = spy[o + TCX];
                bool t1 = (ax == bx) && (ax == cx) && (ay == by) && (ay == cy);
                bool t2 = (ax == cx) && (ax == dx) && (ay == cy) && (ay == dy);
                bool inmap = ax >= 0 && ax < S.npix1 && ay >= 0 && ay < S.npix2;
                if (t1 && t2) {
                    tc.single += 2;
                    if (inmap) {
                        int lx = ax - wax, ly = ay - way;
                        if (lx >= 0 && lx < WW && ly >= 0 && ly < WH) key = ly * WW + lx;
                        else atomicAdd(&S.acc[(size_t)ay * S.npix1 + ax], 2ull << FIXBITS);
                    }
                } else {
                    if (t1 || t2) {
                        ++tc.single;
                        if (inmap) {
                            int lx = ax - wax, ly = ay - way;
                            if (lx >= 0 && lx < WW && ly >= 0 && ly < WH) atomicAdd(&win[ly * WW + lx], 1u);
                            else atomicAdd(&S.acc[(size_t)ay * S.npix1 + ax], 1ull << FIXBITS);
                        }
                    }
                    int slot = atomicAdd(&list_n, (t1 || t2) ? 1 : 2);
                    unsigned short id = (unsigned short)((row * (TCX - 1) + lane) << 1);
                    if (!t1) list[slot++] = id;
                    if (!t2) list[slot] = id | 1;
                }
            }
            window_add_rle(win, key, 2u);
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
            deposit_general(S, su[o], sv[o], su[o1], sv[o1], su[o2], sv[o2], tc);
        }
        // ---- flush the window
        for (int k = threadIdx.x; k < WH * WW; k += blockDim.x) {
            unsigned int c = win[k];
            if (c) atomicAdd(&S.acc[(size_t)(way + k / WW) * S.npix1 + (wax + k % WW)], (unsigned long long)c << FIXBITS);
        }
        __syncthreads();
    }
    flush_counters(S, tc);
}

// Cooperative apportioning of the queued large triangles: one warp per row chunk, lanes across the
// pixels of each row's span; interior pixels get the constant 1/|A| without clipping.
__global__ void __launch_bounds__(256) drain_kernel(ShootDev S) {
    const int lane = threadIdx.x & 31;
    long long nq = (long long)S.counters[C_QUEUE];
    if (nq > S.queue_cap) nq = S.queue_cap;
    long long wid = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5, nw = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long q = wid; q < nq; q += nw) {
        const double *e = S.queue + (size_t)q * QENT;
        TriBox B;
        if (tri_prepare(S, e[0], e[1], e[2], e[3], e[4], e[5], B) != 2) continue;
        int r0 = __double2loint(e[6]), r1 = __double2hiint(e[6]);
        double sgn = (B.A > 0.0) ? 1.0 : -1.0, invA = 1.0 / B.A;
        double inner = fabs(invA);
        // edge functions F_e(x,y) = sgn (dx_e (y - py_e) - dy_e (x - px_e)) >= 0 inside
        double m0[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) m0[k] = fmin(0.0, sgn * B.E.dx[k]) + fmin(0.0, -sgn * B.E.dy[k]);
        for (int py = r0; py < r1; ++py) {
            double yl = (double)py - B.by;                 // strip [yl, yl+1] in local coordinates
            double xmin = 1.0e300, xmax = -1.0e300;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                double vy = B.E.py[k];
                if (vy >= yl && vy <= yl + 1.0) { xmin = fmin(xmin, B.E.px[k]); xmax = fmax(xmax, B.E.px[k]); }
                if (B.E.dy[k] != 0.0) {
                    double ta = (yl - vy) * B.E.idy[k], tb = (yl + 1.0 - vy) * B.E.idy[k];
                    if (ta >= 0.0 && ta <= 1.0) { double xx = fma(ta, B.E.dx[k], B.E.px[k]); xmin = fmin(xmin, xx); xmax = fmax(xmax, xx); }
                    if (tb >= 0.0 && tb <= 1.0) { double xx = fma(tb, B.E.dx[k], B.E.px[k]); xmin = fmin(xmin, xx); xmax = fmax(xmax, xx); }
                }
            }
            if (!(xmax >= xmin)) continue;
            int xs = max(B.lox, (int)fmax(floor(xmin - 1e-6) + B.bx, -1.0e9));
            int xe = min(B.hix, (int)fmin(floor(xmax + 1e-6) + B.bx, 1.0e9));
            for (int px = xs + lane; px <= xe; px += 32) {
                double qx = (double)px - B.bx;
                bool interior = true;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    double F = sgn * (B.E.dx[k] * (yl - B.E.py[k]) - B.E.dy[k] * (qx - B.E.px[k]));
                    interior = interior && (F + m0[k] >= 0.0);
                }
                double frac = interior ? inner : tri_pixel_area(B.E, qx, yl) * invA;
                add_fraction(S, px, py, frac);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// IRS: rays at cell centres (reading G10), floor of a true division (O5), counts.
__global__ void __launch_bounds__(NWARP * 32) shoot_irs_kernel(ShootDev S) {
    __shared__ LeafCache C;
    __shared__ unsigned int win[WH * WW];
    __shared__ int wax, way, anchor_set;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ThreadCounters tc;
    const long long ntiles = (long long)S.ntx * S.tile_rows;
    const long long nrx = S.i1 - S.i0;

    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        long long ty = S.tile_row0 + tile / S.ntx;
        int tx = (int)(tile % S.ntx);
        long long ci0 = S.i0 + (long long)tx * TCX, cj0 = S.j0 + ty * TCY;
        long long ci1 = min(ci0 + TCX, S.i1) - 1, cj1 = min(cj0 + TCY, S.j1) - 1;      // last cell of the tile
        if (threadIdx.x < 4 && S.eval_mode == MLENS_EVAL_FMM)
            cache_find(S, C, threadIdx.x, corner_x(S, (threadIdx.x & 1) ? ci1 : ci0) + 0.5 * S.h1,
                       corner_y(S, (threadIdx.x & 2) ? cj1 : cj0) + 0.5 * S.h2);
        for (int k = threadIdx.x; k < WH * WW; k += blockDim.x) win[k] = 0u;
        if (threadIdx.x == 0) anchor_set = 0;
        __syncthreads();
        if (S.eval_mode == MLENS_EVAL_FMM) cache_fill(S, C);
        __syncthreads();
        // the window is anchored on the tile's central ray, mapped first by warp 0
        int px[TCY / NWARP], py[TCY / NWARP];
#pragma unroll
        for (int r = 0; r < TCY / NWARP; ++r) {
            int row = warp + r * NWARP;
            long long ci = ci0 + lane, cj = cj0 + row;
            px[r] = -1; py[r] = -1;
            if (ci < S.i1 && cj < S.j1) {
                double wx, wy;
                eval_ray(S, C, corner_x(S, ci) + 0.5 * S.h1, corner_y(S, cj) + 0.5 * S.h2, wx, wy, tc);
                if (S.dump1) {
                    size_t d = (size_t)(cj - S.j0) * nrx + (size_t)(ci - S.i0);
                    S.dump1[d] = wx; S.dump2[d] = wy;
                }
                double fx = floor((wx - S.ylo1) / S.p1), fy = floor((wy - S.ylo2) / S.p2);
                if (fx >= 0.0 && fx < (double)S.npix1 && fy >= 0.0 && fy < (double)S.npix2) { px[r] = (int)fx; py[r] = (int)fy; }
                if (atomicCAS(&anchor_set, 0, 1) == 0) { wax = (int)fmin(fmax(fx, -1e9), 1e9) - WW / 2; way = (int)fmin(fmax(fy, -1e9), 1e9) - WH / 2; }
            }
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < TCY / NWARP; ++r) {
            int key = -1;
            if (px[r] >= 0) {
                ++tc.single;
                int lx = px[r] - wax, ly = py[r] - way;
                if (lx >= 0 && lx < WW && ly >= 0 && ly < WH) key = ly * WW + lx;
                else atomicAdd(&S.acc[(size_t)py[r] * S.npix1 + px[r]], 1ull);
            }
            window_add_rle(win, key, 1u);
        }
        __syncthreads();
        for (int k = threadIdx.x; k < WH * WW; k += blockDim.x) {
            unsigned int c = win[k];
            if (c) atomicAdd(&S.acc[(size_t)(way + k / WW) * S.npix1 + (wax + k % WW)], (unsigned long long)c);
        }
        __syncthreads();
    }
    flush_counters(S, tc);
}

// ------------------------------------------------------------------------------------------------
__global__ void finalise_kernel(const unsigned long long *acc, long long n, double scale, int accumulate,
                                double *map, unsigned long long *counts) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    unsigned long long a = acc[i];
    if (map) { double v = (double)a * scale; map[i] = accumulate ? map[i] + v : v; }
    if (counts) counts[i] = accumulate ? counts[i] + a : a;
}

// Geometry of the shooting window and ray grid: eq 14-16, eq A6; O1/O2.
int geometry(const mlens_field *f, const mlens_shoot_desc *d, mlens_grid *g) {
    double a1 = 1.0 - f->kappa_tot + f->gamma, a2 = 1.0 - f->kappa_tot - f->gamma;
    if (a1 == 0.0 || a2 == 0.0) { set_error("macro model is singular (1-kappa+-gamma = 0)"); return MLENS_EINVAL; }
    if (d->npix1 <= 0 || d->npix2 <= 0 || !(d->rays_per_pixel_length > 0) || !(d->half_y1 > 0) || !(d->half_y2 > 0)) {
        set_error("bad map description"); return MLENS_EINVAL;
    }
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
    S.acc = f->acc.p; S.queue = f->queue.p; S.counters = f->counters.p; S.queue_cap = qcap;
    S.dump1 = d->dump_w1; S.dump2 = d->dump_w2;
    if ((S.dump1 == nullptr) != (S.dump2 == nullptr)) { set_error("dump_w1 and dump_w2 go together"); return MLENS_EINVAL; }
    S.eval_mode = d->eval_mode;
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
    for (long long r0 = 0; r0 < nty; r0 += rows_per_band, ++bands) {
        S.tile_row0 = r0;
        S.tile_rows = (nty - r0 < rows_per_band) ? (nty - r0) : rows_per_band;
        long long nt = ntx * S.tile_rows;
        int grid = (int)((nt < (long long)nsm * 16) ? nt : (long long)nsm * 16);
        ML_TRY(mark());
        if (ipm) {
            ML_LAUNCH(shoot_ipm_kernel, grid, NWARP * 32, 0, s, S);
            ML_TRY(mark());
            ML_LAUNCH(drain_kernel, nsm * 8, 256, 0, s, S);
            ML_TRY(mark());
            ML_CUDA(cudaMemsetAsync(f->counters.p, 0, 8, s));     // queue fill count only
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
    ML_LAUNCH(finalise_kernel, (unsigned)((npix + 255) / 256), 256, 0, s, f->acc.p, npix, scale, d->accumulate, map,
                                                                    ipm ? nullptr : counts);
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
            // the last band's closing event is followed by (memset,) finalise, closing event
            ML_CUDA(cudaEventElapsedTime(&ms, ev[ev.size() - 2], ev[ev.size() - 1])); st->ms_finalise = ms;
        }
    } else if (d->sync) {
        ML_CUDA(cudaStreamSynchronize(s));
    }
    for (cudaEvent_t e : ev) cudaEventDestroy(e);
    return MLENS_OK;
}

}  // namespace ml
