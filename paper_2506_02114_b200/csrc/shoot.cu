// shoot.cu -- the two hot loops of the method, fused: evaluate the lens equation on a tile of the ray
// grid (eq 12/23/24) and deposit the mapped cells into the source-plane map without ever writing the
// rays to HBM.
//   IPM: cell -> 2 triangles -> exact area apportioning over the pixel grid.
//   IRS:     one ray per cell centre -> count.
//
// Every WARP is autonomous: it takes 32 x 32-ray tiles from a global counter, builds the
// tile's own expansion (tile.cuh), evaluates four ray rows at a time, keeps the previous row in registers and
// apportions the cells between consecutive rows (deposit.cuh).  There is no block-wide barrier anywhere.
// Accumulation is integer (64-bit fixed point): the IPM map is built as its row-difference array, prefix-
// summed by finalise_kernel; per-warp shared-memory windows absorb most adds before they reach L2.
#include "deposit.cuh"
#include <math.h>
#include <stdlib.h>
#include <limits.h>
#include <mutex>

namespace ml {

static const int SHOOT_WARPS = 2;      // warps per block; blocks only share the shared-memory allocation

__device__ __forceinline__ void flush_counters(const ShootDev &S, ThreadCounters &tc) {
    // order = the C_SINGLE.. block of the counter enum, then C_PX_SMALL
    unsigned int v[9] = {tc.single, tc.small_, tc.queued, tc.chunks, tc.overflow, tc.fallback, tc.rays, tc.near_, tc.px_small};
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        unsigned int x = v[k];
#pragma unroll 1
        for (int o = 16; o; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) == 0 && x) atomicAdd(&S.counters[C_SINGLE + k], (unsigned long long)x);
    }
}

__device__ __forceinline__ long long fetch_tile(const ShootDev &S) {
    long long t = 0;
    if ((threadIdx.x & 31) == 0) t = (long long)atomicAdd(&S.counters[C_TILE], 1ull);
    return __shfl_sync(0xffffffffu, t, 0);
}

struct Pend {
    long long chunk = -1;              // queue chunk this warp is filling
    int used = 0;
};

// General triangles go to the global queue, which drain_kernel apportions at full occupancy.  A warp reserves
// QCHUNK entries at a time (one atomic per chunk); if the queue is full they stay in the warp's own ring and
// are clipped by the (cold) in-kernel copy.
__device__ __forceinline__ void queue_push(const ShootDev &S, const Win &W, WarpSharedIpm &Ws, Pend &P, bool pred, const double (&e)[6], ThreadCounters &tc) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const unsigned m = __ballot_sync(full, pred);
    if (!m) return;
    const int n = __popc(m);
    if (P.chunk < 0 || P.used + n > QCHUNK) {
        long long c = 0;
        if (lane == 0) {
            if (P.chunk >= 0) S.qcount[P.chunk] = P.used;
            c = (long long)atomicAdd(&S.counters[C_QUEUE], 1ull);
        }
        c = __shfl_sync(full, c, 0);
        P.chunk = (c < S.queue_cap) ? c : -1;
        P.used = 0;
    }
    if (P.chunk < 0) {                                          // queue full: apportioned here, 8 at a time (cold)
        if (pred) ++tc.overflow;
        unsigned rem = m;
        while (rem) {
            unsigned take = 0, t = rem;
#pragma unroll 1
            for (int k = 0; k < 8 && t; ++k) { take |= t & (0u - t); t &= t - 1; }
            const int n8 = __popc(take);
            __syncwarp();
            if (pred && ((take >> lane) & 1u)) {
                double *q = Ws.ringE[__popc(take & ((1u << lane) - 1u))];
#pragma unroll
                for (int k = 0; k < QENT; ++k) q[k] = e[k];
            }
            tc.px_small += tri_batch(&S, W.w32, W.ax, W.ay, &Ws, 0, n8);
            if (lane < n8) ++tc.small_;
            rem &= ~take;
        }
        return;
    }
    if (pred) {
        double *q = S.queue + ((size_t)P.chunk * QCHUNK + (size_t)(P.used + __popc(m & ((1u << lane) - 1u)))) * QENT;
#pragma unroll
        for (int k = 0; k < QENT; ++k) q[k] = e[k];
        ++tc.queued;
    }
    P.used += n;
}

// Optional copy of the mapped rays to the caller (tests); out of line: never part of a production run.
static __device__ __noinline__ void dump_rays(const ShootDev *Sp, long long d0, long long stride, unsigned validmask, double w0x, double w0y,
                                              double w1x, double w1y, double w2x, double w2y, double w3x, double w3y) {
    const double wx[4] = {w0x, w1x, w2x, w3x}, wy[4] = {w0y, w1y, w2y, w3y};
    for (int r = 0; r < 4; ++r)
        if ((validmask >> r) & 1u) { Sp->dump1[d0 + (long long)r * stride] = wx[r]; Sp->dump2[d0 + (long long)r * stride] = wy[r]; }
}

// Tile `t` of the band in flight -> its indices on the GLOBAL tile grid.  Column-major by default: the tiles in
// flight at any moment then form a patch of the image plane whose mapped cells fall into a patch of the map that
// L2 holds, whereas a row of tiles spans the whole width of the map.
__device__ __forceinline__ void tile_indices(const ShootDev &S, long long t, long long &tx, long long &ty) {
    long long a, b;
    if (S.colmajor) { a = t / S.tile_rows; b = t - a * S.tile_rows; }
    else { b = t / S.ntx; a = t - b * S.ntx; }
    tx = S.txb + a; ty = S.tyb + S.tile_row0 + b;
}

// The cell row between corner rows `prev` and `prev + 1` of the staged group: lane = cell column.
//   a = (prev, lane), b = (prev, lane+1), c = (prev+1, lane+1), d = (prev+1, lane);  T1 = a, b, c;  T2 = a, c, d  (reading G9)
// Triangles inside one pixel are run-length merged and added at once.  All others that can touch the map only
// leave their name (row, column, which) in the warp's list: process_pending apportions them 32 at a time at the
// end of the row group, every lane busy, from the corners still staged in shared memory.
__device__ __forceinline__ void cell_row(const ShootDev &S, const Win &W, WarpSharedIpm &Ws, int &npend, int prev, bool cellv,
                                         ThreadCounters &tc) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, l1 = min(lane + 1, 31), cur = prev + 1;
    const int pa = Ws.stp[prev][lane], pb = Ws.stp[prev][l1], pc = Ws.stp[cur][l1], pd = Ws.stp[cur][lane];
    const int oa = Ws.sto[prev][lane], ob = Ws.sto[prev][l1], oc = Ws.sto[cur][l1], od = Ws.sto[cur][lane];
    const bool t1 = (pa == pb) && (pa == pc), t2 = (pa == pc) && (pa == pd);
    {
        // single-pixel triangles: equal pixels in consecutive lanes become one deposit
        const int ns = cellv ? (int)t1 + (int)t2 : 0;
        tc.single += ns;
        const int key = (ns > 0 && oa == 0) ? pa : -1;
        const int kprev = __shfl_up_sync(full, key, 1);
        const bool head = (lane == 0) || (key != kprev);
        const unsigned heads = __ballot_sync(full, head);
        const unsigned two = __ballot_sync(full, ns == 2), one = __ballot_sync(full, ns == 1);
        if (head && key >= 0) {
            const unsigned above = (lane == 31) ? 0u : (heads & ~((2u << lane) - 1u));
            const int next = above ? (__ffs(above) - 1) : 32;
            const unsigned run = ((next == 32) ? 0xffffffffu : ((1u << next) - 1u)) & ~((1u << lane) - 1u);
            const unsigned long long n = 2ull * __popc(two & run) + __popc(one & run);
            pix_add(S, W, px_of(pa), py_of(pa), n << FIXBITS);
        }
    }
    const bool act1 = cellv && !t1 && !(oa & ob & oc), act2 = cellv && !t2 && !(oa & oc & od);
    const unsigned b1 = __ballot_sync(full, act1), b2 = __ballot_sync(full, act2);
    const unsigned lt = (1u << lane) - 1u;
    // (the two triangles of a cell next to each other, cells in lane order: neighbours in the mesh stay neighbours in the
    // queue and in the walk list, where walk_kernel pairs the edges they share)
    const int idb = (prev << 6) | (lane << 1), at = npend + __popc(b1 & lt) + __popc(b2 & lt);
    if (act1) Ws.ids[at] = idb;
    if (act2) Ws.ids[at + (act1 ? 1 : 0)] = idb | 1;
    npend += __popc(b1) + __popc(b2);
}

// Apportions the `count` listed triangles of the row group, 32 at a time.  A triangle over two adjacent pixels is
// split in closed form (the fraction of its area beyond the pixel line is the product of two edge ratios); any
// other goes to the global queue.
__device__ __forceinline__ void process_pending(const ShootDev &S, const Win &W, WarpSharedIpm &Ws, Pend &P, int count, ThreadCounters &tc) {
    const int lane = threadIdx.x & 31;
    __syncwarp();
#pragma unroll 1
    for (int h0 = 0; h0 < count; h0 += 32) {
        const bool have = h0 + lane < count;
        const int id = have ? Ws.ids[h0 + lane] : 0;
        const int tt = id & 1, c = (id >> 1) & 31, r = id >> 6, c1 = min(c + 1, 31);
        const int r2 = tt ? r + 1 : r, c3 = tt ? c : c1;                 // vertices (r, c), (r2, c1), (r + 1, c3)
        const int pa = Ws.stp[r][c], p2 = Ws.stp[r2][c1], p3 = Ws.stp[r + 1][c3];
        double e[6];
        e[0] = Ws.stu[r][c]; e[1] = Ws.stv[r][c];
        e[2] = Ws.stu[r2][c1]; e[3] = Ws.stv[r2][c1];
        e[4] = Ws.stu[r + 1][c3]; e[5] = Ws.stv[r + 1][c3];
        const int x1 = px_of(pa), x2 = px_of(p2), x3 = px_of(p3), y1 = py_of(pa), y2 = py_of(p2), y3 = py_of(p3);
        const int mnx = min(x1, min(x2, x3)), mxx = max(x1, max(x2, x3)), mny = min(y1, min(y2, y3)), mxy = max(y1, max(y2, y3));
        const int w = mxx - mnx, h = mxy - mny;
        const bool strip = have && (w + h == 1);
        queue_push(S, W, Ws, P, have && !strip, e, tc);
        if (strip) {
            const bool ay = (h == 1);                                        // pixels stacked in y
            const double line = ay ? (double)(mny + 1) : (double)(mnx + 1);
            const double A2 = (e[2] - e[0]) * (e[5] - e[1]) - (e[4] - e[0]) * (e[3] - e[1]);
            const double d0 = (ay ? e[1] : e[0]) - line, d1 = (ay ? e[3] : e[2]) - line, d2 = (ay ? e[5] : e[4]) - line;
            const unsigned long long a = (A2 == 0.0) ? ((d0 < 0.0) ? FIX_ONE : 0ull) : to_fix(frac_below(d0, d1, d2));
#pragma unroll 1
            for (int k = 0; k < 2; ++k)                             // rolled: one copy of the add in the instruction stream
                pix_add(S, W, mnx + (ay ? 0 : k), mny + (ay ? k : 0), k ? FIX_ONE - a : a);
            ++tc.small_; tc.px_small += 2;
        }
    }
    __syncwarp();
}

template <bool F32>
__global__ void __launch_bounds__(SHOOT_WARPS * 32, 8) shoot_ipm_kernel(const __grid_constant__ ShootDev S) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WarpSharedIpm &Ws = reinterpret_cast<WarpSharedIpm *>(smem_raw)[threadIdx.x >> 5];
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    ThreadCounters tc;
    Pend P;
    TileCtx C;
    Win W; W.w32 = reinterpret_cast<unsigned int *>(Ws.win); W.ax = 0; W.ay = 0;
    const long long ntiles = (long long)S.ntx * S.tile_rows;
    const long long ncx = S.i1 - S.i0 + 1;               // corners per dump row
    int npend = 0;

    // Tiles are anchored on the GLOBAL cell grid (tile (tx, ty) holds the corners [31 tx, 31 tx + 31] x [31 ty, ..]),
    // and a tile evaluates its rays whether or not they belong to the sub-range: a ray then has the same value to the
    // last bit in whatever sub-range it is shot.  Only the cells of the sub-range are deposited.
    for (long long tile = fetch_tile(S); tile < ntiles;) {
        const long long tile_next = fetch_tile(S);       // the hand-out latency hides behind this tile's work
        long long tx, ty;
        tile_indices(S, tile, tx, ty);
        const long long ci0 = tx * (TCX - 1), cj0 = ty * (TCY - 1);
        const long long ci1 = min(ci0 + TCX - 1, S.n1), cj1 = min(cj0 + TCY - 1, S.n2);   // last corner of the tile
        wtile_setup(S, Ws, C, ci0, cj0, ci1, cj1, 0.0);

        const long long ci = ci0 + lane;
        const bool colv = ci <= S.n1, cellv = (lane < TCX - 1) && (ci >= S.i0) && (ci < S.i1);
        // (a corner on a tile border is evaluated by both tiles, each with its own series: the dump takes it from the
        // tile that holds the cell to its left / below, so that it does not depend on which tile runs last)
        const bool dumpc = (ci >= S.i0) && (ci <= S.i1) && (lane > 0 || ci == S.i0);
        const double x = corner_x(S, ci), ux = ((double)lane - 0.5 * (TCX - 1)) * S.dux;
        // row groups that hold a corner row of the sub-range
        const int g_lo = (S.j0 > cj0) ? (int)((S.j0 - cj0) / RPT) : 0;
        const int g_hi = (int)((min(S.j1, cj1) - cj0) / RPT);
#pragma unroll 1
        for (int g = g_lo; g <= g_hi && g < NGRP; ++g) {
            const bool first = (g == g_lo);
            // ---- hot loop A: map RPT corner rows (eq 12)
            double y[RPT], uy[RPT], wx[RPT], wy[RPT];
            bool valid[RPT];
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const int row = g * RPT + r;
                const long long cj = cj0 + row;
                valid[r] = colv && (cj <= S.n2);
                y[r] = corner_y(S, cj);
                uy[r] = ((double)row - 0.5 * (TCY - 1)) * S.duy;
            }
            eval_rays<F32>(S, Ws, C, x, ux, y, uy, valid, wx, wy, tc);
            if (S.dump1) {
                unsigned vm = 0;
#pragma unroll
                for (int r = 0; r < RPT; ++r) {
                    const long long cj = cj0 + g * RPT + r;
                    vm |= (valid[r] && dumpc && cj >= S.j0 && cj <= S.j1 && (g * RPT + r > 0 || cj == S.j0)) ? (1u << r) : 0u;
                }
                dump_rays(&S, (cj0 + g * RPT - S.j0) * ncx + (ci - S.i0), ncx, vm,
                          wx[0], wy[0], wx[1], wy[1], wx[2], wy[2], wx[3], wy[3]);
            }
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const double u = (wx[r] - S.ylo1) * S.inv_p1, v = (wy[r] - S.ylo2) * S.inv_p2;
                const int pk = pack_px(u, v);
                Ws.stu[r + 1][lane] = u; Ws.stv[r + 1][lane] = v; Ws.stp[r + 1][lane] = pk; Ws.sto[r + 1][lane] = out_code(pk, S.npix1, S.npix2);
                if (first && r == 1) {
                    // window anchor: the tile centre extrapolated from the first two rows evaluated (any anchor is correct)
                    const double u0 = Ws.stu[1][lane], v0 = Ws.stv[1][lane];
                    const double rows = 0.5 * (TCY - 1) - (double)(g * RPT);
                    const double cu = __shfl_sync(full, u0 + rows * (u - u0), TCX / 2);
                    const double cv = __shfl_sync(full, v0 + rows * (v - v0), TCX / 2);
                    W.ax = floor_to_int(cu) - WX / 2; W.ay = floor_to_int(cv) - WY / 2;
                }
            }
            __syncwarp();
            // ---- hot loop B: the cell rows between consecutive corner rows (cell row cjp lies between corner rows cjp, cjp + 1)
#pragma unroll 1
            for (int r = first ? 1 : 0; r < RPT; ++r) {
                const long long cjp = cj0 + g * RPT + r - 1;
                if (cjp >= S.j1) break;                                  // warp-uniform
                if (cjp < S.j0) continue;
                cell_row(S, W, Ws, npend, r, cellv, tc);
            }
            process_pending(S, W, Ws, P, npend, tc);
            npend = 0;
            Ws.stu[0][lane] = Ws.stu[RPT][lane]; Ws.stv[0][lane] = Ws.stv[RPT][lane]; Ws.stp[0][lane] = Ws.stp[RPT][lane];
            Ws.sto[0][lane] = Ws.sto[RPT][lane];
            __syncwarp();
        }
        flush_window(S, Ws, W);
        __syncwarp();
        tile = tile_next;
    }
    if (lane == 0 && P.chunk >= 0) S.qcount[P.chunk] = P.used;
    flush_counters(S, tc);
}

// Apportions the queued general triangles at full occupancy: a warp takes a chunk, 32 entries at a time.
// Small boxes are clipped pixel by pixel, the pixels of the 32 triangles spread evenly over the lanes; the
// large ones (among them the faint images of the whole map that every star in the window produces) are
// walked edge by edge by the whole warp, cost ~ perimeter.
static const int DRAIN_WARPS = 8;
// (the walk list is full: cold, and out of line so that its registers are not the drain's)
static __device__ __noinline__ unsigned long long walk_triangle_ool(const ShootDev *Sp, double a0, double a1, double a2, double a3, double a4, double a5,
                                                                    double *scratch) {
    const double v[QENT] = {a0, a1, a2, a3, a4, a5};
    return walk_triangle(*Sp, v, scratch);
}
__global__ void __launch_bounds__(DRAIN_WARPS * 32, 3) drain_kernel(const __grid_constant__ ShootDev S) {
    __shared__ double rec_s[DRAIN_WARPS][32][10];
    double (*rec)[10] = rec_s[threadIdx.x >> 5];
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    long long nq = (long long)S.counters[C_QUEUE];
    if (nq > S.queue_cap) nq = S.queue_cap;
    Win W; W.w32 = nullptr; W.ax = 0; W.ay = 0;
    unsigned long long n_pieces = 0;
    int n_clipped = 0;
    while (true) {
        long long c = 0;
        if (lane == 0) c = (long long)atomicAdd(&S.counters[C_DRAIN], 1ull);
        c = __shfl_sync(full, c, 0);
        if (c >= nq) break;
        const int cnt = S.qcount[c];
        const double *base = S.queue + (size_t)c * QCHUNK * QENT;
#pragma unroll 1
        for (int b0 = 0; b0 < cnt; b0 += 32) {
            unsigned big = apportion_batch<true>(S, W, rec, base, b0, 0x7fffffff, min(32, cnt - b0), n_clipped);
            if (big) {
                // large triangles are handed on one by one (walk_kernel): a chunk from a star's tile is full of them
                const int nb = __popc(big);
                unsigned long long at = 0;
                if (lane == 0) at = atomicAdd(&S.counters[C_BIG], (unsigned long long)nb);
                at = __shfl_sync(full, at, 0);
                if ((long long)(at + nb) <= S.big_cap) {
                    if (big & (1u << lane)) S.biglist[at + __popc(big & ((1u << lane) - 1u))] = (unsigned int)(c * QCHUNK + b0 + lane);
                    big = 0;
                }
            }
            while (big) {                                       // list full: walked here
                const int i = __ffs(big) - 1;
                big &= big - 1;
                double v[QENT];
#pragma unroll
                for (int k = 0; k < QENT; ++k) v[k] = base[(size_t)(b0 + i) * QENT + k];
                n_pieces += walk_triangle_ool(&S, v[0], v[1], v[2], v[3], v[4], v[5], &rec[0][0]);
            }
        }
    }
    if (lane == 0 && n_pieces) atomicAdd(&S.counters[C_PX_EDGE], n_pieces);
    for (int o = 16; o; o >>= 1) n_clipped += __shfl_xor_sync(full, n_clipped, o);
    if (lane == 0 && n_clipped) atomicAdd(&S.counters[C_PX_INT], (unsigned long long)n_clipped);
}

// Edge walk of the large triangles the drain set aside.  A warp takes WB triangles at a time, in list order (the
// list follows the order of the tiles, so the triangles in flight at any moment deposit into neighbouring rows of
// `diff`): lane = triangle for the local frame, lane = edge for the clipped edges (records in shared memory); then the
// RUNS of consecutive steps of all the edges form one index space the lanes stride over, so the set-up is shared by a
// whole batch, a triangle of a few dozen steps costs a few dozen lane-steps, and a lane that walks consecutive steps
// computes every point of its edge once (deposit.cuh).  The next batch is fetched while this one is walked.
static const int WALK_WARPS = 8;
static const int WB = 16;              // triangles per batch
static const int GIANT_STEPS = 1024;   // a triangle with more steps than this is not walked by one warp alone
static const int GIANT_CHUNK = 512;    // but edge by edge in chunks of this many steps: 32 lanes x GIANT_RUN consecutive steps
static const int GIANT_RUN = GIANT_CHUNK / 32;
struct WalkShared {                    // per warp (dynamic shared memory: 8 warps x 7.4 KB)
    double er[3 * WB][EREC];           // edge records
    double tr[WB][8];                  // global vertices, cs, (by, bx) of the triangle's frame
    int pre[3 * WB];                   // inclusive prefix of the runs of the batch's edges
    int pad[3 * WB];
    unsigned int qi[WB];               // queue entry of each triangle
};
__global__ void __launch_bounds__(WALK_WARPS * 32, 3) walk_kernel(const __grid_constant__ ShootDev S) {
    extern __shared__ __align__(16) unsigned char walk_smem[];
    WalkShared &Wk = reinterpret_cast<WalkShared *>(walk_smem)[threadIdx.x >> 5];
    double (*er)[EREC] = Wk.er;
    double (*tr)[8] = Wk.tr;
    int *pre = Wk.pre;
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    long long nb = (long long)S.counters[C_BIG];
    if (nb > S.big_cap) nb = S.big_cap;
    const long long nbatch = (nb + WB - 1) / WB;
    Win W; W.w32 = nullptr; W.ax = 0; W.ay = 0;
    unsigned long long n_pieces = 0;
    long long b = 0;
    if (lane == 0) b = (long long)atomicAdd(&S.counters[C_WALK], 1ull);
    b = __shfl_sync(full, b, 0);
    while (b < nbatch) {
        long long bnext = 0;
        if (lane == 0) bnext = (long long)atomicAdd(&S.counters[C_WALK], 1ull);
        // ---- lane = triangle: frame and weight
        const long long it = b * WB + lane;
        int status = 0;
        unsigned int qidx = 0;
        if (lane < WB && it < nb) {
            qidx = S.biglist[it];
            const double *e = S.queue + (size_t)qidx * QENT;
            double v[QENT];
#pragma unroll
            for (int k = 0; k < QENT; ++k) v[k] = __ldg(&e[k]);
            TriSetup T;
            tri_setup(S, W, v, T);                                  // a degenerate triangle deposits here (reading G12)
            status = T.status;
            if (status == 1) {
                double *q = tr[lane];
#pragma unroll
                for (int k = 0; k < QENT; ++k) q[k] = v[k];
                q[6] = T.cs; q[7] = __hiloint2double(T.by, T.bx);
            }
        }
        if (lane < WB) Wk.qi[lane] = qidx;
        __syncwarp();
        // ---- lane = edge (3 WB of them, two passes): every edge in its own frame and canonical direction
#pragma unroll
        for (int ps = 0; ps < 2; ++ps) {
            const int ed = ps * 32 + lane, ti = ed / 3, e = ed - 3 * ti, tis = min(ti, WB - 1);
            const int st = __shfl_sync(full, status, tis);
            if (ed < 3 * WB) {
                EdgeWalk E;
                E.n = 0; E.majorY = 1; E.sg = 1.0; E.cf = 0; E.bx = 0; E.by = 0; E.fwd = 1;
                E.x0 = E.y0 = E.x1 = E.y1 = E.idx = E.idy = E.ta = E.tb = E.g0 = 0.0;
                double cs = 0.0;
                int by_t = 0;
                if (st == 1) {
                    const int e1 = (e == 2) ? 0 : e + 1;
                    const double *t = tr[ti];
                    edge_setup_canon(S, E, t[2 * e], t[2 * e + 1], t[2 * e1], t[2 * e1 + 1]);
                    cs = t[6]; by_t = __double2hiint(t[7]);
                }
                edge_record(E, cs, by_t, er[ed]);
            }
        }
        __syncwarp();
        // steps per triangle (lane < WB)
        int ntot = 0;
        if (lane < WB) ntot = edge_record_steps(er[3 * lane]) + edge_record_steps(er[3 * lane + 1]) + edge_record_steps(er[3 * lane + 2]);
        // ---- edges shared by two triangles of the batch are walked ONCE, for both (lane = edge, two passes).  T1 and T2 of
        // a cell share its diagonal, T2 and the T1 of the cell before it a vertical edge, and the list keeps them next to
        // each other: about a third of a batch's edges go.  Both triangles set the edge up from the same two end points in
        // the same frame and direction, so the records agree bit for bit and the lower one takes the other's weight: the
        // deposits are exactly those of two walks (deposit.cuh), whichever triangles happen to share a batch.
        {
            int partner[2] = {-1, -1};
            // a 32-bit tag of the edge's geometry first (one integer compare per candidate), the full record on a hit;
            // partners sit within three places of each other in the list
#pragma unroll
            for (int ps = 0; ps < 2; ++ps) {
                const int ed = ps * 32 + lane;
                if (ed < 3 * WB) {
                    const double *q = er[ed];
                    unsigned long long h = (unsigned long long)__double_as_longlong(q[0]) * 0x9E3779B97F4A7C15ull;
                    h = (h ^ (h >> 29) ^ (unsigned long long)__double_as_longlong(q[1])) * 0xBF58476D1CE4E5B9ull;
                    h = (h ^ (h >> 32) ^ (unsigned long long)__double_as_longlong(q[14])) * 0x94D049BB133111EBull;
                    Wk.pad[ed] = (edge_record_steps(q) > 0) ? (int)((h >> 33) | 1ull) : 0;
                }
            }
            __syncwarp();
#pragma unroll
            for (int ps = 0; ps < 2; ++ps) {
                const int ed = ps * 32 + lane, ti = ed / 3;
                const int tag = (ed < 3 * WB) ? Wk.pad[ed] : 0;
                if (tag) {
                    const int j0 = 3 * max(ti - 3, 0), j1 = 3 * min(ti + 4, WB);
#pragma unroll 1
                    for (int j = j0; j < j1; ++j)
                        if (Wk.pad[j] == tag && j != ed && edge_record_same(er[ed], er[j])) partner[ps] = j;
                }
            }
            __syncwarp();
#pragma unroll
            for (int ps = 0; ps < 2; ++ps) { const int ed = ps * 32 + lane; if (ed < 3 * WB) Wk.pad[ed] = partner[ps]; }
            __syncwarp();
            // a pair is made only if both see each other
#pragma unroll
            for (int ps = 0; ps < 2; ++ps) {
                const int ed = ps * 32 + lane, j = partner[ps];
                const int ntj = __shfl_sync(full, ntot, (j >= 0) ? j / 3 : 0);
                bool keep = false, drop = false;
                if (ed < 3 * WB && j >= 0 && ntj > 0 && Wk.pad[j] == ed) {
                    const long long dq = (long long)Wk.qi[j / 3] - (long long)Wk.qi[ed / 3];
                    if (dq >= -127 && dq <= 127) { keep = ed < j; drop = !keep; }
                }
                double c2 = 0.0, d2 = 0.0;
                if (keep) { c2 = er[j][10]; d2 = er[j][11]; }
                __syncwarp();
                if (keep) { er[ed][12] = c2; er[ed][13] = d2; }
                if (drop) er[ed][9] = __hiloint2double(0, __double2loint(er[ed][9]));
                __syncwarp();
            }
        }
        // ---- a triangle that still has more than GIANT_STEPS steps is shared out edge by edge in chunks to walk_giant_kernel;
        // an edge it walks for a neighbour too takes the neighbour along (its queue entry, as an offset, and its edge)
        if (lane < WB) ntot = edge_record_steps(er[3 * lane]) + edge_record_steps(er[3 * lane + 1]) + edge_record_steps(er[3 * lane + 2]);
        if (ntot > GIANT_STEPS) {
            int nch = 0;
#pragma unroll
            for (int e = 0; e < 3; ++e) nch += (edge_record_steps(er[3 * lane + e]) + GIANT_CHUNK - 1) / GIANT_CHUNK;
            unsigned long long at = atomicAdd(&S.counters[C_GIANT], (unsigned long long)nch);
            if ((long long)(at + nch) <= S.giant_cap) {           // (else it stays here; the skipped slots keep their sentinel)
                for (int e = 0; e < 3; ++e) {
                    const double *q = er[3 * lane + e];
                    const int nst = edge_record_steps(q);
                    const int ne = (nst + GIANT_CHUNK - 1) / GIANT_CHUNK;
                    const int fl = __double2loint(q[9]), by_e = __double2hiint(q[14]);
                    unsigned long long ent = ((unsigned long long)qidx << 20) | ((unsigned long long)e << 18);
                    const int j = Wk.pad[3 * lane + e];
                    if (q[12] != 0.0 && j >= 0) {
                        const long long delta = (long long)Wk.qi[j / 3] - (long long)qidx;        // within +-127 (checked when paired)
                        ent |= (1ull << 58) | ((unsigned long long)(j % 3) << 56) | ((unsigned long long)(delta + 128) << 48);
                    }
                    for (int c = 0; c < ne; ++c) {
                        // the block of map rows around the middle step of the chunk (ordering key only)
                        const int m = min(c * GIANT_CHUNK + GIANT_CHUNK / 2, nst - 1);
                        const double ms = q[8] + ((fl & 2) ? -1.0 : 1.0) * (double)(m - 1);
                        const double y = (fl & 1) ? ms : fma(dmin(dmax((ms - q[0]) * q[4], q[6]), q[7]), q[3] - q[1], q[1]);
                        const int row = min(max(__double2int_rd(y) + by_e, 0), S.npix2 - 1);
                        S.giant_key[at] = (unsigned char)min(row >> GIANT_BIN_SHIFT, GIANT_BINS - 2);
                        S.giant[at++] = ent | (unsigned long long)c;
                    }
                }
                ntot = -1;                                          // gone
            }
        }
        // ---- runs per edge and their inclusive prefix (lane = edge, two passes)
        int total = 0;
#pragma unroll
        for (int ps = 0; ps < 2; ++ps) {
            const int ed = ps * 32 + lane, tis = min(ed / 3, WB - 1);
            const int nt = __shfl_sync(full, ntot, tis);
            int inc = (ed < 3 * WB && nt > 0) ? (edge_record_steps(er[ed]) + RUN - 1) / RUN : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(full, inc, o); if (lane >= o) inc += t; }
            if (ed < 3 * WB) pre[ed] = total + inc;
            total += __shfl_sync(full, inc, 31);
        }
        __syncwarp();
        int steps = 0;
#pragma unroll 1
        for (int r0 = 0; r0 < total; r0 += 32) {
            const int r = r0 + lane;
            if (r < total) {
                int lo = 0, hi = 3 * WB - 1;                        // first edge whose inclusive prefix exceeds r
#pragma unroll
                for (int k = 0; k < 6; ++k) { const int mid = (lo + hi) >> 1; const bool up = pre[mid] <= r; lo = up ? mid + 1 : lo; hi = up ? hi : mid; }
                const int ed = min(lo, 3 * WB - 1);
                const double *q = er[ed];
                const int m0 = (r - (ed ? pre[ed - 1] : 0)) * RUN, m1 = min(m0 + RUN, edge_record_steps(q));
                edge_run(S, q, m0, m1);
                steps += m1 - m0;
            }
        }
        __syncwarp();
        n_pieces += (unsigned long long)steps;
        b = __shfl_sync(full, bnext, 0);
    }
    for (int o = 16; o; o >>= 1) n_pieces += __shfl_xor_sync(full, n_pieces, o);
    if (lane == 0 && n_pieces) atomicAdd(&S.counters[C_PX_EDGE], n_pieces);
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(&S.counters[C_CHUNKS], (unsigned long long)nb);   // walked, all bands
}

// The giant triangles walk_kernel set aside, chunk by chunk.  A giant's edges cross the whole map, so its deposits
// touch `diff` rows 80 KB apart: the chunks are first ORDERED by the block of 256 map rows they fall into (counting
// sort: giant_hist_kernel, giant_scatter_kernel), and the warps of walk_giant_kernel take consecutive chunks of that
// order -- at any moment all of them deposit into one or two row blocks (20 MB each), which L2 holds, instead of
// into the whole 1.6 GB of a 10^4 x 10^4 map.
__global__ void __launch_bounds__(256) giant_hist_kernel(const __grid_constant__ ShootDev S) {
    __shared__ unsigned int h[GIANT_BINS];
    for (int k = threadIdx.x; k < GIANT_BINS; k += blockDim.x) h[k] = 0u;
    __syncthreads();
    long long n = (long long)S.counters[C_GIANT];
    if (n > S.giant_cap) n = S.giant_cap;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const unsigned char key = S.giant_key[i];
        if (key < GIANT_BINS - 1) atomicAdd(&h[key], 1u);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < GIANT_BINS; k += blockDim.x) if (h[k]) atomicAdd(&S.giant_hist[k], h[k]);
}
__global__ void __launch_bounds__(256) giant_scatter_kernel(const __grid_constant__ ShootDev S) {
    __shared__ unsigned int base[GIANT_BINS];
    if (threadIdx.x == 0) {
        unsigned int run = 0;
        for (int k = 0; k < GIANT_BINS; ++k) { base[k] = run; run += S.giant_hist[k]; }
        if (blockIdx.x == 0) S.counters[C_GWALK] = run;            // sorted entries (the sentinels are left out)
    }
    __syncthreads();
    long long n = (long long)S.counters[C_GIANT];
    if (n > S.giant_cap) n = S.giant_cap;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const unsigned char key = S.giant_key[i];
        if (key < GIANT_BINS - 1) S.giant_sorted[base[key] + atomicAdd(&S.giant_hist[GIANT_BINS + key], 1u)] = S.giant[i];
    }
}

// One warp per chunk, chunks in sorted order with a grid stride (they cost the same): every lane sets the chunk's
// triangle and edge up for itself from the same vertices (so the chunks' end points agree bit for bit, and no shared
// memory is needed), then walks GIANT_RUN consecutive steps of the chunk.
static const int GIANT_WARPS = 8;
__global__ void __launch_bounds__(GIANT_WARPS * 32, 3) walk_giant_kernel(const __grid_constant__ ShootDev S) {
    const int lane = threadIdx.x & 31;
    const long long n = (long long)S.counters[C_GWALK];
    if (blockIdx.x == 0 && threadIdx.x == 0 && n) atomicAdd(&S.counters[C_ROWS], (unsigned long long)n);    // chunks, all bands
    Win W; W.w32 = nullptr; W.ax = 0; W.ay = 0;
    unsigned long long n_pieces = 0;
    const long long stride = (long long)gridDim.x * GIANT_WARPS;
    long long i = (long long)blockIdx.x * GIANT_WARPS + (threadIdx.x >> 5);
    unsigned long long ent_next = (i < n) ? S.giant_sorted[i] : 0ull;
    for (; i < n; i += stride) {
        const unsigned long long ent = ent_next;                    // (partner: flag, edge, queue offset | queue entry << 20 | edge << 18 | chunk)
        if (i + stride < n) ent_next = S.giant_sorted[i + stride];  // on its way while this chunk is walked
        const int e = (int)((ent >> 18) & 3ull), c = (int)(ent & 0x3ffffull);
        const unsigned int qa = (unsigned int)((ent >> 20) & 0xfffffffull);
        const bool two = ((ent >> 58) & 1ull) != 0;
        const double *p = S.queue + (size_t)qa * QENT;
        const double *p2 = S.queue + (size_t)((long long)qa + (long long)((ent >> 48) & 0xffull) - 128) * QENT;
        double v[QENT], v2[QENT];
#pragma unroll
        for (int k = 0; k < QENT; ++k) v[k] = __ldg(&p[k]);
#pragma unroll
        for (int k = 0; k < QENT; ++k) v2[k] = two ? __ldg(&p2[k]) : 0.0;
        TriSetup T;
        tri_setup(S, W, v, T);
        if (T.status != 1) continue;                                // (cannot happen: walk_kernel found steps to walk)
        const double xa = (e == 0) ? v[0] : (e == 1) ? v[2] : v[4], ya = (e == 0) ? v[1] : (e == 1) ? v[3] : v[5];
        const double xb = (e == 0) ? v[2] : (e == 1) ? v[4] : v[0], yb = (e == 0) ? v[3] : (e == 1) ? v[5] : v[1];
        EdgeWalk E;
        edge_setup_canon(S, E, xa, ya, xb, yb);
        double q[EREC];
        edge_record(E, T.cs, T.by, q);
        if (two) {
            // the neighbour across this edge: its weight, signed for the canonical direction, and its frame
            TriSetup T2;
            tri_setup(S, W, v2, T2);
            if (T2.status == 1) {
                const int e2 = (int)((ent >> 56) & 3ull);
                const double xa2 = (e2 == 0) ? v2[0] : (e2 == 1) ? v2[2] : v2[4], ya2 = (e2 == 0) ? v2[1] : (e2 == 1) ? v2[3] : v2[5];
                const double xb2 = (e2 == 0) ? v2[2] : (e2 == 1) ? v2[4] : v2[0], yb2 = (e2 == 0) ? v2[3] : (e2 == 1) ? v2[5] : v2[1];
                const bool fwd2 = (xa2 < xb2) || (xa2 == xb2 && ya2 <= yb2);
                q[12] = fwd2 ? T2.cs : -T2.cs; q[13] = (double)(E.by - T2.by);
            }
        }
        const int m0 = c * GIANT_CHUNK + lane * GIANT_RUN, m1 = min(m0 + GIANT_RUN, E.n);
        if (m0 < m1) {
            edge_run(S, q, m0, m1);
            n_pieces += (unsigned long long)(m1 - m0);
        }
    }
    for (int o = 16; o; o >>= 1) n_pieces += __shfl_xor_sync(0xffffffffu, n_pieces, o);
    if (lane == 0 && n_pieces) atomicAdd(&S.counters[C_PX_EDGE], n_pieces);
}

// floor(d / p), the pixel rule of O5, exactly, as an integer (saturated; NaN -> INT_MIN, outside every map): the
// product with the rounded reciprocal is within a few ulps of the quotient, so its floor is the quotient's floor
// unless it lies within `tol` of an integer -- only then divide (out of line: an inlined IEEE division is ~30
// instructions, eight of them per row group).  The floor itself is the rounding mode of the conversion.
static __device__ __noinline__ int floor_div_exact(double d, double p) {
    const double f = floor(d / p);
    if (!(f == f)) return INT_MIN;
    return (f >= 2.0e9) ? INT_MAX : (f <= -2.0e9) ? INT_MIN : (int)f;
}
__device__ __forceinline__ int floor_div(double d, double p, double inv_p, double tol) {
    const double q = d * inv_p;
    const int n = __double2int_rd(q);
    const double r = q - (double)n;                       // in [0, 1) unless the conversion saturated (or NaN)
    return (fabs(r - 0.5) < 0.5 - tol) ? n : floor_div_exact(d, p);
}

// ------------------------------------------------------------------------------------------------
// IRS: rays at cell centres (reading G10), floor of a true division (O5), counts.
template <bool F32>
__global__ void __launch_bounds__(SHOOT_WARPS * 32, 12) shoot_irs_kernel(const __grid_constant__ ShootDev S) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WarpShared &Ws = reinterpret_cast<WarpShared *>(smem_raw)[threadIdx.x >> 5];
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    ThreadCounters tc;
    TileCtx C;
    Win W; W.w32 = reinterpret_cast<unsigned int *>(Ws.win); W.ax = 0; W.ay = 0;
    const long long ntiles = (long long)S.ntx * S.tile_rows;
    const long long nrx = S.i1 - S.i0;

    // global tile anchoring as in the IPM kernel: tile (tx, ty) holds the cells [32 tx, 32 tx + 32) x [32 ty, ..)
    for (long long tile = fetch_tile(S); tile < ntiles;) {
        const long long tile_next = fetch_tile(S);
        long long tx, ty;
        tile_indices(S, tile, tx, ty);
        const long long ci0 = tx * TCX, cj0 = ty * TCY;
        const long long ci1 = min(ci0 + TCX, S.n1) - 1, cj1 = min(cj0 + TCY, S.n2) - 1;      // last cell of the tile
        wtile_setup(S, Ws, C, ci0, cj0, ci1, cj1, 0.5);
        const long long ci = ci0 + lane;
        const bool insub = (ci >= S.i0) && (ci < S.i1);
        const double x = corner_x(S, ci) + 0.5 * S.h1, ux = ((double)lane - 0.5 * (TCX - 1)) * S.dux;
        const int g_lo = (S.j0 > cj0) ? (int)((S.j0 - cj0) / RPT) : 0;
        const int g_hi = (int)((min(S.j1 - 1, cj1) - cj0) / RPT);
#pragma unroll 1
        for (int g = g_lo; g <= g_hi && g < NGRP; ++g) {
            double y[RPT], uy[RPT], wx[RPT], wy[RPT];
            bool valid[RPT];
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const int row = g * RPT + r;
                const long long cj = cj0 + row;
                valid[r] = (ci < S.n1) && (cj < S.n2);
                y[r] = corner_y(S, cj) + 0.5 * S.h2;
                uy[r] = ((double)row - 0.5 * (TCY - 1)) * S.duy;
            }
            eval_rays<F32>(S, Ws, C, x, ux, y, uy, valid, wx, wy, tc);
            bool cnt[RPT];                                                  // the rays of the sub-range
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const long long cj = cj0 + g * RPT + r;
                cnt[r] = valid[r] && insub && (cj >= S.j0) && (cj < S.j1);
            }
            int fx[RPT], fy[RPT];
            if (S.dump1) {
                unsigned vm = 0;
#pragma unroll
                for (int r = 0; r < RPT; ++r) vm |= cnt[r] ? (1u << r) : 0u;
                dump_rays(&S, (cj0 + g * RPT - S.j0) * nrx + (ci - S.i0), nrx, vm,
                          wx[0], wy[0], wx[1], wy[1], wx[2], wy[2], wx[3], wy[3]);
            }
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                fx[r] = floor_div(wx[r] - S.ylo1, S.p1, S.inv_p1, S.fd_tol); fy[r] = floor_div(wy[r] - S.ylo2, S.p2, S.inv_p2, S.fd_tol);
            }
            if (g == g_lo) {
                // window anchor: the tile centre extrapolated from the first two rows evaluated (any anchor is correct)
                const int ax0 = max(min(fx[0], 40000), -40000), ax1 = max(min(fx[1], 40000), -40000);
                const int ay0 = max(min(fy[0], 40000), -40000), ay1 = max(min(fy[1], 40000), -40000);
                const int rows2 = (TCY - 1) - 2 * g * RPT;                  // twice the rows from the first one to the centre
                const int cu = __shfl_sync(full, ax0 + (rows2 * (ax1 - ax0)) / 2, TCX / 2);
                const int cv = __shfl_sync(full, ay0 + (rows2 * (ay1 - ay0)) / 2, TCX / 2);
                W.ax = cu - WX / 2; W.ay = cv - WY / 2;
            }
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                int key = -1;
                if (cnt[r] && (unsigned)fx[r] < (unsigned)S.npix1 && (unsigned)fy[r] < (unsigned)S.npix2) {
                    key = (fy[r] << 16) | fx[r];
                    ++tc.single;
                }
                // runs of equal pixels among consecutive lanes become one add
                const int prev = __shfl_up_sync(full, key, 1);
                const bool head = (lane == 0) || (key != prev);
                const unsigned heads = __ballot_sync(full, head);
                if (head && key >= 0) {
                    const unsigned above = (lane == 31) ? 0u : (heads & ~((2u << lane) - 1u));
                    const int next = above ? (__ffs(above) - 1) : 32;
                    pix_add(S, W, key & 0xffff, key >> 16, (unsigned long long)(next - lane));
                }
            }
        }
        __syncwarp();
        flush_window(S, Ws, W);
        __syncwarp();
        tile = tile_next;
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
        unsigned long long a = (i < npix1) ? acc[row + i] : 0ull;
        if (diff) {
            unsigned long long inc = (i < npix1) ? diff[row + i] : 0ull;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
            if (lane == 31) wsum[warp] = inc;
            __syncthreads();
            unsigned long long pre = carry_s;
            for (int w = 0; w < warp; ++w) pre += wsum[w];
            const unsigned long long run = pre + inc;            // inclusive prefix of the differences up to i
            a += run;
            __syncthreads();
            if (threadIdx.x == FIN_T - 1) carry_s = run;
            __syncthreads();
        }
        if (i < npix1) {
            // The sum is read as SIGNED and clamped at 0: in a map that holds only part of the grid's triangles (a
            // slab, a patch) a pixel may be left with a rounding residue of a few quanta below zero by the large
            // triangles that cross it; as an unsigned number that would be 2^64.
            const long long sa = (long long)a;
            if (map) { double v = (double)(sa < 0 ? 0ll : sa) * scale; map[row + i] = accumulate ? map[row + i] + v : v; }
            if (counts) counts[row + i] = accumulate ? counts[row + i] + a : a;
        }
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
    if ((f->quad[0] != 0.0 || f->quad[1] != 0.0 || f->quad[2] != 0.0 || f->quad[3] != 0.0) && d->border_mode != MLENS_BORDER_EXPLICIT) {
        set_error("a field with macro terms beyond linear (mlens_field_set_macro_quadratic) needs an explicit window: "
                  "eq 14-16 enclose the macro-images of a constant kappa, gamma only (MLENS_BORDER_EXPLICIT)");
        return MLENS_EINVAL;
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


namespace {
// `ready` is recorded on the stream the parked buffers were last used on; whoever takes or frees them waits for it.
struct ParkedScratch { DevBuf<double> queue; DevBuf<int> qcount; DevBuf<unsigned int> biglist; int device = -1; cudaEvent_t ready = nullptr; };
ParkedScratch g_parked[ML_MAXDEV];
std::mutex g_parked_mutex;
}  // namespace

void scratch_park(mlens_field *f, cudaStream_t s) {
    std::lock_guard<std::mutex> lock(g_parked_mutex);
    ParkedScratch &P = g_parked[(f->device >= 0 && f->device < ML_MAXDEV) ? f->device : ML_MAXDEV - 1];
    if (!f->queue.p || f->queue.cap <= P.queue.cap) return;                     // the larger one is kept
    if (P.queue.p) {
        if (P.ready) cudaStreamWaitEvent(s, P.ready, 0);
        P.queue.release(s); P.qcount.release(s); P.biglist.release(s);
    }
    if (!P.ready && cudaEventCreateWithFlags(&P.ready, cudaEventDisableTiming) != cudaSuccess) { P.ready = nullptr; cudaGetLastError(); return; }
    P.queue = f->queue; P.qcount = f->qcount; P.biglist = f->biglist; P.device = f->device;
    cudaEventRecord(P.ready, s);
    f->queue = DevBuf<double>(); f->qcount = DevBuf<int>(); f->biglist = DevBuf<unsigned int>();
}

void scratch_take(mlens_field *f, cudaStream_t s) {
    std::lock_guard<std::mutex> lock(g_parked_mutex);
    ParkedScratch &P = g_parked[(f->device >= 0 && f->device < ML_MAXDEV) ? f->device : ML_MAXDEV - 1];
    if (f->queue.p || !P.queue.p || P.device != f->device) return;
    if (P.ready) cudaStreamWaitEvent(s, P.ready, 0);
    f->queue = P.queue; f->qcount = P.qcount; f->biglist = P.biglist;
    f->queue.s_own = s; f->qcount.s_own = s; f->biglist.s_own = s;
    P.queue = DevBuf<double>(); P.qcount = DevBuf<int>(); P.biglist = DevBuf<unsigned int>();
}

static const long long GIANT_CAP = 1ll << 20;       // chunk slots per band (8 MB)

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
        // Queue of general triangles: every band ends with the tails of three kernels, so bands should be few and
        // the queue large -- 8 GiB unless the device is small, never more than the worst case of this map (two
        // triangles per cell); halved until it can be had.  desc.queue_mb overrides.
        size_t mem_free = 0, mem_total = 0;
        cudaMemGetInfo(&mem_free, &mem_total);
        long long qmb = 8192;
        if (mem_total > 0 && (long long)(mem_total >> 24) < qmb) qmb = (long long)(mem_total >> 24);   // <= 1/16 of the device
        const double need_mb = 3.2 * (double)(i1 - i0) * (double)(j1 - j0) * (QENT * 8) / 1048576.0 + 64.0;
        if ((double)qmb > need_mb) qmb = (long long)need_mb;
        const long long qmb_desc = d->queue_mb > 0 ? d->queue_mb : 0;       // the caller's choice, taken as it is
        if (qmb_desc > 0) qmb = qmb_desc;
        if (qmb > 12000) qmb = 12000;                                       // queue entries are named by 28 bits (giant-chunk list)
        scratch_take(f, s);
        for (;;) {
            qcap = qmb * (1ll << 20) / (QCHUNK * QENT * 8);          // chunks
            int rc = f->queue.reserve((size_t)qcap * QCHUNK * QENT, s, false);
            if (rc == MLENS_OK) rc = f->qcount.reserve((size_t)qcap, s, false);
            if (rc == MLENS_OK) rc = f->biglist.reserve((size_t)qcap * QCHUNK / 4, s, false);
            if (rc == MLENS_OK) rc = f->giant.reserve((size_t)GIANT_CAP, s, false);
            if (rc == MLENS_OK) rc = f->giant_sorted.reserve((size_t)GIANT_CAP, s, false);
            if (rc == MLENS_OK) rc = f->giant_key.reserve((size_t)GIANT_CAP, s, false);
            if (rc == MLENS_OK) rc = f->giant_hist.reserve((size_t)2 * GIANT_BINS, s, false);
            if (rc == MLENS_OK) break;
            if (rc != MLENS_ENOMEM || qmb_desc > 0 || qmb <= 256) return rc;
            cudaGetLastError();
            qmb /= 2;
        }
    }
    ShootDev S;
    S.L = make_lens_dev(f);
    S.x0_1 = g->x0_1; S.x0_2 = g->x0_2; S.h1 = g->h1; S.h2 = g->h2;
    S.i0 = i0; S.i1 = i1; S.j0 = j0; S.j1 = j1; S.n1 = g->n1; S.n2 = g->n2;
    S.colmajor = d->tile_traversal == 1 ? 0 : 1;
    S.ylo1 = g->ylo1; S.ylo2 = g->ylo2; S.p1 = g->p1; S.p2 = g->p2; S.inv_p1 = 1.0 / g->p1; S.inv_p2 = 1.0 / g->p2;
    S.npix1 = d->npix1; S.npix2 = d->npix2;
    S.acc = f->acc.p; S.diff = f->diff.p; S.queue = f->queue.p; S.qcount = f->qcount.p; S.biglist = f->biglist.p; S.big_cap = qcap * QCHUNK / 4; S.giant = f->giant.p; S.giant_cap = ipm ? GIANT_CAP : 0; S.giant_sorted = f->giant_sorted.p; S.giant_key = f->giant_key.p; S.giant_hist = f->giant_hist.p; S.counters = f->counters.p; S.queue_cap = qcap;
    S.dump1 = d->dump_w1; S.dump2 = d->dump_w2;
    S.binom = f->binom.p;
    if ((S.dump1 == nullptr) != (S.dump2 == nullptr)) { set_error("dump_w1 and dump_w2 go together"); return MLENS_EINVAL; }
    const bool f32 = d->eval_mode == MLENS_EVAL_FMM_F32;       // same tiles and slow paths as FMM; only the fast path differs
    S.eval_mode = f32 ? MLENS_EVAL_FMM : d->eval_mode;
    S.tq = d->tile_order;
    if (S.tq > TQMAX) S.tq = TQMAX;
    if (S.tq <= 0) S.tq = -1;                                   // chosen below, once the tile radius is known
    else if (S.tq < 2) S.tq = 2;
    S.small_px = d->small_px > 0 ? d->small_px : 24;
    S.fd_tol = 1.0e-9 * (double)((d->npix1 > d->npix2) ? d->npix1 : d->npix2);
    // truncation budget of the tile series: 5 % of the deflection accuracy the field was built for
    S.rt = 0.5 * sqrt((double)((TCX - 1) * (TCX - 1)) * g->h1 * g->h1 + (double)((TCY - 1) * (TCY - 1)) * g->h2 * g->h2) * (1.0 + 1e-9);
    S.inv_rt = 1.0 / S.rt;
    S.dux = g->h1 * S.inv_rt; S.duy = g->h2 * S.inv_rt;
    S.a1_lin = S.L.one_minus_kappa + S.L.gamma + S.L.kappa_star; S.a2_lin = S.L.one_minus_kappa - S.L.gamma + S.L.kappa_star;
    S.eps_far = 0.02 * f->eps * f->theta;
    if (S.tq < 0) {
        // Order of the tile series: term j of a leaf's series shifted to a tile falls like (c rt / L)^j, L the leaf's
        // half-length (c = 1.14 fits the measured optimum on the five configs; sources lie >= 3 L from the leaf's centre);
        // the order that brings it under the truncation budget in the smallest leaves, plus two.  Fewer terms mean
        // more of the near stars summed directly, more terms a longer Horner chain: measured optima 6 (config 3),
        // 8-9 (config 1), 13+ (config 2, one ray per pixel).  Every tile still checks its own bound.
        const double leaf_half_min = f->root_half / (double)(1 << (f->tree.n_levels > 0 ? f->tree.n_levels - 1 : 0));
        const double x = fmin(0.5, 1.14 * S.rt / leaf_half_min);
        int q = (int)ceil(log(0.5 * S.eps_far) / log(x)) - 1 + 2;
        S.tq = q < 4 ? 4 : (q > TQMAX ? TQMAX : q);
        // ... and the same rule for a tile in a larger leaf (tree level l): never more than in the smallest ones
        for (int l = 0; l <= ML_MAXLEV; ++l) {
            const double xl = fmin(0.5, 1.14 * S.rt / (f->root_half / (double)(1 << l)));
            int ql = (int)ceil(log(0.5 * S.eps_far) / log(xl)) - 1 + 2;
            ql = ql < 4 ? 4 : ql;
            S.tq_lev[l] = (signed char)(ql > S.tq ? S.tq : ql);
        }
    } else {
        for (int l = 0; l <= ML_MAXLEV; ++l) S.tq_lev[l] = (signed char)S.tq;       // desc.tile_order: one order everywhere
    }
    S.eps_star = 0.03 * f->eps * f->theta / (double)ML_NEAR;
    const int stepx = ipm ? TCX - 1 : TCX, stepy = ipm ? TCY - 1 : TCY;
    // tiles of the GLOBAL tile grid that hold a cell of the sub-range
    S.txb = i0 / stepx; S.tyb = j0 / stepy;
    long long ntx = (i1 - 1) / stepx - S.txb + 1, nty = (j1 - 1) / stepy - S.tyb + 1;
    if (ntx > 0x7fffffffLL) { set_error("too many tiles per row"); return MLENS_EINVAL; }
    S.ntx = (int)ntx;
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    long long band_cells = d->band_cells > 0 ? d->band_cells : (1ll << 30);
    long long rows_per_band = band_cells / (ntx * stepx * stepy);
    if (rows_per_band < 1) rows_per_band = 1;
    if (!ipm && !d->band_fixed) rows_per_band = nty;                          // IRS has no queue to bound: one launch
    // events of a timed call: destroyed on every way out of the function, error returns included
    struct Events {
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        std::vector<cudaEvent_t> list;
        ~Events() { if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); for (cudaEvent_t e : list) cudaEventDestroy(e); }
    } evs;
    cudaEvent_t &e0 = evs.e0, &e1 = evs.e1;
    const bool timed = st && (d->sync || d->ptr_kind == MLENS_PTR_HOST);
    if (timed) { ML_CUDA(cudaEventCreate(&e0)); ML_CUDA(cudaEventCreate(&e1)); ML_CUDA(cudaEventRecord(e0, s)); }
    int launches = 0, bands = 0;
    // per-kernel device times: events between the back-to-back launches of each band (timed calls only)
    std::vector<cudaEvent_t> &ev = evs.list;
    auto mark = [&]() -> int {
        if (!timed) return MLENS_OK;
        cudaEvent_t e; ML_CUDA(cudaEventCreate(&e)); ML_CUDA(cudaEventRecord(e, s)); ev.push_back(e);
        return MLENS_OK;
    };
    const size_t smem_ipm = SHOOT_WARPS * sizeof(WarpSharedIpm), smem_irs = SHOOT_WARPS * sizeof(WarpShared);
    static std::atomic<int> attr_set[ML_MAXDEV];                     // kernel attributes are per device (context)
    if (!attr_set[device_slot()].load()) {
        ML_CUDA(cudaFuncSetAttribute(walk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(WALK_WARPS * sizeof(WalkShared))));
        ML_CUDA(cudaFuncSetAttribute(shoot_ipm_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ipm));
        ML_CUDA(cudaFuncSetAttribute(shoot_irs_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_irs));
        ML_CUDA(cudaFuncSetAttribute(shoot_ipm_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ipm));
        ML_CUDA(cudaFuncSetAttribute(shoot_irs_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_irs));
        attr_set[device_slot()].store(1);
    }
    int bps_ipm = 1, bps_irs = 1;
    ML_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps_ipm, shoot_ipm_kernel<false>, SHOOT_WARPS * 32, smem_ipm));
    ML_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps_irs, shoot_irs_kernel<false>, SHOOT_WARPS * 32, smem_irs));
    if (bps_ipm < 1 || bps_irs < 1) { set_error("shooting kernels do not fit on this device"); return MLENS_ECUDA; }
    // IPM: the band height follows the rate at which the map's cells produce general triangles (they must fit the
    // queue of one band): the first band assumes the worst case of two per cell, later ones use the measured
    // rate of the bands before.  The host reads two counters after each band's shooting kernel, while the
    // apportioning kernels of that band are already queued behind it.
    const long long nwarps_res = (long long)nsm * (ipm ? bps_ipm : bps_irs) * SHOOT_WARPS;
    const double cap_entries = ipm ? fmax(0.0, 0.8 * (double)qcap - (double)nwarps_res) * (double)QCHUNK * 0.85 : 0.0;
    double rate = -1.0;                                            // general triangles per cell, measured
    const bool adapt = !d->band_fixed;                              // desc.band_fixed: always desc.band_cells (tests)
    unsigned long long q_before = 0;
    for (long long r0 = 0; r0 < nty; r0 += rows_per_band, ++bands) {
        if (ipm && adapt) {
            double cells = (rate < 0.0) ? 0.5 * cap_entries : cap_entries / fmax(rate, 1e-3);
            if (cells > (double)band_cells) cells = (double)band_cells;
            rows_per_band = (long long)(cells / (double)(ntx * stepx * stepy));
            if (rows_per_band < 1) rows_per_band = 1;
        }
        S.tile_row0 = r0;
        S.tile_rows = (nty - r0 < rows_per_band) ? (nty - r0) : rows_per_band;
        long long nt = ntx * S.tile_rows;
        const long long resident = (long long)nsm * (ipm ? bps_ipm : bps_irs);     // persistent blocks, tiles handed out dynamically
        const long long want = (nt + SHOOT_WARPS - 1) / SHOOT_WARPS;
        int grid = (int)((want < resident) ? want : resident);
        ML_CUDA(cudaMemsetAsync(f->counters.p, 0, 16, s));         // queue fill count and tile counter
        ML_CUDA(cudaMemsetAsync(f->counters.p + C_DRAIN, 0, 5 * 8, s));   // drain, big-list, walk and giant counters
        if (ipm) {
            ML_CUDA(cudaMemsetAsync(f->giant_key.p, 0xff, (size_t)GIANT_CAP, s));        // sentinels: slots reserved but not filled
            ML_CUDA(cudaMemsetAsync(f->giant_hist.p, 0, (size_t)2 * GIANT_BINS * 4, s));
        }
        ML_TRY(mark());
        if (ipm) {
            if (f32) ML_LAUNCH(shoot_ipm_kernel<true>, grid, SHOOT_WARPS * 32, smem_ipm, s, S);
            else ML_LAUNCH(shoot_ipm_kernel<false>, grid, SHOOT_WARPS * 32, smem_ipm, s, S);
            ML_TRY(mark());
            if (adapt && r0 + rows_per_band < nty) {             // feedback for the next band's height
                unsigned long long h3[3] = {0, 0, 0};                 // queued, (walked), overflowed: cumulative
                ML_CUDA(cudaMemcpyAsync(h3, f->counters.p + C_QUEUED, 24, cudaMemcpyDeviceToHost, s));
                ML_CUDA(cudaStreamSynchronize(s));
                const unsigned long long hq = h3[0] + h3[2];
                const double cells_done = (double)S.tile_rows * (double)(ntx * stepx * stepy);
                const double r_new = (double)(hq - q_before) / fmax(cells_done, 1.0);
                q_before = hq;
                rate = (rate < 0.0) ? 1.25 * r_new : fmax(1.25 * r_new, 0.7 * rate);   // head-room; forget slowly
            }
            ML_TRY(mark());                                       // after the host's read-back: ms_drain starts here, not at the shooting kernel's end
            ML_LAUNCH(drain_kernel, nsm * 8, DRAIN_WARPS * 32, 0, s, S);
            ML_TRY(mark());
            ML_LAUNCH(walk_kernel, nsm * 3, WALK_WARPS * 32, WALK_WARPS * sizeof(WalkShared), s, S);
            ML_TRY(mark());
            ML_LAUNCH(giant_hist_kernel, nsm, 256, 0, s, S);
            ML_LAUNCH(giant_scatter_kernel, nsm, 256, 0, s, S);
            ML_LAUNCH(walk_giant_kernel, nsm * 3, GIANT_WARPS * 32, 0, s, S);
            ML_TRY(mark());
            launches += 6;
        } else {
            if (f32) ML_LAUNCH(shoot_irs_kernel<true>, grid, SHOOT_WARPS * 32, smem_irs, s, S);
            else ML_LAUNCH(shoot_irs_kernel<false>, grid, SHOOT_WARPS * 32, smem_irs, s, S);
            ML_TRY(mark());
            launches += 1;
        }
        ML_CUDA(cudaGetLastError());
    }
    double scale = ipm ? g->weight / (double)FIX_ONE
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
        st->n_tri_single = (int64_t)h[C_SINGLE]; st->n_tri_strip = (int64_t)h[C_SMALL];
        st->n_tri_queued = (int64_t)h[C_QUEUED]; st->n_tri_walked = (int64_t)h[C_CHUNKS];
        st->n_queue_overflow = (int64_t)h[C_OVERFLOW]; st->n_rays_fallback = (int64_t)h[C_FALLBACK];
        st->n_near_terms = (int64_t)h[C_NEAR];
        st->n_px_strip = (int64_t)h[C_PX_SMALL]; st->n_px_clipped = (int64_t)h[C_PX_INT];
        st->n_edge_steps = (int64_t)h[C_PX_EDGE];
        st->n_tiles_full = (int64_t)h[C_TILES_FULL];
        st->n_giant_chunks = (int64_t)h[C_ROWS];
        st->n_tiles = (int64_t)h[C_TILES]; st->n_near_leaf_sum = (int64_t)h[C_NEAR_LEAF];
        st->tile_order = S.tq;
        st->n_bands = bands; st->gpu_launches = launches; st->n_shoot_launches = bands;
        if (timed) {
            ML_CUDA(cudaEventElapsedTime(&st->ms_total, e0, e1));
            const size_t per = ipm ? 6 : 2;              // events per band: shoot [0,1], (host read-back), drain [2,3], walk [3,4], giants [4,5]
            for (int b = 0; b < bands; ++b) {
                float ms = 0;
                ML_CUDA(cudaEventElapsedTime(&ms, ev[b * per], ev[b * per + 1])); st->ms_shoot += ms;
                if (ipm) {
                    ML_CUDA(cudaEventElapsedTime(&ms, ev[b * per + 2], ev[b * per + 5])); st->ms_drain += ms;
                    ML_CUDA(cudaEventElapsedTime(&ms, ev[b * per + 3], ev[b * per + 4])); st->ms_walk += ms;
                    ML_CUDA(cudaEventElapsedTime(&ms, ev[b * per + 4], ev[b * per + 5])); st->ms_giant += ms;
                }
            }
            float ms = 0;
            ML_CUDA(cudaEventElapsedTime(&ms, ev[ev.size() - 2], ev[ev.size() - 1])); st->ms_finalise = ms;
        }
    } else if (d->sync) {
        ML_CUDA(cudaStreamSynchronize(s));
    }
    return MLENS_OK;
}

}  // namespace ml
