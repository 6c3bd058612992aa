// tile.cuh -- warp-autonomous ray-tile evaluator (hot loop A): every warp owns a 32 x 32 tile of rays,
// builds the tile's own expansion with warp-level primitives only (no block barrier anywhere) and then
// evaluates eq 12 for four rays per lane at a time.
//
// Targets outnumber sources by 10^4..10^5, so the FMM hierarchy is continued on the target side
// (DESIGN.md s5.4): for every ray tile the leaf's local series is shifted to the tile centre (eq C7 once
// more) and the leaf's near-field stars that are far from the tile on the tile's scale are added to it
// (eq C6); what is left per ray is a ~13-term Horner sum plus the few stars within ~10 tile radii.  Both
// truncations are bounded per tile from the coefficients themselves; a tile whose bound fails evaluates
// the leaf's full series and full star list instead.
#pragma once
#include "device.cuh"

namespace ml {

static const int TCX = 32;            // rays per tile row (= warp width, one column per lane)
static const int TCY = 32;            // ray rows per tile
static const int RPT = 4;             // rays a lane evaluates together (independent Horner chains)
static const int NGRP = TCY / RPT;
static const int TQMAX = 15;          // highest order of the tile series
static const int NSLOT = 2;           // leaves a tile keeps a series for (rays in further leaves go through the tree)
static const int WX = 32, WY = 8;     // per-warp shared-memory pixel window
static const int FOLDJ = WX * WY * 8 / (32 * 16);   // series terms per pass of the star folding (scratch = the window)
static const int BN = 2 * ML_P1MAX;   // stride of the Pascal triangle
static const int GIANT_BINS = 128;    // blocks of map rows the giant triangles' chunks are ordered by
static const int GIANT_BIN_SHIFT = 8; // 256 rows per block (a block of `diff` rows stays in L2 while its chunks are walked)

// slots of ShootDev::counters
enum { C_QUEUE = 0, C_TILE, C_SINGLE, C_SMALL, C_QUEUED, C_CHUNKS, C_OVERFLOW, C_FALLBACK, C_RAYS, C_NEAR,
       C_PX_SMALL, C_PX_INT, C_PX_EDGE, C_ROWS, C_TILES_FULL, C_DRAIN, C_BIG, C_WALK, C_GIANT, C_GWALK, C_TILES, C_NEAR_LEAF, C_NCOUNTERS };

// What a shooting kernel needs besides the lens: the ray grid, the map, the accumulators.
struct ShootDev {
    LensDev L;
    double x0_1, x0_2, h1, h2;
    long long i0, i1, j0, j1;          // cell sub-range
    long long n1, n2;                  // cells of the whole grid: tiles are anchored on it, whatever the sub-range
    long long txb, tyb;                // first tile column / row (global tile indices) that holds a cell of the sub-range
    int colmajor;                      // tiles of a band are handed out column by column (else row by row)
    double ylo1, ylo2, p1, p2, inv_p1, inv_p2;
    int npix1, npix2;
    unsigned long long *acc;           // fixed-point pixel sums (IPM) or ray counts (IRS)
    unsigned long long *diff;          // IPM: row-difference array written by the edge walk of large triangles
    double *queue;                     // general-triangle queue: chunks of QCHUNK entries of QENT doubles
    int *qcount;                       // entries in each chunk
    unsigned int *biglist;             // queue entries whose triangles are walked edge by edge (walk_kernel)
    long long big_cap;
    unsigned long long *giant;         // (queue entry << 20 | edge << 18 | chunk) of the triangles with too many steps for one warp
    long long giant_cap;
    unsigned long long *giant_sorted;  // the same entries ordered by the block of map rows their steps fall into
    unsigned char *giant_key;          // that block, per entry (255: none)
    unsigned int *giant_hist;          // [0, GIANT_BINS): entries per block; [GIANT_BINS, 2 GIANT_BINS): scatter cursors
    unsigned long long *counters;
    long long queue_cap;               // chunks
    double *dump1, *dump2;
    const double *binom;               // Pascal triangle, stride BN
    int eval_mode;
    int ntx;                           // tiles along x1
    long long tile_row0, tile_rows;    // band of tile rows handled by this launch
    int tq;                            // highest order of the tile series in this shoot (tiles in the smallest leaves)
    signed char tq_lev[ML_MAXLEV + 1];  // order for a tile in a leaf of tree level l: larger leaves converge faster
    double eps_far, eps_star;          // truncation budgets of the tile series (absolute, units of theta)
    double rt, inv_rt;                 // radius of a ray tile (half its diagonal) and its reciprocal
    double a1_lin, a2_lin;             // inside the star disc w = (a1 x - Re alpha_star, a2 y - Im alpha_star): a = 1 - kappa +- gamma + kappa_star
    double dux, duy;                   // cell size over tile radius: step of the tile series' argument per ray
    double fd_tol;                     // IRS: quotients closer than this to an integer are divided exactly
    int small_px;                      // queued triangles whose clipped bounding box has more pixels than this are walked, not clipped
};

__device__ __forceinline__ double corner_x(const ShootDev &S, long long i) { return __dadd_rn(S.x0_1, __dmul_rn((double)i, S.h1)); }
__device__ __forceinline__ double corner_y(const ShootDev &S, long long j) { return __dadd_rn(S.x0_2, __dmul_rn((double)j, S.h2)); }

// Per-warp shared memory of the evaluator.  `win` doubles as the scratch of the tile set-up (fold terms), which
// is why it is zeroed at the end of the set-up and not by the flush.
struct WarpShared {
    unsigned long long win[WY * WX];                         // 4 KB
    double2 t[NSLOT][TQMAX + 1];                             // conj(alpha)(u) = sum_j t_j u^j, theta^2 included
    double sx[NSLOT][ML_NEAR], sy[NSLOT][ML_NEAR], sm[NSLOT][ML_NEAR];   // direct stars (absolute positions, m theta^2)
    double2 e[ML_P1MAX];                                     // the leaf's derivative series (set-up scratch)
    uint32_t bx0[NSLOT], bx1[NSLOT], by0[NSLOT], by1[NSLOT];
    int leaf[NSLOT], node[NSLOT], nd[NSLOT], mode[NSLOT], q[NSLOT];     // q: order of the slot's series
    double ctx[4];                                           // zt_x, zt_y, 1/rt, fast flag: what the set-up hands back
};
// ... plus what the IPM kernel needs for apportioning
struct WarpSharedIpm : WarpShared {
    double ringE[8][6];                                      // general triangles the global queue could not take, 8 at a time (cold)
    unsigned char ids[256];                                  // triangles of the row group that are not singles: (corner row, column, which of the two)
    double stu[RPT + 1][32], stv[RPT + 1][32];               // mapped corners of the row group in pixel units (row 0 = last row of the previous group)
    int stp[RPT + 1][32];                                    // their packed pixels
    int sto[RPT + 1][32];                                    // and on which sides of the map they lie (0: inside)
    // the per-triangle records of the (cold) in-kernel apportioning live in `e`, which only the tile set-up uses
    __device__ double (*rec())[10] { return reinterpret_cast<double (*)[10]>(e); }
};
static_assert(sizeof(double2) * ML_P1MAX >= 8 * 10 * sizeof(double), "records must fit the set-up scratch");
static_assert(FOLDJ >= 4 && ML_NEAR == 32, "fold scratch must fit the window");

struct TileCtx {                       // warp-uniform registers
    double zt_x, zt_y, inv_rt;
    bool fast;                         // the whole tile sits in one leaf whose tile series passed its bound
    bool lin;                          // the sheet term is -kappa_star z for every ray of the tile: inside the star disc (eq 19), or inside
                                       // the star rectangle with the analytic rest of eq B8 folded into the tile series
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Builds slot `s` of the warp's tile: shifted series + folded stars + direct-star list.
__device__ __forceinline__ void wtile_build_slot(const ShootDev &S, WarpShared &W, const TileCtx &C, int s, double rt, bool with_sheet) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int p = S.L.p;
    const int leaf = W.leaf[s], node = W.node[s];
    const int lev = __ldg(&S.L.level[node]);
    const int Q = S.tq_lev[min(lev, ML_MAXLEV)];
    const double half = S.L.root_half / (double)(1 << lev);
    const double cx = -S.L.root_half + (2.0 * __ldg(&S.L.ix[node]) + 1.0) * half;
    const double cy = -S.L.root_half + (2.0 * __ldg(&S.L.iy[node]) + 1.0) * half;
    const int cnt = __ldg(&S.L.near_cnt[leaf]);
    const double2 *ecoef = with_sheet ? S.L.ecoef_shoot : S.L.ecoef;       // with or without the rectangle sheet's analytic part
    for (int j = lane; j < p; j += 32) W.e[j] = ecoef[(size_t)leaf * S.L.p1 + j];
    __syncwarp();
    // ---- shift of the derivative series to the tile centre: T_j = rho^j sum_m e_{j+m} C(j+m, j) zeta_t^m   (eq C7)
    const double ih = fast_rcp(half);
    const double rho = rt * ih;
    const double zr = (C.zt_x - cx) * ih, zi = (C.zt_y - cy) * ih;
    double tail = 0.0;
    for (int j = lane; j < p; j += 32) {
        double ar = 0.0, ai = 0.0;
#pragma unroll 2
        for (int m = p - 1 - j; m >= 0; --m) {
            double bc = __ldg(&S.binom[(size_t)(j + m) * BN + j]);
            double2 c = W.e[j + m];
            double tr = fma(ar, zr, fma(-ai, zi, bc * c.x));
            double ti = fma(ar, zi, fma(ai, zr, bc * c.y));
            ar = tr; ai = ti;
        }
        double sc = 1.0;
#pragma unroll 1
        for (int k = 0; k < j; ++k) sc *= rho;
        ar *= sc; ai *= sc;
        if (j <= Q) W.t[s][j] = make_double2(ar, ai);
        else tail += fabs(ar) + fabs(ai);
    }
    for (int j = p + lane; j <= Q; j += 32) W.t[s][j] = make_double2(0.0, 0.0);
    tail = warp_sum(tail);
    // ---- near-field stars (lane k = star k): far from the tile on the tile's scale -> series (eq C6), else direct
    double2 *fold = reinterpret_cast<double2 *>(W.win);          // [FOLDJ][32]
    {
        const int k = lane;
        bool have = k < cnt, direct = false;
        double x = 0, y = 0, m = 0;
        double2 term = make_double2(0.0, 0.0), w = make_double2(0.0, 0.0);
        if (have) {
            size_t o = (size_t)leaf * ML_NEAR + k;
            x = S.L.near_x[o]; y = S.L.near_y[o]; m = S.L.near_m[o] * S.L.theta2;
            double dx = x - C.zt_x, dy = y - C.zt_y;
            double d2 = dx * dx + dy * dy, d = sqrt(d2);
            const double id = (d > 0.0) ? fast_rcp(d) : 0.0;
            double r = (d > 0.0) ? rt * id : 2.0;
            direct = true;
            if (r < 0.5) {
                double rq = r;
#pragma unroll 1
                for (int k2 = 0; k2 < Q; ++k2) rq *= r;                  // r^(Q+1)
                double bound = (m * id) * rq * fast_rcp(1.0 - r);
                if (bound <= S.eps_star) {
                    direct = false;
                    // conj(alpha_i) = m/(eta - d) = -(m/d) sum_j (eta/d)^j ; with eta = rt u: term_j = -(m/d)(rt/d)^j
                    double id2 = id * id;
                    term = make_double2(-m * dx * id2, m * dy * id2);     // -m/d = -m conj(d)/|d|^2
                    w = make_double2(rt * dx * id2, -rt * dy * id2);      // rt/d
                }
            }
        }
        const unsigned fm = __ballot_sync(full, have && !direct);
        const unsigned dm = __ballot_sync(full, direct);
        if (direct) {
            int pos = __popc(dm & ((1u << k) - 1u));
            W.sx[s][pos] = x; W.sy[s][pos] = y; W.sm[s][pos] = m;
        }
        if (k == 0) { W.nd[s] = __popc(dm); W.mode[s] = (tail <= S.eps_far) ? 0 : 1; W.q[s] = Q; }
        if (fm) {
            // FOLDJ series terms per pass: lane = star writes its terms, then the warp sums them over the stars
            for (int j0 = 0; j0 <= Q; j0 += FOLDJ) {
                __syncwarp();
#pragma unroll
                for (int j = 0; j < FOLDJ; ++j) { fold[j * 32 + k] = term; term = cmul(term, w); }
                __syncwarp();
                {
                    // lane = (term jj, eighth q): four stars each, then the eighths are summed by shuffles
                    static_assert(FOLDJ == 4, "32 lanes = 4 terms x 8");
                    const int jj = lane >> 3, q = lane & 7;
                    double2 a = fold[jj * 32 + q];
#pragma unroll
                    for (int kk = 1; kk < 4; ++kk) { double2 f = fold[jj * 32 + kk * 8 + q]; a.x += f.x; a.y += f.y; }
#pragma unroll
                    for (int o = 1; o < 8; o <<= 1) { a.x += __shfl_xor_sync(full, a.x, o); a.y += __shfl_xor_sync(full, a.y, o); }
                    if (q == 0 && j0 + jj <= Q) { double2 t0 = W.t[s][j0 + jj]; W.t[s][j0 + jj] = make_double2(t0.x + a.x, t0.y + a.y); }
                }
            }
        }
    }
    __syncwarp();
}

__device__ __forceinline__ void zero_window(WarpShared &W) {
    const int lane = threadIdx.x & 31;
    ulonglong2 *w2 = reinterpret_cast<ulonglong2 *>(W.win);
#pragma unroll
    for (int k = 0; k < WY * WX / 64; ++k) w2[k * 32 + lane] = make_ulonglong2(0ull, 0ull);
}

// Sets up the warp's tile: centre, radius, leaves of the four extreme rays, one slot per distinct leaf.
// off = offset of the rays from the grid corners in cells (0 for IPM, 0.5 for IRS).  Leaves the window zeroed.
static __device__ __noinline__ void wtile_setup_ool(const ShootDev *Sp, WarpShared *Wp, long long ci0, long long cj0,
                                                    long long ci1, long long cj1, double off) {
    const ShootDev &S = *Sp;
    WarpShared &W = *Wp;
    TileCtx C;
    unsigned long long *full_counter = &S.counters[C_TILES_FULL];
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    C.inv_rt = 1.0; C.fast = false; C.zt_x = 0.0; C.zt_y = 0.0;
    if (S.eval_mode != MLENS_EVAL_FMM) {
        zero_window(W);
        if (lane == 0) { W.ctx[0] = 0.0; W.ctx[1] = 0.0; W.ctx[2] = 1.0; W.ctx[3] = 0.0; }
        __syncwarp();
        return;
    }
    const double rt = S.rt;
    C.zt_x = corner_x(S, ci0) + (0.5 * (TCX - 1) + off) * S.h1;
    C.zt_y = corner_y(S, cj0) + (0.5 * (TCY - 1) + off) * S.h2;
    C.inv_rt = S.inv_rt;
    int leaf = -1, node = -1;
    uint32_t b0x = 0, b1x = 0, b0y = 0, b1y = 0;
    if (lane < 4) {
        double x = corner_x(S, (lane & 1) ? ci1 : ci0) + off * S.h1, y = corner_y(S, (lane & 2) ? cj1 : cj0) + off * S.h2;
        uint32_t qx, qy;
        if (quantise(S.L, x, y, qx, qy)) {
            node = find_leaf_node(S.L, qx, qy);
            int lev = __ldg(&S.L.level[node]), ix = __ldg(&S.L.ix[node]), iy = __ldg(&S.L.iy[node]);
            int sh = ML_QBITS - lev;
            leaf = __ldg(&S.L.leaf_id[node]);
            b0x = (uint32_t)ix << sh; b1x = (uint32_t)(ix + 1) << sh;
            b0y = (uint32_t)iy << sh; b1y = (uint32_t)(iy + 1) << sh;
        }
    }
    const int l0 = __shfl_sync(full, leaf, 0), l1 = __shfl_sync(full, leaf, 1), l2 = __shfl_sync(full, leaf, 2), l3 = __shfl_sync(full, leaf, 3);
    const bool one_leaf = l0 >= 0 && l1 == l0 && l2 == l0 && l3 == l0;
    {
        // one slot per distinct leaf, in corner order, at most NSLOT of them
        bool dup = (lane > 0 && leaf == l0) || (lane > 1 && leaf == l1) || (lane > 2 && leaf == l2);
        const bool keep = lane < 4 && leaf >= 0 && !dup;
        const unsigned km = __ballot_sync(full, keep);
        const int slot = __popc(km & ((1u << lane) - 1u));
        if (lane < NSLOT) { W.leaf[lane] = -1; W.node[lane] = -1; W.nd[lane] = 0; W.mode[lane] = -1; }
        __syncwarp();
        if (keep && slot < NSLOT) {
            W.leaf[slot] = leaf; W.node[slot] = node;
            W.bx0[slot] = b0x; W.bx1[slot] = b1x; W.by0[slot] = b0y; W.by1[slot] = b1y;
        }
    }
    __syncwarp();
    // Rectangle sheet inside the rectangle (eq B8): alpha_s = -kappa_star z + conj A(z), A analytic in the open
    // rectangle; the Taylor coefficients of A about every leaf's centre were added to a copy of the leaf's series when the
    // field was made (fmm.cu rect_fold_kernel), so the shift to the tile centre below carries the sheet along: no
    // logarithm per ray (the paper pays four), none per tile.  A tile uses that copy if it lies inside the rectangle
    // and its leaves' copies hold the term (leaves next to the rectangle's border keep eq B7).
    bool fold = false;
    if (S.L.shape == MLENS_SHAPE_RECT && S.L.leaf_fold && W.leaf[0] >= 0)
        fold = fabs(C.zt_x) + rt <= S.L.c1 && fabs(C.zt_y) + rt <= S.L.c2 && __ldg(&S.L.leaf_fold[W.leaf[0]]) != 0 &&
               (W.leaf[1] < 0 || __ldg(&S.L.leaf_fold[W.leaf[1]]) != 0);
    for (int s = 0; s < NSLOT; ++s) {
        if (W.leaf[s] < 0) continue;                              // warp-uniform
        wtile_build_slot(S, W, C, s, rt, fold);
        if (lane == 0 && W.mode[s] == 1 && full_counter) atomicAdd(full_counter, 1ull);
    }
    if (lane == 0 && W.leaf[0] >= 0) {
        // statistics: the near-field list a ray of this tile would sum in the paper's per-ray scheme (roofline accounting)
        atomicAdd(&S.counters[C_TILES], 1ull);
        atomicAdd(&S.counters[C_NEAR_LEAF], (unsigned long long)__ldg(&S.L.near_cnt[W.leaf[0]]));
    }
    // eq 19 inside the disc is linear in z: the farthest ray of the tile decides (the disc is convex)
    const double rmax = sqrt(C.zt_x * C.zt_x + C.zt_y * C.zt_y) + rt;
    // (a field with macro terms beyond linear, reading G23, is never `lin`: its rays take lens_w, which holds that term;
    // make_lens_dev switches the rectangle fold off for such a field, so `fold` is false then)
    const bool lin = !S.L.has_quad && ((S.L.shape == MLENS_SHAPE_DISC && rmax * rmax <= S.L.R2) || fold);
    zero_window(W);
    if (lane == 0) {
        W.ctx[0] = C.zt_x; W.ctx[1] = C.zt_y; W.ctx[2] = C.inv_rt;
        W.ctx[3] = ((one_leaf && W.mode[0] == 0) ? 1.0 : 0.0) + (lin ? 2.0 : 0.0);
    }
    __syncwarp();
}
// Sets up the warp's tile (out of line: once per 1024 rays) and returns its context in registers.
__device__ __forceinline__ void wtile_setup(const ShootDev &S, WarpShared &W, TileCtx &C, long long ci0, long long cj0,
                                            long long ci1, long long cj1, double off) {
    wtile_setup_ool(&S, &W, ci0, cj0, ci1, cj1, off);
    const int flags = (int)W.ctx[3];
    C.zt_x = W.ctx[0]; C.zt_y = W.ctx[1]; C.inv_rt = W.ctx[2]; C.fast = (flags & 1) != 0; C.lin = (flags & 2) != 0;
}

struct ThreadCounters { unsigned int single = 0, small_ = 0, queued = 0, chunks = 0, overflow = 0, fallback = 0, rays = 0, near_ = 0, px_small = 0; };

// One ray of a tile that straddles leaves (or whose series failed its bound), out of line: the slot of the
// ray's leaf if the tile has one for it, else the tree.  Returns alpha_star.
static __device__ __noinline__ double2 eval_one_ool(const ShootDev *Sp, const WarpShared *T, double x, double y, double ux, double uy, int *kind) {
    int s = -1;
    uint32_t qx, qy;
    if (quantise(Sp->L, x, y, qx, qy)) {
#pragma unroll 1
        for (int k = 0; k < NSLOT; ++k)
            if (T->leaf[k] >= 0 && qx >= T->bx0[k] && qx < T->bx1[k] && qy >= T->by0[k] && qy < T->by1[k]) s = k;
    }
    if (s >= 0 && T->mode[s] != 0) s = -1;
    if (s < 0) { *kind = -1; return alpha_fmm_global_ool(&Sp->L, x, y); }
    const int Q = T->q[s];
    double sr = T->t[s][Q].x, si = T->t[s][Q].y;
    for (int j = Q - 1; j >= 0; --j) {
        double2 c = T->t[s][j];
        double tr = fma(sr, ux, fma(-si, uy, c.x));
        double ti = fma(sr, uy, fma(si, ux, c.y));
        sr = tr; si = ti;
    }
    const int nd = T->nd[s];
    for (int k = 0; k < nd; ++k) {
        double dx = x - T->sx[s][k], dy = y - T->sy[s][k];
        double r2 = fma(dx, dx, dy * dy);
        double q = (__double2hiint(r2) >= 0x00100000) ? T->sm[s][k] * fast_rcp(r2) : 0.0;
        sr = fma(q, dx, sr);
        si = fma(-q, dy, si);
    }
    *kind = nd;
    return make_double2(sr, -si);
}

// The RPT rays of one lane when the fast path does not apply (tile straddling leaves, failed bound, partial
// tile, DIRECT mode): one ray at a time, out of line.  Results go through a small local array.
static __device__ __noinline__ void eval_group_ool(const ShootDev *Sp, const WarpShared *T, double x, double ux, double y0, double y1,
                                                   double y2, double y3, double uy0, double duy, unsigned validmask,
                                                   double *w /* [2 RPT] */, int *cnt /* rays, near, fallback */) {
    const ShootDev &S = *Sp;
    static_assert(RPT == 4, "four rows per group");
#pragma unroll 1
    for (int r = 0; r < RPT; ++r) {
        w[2 * r] = 0.0; w[2 * r + 1] = 0.0;
        if (!((validmask >> r) & 1u)) continue;
        const double y = (r == 0) ? y0 : (r == 1) ? y1 : (r == 2) ? y2 : y3;
        ++cnt[0];
        double2 a;
        if (S.eval_mode == MLENS_EVAL_DIRECT) a = direct_all_ool(&S.L, x, y);
        else {
            int kind;
            a = eval_one_ool(Sp, T, x, y, ux, uy0 + duy * (double)r, &kind);
            if (kind >= 0) cnt[1] += kind; else ++cnt[2];
            if (kind >= 0 && S.L.shape == MLENS_SHAPE_RECT && (((int)T->ctx[3]) & 2)) {
                // the slot's series already holds the analytic part of the rectangle sheet (eq B8): only -kappa_star z is left
                w[2 * r] = fma(S.a1_lin, x, -a.x); w[2 * r + 1] = fma(S.a2_lin, y, -a.y);
                continue;
            }
        }
        lens_w(S.L, x, y, a.x, a.y, w[2 * r], w[2 * r + 1]);
    }
}

// Slot of the tile that holds both (x, ya) and (x, yb) -- hence every ray of the column between them, a leaf being
// a box -- with a tile series that passed its bound; -1 if there is none.  Only tiles that straddle leaves ask.
static __device__ __noinline__ int slot_of_column(const ShootDev *Sp, const WarpShared *T, double x, double ya, double yb) {
    uint32_t qx, qa, qb, qx2;
    if (!quantise(Sp->L, x, ya, qx, qa) || !quantise(Sp->L, x, yb, qx2, qb)) return -1;
    int s = -1;
#pragma unroll 1
    for (int k = 0; k < NSLOT; ++k)
        if (T->leaf[k] >= 0 && T->mode[k] == 0 && qx >= T->bx0[k] && qx < T->bx1[k] && qa >= T->by0[k] && qa < T->by1[k] &&
            qb >= T->by0[k] && qb < T->by1[k]) s = k;
    return s;
}

// The full eq 12 from alpha_star where the sheet term is not linear (outside the disc, rectangle): out of line.
static __device__ __noinline__ double2 lens_w_ool(const LensDev *L, double x, double y, double ax, double ay) {
    double wx, wy;
    lens_w(*L, x, y, ax, ay, wx, wy);
    return make_double2(wx, wy);
}

// w(z) of eq 12 for the RPT rays of one lane (same column x, consecutive rows).
// float pairs for the packed single-precision FMA of sm_100 (FFMA2)
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float lo2(unsigned long long v) { return __uint_as_float((unsigned int)v); }
__device__ __forceinline__ float hi2(unsigned long long v) { return __uint_as_float((unsigned int)(v >> 32)); }
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// F32 (the paper's single-precision mode; MLENS_EVAL_FMM_F32): the tile series and the tile's direct stars
// are evaluated in float32 -- the series in the tile's own argument u, the separations from the stars taken in
// float64 and then rounded, so that only the deflection, never a position, is rounded to 24 bits -- and the
// macro terms in float64.
template <bool F32>
__device__ __forceinline__ void eval_rays(const ShootDev &S, const WarpShared &T, const TileCtx &C, double x, double ux,
                                          const double (&y)[RPT], const double (&uy)[RPT],
                                          const bool (&valid)[RPT], double (&wx)[RPT], double (&wy)[RPT], ThreadCounters &tc) {
    bool all = true;
#pragma unroll
    for (int r = 0; r < RPT; ++r) all = all && valid[r];
    int s = 0;
    bool fastlane = C.fast && all;
    if (!C.fast && all && S.eval_mode == MLENS_EVAL_FMM) {
        // a tile over two leaves: the lanes whose four rays share a leaf still take the fast path, each with its slot
        s = slot_of_column(&S, &T, x, y[0], y[RPT - 1]);
        fastlane = s >= 0;
        s = max(s, 0);
    }
    if (fastlane && F32) {
        const int Q = T.q[s];
        const double2 *t = T.t[s];
        const float uxf = (float)ux;
        float uyf[RPT], sr[RPT], si[RPT];
#pragma unroll
        for (int r = 0; r < RPT; ++r) uyf[r] = (float)uy[r];
        // Blackwell's packed FFMA2 (fma.rn.f32x2) does two rays per instruction: the chains of rows (0, 1) and (2, 3)
        // travel as float pairs, eight instructions per two terms and pair instead of sixteen
        static_assert(RPT == 4, "two ray pairs");
        const unsigned long long UX = pack2(uxf, uxf);
        const unsigned long long UYa = pack2(uyf[0], uyf[1]), UYb = pack2(uyf[2], uyf[3]);
        const unsigned long long NUYa = pack2(-uyf[0], -uyf[1]), NUYb = pack2(-uyf[2], -uyf[3]);
        double2 cd = t[Q];
        unsigned long long sra = pack2((float)cd.x, (float)cd.x), sia = pack2((float)cd.y, (float)cd.y), srb = sra, sib = sia;
        int j = Q - 1;
#pragma unroll 1
        for (; j >= 1; j -= 2) {
            const double2 d1 = t[j], d0 = t[j - 1];
            const float c1x = (float)d1.x, c1y = (float)d1.y, c0x = (float)d0.x, c0y = (float)d0.y;
            const unsigned long long C1X = pack2(c1x, c1x), C1Y = pack2(c1y, c1y), C0X = pack2(c0x, c0x), C0Y = pack2(c0y, c0y);
            const unsigned long long tra = fma2(sra, UX, fma2(sia, NUYa, C1X)), tia = fma2(sra, UYa, fma2(sia, UX, C1Y));
            const unsigned long long trb = fma2(srb, UX, fma2(sib, NUYb, C1X)), tib = fma2(srb, UYb, fma2(sib, UX, C1Y));
            sra = fma2(tra, UX, fma2(tia, NUYa, C0X)); sia = fma2(tra, UYa, fma2(tia, UX, C0Y));
            srb = fma2(trb, UX, fma2(tib, NUYb, C0X)); sib = fma2(trb, UYb, fma2(tib, UX, C0Y));
        }
        if (j == 0) {
            cd = t[0];
            const float c0x = (float)cd.x, c0y = (float)cd.y;
            const unsigned long long C0X = pack2(c0x, c0x), C0Y = pack2(c0y, c0y);
            const unsigned long long tra = fma2(sra, UX, fma2(sia, NUYa, C0X)), tia = fma2(sra, UYa, fma2(sia, UX, C0Y));
            const unsigned long long trb = fma2(srb, UX, fma2(sib, NUYb, C0X)), tib = fma2(srb, UYb, fma2(sib, UX, C0Y));
            sra = tra; sia = tia; srb = trb; sib = tib;
        }
        sr[0] = lo2(sra); sr[1] = hi2(sra); sr[2] = lo2(srb); sr[3] = hi2(srb);
        si[0] = lo2(sia); si[1] = hi2(sia); si[2] = lo2(sib); si[3] = hi2(sib);
        const int nd = T.nd[s];
        tc.rays += RPT;
        tc.near_ += (unsigned int)(nd * RPT);
#pragma unroll 1
        for (int k = 0; k < nd; ++k) {
            // the separation is taken in float64 and then rounded: a ray next to a star keeps its relative accuracy
            const double Yd = T.sy[s][k];
            const float M = (float)T.sm[s][k];
            const float dx = (float)(x - T.sx[s][k]);
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const float dy = (float)(y[r] - Yd);
                const float r2 = fmaf(dx, dx, dy * dy);
                const float q = (r2 > 0.0f) ? __fdividef(M, r2) : 0.0f;                   // reading G11: skip r = 0
                sr[r] = fmaf(q, dx, sr[r]);
                si[r] = fmaf(-q, dy, si[r]);
            }
        }
        if (C.lin) {
#pragma unroll
            for (int r = 0; r < RPT; ++r) { wx[r] = fma(S.a1_lin, x, -(double)sr[r]); wy[r] = fma(S.a2_lin, y[r], (double)si[r]); }
        } else {
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const double2 w = lens_w_ool(&S.L, x, y[r], (double)sr[r], -(double)si[r]);
                wx[r] = w.x; wy[r] = w.y;
            }
        }
    } else if (fastlane) {
        // the common case: the four rays in one leaf, RPT independent Horner chains share every coefficient load
        const int Q = T.q[s];
        const double2 *t = T.t[s];
        double sr[RPT], si[RPT];
        double2 c = t[Q];
#pragma unroll
        for (int r = 0; r < RPT; ++r) { sr[r] = c.x; si[r] = c.y; }
        int j = Q - 1;
        // two terms per trip: the chains ping-pong between two register sets, no copies
#pragma unroll 1
        for (; j >= 1; j -= 2) {
            const double2 c1 = t[j], c0 = t[j - 1];
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const double tr = fma(sr[r], ux, fma(-si[r], uy[r], c1.x));
                const double ti = fma(sr[r], uy[r], fma(si[r], ux, c1.y));
                sr[r] = fma(tr, ux, fma(-ti, uy[r], c0.x));
                si[r] = fma(tr, uy[r], fma(ti, ux, c0.y));
            }
        }
        if (j == 0) {
            c = t[0];
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const double tr = fma(sr[r], ux, fma(-si[r], uy[r], c.x));
                const double ti = fma(sr[r], uy[r], fma(si[r], ux, c.y));
                sr[r] = tr; si[r] = ti;
            }
        }
        const int nd = T.nd[s];
        tc.rays += RPT;
        tc.near_ += (unsigned int)(nd * RPT);
#pragma unroll 1
        for (int k = 0; k < nd; ++k) {
            double X = T.sx[s][k], Y = T.sy[s][k], M = T.sm[s][k];
            const double dx = x - X;
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                double dy = y[r] - Y;
                double r2 = fma(dx, dx, dy * dy);
                double q = (__double2hiint(r2) >= 0x00100000) ? M * fast_rcp(r2) : 0.0;   // reading G11: skip r = 0
                sr[r] = fma(q, dx, sr[r]);
                si[r] = fma(-q, dy, si[r]);
            }
        }
        if (C.lin) {
#pragma unroll
            for (int r = 0; r < RPT; ++r) { wx[r] = fma(S.a1_lin, x, -sr[r]); wy[r] = fma(S.a2_lin, y[r], si[r]); }
        } else {
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const double2 w = lens_w_ool(&S.L, x, y[r], sr[r], -si[r]);
                wx[r] = w.x; wy[r] = w.y;
            }
        }
    } else {
        double w[2 * RPT];
        int cnt[3] = {0, 0, 0};
        unsigned vm = 0;
#pragma unroll
        for (int r = 0; r < RPT; ++r) vm |= valid[r] ? (1u << r) : 0u;
        eval_group_ool(&S, &T, x, ux, y[0], y[1], y[2], y[3], uy[0], uy[1] - uy[0], vm, w, cnt);
        tc.rays += cnt[0]; tc.near_ += cnt[1]; tc.fallback += cnt[2];
#pragma unroll
        for (int r = 0; r < RPT; ++r) { wx[r] = w[2 * r]; wy[r] = w[2 * r + 1]; }
    }
}

}  // namespace ml
