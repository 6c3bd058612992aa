// eval.cu -- lens-equation evaluation at caller-given points (the 1e-8 parity surface) and the
// seeded star-field generator.
#include "device.cuh"

namespace ml {

LensDev make_lens_dev(const mlens_field *f) {
    LensDev L;
    L.one_minus_kappa = 1.0 - f->kappa_tot;
    L.gamma = f->gamma;
    L.q111 = f->quad[0]; L.q112 = f->quad[1]; L.q122 = f->quad[2]; L.q222 = f->quad[3];
    L.has_quad = (f->quad[0] != 0.0 || f->quad[1] != 0.0 || f->quad[2] != 0.0 || f->quad[3] != 0.0) ? 1 : 0;
    L.kappa_star = f->kappa_star;
    L.theta2 = f->theta * f->theta;
    L.shape = f->shape;
    L.R2 = f->R * f->R;
    L.c1 = f->c1; L.c2 = f->c2;
    L.root_half = f->root_half;
    L.qscale = (double)(1u << ML_QBITS) / (2.0 * f->root_half);
    const Tree &t = f->tree;
    L.child0 = t.child0.p; L.leaf_id = t.leaf_id.p; L.level = t.level.p; L.ix = t.ix.p; L.iy = t.iy.p;
    L.near_cnt = t.near_cnt.p; L.near_x = t.near_x.p; L.near_y = t.near_y.p; L.near_m = t.near_m.p;
    L.ecoef = t.ecoef.p;
    // (with macro terms beyond linear every ray goes through lens_w, sheet included: no folded series then)
    const bool fold_ok = f->shape == MLENS_SHAPE_RECT && !L.has_quad;
    L.ecoef_shoot = (fold_ok && t.ecoef_shoot.p) ? t.ecoef_shoot.p : t.ecoef.p;
    L.leaf_fold = fold_ok ? t.leaf_fold.p : nullptr;
    L.p = f->order; L.p1 = f->order + 1;
    L.sx = f->sx.p; L.sy = f->sy.p; L.sm = f->sm.p;
    L.n_stars = f->n_stars;
    return L;
}

// FMM evaluation: one thread per point (eq 23).
__global__ void deflect_fmm_kernel(LensDev L, long long n, const double *zx, const double *zy,
                                   double *ox, double *oy, int full_lens) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double x = zx[i], y = zy[i], ax, ay;
    alpha_fmm_global(L, x, y, ax, ay);
    if (full_lens) { double wx, wy; lens_w(L, x, y, ax, ay, wx, wy); ox[i] = wx; oy[i] = wy; }
    else { ox[i] = ax; oy[i] = ay; }
}

// Direct sum over all stars (eq 13): warp-tiled P2P -- every thread owns one point, the block streams its
// share of the stars through shared memory in tiles and each star value is reused by all threads.  The stars
// are split over gridDim.y blocks (few points against many stars must still fill the GPU); each block adds its
// Kahan-compensated partial sum to the accumulators, direct_finish_kernel turns them into the result.
static const int DP_T = 128, DP_TILE = 256;
__global__ void deflect_direct_kernel(LensDev L, long long n, const double *zx, const double *zy, long long stars_per_block,
                                      double *accx, double *accy) {
    __shared__ double tx[DP_TILE], ty[DP_TILE], tm[DP_TILE];
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    bool act = i < n;
    double x = act ? zx[i] : 0.0, y = act ? zy[i] : 0.0;
    double sx = 0.0, sy = 0.0, cx = 0.0, cy = 0.0;         // Kahan-compensated sums
    const long long s0 = blockIdx.y * stars_per_block;
    const long long s1 = (s0 + stars_per_block < L.n_stars) ? s0 + stars_per_block : L.n_stars;
    for (long long base = s0; base < s1; base += DP_TILE) {
        __syncthreads();
        for (int e = threadIdx.x; e < DP_TILE; e += DP_T) {
            long long j = base + e;
            bool v = j < s1;
            tx[e] = v ? L.sx[j] : 0.0; ty[e] = v ? L.sy[j] : 0.0; tm[e] = v ? L.sm[j] : 0.0;
        }
        __syncthreads();
        int cnt = (int)((s1 - base < DP_TILE) ? (s1 - base) : DP_TILE);
#pragma unroll 4
        for (int e = 0; e < cnt; ++e) {
            double dx = x - tx[e], dy = y - ty[e];
            double r2 = dx * dx + dy * dy;
            double q = (r2 > 0.0) ? tm[e] / r2 : 0.0;
            double vx = __dadd_rn(__dmul_rn(q, dx), -cx), vy = __dadd_rn(__dmul_rn(q, dy), -cy);
            double tx_ = __dadd_rn(sx, vx), ty_ = __dadd_rn(sy, vy);
            cx = __dadd_rn(__dadd_rn(tx_, -sx), -vx); cy = __dadd_rn(__dadd_rn(ty_, -sy), -vy);
            sx = tx_; sy = ty_;
        }
    }
    if (!act) return;
    if (gridDim.y == 1) { accx[i] = sx; accy[i] = sy; }
    else { atomicAdd(&accx[i], sx); atomicAdd(&accy[i], sy); }
}
__global__ void direct_finish_kernel(LensDev L, long long n, const double *zx, const double *zy, double *ox, double *oy, int full_lens) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double ax = L.theta2 * ox[i], ay = L.theta2 * oy[i];
    if (full_lens) { double wx, wy; lens_w(L, zx[i], zy[i], ax, ay, wx, wy); ox[i] = wx; oy[i] = wy; }
    else { ox[i] = ax; oy[i] = ay; }
}

int deflect_points(const mlens_field *f, int64_t n, const double *zx, const double *zy, double *ox_, double *oy_,
                   int eval_mode, int full_lens, cudaStream_t s) {
    if (n <= 0) return MLENS_OK;
    LensDev L = make_lens_dev(f);
    if (eval_mode == MLENS_EVAL_FMM) {
        long long blocks = (n + 127) / 128;
        ML_LAUNCH(deflect_fmm_kernel, (unsigned)blocks, 128, 0, s, L, n, zx, zy, ox_, oy_, full_lens);
    } else {
        long long bx = (n + DP_T - 1) / DP_T;
        int dev = 0, nsm = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
        // enough blocks for 8 per SM; a block's share of the stars is whole tiles
        long long by = (8ll * nsm + bx - 1) / bx;
        long long max_by = (L.n_stars + 4 * DP_TILE - 1) / (4 * DP_TILE);
        if (by > max_by) by = max_by;
        if (by < 1) by = 1;
        if (by > 65535) by = 65535;
        long long per = (L.n_stars + by - 1) / by;
        per = (per + DP_TILE - 1) / DP_TILE * DP_TILE;
        if (per < DP_TILE) per = DP_TILE;
        by = (L.n_stars + per - 1) / per;
        if (by < 1) by = 1;
        if (by > 1) {
            ML_CUDA(cudaMemsetAsync(ox_, 0, (size_t)n * 8, s));
            ML_CUDA(cudaMemsetAsync(oy_, 0, (size_t)n * 8, s));
        }
        ML_LAUNCH(deflect_direct_kernel, dim3((unsigned)bx, (unsigned)by), DP_T, 0, s, L, n, zx, zy, per, ox_, oy_);
        ML_LAUNCH(direct_finish_kernel, (unsigned)((n + 255) / 256), 256, 0, s, L, n, zx, zy, ox_, oy_, full_lens);
    }
    ML_CUDA(cudaGetLastError());
    return MLENS_OK;
}

// ------------------------------------------------------------------------------------------------
// Seeded star field (generator spec: DESIGN.md section 4).
// draw(seed, n) = fin(fin(seed) + (n+1) * 0x9E3779B97F4A7C15), fin = the SplitMix64 finaliser;
// u = (draw >> 11) * 2^-53.  Star i uses counters 3i (radius or x1), 3i+1 (angle or x2), 3i+2 (mass).
__device__ __forceinline__ unsigned long long sm64_fin(unsigned long long x) {
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull;
    x ^= x >> 27; x *= 0x94D049BB133111EBull;
    x ^= x >> 31;
    return x;
}
__device__ __forceinline__ double sm64_u(unsigned long long seed_fin, unsigned long long n) {
    unsigned long long r = sm64_fin(seed_fin + (n + 1ull) * 0x9E3779B97F4A7C15ull);
    return (double)(r >> 11) * 0x1.0p-53;
}

// (cos, sin)(2 pi v) by octant reduction and fixed Taylor polynomials (fma Horner): the spec fixes the
// polynomial so that positions are reproducible bit for bit on any IEEE-754 machine.
__device__ __forceinline__ void unit_vec(double v, double &c_out, double &s_out) {
    double t8 = 8.0 * v;
    int k = (int)t8;
    double fr = t8 - (double)k;
    if (k & 1) fr = 1.0 - fr;
    double th = __dmul_rn(fr, 0.78539816339744830962);
    double q = __dmul_rn(th, th);
    double S = 1.0 / 355687428096000.0;
    S = fma(S, q, -1.0 / 1307674368000.0);
    S = fma(S, q, 1.0 / 6227020800.0);
    S = fma(S, q, -1.0 / 39916800.0);
    S = fma(S, q, 1.0 / 362880.0);
    S = fma(S, q, -1.0 / 5040.0);
    S = fma(S, q, 1.0 / 120.0);
    S = fma(S, q, -1.0 / 6.0);
    S = fma(S, q, 1.0);
    double sn = __dmul_rn(th, S);
    double C = 1.0 / 6402373705728000.0;
    C = fma(C, q, -1.0 / 20922789888000.0);
    C = fma(C, q, 1.0 / 87178291200.0);
    C = fma(C, q, -1.0 / 479001600.0);
    C = fma(C, q, 1.0 / 3628800.0);
    C = fma(C, q, -1.0 / 40320.0);
    C = fma(C, q, 1.0 / 720.0);
    C = fma(C, q, -1.0 / 24.0);
    C = fma(C, q, 0.5);
    double cs = fma(-C, q, 1.0);
    switch (k & 7) {
        case 0: c_out = cs; s_out = sn; break;
        case 1: c_out = sn; s_out = cs; break;
        case 2: c_out = -sn; s_out = cs; break;
        case 3: c_out = -cs; s_out = sn; break;
        case 4: c_out = -cs; s_out = -sn; break;
        case 5: c_out = -sn; s_out = -cs; break;
        case 6: c_out = sn; s_out = -cs; break;
        default: c_out = cs; s_out = -sn; break;
    }
}

__global__ void starfield_kernel(unsigned long long seed_fin, long long n, int shape, double a1, double a2,
                                 int mass_law, double inv_e, double loe, double dhe, double inv_mean,
                                 double *x, double *y, double *m) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double u1 = sm64_u(seed_fin, 3ull * i), u2 = sm64_u(seed_fin, 3ull * i + 1ull), u3 = sm64_u(seed_fin, 3ull * i + 2ull);
    if (shape == MLENS_SHAPE_DISC) {
        double r = __dmul_rn(a1, sqrt(u1)), c, s;
        unit_vec(u2, c, s);
        x[i] = __dmul_rn(r, c); y[i] = __dmul_rn(r, s);
    } else {
        x[i] = __dmul_rn(a1, __dadd_rn(__dmul_rn(2.0, u1), -1.0));
        y[i] = __dmul_rn(a2, __dadd_rn(__dmul_rn(2.0, u2), -1.0));
    }
    m[i] = (mass_law == MLENS_MASS_POWER) ? pow(__dadd_rn(loe, __dmul_rn(u3, dhe)), inv_e) * inv_mean : 1.0;
}

int generate_stars(uint64_t seed, int64_t n, int shape, double a1, double a2, int mass_law, double a,
                   double lo, double hi, double *x, double *y, double *m, cudaStream_t s) {
    if (n <= 0) return MLENS_OK;
    unsigned long long sf = seed;
    sf ^= sf >> 30; sf *= 0xBF58476D1CE4E5B9ull; sf ^= sf >> 27; sf *= 0x94D049BB133111EBull; sf ^= sf >> 31;
    double e = 1.0 - a, loe = 0, dhe = 0, inv_mean = 1.0, inv_e = 1.0;
    if (mass_law == MLENS_MASS_POWER) {
        if (!(lo > 0) || !(hi > lo) || e == 0.0 || e == -1.0) { set_error("bad mass law"); return MLENS_EINVAL; }
        loe = pow(lo, e); double hie = pow(hi, e);
        dhe = hie - loe;
        double mean = (e / (e + 1.0)) * (pow(hi, e + 1.0) - pow(lo, e + 1.0)) / (hie - loe);
        inv_mean = 1.0 / mean; inv_e = 1.0 / e;
    }
    long long blocks = (n + 255) / 256;
    ML_LAUNCH(starfield_kernel, (unsigned)blocks, 256, 0, s, sf, n, shape, a1, a2, mass_law, inv_e, loe, dhe, inv_mean, x, y, m);
    ML_CUDA(cudaGetLastError());
    return MLENS_OK;
}

}  // namespace ml
