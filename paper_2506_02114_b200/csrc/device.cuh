// device.cuh -- device-side building blocks shared by the evaluation and shooting kernels.
#pragma once
#include "common.cuh"

namespace ml {

// ---- complex arithmetic on double2 (x = re, y = im)
__host__ __device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__host__ __device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ double2 cscale(double2 a, double s) { return make_double2(a.x * s, a.y * s); }
__host__ __device__ __forceinline__ double2 cinv(double2 a) {
    double r = 1.0 / (a.x * a.x + a.y * a.y);
    return make_double2(a.x * r, -a.y * r);
}
__host__ __device__ __forceinline__ double2 cpowi(double2 a, int n) {     // a^n, n >= 0, binary powering
    double2 r = make_double2(1.0, 0.0);
    while (n) {
        if (n & 1) r = cmul(r, a);
        a = cmul(a, a);
        n >>= 1;
    }
    return r;
}

// 1/a to double precision from the 20-bit hardware seed: one cubic step, e^3 ~ 2^-60 (a normal, finite, > 0)
__device__ __forceinline__ double fast_rcp(double a) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double e = fma(-a, y, 1.0);
    double t = fma(e, e, e);
    return fma(y, t, y);
}

// ---- everything a kernel needs to evaluate the lens equation (eq 12)
struct LensDev {
    double one_minus_kappa, gamma, kappa_star, theta2;
    double q111, q112, q122, q222;      // macro potential's third derivatives at the origin (App. D, reading G23)
    int has_quad;                       // 0: constant kappa, gamma (the terms are not even touched)
    int shape;
    double R2, c1, c2;
    // tree
    double root_half, qscale;           // quantised coordinate = floor((x + root_half) * qscale)
    const int *child0, *leaf_id, *level, *ix, *iy;
    const int *near_cnt;
    const double *near_x, *near_y, *near_m;
    const double2 *ecoef;
    const double2 *ecoef_shoot;         // rectangle fields: ecoef + the Taylor series of the sheet's analytic part (else = ecoef)
    const unsigned char *leaf_fold;     // rectangle fields: 1 where ecoef_shoot holds that part
    int p, p1;                          // order, coefficients per expansion (stride of ecoef)
    // all stars (DIRECT mode and out-of-root fallback)
    const double *sx, *sy, *sm;
    long long n_stars;
};

// Quantised coordinate used for tree membership (stars and rays alike).
__device__ __forceinline__ bool quantise(const LensDev &L, double x, double y, uint32_t &qx, uint32_t &qy) {
    double fx = (x + L.root_half) * L.qscale, fy = (y + L.root_half) * L.qscale;
    const double lim = (double)(1u << ML_QBITS);
    bool inside = (fx >= 0.0) && (fy >= 0.0) && (fx < lim) && (fy < lim);
    qx = inside ? (uint32_t)fx : 0u;
    qy = inside ? (uint32_t)fy : 0u;
    return inside;
}

// Descend from the root to the childless node that owns (qx, qy).
__device__ __forceinline__ int find_leaf_node(const LensDev &L, uint32_t qx, uint32_t qy) {
    int node = 0, lev = 0;
    int c = __ldg(&L.child0[0]);
    while (c >= 0) {
        int sh = ML_QBITS - 1 - lev;
        node = c + (int)((qx >> sh) & 1u) + 2 * (int)((qy >> sh) & 1u);
        ++lev;
        c = __ldg(&L.child0[node]);
    }
    return node;
}

// Near-field direct sum, eq 13 restricted to the leaf's list (reading G11: skip r = 0).
// Returns sum m (z - z_i)/|z - z_i|^2 (without theta^2).
__device__ __forceinline__ void near_sum(const double *nx, const double *ny, const double *nm, int cnt,
                                         double x, double y, double &ax, double &ay) {
    double sx = 0.0, sy = 0.0;
    for (int i = 0; i < cnt; ++i) {
        double dx = x - nx[i], dy = y - ny[i];
        double r2 = dx * dx + dy * dy;
        double q = (r2 > 0.0) ? nm[i] / r2 : 0.0;
        sx = fma(q, dx, sx);
        sy = fma(q, dy, sy);
    }
    ax = sx; ay = sy;
}

// Far field: alpha_far = conj( sum_{l=0}^{p-1} e_l zeta^l ), e_l = (l+1) c_{l+1} theta^2 / L
// (eq 24 / C4; reading G1), Horner.
__device__ __forceinline__ void far_horner(const double2 *e, int p, double zr, double zi, double &ax, double &ay) {
    double sr = 0.0, si = 0.0;
    for (int l = p - 1; l >= 0; --l) {
        double2 c = e[l];
        double tr = fma(sr, zr, fma(-si, zi, c.x));
        double ti = fma(sr, zi, fma(si, zr, c.y));
        sr = tr; si = ti;
    }
    ax = sr; ay = -si;
}

// z log z with 0 log 0 = 0, principal branch
__device__ __forceinline__ double2 zlogz(double2 v) {
    if (v.x == 0.0 && v.y == 0.0) return make_double2(0.0, 0.0);
    double2 lg = make_double2(0.5 * log(v.x * v.x + v.y * v.y), atan2(v.y, v.x));
    return cmul(v, lg);
}

// Smooth-sheet deflection alpha_s of a rectangle, eq B7.  Kept out of line: four complex logarithms.
static __device__ __noinline__ double2 sheet_rect(double c1, double c2, double ks, double x, double y) {
    // conj z = (x, -y); corners c = (c1, c2), conj c = (c1, -c2)
    double2 t1 = zlogz(make_double2(c1 - x, c2 + y));       //  c - conj z
    double2 t2 = zlogz(make_double2(c1 - x, -c2 + y));      //  conj c - conj z
    double2 t3 = zlogz(make_double2(-c1 - x, -c2 + y));     // -c - conj z
    double2 t4 = zlogz(make_double2(-c1 - x, c2 + y));      // -conj c - conj z
    double Sr = t1.x - t2.x + t3.x - t4.x, Si = t1.y - t2.y + t3.y - t4.y;
    const double inv_pi = 0.31830988618379067154;
    // (-ks i/pi) * S = (ks/pi) (Si, -Sr)
    double rx = ks * inv_pi * Si, ry = -ks * inv_pi * Sr;
    bool in2 = (y >= -c2) && (y <= c2);
    if (in2 && x >= -c1 && x <= c1) rx -= ks * (2.0 * c1 + 2.0 * x);
    if (in2 && x - c1 >= 0.0) rx -= ks * 4.0 * c1;
    return make_double2(rx, ry);
}

// Smooth-sheet deflection alpha_s: disc eq 19, rectangle eq B7.
__device__ __forceinline__ void sheet(const LensDev &L, double x, double y, double &ax, double &ay) {
    if (L.shape == MLENS_SHAPE_DISC) {
        double r2 = x * x + y * y;
        if (r2 <= L.R2) { ax = -L.kappa_star * x; ay = -L.kappa_star * y; }
        else { double q = L.kappa_star * L.R2 * fast_rcp(r2); ax = -q * x; ay = -q * y; }
        return;
    }
    double2 a = sheet_rect(L.c1, L.c2, L.kappa_star, x, y);
    ax = a.x; ay = a.y;
}

// All stars, for DIRECT mode and rays outside the root square.
__device__ __forceinline__ void direct_all(const LensDev &L, double x, double y, double &ax, double &ay) {
    double sx = 0.0, sy = 0.0;
    for (long long i = 0; i < L.n_stars; ++i) {
        double dx = x - __ldg(&L.sx[i]), dy = y - __ldg(&L.sy[i]);
        double r2 = dx * dx + dy * dy;
        double q = (r2 > 0.0) ? __ldg(&L.sm[i]) / r2 : 0.0;
        sx = fma(q, dx, sx);
        sy = fma(q, dy, sy);
    }
    ax = sx; ay = sy;
}

// alpha_star(z)/theta^2-scaled pieces from global memory for one point: FMM evaluation (eq 23).
__device__ __forceinline__ void alpha_fmm_global(const LensDev &L, double x, double y, double &ax, double &ay) {
    uint32_t qx, qy;
    if (!quantise(L, x, y, qx, qy)) {                // outside the root: plain sum over all stars
        direct_all(L, x, y, ax, ay);
        ax *= L.theta2; ay *= L.theta2;
        return;
    }
    int node = find_leaf_node(L, qx, qy);
    int leaf = __ldg(&L.leaf_id[node]);
    int lev = __ldg(&L.level[node]);
    double half = L.root_half / (double)(1 << lev);
    double cx = -L.root_half + (2.0 * __ldg(&L.ix[node]) + 1.0) * half;
    double cy = -L.root_half + (2.0 * __ldg(&L.iy[node]) + 1.0) * half;
    double nx_, ny_, fx, fy;
    near_sum(L.near_x + (size_t)leaf * ML_NEAR, L.near_y + (size_t)leaf * ML_NEAR,
             L.near_m + (size_t)leaf * ML_NEAR, __ldg(&L.near_cnt[leaf]), x, y, nx_, ny_);
    double inv = 1.0 / half;
    far_horner(L.ecoef + (size_t)leaf * L.p1, L.p, (x - cx) * inv, (y - cy) * inv, fx, fy);
    ax = fma(L.theta2, nx_, fx);
    ay = fma(L.theta2, ny_, fy);
}

// Out-of-line copies for the shooting kernels' rare paths (keeps their hot loops inside the instruction cache).
static __device__ __noinline__ double2 alpha_fmm_global_ool(const LensDev *L, double x, double y) {
    double ax, ay;
    alpha_fmm_global(*L, x, y, ax, ay);
    return make_double2(ax, ay);
}
static __device__ __noinline__ double2 direct_all_ool(const LensDev *L, double x, double y) {
    double ax, ay;
    direct_all(*L, x, y, ax, ay);
    return make_double2(ax * L->theta2, ay * L->theta2);
}

// Second-order term of the macro deflection (App. D; reading G23): w -= (1/2) psi_ijk x_j x_k.  A uniform
// branch: fields without it (every BASELINE config) execute one predicate.
__device__ __forceinline__ void macro_quad(const LensDev &L, double x, double y, double &wx, double &wy) {
    if (L.has_quad) {
        wx -= 0.5 * (L.q111 * x * x + 2.0 * L.q112 * x * y + L.q122 * y * y);
        wy -= 0.5 * (L.q112 * x * x + 2.0 * L.q122 * x * y + L.q222 * y * y);
    }
}

// w of eq 12 from alpha_star: w = (1-kappa) z + gamma conj z - alpha_star - alpha_s
__device__ __forceinline__ void lens_w(const LensDev &L, double x, double y, double ax, double ay,
                                       double &wx, double &wy) {
    double sx_, sy_;
    sheet(L, x, y, sx_, sy_);
    wx = (L.one_minus_kappa + L.gamma) * x - ax - sx_;
    wy = (L.one_minus_kappa - L.gamma) * y - ay - sy_;
    macro_quad(L, x, y, wx, wy);
}

LensDev make_lens_dev(const mlens_field *f);

}  // namespace ml
