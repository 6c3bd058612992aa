/* mlens_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct restatement of what the hot path of
 * arXiv 2506.02114 computes ("P:n" = /root/reference/PAPER.md line n):
 *   - the lens equation in complex form with a DIRECT SUM over ALL stars
 *     (no tree, no multipoles), accumulated in long double;
 *   - the smooth-sheet term for a disc (eq 19) or a rectangle (eq B7);
 *   - the image-plane ray grid (eq 14-16, A6);
 *   - inverse polygon mapping by brute force: every mapped triangle is clipped
 *     (Sutherland-Hodgman) against EVERY pixel of its bounding box;
 *   - inverse ray shooting counts;
 *   - the seeded star-field generator (own implementation of the counter RNG
 *     specified in DESIGN.md section 4);
 *   - the FMM expansion coefficients BY THEIR DEFINITIONS (eq C2, eq C6 summed
 *     over stars), used only to pin the CUDA operators;
 *   - what the paper reads off a map: a light curve along a straight track (Fig 4 P:212,
 *     Fig 8) and the histogram of log10(mu/mu_ref) (Fig 5, Fig 10).
 * It shares no code, header, table or constant with the CUDA library and is
 * never tuned.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline
 * / --impl reference legs may load it.
 *
 * Parity pins (tests/test_oracle_*.py): point-lens magnification, Chang-Refsdal
 * caustic cusps, rectangle sheet vs 2-D quadrature of eq B1, affine-map
 * exactness of IPM, area conservation, mean magnification, Monte-Carlo area on
 * tiny inputs, RNG uniformity and closed-form moments; the second-order macro
 * terms (reading G23) by the closed-form fold map (image positions, flux per
 * pixel column, pixel means) and a finite-difference Jacobian.  Unpinned: the paper's
 * own absolute map values (its figures and star files are not available).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

typedef struct {
    double kappa_tot, kappa_star, gamma, theta_star;
    int32_t shape;      /* 0 = disc of radius R, 1 = rectangle with corner (c1, c2) */
    int32_t pad_;
    double R, c1, c2;
    int64_t n_stars;
    const double *x, *y, *m;
    /* Macro model beyond linear (App. D, P:694-702 gives the idea -- "the chosen order to which the potential is Taylor
     * expanded" -- and no formula; reading G23): third derivatives psi_111, psi_112, psi_122, psi_222 of the
     * macro potential at the origin.  All zero = the paper's constant kappa, gamma. */
    double t111, t112, t122, t222;
} orc_field;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* Star deflection, eq 13: alpha_star(z) = theta^2 sum m_i/(conj z - conj z_i)
 * = theta^2 sum m_i (z - z_i)/|z - z_i|^2  (eq 8).  All stars, long double.
 * Reading G11: a ray exactly on a star skips that star.                      */
static void alpha_star_1(const orc_field *f, double zx, double zy, ld *ax, ld *ay)
{
    ld sx = 0, sy = 0;
    for (int64_t i = 0; i < f->n_stars; ++i) {
        ld dx = (ld)zx - (ld)f->x[i], dy = (ld)zy - (ld)f->y[i];
        ld r2 = dx * dx + dy * dy;
        if (r2 == 0) continue;
        ld q = (ld)f->m[i] / r2;
        sx += q * dx;
        sy += q * dy;
    }
    ld t2 = (ld)f->theta_star * (ld)f->theta_star;
    *ax = t2 * sx;
    *ay = t2 * sy;
}

/* z log z with 0 log 0 = 0 (principal branch, cut on the negative real axis) */
static long double complex zlogz(long double complex v)
{
    if (creall(v) == 0 && cimagl(v) == 0) return 0;
    return v * clogl(v);
}

/* Smooth sheet: disc eq 19; rectangle eq B7. */
static void alpha_smooth_1(const orc_field *f, double zx, double zy, ld *ax, ld *ay)
{
    ld ks = f->kappa_star;
    if (f->shape == 0) {
        ld r2 = (ld)zx * zx + (ld)zy * zy, R2 = (ld)f->R * f->R;
        if (r2 <= R2) { *ax = -ks * zx; *ay = -ks * zy; }
        else { /* -ks R^2 / conj(z) = -ks R^2 z/|z|^2 */
            *ax = -ks * R2 * zx / r2; *ay = -ks * R2 * zy / r2;
        }
        return;
    }
    const ld PI = 3.14159265358979323846264338327950288L;
    long double complex z = (ld)zx + (ld)zy * I, zb = conjl(z);
    long double complex c = (ld)f->c1 + (ld)f->c2 * I, cb = conjl(c);
    long double complex S = zlogz(c - zb) - zlogz(cb - zb) + zlogz(-c - zb) - zlogz(-cb - zb);
    long double complex a = (-ks * I / PI) * S;
    int in2 = (zy >= -f->c2 && zy <= f->c2);
    int box = in2 && (zx >= -f->c1 && zx <= f->c1);
    if (box) a += -ks * (c + cb + z + zb);
    if (in2 && zx - f->c1 >= 0) a += -ks * 2 * (c + cb);   /* B_(inf,c2) * H(Re z - c1) */
    *ax = creall(a);
    *ay = cimagl(a);
}

void orc_alpha_star(const orc_field *f, int64_t n, const double *zx, const double *zy,
                    double *ax, double *ay)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t k = 0; k < n; ++k) {
        ld a, b;
        alpha_star_1(f, zx[k], zy[k], &a, &b);
        ax[k] = (double)a; ay[k] = (double)b;
    }
}

void orc_alpha_smooth(const orc_field *f, int64_t n, const double *zx, const double *zy,
                      double *ax, double *ay)
{
    for (int64_t k = 0; k < n; ++k) {
        ld a, b;
        alpha_smooth_1(f, zx[k], zy[k], &a, &b);
        ax[k] = (double)a; ay[k] = (double)b;
    }
}

/* Lens equation, eq 12: w = (1-kappa) z + gamma conj(z) - alpha_star - alpha_s
 * and, reading G23 (App. D: the macro potential Taylor-expanded one order further), minus the second-order term
 * of the macro deflection grad(psi):  alpha_i += (1/2) sum_jk psi_ijk x_j x_k, i.e.
 *   alpha_1 += (psi_111 x1^2 + 2 psi_112 x1 x2 + psi_122 x2^2)/2,  alpha_2 += (psi_112 x1^2 + 2 psi_122 x1 x2 + psi_222 x2^2)/2. */
static void lens_map_1(const orc_field *f, double zx, double zy, double *wx, double *wy)
{
    ld asx, asy, amx, amy;
    alpha_star_1(f, zx, zy, &asx, &asy);
    alpha_smooth_1(f, zx, zy, &amx, &amy);
    ld k = f->kappa_tot, g = f->gamma;
    ld x1 = zx, x2 = zy;
    ld q1 = (f->t111 * x1 * x1 + 2 * f->t112 * x1 * x2 + f->t122 * x2 * x2) / 2;
    ld q2 = (f->t112 * x1 * x1 + 2 * f->t122 * x1 * x2 + f->t222 * x2 * x2) / 2;
    *wx = (double)((1 - k) * zx + g * zx - asx - amx - q1);
    *wy = (double)((1 - k) * zy - g * zy - asy - amy - q2);
}

void orc_lens_map(const orc_field *f, int64_t n, const double *zx, const double *zy,
                  double *wx, double *wy)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t k = 0; k < n; ++k) lens_map_1(f, zx[k], zy[k], &wx[k], &wy[k]);
}

/* ------------------------------------------------------------------------- */
/* Geometry of the shooting window and ray grid (readings O1/O2 of DESIGN.md). */
typedef struct {
    /* inputs */
    double kappa_tot, kappa_star, gamma, theta_star, m2_over_m;
    double Y1, Y2;           /* map centre (source plane) */
    double dY1, dY2;         /* map half-sizes */
    int32_t npix1, npix2;
    double k;                /* rays per pixel LENGTH: cell = pixel / k */
    int32_t border_mode;     /* 0 eq16, 1 A6(f), 2 margin(frac), 3 explicit */
    int32_t pad_;
    double border_param, He1, He2;
    /* outputs */
    double X1, X2;           /* window centre, eq 14 */
    double H1, H2;           /* half-sizes after growing to whole cells */
    double h1, h2;           /* cell sizes */
    double p1, p2;           /* pixel sizes */
    double x0_1, x0_2;       /* coordinates of corner (0,0) */
    double ylo1, ylo2;       /* lower-left of the map */
    int64_t n1, n2;          /* cells along x1, x2 */
    double weight;           /* magnification deposited by one whole triangle = h1 h2/(2 p1 p2) */
} orc_geom;

int orc_geometry(orc_geom *g)
{
    double a1 = 1.0 - g->kappa_tot + g->gamma, a2 = 1.0 - g->kappa_tot - g->gamma;
    if (a1 == 0.0 || a2 == 0.0 || g->npix1 <= 0 || g->npix2 <= 0 || !(g->k > 0)) return -1;
    g->p1 = 2.0 * g->dY1 / g->npix1;
    g->p2 = 2.0 * g->dY2 / g->npix2;
    g->h1 = g->p1 / g->k;
    g->h2 = g->p2 / g->k;
    g->X1 = g->Y1 / a1;                       /* eq 14 */
    g->X2 = g->Y2 / a2;
    double b1, b2;                            /* source-plane half-size incl. border */
    switch (g->border_mode) {
    case 0: {                                 /* eq 16 */
        double r = 10.0 * g->theta_star * sqrt(g->kappa_star);
        b1 = g->dY1 + r; b2 = g->dY2 + r; break; }
    case 1: {                                 /* eq A6 */
        double r = g->theta_star * sqrt(g->kappa_star * g->m2_over_m / g->border_param);
        b1 = g->dY1 + r; b2 = g->dY2 + r; break; }
    case 2:                                   /* multiplicative margin */
        b1 = g->dY1 * (1.0 + g->border_param); b2 = g->dY2 * (1.0 + g->border_param); break;
    case 3:
        b1 = b2 = 0; break;
    default: return -1;
    }
    double H1 = (g->border_mode == 3) ? g->He1 : b1 / fabs(a1);   /* eq 15/16 */
    double H2 = (g->border_mode == 3) ? g->He2 : b2 / fabs(a2);
    g->n1 = (int64_t)ceil(2.0 * H1 / g->h1);
    g->n2 = (int64_t)ceil(2.0 * H2 / g->h2);
    if (g->n1 < 1 || g->n2 < 1) return -1;
    g->H1 = 0.5 * ((double)g->n1 * g->h1);
    g->H2 = 0.5 * ((double)g->n2 * g->h2);
    g->x0_1 = g->X1 - g->H1;
    g->x0_2 = g->X2 - g->H2;
    g->ylo1 = g->Y1 - g->dY1;
    g->ylo2 = g->Y2 - g->dY2;
    g->weight = (g->h1 * g->h2) / (2.0 * (g->p1 * g->p2));
    return 0;
}

/* corner (i, j) of the ray grid: one multiply, one add per axis (reading O2) */
static inline double corner1(const orc_geom *g, int64_t i) { return g->x0_1 + (double)i * g->h1; }
static inline double corner2(const orc_geom *g, int64_t j) { return g->x0_2 + (double)j * g->h2; }

/* ------------------------------------------------------------------------- */
/* Brute-force apportioning of one mapped triangle.
 * Vertices in PIXEL UNITS relative to the map's lower-left.  Every pixel of the
 * bounding box (clipped to the map) is intersected with the triangle by
 * Sutherland-Hodgman clipping against the pixel's four half-planes; shoelace
 * area; weight * A_piece / A_triangle is added (reading G16).                  */
typedef struct { double x, y; } pt;

static int clip_halfplane(const pt *in, int n, pt *out, int axis, double bound, int keep_ge)
{
    int m = 0;
    for (int a = 0; a < n; ++a) {
        pt P = in[a], Q = in[(a + 1) % n];
        double pv = axis ? P.y : P.x, qv = axis ? Q.y : Q.x;
        int pin = keep_ge ? (pv >= bound) : (pv <= bound);
        int qin = keep_ge ? (qv >= bound) : (qv <= bound);
        if (pin) out[m++] = P;
        if (pin != qin) {
            double t = (bound - pv) / (qv - pv);
            pt X;
            X.x = axis ? P.x + t * (Q.x - P.x) : bound;
            X.y = axis ? bound : P.y + t * (Q.y - P.y);
            out[m++] = X;
        }
    }
    return m;
}

static double shoelace(const pt *p, int n)
{
    double s = 0;
    for (int a = 0; a < n; ++a) {
        pt P = p[a], Q = p[(a + 1) % n];
        s += P.x * Q.y - Q.x * P.y;
    }
    return 0.5 * s;
}

/* signed area of triangle ∩ unit pixel [px,px+1]x[py,py+1] */
double orc_triangle_pixel_area(const double *tri /* x0 y0 x1 y1 x2 y2 */, double px, double py)
{
    pt a[16], b[16];
    for (int v = 0; v < 3; ++v) { a[v].x = tri[2 * v]; a[v].y = tri[2 * v + 1]; }
    int n = 3;
    n = clip_halfplane(a, n, b, 0, px, 1);        if (n < 3) return 0;
    n = clip_halfplane(b, n, a, 0, px + 1.0, 0);  if (n < 3) return 0;
    n = clip_halfplane(a, n, b, 1, py, 1);        if (n < 3) return 0;
    n = clip_halfplane(b, n, a, 1, py + 1.0, 0);  if (n < 3) return 0;
    return shoelace(a, n);
}

static void deposit_triangle(double ux0, double uy0, double ux1, double uy1, double ux2, double uy2,
                             int32_t npix1, int32_t npix2, double weight, double *map)
{
    double mnx = fmin(ux0, fmin(ux1, ux2)), mxx = fmax(ux0, fmax(ux1, ux2));
    double mny = fmin(uy0, fmin(uy1, uy2)), mxy = fmax(uy0, fmax(uy1, uy2));
    if (!(mxx >= 0) || !(mxy >= 0) || !(mnx < npix1) || !(mny < npix2)) return;  /* also drops NaN */
    double bx = floor(mnx), by = floor(mny);
    /* local coordinates: subtract the integer lower-left of the bounding box */
    double t[6] = { ux0 - bx, uy0 - by, ux1 - bx, uy1 - by, ux2 - bx, uy2 - by };
    double A = 0.5 * ((t[2] - t[0]) * (t[5] - t[1]) - (t[4] - t[0]) * (t[3] - t[1]));
    if (A == 0.0) {                              /* reading G12 */
        double fx = floor(ux0), fy = floor(uy0);
        if (fx >= 0 && fx < npix1 && fy >= 0 && fy < npix2)
            map[(int64_t)fy * npix1 + (int64_t)fx] += weight;
        return;
    }
    double ex = floor(mxx), ey = floor(mxy);
    double lox = fmax(bx, 0.0), hix = fmin(ex, (double)npix1 - 1.0);
    double loy = fmax(by, 0.0), hiy = fmin(ey, (double)npix2 - 1.0);
    for (double qy = loy; qy <= hiy; qy += 1.0)
        for (double qx = lox; qx <= hix; qx += 1.0) {
            double a = orc_triangle_pixel_area(t, qx - bx, qy - by);
            if (a != 0.0) map[(int64_t)qy * npix1 + (int64_t)qx] += weight * (a / A);
        }
}

/* IPM deposit of a grid of already-mapped corners: w[(j)*nc1 + i], i along x1.
 * Cell (i,j) -> T1 = (i,j),(i+1,j),(i+1,j+1); T2 = (i,j),(i+1,j+1),(i,j+1)  (reading G9). */
void orc_deposit_ipm(const double *wx, const double *wy, int64_t nc1, int64_t nc2,
                     double ylo1, double ylo2, double p1, double p2,
                     int32_t npix1, int32_t npix2, double weight, double *map)
{
    for (int64_t j = 0; j + 1 < nc2; ++j)
        for (int64_t i = 0; i + 1 < nc1; ++i) {
            int64_t a = j * nc1 + i, b = a + 1, c = a + nc1 + 1, d = a + nc1;
            double ua = (wx[a] - ylo1) / p1, va = (wy[a] - ylo2) / p2;
            double ub = (wx[b] - ylo1) / p1, vb = (wy[b] - ylo2) / p2;
            double uc = (wx[c] - ylo1) / p1, vc = (wy[c] - ylo2) / p2;
            double ud = (wx[d] - ylo1) / p1, vd = (wy[d] - ylo2) / p2;
            deposit_triangle(ua, va, ub, vb, uc, vc, npix1, npix2, weight, map);
            deposit_triangle(ua, va, uc, vc, ud, vd, npix1, npix2, weight, map);
        }
}

/* IRS binning (reading O5/G15): floor of a TRUE division, lower edge inclusive. */
void orc_bin_irs(const double *wx, const double *wy, int64_t n, double ylo1, double ylo2,
                 double p1, double p2, int32_t npix1, int32_t npix2, uint64_t *counts)
{
    for (int64_t r = 0; r < n; ++r) {
        double fx = floor((wx[r] - ylo1) / p1), fy = floor((wy[r] - ylo2) / p2);
        if (fx >= 0 && fx < npix1 && fy >= 0 && fy < npix2)
            counts[(int64_t)fy * npix1 + (int64_t)fx] += 1;
    }
}

/* Mapped corners of the cell sub-range [i0,i1) x [j0,j1): (i1-i0+1) x (j1-j0+1) corners. */
void orc_map_corners(const orc_field *f, const orc_geom *g, int64_t i0, int64_t i1,
                     int64_t j0, int64_t j1, double *wx, double *wy)
{
    int64_t nc1 = i1 - i0 + 1, nc2 = j1 - j0 + 1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < nc2; ++j)
        for (int64_t i = 0; i < nc1; ++i)
            lens_map_1(f, corner1(g, i0 + i), corner2(g, j0 + j), &wx[j * nc1 + i], &wy[j * nc1 + i]);
}

/* Mapped cell CENTRES (IRS rays, reading G10) of the same sub-range: (i1-i0) x (j1-j0) rays. */
void orc_map_centres(const orc_field *f, const orc_geom *g, int64_t i0, int64_t i1,
                     int64_t j0, int64_t j1, double *wx, double *wy)
{
    int64_t n1 = i1 - i0, n2 = j1 - j0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t j = 0; j < n2; ++j)
        for (int64_t i = 0; i < n1; ++i)
            lens_map_1(f, corner1(g, i0 + i) + 0.5 * g->h1, corner2(g, j0 + j) + 0.5 * g->h2,
                       &wx[j * n1 + i], &wy[j * n1 + i]);
}

/* The whole path on a cell sub-range: mode 0 = IPM into map (accumulates), 1 = IRS into counts. */
int orc_shoot(const orc_field *f, const orc_geom *g, int64_t i0, int64_t i1, int64_t j0, int64_t j1,
              int mode, double *map, uint64_t *counts)
{
    if (i0 < 0 || j0 < 0 || i1 > g->n1 || j1 > g->n2 || i1 <= i0 || j1 <= j0) return -1;
    int64_t nc1 = i1 - i0 + (mode == 0), nc2 = j1 - j0 + (mode == 0);
    double *wx = (double *)malloc(sizeof(double) * nc1 * nc2);
    double *wy = (double *)malloc(sizeof(double) * nc1 * nc2);
    if (!wx || !wy) { free(wx); free(wy); return -2; }
    if (mode == 0) {
        orc_map_corners(f, g, i0, i1, j0, j1, wx, wy);
        orc_deposit_ipm(wx, wy, nc1, nc2, g->ylo1, g->ylo2, g->p1, g->p2, g->npix1, g->npix2,
                        g->weight, map);
    } else {
        orc_map_centres(f, g, i0, i1, j0, j1, wx, wy);
        orc_bin_irs(wx, wy, nc1 * nc2, g->ylo1, g->ylo2, g->p1, g->p2, g->npix1, g->npix2, counts);
    }
    free(wx); free(wy);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Seeded star field (eq 9).  Counter-based generator specified in
 * DESIGN.md section 4 (splitmix64 finaliser over a Weyl sequence); star i consumes
 * counters 3i (radius / x1), 3i+1 (angle / x2), 3i+2 (mass).  The angle uses a fixed
 * Taylor polynomial on one octant so that positions are bit-reproducible by any
 * IEEE-754 implementation with fma.                                            */
static uint64_t rng_fin(uint64_t x)
{
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ULL;
    x ^= x >> 27; x *= 0x94D049BB133111EBULL;
    x ^= x >> 31;
    return x;
}
uint64_t orc_rng_draw(uint64_t seed, uint64_t n)
{
    return rng_fin(rng_fin(seed) + (n + 1) * 0x9E3779B97F4A7C15ULL);
}
static double rng_u(uint64_t seed, uint64_t n)
{
    return (double)(orc_rng_draw(seed, n) >> 11) * 0x1.0p-53;
}

/* (cos, sin) of 2 pi v, v in [0,1): octant k = floor(8v), f = 8v - k (mirrored for odd k),
 * theta = f pi/4, Taylor series of sin to theta^17 and cos to theta^18 by Horner with fma. */
static void unit_vector(double v, double *c_out, double *s_out)
{
    double t8 = 8.0 * v;
    int k = (int)t8;
    double f = t8 - (double)k;
    if (k & 1) f = 1.0 - f;
    double th = f * 0.78539816339744830962;
    double q = th * th;
    double S = 1.0 / 355687428096000.0;                 /* 1/17! */
    S = fma(S, q, -1.0 / 1307674368000.0);              /* 15! */
    S = fma(S, q, 1.0 / 6227020800.0);                  /* 13! */
    S = fma(S, q, -1.0 / 39916800.0);                   /* 11! */
    S = fma(S, q, 1.0 / 362880.0);                      /* 9! */
    S = fma(S, q, -1.0 / 5040.0);                       /* 7! */
    S = fma(S, q, 1.0 / 120.0);                         /* 5! */
    S = fma(S, q, -1.0 / 6.0);                          /* 3! */
    S = fma(S, q, 1.0);
    double s = th * S;
    double C = 1.0 / 6402373705728000.0;                /* 1/18! */
    C = fma(C, q, -1.0 / 20922789888000.0);             /* 16! */
    C = fma(C, q, 1.0 / 87178291200.0);                 /* 14! */
    C = fma(C, q, -1.0 / 479001600.0);                  /* 12! */
    C = fma(C, q, 1.0 / 3628800.0);                     /* 10! */
    C = fma(C, q, -1.0 / 40320.0);                      /* 8! */
    C = fma(C, q, 1.0 / 720.0);                         /* 6! */
    C = fma(C, q, -1.0 / 24.0);                         /* 4! */
    C = fma(C, q, 0.5);                                 /* 2! */
    double c = fma(-C, q, 1.0);
    double cc, ss;
    switch (k & 7) {
    case 0: cc = c;  ss = s;  break;     /* phi = theta          */
    case 1: cc = s;  ss = c;  break;     /* phi = pi/2 - theta'  */
    case 2: cc = -s; ss = c;  break;     /* phi = pi/2 + theta   */
    case 3: cc = -c; ss = s;  break;     /* phi = pi - theta'    */
    case 4: cc = -c; ss = -s; break;     /* phi = pi + theta     */
    case 5: cc = -s; ss = -c; break;     /* phi = 3pi/2 - theta' */
    case 6: cc = s;  ss = -c; break;     /* phi = 3pi/2 + theta  */
    default: cc = c; ss = -s; break;     /* phi = 2pi - theta'   */
    }
    *c_out = cc; *s_out = ss;
}

/* shape 0: disc radius a1 (r = R sqrt(u)); shape 1: rectangle corner (a1, a2).
 * mass_law 0: m = 1; 1: dN/dm ~ m^-a on [lo, hi] by inverse CDF, divided by the
 * theoretical mean (reading G22).                                              */
void orc_starfield(uint64_t seed, int64_t n, int shape, double a1, double a2,
                   int mass_law, double a, double lo, double hi,
                   double *x, double *y, double *m)
{
    double e = 1.0 - a, loe = 0, hie = 0, mean = 1.0;
    if (mass_law == 1) {
        loe = pow(lo, e); hie = pow(hi, e);
        mean = (e / (e + 1.0)) * (pow(hi, e + 1.0) - pow(lo, e + 1.0)) / (hie - loe);
    }
    for (int64_t i = 0; i < n; ++i) {
        double u1 = rng_u(seed, 3 * (uint64_t)i), u2 = rng_u(seed, 3 * (uint64_t)i + 1);
        double u3 = rng_u(seed, 3 * (uint64_t)i + 2);
        if (shape == 0) {
            double r = a1 * sqrt(u1), c, s;
            unit_vector(u2, &c, &s);
            x[i] = r * c; y[i] = r * s;
        } else {
            x[i] = a1 * (2.0 * u1 - 1.0);
            y[i] = a2 * (2.0 * u2 - 1.0);
        }
        m[i] = (mass_law == 1) ? pow(loe + u3 * (hie - loe), 1.0 / e) / mean : 1.0;
    }
}

/* ------------------------------------------------------------------------- */
/* FMM coefficients by their definitions, used to pin the CUDA operators.
 * Multipole, eq C2: a_0 = sum m, a_k = -(1/k) sum m zeta^k,
 * zeta = (z_i - centre)/L.   out[2k], out[2k+1] = Re, Im of a_k, k = 0..p.      */
void orc_multipole_def(int64_t n, const double *x, const double *y, const double *m,
                       double cx, double cy, double L, int p, double *out)
{
    for (int k = 0; k <= p; ++k) {
        long double complex s = 0;
        for (int64_t i = 0; i < n; ++i) {
            long double complex zeta = (((ld)x[i] - cx) + ((ld)y[i] - cy) * I) / (ld)L;
            if (k == 0) s += (ld)m[i];
            else s += -(ld)m[i] * cpowl(zeta, k) / (ld)k;
        }
        out[2 * k] = (double)creall(s); out[2 * k + 1] = (double)cimagl(s);
    }
}

/* Local (Taylor) coefficients straight from stars, eq C6:
 * c_l = sum -m/(l zeta_i^l), l >= 1;  c_0 = sum m log(-zeta_i) + m log L.        */
void orc_local_def(int64_t n, const double *x, const double *y, const double *m,
                   double cx, double cy, double L, int p, double *out)
{
    for (int l = 0; l <= p; ++l) {
        long double complex s = 0;
        for (int64_t i = 0; i < n; ++i) {
            long double complex zeta = (((ld)x[i] - cx) + ((ld)y[i] - cy) * I) / (ld)L;
            if (l == 0) s += (ld)m[i] * (clogl(-zeta) + logl((ld)L));
            else s += -(ld)m[i] / ((ld)l * cpowl(zeta, l));
        }
        out[2 * l] = (double)creall(s); out[2 * l + 1] = (double)cimagl(s);
    }
}

/* Far-field deflection from a local expansion, eq 24 / C4 (reading G1):
 * alpha_far = theta^2 conj( sum_{l>=1} l c_l zeta^(l-1) ) / L,  zeta = (z - centre)/L.   */
void orc_local_eval(const double *coef, int p, double cx, double cy, double L, double theta,
                    double zx, double zy, double *ax, double *ay)
{
    long double complex zeta = (((ld)zx - cx) + ((ld)zy - cy) * I) / (ld)L, s = 0, pw = 1;
    for (int l = 1; l <= p; ++l) {
        long double complex c = (ld)coef[2 * l] + (ld)coef[2 * l + 1] * I;
        s += (ld)l * c * pw;
        pw *= zeta;
    }
    s = conjl(s) * (ld)theta * (ld)theta / (ld)L;
    *ax = (double)creall(s); *ay = (double)cimagl(s);
}

/* ---- map consumers --------------------------------------------------------
 * Light curve: sample i of n at y = ya + (yb - ya) i/(n-1); pixel units u = (y - ylo)/p (true division).
 * mode 0: value of the pixel holding the point (floor rule); mode 1: bilinear between the four nearest pixel
 * centres (centres at integer + 1/2, indices clamped at the border).  Outside the map: NaN. */
void orc_light_curve(const double *map, int32_t npix1, int32_t npix2, double ylo1, double ylo2, double p1, double p2,
                     double ya1, double ya2, double yb1, double yb2, int64_t n, int32_t mode, double *mu)
{
    for (int64_t i = 0; i < n; ++i) {
        double t = (n > 1) ? (double)i / (double)(n - 1) : 0.0;
        double y1 = ya1 + (yb1 - ya1) * t, y2 = ya2 + (yb2 - ya2) * t;
        double u = (y1 - ylo1) / p1, v = (y2 - ylo2) / p2;
        mu[i] = NAN;
        if (!(u >= 0.0 && v >= 0.0 && u < (double)npix1 && v < (double)npix2)) continue;
        if (mode == 0) {
            mu[i] = map[(size_t)floor(v) * (size_t)npix1 + (size_t)floor(u)];
        } else {
            double uc = u - 0.5, vc = v - 0.5;
            long iu = (long)floor(uc), iv = (long)floor(vc);
            double a = uc - (double)iu, b = vc - (double)iv;
            long i0 = iu < 0 ? 0 : iu, i1 = iu + 1 > npix1 - 1 ? npix1 - 1 : iu + 1;
            long j0 = iv < 0 ? 0 : iv, j1 = iv + 1 > npix2 - 1 ? npix2 - 1 : iv + 1;
            double m00 = map[j0 * npix1 + i0], m10 = map[j0 * npix1 + i1], m01 = map[j1 * npix1 + i0], m11 = map[j1 * npix1 + i1];
            mu[i] = (1.0 - b) * ((1.0 - a) * m00 + a * m10) + b * ((1.0 - a) * m01 + a * m11);
        }
    }
}

/* Histogram of x = log10(mu/mu_ref) in nbins equal bins of [lo, hi): bin j holds edge_j <= mu < edge_{j+1},
 * edge_j = mu_ref 10^(lo + j (hi-lo)/nbins).  counts[0]: below edge_0 (also mu <= 0, NaN); counts[1+j]: bin j;
 * counts[nbins+1]: at or above edge_nbins.  Plain linear scan over the edges. */
void orc_histogram(const double *map, int64_t n, double mu_ref, double lo, double hi, int32_t nbins, uint64_t *counts)
{
    double *edge = (double *)malloc((size_t)(nbins + 1) * sizeof(double));
    for (int j = 0; j <= nbins; ++j) edge[j] = mu_ref * pow(10.0, lo + (double)j * (hi - lo) / (double)nbins);
    for (int j = 0; j < nbins + 2; ++j) counts[j] = 0;
    for (int64_t i = 0; i < n; ++i) {
        double mu = map[i];
        int slot = 0;
        if (mu >= edge[0]) {
            slot = nbins + 1;
            for (int j = 0; j < nbins; ++j)
                if (mu < edge[j + 1]) { slot = 1 + j; break; }
        }
        counts[slot]++;
    }
    free(edge);
}

