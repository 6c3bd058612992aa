/* mlens.h -- C ABI of libmlens: microlensing magnification maps on one NVIDIA B200 (sm_100a).
 *
 * Hot path of arXiv 2506.02114 ("P:n" = line n of the paper text):
 *   lens equation in complex form        w = (1-kappa) z + gamma conj(z) - alpha_star(z) - alpha_s(z)   (eq 12)
 *   star deflection                      alpha_star = theta^2 sum m_i/(conj z - conj z_i)               (eq 13)
 *     summed by an adaptive-quadtree fast multipole method (App. C)
 *   smooth sheet                         disc eq 19 or rectangle eq B7
 *   shooting window                      eq 14-16, eq A6
 *   inverse polygon mapping (IPM)        cells -> 2 triangles -> exact area apportioning
 *   inverse ray shooting (IRS)           ray counts per pixel
 *
 * Conventions
 *   - every call returns an int status (MLENS_OK = 0, negative = error); nothing throws across the ABI;
 *     mlens_last_error() returns a thread-local message for the last failing call.
 *   - the library owns the opaque mlens_field; THE CALLER OWNS EVERY ARRAY it passes in or receives
 *     into.  Arrays are DEVICE pointers (e.g. torch allocations) when ptr_kind = MLENS_PTR_DEVICE and
 *     HOST pointers when MLENS_PTR_HOST (then the call copies host<->device itself and synchronises).
 *     Inputs are copied at create time, never aliased.
 *   - all work is enqueued on the cudaStream_t passed as `stream` (void*, NULL = default stream).
 *     Calls that return scalars to the host (create, grid_info, stats) synchronise that stream; an IPM
 *     shoot also waits on it between row bands (it sizes each band from the counters of the one before).
 *   - there is NO CPU fallback: without a CUDA device every compute call fails with MLENS_ECUDA.
 *   - maps are row-major double[npix2][npix1], row index = x2 (y2) ascending, i.e. map[iy*npix1+ix];
 *     a pixel owns its lower edges (floor rule).  IPM maps are in magnification units (an identity
 *     lens gives 1.0); IRS count maps are raw ray counts, the IRS double map is counts / k^2.
 */
#ifndef MLENS_H
#define MLENS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MLENS_VERSION 200 /* 0.2.0: tuning fields in mlens_shoot_desc, more mlens_stats, benchmarks moved to mlens_bench.h */

enum { MLENS_OK = 0, MLENS_EINVAL = -1, MLENS_ENOMEM = -2, MLENS_ECUDA = -3,
       MLENS_ERANGE = -4 /* requested accuracy not attainable with order <= MLENS_MAX_ORDER, or tree depth exhausted */,
       MLENS_ESTATE = -5 };

enum { MLENS_PTR_DEVICE = 0, MLENS_PTR_HOST = 1 };
enum { MLENS_SHAPE_DISC = 0, MLENS_SHAPE_RECT = 1 };          /* star-region shape */
enum { MLENS_MASS_EQUAL = 0, MLENS_MASS_POWER = 1 };          /* dN/dm ~ m^-a on [lo,hi] / theoretical mean */
enum { MLENS_EVAL_FMM = 0, MLENS_EVAL_DIRECT = 1,             /* DIRECT = the paper's "no FMM" mode (Table 1) */
       MLENS_EVAL_FMM_F32 = 2 };  /* mlens_shoot only: the paper's single-precision mode: far-field series and
                                     near-field stars of a ray tile in float32, relative to the tile centre; macro
                                     terms, pixel arithmetic and accumulation stay float64.  Deflections are then
                                     good to ~1e-7 of their magnitude (not to eps_deflection). */
enum { MLENS_MAP_IPM = 0, MLENS_MAP_IRS = 1 };
enum { MLENS_BORDER_EQ16 = 0,      /* dY + 10 theta sqrt(kappa_star)                      (eq 16) */
       MLENS_BORDER_A6 = 1,        /* dY + theta sqrt(kappa_star <m^2>/(f <m>)), param=f (eq A6) */
       MLENS_BORDER_MARGIN = 2,    /* dY (1 + param)   (multiplicative margin)                   */
       MLENS_BORDER_EXPLICIT = 3 };/* window half-sizes He1, He2 given by the caller                    */

#define MLENS_MAX_ORDER 47         /* expansion order p <= 47 (48 coefficients; the paper caps at 31) */
#define MLENS_MAX_DIRECT 32        /* stars used directly per leaf */

typedef struct mlens_field mlens_field;

/* Lens field from caller-given stars (eq 12).  Exactly one of kappa_star / kappa_smooth may be NaN
 * and is then derived from kappa_tot (eq 10).  kappa_star is TAKEN AS GIVEN, never recomputed
 * from the stars (reading G17); mlens_field_get_info reports the actual value of eq 9. */
typedef struct {
    double kappa_tot, kappa_star, kappa_smooth, gamma;
    double theta_star;             /* Einstein radius of unit mass; 1 in all configs */
    int32_t shape;                 /* MLENS_SHAPE_* of the region the sheet compensates */
    int32_t ptr_kind;              /* where x, y, m live */
    double R;                      /* disc radius (shape DISC) */
    double c1, c2;                 /* rectangle corner (shape RECT), region |x1|<=c1, |x2|<=c2, centred at 0 */
    int64_t n_stars;               /* may be 0 */
    const double *x, *y, *m;       /* star positions and masses, length n_stars */
    double eps_deflection;         /* absolute accuracy wanted for alpha_star, units of theta_star; <=0 -> 1e-8 */
    int32_t max_direct;            /* <=0 -> 32; at most MLENS_MAX_DIRECT */
    int32_t order;                 /* expansion order p; <=0 -> chosen from eq C9 and verified on device */
    void *stream;
} mlens_field_desc;

/* Seeded star field: n_stars positions uniform in the region, masses equal
 * or power law.  The region size follows from eq 9 with <m> = 1:  disc R = theta sqrt(N/kappa_star);
 * rectangle 4 c1 c2 = pi theta^2 N / kappa_star with c1/c2 = rect_aspect.  Generator: DESIGN.md s4. */
typedef struct {
    double kappa_tot, kappa_star, kappa_smooth, gamma, theta_star;
    int32_t shape, mass_law;
    double rect_aspect;            /* c1/c2 for shape RECT */
    double mass_a, mass_lo, mass_hi;
    int64_t n_stars;
    uint64_t seed;
    double eps_deflection;
    int32_t max_direct, order;
    void *stream;
} mlens_seed_desc;

typedef struct {
    int64_t n_stars;
    int32_t order;                 /* expansion order p in use */
    int32_t n_levels;              /* deepest level + 1 */
    int64_t n_nodes, n_leaves;
    double root_half;              /* half-length of the root square (centred at the origin) */
    double leaf_half_min;          /* smallest leaf half-length */
    double kappa_star_actual;      /* theta^2 sum(m) / R^2  or  pi theta^2 sum(m)/(4 c1 c2)   (eq 9) */
    double mean_m, mean_m2;        /* <m>, <m^2> of the stars */
    double R, c1, c2;
    double spot_check_err;         /* max |alpha_fmm - alpha_direct| over the on-device spot check */
    int32_t max_near;              /* largest near-field list */
    int32_t max_m2l, max_p2l;      /* largest same-level / coarser-level interaction lists */
} mlens_field_info;

/* What to shoot.  Cell (i,j), 0<=i<n1, 0<=j<n2, has corners (i,j),(i+1,j),(i+1,j+1),(i,j+1) of the ray
 * grid z(i,j) = (x0_1 + i h1) + i (x0_2 + j h2); IPM rays are the corners, IRS rays the cell centres. */
typedef struct {
    double center_y1, center_y2;   /* map centre (Y1, Y2) in the source plane */
    double half_y1, half_y2;       /* map half-sizes (dY1, dY2) */
    int32_t npix1, npix2;
    double rays_per_pixel_length;  /* k: cell = pixel / k (Table 1 caption) */
    int32_t map_mode;              /* MLENS_MAP_IPM / MLENS_MAP_IRS */
    int32_t eval_mode;             /* MLENS_EVAL_FMM / MLENS_EVAL_DIRECT / MLENS_EVAL_FMM_F32 */
    int32_t border_mode;           /* MLENS_BORDER_* */
    int32_t accumulate;            /* 0: overwrite map/counts, 1: add to their current contents */
    double border_param, He1, He2;
    int64_t i0, i1, j0, j1;        /* cell sub-range [i0,i1) x [j0,j1); i1<=0 or j1<=0 -> whole grid */
    int32_t ptr_kind;              /* where map / counts / dump live */
    int32_t sync;                  /* 1: synchronise the stream before returning (always for host pointers) */
    double *dump_w1, *dump_w2;     /* optional: mapped ray positions of the sub-range, written by the SAME
                                      kernel that deposits them.  IPM: (j1-j0+1) x (i1-i0+1) corners;
                                      IRS: (j1-j0) x (i1-i0) centres; row-major, x1 fastest. May be NULL. */
    /* Tuning knobs; 0 = the library's default everywhere.  None of them changes what is computed: a map is the
     * same to the last bit for any setting except tile_order (which moves the rays within the tile series'
     * truncation budget, 5 % of eps_deflection) and small_px (which selects between two exact area formulas). */
    int32_t queue_mb;              /* size of the general-triangle queue in MiB (default: up to 8192) */
    int32_t tile_order;            /* order of the per-tile series, 2..15 (default: chosen per shoot from the tile size) */
    int32_t small_px;              /* queued triangles whose box holds more pixels than this are walked along their
                                      edges instead of clipped pixel by pixel (default 24) */
    int32_t band_fixed;            /* 1: IPM bands of exactly band_cells cells (default: sized from the measured rate
                                      of general triangles per cell) */
    int64_t band_cells;            /* upper bound of the cells per band (default 2^30) */
    int32_t tile_traversal;        /* order in which a band's ray tiles are handed out: 0 = default (column-major:
                                      the deposits of the tiles in flight stay within a patch of the map that L2
                                      holds), 1 = row-major */
    int32_t pad_;
} mlens_shoot_desc;

typedef struct {
    double X1, X2;                 /* window centre (eq 14) */
    double H1, H2;                 /* window half-sizes, grown to whole cells */
    double h1, h2, p1, p2;         /* cell and pixel sizes */
    double x0_1, x0_2;             /* position of corner (0,0) */
    double ylo1, ylo2;             /* lower-left of the map */
    int64_t n1, n2;                /* cells along x1, x2 */
    double weight;                 /* magnification carried by one whole triangle: h1 h2/(2 p1 p2) */
    int32_t order;
} mlens_grid;

typedef struct {
    int64_t n_rays;                /* lens-equation evaluations performed (incl. tile-border duplicates) */
    int64_t n_cells;
    int64_t n_tri_single;          /* triangles wholly inside one pixel */
    int64_t n_tri_strip;           /* triangles over two adjacent pixels (closed-form split in the shooting kernel) */
    int64_t n_tri_queued;          /* general triangles handed to the apportioning kernels through the global queue */
    int64_t n_tri_walked;          /* ... of which walked edge by edge (large boxes), the rest clipped pixel by pixel */
    int64_t n_queue_overflow;      /* general triangles apportioned by the shooting kernel itself: queue full */
    int64_t n_rays_fallback;       /* rays evaluated through the tree instead of the tile's series */
    int32_t n_bands;               /* row bands the sub-range was processed in */
    int32_t gpu_launches;          /* kernels launched by this call */
    float ms_total;                /* device time of the call (CUDA events), only when sync = 1 */
    float ms_shoot;                /* summed device time of the fused evaluate+deposit launches (IPM or IRS) */
    float ms_drain;                /* summed device time of the apportioning launches (drain + walk kernels, IPM) */
    float ms_finalise;             /* device time of the fixed-point -> double conversion */
    int32_t n_shoot_launches;      /* launches behind ms_shoot */
    int64_t n_near_terms;          /* near-field star terms summed directly over all rays (eq 23 direct part) */
    int64_t n_px_strip;            /* pixel deposits of the strips */
    int64_t n_px_clipped;          /* (triangle, pixel) pairs clipped exactly by the drain kernel */
    int64_t n_edge_steps;          /* major-axis steps of the edge walk (an edge walked once for the two triangles that share
                                      it counts once) */
    int64_t reserved_;
    int64_t n_tiles_full;          /* tile slots whose truncation bound failed (evaluated with the leaf's full series) */
    int32_t tile_order;            /* order of the per-tile series */
    int32_t pad_;
    float ms_walk;                 /* of ms_drain: the edge-walk launches (walk_kernel) */
    float ms_giant;                /* of ms_drain: the launches that walk the giant triangles chunk by chunk */
    int64_t n_giant_chunks;        /* chunks of edge steps the giant triangles were shared out in */
    int64_t n_tiles;               /* ray tiles (32 x 32 rays) evaluated with a leaf under their first corner */
    int64_t n_near_leaf_sum;       /* sum over those tiles of the near-field list length of that leaf: divided by n_tiles,
                                      the mean number of stars the paper's per-ray scheme sums directly (eq 23) */
} mlens_stats;

int mlens_version(void);
const char *mlens_last_error(void);
/* Kernels launched by the library in this process so far (every launch site counts itself). */
int64_t mlens_launch_count(void);

int mlens_field_create(const mlens_field_desc *desc, mlens_field **out);
int mlens_field_create_seeded(const mlens_seed_desc *desc, mlens_field **out);
/* Frees everything the field owns WITHOUT synchronising the device: the frees are stream-ordered on the stream of the
 * most recent call made on this field (create, deflect, lens_map, get_stars, shoot), after the work already enqueued
 * there.  That stream must therefore still exist when the field is destroyed (destroy the field first, then the
 * stream); a caller that used the field on several streams orders them before destroying it.  Should a stream-ordered
 * free fail all the same (e.g. the stream is gone), destroy falls back to a device synchronisation and plain frees. */
int mlens_field_destroy(mlens_field *f);
int mlens_field_get_info(const mlens_field *f, mlens_field_info *info);

/* Macro model beyond linear, for maps next to a macro-caustic (App. D: "the chosen order to which the
 * potential is Taylor expanded"; the paper prints no formula, reading G23).  The macro deflection grad(psi)
 * gets its second-order Taylor term about the origin, from the four third derivatives of the macro potential there:
 *   w1 -= (psi_111 x1^2 + 2 psi_112 x1 x2 + psi_122 x2^2) / 2,   w2 -= (psi_112 x1^2 + 2 psi_122 x1 x2 + psi_222 x2^2) / 2
 * in eq 12 (mlens_lens_map and every ray of mlens_shoot; mlens_deflect, the stars' part, is untouched).  All four zero
 * (the state after create) is the paper's constant kappa and gamma, to the last bit.  With any of them non-zero the
 * shooting window of eq 14-16 no longer encloses the macro-images, so mlens_shoot / mlens_grid_info then take
 * MLENS_BORDER_EXPLICIT only (MLENS_EINVAL otherwise): choosing the window is the part the paper leaves to other work.
 * Host-side state only (no device work); affects the calls made after it. */
int mlens_field_set_macro_quadratic(mlens_field *f, double psi_111, double psi_112, double psi_122, double psi_222);

/* Copies the stars (positions in units of theta_star's length, masses as used in eq 13; for a seeded field
 * the draws of P:159-165), in the caller's original order, into x, y, m (length n_stars each). */
int mlens_field_get_stars(const mlens_field *f, double *x, double *y, double *m, int32_t ptr_kind, void *stream);

/* alpha_star (eq 13) at n points: FMM (near-field direct sum + local expansion, eq 23-24)
 * or DIRECT (all stars).  Outputs ax, ay length n. */
int mlens_deflect(const mlens_field *f, int64_t n, const double *zx, const double *zy,
                  double *ax, double *ay, int32_t eval_mode, int32_t ptr_kind, void *stream);

/* w of eq 12 at n points (macro + stars + sheet). */
int mlens_lens_map(const mlens_field *f, int64_t n, const double *zx, const double *zy,
                   double *wx, double *wy, int32_t eval_mode, int32_t ptr_kind, void *stream);

/* The integers and lengths the shoot call will use (host-side arithmetic only): window centre X = Y/(1-kappa -+ gamma)
 * (eq 14), half-sizes from the map's half-sizes plus the border of eq 16 / eq A6 / the caller's
 * choice, grown to whole cells of pixel/k (Table 1 caption). */
int mlens_grid_info(const mlens_field *f, const mlens_shoot_desc *desc, mlens_grid *out);

/* Shoots the (sub-range of the) ray grid and builds the map.  map: double[npix2*npix1] or NULL;
 * counts: uint64[npix2*npix1], the IRS ray counts, or NULL -- it must be NULL for MLENS_MAP_IPM (MLENS_EINVAL
 * otherwise: an IPM map has no counts); stats may be NULL.
 * IPM: cells -> two triangles -> exact area apportioning; IRS: one ray per cell centre, counted in the
 * pixel it falls into.  Window and grid are those of mlens_grid_info.
 * Ray tiles are anchored on the GLOBAL cell grid, so a ray has the same value to the last bit in whatever
 * sub-range it is shot, and within ONE call every deposit is an integer (fixed-point) addition.  Across calls the
 * sum is taken in float64: each sub-range shoot converts its integers to double once (clamping a negative
 * rounding residue to 0) and `accumulate` or the all-reduce of row slabs adds those doubles.  Maps put together
 * from sub-ranges or slabs therefore equal the one-call map up to one float64 rounding per part and pixel (plus
 * the residues of the fixed-point quantum, 2^-36 of a triangle's weight), not to the last bit. */
int mlens_shoot(mlens_field *f, const mlens_shoot_desc *desc, double *map, uint64_t *counts,
                mlens_stats *stats, void *stream);

/* Tree introspection for tests (HOST buffers, any may be NULL).  Node arrays have n_nodes entries;
 * coefficient arrays n_nodes*(order+1) complex numbers as (re,im) pairs, in units of the node
 * half-length: multipole eq C1-C3, local eq C4-C7.  Leaf arrays have n_leaves entries;
 * near_* are n_leaves*MLENS_MAX_DIRECT.  m2l_list is n_nodes*27, p2l_list n_nodes*8 (node indices, -1 pad). */
typedef struct {
    int32_t *level, *ix, *iy, *parent, *child0, *star_lo, *star_n, *leaf_id;
    int32_t *nbr;                  /* n_nodes*8, same-level neighbour node or -1 */
    int32_t *m2l_cnt, *m2l_list, *p2l_cnt, *p2l_list;
    double *multipole, *local;
    int32_t *near_cnt;
    double *near_x, *near_y, *near_m;
    double *sorted_x, *sorted_y, *sorted_m;   /* stars in Morton order, n_stars each */
} mlens_tree_view;
int mlens_field_get_tree(const mlens_field *f, mlens_tree_view *view);

/* ---- Map consumers: what the paper reads off its maps ---------------------------------
 * The map is double[npix2*npix1], row = y2 ascending, pixel (ix, iy) covering
 * [ylo1 + ix p1, ylo1 + (ix+1) p1) x [ylo2 + iy p2, ylo2 + (iy+1) p2)   (mlens_grid: ylo1, ylo2, p1, p2).
 *
 * Light curve (Fig 4, Fig 8: the magnification along a straight source track): n >= 1 samples at
 * y_i = ya + (yb - ya) i/(n-1) (i = 0 if n = 1).  interp = MLENS_INTERP_NEAREST: the value of the pixel holding
 * y_i (floor rule, lower edge inclusive); MLENS_INTERP_BILINEAR: bilinear between the four nearest pixel CENTRES
 * (indices clamped at the border).  A sample outside the map gives NaN.  mu: double[n]. */
enum { MLENS_INTERP_NEAREST = 0, MLENS_INTERP_BILINEAR = 1 };
int mlens_map_light_curve(const double *map, int32_t npix1, int32_t npix2, double ylo1, double ylo2, double p1, double p2,
                          double ya1, double ya2, double yb1, double yb2, int64_t n, int32_t interp,
                          double *mu, int32_t ptr_kind, void *stream);

/* Magnification histogram (Fig 5, Fig 10): counts of x = log10(mu / mu_ref) in nbins equal bins of
 * [lo, hi).  Bin j holds edge_j <= mu < edge_{j+1} with edge_j = mu_ref 10^(lo + j (hi-lo)/nbins) evaluated once in
 * float64 on the host: the decision is a comparison of mu with those edges, never a logarithm of mu.
 * counts: uint64[nbins + 2] = { below edge_0 (also mu <= 0 and NaN), the bins, at or above edge_nbins }; overwritten.
 * 1 <= nbins <= 4096, n = number of pixels, mu_ref > 0, hi > lo. */
int mlens_map_histogram(const double *map, int64_t n, double mu_ref, double lo, double hi, int32_t nbins,
                        uint64_t *counts, int32_t ptr_kind, void *stream);

/* The same histogram (Fig 5, Fig 10; same bins, same counts to the last unit) for callers that cannot let
 * the library allocate device memory.  That is the case in a process whose memory manager has claimed the whole GPU up
 * front (an inference server, a framework's caching allocator at its cap: any allocation of ours would fail there), and
 * on paths where an allocation's hidden costs are not acceptable (it can serialise against work on other streams, and
 * it can fail at a moment the caller cannot recover from).  mlens_map_histogram takes the device copy of its bin-edge
 * table from the device's memory pool on every call; this entry point keeps that table in a fixed array inside the
 * library image instead and calls no cudaMalloc / cudaMallocAsync / cudaFree or other allocating routine.
 *   - map (n values) and counts (nbins + 2, overwritten) are DEVICE pointers owned by the caller; host pointers are
 *     refused with MLENS_EINVAL (copying them over would need a buffer).
 *   - nbins <= MLENS_HIST_STATIC_MAXBINS; more is refused with MLENS_EINVAL and a message naming the limit.  The table
 *     costs (MLENS_HIST_STATIC_MAXBINS + 1) * 8 bytes = 32 KB on every GPU the library is loaded on, until the process ends.
 *   - the first call on each device looks the table's device address up (with that device current) and sets the
 *     kernel's attributes; make that first call before any stream capture starts.
 *   - all calls on a device share the one table.  A call overwrites the entries it uses before its kernel reads them,
 *     so leftovers of earlier calls are never seen and nothing needs clearing; calls on the same stream are ordered
 *     and safe, but two calls whose work can overlap on the GPU (different streams, different host threads) race on
 *     the table and may count with each other's edges: serialise them.
 *   - work is enqueued on `stream`; the call returns without waiting for the kernel (its copy of the edges from
 *     pageable host memory may wait for earlier work on that stream). */
#define MLENS_HIST_STATIC_MAXBINS 4096
int mlens_map_histogram_static(const double *map, int64_t n, double mu_ref, double lo, double hi, int32_t nbins,
                               uint64_t *counts, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* MLENS_H */
