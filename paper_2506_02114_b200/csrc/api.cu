// api.cu -- the C ABI of include/mlens.h: argument checking, host<->device marshalling, handle life
// cycle, expansion-order selection (eq C9) with an on-device a-posteriori check.
#include "device.cuh"
#include <math.h>
#include <stdarg.h>
#include <string.h>

namespace ml {
std::atomic<long long> g_launches{0};
static thread_local char g_err[512] = "";
void set_error(const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int pool_init() {
    static std::atomic<int> done[ML_MAXDEV];                        // per device (zero-initialised)
    int dev = 0;
    ML_CUDA(cudaGetDevice(&dev));
    const int slot = device_slot();
    if (done[slot].load()) return MLENS_OK;
    cudaMemPool_t pool;
    ML_CUDA(cudaDeviceGetDefaultMemPool(&pool, dev));
    unsigned long long keep = ~0ull;
    ML_CUDA(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
    done[slot].store(1);
    return MLENS_OK;
}

static int check_device() {
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n <= 0) {
        set_error("no CUDA device available (%s); libmlens has no CPU fallback", cudaGetErrorString(e));
        cudaGetLastError();
        return MLENS_ECUDA;
    }
    return MLENS_OK;
}

// staging of caller arrays: device pointers pass through, host pointers are copied
struct Stage {
    std::vector<void *> owned;
    cudaStream_t s_;
    explicit Stage(cudaStream_t s) : s_(s) {}
    ~Stage() { for (void *p : owned) cudaFreeAsync(p, s_); }       // stream-ordered: after the copies back
    template <typename T>
    int in(const T *src, size_t n, int kind, cudaStream_t s, const T **out) {
        if (kind == MLENS_PTR_DEVICE || n == 0) { *out = src; return MLENS_OK; }
        T *d = nullptr;
        ML_TRY(pool_init());
        ML_CUDA(cudaMallocAsync(&d, n * sizeof(T), s));
        owned.push_back(d);
        ML_CUDA(cudaMemcpyAsync(d, src, n * sizeof(T), cudaMemcpyHostToDevice, s));
        *out = d;
        return MLENS_OK;
    }
    template <typename T>
    int out(T *dst, size_t n, int kind, T **dev) {
        if (kind == MLENS_PTR_DEVICE || n == 0 || dst == nullptr) { *dev = dst; return MLENS_OK; }
        T *d = nullptr;
        ML_TRY(pool_init());
        ML_CUDA(cudaMallocAsync(&d, n * sizeof(T), s_));
        owned.push_back(d);
        *dev = d;
        return MLENS_OK;
    }
    template <typename T>
    int back(T *dst, const T *dev, size_t n, int kind, cudaStream_t s) {
        if (kind == MLENS_PTR_DEVICE || n == 0 || dst == nullptr) return MLENS_OK;
        ML_CUDA(cudaMemcpyAsync(dst, dev, n * sizeof(T), cudaMemcpyDeviceToHost, s));
        return MLENS_OK;
    }
};

// sample points for the a-posteriori accuracy check: around stars at the scale of the smallest leaves
// (where the expansions are coarsest relative to the masses) and uniformly over the star region
__global__ void spot_points_kernel(const double *sx, const double *sy, long long n, double leaf_half, double root_half,
                                   int npts, double *zx, double *zy) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npts) return;
    unsigned long long h = (unsigned long long)(i + 1) * 0x9E3779B97F4A7C15ull;
    h ^= h >> 29; h *= 0xBF58476D1CE4E5B9ull; h ^= h >> 32;
    double u1 = (double)(h & 0xFFFFF) / 1048576.0, u2 = (double)((h >> 20) & 0xFFFFF) / 1048576.0;
    double u3 = (double)((h >> 40) & 0xFFFFF) / 1048576.0;
    if ((i & 3) == 3 || n == 0) {
        zx[i] = root_half * 0.7 * (2.0 * u1 - 1.0); zy[i] = root_half * 0.7 * (2.0 * u2 - 1.0);
    } else {
        long long j = (long long)(u3 * (double)n); if (j >= n) j = n - 1;
        double r = leaf_half * (0.05 + 3.0 * u1), a = 6.283185307179586 * u2;
        zx[i] = sx[j] + r * cos(a); zy[i] = sy[j] + r * sin(a);
    }
}
__global__ void max_diff_kernel(const double *ax, const double *ay, const double *bx, const double *by, int n,
                                unsigned long long *out_bits) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    double d = 0.0;
    if (i < n) d = hypot(ax[i] - bx[i], ay[i] - by[i]);
    if (!(d == d)) d = 1.0e300;
    for (int o = 16; o; o >>= 1) d = fmax(d, __shfl_xor_sync(0xffffffffu, d, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out_bits, (unsigned long long)__double_as_longlong(d));
}

static int spot_check(mlens_field *f, cudaStream_t s, double *err) {
    const int NP = 1024;
    ScratchBuf<double> b; ScratchBuf<unsigned long long> bits;
    ML_TRY(b.reserve(6 * NP, s, false)); ML_TRY(bits.reserve(1, s, false));
    double *zx = b.p, *zy = b.p + NP, *ax = b.p + 2 * NP, *ay = b.p + 3 * NP, *bx = b.p + 4 * NP, *by = b.p + 5 * NP;
    double leaf_half = f->root_half / (double)(1 << (f->tree.n_levels - 1));
    ML_LAUNCH(spot_points_kernel, (NP + 127) / 128, 128, 0, s, f->sx.p, f->sy.p, f->n_stars, leaf_half, f->root_half, NP, zx, zy);
    ML_TRY(deflect_points(f, NP, zx, zy, ax, ay, MLENS_EVAL_FMM, 0, s));
    ML_TRY(deflect_points(f, NP, zx, zy, bx, by, MLENS_EVAL_DIRECT, 0, s));
    ML_CUDA(cudaMemsetAsync(bits.p, 0, 8, s));
    ML_LAUNCH(max_diff_kernel, (NP + 127) / 128, 128, 0, s, ax, ay, bx, by, NP, bits.p);
    unsigned long long h = 0;
    ML_CUDA(cudaMemcpyAsync(&h, bits.p, 8, cudaMemcpyDeviceToHost, s));
    ML_CUDA(cudaStreamSynchronize(s));
    ML_CUDA(cudaGetLastError());
    memcpy(err, &h, 8);
    b.release(); bits.release();
    return MLENS_OK;
}

static int finish_create(mlens_field *f, int order_req, cudaStream_t s) {
    ML_TRY(build_tree(f, s));
    ML_TRY(fmm_prepare_tables(f, s));
    double leaf_half = f->root_half / (double)(1 << (f->tree.n_levels - 1));
    int p;
    if (order_req > 0) p = order_req;
    else {
        // eq C9: p > log2( theta^2 <m^2>/<m> / (L eps) ), L = smallest leaf half-length (reading G5)
        double m2m = (f->mean_m > 0) ? f->mean_m2 / f->mean_m : 1.0;
        double v = log2(f->theta * f->theta * m2m / (leaf_half * f->eps));
        p = (int)ceil(v) + 1;
        if (p < 4) p = 4;
    }
    if (p > MLENS_MAX_ORDER) p = MLENS_MAX_ORDER;
    while (true) {
        f->order = p;
        ML_TRY(fmm_passes(f, s));
        if (f->n_stars == 0) { f->spot_err = 0; break; }
        ML_TRY(spot_check(f, s, &f->spot_err));
        if (order_req > 0 || f->spot_err <= 0.5 * f->eps) break;
        if (p >= MLENS_MAX_ORDER) {
            set_error("deflection accuracy %.3g not reached at the maximum order %d (error %.3g)", f->eps, p, f->spot_err);
            return MLENS_ERANGE;
        }
        p = (p + 3 > MLENS_MAX_ORDER) ? MLENS_MAX_ORDER : p + 3;
    }
    if (f->shape == MLENS_SHAPE_RECT) ML_TRY(rect_fold(f, s));
    return MLENS_OK;
}

static int resolve_kappa(double kt, double &ks, double &km) {
    bool ns = ks != ks, nm = km != km;
    if (ns && nm) { set_error("give kappa_star or kappa_smooth"); return MLENS_EINVAL; }
    if (ns) ks = kt - km;
    if (nm) km = kt - ks;
    if (fabs(ks + km - kt) > 1e-12 * (1.0 + fabs(kt))) { set_error("kappa_star + kappa_smooth != kappa_tot"); return MLENS_EINVAL; }
    if (ks < 0) { set_error("kappa_star < 0"); return MLENS_EINVAL; }
    return MLENS_OK;
}
}  // namespace ml

using namespace ml;

extern "C" {

int mlens_version(void) { return MLENS_VERSION; }
const char *mlens_last_error(void) { return g_err; }
int64_t mlens_launch_count(void) { return (int64_t)g_launches.load(); }

int mlens_field_create(const mlens_field_desc *d, mlens_field **out) {
    if (!d || !out) { set_error("null argument"); return MLENS_EINVAL; }
    *out = nullptr;
    ML_TRY(check_device());
    if (d->n_stars < 0 || (d->n_stars > 0 && (!d->x || !d->y || !d->m))) { set_error("bad star arrays"); return MLENS_EINVAL; }
    if (d->shape != MLENS_SHAPE_DISC && d->shape != MLENS_SHAPE_RECT) { set_error("bad shape"); return MLENS_EINVAL; }
    if (d->shape == MLENS_SHAPE_DISC && !(d->R > 0)) { set_error("disc needs R > 0"); return MLENS_EINVAL; }
    if (d->shape == MLENS_SHAPE_RECT && (!(d->c1 > 0) || !(d->c2 > 0))) { set_error("rectangle needs c1, c2 > 0"); return MLENS_EINVAL; }
    if (d->order > MLENS_MAX_ORDER || d->max_direct > MLENS_MAX_DIRECT) { set_error("order or max_direct too large"); return MLENS_EINVAL; }
    double ks = d->kappa_star, km = d->kappa_smooth;
    ML_TRY(resolve_kappa(d->kappa_tot, ks, km));
    cudaStream_t s = (cudaStream_t)d->stream;
    mlens_field *f = new (std::nothrow) mlens_field();
    if (!f) return MLENS_ENOMEM;
    f->kappa_tot = d->kappa_tot; f->kappa_star = ks; f->kappa_smooth = km; f->gamma = d->gamma;
    f->theta = (d->theta_star > 0) ? d->theta_star : 1.0;
    f->shape = d->shape; f->R = d->R; f->c1 = d->c1; f->c2 = d->c2;
    f->eps = (d->eps_deflection > 0) ? d->eps_deflection : 1e-8;
    f->max_direct = (d->max_direct > 0) ? d->max_direct : MLENS_MAX_DIRECT;
    f->n_stars = d->n_stars;
    cudaGetDevice(&f->device);
    f->last_stream = s;
    int rc = MLENS_OK;
    size_t n = (size_t)d->n_stars;
    cudaMemcpyKind kind = d->ptr_kind == MLENS_PTR_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    auto body = [&]() -> int {
        ML_TRY(f->ox.reserve(n + 1, s, false)); ML_TRY(f->oy.reserve(n + 1, s, false)); ML_TRY(f->om.reserve(n + 1, s, false));
        if (n) {
            ML_CUDA(cudaMemcpyAsync(f->ox.p, d->x, n * 8, kind, s));
            ML_CUDA(cudaMemcpyAsync(f->oy.p, d->y, n * 8, kind, s));
            ML_CUDA(cudaMemcpyAsync(f->om.p, d->m, n * 8, kind, s));
        }
        return finish_create(f, d->order, s);
    };
    rc = body();
    if (rc != MLENS_OK) { mlens_field_destroy(f); return rc; }
    *out = f;
    return MLENS_OK;
}

int mlens_field_create_seeded(const mlens_seed_desc *d, mlens_field **out) {
    if (!d || !out) { set_error("null argument"); return MLENS_EINVAL; }
    *out = nullptr;
    ML_TRY(check_device());
    if (d->n_stars <= 0) { set_error("n_stars must be positive"); return MLENS_EINVAL; }
    if (d->order > MLENS_MAX_ORDER || d->max_direct > MLENS_MAX_DIRECT) { set_error("order or max_direct too large"); return MLENS_EINVAL; }
    double ks = d->kappa_star, km = d->kappa_smooth;
    ML_TRY(resolve_kappa(d->kappa_tot, ks, km));
    if (!(ks > 0)) { set_error("a seeded field needs kappa_star > 0"); return MLENS_EINVAL; }
    cudaStream_t s = (cudaStream_t)d->stream;
    mlens_field *f = new (std::nothrow) mlens_field();
    if (!f) return MLENS_ENOMEM;
    f->kappa_tot = d->kappa_tot; f->kappa_star = ks; f->kappa_smooth = km; f->gamma = d->gamma;
    f->theta = (d->theta_star > 0) ? d->theta_star : 1.0;
    f->shape = d->shape;
    f->eps = (d->eps_deflection > 0) ? d->eps_deflection : 1e-8;
    f->max_direct = (d->max_direct > 0) ? d->max_direct : MLENS_MAX_DIRECT;
    f->n_stars = d->n_stars;
    cudaGetDevice(&f->device);
    f->last_stream = s;
    // eq 9 with <m> = 1: area = pi theta^2 N / kappa_star
    double a1, a2 = 0.0;
    if (d->shape == MLENS_SHAPE_DISC) {
        f->R = f->theta * sqrt((double)d->n_stars / ks);
        a1 = f->R;
    } else if (d->shape == MLENS_SHAPE_RECT) {
        if (!(d->rect_aspect > 0)) { delete f; set_error("rect_aspect must be > 0"); return MLENS_EINVAL; }
        double area = 3.14159265358979323846 * f->theta * f->theta * (double)d->n_stars / ks;
        f->c2 = sqrt(area / (4.0 * d->rect_aspect));
        f->c1 = d->rect_aspect * f->c2;
        a1 = f->c1; a2 = f->c2;
    } else { delete f; set_error("bad shape"); return MLENS_EINVAL; }
    size_t n = (size_t)d->n_stars;
    auto body = [&]() -> int {
        ML_TRY(f->ox.reserve(n + 1, s, false)); ML_TRY(f->oy.reserve(n + 1, s, false)); ML_TRY(f->om.reserve(n + 1, s, false));
        ML_TRY(generate_stars(d->seed, d->n_stars, d->shape, a1, a2, d->mass_law, d->mass_a, d->mass_lo, d->mass_hi,
                              f->ox.p, f->oy.p, f->om.p, s));
        return finish_create(f, d->order, s);
    };
    int rc = body();
    if (rc != MLENS_OK) { mlens_field_destroy(f); return rc; }
    *out = f;
    return MLENS_OK;
}

// Everything a field owns is freed in stream order on the stream of the field's most recent call: no device-wide
// synchronisation.  (A caller that used the field on several streams orders them before destroying it, as for
// any other stream-ordered resource.)
int mlens_field_destroy(mlens_field *f) {
    if (!f) return MLENS_OK;
    int cur = 0;
    cudaGetDevice(&cur);
    if (cur != f->device) cudaSetDevice(f->device);
    cudaStream_t s = f->last_stream;
    f->ox.release(s); f->oy.release(s); f->om.release(s); f->sx.release(s); f->sy.release(s); f->sm.release(s);
    f->sqx.release(s); f->sqy.release(s); f->acc.release(s); f->diff.release(s);
    f->binom.p = nullptr; f->tab.p = nullptr;                     // borrowed from the per-device tables (fmm.cu)
    scratch_park(f, s);
    f->queue.release(s); f->qcount.release(s); f->biglist.release(s); f->giant.release(s); f->giant_sorted.release(s); f->giant_key.release(s); f->giant_hist.release(s); f->counters.release(s);
    f->tree.release(s);
    if (cur != f->device) cudaSetDevice(cur);
    delete f;
    return MLENS_OK;
}

int mlens_field_set_macro_quadratic(mlens_field *f, double psi_111, double psi_112, double psi_122, double psi_222) {
    if (!f) { set_error("null argument"); return MLENS_EINVAL; }
    const double t[4] = {psi_111, psi_112, psi_122, psi_222};
    for (int i = 0; i < 4; ++i) if (!(t[i] == t[i]) || fabs(t[i]) > 1e300) { set_error("macro coefficients must be finite"); return MLENS_EINVAL; }
    for (int i = 0; i < 4; ++i) f->quad[i] = t[i];
    return MLENS_OK;
}

int mlens_field_get_info(const mlens_field *f, mlens_field_info *o) {
    if (!f || !o) { set_error("null argument"); return MLENS_EINVAL; }
    memset(o, 0, sizeof(*o));
    o->n_stars = f->n_stars; o->order = f->order; o->n_levels = f->tree.n_levels;
    o->n_nodes = f->tree.n_nodes; o->n_leaves = f->tree.n_leaves;
    o->root_half = f->root_half;
    o->leaf_half_min = f->root_half / (double)(1 << (f->tree.n_levels - 1));
    double area = (f->shape == MLENS_SHAPE_DISC) ? 3.14159265358979323846 * f->R * f->R : 4.0 * f->c1 * f->c2;
    o->kappa_star_actual = 3.14159265358979323846 * f->theta * f->theta * f->sum_m / area;
    o->mean_m = f->mean_m; o->mean_m2 = f->mean_m2;
    o->R = f->R; o->c1 = f->c1; o->c2 = f->c2;
    o->spot_check_err = f->spot_err;
    o->max_near = f->max_near; o->max_m2l = f->max_m2l; o->max_p2l = f->max_p2l;
    return MLENS_OK;
}

int mlens_field_get_stars(const mlens_field *f, double *x, double *y, double *m, int32_t ptr_kind, void *stream) {
    if (!f || !x || !y || !m) { set_error("null argument"); return MLENS_EINVAL; }
    cudaStream_t s = (cudaStream_t)stream;
    size_t n = (size_t)f->n_stars;
    if (!n) return MLENS_OK;
    cudaMemcpyKind kind = ptr_kind == MLENS_PTR_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    ML_CUDA(cudaMemcpyAsync(x, f->ox.p, n * 8, kind, s));
    ML_CUDA(cudaMemcpyAsync(y, f->oy.p, n * 8, kind, s));
    ML_CUDA(cudaMemcpyAsync(m, f->om.p, n * 8, kind, s));
    if (ptr_kind == MLENS_PTR_HOST) ML_CUDA(cudaStreamSynchronize(s));
    return MLENS_OK;
}

static int points_call(const mlens_field *f, int64_t n, const double *zx, const double *zy, double *ox, double *oy,
                       int eval_mode, int full, int ptr_kind, void *stream) {
    if (!f || n < 0 || (n > 0 && (!zx || !zy || !ox || !oy))) { set_error("bad arguments"); return MLENS_EINVAL; }
    if (eval_mode != MLENS_EVAL_FMM && eval_mode != MLENS_EVAL_DIRECT) { set_error("bad eval mode"); return MLENS_EINVAL; }
    cudaStream_t s = (cudaStream_t)stream;
    const_cast<mlens_field *>(f)->last_stream = s;
    Stage st(s);
    const double *dzx, *dzy; double *dox, *doy;
    ML_TRY(st.in(zx, (size_t)n, ptr_kind, s, &dzx)); ML_TRY(st.in(zy, (size_t)n, ptr_kind, s, &dzy));
    ML_TRY(st.out(ox, (size_t)n, ptr_kind, &dox)); ML_TRY(st.out(oy, (size_t)n, ptr_kind, &doy));
    ML_TRY(deflect_points(f, n, dzx, dzy, dox, doy, eval_mode, full, s));
    ML_TRY(st.back(ox, dox, (size_t)n, ptr_kind, s)); ML_TRY(st.back(oy, doy, (size_t)n, ptr_kind, s));
    if (ptr_kind == MLENS_PTR_HOST) ML_CUDA(cudaStreamSynchronize(s));
    return MLENS_OK;
}

int mlens_deflect(const mlens_field *f, int64_t n, const double *zx, const double *zy, double *ax, double *ay,
                  int32_t eval_mode, int32_t ptr_kind, void *stream) {
    return points_call(f, n, zx, zy, ax, ay, eval_mode, 0, ptr_kind, stream);
}
int mlens_lens_map(const mlens_field *f, int64_t n, const double *zx, const double *zy, double *wx, double *wy,
                   int32_t eval_mode, int32_t ptr_kind, void *stream) {
    return points_call(f, n, zx, zy, wx, wy, eval_mode, 1, ptr_kind, stream);
}

int mlens_grid_info(const mlens_field *f, const mlens_shoot_desc *d, mlens_grid *out) {
    if (!f || !d || !out) { set_error("null argument"); return MLENS_EINVAL; }
    return geometry(f, d, out);
}

int mlens_shoot(mlens_field *f, const mlens_shoot_desc *d, double *map, uint64_t *counts, mlens_stats *stats, void *stream) {
    if (!f || !d) { set_error("null argument"); return MLENS_EINVAL; }
    if (d->map_mode != MLENS_MAP_IPM && d->map_mode != MLENS_MAP_IRS) { set_error("bad map mode"); return MLENS_EINVAL; }
    if (d->eval_mode != MLENS_EVAL_FMM && d->eval_mode != MLENS_EVAL_DIRECT && d->eval_mode != MLENS_EVAL_FMM_F32) { set_error("bad eval mode"); return MLENS_EINVAL; }
    if (d->map_mode == MLENS_MAP_IPM && counts) { set_error("an IPM map has no ray counts: counts must be NULL"); return MLENS_EINVAL; }
    mlens_grid g;
    ML_TRY(geometry(f, d, &g));
    cudaStream_t s = (cudaStream_t)stream;
    f->last_stream = s;
    size_t npix = (size_t)d->npix1 * d->npix2;
    Stage st(s);
    double *dmap = nullptr; unsigned long long *dcnt = nullptr;
    ML_TRY(st.out(map, npix, d->ptr_kind, &dmap));
    ML_TRY(st.out((unsigned long long *)counts, npix, d->ptr_kind, &dcnt));
    mlens_shoot_desc dd = *d;
    long long i0 = d->i0, i1 = d->i1, j0 = d->j0, j1 = d->j1;
    if (i1 <= 0 || j1 <= 0) { i0 = 0; i1 = g.n1; j0 = 0; j1 = g.n2; }
    size_t ndump = 0;
    if (d->dump_w1) {
        ndump = d->map_mode == MLENS_MAP_IPM ? (size_t)(i1 - i0 + 1) * (size_t)(j1 - j0 + 1) : (size_t)(i1 - i0) * (size_t)(j1 - j0);
        ML_TRY(st.out(d->dump_w1, ndump, d->ptr_kind, &dd.dump_w1));
        ML_TRY(st.out(d->dump_w2, ndump, d->ptr_kind, &dd.dump_w2));
    }
    if (d->ptr_kind == MLENS_PTR_HOST && d->accumulate) {
        if (map) ML_CUDA(cudaMemcpyAsync(dmap, map, npix * 8, cudaMemcpyHostToDevice, s));
        if (counts) ML_CUDA(cudaMemcpyAsync(dcnt, counts, npix * 8, cudaMemcpyHostToDevice, s));
    }
    ML_TRY(shoot(f, &dd, &g, dmap, dcnt, stats, s));
    ML_TRY(st.back(map, dmap, npix, d->ptr_kind, s));
    ML_TRY(st.back((unsigned long long *)counts, dcnt, npix, d->ptr_kind, s));
    if (ndump) { ML_TRY(st.back(d->dump_w1, dd.dump_w1, ndump, d->ptr_kind, s)); ML_TRY(st.back(d->dump_w2, dd.dump_w2, ndump, d->ptr_kind, s)); }
    if (d->ptr_kind == MLENS_PTR_HOST || d->sync) ML_CUDA(cudaStreamSynchronize(s));
    return MLENS_OK;
}

int mlens_map_light_curve(const double *map, int32_t npix1, int32_t npix2, double ylo1, double ylo2, double p1, double p2,
                          double ya1, double ya2, double yb1, double yb2, int64_t n, int32_t interp,
                          double *mu, int32_t ptr_kind, void *stream) {
    ML_TRY(check_device());
    if (!map || npix1 <= 0 || npix2 <= 0 || !(p1 > 0) || !(p2 > 0) || n < 0 || (n > 0 && !mu)) { set_error("bad arguments"); return MLENS_EINVAL; }
    if (interp != MLENS_INTERP_NEAREST && interp != MLENS_INTERP_BILINEAR) { set_error("bad interpolation mode"); return MLENS_EINVAL; }
    cudaStream_t s = (cudaStream_t)stream;
    Stage st(s);
    const size_t np = (size_t)npix1 * (size_t)npix2;
    const double *dmap; double *dmu;
    ML_TRY(st.in(map, np, ptr_kind, s, &dmap));
    ML_TRY(st.out(mu, (size_t)n, ptr_kind, &dmu));
    ML_TRY(map_light_curve(dmap, npix1, npix2, ylo1, ylo2, p1, p2, ya1, ya2, yb1, yb2, n, interp, dmu, s));
    ML_TRY(st.back(mu, dmu, (size_t)n, ptr_kind, s));
    if (ptr_kind == MLENS_PTR_HOST) ML_CUDA(cudaStreamSynchronize(s));
    return MLENS_OK;
}

int mlens_map_histogram(const double *map, int64_t n, double mu_ref, double lo, double hi, int32_t nbins,
                        uint64_t *counts, int32_t ptr_kind, void *stream) {
    ML_TRY(check_device());
    if (!counts || n < 0 || (n > 0 && !map) || nbins < 1 || nbins > 4096 || !(mu_ref > 0) || !(hi > lo)) { set_error("bad arguments"); return MLENS_EINVAL; }
    cudaStream_t s = (cudaStream_t)stream;
    Stage st(s);
    std::vector<double> edges((size_t)nbins + 1);
    for (int j = 0; j <= nbins; ++j) edges[j] = mu_ref * pow(10.0, lo + (double)j * (hi - lo) / (double)nbins);
    for (int j = 1; j <= nbins; ++j) if (!(edges[j] > edges[j - 1])) { set_error("bins too narrow for float64 edges"); return MLENS_EINVAL; }
    const double *dmap, *dedges; unsigned long long *dcounts;
    ML_TRY(st.in(map, (size_t)n, ptr_kind, s, &dmap));
    ML_TRY(st.in(edges.data(), edges.size(), MLENS_PTR_HOST, s, &dedges));
    ML_TRY(st.out(reinterpret_cast<unsigned long long *>(counts), (size_t)nbins + 2, ptr_kind, &dcounts));
    ML_TRY(map_histogram(dmap, n, dedges, nbins, dcounts, s));
    ML_TRY(st.back(reinterpret_cast<unsigned long long *>(counts), dcounts, (size_t)nbins + 2, ptr_kind, s));
    ML_CUDA(cudaStreamSynchronize(s));                              // `edges` is host memory of this call
    return MLENS_OK;
}

int mlens_field_get_tree(const mlens_field *f, mlens_tree_view *v) {
    if (!f || !v) { set_error("null argument"); return MLENS_EINVAL; }
    ML_CUDA(cudaStreamSynchronize(f->last_stream));
    const Tree &t = f->tree;
    size_t nn = (size_t)t.n_nodes, nl = (size_t)t.n_leaves, p1 = (size_t)f->order + 1, ns = (size_t)f->n_stars;
#define CP(dst, src, count) if (dst && (count)) ML_CUDA(cudaMemcpy(dst, src, (count) * sizeof(*(dst)), cudaMemcpyDeviceToHost))
    CP(v->level, t.level.p, nn); CP(v->ix, t.ix.p, nn); CP(v->iy, t.iy.p, nn); CP(v->parent, t.parent.p, nn);
    CP(v->child0, t.child0.p, nn); CP(v->star_lo, t.lo.p, nn); CP(v->star_n, t.n.p, nn); CP(v->leaf_id, t.leaf_id.p, nn);
    CP(v->nbr, t.nbr.p, nn * 8);
    CP(v->m2l_cnt, t.m2l_cnt.p, nn); CP(v->m2l_list, t.m2l_list.p, nn * 27);
    CP(v->p2l_cnt, t.p2l_cnt.p, nn); CP(v->p2l_list, t.p2l_list.p, nn * 8);
    CP(v->multipole, (const double *)t.mp.p, nn * p1 * 2); CP(v->local, (const double *)t.loc.p, nn * p1 * 2);
    CP(v->near_cnt, t.near_cnt.p, nl);
    CP(v->near_x, t.near_x.p, nl * ML_NEAR); CP(v->near_y, t.near_y.p, nl * ML_NEAR); CP(v->near_m, t.near_m.p, nl * ML_NEAR);
    CP(v->sorted_x, f->sx.p, ns); CP(v->sorted_y, f->sy.p, ns); CP(v->sorted_m, f->sm.p, ns);
#undef CP
    return MLENS_OK;
}

}  // extern "C"
