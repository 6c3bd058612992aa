// consume.cu -- what the paper reads off a finished magnification map: light curves
// along straight source tracks (Fig 4, Fig 8) and magnification histograms (Fig 5, Fig 10).
// Both are HBM-bandwidth work: the histogram reads the map once, privatised per block in shared memory.
#include "common.cuh"
#include <math.h>

namespace ml {

static const int HIST_T = 256;
static const int HIST_MAXBINS = 4096;

// counts[0] = below edge[0] (also mu <= 0 and NaN), counts[1 + j] = edge[j] <= mu < edge[j+1], counts[nbins + 1] = the rest.
// The bin is DECIDED by comparisons with the float64 edges, so the decision is the same on any machine; a float32
// logarithm only proposes where to start comparing (the bins are equal in log mu, so it is off by one at most
// except next to an edge).
__device__ __forceinline__ int hist_slot(double mu, const double *se, int nbins, float lg_lo, float inv_w) {
    if (!(mu >= se[0])) return 0;                                                    // also NaN
    if (mu >= se[nbins]) return nbins + 1;
    int j = (int)((__log2f((float)mu) - lg_lo) * inv_w);                             // proposal
    j = min(max(j, 0), nbins - 1);
    while (mu < se[j]) --j;                                                          // se[0] <= mu < se[nbins]: both loops end inside
    while (mu >= se[j + 1]) ++j;
    return 1 + j;
}

__global__ void __launch_bounds__(HIST_T) histogram_kernel(const double *__restrict__ map, long long n, const double *__restrict__ edge,
                                                           int nbins, int rep, unsigned long long *counts) {
    extern __shared__ unsigned char smem_raw[];
    double *se = reinterpret_cast<double *>(smem_raw);                               // nbins + 1 edges
    unsigned int *sc = reinterpret_cast<unsigned int *>(se + nbins + 1);             // (nbins + 2) counters, `rep` copies of each
    for (int i = threadIdx.x; i <= nbins; i += HIST_T) se[i] = edge[i];
    for (int i = threadIdx.x; i < (nbins + 2) * rep; i += HIST_T) sc[i] = 0u;
    __syncthreads();
    const float lg_lo = __log2f((float)se[0]);
    const float inv_w = (float)nbins / (__log2f((float)se[nbins]) - lg_lo);
    const int r = threadIdx.x & (rep - 1);                                           // maps pile up in a few bins: lanes spread over the copies
    const long long stride = (long long)gridDim.x * HIST_T;
    const long long n4 = n / (4 * stride) * (4 * stride);                            // whole rounds of four coalesced loads per thread
    for (long long i = (long long)blockIdx.x * HIST_T + threadIdx.x; i < n4; i += 4 * stride) {
        double mu[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) mu[k] = __ldcs(&map[i + k * stride]);
#pragma unroll
        for (int k = 0; k < 4; ++k) atomicAdd(&sc[hist_slot(mu[k], se, nbins, lg_lo, inv_w) * rep + r], 1u);
    }
    for (long long i = n4 + (long long)blockIdx.x * HIST_T + threadIdx.x; i < n; i += stride)
        atomicAdd(&sc[hist_slot(map[i], se, nbins, lg_lo, inv_w) * rep + r], 1u);
    __syncthreads();
    for (int k = threadIdx.x; k < nbins + 2; k += HIST_T) {
        unsigned long long t = 0;
        for (int q = 0; q < rep; ++q) t += sc[k * rep + q];
        if (t) atomicAdd(&counts[k], t);
    }
}

int map_histogram(const double *map, long long n, const double *edges_dev, int nbins, unsigned long long *counts, cudaStream_t s) {
    ML_CUDA(cudaMemsetAsync(counts, 0, (size_t)(nbins + 2) * 8, s));
    if (n <= 0) return MLENS_OK;
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    long long want = (n + HIST_T - 1) / HIST_T;
    const long long cap = (long long)nsm * 8;                      // 2048 threads per SM
    const unsigned grid = (unsigned)(want < cap ? want : cap);
    int rep = 16;                                                  // copies of every counter: as many as 48 KB allow
    while (rep > 1 && (size_t)(nbins + 1) * 8 + (size_t)(nbins + 2) * 4 * rep > 48 * 1024) rep >>= 1;
    const size_t smem = (size_t)(nbins + 1) * 8 + (size_t)(nbins + 2) * 4 * rep;
    static std::atomic<int> attr_set[ML_MAXDEV];                   // kernel attributes are per device (context)
    if (!attr_set[device_slot()].load()) {
        ML_CUDA(cudaFuncSetAttribute(histogram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (HIST_MAXBINS + 1) * 8 + (HIST_MAXBINS + 2) * 4));
        attr_set[device_slot()].store(1);
    }
    if (n / grid >= (1ll << 32)) { set_error("map too large for the histogram's 32-bit block counters"); return MLENS_EINVAL; }
    ML_LAUNCH(histogram_kernel, grid, HIST_T, smem, s, map, n, edges_dev, nbins, rep, counts);
    ML_CUDA(cudaGetLastError());
    return MLENS_OK;
}

// One thread per sample.  Pixel of a point: floor((y - ylo)/p) with a true division (the rule of the map itself).
__global__ void light_curve_kernel(const double *__restrict__ map, int npix1, int npix2, double ylo1, double ylo2, double p1, double p2,
                                   double ya1, double ya2, double yb1, double yb2, long long n, int interp, double *mu) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double t = (n > 1) ? (double)i / (double)(n - 1) : 0.0;
    const double y1 = ya1 + (yb1 - ya1) * t, y2 = ya2 + (yb2 - ya2) * t;
    const double u = (y1 - ylo1) / p1, v = (y2 - ylo2) / p2;                         // pixel units
    double out = nan("");
    if (u >= 0.0 && v >= 0.0 && u < (double)npix1 && v < (double)npix2) {
        if (interp == MLENS_INTERP_NEAREST) {
            out = map[(size_t)(int)floor(v) * npix1 + (int)floor(u)];
        } else {
            // centres sit at integer + 0.5: the cell of centres that holds the point, indices clamped at the border
            const double uc = u - 0.5, vc = v - 0.5;
            const double fu = floor(uc), fv = floor(vc);
            const double a = uc - fu, b = vc - fv;
            const int i0 = max((int)fu, 0), i1 = min((int)fu + 1, npix1 - 1);
            const int j0 = max((int)fv, 0), j1 = min((int)fv + 1, npix2 - 1);
            const double m00 = map[(size_t)j0 * npix1 + i0], m10 = map[(size_t)j0 * npix1 + i1];
            const double m01 = map[(size_t)j1 * npix1 + i0], m11 = map[(size_t)j1 * npix1 + i1];
            out = (1.0 - b) * ((1.0 - a) * m00 + a * m10) + b * ((1.0 - a) * m01 + a * m11);
        }
    }
    mu[i] = out;
}

int map_light_curve(const double *map, int npix1, int npix2, double ylo1, double ylo2, double p1, double p2,
                    double ya1, double ya2, double yb1, double yb2, long long n, int interp, double *mu, cudaStream_t s) {
    if (n <= 0) return MLENS_OK;
    const int T = 256;
    ML_LAUNCH(light_curve_kernel, (unsigned)((n + T - 1) / T), T, 0, s, map, npix1, npix2, ylo1, ylo2, p1, p2, ya1, ya2, yb1, yb2, n, interp, mu);
    ML_CUDA(cudaGetLastError());
    return MLENS_OK;
}

}  // namespace ml

// ---- mlens_map_histogram_static: the histogram for callers that must not allocate device memory -------------------
// histogram_kernel reads its bin edges from global memory.  mlens_map_histogram gets that table from the device's
// memory pool on every call; here it lives in the library's own image instead: one fixed array per GPU, there from the
// moment the library is loaded on that GPU until the process ends, shared by every call of this entry point.
static __device__ __align__(256) double g_static_hist_edges[MLENS_HIST_STATIC_MAXBINS + 1];

namespace ml {
// In host code `g_static_hist_edges` is only a handle for the runtime's symbol calls, not somewhere a kernel can read:
// the array's address on the CURRENT device is asked for once per device and kept here.
static int static_hist_edges(double **out) {
    static std::atomic<double *> addr[ML_MAXDEV];                   // zero-initialised; one slot per device
    int dev = 0;
    ML_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= ML_MAXDEV) { set_error("device ordinal %d beyond the %d this table holds", dev, ML_MAXDEV); return MLENS_EINVAL; }
    double *p = addr[dev].load();
    if (!p) {
        ML_CUDA(cudaGetSymbolAddress((void **)&p, g_static_hist_edges));
        if (!p) { set_error("cudaGetSymbolAddress gave a null address for the static edge table"); return MLENS_ECUDA; }
        addr[dev].store(p);                                         // two threads racing here store the same value
    }
    *out = p;
    return MLENS_OK;
}

static int must_be_device_memory(const void *p, const char *what) {
    cudaPointerAttributes a;
    ML_CUDA(cudaPointerGetAttributes(&a, p));
    if (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged) {
        set_error("%s must be device memory: this entry point stages nothing (it may not allocate)", what);
        return MLENS_EINVAL;
    }
    return MLENS_OK;
}
}  // namespace ml

extern "C" int mlens_map_histogram_static(const double *map, int64_t n, double mu_ref, double lo, double hi, int32_t nbins,
                                          uint64_t *counts, void *stream) {
    using namespace ml;
    if (nbins > MLENS_HIST_STATIC_MAXBINS) {
        set_error("nbins = %d is more than the static edge table holds (MLENS_HIST_STATIC_MAXBINS = %d); "
                  "use mlens_map_histogram, which allocates", nbins, MLENS_HIST_STATIC_MAXBINS);
        return MLENS_EINVAL;
    }
    if (!counts || n < 0 || (n > 0 && !map) || nbins < 1 || !(mu_ref > 0) || !(hi > lo)) { set_error("bad arguments"); return MLENS_EINVAL; }
    ML_TRY(must_be_device_memory(counts, "counts"));
    if (n > 0) ML_TRY(must_be_device_memory(map, "map"));
    // the same expression as mlens_map_histogram (api.cu), so the two entry points decide every pixel alike
    double edges[MLENS_HIST_STATIC_MAXBINS + 1];                     // 32 KB of stack, no heap
    for (int j = 0; j <= nbins; ++j) edges[j] = mu_ref * pow(10.0, lo + (double)j * (hi - lo) / (double)nbins);
    for (int j = 1; j <= nbins; ++j) if (!(edges[j] > edges[j - 1])) { set_error("bins too narrow for float64 edges"); return MLENS_EINVAL; }
    double *dedges = nullptr;
    ML_TRY(static_hist_edges(&dedges));                              // first call on a device: looks the array up
    cudaStream_t s = (cudaStream_t)stream;
    // Entries 0..nbins are overwritten, the kernel reads no others: whatever an earlier call left behind is never seen
    // and nothing has to be zeroed.  `edges` is pageable, so the runtime has taken its copy when this returns.
    ML_CUDA(cudaMemcpyAsync(dedges, edges, (size_t)(nbins + 1) * sizeof(double), cudaMemcpyHostToDevice, s));
    return map_histogram(map, n, dedges, nbins, reinterpret_cast<unsigned long long *>(counts), s);
}
