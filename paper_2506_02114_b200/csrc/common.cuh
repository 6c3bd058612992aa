// common.cuh -- internal declarations of libmlens (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
#include <vector>
#include <new>
#include <atomic>

#include "../../include/mlens.h"

#define ML_P1MAX (MLENS_MAX_ORDER + 1)   // coefficients per expansion
#define ML_QBITS 24                      // quantised star / ray coordinate bits per axis
#define ML_MAXLEV 20                     // deepest tree level
#define ML_NEAR MLENS_MAX_DIRECT

namespace ml {

void set_error(const char *fmt, ...);

// every kernel the library launches goes through ML_LAUNCH so that mlens_launch_count() is a count, not a guess
extern std::atomic<long long> g_launches;
#define ML_LAUNCH(kernel, grid, block, smem, stream, ...)                         \
    do {                                                                          \
        ++ml::g_launches;                                                         \
        kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);               \
    } while (0)

#define ML_CUDA(call)                                                                  \
    do {                                                                               \
        cudaError_t e_ = (call);                                                       \
        if (e_ != cudaSuccess) {                                                       \
            ml::set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return (e_ == cudaErrorMemoryAllocation) ? MLENS_ENOMEM : MLENS_ECUDA;      \
        }                                                                              \
    } while (0)

#define ML_TRY(call)                 \
    do {                             \
        int rc_ = (call);            \
        if (rc_ != MLENS_OK) return rc_; \
    } while (0)

// Device memory comes from the stream-ordered pool of the device (cudaMallocAsync), with the pool told to keep
// what is freed: creating and destroying fields in a loop then costs no driver allocation at all.
int pool_init();

// One-time set-ups (memory-pool threshold, kernel attributes) are per DEVICE, not per process: a process may drive
// several GPUs.  Returns the current device's slot in such tables.
static const int ML_MAXDEV = 64;
inline int device_slot() {
    int dev = 0;
    cudaGetDevice(&dev);
    return (dev >= 0 && dev < ML_MAXDEV) ? dev : ML_MAXDEV - 1;
}

// Growable device array that keeps its contents on reserve().  Memory is stream-ordered: `s_own` is the stream of
// the last reserve (all of the library's work on a buffer is enqueued on the caller's stream), and a release is
// ordered after the work already enqueued there -- no device-wide synchronisation anywhere.
template <typename T>
struct DevBuf {
    T *p = nullptr;
    size_t cap = 0;
    cudaStream_t s_own = nullptr;
    int reserve(size_t n, cudaStream_t s, bool keep = true) {
        s_own = s;
        if (n <= cap) return MLENS_OK;
        ML_TRY(pool_init());
        size_t ncap = n + n / 4 + 64;
        T *q = nullptr;
        ML_CUDA(cudaMallocAsync(&q, ncap * sizeof(T), s));
        if (p && keep && cap) ML_CUDA(cudaMemcpyAsync(q, p, cap * sizeof(T), cudaMemcpyDeviceToDevice, s));
        if (p) ML_CUDA(cudaFreeAsync(p, s));
        p = q; cap = ncap;
        return MLENS_OK;
    }
    // A stream-ordered free can fail (the stream was destroyed before the buffer's owner): then the error is cleared
    // and the buffer is freed the plain way after a device synchronisation, so that nothing leaks silently.
    void release(cudaStream_t s) {
        if (p && cudaFreeAsync(p, s) != cudaSuccess) {
            cudaGetLastError();
            cudaDeviceSynchronize();
            if (cudaFreeAsync(p, nullptr) != cudaSuccess) { cudaGetLastError(); cudaFree(p); cudaGetLastError(); }
        }
        p = nullptr; cap = 0;
    }
    void release() { release(s_own); }
};
// Local scratch of a host function: freed (stream-ordered) on every way out of the scope, early returns included.
template <typename T>
struct ScratchBuf : DevBuf<T> {
    ScratchBuf() = default;
    ScratchBuf(const ScratchBuf &) = delete;
    ScratchBuf &operator=(const ScratchBuf &) = delete;
    ~ScratchBuf() { this->release(); }
};

struct Tree {
    int n_nodes = 0, n_leaves = 0, n_levels = 0;
    int level_off[ML_MAXLEV + 2] = {0};          // nodes of level l are [level_off[l], level_off[l+1])
    DevBuf<int> level, ix, iy, parent, child0, lo, n, leaf_id, nbr;   // nbr: 8 per node
    DevBuf<int> m2l_cnt, m2l_list, p2l_cnt, p2l_list;                 // 27 / 8 per node
    DevBuf<double2> mp, loc;                     // n_nodes * P1
    DevBuf<int> leaf_node;                       // n_leaves
    DevBuf<int> near_cnt;                        // n_leaves
    DevBuf<double> near_x, near_y, near_m;       // n_leaves * ML_NEAR
    DevBuf<double2> ecoef;                       // n_leaves * P1: (l+1) c_{l+1} theta^2/L, l = 0..p-1
    DevBuf<double2> ecoef_shoot;                 // rectangle fields: + the sheet's analytic part (fmm.cu rect_fold)
    DevBuf<unsigned char> leaf_fold;             // n_leaves
    void release(cudaStream_t s);
};

}  // namespace ml

struct mlens_field {
    // lens
    double kappa_tot = 0, kappa_star = 0, kappa_smooth = 0, gamma = 0, theta = 1;
    int shape = 0;
    double R = 0, c1 = 0, c2 = 0;
    double eps = 1e-8;
    double quad[4] = {0, 0, 0, 0};  // psi_111, psi_112, psi_122, psi_222 of the macro potential (reading G23); all zero = off
    int max_direct = 32;
    int order = 0;                 // p
    int64_t n_stars = 0;
    // stars: original order and Morton order
    ml::DevBuf<double> ox, oy, om, sx, sy, sm;
    ml::DevBuf<uint32_t> sqx, sqy;
    double root_half = 1.0;
    double mean_m = 0, mean_m2 = 0, sum_m = 0;
    double spot_err = 0;
    int max_near = 0, max_m2l = 0, max_p2l = 0;
    ml::Tree tree;
    // tables
    ml::DevBuf<double> binom;      // (2*P1MAX) x (2*P1MAX) Pascal triangle
    ml::DevBuf<double2> tab;       // power tables, see fmm.cu
    // shoot scratch
    ml::DevBuf<unsigned long long> acc;  // fixed-point / count accumulator, npix
    ml::DevBuf<unsigned long long> diff; // row-difference array of interior runs (IPM), npix
    ml::DevBuf<double> queue;            // general-triangle queue
    ml::DevBuf<int> qcount;              // entries per queue chunk
    ml::DevBuf<unsigned int> biglist;    // queue entries to be walked edge by edge
    ml::DevBuf<unsigned long long> giant; // chunks of the giant triangles among them
    ml::DevBuf<unsigned long long> giant_sorted;
    ml::DevBuf<unsigned char> giant_key;
    ml::DevBuf<unsigned int> giant_hist;
    ml::DevBuf<unsigned long long> counters;
    int device = 0;
    cudaStream_t last_stream = nullptr;   // stream of the most recent call on this field: destroy frees in its order
};

namespace ml {
// tree.cu
int build_tree(mlens_field *f, cudaStream_t s);
// fmm.cu
int fmm_prepare_tables(mlens_field *f, cudaStream_t s);
int fmm_passes(mlens_field *f, cudaStream_t s);     // upward + downward + leaf coefficients for f->order
int rect_fold(mlens_field *f, cudaStream_t s);      // rectangle fields: the sheet's analytic part into a copy of the leaf series
// eval.cu
int deflect_points(const mlens_field *f, int64_t n, const double *zx, const double *zy, double *ox_, double *oy_,
                   int eval_mode, int full_lens, cudaStream_t s);
// starfield.cu
int generate_stars(uint64_t seed, int64_t n, int shape, double a1, double a2, int mass_law, double a,
                   double lo, double hi, double *x, double *y, double *m, cudaStream_t s);
// shoot.cu
// The general-triangle queue is gigabytes of scratch that belongs to no field in particular: a destroyed field
// parks it here (with an event on its stream) and the next field that shoots on that device takes it (after the event),
// so that creating and destroying fields in a loop never allocates it again.
void scratch_park(mlens_field *f, cudaStream_t s);
void scratch_take(mlens_field *f, cudaStream_t s);
int geometry(const mlens_field *f, const mlens_shoot_desc *d, mlens_grid *g);
int shoot(mlens_field *f, const mlens_shoot_desc *d, const mlens_grid *g, double *map,
          unsigned long long *counts, mlens_stats *st, cudaStream_t s);
// consume.cu
int map_histogram(const double *map, long long n, const double *edges_dev, int nbins, unsigned long long *counts, cudaStream_t s);
int map_light_curve(const double *map, int npix1, int npix2, double ylo1, double ylo2, double p1, double p2,
                    double ya1, double ya2, double yb1, double yb2, long long n, int interp, double *mu, cudaStream_t s);
}  // namespace ml
