// tree.cu -- GPU adaptive quadtree (App. C1): Morton keys, LSD radix sort,
// level-by-level subdivision, neighbour / interaction / near-field lists.
//
// Membership of a star (or ray) in a node is decided by its ML_QBITS-bit quantised coordinates in the
// root square.  A node at level l is split into 4 children when the 3x3 block of level-l cells around
// it holds more than max_direct stars (reading R-tree); this alone keeps neighbouring leaves
// within one level of each other, the same-level interaction list <= 27 and the direct list <= max_direct.
#include "common.cuh"

namespace ml {

// ------------------------------------------------------------------------------------------------
// exclusive scan of int32 (in place), any n, recursive over block sums
static const int SCAN_T = 512, SCAN_E = 4, SCAN_B = SCAN_T * SCAN_E;

__global__ void scan_block_kernel(int *data, int n, int *block_sums) {
    __shared__ int warp_tot[SCAN_T / 32];
    int base = blockIdx.x * SCAN_B + threadIdx.x * SCAN_E;
    int v[SCAN_E], run = 0;
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) {
        int idx = base + e;
        v[e] = (idx < n) ? data[idx] : 0;
        run += v[e];
    }
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        int w = (lane < SCAN_T / 32) ? warp_tot[lane] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o) w += t;
        }
        if (lane < SCAN_T / 32) warp_tot[lane] = w;   // inclusive over warps
    }
    __syncthreads();
    int excl = inc - run + (warp ? warp_tot[warp - 1] : 0);
#pragma unroll
    for (int e = 0; e < SCAN_E; ++e) {
        int idx = base + e;
        if (idx < n) data[idx] = excl;
        excl += v[e];
    }
    if (threadIdx.x == SCAN_T - 1 && block_sums) block_sums[blockIdx.x] = warp_tot[SCAN_T / 32 - 1];
}

__global__ void scan_add_kernel(int *data, int n, const int *block_offsets) {
    int idx = blockIdx.x * SCAN_B + threadIdx.x;
    int off = block_offsets[blockIdx.x];
    for (int e = 0; e < SCAN_E; ++e, idx += SCAN_T)
        if (idx < n) data[idx] += off;
}

// scratch must hold at least n/SCAN_B + n/SCAN_B^2 + 8 ints
static int exclusive_scan(int *data, int n, int *scratch, cudaStream_t s) {
    if (n <= 0) return MLENS_OK;
    int nb = (n + SCAN_B - 1) / SCAN_B;
    ML_LAUNCH(scan_block_kernel, nb, SCAN_T, 0, s, data, n, nb > 1 ? scratch : nullptr);
    if (nb > 1) {
        ML_TRY(exclusive_scan(scratch, nb, scratch + nb, s));
        ML_LAUNCH(scan_add_kernel, nb, SCAN_T, 0, s, data, n, scratch);
    }
    ML_CUDA(cudaGetLastError());
    return MLENS_OK;
}
static size_t scan_scratch_ints(size_t n) { return n / SCAN_B + n / ((size_t)SCAN_B * SCAN_B) + 64; }

// ------------------------------------------------------------------------------------------------
// Morton keys: bit i of qx -> key bit 2i, bit i of qy -> key bit 2i+1 (child index = bx + 2 by)
__device__ __forceinline__ unsigned long long spread_bits(uint32_t v) {
    unsigned long long x = v;
    x = (x | (x << 16)) & 0x0000FFFF0000FFFFull;
    x = (x | (x << 8)) & 0x00FF00FF00FF00FFull;
    x = (x | (x << 4)) & 0x0F0F0F0F0F0F0F0Full;
    x = (x | (x << 2)) & 0x3333333333333333ull;
    x = (x | (x << 1)) & 0x5555555555555555ull;
    return x;
}

__global__ void extent_kernel(const double *x, const double *y, long long n, unsigned long long *out_bits) {
    double m = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        m = fmax(m, fmax(fabs(x[i]), fabs(y[i])));
    for (int o = 16; o; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out_bits, (unsigned long long)__double_as_longlong(m));  // m >= 0
}

__global__ void moments_kernel(const double *m, long long n, double *out /* sum m, sum m^2 */) {
    double a = 0.0, b = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double v = m[i];
        a += v; b += v * v;
    }
    for (int o = 16; o; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&out[0], a); atomicAdd(&out[1], b); }
}

__global__ void keys_kernel(const double *x, const double *y, int n, double root_half, double qscale,
                            unsigned long long *keys, int *idx) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double lim = (double)(1u << ML_QBITS) - 1.0;
    double fx = fmin(fmax(floor((x[i] + root_half) * qscale), 0.0), lim);
    double fy = fmin(fmax(floor((y[i] + root_half) * qscale), 0.0), lim);
    keys[i] = spread_bits((uint32_t)fx) | (spread_bits((uint32_t)fy) << 1);
    idx[i] = i;
}

// ---- LSD radix sort, 8-bit digits, stable.  Each block owns a contiguous chunk of RS_CHUNK elements.
static const int RS_T = 256, RS_CHUNK = 4096;

__global__ void rs_hist_kernel(const unsigned long long *keys, int n, int shift, int *hist, int nblocks) {
    __shared__ int h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    int base = blockIdx.x * RS_CHUNK;
    for (int e = threadIdx.x; e < RS_CHUNK; e += RS_T) {
        int i = base + e;
        if (i < n) atomicAdd(&h[(int)((keys[i] >> shift) & 255ull)], 1);
    }
    __syncthreads();
    hist[threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];   // digit-major so one scan gives global offsets
}

__global__ void rs_scatter_kernel(const unsigned long long *keys, const int *vals, int n, int shift,
                                  const int *offsets, int nblocks, unsigned long long *keys_out, int *vals_out) {
    __shared__ int base[256];                 // running output position of each digit for this block
    __shared__ int wcount[RS_T / 32][256];    // per-warp digit counts of the current round
    int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    base[tid] = offsets[tid * nblocks + blockIdx.x];
    int start = blockIdx.x * RS_CHUNK;
    for (int r = 0; r < RS_CHUNK; r += RS_T) {
        for (int w = 0; w < RS_T / 32; ++w) wcount[w][tid] = 0;
        __syncthreads();
        int i = start + r + tid;
        bool valid = i < n;
        unsigned long long k = valid ? keys[i] : 0ull;
        int d = valid ? (int)((k >> shift) & 255ull) : 256 + lane;   // invalid lanes never match
        unsigned m = __match_any_sync(0xffffffffu, d);
        int rank = __popc(m & ((1u << lane) - 1u));
        if (valid && rank == 0) wcount[warp][d] = __popc(m);
        __syncthreads();
        // thread `tid` owns digit `tid`: exclusive prefix over warps, then advance the base
        int run = 0;
        for (int w = 0; w < RS_T / 32; ++w) { int c = wcount[w][tid]; wcount[w][tid] = run; run += c; }
        int b0 = base[tid];
        __syncthreads();
        if (valid) {
            int pos = base[d] + wcount[warp][d] + rank;
            keys_out[pos] = k;
            vals_out[pos] = vals[i];
        }
        __syncthreads();
        base[tid] = b0 + run;
        __syncthreads();
    }
}

__global__ void gather_kernel(const int *idx, int n, const double *x, const double *y, const double *m,
                              const unsigned long long *keys, double *sx, double *sy, double *sm,
                              uint32_t *sqx, uint32_t *sqy) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int j = idx[i];
    sx[i] = x[j]; sy[i] = y[j]; sm[i] = m[j];
    unsigned long long k = keys[i];
    uint32_t qx = 0, qy = 0;
    for (int b = 0; b < ML_QBITS; ++b) {
        qx |= (uint32_t)((k >> (2 * b)) & 1ull) << b;
        qy |= (uint32_t)((k >> (2 * b + 1)) & 1ull) << b;
    }
    sqx[i] = qx; sqy[i] = qy;
}

// ------------------------------------------------------------------------------------------------
// tree levels
__constant__ int c_dx[8] = {-1, 0, 1, -1, 1, -1, 0, 1};
__constant__ int c_dy[8] = {-1, -1, -1, 0, 0, 1, 1, 1};
__device__ __forceinline__ int dir_index(int dx, int dy) {      // inverse of (c_dx, c_dy)
    int t = (dy + 1) * 3 + (dx + 1);                             // 0..8, 4 = centre
    return t < 4 ? t : t - 1;
}

struct TreeDev {
    int *level, *ix, *iy, *parent, *child0, *lo, *n, *nbr;
    const uint32_t *sqx, *sqy;
};

// stars of childless node Q that fall in cell (cx, cy) of level lev
__device__ __forceinline__ int count_in_cell(const TreeDev &T, int Q, int cx, int cy, int lev) {
    int sh = ML_QBITS - lev, c = 0;
    int lo = T.lo[Q], n = T.n[Q];
    for (int i = lo; i < lo + n; ++i)
        c += ((int)(T.sqx[i] >> sh) == cx) && ((int)(T.sqy[i] >> sh) == cy);
    return c;
}

// neighbours of every node of one level + the split decision
// The nodes of level `lev` are [range[lev], range[lev+1]): the level sizes stay on the device while the tree is built
// (the host launches every level with an upper bound of its size and reads the ranges back once).
__global__ void link_level_kernel(TreeDev T, const int *range, int lev, int max_direct, int *flags, int *overflow) {
    const int a = range[lev], b = range[lev + 1];
    int me = a + blockIdx.x * blockDim.x + threadIdx.x;
    if (me >= b) return;
    int ix = T.ix[me], iy = T.iy[me], P = T.parent[me];
    int count = T.n[me];
    int side = 1 << lev;
    for (int d = 0; d < 8; ++d) {
        int nx = ix + c_dx[d], ny = iy + c_dy[d];
        int res = -1;
        if (lev > 0 && nx >= 0 && ny >= 0 && nx < side && ny < side) {
            int ddx = (nx >> 1) - (ix >> 1), ddy = (ny >> 1) - (iy >> 1);
            int Q = (ddx == 0 && ddy == 0) ? P : T.nbr[(size_t)P * 8 + dir_index(ddx, ddy)];
            if (Q >= 0) {
                int c = T.child0[Q];
                if (c >= 0) {
                    res = c + (nx & 1) + 2 * (ny & 1);
                    count += T.n[res];
                } else {
                    res = -2 - Q;                                   // cell lies inside the coarser leaf Q
                    count += count_in_cell(T, Q, nx, ny, lev);
                }
            }
        }
        T.nbr[(size_t)me * 8 + d] = res;
    }
    int split = count > max_direct;
    if (split && lev >= ML_MAXLEV) { split = 0; atomicExch(overflow, 1); }
    flags[me - a] = split;
}

// range[lev+2] = end of the next level: the split nodes' children, unless they would not fit the node arrays (then
// nobody splits and *overflow is set: the host starts again with more room).
__global__ void next_level_kernel(int *range, int lev, const int *nsplit, int cap, int *overflow) {
    const int b = range[lev + 1];
    long long nb = (long long)b + 4ll * (long long)(*nsplit);
    if (nb > (long long)cap) { nb = b; atomicExch(overflow, 2); }
    range[lev + 2] = (int)nb;
}

__global__ void make_children_kernel(TreeDev T, const int *range, int lev, const int *flags, const int *rank,
                                     const unsigned long long *keys) {
    const int a = range[lev], b = range[lev + 1];
    int me = a + blockIdx.x * blockDim.x + threadIdx.x;
    if (me >= b) return;
    // flags were scanned in place into `rank`; a node splits iff rank[next] - rank[me] == 1, so the
    // caller passes the original flags separately
    if (!flags[me - a] || range[lev + 2] == b) { T.child0[me] = -1; return; }
    int c0 = b + 4 * rank[me - a];
    T.child0[me] = c0;
    int lo = T.lo[me], n = T.n[me];
    int sh = 2 * (ML_QBITS - 1 - lev);
    int bound[5];
    bound[0] = lo; bound[4] = lo + n;
    for (int q = 1; q < 4; ++q) {                 // first star whose child digit >= q
        int l = lo, r = lo + n;
        while (l < r) {
            int mid = (l + r) >> 1;
            if ((int)((keys[mid] >> sh) & 3ull) < q) l = mid + 1; else r = mid;
        }
        bound[q] = l;
    }
    int ix = T.ix[me], iy = T.iy[me];
    for (int q = 0; q < 4; ++q) {
        int c = c0 + q;
        T.level[c] = lev + 1;
        T.ix[c] = 2 * ix + (q & 1);
        T.iy[c] = 2 * iy + (q >> 1);
        T.parent[c] = me;
        T.child0[c] = -1;
        T.lo[c] = bound[q];
        T.n[c] = bound[q + 1] - bound[q];
    }
}

__global__ void init_tree_kernel(int *level, int *ix, int *iy, int *parent, int *child0, int *lo, int *nn, int n, int *range, int nr) {
    if (threadIdx.x == 0) { level[0] = 0; ix[0] = 0; iy[0] = 0; parent[0] = -1; child0[0] = -1; lo[0] = 0; nn[0] = n; }
    for (int l = threadIdx.x; l < nr; l += blockDim.x) range[l] = (l == 0) ? 0 : 1;
}

__global__ void leaf_flag_kernel(const int *child0, int n, int *flag) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) flag[i] = child0[i] < 0;
}

// interaction lists for every node + near-field lists for leaves
__global__ void lists_kernel(TreeDev T, int n_nodes, int *leaf_id /* in: exclusive scan of leaf flags */,
                             int *leaf_node, int *m2l_cnt, int *m2l_list, int *p2l_cnt, int *p2l_list,
                             int *near_cnt, double *near_x, double *near_y, double *near_m,
                             const double *sx, const double *sy, const double *sm, int *maxima) {
    int me = blockIdx.x * blockDim.x + threadIdx.x;
    if (me >= n_nodes) return;
    int lev = T.level[me], ix = T.ix[me], iy = T.iy[me], P = T.parent[me];
    int nm = 0, np = 0;
    if (lev >= 2) {
        for (int d = 0; d < 8; ++d) {
            int Q = T.nbr[(size_t)P * 8 + d];
            if (Q < 0) continue;                     // outside the root (a split node's neighbours all exist)
            int c = T.child0[Q];
            if (c >= 0) {
                int qx = T.ix[Q], qy = T.iy[Q];
                for (int q = 0; q < 4; ++q) {
                    int sx_ = 2 * qx + (q & 1), sy_ = 2 * qy + (q >> 1);
                    if (abs(sx_ - ix) > 1 || abs(sy_ - iy) > 1) m2l_list[(size_t)me * 27 + nm++] = c + q;
                }
            } else if (T.n[Q] > 0) {
                p2l_list[(size_t)me * 8 + np++] = Q;  // its stars outside the 3x3 block go through eq C6
            }
        }
    }
    m2l_cnt[me] = nm; p2l_cnt[me] = np;
    for (int k = nm; k < 27; ++k) m2l_list[(size_t)me * 27 + k] = -1;
    for (int k = np; k < 8; ++k) p2l_list[(size_t)me * 8 + k] = -1;
    atomicMax(&maxima[1], nm); atomicMax(&maxima[2], np);
    if (T.child0[me] >= 0) { leaf_id[me] = -1; return; }
    int leaf = leaf_id[me];
    leaf_node[leaf] = me;
    size_t o = (size_t)leaf * ML_NEAR;
    int cnt = 0;
    for (int i = T.lo[me]; i < T.lo[me] + T.n[me]; ++i, ++cnt)
        if (cnt < ML_NEAR) { near_x[o + cnt] = sx[i]; near_y[o + cnt] = sy[i]; near_m[o + cnt] = sm[i]; }
    int sh = ML_QBITS - lev;
    for (int d = 0; d < 8; ++d) {
        int nb = T.nbr[(size_t)me * 8 + d];
        if (nb >= 0) {
            for (int i = T.lo[nb]; i < T.lo[nb] + T.n[nb]; ++i, ++cnt)
                if (cnt < ML_NEAR) { near_x[o + cnt] = sx[i]; near_y[o + cnt] = sy[i]; near_m[o + cnt] = sm[i]; }
        } else if (nb <= -2) {
            int Q = -2 - nb, nx = ix + c_dx[d], ny = iy + c_dy[d];
            for (int i = T.lo[Q]; i < T.lo[Q] + T.n[Q]; ++i)
                if ((int)(T.sqx[i] >> sh) == nx && (int)(T.sqy[i] >> sh) == ny) {
                    if (cnt < ML_NEAR) { near_x[o + cnt] = sx[i]; near_y[o + cnt] = sy[i]; near_m[o + cnt] = sm[i]; }
                    ++cnt;
                }
        }
    }
    near_cnt[leaf] = min(cnt, ML_NEAR);
    atomicMax(&maxima[0], cnt);
}

// ------------------------------------------------------------------------------------------------
void Tree::release(cudaStream_t s) {
    level.release(s); ix.release(s); iy.release(s); parent.release(s); child0.release(s); lo.release(s); n.release(s);
    leaf_id.release(s); nbr.release(s); m2l_cnt.release(s); m2l_list.release(s); p2l_cnt.release(s); p2l_list.release(s);
    mp.release(s); loc.release(s); leaf_node.release(s); near_cnt.release(s); near_x.release(s); near_y.release(s);
    near_m.release(s); ecoef.release(s); ecoef_shoot.release(s); leaf_fold.release(s);
}

static int reserve_nodes(Tree &t, size_t n, cudaStream_t s) {
    ML_TRY(t.level.reserve(n, s)); ML_TRY(t.ix.reserve(n, s)); ML_TRY(t.iy.reserve(n, s));
    ML_TRY(t.parent.reserve(n, s)); ML_TRY(t.child0.reserve(n, s)); ML_TRY(t.lo.reserve(n, s));
    ML_TRY(t.n.reserve(n, s)); ML_TRY(t.nbr.reserve(n * 8, s));
    return MLENS_OK;
}

int build_tree(mlens_field *f, cudaStream_t s) {
    const long long N = f->n_stars;
    if (N > 0x7fffffffLL - 8) { set_error("too many stars"); return MLENS_EINVAL; }
    const int n = (int)N;
    Tree &t = f->tree;

    // ---- extent, moments
    ScratchBuf<unsigned long long> d_bits; ScratchBuf<double> d_mom;
    ML_TRY(d_bits.reserve(1, s)); ML_TRY(d_mom.reserve(2, s));
    ML_CUDA(cudaMemsetAsync(d_bits.p, 0, sizeof(unsigned long long), s));
    ML_CUDA(cudaMemsetAsync(d_mom.p, 0, 2 * sizeof(double), s));
    double extent = 0.0, mom[2] = {0, 0};
    if (n > 0) {
        int blocks = (int)((N + 255) / 256); if (blocks > 1184) blocks = 1184;
        ML_LAUNCH(extent_kernel, blocks, 256, 0, s, f->ox.p, f->oy.p, N, d_bits.p);
        ML_LAUNCH(moments_kernel, blocks, 256, 0, s, f->om.p, N, d_mom.p);
        unsigned long long bits = 0;
        ML_CUDA(cudaMemcpyAsync(&bits, d_bits.p, sizeof(bits), cudaMemcpyDeviceToHost, s));
        ML_CUDA(cudaMemcpyAsync(mom, d_mom.p, sizeof(mom), cudaMemcpyDeviceToHost, s));
        ML_CUDA(cudaStreamSynchronize(s));
        memcpy(&extent, &bits, sizeof(double));
    }
    d_bits.release(); d_mom.release();
    if (!(extent == extent) || extent > 1e300) { set_error("star coordinates are not finite"); return MLENS_EINVAL; }
    f->sum_m = mom[0];
    f->mean_m = n ? mom[0] / n : 0.0;
    f->mean_m2 = n ? mom[1] / n : 0.0;
    // The root square is twice the stars' extent: shooting windows reach a little past the star region
    // (config 1: H2 = 211.4 > R = 210.8), and rays outside the root can only be summed directly.
    f->root_half = 2.0 * extent * (1.0 + 1e-6);
    if (f->root_half < f->theta) f->root_half = f->theta;
    const double qscale = (double)(1u << ML_QBITS) / (2.0 * f->root_half);

    // ---- Morton sort
    ML_TRY(f->sx.reserve(n + 1, s, false)); ML_TRY(f->sy.reserve(n + 1, s, false)); ML_TRY(f->sm.reserve(n + 1, s, false));
    ML_TRY(f->sqx.reserve(n + 1, s, false)); ML_TRY(f->sqy.reserve(n + 1, s, false));
    ScratchBuf<unsigned long long> k0, k1; ScratchBuf<int> v0, v1, hist, scratch;
    if (n > 0) {
        ML_TRY(k0.reserve(n, s, false)); ML_TRY(k1.reserve(n, s, false));
        ML_TRY(v0.reserve(n, s, false)); ML_TRY(v1.reserve(n, s, false));
        int nb = (n + RS_CHUNK - 1) / RS_CHUNK;
        ML_TRY(hist.reserve((size_t)256 * nb, s, false));
        ML_TRY(scratch.reserve(scan_scratch_ints((size_t)256 * nb), s, false));
        ML_LAUNCH(keys_kernel, (n + 255) / 256, 256, 0, s, f->ox.p, f->oy.p, n, f->root_half, qscale, k0.p, v0.p);
        unsigned long long *ka = k0.p, *kb = k1.p; int *va = v0.p, *vb = v1.p;
        for (int shift = 0; shift < 2 * ML_QBITS; shift += 8) {
            ML_LAUNCH(rs_hist_kernel, nb, RS_T, 0, s, ka, n, shift, hist.p, nb);
            ML_TRY(exclusive_scan(hist.p, 256 * nb, scratch.p, s));
            ML_LAUNCH(rs_scatter_kernel, nb, RS_T, 0, s, ka, va, n, shift, hist.p, nb, kb, vb);
            std::swap(ka, kb); std::swap(va, vb);
        }
        ML_CUDA(cudaGetLastError());
        ML_LAUNCH(gather_kernel, (n + 255) / 256, 256, 0, s, va, n, f->ox.p, f->oy.p, f->om.p, ka, f->sx.p, f->sy.p, f->sm.p,
                                                      f->sqx.p, f->sqy.p);
        if (ka != k0.p) ML_CUDA(cudaMemcpyAsync(k0.p, ka, (size_t)n * sizeof(unsigned long long), cudaMemcpyDeviceToDevice, s));
        ML_CUDA(cudaGetLastError());
    }
    const unsigned long long *keys = k0.p;   // sorted keys

    // ---- levels: the loop runs on the device's own counts.  Level l is launched with an upper bound of its size
    // (four times the bound of the level above, at most the node capacity); the ranges come back once per chunk of
    // levels -- log4(n) + 3 levels in the first chunk, which is all of them for any star field that is not clustered.
    ScratchBuf<int> flags, rank, d_over, d_range;
    ML_TRY(d_over.reserve(1, s)); ML_TRY(d_range.reserve(ML_MAXLEV + 3, s));
    size_t cap = 2 * (size_t)n + 4096;
    int h_range[ML_MAXLEV + 3];
    for (;;) {                                                   // (again with more room if the nodes did not fit)
        if (cap > 0x7ffffff0u) { set_error("tree too large"); return MLENS_ERANGE; }
        ML_TRY(reserve_nodes(t, cap, s));
        {
            // root node, level ranges (level 0 = [0, 1), nothing below yet) and flags, written by a kernel: copies
            // from pageable host memory would make the host wait for the sort
            ML_LAUNCH(init_tree_kernel, 1, 32, 0, s, t.level.p, t.ix.p, t.iy.p, t.parent.p, t.child0.p, t.lo.p, t.n.p, n,
                      d_range.p, ML_MAXLEV + 3);
            ML_CUDA(cudaMemsetAsync(d_over.p, 0, 4, s));
        }
        TreeDev T{t.level.p, t.ix.p, t.iy.p, t.parent.p, t.child0.p, t.lo.p, t.n.p, t.nbr.p, f->sqx.p, f->sqy.p};
        int lev = 0, h_over = 0, n_levels = 0;
        long long ub = 1;                                        // upper bound of the size of level `lev`
        int chunk = 3;
        for (long long q = 1; q < (long long)n; q *= 4) ++chunk;
        while (n_levels == 0) {
            const int lev_end = (lev + chunk < ML_MAXLEV + 1) ? lev + chunk : ML_MAXLEV + 1;
            for (; lev < lev_end; ++lev) {
                const int u = (int)ub;
                ML_TRY(flags.reserve((size_t)u + 1, s, false)); ML_TRY(rank.reserve((size_t)u + 1, s, false));
                ML_TRY(scratch.reserve(scan_scratch_ints((size_t)u + 1), s, false));
                ML_CUDA(cudaMemsetAsync(flags.p, 0, ((size_t)u + 1) * 4, s));
                ML_LAUNCH(link_level_kernel, (u + 127) / 128, 128, 0, s, T, d_range.p, lev, f->max_direct, flags.p, d_over.p);
                ML_CUDA(cudaMemcpyAsync(rank.p, flags.p, ((size_t)u + 1) * 4, cudaMemcpyDeviceToDevice, s));
                ML_TRY(exclusive_scan(rank.p, u + 1, scratch.p, s));
                ML_LAUNCH(next_level_kernel, 1, 1, 0, s, d_range.p, lev, rank.p + u, (int)cap, d_over.p);
                ML_LAUNCH(make_children_kernel, (u + 127) / 128, 128, 0, s, T, d_range.p, lev, flags.p, rank.p, keys);
                ub = (4 * ub < (long long)cap) ? 4 * ub : (long long)cap;
            }
            ML_CUDA(cudaGetLastError());
            ML_CUDA(cudaMemcpyAsync(h_range, d_range.p, sizeof(h_range), cudaMemcpyDeviceToHost, s));
            ML_CUDA(cudaMemcpyAsync(&h_over, d_over.p, 4, cudaMemcpyDeviceToHost, s));
            ML_CUDA(cudaStreamSynchronize(s));
            if (h_over) break;
            for (int l = 0; l < lev; ++l)
                if (h_range[l + 2] == h_range[l + 1]) { n_levels = l + 1; break; }       // level l split nobody: it is the last
            if (n_levels == 0 && lev > ML_MAXLEV) n_levels = ML_MAXLEV + 1;
            if (n_levels == 0) { ub = h_range[lev + 1] - h_range[lev]; chunk = 4; }       // go on from the true size of the next level
        }
        if (h_over == 1) {
            set_error("more than max_direct stars within one cell of the deepest tree level (%d)", ML_MAXLEV);
            return MLENS_ERANGE;
        }
        if (h_over == 2) { cap *= 2; continue; }
        t.n_levels = n_levels;
        for (int l = 0; l <= n_levels; ++l) t.level_off[l] = h_range[l];
        t.n_nodes = h_range[n_levels];
        break;
    }
    d_over.release(); d_range.release();

    // ---- leaves and lists
    const int nn = t.n_nodes;
    ML_TRY(t.leaf_id.reserve(nn + 1, s, false));
    ML_TRY(scratch.reserve(scan_scratch_ints(nn + 1), s, false));
    ML_LAUNCH(leaf_flag_kernel, (nn + 255) / 256, 256, 0, s, t.child0.p, nn, t.leaf_id.p);
    ML_CUDA(cudaMemsetAsync(t.leaf_id.p + nn, 0, 4, s));
    ML_TRY(exclusive_scan(t.leaf_id.p, nn + 1, scratch.p, s));
    int nleaf = 0;
    ML_CUDA(cudaMemcpyAsync(&nleaf, t.leaf_id.p + nn, 4, cudaMemcpyDeviceToHost, s));
    ML_CUDA(cudaStreamSynchronize(s));
    t.n_leaves = nleaf;
    ML_TRY(t.leaf_node.reserve(nleaf, s, false)); ML_TRY(t.near_cnt.reserve(nleaf, s, false));
    ML_TRY(t.near_x.reserve((size_t)nleaf * ML_NEAR, s, false));
    ML_TRY(t.near_y.reserve((size_t)nleaf * ML_NEAR, s, false));
    ML_TRY(t.near_m.reserve((size_t)nleaf * ML_NEAR, s, false));
    ML_TRY(t.m2l_cnt.reserve(nn, s, false)); ML_TRY(t.m2l_list.reserve((size_t)nn * 27, s, false));
    ML_TRY(t.p2l_cnt.reserve(nn, s, false)); ML_TRY(t.p2l_list.reserve((size_t)nn * 8, s, false));
    ML_CUDA(cudaMemsetAsync(t.near_x.p, 0, (size_t)nleaf * ML_NEAR * 8, s));
    ML_CUDA(cudaMemsetAsync(t.near_y.p, 0, (size_t)nleaf * ML_NEAR * 8, s));
    ML_CUDA(cudaMemsetAsync(t.near_m.p, 0, (size_t)nleaf * ML_NEAR * 8, s));
    ScratchBuf<int> maxima; ML_TRY(maxima.reserve(4, s)); ML_CUDA(cudaMemsetAsync(maxima.p, 0, 16, s));
    TreeDev T{t.level.p, t.ix.p, t.iy.p, t.parent.p, t.child0.p, t.lo.p, t.n.p, t.nbr.p, f->sqx.p, f->sqy.p};
    ML_LAUNCH(lists_kernel, (nn + 127) / 128, 128, 0, s, T, nn, t.leaf_id.p, t.leaf_node.p, t.m2l_cnt.p, t.m2l_list.p,
                                                  t.p2l_cnt.p, t.p2l_list.p, t.near_cnt.p, t.near_x.p, t.near_y.p,
                                                  t.near_m.p, f->sx.p, f->sy.p, f->sm.p, maxima.p);
    int h_max[4];
    ML_CUDA(cudaMemcpyAsync(h_max, maxima.p, 16, cudaMemcpyDeviceToHost, s));
    ML_CUDA(cudaStreamSynchronize(s));
    ML_CUDA(cudaGetLastError());
    maxima.release();
    f->max_near = h_max[0]; f->max_m2l = h_max[1]; f->max_p2l = h_max[2];
    if (h_max[0] > ML_NEAR) { set_error("near-field list overflow (%d)", h_max[0]); return MLENS_ERANGE; }
    k0.release(); k1.release(); v0.release(); v1.release(); hist.release(); scratch.release();
    flags.release(); rank.release();
    return MLENS_OK;
}

}  // namespace ml
