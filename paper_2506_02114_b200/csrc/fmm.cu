// fmm.cu -- upward pass (P2M eq C2, M2M eq C3), downward pass (M2L eq C5, P2L eq C6, L2L eq C7) and the
// per-leaf Taylor coefficients used by the ray evaluator (eq 24 / C4).  App. C2 of the paper.
// All coefficients are in units of the node half-length.  c_0 and every logarithm are
// dropped: they never enter a deflection (reading G1).
#include "device.cuh"
#include <mutex>

namespace ml {

// table layout inside mlens_field::tab (double2 entries, ML_P1MAX per row)
static const int TAB_M2M = 0;                  // 4 rows: z0^n, z0 = (+-1 +- i), row = bx + 2 by
static const int TAB_L2L = 4;                  // 4 rows: (z0/2)^n
static const int TAB_M2L = 8;                  // 49 rows: (-1/z0)^n, z0 = 2(dx + i dy), row = (dy+3)*7 + dx+3
static const int TAB_ROWS = 8 + 49;
static const int BN = 2 * ML_P1MAX;            // Pascal triangle stride

// The tables depend on nothing but compile-time constants: they are built and uploaded once per device and process,
// and every field borrows them (mlens_field_destroy does not free them).
static int build_tables(DevBuf<double> &binom, DevBuf<double2> &tabd, cudaStream_t s) {
    std::vector<double> bin((size_t)BN * BN, 0.0);
    for (int n = 0; n < BN; ++n) {
        bin[(size_t)n * BN] = 1.0;
        for (int k = 1; k <= n; ++k)
            bin[(size_t)n * BN + k] = bin[(size_t)(n - 1) * BN + k - 1] + (k <= n - 1 ? bin[(size_t)(n - 1) * BN + k] : 0.0);
    }
    std::vector<double2> tab((size_t)TAB_ROWS * ML_P1MAX);
    for (int q = 0; q < 4; ++q) {
        double2 z0 = make_double2((q & 1) ? 1.0 : -1.0, (q >> 1) ? 1.0 : -1.0);
        double2 zh = make_double2(0.5 * z0.x, 0.5 * z0.y);
        for (int n = 0; n < ML_P1MAX; ++n) {
            tab[(size_t)(TAB_M2M + q) * ML_P1MAX + n] = cpowi(z0, n);
            tab[(size_t)(TAB_L2L + q) * ML_P1MAX + n] = cpowi(zh, n);
        }
    }
    for (int dy = -3; dy <= 3; ++dy)
        for (int dx = -3; dx <= 3; ++dx) {
            int row = TAB_M2L + (dy + 3) * 7 + dx + 3;
            double2 w = make_double2(0.0, 0.0);
            if (dx || dy) { double2 z0 = make_double2(2.0 * dx, 2.0 * dy); w = cinv(z0); w.x = -w.x; w.y = -w.y; }
            for (int n = 0; n < ML_P1MAX; ++n) tab[(size_t)row * ML_P1MAX + n] = cpowi(w, n);
        }
    ML_TRY(binom.reserve(bin.size(), s, false));
    ML_TRY(tabd.reserve(tab.size(), s, false));
    ML_CUDA(cudaMemcpyAsync(binom.p, bin.data(), bin.size() * sizeof(double), cudaMemcpyHostToDevice, s));
    ML_CUDA(cudaMemcpyAsync(tabd.p, tab.data(), tab.size() * sizeof(double2), cudaMemcpyHostToDevice, s));
    ML_CUDA(cudaStreamSynchronize(s));
    return MLENS_OK;
}

int fmm_prepare_tables(mlens_field *f, cudaStream_t s) {
    static const int MAXDEV = 64;
    static std::mutex mtx;
    static DevBuf<double> c_binom[MAXDEV];
    static DevBuf<double2> c_tab[MAXDEV];
    if (f->device < 0 || f->device >= MAXDEV) { set_error("device index out of range"); return MLENS_EINVAL; }
    std::lock_guard<std::mutex> lock(mtx);
    if (!c_binom[f->device].p || !c_tab[f->device].p) ML_TRY(build_tables(c_binom[f->device], c_tab[f->device], s));
    f->binom.p = c_binom[f->device].p; f->binom.cap = 0;          // borrowed
    f->tab.p = c_tab[f->device].p; f->tab.cap = 0;
    return MLENS_OK;
}

struct FmmDev {
    const int *level, *ix, *iy, *parent, *child0, *lo, *n;
    const int *m2l_cnt, *m2l_list, *p2l_cnt, *p2l_list, *leaf_node;
    const double *sx, *sy, *sm;
    const uint32_t *sqx, *sqy;
    double2 *mp, *loc, *ecoef;
    const double *binom;
    const double2 *tab;
    double root_half, theta2;
    int p, p1;
};

__device__ __forceinline__ void node_geom(const FmmDev &F, int node, double &cx, double &cy, double &half) {
    int lev = F.level[node];
    half = F.root_half / (double)(1 << lev);
    cx = -F.root_half + (2.0 * F.ix[node] + 1.0) * half;
    cy = -F.root_half + (2.0 * F.iy[node] + 1.0) * half;
}

// P2M, eq C2: a_0 = sum m, a_k = -(1/k) sum m zeta^k.  One block per childless node,
// thread k owns coefficient k ("done in parallel").  Also serves the childless nodes of the
// coarser levels.
__global__ void p2m_kernel(FmmDev F, int n_leaves) {
    int leaf = blockIdx.x;
    int k = threadIdx.x;
    if (leaf >= n_leaves || k > F.p) return;
    int node = F.leaf_node[leaf];
    double cx, cy, half;
    node_geom(F, node, cx, cy, half);
    double inv = 1.0 / half;
    int lo = F.lo[node], n = F.n[node];
    double2 acc = make_double2(0.0, 0.0);
    for (int i = lo; i < lo + n; ++i) {
        double m = F.sm[i];
        if (k == 0) { acc.x += m; continue; }
        double2 zeta = make_double2((F.sx[i] - cx) * inv, (F.sy[i] - cy) * inv);
        double2 pw = cpowi(zeta, k);
        acc.x -= m * pw.x; acc.y -= m * pw.y;
    }
    if (k > 0) { acc.x /= (double)k; acc.y /= (double)k; }
    F.mp[(size_t)node * F.p1 + k] = acc;
}

// M2M, eq C3: b_l = -a_0 z0^l/l + sum_{k=1}^{l} a_k z0^(l-k) C(l-1,k-1), then / 2^l; the
// four shifted children are added.  One block per node of the level, thread l owns b_l.
__global__ void m2m_kernel(FmmDev F, int a, int b) {
    __shared__ double2 ch[4][ML_P1MAX];
    int node = a + blockIdx.x;
    if (node >= b) return;
    int c0 = F.child0[node];
    if (c0 < 0) return;                       // childless: P2M already wrote its coefficients
    int l = threadIdx.x;
    if (l <= F.p)
        for (int q = 0; q < 4; ++q) ch[q][l] = F.mp[(size_t)(c0 + q) * F.p1 + l];
    __syncthreads();
    if (l > F.p) return;
    double2 acc = make_double2(0.0, 0.0);
    for (int q = 0; q < 4; ++q) {
        const double2 *zp = F.tab + (size_t)(TAB_M2M + q) * ML_P1MAX;
        if (l == 0) { acc.x += ch[q][0].x; acc.y += ch[q][0].y; continue; }
        double2 t = cscale(zp[l], -ch[q][0].x / (double)l);       // a_0 is real
        for (int k = 1; k <= l; ++k) {
            double bc = F.binom[(size_t)(l - 1) * BN + (k - 1)];
            double2 u = cmul(ch[q][k], zp[l - k]);
            t.x = fma(bc, u.x, t.x); t.y = fma(bc, u.y, t.y);
        }
        acc.x += t.x; acc.y += t.y;
    }
    double sc = scalbn(1.0, -l);
    F.mp[(size_t)node * F.p1 + l] = cscale(acc, sc);
}

// Downward pass for the nodes [a, b) of one level: L2L from the parent (eq C7), M2L over the same-level
// interaction list (eq C5), P2L from the stars of childless coarser nodes (eq C6).  One block per node,
// thread l owns local coefficient l; source coefficients are staged (pre-scaled) in shared memory.
__global__ void downward_kernel(FmmDev F, int a, int b) {
    __shared__ double2 src[ML_P1MAX];
    int node = a + blockIdx.x;
    if (node >= b) return;
    const int l = threadIdx.x, p = F.p;
    const bool act = (l <= p);
    int P = F.parent[node];
    int ix = F.ix[node], iy = F.iy[node], lev = F.level[node];
    double2 acc = make_double2(0.0, 0.0);

    // ---- L2L (eq C7 with z0 = (child - parent)/L_parent, reading G3): d_l = sum_{k>=l} c_k C(k,l) z0^(k-l) / 2^l
    if (act) src[l] = F.loc[(size_t)P * F.p1 + l];
    __syncthreads();
    if (act && l >= 1) {
        int q = (ix & 1) + 2 * (iy & 1);
        const double2 *zp = F.tab + (size_t)(TAB_L2L + q) * ML_P1MAX;
        double2 t = make_double2(0.0, 0.0);
        for (int k = l; k <= p; ++k) {
            double bc = F.binom[(size_t)k * BN + l];
            double2 u = cmul(src[k], zp[k - l]);
            t.x = fma(bc, u.x, t.x); t.y = fma(bc, u.y, t.y);
        }
        acc = cscale(t, scalbn(1.0, -l));
    }

    // ---- M2L (eq C5): c_l = z0^-l [ -b_0/l + sum_{k=1}^{p} b_k (-z0)^-k C(l+k-1,k-1) ]
    int nm = F.m2l_cnt[node];
    for (int e = 0; e < nm; ++e) {
        int S = F.m2l_list[(size_t)node * 27 + e];
        int dx = F.ix[S] - ix, dy = F.iy[S] - iy;
        const double2 *wp = F.tab + (size_t)(TAB_M2L + (dy + 3) * 7 + dx + 3) * ML_P1MAX;   // (-1/z0)^n
        __syncthreads();
        if (act) src[l] = cmul(F.mp[(size_t)S * F.p1 + l], wp[l]);
        __syncthreads();
        if (act && l >= 1) {
            double2 t = make_double2(-src[0].x / (double)l, 0.0);
            for (int k = 1; k <= p; ++k) {
                double bc = F.binom[(size_t)(l + k - 1) * BN + (k - 1)];
                t.x = fma(bc, src[k].x, t.x); t.y = fma(bc, src[k].y, t.y);
            }
            double2 zi = wp[l];                                   // (1/z0)^l = (-1)^l (-1/z0)^l
            if (l & 1) { zi.x = -zi.x; zi.y = -zi.y; }
            double2 u = cmul(t, zi);
            acc.x += u.x; acc.y += u.y;
        }
    }

    // ---- P2L (eq C6): c_l = sum -m/(l zeta^l) over the stars of coarser childless nodes that lie
    // outside this node's 3x3 block (those inside are in the near-field list)
    int np = F.p2l_cnt[node];
    if (np > 0 && act && l >= 1) {
        double cx, cy, half;
        node_geom(F, node, cx, cy, half);
        int sh = ML_QBITS - lev;
        for (int e = 0; e < np; ++e) {
            int Q = F.p2l_list[(size_t)node * 8 + e];
            int lo = F.lo[Q], n = F.n[Q];
            for (int i = lo; i < lo + n; ++i) {
                int cxq = (int)(F.sqx[i] >> sh), cyq = (int)(F.sqy[i] >> sh);
                if (abs(cxq - ix) <= 1 && abs(cyq - iy) <= 1) continue;
                double2 zeta = make_double2((F.sx[i] - cx) / half, (F.sy[i] - cy) / half);
                double2 w = cpowi(cinv(zeta), l);
                double f = -F.sm[i] / (double)l;
                acc.x = fma(f, w.x, acc.x); acc.y = fma(f, w.y, acc.y);
            }
        }
    }
    if (act) F.loc[(size_t)node * F.p1 + l] = (l >= 1) ? acc : make_double2(0.0, 0.0);
}

// The downward pass for orders p <= 31: one WARP per node, lane = coefficient l, no block barriers.  M2L is a
// real p x p binomial matrix (the same for every pair, eq C5) times the complex source vectors scaled by powers of
// -1/z0: the matrix sits transposed in shared memory (lane-contiguous, conflict free), DW_NP source vectors are
// staged per pass so that one matrix element feeds 2 DW_NP FMAs, and the inner loop is bound by the FP64 pipe.
static const int DW_WARPS = 8, DW_NP = 4, DW_PMAX = 31;
__global__ void __launch_bounds__(DW_WARPS * 32) downward_warp_kernel(FmmDev F, int a, int b) {
    __shared__ double Bt[DW_PMAX * 32];                         // Bt[(k-1) 32 + l] = C(l+k-1, k-1)
    __shared__ double2 src_s[DW_WARPS][DW_NP][32];
    const unsigned full = 0xffffffffu;
    const int p = F.p, l = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < p * 32; i += blockDim.x) {
        const int k = i / 32 + 1, ll = i % 32;
        Bt[i] = (ll >= 1 && ll <= p) ? F.binom[(size_t)(ll + k - 1) * BN + (k - 1)] : 0.0;
    }
    __syncthreads();
    double2 (*src)[32] = src_s[warp];
    const bool act = (l <= p), row = act && (l >= 1);
    const double inv_l = (l >= 1) ? 1.0 / (double)l : 0.0;
    for (int node = a + blockIdx.x * DW_WARPS + warp; node < b; node += gridDim.x * DW_WARPS) {
        const int P = F.parent[node], ix = F.ix[node], iy = F.iy[node], lev = F.level[node];
        double2 acc = make_double2(0.0, 0.0);
        // ---- L2L (eq C7, reading G3)
        __syncwarp(full);
        if (act) src[0][l] = F.loc[(size_t)P * F.p1 + l];
        __syncwarp(full);
        if (row) {
            const int q = (ix & 1) + 2 * (iy & 1);
            const double2 *zp = F.tab + (size_t)(TAB_L2L + q) * ML_P1MAX;
            double2 t = make_double2(0.0, 0.0);
            for (int k = l; k <= p; ++k) {
                const double bc = F.binom[(size_t)k * BN + l];
                const double2 u = cmul(src[0][k], zp[k - l]);
                t.x = fma(bc, u.x, t.x); t.y = fma(bc, u.y, t.y);
            }
            acc = cscale(t, scalbn(1.0, -l));
        }
        // ---- M2L (eq C5), DW_NP pairs per pass
        const int nm = F.m2l_cnt[node];
        for (int e0 = 0; e0 < nm; e0 += DW_NP) {
            const double2 *wp[DW_NP];
            __syncwarp(full);
#pragma unroll
            for (int q = 0; q < DW_NP; ++q) {
                double2 v = make_double2(0.0, 0.0);
                wp[q] = F.tab + (size_t)(TAB_M2L + 3 * 7 + 3) * ML_P1MAX;       // offset (0, 0): all zeros beyond n = 0
                if (e0 + q < nm) {
                    const int S = F.m2l_list[(size_t)node * 27 + e0 + q];
                    const int dx = F.ix[S] - ix, dy = F.iy[S] - iy;
                    wp[q] = F.tab + (size_t)(TAB_M2L + (dy + 3) * 7 + dx + 3) * ML_P1MAX;   // (-1/z0)^n
                    if (act) v = cmul(F.mp[(size_t)S * F.p1 + l], wp[q][l]);
                }
                src[q][l] = v;
            }
            __syncwarp(full);
            double2 t[DW_NP];
#pragma unroll
            for (int q = 0; q < DW_NP; ++q) t[q] = make_double2(-src[q][0].x * inv_l, 0.0);
#pragma unroll 2
            for (int k = 1; k <= p; ++k) {
                const double bc = Bt[(k - 1) * 32 + l];
#pragma unroll
                for (int q = 0; q < DW_NP; ++q) {
                    const double2 sv = src[q][k];
                    t[q].x = fma(bc, sv.x, t[q].x); t[q].y = fma(bc, sv.y, t[q].y);
                }
            }
            if (row) {
#pragma unroll
                for (int q = 0; q < DW_NP; ++q) {
                    if (e0 + q < nm) {
                        double2 zi = wp[q][l];                        // (1/z0)^l = (-1)^l (-1/z0)^l
                        if (l & 1) { zi.x = -zi.x; zi.y = -zi.y; }
                        const double2 u = cmul(t[q], zi);
                        acc.x += u.x; acc.y += u.y;
                    }
                }
            }
        }
        // ---- P2L (eq C6): stars of coarser childless nodes outside this node's 3x3 block
        const int np = F.p2l_cnt[node];
        if (np > 0 && row) {
            double cx, cy, half;
            node_geom(F, node, cx, cy, half);
            const int sh = ML_QBITS - lev;
            for (int e = 0; e < np; ++e) {
                const int Q = F.p2l_list[(size_t)node * 8 + e];
                const int lo = F.lo[Q], n = F.n[Q];
                for (int i = lo; i < lo + n; ++i) {
                    const int cxq = (int)(F.sqx[i] >> sh), cyq = (int)(F.sqy[i] >> sh);
                    if (abs(cxq - ix) <= 1 && abs(cyq - iy) <= 1) continue;
                    const double2 zeta = make_double2((F.sx[i] - cx) / half, (F.sy[i] - cy) / half);
                    const double2 w = cpowi(cinv(zeta), l);
                    const double f = -F.sm[i] * inv_l;
                    acc.x = fma(f, w.x, acc.x); acc.y = fma(f, w.y, acc.y);
                }
            }
        }
        if (act) F.loc[(size_t)node * F.p1 + l] = row ? acc : make_double2(0.0, 0.0);
    }
}

// e_l = (l+1) c_{l+1} theta^2 / L for l < p: the derivative series of eq C4 the evaluator sums (eq 24)
__global__ void leaf_coef_kernel(FmmDev F, int n_leaves) {
    int leaf = blockIdx.x, l = threadIdx.x;
    if (leaf >= n_leaves || l > F.p) return;
    int node = F.leaf_node[leaf];
    double half = F.root_half / (double)(1 << F.level[node]);
    double2 v = make_double2(0.0, 0.0);
    if (l < F.p) v = cscale(F.loc[(size_t)node * F.p1 + l + 1], (double)(l + 1) * F.theta2 / half);
    F.ecoef[(size_t)leaf * F.p1 + l] = v;
}

// Rectangle sheet inside the star rectangle (eq B8):  alpha_s = -kappa_star z + conj A(z),
//   A(z) = (kappa_star i/pi) G(z) - kappa_star (2 c1 + z),   G(z) = sum_i s_i (a_i - z) log(a_i - z),
// a_i = conj c, c, -conj c, -c and s_i = +1, -1, +1, -1: analytic in the open rectangle (the logarithms' cuts lie on its
// upper and lower edges).  Its Taylor series about a leaf's centre z_c, in the leaf's variable zeta = (z - z_c)/L, is
//   T_0 = A(z_c),  T_1 = A'(z_c) L  with G' = -sum s_i log(a_i - z),
//   T_l = (kappa_star i/pi) sum_i s_i d_i w_i^l / (l (l-1)),  d_i = a_i - z_c,  w_i = L/d_i        (l >= 2)
// and is ADDED to a copy of the leaf's derivative series (which sums to conj alpha_far): the shooting kernels' tiles shift
// that copy to their centres and never see a logarithm.  A leaf whose square is not inside the rectangle, or so close to a
// corner that the series converges slower than 0.4^l, keeps the plain series (flag 0): its tiles evaluate eq B7.
// So does a leaf where the series, cut at the field's order p, would leave more than `rem_budget` of the sheet's
// deflection behind: with r_i = sqrt2 L/|d_i| the four tails are bounded by
//   sum_i (kappa_star/pi) |d_i| r_i^p / (p (p-1) (1 - r_i)),
// which matters when the caller fixed a low order (~1e-4 theta at p = 8 next to a corner).
__global__ void rect_fold_kernel(FmmDev F, int n_leaves, double c1, double c2, double kappa_star, double rem_budget,
                                 double2 *ecoef_shoot, unsigned char *leaf_fold) {
    const int leaf = blockIdx.x, l = threadIdx.x;
    if (leaf >= n_leaves) return;
    const int node = F.leaf_node[leaf];
    const double half = F.root_half / (double)(1 << F.level[node]);
    const double cx = -F.root_half + (2.0 * F.ix[node] + 1.0) * half, cy = -F.root_half + (2.0 * F.iy[node] + 1.0) * half;
    const double ks_pi = kappa_star * 0.31830988618379067154;
    bool ok = fabs(cx) + half <= c1 && fabs(cy) + half <= c2 && F.p >= 2;
    double rem = 0.0;
#pragma unroll 1
    for (int i = 0; i < 4; ++i) {                                                                // the verdict first: the same for every l
        const double dx = ((i < 2) ? c1 : -c1) - cx, dy = ((i == 0 || i == 3) ? -c2 : c2) - cy;
        const double d2 = dx * dx + dy * dy;
        if (!(2.0 * half * half < 0.16 * d2)) { ok = false; continue; }                          // (sqrt2 L / |d|)^2 < 0.4^2
        const double r = sqrt(2.0 * half * half / d2);
        rem += ks_pi * sqrt(d2) * pow(r, (double)F.p) / ((double)F.p * (double)(F.p - 1) * (1.0 - r));
    }
    if (!(rem <= rem_budget)) ok = false;
    double2 T = make_double2(0.0, 0.0);
#pragma unroll 1
    for (int i = 0; i < 4; ++i) {
        const double sg = (i & 1) ? -1.0 : 1.0;
        const double ax = (i < 2) ? c1 : -c1, ay = (i == 0 || i == 3) ? -c2 : c2;             // conj c, c, -conj c, -c
        const double2 d = make_double2(ax - cx, ay - cy);
        const double d2 = d.x * d.x + d.y * d.y;
        if (!ok || l >= F.p) continue;
        if (l == 0) {
            const double lg = 0.5 * log(d2), ar = atan2(d.y, d.x);
            T.x += sg * (d.x * lg - d.y * ar); T.y += sg * (d.x * ar + d.y * lg);
        } else if (l == 1) {
            T.x -= sg * 0.5 * log(d2) * half; T.y -= sg * atan2(d.y, d.x) * half;
        } else {
            const double2 w = make_double2(half * d.x / d2, -half * d.y / d2);
            const double2 t = cmul(d, cpowi(w, l));
            const double f = sg / (double)(l * (l - 1));
            T.x += f * t.x; T.y += f * t.y;
        }
    }
    T = make_double2(-ks_pi * T.y, ks_pi * T.x);
    if (l == 0) { T.x -= kappa_star * (2.0 * c1 + cx); T.y -= kappa_star * cy; }
    if (l == 1) T.x -= kappa_star * half;
    if (l <= F.p) {
        double2 e = F.ecoef[(size_t)leaf * F.p1 + l];
        if (ok && l < F.p) { e.x += T.x; e.y += T.y; }
        ecoef_shoot[(size_t)leaf * F.p1 + l] = e;
    }
    if (l == 0) leaf_fold[leaf] = ok ? 1 : 0;
}

int rect_fold(mlens_field *f, cudaStream_t s) {
    Tree &t = f->tree;
    const int p = f->order, p1 = p + 1;
    const size_t nl = (size_t)t.n_leaves;
    if (!nl) return MLENS_OK;
    ML_TRY(t.ecoef_shoot.reserve(nl * p1, s, false));
    ML_TRY(t.leaf_fold.reserve(nl, s, false));
    FmmDev F{t.level.p, t.ix.p, t.iy.p, t.parent.p, t.child0.p, t.lo.p, t.n.p,
             t.m2l_cnt.p, t.m2l_list.p, t.p2l_cnt.p, t.p2l_list.p, t.leaf_node.p,
             f->sx.p, f->sy.p, f->sm.p, f->sqx.p, f->sqy.p, t.mp.p, t.loc.p, t.ecoef.p,
             f->binom.p, f->tab.p, f->root_half, f->theta * f->theta, p, p1};
    // a tenth of the field's accuracy target for the sheet's truncation (orders chosen from eq C9 stay far below it)
    ML_LAUNCH(rect_fold_kernel, (unsigned)nl, 64, 0, s, F, (int)nl, f->c1, f->c2, f->kappa_star, 0.1 * f->eps * f->theta,
              t.ecoef_shoot.p, t.leaf_fold.p);
    ML_CUDA(cudaGetLastError());
    return MLENS_OK;
}

int fmm_passes(mlens_field *f, cudaStream_t s) {
    Tree &t = f->tree;
    const int p = f->order, p1 = p + 1;
    const size_t nn = (size_t)t.n_nodes, nl = (size_t)t.n_leaves;
    ML_TRY(t.mp.reserve(nn * p1, s, false));
    ML_TRY(t.loc.reserve(nn * p1, s, false));
    ML_TRY(t.ecoef.reserve(nl * p1, s, false));
    ML_CUDA(cudaMemsetAsync(t.loc.p, 0, nn * p1 * sizeof(double2), s));
    FmmDev F{t.level.p, t.ix.p, t.iy.p, t.parent.p, t.child0.p, t.lo.p, t.n.p,
             t.m2l_cnt.p, t.m2l_list.p, t.p2l_cnt.p, t.p2l_list.p, t.leaf_node.p,
             f->sx.p, f->sy.p, f->sm.p, f->sqx.p, f->sqy.p, t.mp.p, t.loc.p, t.ecoef.p,
             f->binom.p, f->tab.p, f->root_half, f->theta * f->theta, p, p1};
    const int T = 64;   // >= ML_P1MAX
    static_assert(ML_P1MAX <= 64, "one thread per coefficient");
    ML_LAUNCH(p2m_kernel, (unsigned)nl, T, 0, s, F, (int)nl);
    for (int lev = t.n_levels - 2; lev >= 0; --lev) {
        int a = t.level_off[lev], b = t.level_off[lev + 1];
        ML_LAUNCH(m2m_kernel, b - a, T, 0, s, F, a, b);
    }
    for (int lev = 2; lev < t.n_levels; ++lev) {
        int a = t.level_off[lev], b = t.level_off[lev + 1];
        if (p <= DW_PMAX) {
            int nsm = 148;
            cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, f->device);
            const int want = (b - a + DW_WARPS - 1) / DW_WARPS, cap = nsm * 6;
            ML_LAUNCH(downward_warp_kernel, (want < cap) ? want : cap, DW_WARPS * 32, 0, s, F, a, b);
        } else {
            ML_LAUNCH(downward_kernel, b - a, T, 0, s, F, a, b);
        }
    }
    ML_LAUNCH(leaf_coef_kernel, (unsigned)nl, T, 0, s, F, (int)nl);
    ML_CUDA(cudaGetLastError());
    return MLENS_OK;
}

}  // namespace ml
