// qmc_project.cu -- S10, the projection pass that feeds the variance-reduction fit
// (Eq. 20; the paper's `evaluate`, keeps all n samples on the host and
// sorts them per dimension, P:L958-L960 -- here replaced by a device histogram, C-8):
//
//     H[j][b] = sum_k |f(x_k)| [ floor(B x_{k,j}) == b ],   x_k = { k z / n + Delta_0 },
//
// transform None, weight 1, first shift only, all n lattice points.
//
// Determinism: a tile is a fixed range of lattice indices; inside a tile every warp owns a private
// shared-memory histogram.  Per step the 32 lanes evaluate their points and stage (x, |f|) in shared
// memory; then lane L adds the 32 staged points, in lane order, to the histogram row of dimension L:
// rows are private to a lane, so there is no conflict to resolve and no floating-point atomic (round 1
// resolved same-bin lanes with __match_any_sync and a vote loop per dimension: 10 times slower).  Warp
// histograms are merged in warp order, tile histograms in tile order (compensated) by
// project_merge_kernel.  The result does not depend on the grid size, the SM count or the scheduling order.
#include <algorithm>
#include <cmath>
#include <cstring>

#include "qmc_device.cuh"
#include "qmc_kernels.h"

namespace qmc {
namespace {

constexpr int kProjTilesTarget = 148;       // one tile per SM of a B200: fixed, so the tiling is a function of n only
constexpr int kProjSmemBudget = 200 * 1024; // bytes of warp-private histograms per CTA

struct ProjArgs {
    const double* params;
    const unsigned long long* z;
    const double* shift;        // first shift, dim entries
    unsigned long long n;
    double inv_n;
    int family, dim, n_params, bins;
    int steps;                  // lattice indices per thread per tile
    int tiles;
    int dchunk;                 // dimensions histogrammed per CTA
    int nchunks;
    double* tile_hist;          // [tile][dim][bins]
    double* out_hist;           // [dim][bins]
};

// |f(x)| for the four families, straight from the caller's parameter block (layouts: qmc_lattice.h).
__device__ double abs_integrand(const ProjArgs& a, const double* x) {
    const double* p = a.params;
    const int d = a.dim;
    if (a.family == QMC_FAMILY_GENZ_OSC) {
        double ph = __dmul_rn(6.283185307179586476925286766559, p[0]);
        for (int j = 0; j < d; ++j) ph = __fma_rn(p[1 + j], x[j], ph);
        return fabs(cos(ph));
    }
    if (a.family == QMC_FAMILY_GENZ_PRODPEAK) {
        double den = 1.0;
        for (int j = 0; j < d; ++j) {
            const double c = p[j], t = x[j] - p[d + j];
            den *= __fma_rn(t, t, 1.0 / (c * c));
        }
        return fabs(1.0 / den);
    }
    if (a.family == QMC_FAMILY_CEXP_POLY) {                                  // |exp(i phase)| = 1
        double pr = 1.0;
        for (int j = 0; j < d; ++j) pr *= __fma_rn(p[d + j], x[j], 1.0);
        return fabs(pr);
    }
    if (a.family == QMC_FAMILY_GENZ_CORNER) {
        double b = 1.0;
        for (int j = 0; j < d; ++j) b = __fma_rn(p[j], x[j], b);
        return fabs(1.0 / ipow_small(b, d + 1));
    }
    if (a.family == QMC_FAMILY_GENZ_GAUSSIAN || a.family == QMC_FAMILY_GENZ_C0) {
        double e = 0.0;
        for (int j = 0; j < d; ++j) {
            const double t = x[j] - p[d + j];
            e += (a.family == QMC_FAMILY_GENZ_GAUSSIAN) ? p[j] * p[j] * t * t : p[j] * fabs(t);
        }
        return exp(-e);
    }
    if (a.family == QMC_FAMILY_GENZ_DISCONT) {
        double e = 0.0;
        bool zero = false;
        for (int j = 0; j < d; ++j) { e = __fma_rn(p[j], x[j], e); zero = zero || (j < 2 && x[j] > p[d + j]); }
        return zero ? 0.0 : exp(e);
    }
    const int pa = (int)p[0], pb = (int)p[1], nU = (int)p[2], nF = (int)p[3];
    double pre = 1.0;
    for (int j = 0; j < d; ++j) pre *= ipow_small(x[j], (int)p[4 + j]);
    const double* base = p + 4 + d;
    if (a.family == QMC_FAMILY_SECTOR_COMPLEX) {                             // |f| = pre |U|^a / |F|^b (|Log| factor: modulus of the power)
        double re[2], im[2];
        const int cnt2[2] = {nU, nF};
        for (int w = 0; w < 2; ++w) {
            const double* cr = base;
            const double* ci = base + cnt2[w];
            const double* e = base + 2 * cnt2[w];
            double sr = 0.0, si = 0.0;
            for (int t = 0; t < cnt2[w]; ++t) {
                double mon = 1.0;
                for (int j = 0; j < d; ++j) mon *= ipow_small(x[j], (int)e[t * d + j]);
                sr = __fma_rn(cr[t], mon, sr); si = __fma_rn(ci[t], mon, si);
            }
            re[w] = sr; im[w] = si;
            base += cnt2[w] * (2 + d);
        }
        const double mu = sqrt(re[0] * re[0] + im[0] * im[0]), mf = sqrt(re[1] * re[1] + im[1] * im[1]);
        double f = pre * ipow_small(mu, pa) / ipow_small(mf, pb);
        if (a.n_params == 4 + d + (nU + nF) * (2 + d) + 3) {
            const double* t = p + a.n_params - 3;
            const double Lr = t[0] * log(mu) + t[1] * log(mf), Li = t[0] * atan2(im[0], re[0]) + t[1] * atan2(im[1], re[1]);
            f *= ipow_small(sqrt(Lr * Lr + Li * Li), (int)t[2]);
        }
        return fabs(f);
    }
    double poly[2];
    const int cnt[2] = {nU, nF};
    for (int w = 0; w < 2; ++w) {
        const double* c = base;
        const double* e = base + cnt[w];
        double s = 0.0;
        for (int t = 0; t < cnt[w]; ++t) {
            double mon = c[t];
            for (int j = 0; j < d; ++j) mon *= ipow_small(x[j], (int)e[t * d + j]);
            s += mon;
        }
        poly[w] = s;
        base += cnt[w] * (1 + d);
    }
    double f = pre * ipow_small(poly[0], pa) / ipow_small(poly[1], pb);
    if (a.n_params == 4 + d + (nU + nF) * (1 + d) + 3) {                     // trailing [lu, lf, p]: log factors of the sector family
        const double* t = p + a.n_params - 3;
        f *= ipow_small(t[0] * log(poly[0]) + t[1] * log(poly[1]), (int)t[2]);
    }
    return fabs(f);
}

template <bool WIDE>
__global__ void __launch_bounds__(kThreads) project_kernel(ProjArgs a) {   // a: by value, a.params is redirected to shared memory
    typedef typename Res<WIDE>::T RT;
    extern __shared__ double hist[];                    // [warp][dchunk][bins], then the parameter block
    __shared__ int block_status;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x / a.nchunks, chunk = blockIdx.x - tile * a.nchunks;
    const int j0 = chunk * a.dchunk, j1 = min(a.dim, j0 + a.dchunk);
    const int hsize = a.dchunk * a.bins;
    for (int i = tid; i < kWarps * hsize; i += kThreads) hist[i] = 0.0;
    // the parameter block is read from shared memory in the point loop; a sector block is validated first (on the device:
    // the host sees only the struct) -- a block that fails is never interpreted and the histograms become NaN
    double* sp = hist + kWarps * hsize;
    for (int i = tid; i < a.n_params; i += kThreads) sp[i] = a.params[i];
    if (tid == 0) block_status = is_sector_family(a.family) ? sector_block_status(a.params, a.n_params, a.dim, a.family == QMC_FAMILY_SECTOR_COMPLEX) : 0;
    __syncthreads();
    a.params = sp;
    if (block_status != 0) {
        for (int i = tid; i < (j1 - j0) * a.bins; i += kThreads) a.tile_hist[((size_t)tile * a.dim + j0) * a.bins + i] = nan("");
        return;
    }
    double* mine = hist + warp * hsize;
    double* stage = sp + ((a.n_params + 1) & ~1) + (size_t)warp * 32 * (QMC_MAX_DIM + 1);   // [point of the warp][x_0 .. x_(dim-1), |f|]

    const unsigned long long n = a.n;
    const unsigned long long tile_len = (unsigned long long)a.steps * kThreads;
    const unsigned long long k0 = (unsigned long long)tile * tile_len;
    const unsigned long long kend = (k0 + tile_len < n) ? k0 + tile_len : n;
    RT r[QMC_MAX_DIM], step[QMC_MAX_DIM];
    double x[QMC_MAX_DIM];
    for (int j = 0; j < a.dim; ++j) {
        const unsigned long long z = a.z[j] % n;
        r[j] = (RT)mulmod_u64((k0 + tid) % n, z, n);
        step[j] = (RT)mulmod_u64((unsigned long long)kThreads % n, z, n);
    }
    unsigned long long k = k0 + tid;
    const int row = QMC_MAX_DIM + 1;
    for (int i = 0; i < a.steps; ++i, k += kThreads) {
        // every lane evaluates its point and stages (x, |f|); a dead lane (beyond the lattice) stages |f| = -1
        const bool live = k < kend;
        double v = -1.0;
        if (live) {
            for (int j = 0; j < a.dim; ++j) x[j] = wrap_u(coord_t(Res<WIDE>::to_double(r[j]), a.inv_n, a.shift[j]));
            v = abs_integrand(a, x);
            for (int j = j0; j < j1; ++j) stage[lane * row + j] = x[j];
        }
        stage[lane * row + QMC_MAX_DIM] = v;
        __syncwarp();
        // lane L < (j1 - j0) owns dimension j0 + L of the warp's private histogram and adds the 32 points in lane order: no two
        // lanes touch the same row, so there is nothing to resolve and the order of the additions is fixed
        const int j = j0 + lane;
        if (j < j1) {
            double* hrow = mine + (size_t)lane * a.bins;
            const double fb = (double)a.bins;
#pragma unroll 4
            for (int p = 0; p < 32; ++p) {
                const double pv = stage[p * row + QMC_MAX_DIM];
                if (pv >= 0.0) {
                    int b = (int)floor(fb * stage[p * row + j]);
                    if (b >= a.bins) b = a.bins - 1;
                    hrow[b] += pv;
                }
            }
        }
        __syncwarp();
        for (int j = 0; j < a.dim; ++j) r[j] = add_mod<RT>(r[j], step[j], (RT)n);
    }
    __syncthreads();
    // merge the warp histograms in warp order and publish the tile's histogram
    for (int i = tid; i < (j1 - j0) * a.bins; i += kThreads) {
        double s = hist[i];
#pragma unroll
        for (int w = 1; w < kWarps; ++w) s += hist[w * hsize + i];
        a.tile_hist[((size_t)tile * a.dim + j0) * a.bins + i] = s;
    }
}

__global__ void __launch_bounds__(256) project_merge_kernel(ProjArgs a) {
    const int cells = a.dim * a.bins;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < cells; i += gridDim.x * blockDim.x) {
        CompSum cs;
        for (int t = 0; t < a.tiles; ++t) cs.add(a.tile_hist[(size_t)t * cells + i]);
        a.out_hist[i] = cs.value();
    }
}

// ---------------------------------------------------------------------------------------------
// S10b: the paper's own CDF sampling (all samples sorted per dimension, every fitstepsize-th
// kept; reading C-8b) WITHOUT a sort.  In dimension j the coordinate of lattice index k is x = wrap(fma(r, 1/n, Delta_j)),
// r = k z_j mod n, and both branches of the wrap are increasing in r: sorted by x the samples come in the cyclic residue
// order r0, r0+1, ..., n-1, 0, ..., r0-1 with r0 the first residue that wraps.  The rank of sample k is therefore
// (r - r0) mod n: the samples are SCATTERED to their ranks, summed in buckets of `step` consecutive ranks and scanned.
// Fixed shapes (a function of n and step only): deterministic, no floating-point atomics.
//   cdf_eval_kernel     v[k] = |f(x_k)|
//   cdf_scatter_kernel  vs[j][rank_j(k)] = v[k]
//   cdf_scan_kernel     one CTA per dimension: bucket sums, block scan, total; writes x_t and CDF_t, t = 1..K
// ---------------------------------------------------------------------------------------------
struct CdfArgs {
    ProjArgs pa;                 // params, z, shift, n, inv_n, family, dim, n_params (bins unused)
    int step;                    // fitstepsize
    long long K;                 // kept points per dimension = n / step
    double* v;                   // [n]
    double* vs;                  // [dim][n]
    unsigned long long* r0;      // [dim] first residue whose coordinate wraps (n if none)
    double* out_x;               // [dim][K]
    double* out_cdf;             // [dim][K]
    int* status;                 // device flag: sector block invalid -> outputs NaN
};

// first residue r with fma(r, 1/n, delta) >= 1 (the sum is non-decreasing in r), n if there is none
__device__ unsigned long long first_wrapping_residue(unsigned long long n, double inv_n, double delta) {
    unsigned long long lo = 0, hi = n;                       // answer in [lo, hi]
    while (lo < hi) {
        const unsigned long long mid = lo + (hi - lo) / 2;
        if (ge_one(coord_t((double)mid, inv_n, delta))) hi = mid; else lo = mid + 1;
    }
    return lo;
}

__global__ void __launch_bounds__(256) cdf_eval_kernel(CdfArgs c) {
    extern __shared__ double sp[];                           // the parameter block
    __shared__ int block_status;
    ProjArgs a = c.pa;
    for (int i = threadIdx.x; i < a.n_params; i += blockDim.x) sp[i] = a.params[i];
    if (threadIdx.x == 0) block_status = is_sector_family(a.family) ? sector_block_status(a.params, a.n_params, a.dim, a.family == QMC_FAMILY_SECTOR_COMPLEX) : 0;
    __syncthreads();
    if (block_status != 0) { if (blockIdx.x == 0 && threadIdx.x == 0) *c.status = block_status; return; }
    if (blockIdx.x == 0 && threadIdx.x < a.dim) c.r0[threadIdx.x] = first_wrapping_residue(a.n, a.inv_n, a.shift[threadIdx.x]);
    a.params = sp;
    const unsigned long long n = a.n, stride = (unsigned long long)gridDim.x * blockDim.x;
    double x[QMC_MAX_DIM];
    for (unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += stride) {
        for (int j = 0; j < a.dim; ++j) x[j] = wrap_u(coord_t((double)mulmod_u64(k, a.z[j] % n, n), a.inv_n, a.shift[j]));
        c.v[k] = abs_integrand(a, x);
    }
}

__global__ void __launch_bounds__(256) cdf_scatter_kernel(CdfArgs c) {
    const unsigned long long n = c.pa.n, stride = (unsigned long long)gridDim.x * blockDim.x;
    const int j = blockIdx.y;
    const unsigned long long z = c.pa.z[j] % n, r0 = c.r0[j];
    double* vs = c.vs + (size_t)j * n;
    for (unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += stride) {
        const unsigned long long r = mulmod_u64(k, z, n);
        vs[r >= r0 ? r - r0 : r + (n - r0)] = c.v[k];
    }
}

constexpr int kCdfScanThreads = 1024;
__global__ void __launch_bounds__(kCdfScanThreads) cdf_scan_kernel(CdfArgs c) {
    __shared__ double part[kCdfScanThreads];
    const int j = blockIdx.x, tid = threadIdx.x;
    const unsigned long long n = c.pa.n;
    const long long K = c.K;
    const int step = c.step;
    double* ox = c.out_x + (size_t)j * K;
    double* oc = c.out_cdf + (size_t)j * K;
    if (*c.status != 0) {
        for (long long t = tid; t < K; t += kCdfScanThreads) { ox[t] = nan(""); oc[t] = nan(""); }
        return;
    }
    const double* vs = c.vs + (size_t)j * n;
    // thread `tid` owns the kept points t in [t0, t1): a contiguous chunk, the same split for every dimension
    const long long per = (K + kCdfScanThreads - 1) / kCdfScanThreads;
    const long long t0 = min(K, (long long)tid * per), t1 = min(K, t0 + per);
    double local = 0.0;
    for (long long t = t0; t < t1; ++t) {
        double b = 0.0;
        for (int i = 0; i < step; ++i) b += vs[(size_t)t * step + i];
        local += b;
    }
    // samples beyond the last kept point (fewer than step of them) belong to the total only: the last thread adds them
    double tail = 0.0;
    if (tid == kCdfScanThreads - 1)
        for (unsigned long long i = (unsigned long long)K * step; i < n; ++i) tail += vs[i];
    part[tid] = local;
    __syncthreads();
    // inclusive block scan (Hillis-Steele, fixed shape)
    for (int off = 1; off < kCdfScanThreads; off <<= 1) {
        const double add = tid >= off ? part[tid - off] : 0.0;
        __syncthreads();
        part[tid] += add;
        __syncthreads();
    }
    __shared__ double total;
    if (tid == kCdfScanThreads - 1) total = part[tid] + tail;
    __syncthreads();
    double run = part[tid] - local;                           // exclusive prefix of this thread's chunk
    const unsigned long long r0 = c.r0[j];
    const double delta = c.pa.shift[j];
    for (long long t = t0; t < t1; ++t) {
        double b = 0.0;
        for (int i = 0; i < step; ++i) b += vs[(size_t)t * step + i];
        run += b;
        const unsigned long long rank = (unsigned long long)t * step + (step - 1);
        const unsigned long long r = rank < n - r0 ? r0 + rank : rank - (n - r0);
        ox[t] = wrap_u(coord_t((double)r, c.pa.inv_n, delta));
        oc[t] = __ddiv_rn(run, total);
    }
}

int plan_project(const qmc_problem* p, int bins, ProjArgs* a) {
    if (!p) return QMC_ERR_NULL;
    if (p->family < 0 || p->family > QMC_FAMILY_SECTOR_COMPLEX) return QMC_ERR_FAMILY;
    if (p->dim < 1 || p->dim > QMC_MAX_DIM) return QMC_ERR_DIM;
    if (is_sector_family(p->family) && p->dim > QMC_MAX_SECTOR_DIM) return QMC_ERR_DIM;          // the same limits as the integration entries
    if (p->n < 2 || p->n >= (1ull << 53)) return QMC_ERR_N;
    if (bins < 2 || bins > 1024) return QMC_ERR_N;
    if (p->m < 1) return QMC_ERR_M;
    if (!p->params || !p->z || !p->shifts) return QMC_ERR_NULL;
    if (p->family == QMC_FAMILY_GENZ_OSC && p->n_params != 1 + p->dim) return QMC_ERR_PARAMS;
    if ((p->family == QMC_FAMILY_GENZ_PRODPEAK || p->family == QMC_FAMILY_CEXP_POLY) && p->n_params != 2 * p->dim) return QMC_ERR_PARAMS;
    if (p->family == QMC_FAMILY_GENZ_CORNER && p->n_params != p->dim) return QMC_ERR_PARAMS;
    if ((p->family == QMC_FAMILY_GENZ_GAUSSIAN || p->family == QMC_FAMILY_GENZ_C0) && p->n_params != 2 * p->dim) return QMC_ERR_PARAMS;
    if (p->family == QMC_FAMILY_GENZ_DISCONT && p->n_params != p->dim + (p->dim < 2 ? p->dim : 2)) return QMC_ERR_PARAMS;
    if (is_sector_family(p->family)) {                  // struct-level layout check as in qmc_host.cu; the values are checked on the device
        const int rest = p->n_params - 4 - p->dim, rec = sector_mono_stride(p->family, p->dim);
        const bool plain = rest % rec == 0, with_log = rest >= 3 && (rest - 3) % rec == 0;
        if (rest < 2 * rec || !(plain || with_log) || rest / rec > 2 * kMaxSectorMono) return QMC_ERR_PARAMS;
    }
    std::memset(a, 0, sizeof(*a));
    a->params = p->params;
    a->z = reinterpret_cast<const unsigned long long*>(p->z);
    a->shift = p->shifts;
    a->n = p->n;
    a->inv_n = 1.0 / (double)p->n;                                    // reading C-2
    a->family = p->family; a->dim = p->dim; a->n_params = p->n_params; a->bins = bins;
    const unsigned long long per = (unsigned long long)kThreads * kProjTilesTarget;
    const unsigned long long steps = std::max<unsigned long long>(1, (p->n + per - 1) / per);
    if (steps > 0x7fffffffull) return QMC_ERR_N;
    a->steps = (int)steps;
    a->tiles = (int)((p->n + steps * kThreads - 1) / (steps * kThreads));
    a->dchunk = std::max(1, std::min(std::min(p->dim, 32), (kProjSmemBudget - p->n_params * 8 - kWarps * 32 * (QMC_MAX_DIM + 1) * 8) / (kWarps * bins * 8)));   // <= 32: one lane per dimension of the chunk
    a->nchunks = (p->dim + a->dchunk - 1) / a->dchunk;
    return QMC_OK;
}

}  // namespace
}  // namespace qmc

using namespace qmc;

extern "C" size_t qmc_project_workspace_bytes(const qmc_problem* p, int bins) {
    ProjArgs a;
    if (plan_project(p, bins, &a) != QMC_OK) return 0;
    return ((size_t)a.tiles * a.dim * bins * 8 + 255) / 256 * 256;
}

extern "C" int qmc_lattice_project(const qmc_problem* p, int bins, double* out_hist, void* workspace, size_t workspace_bytes,
                                   void* cuda_stream) {
    ProjArgs a;
    const int st = plan_project(p, bins, &a);
    if (st != QMC_OK) return st;
    if (!out_hist) return QMC_ERR_NULL;
    const size_t need = ((size_t)a.tiles * a.dim * bins * 8 + 255) / 256 * 256;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need) return QMC_ERR_WORKSPACE;
    a.tile_hist = static_cast<double*>(workspace);
    a.out_hist = out_hist;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const size_t smem = (size_t)kWarps * a.dchunk * bins * 8 + (size_t)((a.n_params + 1) & ~1) * 8 + (size_t)kWarps * 32 * (QMC_MAX_DIM + 1) * 8;   // histograms, parameter block, staging
    const bool wide = p->n >= (1ull << 31);
    cudaError_t e;
    if (wide) {
        e = cudaFuncSetAttribute(project_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) project_kernel<true><<<a.tiles * a.nchunks, kThreads, smem, stream>>>(a);
    } else {
        e = cudaFuncSetAttribute(project_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) project_kernel<false><<<a.tiles * a.nchunks, kThreads, smem, stream>>>(a);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) {
        const int cells = a.dim * bins;
        project_merge_kernel<<<(cells + 255) / 256, 256, 0, stream>>>(a);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return report_cuda_error(e, "qmc_lattice_project");
    return QMC_OK;
}


// ---- sort-based CDF sampling (S10b) -----------------------------------------------------------------
namespace {
size_t cdf_layout(const qmc_problem* p, long long K, size_t* off_vs, size_t* off_r0, size_t* off_status) {
    size_t o = 0;
    o = ((size_t)p->n * 8 + 255) / 256 * 256;                // v
    *off_vs = o; o += ((size_t)p->dim * p->n * 8 + 255) / 256 * 256;
    *off_r0 = o; o += 256;
    *off_status = o; o += 256;
    (void)K;
    return o;
}
}  // namespace

extern "C" long long qmc_cdf_sample_count(uint64_t n, int fitstepsize) {
    if (fitstepsize < 1 || (uint64_t)fitstepsize > n) return 0;
    return (long long)(n / (uint64_t)fitstepsize);
}

extern "C" size_t qmc_cdf_workspace_bytes(const qmc_problem* p, int fitstepsize) {
    qmc::ProjArgs a;
    if (qmc::plan_project(p, 2, &a) != QMC_OK || qmc_cdf_sample_count(p->n, fitstepsize) == 0) return 0;
    size_t o1, o2, o3;
    return cdf_layout(p, 0, &o1, &o2, &o3);
}

extern "C" int qmc_lattice_cdf_samples(const qmc_problem* p, int fitstepsize, double* out_x, double* out_cdf, void* workspace,
                                       size_t workspace_bytes, void* cuda_stream) {
    qmc::ProjArgs a;
    const int st = qmc::plan_project(p, 2, &a);
    if (st != QMC_OK) return st;
    const long long K = qmc_cdf_sample_count(p->n, fitstepsize);
    if (K < 1) return QMC_ERR_N;
    if (!out_x || !out_cdf) return QMC_ERR_NULL;
    size_t off_vs, off_r0, off_status;
    const size_t need = cdf_layout(p, K, &off_vs, &off_r0, &off_status);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < need) return QMC_ERR_WORKSPACE;
    char* ws = static_cast<char*>(workspace);
    qmc::CdfArgs c;
    c.pa = a; c.step = fitstepsize; c.K = K;
    c.v = reinterpret_cast<double*>(ws);
    c.vs = reinterpret_cast<double*>(ws + off_vs);
    c.r0 = reinterpret_cast<unsigned long long*>(ws + off_r0);
    c.status = reinterpret_cast<int*>(ws + off_status);
    c.out_x = out_x; c.out_cdf = out_cdf;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t e = cudaMemsetAsync(c.status, 0, sizeof(int), stream);
    const int blocks = (int)std::min<unsigned long long>((p->n + 255) / 256, 148ull * 8);
    if (e == cudaSuccess) {
        qmc::cdf_eval_kernel<<<blocks, 256, (size_t)a.n_params * 8, stream>>>(c);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        qmc::cdf_scatter_kernel<<<dim3(blocks, p->dim), 256, 0, stream>>>(c);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        qmc::cdf_scan_kernel<<<p->dim, qmc::kCdfScanThreads, 0, stream>>>(c);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return qmc::report_cuda_error(e, "qmc_lattice_cdf_samples");
    return QMC_OK;
}
