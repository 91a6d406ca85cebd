// qmc_adaptive.cu -- the paper's `integrate` iteration (section 3.3.1) as a thin host loop around the
// stream-ordered hot path (qmc_lattice_integrate_batch + qmc_finalize_means).  SURVEY.md 8(f) row f-1.
// Every lattice evaluation runs in the fused kernels; this file only chooses the next lattice / shift count.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

#include <cuda_runtime.h>

#include "qmc_kernels.h"

namespace {

// CUDA failures are recorded for qmc_last_cuda_error() (qmc_host.cu)
#define ADAPT_CUDA(call)                                                        \
    do {                                                                        \
        cudaError_t e_ = (call);                                                \
        if (e_ != cudaSuccess) return qmc::report_cuda_error(e_, #call);        \
    } while (0)

struct DeviceBlock {              // one stream-ordered allocation, freed when the call returns
    char* p = nullptr;
    cudaStream_t st = 0;
    ~DeviceBlock() { if (p) cudaFreeAsync(p, st); }
};
inline size_t up256(size_t v) { return (v + 255) / 256 * 256; }

// error goal of P:L899 (real) and P:L915-L920 (complex: errormode all / largest)
bool goal_met(const double* mean, const double* err, int nc, double epsrel, double epsabs, int errormode, double* ratio) {
    double worst = 0.0;
    if (nc == 1 || errormode == 0) {
        for (int c = 0; c < nc; ++c) {
            const double goal = std::fmax(epsabs, epsrel * std::fabs(mean[c]));
            worst = std::fmax(worst, goal > 0.0 ? err[c] / goal : (err[c] > 0.0 ? INFINITY : 0.0));
        }
    } else {
        const double goal = std::fmax(epsabs, epsrel * std::fmax(std::fabs(mean[0]), std::fabs(mean[1])));
        const double e = std::fmax(err[0], err[1]);
        worst = goal > 0.0 ? e / goal : (e > 0.0 ? INFINITY : 0.0);
    }
    *ratio = worst;
    return worst <= 1.0;
}

}  // namespace

extern "C" int qmc_integrate(int family, const double* params, int n_params, int dim, int transform, const double* fit_coeffs,
                             int n_lattices, const uint64_t* ladder_n, const uint64_t* ladder_z, const double* shifts,
                             uint64_t min_n, int min_m, int max_m, double epsrel, double epsabs, uint64_t maxeval, int errormode,
                             qmc_result* out) {
    if (!params || !ladder_n || !ladder_z || !shifts || !out) return QMC_ERR_NULL;
    const int nc = qmc_num_components(family);
    if (nc < 0) return QMC_ERR_FAMILY;
    if (n_lattices < 1) return QMC_ERR_N;
    if (min_m < 2 || max_m < min_m || max_m > QMC_MAX_M) return QMC_ERR_M;
    if (!(epsrel >= 0.0) || !(epsabs >= 0.0) || errormode < 0 || errormode > 1) return QMC_ERR_PARAMS;
    for (int i = 1; i < n_lattices; ++i)
        if (ladder_n[i] <= ladder_n[i - 1]) return QMC_ERR_N;
    // full value validation of every lattice before anything is launched
    qmc_problem hp;
    hp.family = family; hp.dim = dim; hp.m = max_m; hp.transform = transform; hp.params = params; hp.n_params = n_params;
    hp.shifts = shifts; hp.fit_coeffs = fit_coeffs;
    size_t ws_bytes = 0;
    for (int i = 0; i < n_lattices; ++i) {
        hp.n = ladder_n[i]; hp.z = ladder_z + (size_t)i * dim;
        const int st = qmc_validate_problem_host(&hp);
        if (st != QMC_OK) return st;
        ws_bytes = std::max(ws_bytes, qmc_workspace_bytes(1, &hp));
    }

    cudaStream_t st = 0;
    const size_t b_params = up256((size_t)n_params * 8), b_z = up256((size_t)n_lattices * dim * 8),
                 b_sh = up256((size_t)max_m * dim * 8), b_fit = up256((size_t)dim * 6 * 8), b_sm = up256((size_t)max_m * 2 * 8),
                 b_out = 256;
    DeviceBlock blk;
    blk.st = st;
    ADAPT_CUDA(cudaMallocAsync(reinterpret_cast<void**>(&blk.p), b_params + b_z + b_sh + b_fit + 2 * b_sm + b_out + ws_bytes, st));
    char* d_params = blk.p;
    char* d_z = d_params + b_params;
    char* d_sh = d_z + b_z;
    char* d_fit = d_sh + b_sh;
    double* d_sm = reinterpret_cast<double*>(d_fit + b_fit);            // per-shift means of the current lattice, all shifts
    double* d_sm_new = reinterpret_cast<double*>(reinterpret_cast<char*>(d_sm) + b_sm);   // means of an extension
    double* d_out = reinterpret_cast<double*>(reinterpret_cast<char*>(d_sm_new) + b_sm);  // mean(2), err(2)
    char* d_ws = reinterpret_cast<char*>(d_out) + b_out;
    ADAPT_CUDA(cudaMemcpyAsync(d_params, params, (size_t)n_params * 8, cudaMemcpyHostToDevice, st));
    ADAPT_CUDA(cudaMemcpyAsync(d_z, ladder_z, (size_t)n_lattices * dim * 8, cudaMemcpyHostToDevice, st));
    ADAPT_CUDA(cudaMemcpyAsync(d_sh, shifts, (size_t)max_m * dim * 8, cudaMemcpyHostToDevice, st));
    if (fit_coeffs) ADAPT_CUDA(cudaMemcpyAsync(d_fit, fit_coeffs, (size_t)dim * 6 * 8, cudaMemcpyHostToDevice, st));

    qmc_problem dp = hp;
    dp.params = reinterpret_cast<const double*>(d_params);
    dp.fit_coeffs = fit_coeffs ? reinterpret_cast<const double*>(d_fit) : nullptr;

    std::memset(out, 0, sizeof(*out));
    int li = 0;                                                          // smallest ladder lattice with n >= min_n
    while (li + 1 < n_lattices && ladder_n[li] < min_n) ++li;
    int m = min_m, m_have = 0;                                           // m_have: shifts of lattice li already in d_sm
    double host_out[4];
    for (;;) {
        // sample shifts [m_have, m) of lattice li (a fresh lattice has m_have = 0)
        const int m_add = m - m_have;
        dp.n = ladder_n[li];
        dp.z = reinterpret_cast<const uint64_t*>(d_z) + (size_t)li * dim;
        dp.shifts = reinterpret_cast<const double*>(d_sh) + (size_t)m_have * dim;
        dp.m = m_add;
        double* sm_dst = m_have == 0 ? d_sm : d_sm_new;
        int rc = qmc_lattice_integrate_batch(1, &dp, d_out, d_out + 2, sm_dst, d_ws, ws_bytes, st);
        if (rc != QMC_OK) return rc;
        if (m_have > 0) {                                                // extension: append the new means, redo Eq. 2-3 over all
            ADAPT_CUDA(cudaMemcpyAsync(d_sm + (size_t)m_have * nc, d_sm_new, (size_t)m_add * nc * 8, cudaMemcpyDeviceToDevice, st));
            rc = qmc_finalize_means(d_sm, m, nc, d_out, d_out + 2, st);
            if (rc != QMC_OK) return rc;
        }
        ADAPT_CUDA(cudaMemcpyAsync(host_out, d_out, sizeof(host_out), cudaMemcpyDeviceToHost, st));
        ADAPT_CUDA(cudaStreamSynchronize(st));
        out->iterations += 1;
        out->evaluations += (uint64_t)m_add * ladder_n[li];
        out->n = ladder_n[li];
        out->m = m;
        for (int c = 0; c < 2; ++c) { out->integral[c] = c < nc ? host_out[c] : 0.0; out->error[c] = c < nc ? host_out[2 + c] : 0.0; }
        for (int c = 0; c < nc; ++c)
            if (!std::isfinite(host_out[c]) || !std::isfinite(host_out[2 + c])) return QMC_ERR_NONFINITE;
        double ratio;
        if (goal_met(out->integral, out->error, nc, epsrel, epsabs, errormode, &ratio)) return QMC_OK;
        if (out->evaluations >= maxeval) return QMC_ERR_MAXEVAL;
        const uint64_t budget = maxeval - out->evaluations;
        bool enlarged = false;
        if (li + 1 < n_lattices) {
            // larger lattice: smallest ladder n >= n * max(2, err/goal), limited by what maxeval still allows: a lattice
            // whose min_m samples do not fit the remaining budget is not tried
            const double want = (double)ladder_n[li] * std::fmax(2.0, std::isfinite(ratio) ? ratio : 2.0);
            int nx = li + 1;
            while (nx + 1 < n_lattices && (double)ladder_n[nx] < want) ++nx;
            while (nx > li && (uint64_t)min_m * ladder_n[nx] > budget) --nx;
            if (nx > li) {
                li = nx;
                m = min_m;
                m_have = 0;                                              // earlier results are discarded
                enlarged = true;
            }
        }
        if (!enlarged) {
            // ladder exhausted (or no larger lattice affordable): add shifts on the current lattice, Monte Carlo scaling err ~ m^-1/2
            if (m >= max_m) return QMC_ERR_MAXEVAL;
            double grow = std::isfinite(ratio) ? ratio * ratio : 2.0;
            long long m_next = (long long)std::ceil((double)m * std::fmin(std::fmax(grow, 1.25), 4.0));
            m_next = std::max<long long>(m_next, m + 2);                 // an extension samples at least two shifts
            const long long afford = (long long)(budget / ladder_n[li]);
            if (afford < 2) return QMC_ERR_MAXEVAL;
            m_next = std::min<long long>(std::min<long long>(m_next, m + afford), max_m);
            if (m_next - m < 2) { if (max_m - m >= 2) m_next = m + 2; else return QMC_ERR_MAXEVAL; }
            m_have = m;
            m = (int)m_next;
        }
    }
}
