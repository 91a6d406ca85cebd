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

// What the iteration does after a lattice evaluation (reading C-14): done (QMC_OK), out of budget / lattices /
// shifts (QMC_ERR_MAXEVAL), or kContinue with the next lattice index li, shift count m and the shifts already sampled on that
// lattice (m_have > 0: an extension of the current lattice; 0: a fresh, larger lattice whose predecessors are discarded).
constexpr int kContinue = 1;
int next_step(const qmc_result* out, int nc, int n_lattices, const uint64_t* ladder_n, int min_m, int max_m, double epsrel, double epsabs,
              uint64_t maxeval, int errormode, int* li_io, int* m_io, int* m_have_io) {
    int li = *li_io, m = *m_io;
    double ratio;
    if (goal_met(out->integral, out->error, nc, epsrel, epsabs, errormode, &ratio)) return QMC_OK;
    if (out->evaluations >= maxeval) return QMC_ERR_MAXEVAL;
    const uint64_t budget = maxeval - out->evaluations;
    if (li + 1 < n_lattices) {
        // larger lattice: smallest ladder n >= n * max(2, err/goal), limited by what maxeval still allows: a lattice
        // whose min_m samples do not fit the remaining budget is not tried
        const double want = (double)ladder_n[li] * std::fmax(2.0, std::isfinite(ratio) ? ratio : 2.0);
        int nx = li + 1;
        while (nx + 1 < n_lattices && (double)ladder_n[nx] < want) ++nx;
        while (nx > li && (uint64_t)min_m * ladder_n[nx] > budget) --nx;
        if (nx > li) {
            *li_io = nx; *m_io = min_m; *m_have_io = 0;             // earlier results are discarded
            return kContinue;
        }
    }
    // ladder exhausted (or no larger lattice affordable): add shifts on the current lattice, Monte Carlo scaling err ~ m^-1/2
    if (m >= max_m) return QMC_ERR_MAXEVAL;
    double grow = std::isfinite(ratio) ? ratio * ratio : 2.0;
    long long m_next = (long long)std::ceil((double)m * std::fmin(std::fmax(grow, 1.25), 4.0));
    m_next = std::max<long long>(m_next, m + 2);                    // an extension samples at least two shifts
    const long long afford = (long long)(budget / ladder_n[li]);
    if (afford < 2) return QMC_ERR_MAXEVAL;
    m_next = std::min<long long>(std::min<long long>(m_next, m + afford), max_m);
    if (m_next - m < 2) { if (max_m - m >= 2) m_next = m + 2; else return QMC_ERR_MAXEVAL; }
    *m_have_io = m;
    *m_io = (int)m_next;
    return kContinue;
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
        const int next = next_step(out, nc, n_lattices, ladder_n, min_m, max_m, epsrel, epsabs, maxeval, errormode, &li, &m, &m_have);
        if (next != kContinue) return next;
    }
}

// ---- the iteration for MANY integrands at once ------------------------------------------------------------------------------
// Every integrand runs the iteration of qmc_integrate (the same next_step), but the lattice evaluations of one round -- each
// integrand on its own current lattice and shift range -- share ONE batched launch of the fused kernels (S9: tiles of unequal
// cost in one persistent grid).  With a module the sectors run as compiled code.  One device-to-host copy and one
// synchronisation per round instead of one per integrand and iteration.
namespace {

struct IntegrandState {
    int li = 0, m = 0, m_have = 0;
    bool active = true;
};

}  // namespace

extern "C" int qmc_integrate_batch(int count, const qmc_integrand* integrands, qmc_sector_module* module, int n_lattices,
                                   const uint64_t* ladder_n, const uint64_t* ladder_z, int ladder_dim, const double* shifts, uint64_t min_n,
                                   int min_m, int max_m, double epsrel, double epsabs, uint64_t maxeval, int errormode, qmc_result* out,
                                   int* out_status) {
    if (!integrands || !ladder_n || !ladder_z || !shifts || !out || !out_status) return QMC_ERR_NULL;
    if (count < 1 || n_lattices < 1) return QMC_ERR_N;
    if (ladder_dim < 1 || ladder_dim > QMC_MAX_DIM) return QMC_ERR_DIM;
    if (min_m < 2 || max_m < min_m || max_m > QMC_MAX_M) return QMC_ERR_M;
    if (!(epsrel >= 0.0) || !(epsabs >= 0.0) || errormode < 0 || errormode > 1) return QMC_ERR_PARAMS;
    for (int i = 1; i < n_lattices; ++i)
        if (ladder_n[i] <= ladder_n[i - 1]) return QMC_ERR_N;

    // host images: per distinct dimension d the ladder vectors [n_lattices][d] and the shifts [max_m][d] (the first d components
    // of the caller's ladder_dim-dimensional ones); per integrand its parameter block and fit map
    int dim_slot[QMC_MAX_DIM + 1];
    for (int d = 0; d <= QMC_MAX_DIM; ++d) dim_slot[d] = -1;
    std::vector<int> dims;
    std::vector<int> ncs(count);
    for (int p = 0; p < count; ++p) {
        const qmc_integrand& g = integrands[p];
        if (!g.params) return QMC_ERR_NULL;
        ncs[p] = qmc_num_components(g.family);
        if (ncs[p] < 0) return QMC_ERR_FAMILY;
        if (g.dim < 1 || g.dim > ladder_dim) return QMC_ERR_DIM;
        if (g.n_params < 1) return QMC_ERR_PARAMS;
        if (dim_slot[g.dim] < 0) { dim_slot[g.dim] = (int)dims.size(); dims.push_back(g.dim); }
    }
    std::vector<size_t> off_z(dims.size()), off_sh(dims.size()), off_params(count), off_fit(count);
    std::vector<char> blob;
    auto reserve = [&](size_t bytes) { const size_t at = blob.size(); blob.resize(at + up256(bytes)); return at; };
    for (size_t k = 0; k < dims.size(); ++k) {
        const int d = dims[k];
        off_z[k] = reserve((size_t)n_lattices * d * 8);
        off_sh[k] = reserve((size_t)max_m * d * 8);
    }
    for (int p = 0; p < count; ++p) {
        off_params[p] = reserve((size_t)integrands[p].n_params * 8);
        off_fit[p] = integrands[p].fit_coeffs ? reserve((size_t)integrands[p].dim * 6 * 8) : 0;
    }
    for (size_t k = 0; k < dims.size(); ++k) {                     // every reserve is done: blob.data() is stable from here on
        const int d = dims[k];
        uint64_t* hz = reinterpret_cast<uint64_t*>(blob.data() + off_z[k]);
        double* hs = reinterpret_cast<double*>(blob.data() + off_sh[k]);
        for (int l = 0; l < n_lattices; ++l)
            for (int j = 0; j < d; ++j) hz[(size_t)l * d + j] = ladder_z[(size_t)l * ladder_dim + j];
        for (int s = 0; s < max_m; ++s)
            for (int j = 0; j < d; ++j) hs[(size_t)s * d + j] = shifts[(size_t)s * ladder_dim + j];
    }
    for (int p = 0; p < count; ++p) {
        std::memcpy(blob.data() + off_params[p], integrands[p].params, (size_t)integrands[p].n_params * 8);
        if (integrands[p].fit_coeffs) std::memcpy(blob.data() + off_fit[p], integrands[p].fit_coeffs, (size_t)integrands[p].dim * 6 * 8);
    }
    // full value validation of every integrand on every lattice, on the host images, before anything is launched
    for (int p = 0; p < count; ++p) {
        const qmc_integrand& g = integrands[p];
        const int k = dim_slot[g.dim];
        qmc_problem hp;
        hp.family = g.family; hp.dim = g.dim; hp.m = max_m; hp.transform = g.transform; hp.n_params = g.n_params;
        hp.params = reinterpret_cast<const double*>(blob.data() + off_params[p]);
        hp.shifts = reinterpret_cast<const double*>(blob.data() + off_sh[k]);
        hp.fit_coeffs = g.fit_coeffs ? reinterpret_cast<const double*>(blob.data() + off_fit[p]) : nullptr;
        for (int l = 0; l < n_lattices; ++l) {
            hp.n = ladder_n[l];
            hp.z = reinterpret_cast<const uint64_t*>(blob.data() + off_z[k]) + (size_t)l * g.dim;
            const int st = qmc_validate_problem_host(&hp);
            if (st != QMC_OK) return st;
        }
    }

    cudaStream_t st = 0;
    // device block: [inputs | shift means: rows 2p (all shifts of integrand p's current lattice) and 2p + 1 (an extension's new
    // shifts), stride 2 max_m | means, errors: rows as the shift means, 2 doubles each]
    const int stride = 2 * max_m;
    const size_t b_in = blob.size(), b_sm = up256((size_t)2 * count * stride * 8), b_res = up256((size_t)2 * count * 2 * 8);
    DeviceBlock blk;
    blk.st = st;
    ADAPT_CUDA(cudaMallocAsync(reinterpret_cast<void**>(&blk.p), b_in + b_sm + 2 * b_res, st));
    char* d_in = blk.p;
    double* d_sm = reinterpret_cast<double*>(d_in + b_in);
    double* d_means = reinterpret_cast<double*>(d_in + b_in + b_sm);
    double* d_errs = reinterpret_cast<double*>(d_in + b_in + b_sm + b_res);
    ADAPT_CUDA(cudaMemcpyAsync(d_in, blob.data(), b_in, cudaMemcpyHostToDevice, st));
    DeviceBlock ws;                                                   // the batch workspace, grown when a round needs more
    ws.st = st;
    size_t ws_bytes = 0;

    std::vector<IntegrandState> state(count);
    for (int p = 0; p < count; ++p) {
        std::memset(&out[p], 0, sizeof(qmc_result));
        out_status[p] = QMC_ERR_MAXEVAL;
        int li = 0;                                                   // smallest ladder lattice with n >= min_n
        while (li + 1 < n_lattices && ladder_n[li] < min_n) ++li;
        state[p].li = li; state[p].m = min_m; state[p].m_have = 0;
    }
    std::vector<qmc_problem> batch;
    std::vector<int> who, rows, in_module;
    std::vector<double> h_res((size_t)2 * count * 2 * 2);
    for (;;) {
        batch.clear(); who.clear(); rows.clear(); in_module.clear();
        for (int p = 0; p < count; ++p) {
            if (!state[p].active) continue;
            const qmc_integrand& g = integrands[p];
            const IntegrandState& s = state[p];
            const int k = dim_slot[g.dim];
            qmc_problem dp;
            dp.family = g.family; dp.dim = g.dim; dp.transform = g.transform; dp.n_params = g.n_params;
            dp.n = ladder_n[s.li];
            dp.m = s.m - s.m_have;                                    // shifts [m_have, m) of lattice li
            dp.params = reinterpret_cast<const double*>(d_in + off_params[p]);
            dp.z = reinterpret_cast<const uint64_t*>(d_in + off_z[k]) + (size_t)s.li * g.dim;
            dp.shifts = reinterpret_cast<const double*>(d_in + off_sh[k]) + (size_t)s.m_have * g.dim;
            dp.fit_coeffs = g.fit_coeffs ? reinterpret_cast<const double*>(d_in + off_fit[p]) : nullptr;
            batch.push_back(dp);
            who.push_back(p);
            rows.push_back(2 * p + (s.m_have > 0 ? 1 : 0));
            in_module.push_back(p);
        }
        if (batch.empty()) break;
        const int nb = (int)batch.size();
        const size_t need = qmc::routed_workspace_bytes(nb, batch.data(), module, module ? in_module.data() : nullptr);
        if (need == 0) return QMC_ERR_WORKSPACE;
        if (need > ws_bytes) {
            if (ws.p) { ADAPT_CUDA(cudaFreeAsync(ws.p, st)); ws.p = nullptr; }
            ws_bytes = need + need / 2;
            ADAPT_CUDA(cudaMallocAsync(reinterpret_cast<void**>(&ws.p), ws_bytes, st));
        }
        int rc = qmc::run_batch_routed(nb, batch.data(), d_means, d_errs, d_sm, ws.p, ws_bytes, st, module, module ? in_module.data() : nullptr,
                                       rows.data(), stride);
        if (rc != QMC_OK) return rc;
        for (int i = 0; i < nb; ++i) {                                // extensions: append the new means, redo Eq. 2-3 over all shifts
            const int p = who[i];
            const IntegrandState& s = state[p];
            if (s.m_have == 0) continue;
            double* all = d_sm + (size_t)(2 * p) * stride;
            ADAPT_CUDA(cudaMemcpyAsync(all + (size_t)s.m_have * ncs[p], d_sm + (size_t)(2 * p + 1) * stride,
                                       (size_t)(s.m - s.m_have) * ncs[p] * 8, cudaMemcpyDeviceToDevice, st));
            rc = qmc_finalize_means(all, s.m, ncs[p], d_means + (size_t)(2 * p) * 2, d_errs + (size_t)(2 * p) * 2, st);
            if (rc != QMC_OK) return rc;
        }
        ADAPT_CUDA(cudaMemcpyAsync(h_res.data(), d_means, (size_t)2 * count * 2 * 8, cudaMemcpyDeviceToHost, st));
        ADAPT_CUDA(cudaMemcpyAsync(h_res.data() + (size_t)2 * count * 2, d_errs, (size_t)2 * count * 2 * 8, cudaMemcpyDeviceToHost, st));
        ADAPT_CUDA(cudaStreamSynchronize(st));
        for (int i = 0; i < nb; ++i) {
            const int p = who[i], nc = ncs[p];
            IntegrandState& s = state[p];
            qmc_result& r = out[p];
            const double* mean = h_res.data() + (size_t)(2 * p) * 2;
            const double* err = h_res.data() + (size_t)2 * count * 2 + (size_t)(2 * p) * 2;
            r.iterations += 1;
            r.evaluations += (uint64_t)(s.m - s.m_have) * ladder_n[s.li];
            r.n = ladder_n[s.li];
            r.m = s.m;
            bool finite = true;
            for (int c = 0; c < 2; ++c) {
                r.integral[c] = c < nc ? mean[c] : 0.0;
                r.error[c] = c < nc ? err[c] : 0.0;
                if (c < nc) finite = finite && std::isfinite(mean[c]) && std::isfinite(err[c]);
            }
            if (!finite) { s.active = false; out_status[p] = QMC_ERR_NONFINITE; continue; }
            const int next = next_step(&r, nc, n_lattices, ladder_n, min_m, max_m, epsrel, epsabs, maxeval, errormode, &s.li, &s.m, &s.m_have);
            if (next != kContinue) { s.active = false; out_status[p] = next; }
        }
    }
    int worst = QMC_OK;
    for (int p = 0; p < count; ++p)
        if (out_status[p] != QMC_OK && (worst == QMC_OK || out_status[p] == QMC_ERR_NONFINITE)) worst = out_status[p];
    return worst;
}
