// qmc_host.cu -- the C ABI of include/qmc_lattice.h: validation, launch planning, workspace layout
// and launches.  Every step of the hot path runs in the CUDA kernels; there is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>
#include <string>
#include <vector>

#include "qmc_fused.cuh"
#include "qmc_kernels.h"
#include "qmc_spec.h"

namespace qmc {
namespace {

// Per-thread measurement and staging state (include/qmc_lattice.h, "Conventions"): the text of the last CUDA error, the launch
// count of the last batch call, the profiling events (created on first use for the device that is current then) and the
// staging arena of the synchronous HOST-pointer entries.  Everything is released by qmc_release_thread_resources() and by
// the destructor at thread exit.
struct ThreadState {
    std::string last_error;
    int last_launches = 0;
    bool profile = false;                            // qmc_profile_enable
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    int ev_device = -1;
    bool ev_valid = false;
    // staging arena of the HOST-pointer entries: pinned host block + device block, grown on demand, bound to one device
    char* pinned = nullptr;
    char* device = nullptr;
    size_t pinned_bytes = 0, device_bytes = 0;
    int arena_device = -1;
    void release() {
        if (ev0) { cudaEventDestroy(ev0); cudaEventDestroy(ev1); ev0 = ev1 = nullptr; }
        ev_valid = false; ev_device = -1;
        if (pinned) { cudaFreeHost(pinned); pinned = nullptr; pinned_bytes = 0; }
        if (device) { cudaFree(device); device = nullptr; device_bytes = 0; }
        arena_device = -1;
    }
    ~ThreadState() { release(); }                    // errors (context already gone at process exit) are ignored
};
thread_local ThreadState g_ts;

int cuda_fail(cudaError_t e, const char* where) {
    g_ts.last_error = std::string(where) + ": " + cudaGetErrorString(e);
    return QMC_ERR_CUDA;
}
}  // namespace
// shared with the other translation units (qmc_kernels.h): records the text for qmc_last_cuda_error()
int report_cuda_error(cudaError_t e, const char* where) { return cuda_fail(e, where); }
namespace {
#define QMC_CUDA(call)                                              \
    do {                                                            \
        cudaError_t e_ = (call);                                    \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);         \
    } while (0)

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

int ncomp_of(int family) {
    if (family == QMC_FAMILY_CEXP_POLY || family == QMC_FAMILY_SECTOR_COMPLEX) return 2;
    if (family >= 0 && family <= QMC_FAMILY_GENZ_DISCONT) return 1;
    return -1;
}

// dimension slots of the kernel variant that serves (family, dim, residue width); slots beyond dim are padded
int dim_slots(int family, int dim, bool wide) {
    if (is_sector_family(family)) return dim <= 4 ? 4 : (dim <= 6 ? 6 : (dim <= 8 ? 8 : (dim <= 16 ? 16 : -1)));   // = sector_dim_slots (qmc_sector.cuh)
    if (wide) return dim <= 8 ? 8 : (dim <= 16 ? 16 : 32);
    return dim <= 4 ? 4 : (dim <= 6 ? 6 : (dim <= 8 ? 8 : (dim <= 12 ? 12 : (dim <= 16 ? 16 : 32))));
}
bool is_wide(unsigned long long n, const qmc_plan_options& o) { return n >= (1ull << 31) || o.force_wide != 0; }
// residue width of the kernel variant: 64-bit for n >= 2^31, and for the 32-slot closed-form kernels (dim > 16), which
// exist only with wide residues
bool variant_wide(int family, int dim, unsigned long long n, const qmc_plan_options& o) {
    return is_wide(n, o) || (!is_sector_family(family) && dim > 16);
}

// transform id -> tile-loop kind, symmetric Korobov weight r (0 if none) and the generic-transform code
// gen = GEN_* | r0 << 4 | r1 << 8 (Table A.2)
bool decode_transform(int transform, int* kind, int* r, int* gen = nullptr) {
    int g = 0;
    bool ok = false;
    *r = 0;
    if (transform == QMC_TRANSFORM_NONE) { *kind = TR_NONE; g = GEN_NONE; ok = true; }
    else if (transform == QMC_TRANSFORM_BAKER) { *kind = TR_BAKER; g = GEN_BAKER; ok = true; }
    else if (transform >= QMC_TRANSFORM_KOROBOV + 1 && transform <= QMC_TRANSFORM_KOROBOV + 6) {
        *r = transform - QMC_TRANSFORM_KOROBOV;
        *kind = (*r == 3) ? TR_KOR3 : TR_KORR;
        g = GEN_KOROBOV_SYM | (*r << 4) | (*r << 8);
        ok = true;
    } else if (transform >= QMC_TRANSFORM_SIDI + 1 && transform <= QMC_TRANSFORM_SIDI + 6) {
        *kind = TR_KORR;
        g = GEN_SIDI | ((transform - QMC_TRANSFORM_SIDI) << 4);
        ok = true;
    } else if (transform >= QMC_TRANSFORM_KOROBOV_ASYM) {
        const int r0 = (transform - QMC_TRANSFORM_KOROBOV_ASYM) / 16, r1 = (transform - QMC_TRANSFORM_KOROBOV_ASYM) % 16;
        if (r0 >= 1 && r0 <= 6 && r1 >= 1 && r1 <= 6) {
            if (r0 == r1) return decode_transform(QMC_TRANSFORM_KOROBOV + r0, kind, r, gen);
            *kind = TR_KORR;
            g = GEN_KOROBOV_ASYM | (r0 << 4) | (r1 << 8);
            ok = true;
        }
    }
    if (gen) *gen = ok ? g : 0;
    return ok;
}

// C(a, b) for the small arguments of the transform tables (a <= 12): exact integer Pascal recurrence
double binom(int a, int b) {
    unsigned long long row[16] = {1};
    for (int n = 1; n <= a; ++n)
        for (int k = n; k >= 1; --k) row[k] += row[k - 1];
    return (b < 0 || b > a) ? 0.0 : (double)row[b];
}

// struct-level validation (no dereference of the data pointers)
int validate_struct(const qmc_problem& p, bool need_two_shifts) {
    if (ncomp_of(p.family) < 0) return QMC_ERR_FAMILY;
    if (p.dim < 1 || p.dim > QMC_MAX_DIM) return QMC_ERR_DIM;
    if (dim_slots(p.family, p.dim, false) < 0) return QMC_ERR_DIM;
    if (p.n < 2 || p.n >= (1ull << 53)) return QMC_ERR_N;
    if (p.m < (need_two_shifts ? 2 : 1) || p.m > QMC_MAX_M) return QMC_ERR_M;
    int kind, r;
    if (!decode_transform(p.transform, &kind, &r)) return QMC_ERR_TRANSFORM;
    if (!p.params || !p.z || !p.shifts) return QMC_ERR_NULL;
    if (p.family == QMC_FAMILY_GENZ_OSC && p.n_params != 1 + p.dim) return QMC_ERR_PARAMS;
    if ((p.family == QMC_FAMILY_GENZ_PRODPEAK || p.family == QMC_FAMILY_CEXP_POLY) && p.n_params != 2 * p.dim) return QMC_ERR_PARAMS;
    if (p.family == QMC_FAMILY_GENZ_CORNER && p.n_params != p.dim) return QMC_ERR_PARAMS;
    if ((p.family == QMC_FAMILY_GENZ_GAUSSIAN || p.family == QMC_FAMILY_GENZ_C0) && p.n_params != 2 * p.dim) return QMC_ERR_PARAMS;
    if (p.family == QMC_FAMILY_GENZ_DISCONT && p.n_params != p.dim + std::min(p.dim, 2)) return QMC_ERR_PARAMS;
    if (is_sector_family(p.family)) {
        const int rest = p.n_params - 4 - p.dim, rec = sector_mono_stride(p.family, p.dim);
        const bool plain = rest % rec == 0, with_log = rest >= 3 && (rest - 3) % rec == 0;   // optional trailing [lu, lf, p]
        if (rest < 2 * rec || !(plain || with_log) || rest / rec > 2 * kMaxSectorMono) return QMC_ERR_PARAMS;
    }
    return QMC_OK;
}

// ---- launch plan: tiles, kernel variants, workspace layout (pure function of the problem structs) ----
struct Variant {
    int family, dp;                  // kernel family (kernel_family(public id), or kKernelFamilySpec), dimension slots
    bool wide;
    std::vector<int> plist;          // problem indices, queue order (most expensive tiles first)
    long long total_tiles = 0;
    int spec_kernel = -1;            // kKernelFamilySpec: the module's kernel
    int group = kGroup;              // closed-form families: shifts per group of the kernel (4, or 8: pick_group)
    int gen_kind = -1;               // closed-form families: GEN_* kind of a dedicated generic kernel, or -1
};

struct Plan {
    std::vector<DevProblem> dev;
    std::vector<Variant> variants;
    int max_m = 0;
    size_t off_counters = 0, off_probs = 0, off_plist = 0, off_prefix = 0, off_aux = 0, off_prog = 0, off_means = 0,
           off_partials = 0, total = 0;
    size_t prog_words = 0, means_doubles = 0, partial_doubles = 0;
    long long total_tiles = 0;
};

const qmc_plan_options kDefaultOptions = {0, 0, 0, 0};

// Shifts per group of a closed-form kernel.  The product-peak kernels of <= 8 dimension slots exist with 4 and with 8 shifts per
// lattice index: 8 amortise the residue walk over twice the shifts and give every warp twice the independent chains (configs[1]:
// 0.141 -> 0.130 ms), but a ragged last group evaluates idle slots, so the choice follows m: the fewer slots, an 8-group slot
// counted as kGroup8Cost of a 4-group slot.  Measured for every family at 4 / 6 / 8 slots and m = 32: the other families (longer
// per-point chains, more live registers at the same 128-register cap) lose 1-20 % with 8, and so does the product peak with a fit
// map: they keep 4.
constexpr double kGroup8Cost = 0.95;
int pick_group(int kernel_fam, int dp, bool wide, int m, bool has_fit, const qmc_plan_options& opt) {
    if (!closed_has_group8(kernel_fam, dp, wide)) return kGroup;
    if (opt.group == kGroup || opt.group == kGroupWide) return opt.group;
    if (has_fit) return kGroup;
    const double slots4 = (double)((m + kGroup - 1) / kGroup * kGroup);
    const double slots8 = (double)((m + kGroupWide - 1) / kGroupWide * kGroupWide) * kGroup8Cost;
    return slots8 < slots4 ? kGroupWide : kGroup;
}

int make_plan(int count, const qmc_problem* problems, bool need_two_shifts, Plan* plan, const qmc_plan_options& opt = kDefaultOptions,
              const qmc_sector_module* module = nullptr, const int* module_index = nullptr) {
    if (count < 1 || !problems) return count < 1 ? QMC_ERR_N : QMC_ERR_NULL;
    // the batch the module was built from, in its order -- or (internal callers: the batched iteration) any selection of its
    // problems, problems[i] being problem module_index[i] of the module's batch
    auto in_module = [&](int i) { return module_index ? module_index[i] : i; };
    if (module) {
        if (!module_index && spec_problem_count(module) != count) return QMC_ERR_N;
        const SpecProblem* sp = spec_problems(module);
        for (int i = 0; i < count; ++i) {
            const int k = in_module(i);
            if (k < 0 || k >= spec_problem_count(module)) return QMC_ERR_N;
            if (sp[k].family != problems[i].family || sp[k].dim != problems[i].dim || sp[k].n_params != problems[i].n_params) return QMC_ERR_PARAMS;
        }
    }
    plan->dev.resize(count);
    long long means_off = 0;
    size_t prog_off = 0;
    for (int i = 0; i < count; ++i) {
        const qmc_problem& p = problems[i];
        const int st = validate_struct(p, need_two_shifts);
        if (st != QMC_OK) return st;
        DevProblem d;
        std::memset(&d, 0, sizeof(d));
        d.params = p.params; d.z = reinterpret_cast<const unsigned long long*>(p.z); d.shifts = p.shifts; d.fit = p.fit_coeffs;
        d.n = p.n;
        d.inv_n = 1.0 / (double)p.n;                                   // reading C-2
        d.family = p.family; d.dim = p.dim; d.m = p.m; d.ncomp = ncomp_of(p.family);
        decode_transform(p.transform, &d.tr_kind, &d.kor_r, &d.gen);
        d.has_fit = p.fit_coeffs ? 1 : 0;
        d.n_params = p.n_params;
        d.out_index = i;
        d.wconst = 1.0;
        const int npad = dim_slots(p.family, p.dim, variant_wide(p.family, p.dim, p.n, opt)) - p.dim;   // padded dimension slots sit at u = 1/2 (qmc_fused.cuh)
        if (d.kor_r > 0) {
            // Eq. 15: c_r = (2r+1) C(2r,r); centred antiderivative coefficients of Eq. 14 (see qmc_device.cuh)
            const int r = d.kor_r;
            const double cr = (2.0 * r + 1.0) * binom(2 * r, r);
            for (int k = 0; k <= r; ++k)
                d.kor[k] = cr * binom(r, k) * std::ldexp(1.0, 2 * (k - r)) * ((k & 1) ? -1.0 : 1.0) / (double)(2 * k + 1);
            for (int j = 0; j < p.dim; ++j) d.wconst *= cr;
            d.wconst = std::ldexp(d.wconst, 2 * r * npad);               // a padded slot contributes (1/4)^r: exact compensation
        } else if ((d.gen & 15) == GEN_KOROBOV_ASYM) {
            // Eq. 15 with r0 != r1: c = (r0+r1+1) C(r0+r1,r0); phi(u) = c sum_i C(r1,i)(-1)^i u^(r0+1+i)/(r0+1+i) (Eq. 14)
            const int r0 = (d.gen >> 4) & 15, r1 = (d.gen >> 8) & 15;
            const double c = (double)(r0 + r1 + 1) * binom(r0 + r1, r0);
            for (int k = 0; k <= r1; ++k) d.kor[k] = c * binom(r1, k) * ((k & 1) ? -1.0 : 1.0) / (double)(r0 + 1 + k);
            for (int k = 0; k <= r0; ++k) d.kor[8 + k] = c * binom(r0, k) * ((k & 1) ? -1.0 : 1.0) / (double)(r1 + 1 + k);
            for (int j = 0; j < p.dim; ++j) d.wconst *= c;
            d.wconst = std::ldexp(d.wconst, (r0 + r1) * npad);           // a padded slot contributes (1/2)^(r0+r1)
        } else if ((d.gen & 15) == GEN_SIDI && d.gen) {
            // Eq. 16: K_r = pi / 2^r Gamma(r+1) / Gamma((r+1)/2)^2; a padded slot has sin(pi/2)^r = 1
            const int r = (d.gen >> 4) & 15;
            const double gh = std::tgamma(0.5 * (r + 1));
            const double K = 3.141592653589793238462643383279 / std::ldexp(1.0, r) * std::tgamma(r + 1.0) / (gh * gh);
            d.kor[0] = K / 3.141592653589793238462643383279;
            for (int j = 0; j < p.dim; ++j) d.wconst *= K;
        }
        if (is_sector_family(p.family)) {
            const int nmono = (p.n_params - 4 - p.dim) / sector_mono_stride(p.family, p.dim);
            d.aux_off = (int)prog_off;
            d.aux_len = sector_slot_words(nmono, p.family == QMC_FAMILY_SECTOR_COMPLEX) + 2 * nmono + 1;   // coefficient slots + 16 one-byte steps per monomial + end steps / padding
            prog_off += (size_t)d.aux_len;
        }
        d.means_off = means_off;
        means_off += (long long)p.m * d.ncomp;
        plan->max_m = std::max(plan->max_m, p.m);
        plan->dev[i] = d;
    }
    // kernel variants
    for (int i = 0; i < count; ++i) {
        const DevProblem& d = plan->dev[i];
        const bool wide = variant_wide(d.family, d.dim, d.n, opt);
        const int dp = dim_slots(d.family, d.dim, wide);
        // a specialised kernel holds the sector's code and serves the default tile loop only (Korobov-3, no fit map, narrow residues)
        int kfam = kernel_family(d.family), spec_kernel = -1;
        if (module && is_sector_family(d.family) && !wide && d.tr_kind == TR_KOR3 && !d.has_fit && spec_problems(module)[in_module(i)].kernel >= 0) {
            kfam = kKernelFamilySpec;
            spec_kernel = spec_problems(module)[in_module(i)].kernel;
            plan->dev[i].spec_case = spec_problems(module)[in_module(i)].kase;
        }
        const int group = pick_group(kfam, dp, wide, d.m, d.has_fit != 0, opt);
        // Korobov r != 3, Korobov (r0, r1) and Sidi without a fit map, 32-bit residues, <= 16 slots: the dedicated generic kernels
        int gen_kind = -1;
        const bool closed = kfam == 0 || kfam == 1 || kfam == 2 || kfam == kKernelFamilyGenzMisc;
        if (closed && !wide && dp <= 16 && d.tr_kind == TR_KORR && !d.has_fit && (d.gen & 15) < kGenKinds && !opt.generic_call)
            gen_kind = d.gen & 15;
        Variant* v = nullptr;
        for (auto& c : plan->variants)
            if (c.family == kfam && c.dp == dp && c.wide == wide && c.spec_kernel == spec_kernel && c.group == group && c.gen_kind == gen_kind) v = &c;
        if (!v) { plan->variants.push_back(Variant{kfam, dp, wide, {}, 0, spec_kernel, group, gen_kind}); v = &plan->variants.back(); }
        v->plist.push_back(i);
    }
    if (plan->variants.size() > 64) return QMC_ERR_WORKSPACE;
    // tiling (S9): per kernel variant aim at kWaves x (resident CTAs of a B200) tiles, shared among the variant's problems
    // in proportion to their cost; a tile is at least one index per thread and at most kMaxSteps (bounds the fp64 chains)
    for (auto& v : plan->variants) {
        const bool sector_variant = v.family == QMC_FAMILY_SECTOR || v.family == kKernelFamilyCSector || v.family == kKernelFamilySpec;
        const int resident = kPlanSMs * (sector_variant ? min_blocks_sector(v.dp) : (v.gen_kind >= 0 ? min_blocks_generic(v.dp) : min_blocks_closed(v.dp, v.wide)));
        const int threads = v.family == kKernelFamilySpec ? spec_kernel_threads(module, v.spec_kernel)
                            : (v.family == QMC_FAMILY_SECTOR ? sector_threads(v.dp) : (v.family == kKernelFamilyCSector ? kCSectorThreads : kThreads));   // CTA size of the variant's kernel
        const int env = opt.tiles_target > 0 ? opt.tiles_target : 0;
        // one problem: equal tiles, 2 per resident CTA (the queue evens out SM speed differences over a long kernel) -- or
        // exactly 1 when the whole kernel is short (< kShortEvalsPerCta evaluations per CTA: per-tile overhead and the
        // queue reset matter more than balance); a batch of unequal problems: 8 per resident CTA
        int waves = kWavesBatch;
        if (v.plist.size() == 1) {
            const DevProblem& d0 = plan->dev[v.plist[0]];
            waves = ((double)d0.n * d0.m < (double)kShortEvalsPerCta * resident) ? 1 : kWavesSingle;
        }
        const double target = env > 0 ? env : resident * waves;
        double total_cost = 0.0;
        for (int i : v.plist) total_cost += (double)plan->dev[i].n * plan->dev[i].m * (12.0 * plan->dev[i].dim + 0.5 * plan->dev[i].n_params + 40.0);
        for (int i : v.plist) {
            DevProblem& d = plan->dev[i];
            const double cost = (double)d.n * d.m * (12.0 * d.dim + 0.5 * d.n_params + 40.0);
            const double want = std::max(1.0, std::floor(target * cost / total_cost));
            unsigned long long tile_len = (unsigned long long)std::ceil((double)d.n / want);
            const unsigned long long max_len = (unsigned long long)kMaxSteps * threads;
            if (tile_len > max_len && v.plist.size() == 1 && env == 0) {
                // a lattice too long for `target` tiles of at most kMaxSteps indices per thread: more tiles, in whole waves --
                // a multiple of the resident CTAs, all of equal length, so that the last wave is as full as the others
                // (configs[4]: 8436 tiles = 19 waves of 444 instead of 8192 = 18.45)
                unsigned long long tiles_min = (d.n + max_len - 1) / max_len;
                tiles_min = (tiles_min + resident - 1) / resident * resident;
                tile_len = (d.n + tiles_min - 1) / tiles_min;
            }
            tile_len = std::min<unsigned long long>(std::max<unsigned long long>(tile_len, threads), max_len);
            const unsigned long long tiles = (d.n + tile_len - 1) / tile_len;
            if (tiles > 0x7fffffffull) return QMC_ERR_N;
            d.tile_len = (long long)tile_len;
            d.steps = (int)((tile_len + threads - 1) / threads);
            d.tiles = (int)tiles;
        }
    }
    long long partial_off = 0;
    for (int i = 0; i < count; ++i) {
        plan->dev[i].partial_off = partial_off;
        partial_off += (long long)plan->dev[i].tiles * plan->dev[i].m * plan->dev[i].ncomp;
    }
    for (auto& v : plan->variants) {
        // most expensive tiles first (S9); cost ~ indices x shifts x (dimension work + integrand size)
        auto cost = [&](int i) {
            const DevProblem& d = plan->dev[i];
            return (double)d.tile_len * d.m * (12.0 * d.dim + 0.5 * d.n_params + 40.0);
        };
        std::stable_sort(v.plist.begin(), v.plist.end(), [&](int a, int b) { return cost(a) > cost(b); });
        for (int i : v.plist) { plan->dev[i].tile_begin = v.total_tiles; v.total_tiles += plan->dev[i].tiles; }
        plan->total_tiles += v.total_tiles;
    }
    plan->prog_words = prog_off;
    plan->means_doubles = (size_t)means_off;
    plan->partial_doubles = (size_t)partial_off;
    size_t o = 0;
    plan->off_counters = o; o = align_up(o + 64 * sizeof(unsigned long long), 256);
    plan->off_probs = o; o = align_up(o + (size_t)count * sizeof(DevProblem), 256);
    plan->off_plist = o; o = align_up(o + (size_t)count * sizeof(int), 256);
    plan->off_prefix = o; o = align_up(o + ((size_t)count + 64) * sizeof(long long), 256);   // <= 64 variants: the size does not depend on the routing
    plan->off_aux = o; o = align_up(o + (size_t)count * sizeof(DevAux), 256);
    plan->off_prog = o; o = align_up(o + plan->prog_words * 8, 256);
    plan->off_means = o; o = align_up(o + plan->means_doubles * 8, 256);
    plan->off_partials = o; o = align_up(o + plan->partial_doubles * 8, 256);
    plan->total = o;
    return QMC_OK;
}

// Immutable device attributes, cached per device ordinal (written once with the same value by whichever thread asks first).
constexpr int kMaxDevices = 64;
int current_device() {
    int dev = 0;
    return cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < kMaxDevices ? dev : -1;
}
int sm_count() {
    static int cache[kMaxDevices];
    const int dev = current_device();
    if (dev < 0) return 0;
    if (cache[dev] > 0) return cache[dev];
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    cache[dev] = n;
    return n;
}

// closed-form families: the kernel variants live in four parts per family (+ one of the product peak with 8 shifts per group) (qmc_fused_closed.inc); try each
#define QMC_TRY_PARTS(FAM, PREFIX, FAIL, ...)                                                             \
    {                                                                                                    \
        auto r0 = PREFIX##FAM##_0(__VA_ARGS__); if (r0 != FAIL) return r0;                               \
        auto r1 = PREFIX##FAM##_1(__VA_ARGS__); if (r1 != FAIL) return r1;                               \
        auto r2 = PREFIX##FAM##_2(__VA_ARGS__); if (r2 != FAIL) return r2;                               \
        return PREFIX##FAM##_3(__VA_ARGS__);                                                             \
    }
cudaError_t launch_closed(int family, int dp, bool wide, int group, int grid, cudaStream_t st, const FusedLaunch& a) {
    switch (family) {
        case 0: QMC_TRY_PARTS(0, launch_fused_part_, cudaErrorInvalidValue, dp, wide, group, grid, st, a)
        case 1:
            if (group == kGroupWide) return launch_fused_part_1_4(dp, wide, group, grid, st, a);
            QMC_TRY_PARTS(1, launch_fused_part_, cudaErrorInvalidValue, dp, wide, group, grid, st, a)
        case 2: QMC_TRY_PARTS(2, launch_fused_part_, cudaErrorInvalidValue, dp, wide, group, grid, st, a)
        case 4: QMC_TRY_PARTS(4, launch_fused_part_, cudaErrorInvalidValue, dp, wide, group, grid, st, a)
    }
    return cudaErrorInvalidValue;
}
int occupancy_closed(int family, int dp, bool wide, int group) {
    switch (family) {
        case 0: QMC_TRY_PARTS(0, occupancy_fused_part_, -1, dp, wide, group)
        case 1:
            if (group == kGroupWide) return occupancy_fused_part_1_4(dp, wide, group);
            QMC_TRY_PARTS(1, occupancy_fused_part_, -1, dp, wide, group)
        case 2: QMC_TRY_PARTS(2, occupancy_fused_part_, -1, dp, wide, group)
        case 4: QMC_TRY_PARTS(4, occupancy_fused_part_, -1, dp, wide, group)
    }
    return -1;
}
#undef QMC_TRY_PARTS

#define QMC_GENERIC_KINDS(FAM, PREFIX, ...)                      \
    switch (kind) {                                               \
        case 0: return PREFIX##FAM##_0(__VA_ARGS__);              \
    }                                                             \
    break;
cudaError_t launch_generic(int family, int kind, int dp, int grid, cudaStream_t st, const FusedLaunch& a) {
    switch (family) {
        case 0: QMC_GENERIC_KINDS(0, launch_fused_generic_, dp, grid, st, a)
        case 1: QMC_GENERIC_KINDS(1, launch_fused_generic_, dp, grid, st, a)
        case 2: QMC_GENERIC_KINDS(2, launch_fused_generic_, dp, grid, st, a)
        case 4: QMC_GENERIC_KINDS(4, launch_fused_generic_, dp, grid, st, a)
    }
    return cudaErrorInvalidValue;
}
int occupancy_generic_uncached(int family, int kind, int dp) {
    switch (family) {
        case 0: QMC_GENERIC_KINDS(0, occupancy_fused_generic_, dp)
        case 1: QMC_GENERIC_KINDS(1, occupancy_fused_generic_, dp)
        case 2: QMC_GENERIC_KINDS(2, occupancy_fused_generic_, dp)
        case 4: QMC_GENERIC_KINDS(4, occupancy_fused_generic_, dp)
    }
    return -1;
}
#undef QMC_GENERIC_KINDS
int occupancy_generic(int family, int kind, int dp) {
    static int cache[kMaxDevices][kKernelFamilies][kGenKinds][17];
    const int dev = current_device();
    if (dev < 0 || kind < 0 || kind >= kGenKinds || dp > 16) return -1;
    int& c = cache[dev][family][kind][dp];
    if (c > 0) return c;
    const int v = occupancy_generic_uncached(family, kind, dp);
    if (v > 0) c = v;
    return v;
}

int occupancy(int family, int dp, bool wide, int group = kGroup) {
    static int cache[kMaxDevices][kKernelFamilies][33][2][2];
    const int dev = current_device();
    if (dev < 0) return -1;
    int& c = cache[dev][family][dp][wide ? 1 : 0][group == kGroupWide ? 1 : 0];
    if (c > 0) return c;
    int v = -1;
    switch (family) {
        case 0: case 1: case 2: case 4: v = occupancy_closed(family, dp, wide, group); break;
        case 3: v = occupancy_fused_f3(dp, wide); break;
        case kKernelFamilyCSector: v = occupancy_fused_f8(dp, wide); break;
    }
    if (v > 0) c = v;
    return v;
}

// the thread's staging arena (pinned host + device), grown on demand; bound to the device that is current
int arena_reserve(size_t pinned_bytes, size_t device_bytes) {
    ThreadState& t = g_ts;
    const int dev = current_device();
    if (dev < 0) return cuda_fail(cudaErrorNoDevice, "no CUDA device");
    if (t.arena_device != dev && (t.pinned || t.device)) {
        if (t.pinned) { cudaFreeHost(t.pinned); t.pinned = nullptr; t.pinned_bytes = 0; }
        if (t.device) { cudaFree(t.device); t.device = nullptr; t.device_bytes = 0; }
    }
    t.arena_device = dev;
    if (pinned_bytes > t.pinned_bytes) {
        if (t.pinned) { cudaFreeHost(t.pinned); t.pinned = nullptr; t.pinned_bytes = 0; }
        const size_t want = std::max<size_t>(pinned_bytes + pinned_bytes / 2, 1 << 16);
        cudaError_t e = cudaHostAlloc(reinterpret_cast<void**>(&t.pinned), want, cudaHostAllocMapped | cudaHostAllocPortable);   // the results are written here by the device
        if (e != cudaSuccess) return cuda_fail(e, "cudaMallocHost (staging arena)");
        t.pinned_bytes = want;
    }
    if (device_bytes > t.device_bytes) {
        if (t.device) { cudaFree(t.device); t.device = nullptr; t.device_bytes = 0; }
        const size_t want = std::max<size_t>(device_bytes + device_bytes / 2, 1 << 20);
        cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&t.device), want);
        if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc (staging arena)");
        t.device_bytes = want;
    }
    return QMC_OK;
}

// phases of a batch call: a prepared batch (qmc_batch_*) uploads and prepares once (kPhaseSetup) and then only launches
// (kPhaseLaunch: one memset of the queue heads + the kernels, nothing read from host memory)
constexpr int kPhaseAll = 0, kPhaseSetup = 1, kPhaseLaunch = 2;

int run_batch(int count, const qmc_problem* problems, double* out_means, double* out_errs, double* out_shift_means,
              void* workspace, size_t workspace_bytes, cudaStream_t st, const qmc_plan_options& opt = kDefaultOptions,
              char* pinned_blob = nullptr, Plan* prebuilt = nullptr, qmc_sector_module* module = nullptr, int sm_stride = 0,
              int phase = kPhaseAll) {
    g_ts.last_launches = 0;
    if (phase != kPhaseSetup && (!out_means || !out_errs)) return QMC_ERR_NULL;
    Plan local_plan;
    Plan& plan = prebuilt ? *prebuilt : local_plan;          // the HOST-pointer entry plans once and patches the data pointers
    if (!prebuilt) {
        const int pst = make_plan(count, problems, true, &local_plan, opt, module);
        if (pst != QMC_OK) return pst;
    }
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255u) || workspace_bytes < plan.total) return QMC_ERR_WORKSPACE;
    const int sms = sm_count();
    if (sms <= 0) return cuda_fail(cudaErrorNoDevice, "no CUDA device");
    char* ws = static_cast<char*>(workspace);

    const DevProblem* dprobs = reinterpret_cast<const DevProblem*>(ws + plan.off_probs);
    DevAux* daux = reinterpret_cast<DevAux*>(ws + plan.off_aux);
    unsigned long long* dprog = reinterpret_cast<unsigned long long*>(ws + plan.off_prog);
    double* dmeans = reinterpret_cast<double*>(ws + plan.off_means);
    double* dpart = reinterpret_cast<double*>(ws + plan.off_partials);
    bool any_sector = false;
    for (const DevProblem& d : plan.dev) any_sector = any_sector || is_sector_family(d.family);
    // single mode: one closed-form problem travels in the kernel parameter; nothing is uploaded, reset or prepared
    const bool single = count == 1 && !any_sector;
    FusedLaunch base;
    std::memset(&base, 0, sizeof(base));
    base.probs = dprobs; base.aux = daux; base.prog = dprog; base.partials = dpart;
    base.single = single ? 1 : 0;
    if (single) base.one = plan.dev[0];

    std::vector<VariantQueue> queues(plan.variants.size());
    if (!single) {
        // host image of [queue heads (zero) | probs | plist | prefix]: one upload resets the queues too
        // (the synchronous HOST-pointer entries pass a pinned staging block; the stream-ordered entry copies from pageable memory,
        // which the runtime stages before cudaMemcpyAsync returns -- the call does not wait for the device)
        const size_t blob_bytes = plan.off_aux - plan.off_counters;
        std::vector<char> pageable;
        char* blob = pinned_blob;
        if (!blob) { pageable.assign(blob_bytes, 0); blob = pageable.data(); }
        else std::memset(blob, 0, blob_bytes);
        std::memcpy(blob + (plan.off_probs - plan.off_counters), plan.dev.data(), (size_t)count * sizeof(DevProblem));
        int* plist = reinterpret_cast<int*>(blob + (plan.off_plist - plan.off_counters));
        long long* prefix = reinterpret_cast<long long*>(blob + (plan.off_prefix - plan.off_counters));
        size_t pl = 0, pf = 0;
        int vi = 0;
        for (auto& v : plan.variants) {
            VariantQueue& q = queues[vi];
            q.plist = reinterpret_cast<const int*>(ws + plan.off_plist) + pl;
            q.tile_prefix = reinterpret_cast<const long long*>(ws + plan.off_prefix) + pf;
            q.plist_len = (int)v.plist.size();
            q.total_tiles = v.total_tiles;
            q.counter = reinterpret_cast<unsigned long long*>(ws + plan.off_counters) + vi;
            long long acc = 0;
            for (int i : v.plist) { plist[pl++] = i; prefix[pf++] = acc; acc += plan.dev[i].tiles; }
            prefix[pf++] = acc;
            ++vi;
        }
        if (phase == kPhaseLaunch) {                        // plan and programs are in the workspace already: reset the queue heads
            QMC_CUDA(cudaMemsetAsync(ws + plan.off_counters, 0, 64 * sizeof(unsigned long long), st));
        } else {
            QMC_CUDA(cudaMemcpyAsync(ws + plan.off_counters, blob, blob_bytes, cudaMemcpyHostToDevice, st));
            if (any_sector) {                               // S0 for the sector family: tables + device-side program compiler
                QMC_CUDA(launch_prepare(count, st, dprobs, daux, dprog));
                ++g_ts.last_launches;
            }
        }
    } else if (phase == kPhaseSetup) {
        return QMC_OK;                                      // a single closed-form problem needs no set-up
    } else {
        std::memset(&queues[0], 0, sizeof(VariantQueue));
        queues[0].total_tiles = plan.variants[0].total_tiles;
        const Variant& v0 = plan.variants[0];
        if (v0.total_tiles > (long long)sms * std::max(1, (v0.gen_kind >= 0 ? occupancy_generic(v0.family, v0.gen_kind, v0.dp) : occupancy(v0.family, v0.dp, v0.wide, v0.group)))) {
            // more tiles than resident CTAs: dynamic queue (one 8-byte reset); otherwise every CTA owns one tile
            queues[0].counter = reinterpret_cast<unsigned long long*>(ws + plan.off_counters);
            QMC_CUDA(cudaMemsetAsync(queues[0].counter, 0, sizeof(unsigned long long), st));
        }
    }
    if (phase == kPhaseSetup) return QMC_OK;
    g_ts.ev_valid = false;
    if (g_ts.profile) {
        const int dev = current_device();
        if (g_ts.ev0 && g_ts.ev_device != dev) { cudaEventDestroy(g_ts.ev0); cudaEventDestroy(g_ts.ev1); g_ts.ev0 = g_ts.ev1 = nullptr; }
        if (!g_ts.ev0) { QMC_CUDA(cudaEventCreate(&g_ts.ev0)); QMC_CUDA(cudaEventCreate(&g_ts.ev1)); g_ts.ev_device = dev; }
        QMC_CUDA(cudaEventRecord(g_ts.ev0, st));
    }
    for (size_t vi = 0; vi < plan.variants.size(); ++vi) {
        const Variant& v = plan.variants[vi];
        const int occ = v.family == kKernelFamilySpec ? spec_occupancy(module, v.spec_kernel) : (v.gen_kind >= 0 ? occupancy_generic(v.family, v.gen_kind, v.dp) : occupancy(v.family, v.dp, v.wide, v.group));
        if (occ <= 0 && v.family == kKernelFamilySpec) return QMC_ERR_CUDA;      // the loader left the text
        if (occ <= 0) return cuda_fail(cudaErrorInvalidDeviceFunction, "occupancy query (is the sm_100a image loadable on this device?)");
        const long long cap = (long long)sms * occ;
        const int grid = (int)std::min<long long>(cap, v.total_tiles);
        FusedLaunch a = base;
        a.vq = queues[vi];
        if (v.family == kKernelFamilySpec) {
            const int rc = spec_launch(module, v.spec_kernel, grid, st, a);
            if (rc != QMC_OK) return rc;
            ++g_ts.last_launches;
            continue;
        }
        cudaError_t e = cudaErrorInvalidValue;
        switch (v.family) {
            case 0: case 1: case 2: case 4:
                e = v.gen_kind >= 0 ? launch_generic(v.family, v.gen_kind, v.dp, grid, st, a) : launch_closed(v.family, v.dp, v.wide, v.group, grid, st, a);
                break;
            case 3: e = launch_fused_f3(v.dp, v.wide, grid, st, a); break;
            case kKernelFamilyCSector: e = launch_fused_f8(v.dp, v.wide, grid, st, a); break;
        }
        if (e != cudaSuccess) return cuda_fail(e, "fused kernel launch");
        ++g_ts.last_launches;
    }
    if (g_ts.profile) { QMC_CUDA(cudaEventRecord(g_ts.ev1, st)); g_ts.ev_valid = true; }
    QMC_CUDA(launch_finalize(count, st, base, dmeans, out_means, out_errs, out_shift_means, sm_stride > 0 ? sm_stride : 2 * plan.max_m));
    ++g_ts.last_launches;
    return QMC_OK;
}

}  // namespace

// Internal (qmc_kernels.h; the batched iteration of qmc_adaptive.cu): a batch call whose problems are a selection of a module's
// batch (module_index, may be null without a module) and whose results land in caller-chosen rows: problem i writes
// out_means / out_errs [out_row[i] * 2 + c] and out_shift_means [out_row[i] * sm_stride + s * ncomp + c].
size_t routed_workspace_bytes(int count, const qmc_problem* problems, const qmc_sector_module* module, const int* module_index) {
    Plan plan;
    if (make_plan(count, problems, false, &plan, kDefaultOptions, module, module_index) != QMC_OK) return 0;
    return plan.total;
}
int run_batch_routed(int count, const qmc_problem* problems, double* out_means, double* out_errs, double* out_shift_means,
                     void* workspace, size_t workspace_bytes, cudaStream_t st, qmc_sector_module* module, const int* module_index,
                     const int* out_row, int sm_stride) {
    Plan plan;
    const int pst = make_plan(count, problems, true, &plan, kDefaultOptions, module, module_index);
    if (pst != QMC_OK) return pst;
    int max_m = 0;
    for (int i = 0; i < count; ++i) { plan.dev[i].out_index = out_row[i]; max_m = std::max(max_m, plan.dev[i].m * plan.dev[i].ncomp); }
    if (sm_stride < max_m) return QMC_ERR_M;
    return run_batch(count, problems, out_means, out_errs, out_shift_means, workspace, workspace_bytes, st, kDefaultOptions, nullptr, &plan,
                     module, sm_stride);
}

namespace {
// ---- full value validation of host-resident data --------------------------------------------------
unsigned long long gcd_u64(unsigned long long a, unsigned long long b) {
    while (b) { const unsigned long long t = a % b; a = b; b = t; }
    return a;
}

int validate_values(const qmc_problem& p) {
    const int st = validate_struct(p, true);
    if (st != QMC_OK) return st;
    for (int j = 0; j < p.dim; ++j) {
        const unsigned long long z = p.z[j];
        if (z < 1 || z >= p.n || gcd_u64(z, p.n) != 1) return QMC_ERR_Z;          // "coprime to n"
    }
    for (long long i = 0; i < (long long)p.m * p.dim; ++i)
        if (!(p.shifts[i] >= 0.0 && p.shifts[i] < 1.0)) return QMC_ERR_SHIFT;      // Delta in [0,1)
    for (int i = 0; i < p.n_params; ++i)
        if (!std::isfinite(p.params[i])) return QMC_ERR_PARAMS;
    if (p.family == QMC_FAMILY_GENZ_PRODPEAK)
        for (int j = 0; j < p.dim; ++j)
            if (p.params[j] == 0.0) return QMC_ERR_PARAMS;
    if (is_sector_family(p.family)) {
        const double* q = p.params;
        for (int k = 0; k < 4; ++k)
            if (q[k] != std::floor(q[k]) || q[k] < 0.0) return QMC_ERR_PARAMS;
        if (q[0] > 8 || q[1] > 8 || q[2] < 1 || q[3] < 1 || q[2] > kMaxSectorMono || q[3] > kMaxSectorMono) return QMC_ERR_PARAMS;
        const int base = 4 + p.dim + ((int)q[2] + (int)q[3]) * sector_mono_stride(p.family, p.dim);
        if (p.n_params == base + 3) {                                            // log factor: p an integer in 1..4
            if (!(q[base + 2] >= 1.0 && q[base + 2] <= 4.0) || q[base + 2] != std::floor(q[base + 2])) return QMC_ERR_PARAMS;
        } else if (p.n_params != base) return QMC_ERR_PARAMS;
    }
    if (p.fit_coeffs) {
        for (int j = 0; j < p.dim; ++j) {
            const double* a = p.fit_coeffs + 6 * j;
            for (int k = 0; k < 6; ++k)
                if (!std::isfinite(a[k])) return QMC_ERR_FIT;
            const double a4 = a[4], a5 = a[5], a6 = 1.0 - a[2] - a[3] - a4 - a5;
            if (a[2] == 0.0 && a[3] == 0.0) {
                // cubic map: p'(y) = a4 + 2 a5 y + 3 a6 y^2 must stay positive on [0,1] (monotone map, Eq. 18)
                double mn = std::fmin(a4, a4 + 2.0 * a5 + 3.0 * a6);
                if (a6 != 0.0) {
                    const double yv = -a5 / (3.0 * a6);
                    if (yv > 0.0 && yv < 1.0) mn = std::fmin(mn, a4 + yv * (2.0 * a5 + 3.0 * a6 * yv));
                }
                if (!(mn > 0.0)) return QMC_ERR_FIT;
            } else {
                // pole terms: the bounds of P:L231 keep the poles outside [0,1]; monotonicity is checked on a fine grid
                if (!(a[0] >= 1.001) || !(a[1] <= -0.001) || !(a[2] >= 0.0) || !(a[3] >= 0.0)) return QMC_ERR_FIT;
                for (int i = 0; i <= 1024; ++i) {
                    const double y = (double)i / 1024.0;
                    const double dp = a[2] * a[0] * (a[0] - 1.0) / ((a[0] - y) * (a[0] - y)) + a[3] * a[1] * (a[1] - 1.0) / ((a[1] - y) * (a[1] - y)) +
                                      a4 + y * (2.0 * a5 + 3.0 * a6 * y);
                    if (!(dp > 0.0)) return QMC_ERR_FIT;
                }
            }
        }
    }
    return QMC_OK;
}

int family_param_count(int family, const double* params, int dim) {
    if (family == QMC_FAMILY_GENZ_OSC) return 1 + dim;
    if (family == QMC_FAMILY_GENZ_PRODPEAK || family == QMC_FAMILY_CEXP_POLY) return 2 * dim;
    if (family == QMC_FAMILY_GENZ_CORNER) return dim;
    if (family == QMC_FAMILY_GENZ_GAUSSIAN || family == QMC_FAMILY_GENZ_C0) return 2 * dim;
    if (family == QMC_FAMILY_GENZ_DISCONT) return dim + std::min(dim, 2);
    if (is_sector_family(family) && params) {
        const double nU = params[2], nF = params[3];
        if (!(nU >= 1 && nU <= kMaxSectorMono && nF >= 1 && nF <= kMaxSectorMono)) return -1;
        return 4 + dim + ((int)nU + (int)nF) * sector_mono_stride(family, dim);
    }
    return -1;
}

}  // namespace
}  // namespace qmc

using namespace qmc;

extern "C" {

int qmc_num_components(int family) { return ncomp_of(family); }

const char* qmc_status_string(int status) {
    switch (status) {
        case QMC_OK: return "ok";
        case QMC_ERR_NULL: return "null pointer";
        case QMC_ERR_DIM: return "dimension out of range";
        case QMC_ERR_N: return "lattice size / count out of range";
        case QMC_ERR_Z: return "generating vector component out of range or not coprime to n";
        case QMC_ERR_SHIFT: return "shift outside [0,1)";
        case QMC_ERR_M: return "number of shifts out of range";
        case QMC_ERR_TRANSFORM: return "unknown periodizing transform";
        case QMC_ERR_FAMILY: return "unknown integrand family";
        case QMC_ERR_PARAMS: return "integrand parameter block invalid";
        case QMC_ERR_FIT: return "fit map invalid";
        case QMC_ERR_WORKSPACE: return "workspace null, misaligned or too small";
        case QMC_ERR_CUDA: return "CUDA error";
        case QMC_ERR_NONFINITE: return "non-finite result";
        case QMC_ERR_MAXEVAL: return "error goal not reached within maxeval / the available lattices and shifts";
    }
    return "unknown status";
}

const char* qmc_last_cuda_error(void) { return g_ts.last_error.c_str(); }
int qmc_last_launch_count(void) { return g_ts.last_launches; }

int qmc_profile_enable(int on) { g_ts.profile = on != 0; return QMC_OK; }

int qmc_release_thread_resources(void) {
    g_ts.release();
    return QMC_OK;
}

int qmc_profile_last_fused_ms(double* out_ms) {
    if (!out_ms) return QMC_ERR_NULL;
    if (!g_ts.ev_valid) return QMC_ERR_N;
    QMC_CUDA(cudaEventSynchronize(g_ts.ev1));
    float ms = 0.f;
    QMC_CUDA(cudaEventElapsedTime(&ms, g_ts.ev0, g_ts.ev1));
    *out_ms = (double)ms;
    return QMC_OK;
}

size_t qmc_workspace_bytes_opts(int count, const qmc_problem* problems, const qmc_plan_options* opts) {
    Plan plan;
    if (make_plan(count, problems, true, &plan, opts ? *opts : kDefaultOptions) != QMC_OK) return 0;
    return plan.total;
}
size_t qmc_workspace_bytes(int count, const qmc_problem* problems) { return qmc_workspace_bytes_opts(count, problems, nullptr); }
size_t qmc_sector_module_workspace_bytes(const qmc_sector_module* module, int count, const qmc_problem* problems) {
    Plan plan;
    if (!module || make_plan(count, problems, true, &plan, kDefaultOptions, module) != QMC_OK) return 0;
    return plan.total;
}

int qmc_plan_info(int count, const qmc_problem* problems, long long* out_tiles, int* out_ctas, long long* out_tile_len0) {
    Plan plan;
    const int st = make_plan(count, problems, true, &plan);
    if (st != QMC_OK) return st;
    if (out_tiles) *out_tiles = plan.total_tiles;
    if (out_tile_len0) *out_tile_len0 = plan.dev[0].tile_len;
    if (out_ctas) {
        int ctas = 0;
        const int sms = sm_count();
        for (auto& v : plan.variants) {
            const int occ = sms > 0 ? (v.gen_kind >= 0 ? occupancy_generic(v.family, v.gen_kind, v.dp) : occupancy(v.family, v.dp, v.wide, v.group)) : 0;
            ctas += (int)std::min<long long>((long long)sms * std::max(occ, 0), v.total_tiles);
        }
        *out_ctas = ctas;
    }
    return QMC_OK;
}

int qmc_validate_problem_host(const qmc_problem* p) {
    if (!p) return QMC_ERR_NULL;
    return validate_values(*p);
}

int qmc_lattice_integrate_batch_opts(int count, const qmc_problem* problems, double* out_means, double* out_errs,
                                     double* out_shift_means, void* workspace, size_t workspace_bytes, void* cuda_stream,
                                     const qmc_plan_options* opts) {
    return run_batch(count, problems, out_means, out_errs, out_shift_means, workspace, workspace_bytes,
                     static_cast<cudaStream_t>(cuda_stream), opts ? *opts : kDefaultOptions);
}
// ---- prepared batches: plan, upload and prepare once; every later call is kernel launches only ---------------------------------
struct qmc_batch {
    Plan plan;
    std::vector<qmc_problem> problems;
    qmc_sector_module* module = nullptr;
    void* workspace = nullptr;
    size_t workspace_bytes = 0;
    int device = -1;
};

int qmc_batch_create(int count, const qmc_problem* problems, qmc_sector_module* module, void* workspace, size_t workspace_bytes,
                     void* cuda_stream, qmc_batch** out) {
    if (!out) return QMC_ERR_NULL;
    *out = nullptr;
    qmc_batch* b = new qmc_batch;
    const int pst = make_plan(count, problems, true, &b->plan, kDefaultOptions, module);
    if (pst != QMC_OK) { delete b; return pst; }
    b->problems.assign(problems, problems + count);
    b->module = module; b->workspace = workspace; b->workspace_bytes = workspace_bytes; b->device = current_device();
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int rc = run_batch(count, b->problems.data(), nullptr, nullptr, nullptr, workspace, workspace_bytes, st, kDefaultOptions, nullptr, &b->plan,
                       module, 0, kPhaseSetup);
    if (rc == QMC_OK && module) {                        // load the module's kernels on this device now, not inside the first launch
        for (const Variant& v : b->plan.variants)
            if (v.family == kKernelFamilySpec && spec_occupancy(module, v.spec_kernel) <= 0) rc = QMC_ERR_CUDA;
    }
    if (rc == QMC_OK) {
        for (const Variant& v : b->plan.variants)        // fill the occupancy cache (a query is not a launch, but it is not capturable either)
            if (v.family != kKernelFamilySpec && (v.gen_kind >= 0 ? occupancy_generic(v.family, v.gen_kind, v.dp) : occupancy(v.family, v.dp, v.wide, v.group)) <= 0)
                rc = cuda_fail(cudaErrorInvalidDeviceFunction, "occupancy query (is the sm_100a image loadable on this device?)");
    }
    // the plan was staged from host memory that dies with this call
    if (rc == QMC_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = cuda_fail(cudaGetLastError(), "cudaStreamSynchronize (qmc_batch_create)");
    if (rc != QMC_OK) { delete b; return rc; }
    *out = b;
    return QMC_OK;
}

int qmc_batch_launch(qmc_batch* b, double* out_means, double* out_errs, double* out_shift_means, void* cuda_stream) {
    if (!b) return QMC_ERR_NULL;
    if (current_device() != b->device) return cuda_fail(cudaErrorInvalidDevice, "qmc_batch_launch: the batch was created on another device");
    return run_batch((int)b->problems.size(), b->problems.data(), out_means, out_errs, out_shift_means, b->workspace, b->workspace_bytes,
                     static_cast<cudaStream_t>(cuda_stream), kDefaultOptions, nullptr, &b->plan, b->module, 0, kPhaseLaunch);
}

void qmc_batch_destroy(qmc_batch* b) { delete b; }

int qmc_lattice_integrate_batch_module(qmc_sector_module* module, int count, const qmc_problem* problems, double* out_means,
                                       double* out_errs, double* out_shift_means, void* workspace, size_t workspace_bytes,
                                       void* cuda_stream) {
    if (!module) return QMC_ERR_NULL;
    return run_batch(count, problems, out_means, out_errs, out_shift_means, workspace, workspace_bytes,
                     static_cast<cudaStream_t>(cuda_stream), kDefaultOptions, nullptr, nullptr, module);
}
int qmc_lattice_integrate_batch(int count, const qmc_problem* problems, double* out_means, double* out_errs,
                                double* out_shift_means, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    return qmc_lattice_integrate_batch_opts(count, problems, out_means, out_errs, out_shift_means, workspace, workspace_bytes,
                                            cuda_stream, nullptr);
}

// Synchronous HOST-pointer batch: every input of every problem travels in ONE host-to-device copy from the thread's pinned
// staging block, the results come back in one device-to-host copy; device memory comes from the thread's arena.
int qmc_lattice_integrate_batch_host(int count, const qmc_problem* problems, double* out_means, double* out_errs,
                                     double* out_shift_means) {
    return qmc_lattice_integrate_batch_host_module(nullptr, count, problems, out_means, out_errs, out_shift_means);
}

int qmc_lattice_integrate_batch_host_module(qmc_sector_module* module, int count, const qmc_problem* problems, double* out_means,
                                            double* out_errs, double* out_shift_means) {
    if (count < 1) return QMC_ERR_N;
    if (!problems || !out_means || !out_errs) return QMC_ERR_NULL;
    int max_m = 0;
    size_t in_bytes = 0;
    for (int i = 0; i < count; ++i) {
        const int vst = validate_values(problems[i]);
        if (vst != QMC_OK) return vst;
        const qmc_problem& p = problems[i];
        max_m = std::max(max_m, p.m);
        in_bytes += align_up((size_t)p.n_params * 8, 256) + align_up((size_t)p.dim * 8, 256) + align_up((size_t)p.m * p.dim * 8, 256) +
                    (p.fit_coeffs ? align_up((size_t)p.dim * 6 * 8, 256) : 0);
    }
    const size_t out_doubles = (size_t)count * (4 + 2 * (size_t)max_m);     // means (2), errs (2), shift means (2 max_m) per problem
    const size_t out_bytes = align_up(out_doubles * 8, 256);
    Plan plan;
    const int pst = make_plan(count, problems, true, &plan, kDefaultOptions, module);
    if (pst != QMC_OK) return pst;
    const size_t blob_bytes = align_up(plan.off_aux - plan.off_counters, 256);
    const int ast = arena_reserve(in_bytes + blob_bytes + out_bytes, in_bytes + plan.total + 256);
    if (ast != QMC_OK) return ast;
    char* h_in = g_ts.pinned;                         // [inputs | plan blob | results]
    char* h_blob = h_in + in_bytes;
    char* h_out = h_blob + blob_bytes;
    char* d_in = g_ts.device;
    // the finalize kernel writes the results (a few KB) straight into the mapped staging block: no device-to-host copy to wait for
    double* d_out = nullptr;
    QMC_CUDA(cudaHostGetDevicePointer(reinterpret_cast<void**>(&d_out), h_out, 0));
    char* d_ws = d_in + in_bytes;
    size_t off = 0;
    for (int i = 0; i < count; ++i) {
        const qmc_problem& p = problems[i];
        auto put = [&](const void* src, size_t bytes) {
            std::memcpy(h_in + off, src, bytes);
            const char* dev = d_in + off;
            off += align_up(bytes, 256);
            return dev;
        };
        DevProblem& d = plan.dev[i];                         // planned from the HOST structs: redirect the data pointers to the device copies
        d.params = reinterpret_cast<const double*>(put(p.params, (size_t)p.n_params * 8));
        d.z = reinterpret_cast<const unsigned long long*>(put(p.z, (size_t)p.dim * 8));
        d.shifts = reinterpret_cast<const double*>(put(p.shifts, (size_t)p.m * p.dim * 8));
        d.fit = p.fit_coeffs ? reinterpret_cast<const double*>(put(p.fit_coeffs, (size_t)p.dim * 6 * 8)) : nullptr;
    }
    cudaStream_t st = 0;
    double* d_means = d_out;
    double* d_errs = d_out + (size_t)count * 2;
    double* d_sm = d_out + (size_t)count * 4;
    QMC_CUDA(cudaMemcpyAsync(d_in, h_in, in_bytes, cudaMemcpyHostToDevice, st));
    const int status = run_batch(count, problems, d_means, d_errs, d_sm, d_ws, plan.total, st, kDefaultOptions, h_blob, &plan, module);
    if (status != QMC_OK) { cudaStreamSynchronize(st); return status; }
    QMC_CUDA(cudaStreamSynchronize(st));
    const double* r = reinterpret_cast<const double*>(h_out);
    bool finite = true;
    for (int i = 0; i < count; ++i) {
        const int nc = ncomp_of(problems[i].family);
        for (int c = 0; c < 2; ++c) {
            out_means[(size_t)i * 2 + c] = r[(size_t)i * 2 + c];
            out_errs[(size_t)i * 2 + c] = r[(size_t)count * 2 + (size_t)i * 2 + c];
            if (c < nc) finite = finite && std::isfinite(out_means[(size_t)i * 2 + c]) && std::isfinite(out_errs[(size_t)i * 2 + c]);
        }
    }
    if (out_shift_means) std::memcpy(out_shift_means, r + (size_t)count * 4, (size_t)count * 2 * max_m * 8);
    return finite ? QMC_OK : QMC_ERR_NONFINITE;
}

int qmc_lattice_integrate_ex(int family, const double* params, int n_params, int dim, uint64_t n, const uint64_t* z,
                             const double* shifts, int m, int transform, const double* fit_coeffs, double* out_mean,
                             double* out_err, double* out_shift_means) {
    if (!params || !z || !shifts || !out_mean || !out_err) return QMC_ERR_NULL;
    qmc_problem hp;
    hp.family = family; hp.dim = dim; hp.m = m; hp.transform = transform; hp.n = n;
    hp.params = params; hp.n_params = n_params; hp.z = z; hp.shifts = shifts; hp.fit_coeffs = fit_coeffs;
    const int vst = validate_values(hp);                       // before the arrays below are sized from m
    if (vst != QMC_OK) return vst;
    double means[2], errs[2];
    std::vector<double> sm(out_shift_means ? (size_t)2 * m : 0);
    const int st = qmc_lattice_integrate_batch_host(1, &hp, means, errs, out_shift_means ? sm.data() : nullptr);
    if (st != QMC_OK && st != QMC_ERR_NONFINITE) return st;
    const int nc = ncomp_of(family);
    for (int c = 0; c < nc; ++c) { out_mean[c] = means[c]; out_err[c] = errs[c]; }
    if (out_shift_means)
        for (int i = 0; i < m * nc; ++i) out_shift_means[i] = sm[i];
    return st;
}

// Inspection: the interpreter program the device-side compiler makes of a sector parameter block (qmc_sector.cuh).
int qmc_sector_compile(const double* params, int n_params, int dim, unsigned char* out_steps, int steps_cap, int* out_n_steps,
                       double* out_slots, int slots_cap, int* out_n_slots, double* out_c0) {
    if (!params || !out_n_steps || !out_n_slots || !out_c0) return QMC_ERR_NULL;
    if (dim < 1 || dim > 16) return QMC_ERR_DIM;
    // a one-point problem around the block: only the struct-level checks and the program matter here
    const uint64_t z1[16] = {1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1};
    std::vector<double> sh((size_t)2 * dim, 0.25);
    qmc_problem hp;
    hp.family = QMC_FAMILY_SECTOR; hp.dim = dim; hp.m = 2; hp.transform = QMC_TRANSFORM_NONE; hp.n = 2;
    hp.params = params; hp.n_params = n_params; hp.z = z1; hp.shifts = sh.data(); hp.fit_coeffs = nullptr;
    Plan plan;
    const int pst = make_plan(1, &hp, true, &plan);
    if (pst != QMC_OK) return pst;
    const size_t b_params = align_up((size_t)n_params * 8, 256), b_z = 256;
    const size_t blob_bytes = align_up(plan.off_aux - plan.off_counters, 256);
    const size_t prog_bytes = plan.prog_words * 8, back_bytes = align_up(sizeof(DevAux) + prog_bytes, 256);
    const int ast = arena_reserve(b_params + b_z + blob_bytes + back_bytes, b_params + b_z + plan.total + 256);
    if (ast != QMC_OK) return ast;
    char* h = g_ts.pinned;
    char* d = g_ts.device;
    std::memcpy(h, params, (size_t)n_params * 8);
    std::memcpy(h + b_params, z1, (size_t)dim * 8);
    cudaStream_t st = 0;
    QMC_CUDA(cudaMemcpyAsync(d, h, b_params + b_z, cudaMemcpyHostToDevice, st));
    DevProblem dv = plan.dev[0];
    dv.params = reinterpret_cast<const double*>(d);
    dv.z = reinterpret_cast<const unsigned long long*>(d + b_params);
    dv.shifts = reinterpret_cast<const double*>(d);            // never read by the prepare kernel
    char* ws = d + b_params + b_z;
    char* h_blob = h + b_params + b_z;
    std::memset(h_blob, 0, blob_bytes);
    std::memcpy(h_blob + (plan.off_probs - plan.off_counters), &dv, sizeof(DevProblem));
    QMC_CUDA(cudaMemcpyAsync(ws + plan.off_counters, h_blob, plan.off_aux - plan.off_counters, cudaMemcpyHostToDevice, st));
    QMC_CUDA(launch_prepare(1, st, reinterpret_cast<const DevProblem*>(ws + plan.off_probs), reinterpret_cast<DevAux*>(ws + plan.off_aux),
                            reinterpret_cast<unsigned long long*>(ws + plan.off_prog)));
    char* h_back = h_blob + blob_bytes;
    QMC_CUDA(cudaMemcpyAsync(h_back, ws + plan.off_aux, sizeof(DevAux), cudaMemcpyDeviceToHost, st));
    QMC_CUDA(cudaMemcpyAsync(h_back + sizeof(DevAux), ws + plan.off_prog, prog_bytes, cudaMemcpyDeviceToHost, st));
    QMC_CUDA(cudaStreamSynchronize(st));
    DevAux aux;
    std::memcpy(&aux, h_back, sizeof(DevAux));
    if (aux.status != 0) return aux.status;
    const int nmono = (n_params - 4 - dim) / (1 + dim);
    const double* slots = reinterpret_cast<const double*>(h_back + sizeof(DevAux));
    const unsigned char* steps = reinterpret_cast<const unsigned char*>(h_back + sizeof(DevAux)) + (size_t)sector_slot_words(nmono) * 8;
    const int n_steps = aux.sec_nops[0] * 4, n_slots = aux.sec_ncoef[0];
    *out_n_steps = n_steps;
    *out_n_slots = n_slots;
    out_c0[0] = aux.sec_c0[0]; out_c0[1] = aux.sec_c0[1];
    if (out_steps) { if (steps_cap < n_steps) return QMC_ERR_WORKSPACE; std::memcpy(out_steps, steps, (size_t)n_steps); }
    if (out_slots) { if (slots_cap < n_slots) return QMC_ERR_WORKSPACE; std::memcpy(out_slots, slots, (size_t)n_slots * 16); }
    return QMC_OK;
}

int qmc_lattice_integrate(int family, const double* params, int dim, uint64_t n, const uint64_t* z, const double* shifts,
                          int m, int transform, const double* fit_coeffs, double* out_mean, double* out_err) {
    if (!params) return QMC_ERR_NULL;
    if (ncomp_of(family) < 0) return QMC_ERR_FAMILY;
    if (dim < 1 || dim > QMC_MAX_DIM) return QMC_ERR_DIM;
    const int n_params = family_param_count(family, params, dim);
    if (n_params < 0) return QMC_ERR_PARAMS;
    return qmc_lattice_integrate_ex(family, params, n_params, dim, n, z, shifts, m, transform, fit_coeffs, out_mean, out_err,
                                    nullptr);
}

int qmc_finalize_means(const double* shift_means, int m, int ncomp, double* out_mean, double* out_err, void* cuda_stream) {
    if (!shift_means || !out_mean || !out_err) return QMC_ERR_NULL;
    if (m < 2 || m > QMC_MAX_M) return QMC_ERR_M;
    if (ncomp < 1 || ncomp > 2) return QMC_ERR_FAMILY;
    QMC_CUDA(launch_finalize_means(static_cast<cudaStream_t>(cuda_stream), shift_means, m, ncomp, out_mean, out_err));
    return QMC_OK;
}

int qmc_lattice_points(uint64_t n, int dim, const uint64_t* z, const double* shift, uint64_t k0, uint64_t count,
                       uint64_t* out_r, double* out_u, void* cuda_stream) {
    if (!z || !shift) return QMC_ERR_NULL;
    if (dim < 1 || dim > QMC_MAX_DIM) return QMC_ERR_DIM;
    if (n < 2 || n >= (1ull << 53)) return QMC_ERR_N;
    PointsArgs a;
    std::memset(&a, 0, sizeof(a));
    for (int j = 0; j < dim; ++j) {
        if (z[j] < 1 || z[j] >= n || gcd_u64(z[j], n) != 1) return QMC_ERR_Z;
        if (!(shift[j] >= 0.0 && shift[j] < 1.0)) return QMC_ERR_SHIFT;
        a.z[j] = z[j];
        a.shift[j] = shift[j];
    }
    a.n = n; a.k0 = k0; a.count = count; a.inv_n = 1.0 / (double)n; a.dim = dim;
    a.out_r = reinterpret_cast<unsigned long long*>(out_r);
    a.out_u = out_u;
    const int sms = sm_count();
    if (sms <= 0) return cuda_fail(cudaErrorNoDevice, "no CUDA device");
    QMC_CUDA(launch_points(static_cast<cudaStream_t>(cuda_stream), a, sms));
    return QMC_OK;
}

int qmc_fp64_peak_probe(int iters, double* out_rate, double* out_ms, void* cuda_stream) {
    if (!out_rate) return QMC_ERR_NULL;
    if (iters < 1) return QMC_ERR_N;
    const int sms = sm_count();
    if (sms <= 0) return cuda_fail(cudaErrorNoDevice, "no CUDA device");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int blocks = sms * 8;
    double* buf = nullptr;
    QMC_CUDA(cudaMalloc(reinterpret_cast<void**>(&buf), (size_t)blocks * 256 * 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaError_t e = launch_dfma_probe(st, buf, blocks, 16);       // warm-up
    float ms = 0.f;
    if (e == cudaSuccess) {
        cudaEventRecord(e0, st);
        e = launch_dfma_probe(st, buf, blocks, iters);
        cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) return cuda_fail(e, "dfma probe");
    const double instr = (double)blocks * 256.0 * (double)iters * 64.0;   // 8 chains x 8 unrolled, per thread per iteration
    *out_rate = instr / ((double)ms * 1e-3);
    if (out_ms) *out_ms = (double)ms;
    return QMC_OK;
}

}  // extern "C"

// (the host-side fits are in qmc_fit.cu)
