// qmc_internal.h -- types shared by the host side (qmc_host.cu) and the kernels of the CUDA path.
// Nothing here is shared with oracle/ (the CPU oracle is an independent translation unit).
#pragma once
#include <cstddef>
#include <cstdint>

#include "../../include/qmc_lattice.h"

namespace qmc {

constexpr int kThreads = 128;          // threads per CTA of the fused kernels (4 warps)
constexpr int kWarps = kThreads / 32;
constexpr int kGroup = 4;             // shifts evaluated together per lattice index (register-resident)
constexpr int kGroupWide = 8;          // ... the product-peak kernels of <= 8 dimension slots also exist with 8 (chosen by the plan from m)
constexpr bool closed_has_group8(int kernel_family, int dp, bool wide) { return kernel_family == QMC_FAMILY_GENZ_PRODPEAK && dp <= 8 && !wide; }
constexpr int kMaxSteps = 1024;        // max lattice indices per thread per tile (bounds the naive fp64 chain length)
constexpr int kPlanSMs = 148;          // the tiling is planned for a B200 (a pure function of the problem structs: results
                                       // are bit-identical on any device, only the balance is tuned for 148 SMs)
constexpr int kWavesSingle = 2;        // tiles per resident CTA when a kernel variant serves one problem (equal-cost tiles)
constexpr int kShortEvalsPerCta = 200000;   // below this many evaluations per resident CTA a single problem gets 1 tile per CTA
constexpr int kWavesBatch = 8;         // ... and when it serves a batch of unequal problems (dynamic balance)

// resident CTAs per SM each fused kernel is register-budgeted for (its __launch_bounds__ minimum)
constexpr int min_blocks_closed(int dp, bool wide) { return (dp <= 8 || (dp <= 12 && !wide)) ? 4 : (dp <= 16 ? (wide ? 2 : 3) : 2); }
constexpr int sector_group(int dp) { return dp <= 8 ? 8 : 4; }                       // shifts per group, sector family
constexpr int csector_group(int dp) { return dp <= 8 ? 4 : 2; }                      // complex sector family: paired accumulators
constexpr int kCSectorThreads = 384;
// The sector kernels run ONE CTA per SM, as large as the registers allow (x[G][DP] lives in registers): every warp of an SM then
// interprets the same program, whose cases stay in the L0 instruction cache.
__host__ __device__ constexpr int sector_threads(int dp) { return dp <= 6 ? 384 : 256; }
constexpr int min_blocks_sector(int) { return 1; }
constexpr int kDeltaCache = 768;       // doubles of shared memory per CTA that cache the shifts of all groups of a problem
constexpr int kMaxSectorMono = 64;     // monomials per polynomial
constexpr int kMaxSectorOps = 2 * kMaxSectorMono * 16 + 64;   // step bytes of a program: <= one per unit of degree (<= 16 per monomial) + end steps, padding
// coefficient region of a program in 8-byte words: one 16-byte slot {cf, cf2} per non-constant monomial, one for the end of U,
// one of read-ahead
// (complex family: 32-byte slots {cf_re, cf_im, cf2_re, cf2_im})
__host__ __device__ constexpr int sector_slot_words(int nmono, bool cplx = false) { return (cplx ? 4 : 2) * (nmono + 2); }

// kernel family of a public family id: the four remaining Genz functions share one fused kernel (runtime sub-kind); the complex
// sector family has its own
constexpr int kKernelFamilyGenzMisc = 4;
constexpr int kKernelFamilyCSector = 5;
constexpr int kKernelFamilies = 6;
__host__ __device__ constexpr int kernel_family(int family) {
    return family <= QMC_FAMILY_SECTOR ? family : (family == QMC_FAMILY_SECTOR_COMPLEX ? kKernelFamilyCSector : kKernelFamilyGenzMisc);
}
__host__ __device__ constexpr bool is_sector_family(int family) { return family == QMC_FAMILY_SECTOR || family == QMC_FAMILY_SECTOR_COMPLEX; }
// monomial record of a sector block: coefficient (re [, im]) + dim exponents
__host__ __device__ constexpr int sector_mono_stride(int family, int dim) { return (family == QMC_FAMILY_SECTOR_COMPLEX ? 2 : 1) + dim; }

// transform kinds after host-side decoding
enum : int { TR_NONE = 0, TR_BAKER = 1, TR_KOR3 = 2, TR_KORR = 3 };   // TR_KORR = the generic tile loop, see GEN_*
// template-only codes of the dedicated generic kernels (fused_generic_kernel): TR_GEN0 + GEN_* kind, kind < kGenKinds, no fit map
enum : int { TR_GEN0 = 4 };
constexpr int kGenKinds = 1;           // GEN_KOROBOV_SYM only: Korobov (r0, r1) and Sidi measured slower as one basic block
constexpr int min_blocks_generic(int dp) { return dp <= 8 ? 4 : 3; }   // resident CTAs per SM of the dedicated generic kernels
// The generic tile loop serves every transform (selected per coordinate by DevProblem::gen = kind | r0 << 4 | r1 << 8)
// and every fit mode at run time; the specialised loops are none / baker / Korobov-3 x (no fit, cubic fit).
enum : int { GEN_KOROBOV_SYM = 0, GEN_KOROBOV_ASYM = 1, GEN_SIDI = 2, GEN_NONE = 3, GEN_BAKER = 4 };
constexpr int FIT_RT = 3;              // template value "fit mode decided at run time" (0 none, 1 cubic, 2 cubic + poles)

// Device-resident description of one problem (built on the host, copied into the workspace).
struct alignas(16) DevProblem {
    const double* params;      // DEVICE, user layout
    const unsigned long long* z;
    const double* shifts;      // [m][dim]
    const double* fit;         // [dim][6] or nullptr
    unsigned long long n;
    double inv_n;              // fl(1/double(n))  (reading C-2)
    double wconst;             // Korobov: c_r^dim ; else 1
    double kor[16];            // transform tables: symmetric Korobov: centred polynomial g_r, kor[i], i <= r (degree r in c^2);
                               // asymmetric Korobov: kor[0..7] = phi series below 1/2, kor[8..15] = mirrored series above
                               // (zero padded to degree 6); Sidi: kor[0] = K_r / pi
    long long partial_off;     // offset in doubles into the partial-sum area
    long long means_off;       // offset in doubles into the per-shift means area
    long long tile_begin;      // first tile index (within this problem's kernel variant queue)
    long long tile_len;        // lattice indices per tile (the last tile is shorter); steps = ceil(tile_len / kThreads)
    int tiles;                 // number of k-tiles
    int steps;                 // I: lattice indices per thread per tile; tile length = steps*kThreads
    int family, dim, m, ncomp;
    int tr_kind;               // TR_*
    int kor_r;                 // symmetric Korobov weight r (1..6) or 0
    int has_fit;               // 0 none, 1 fit map of Eq. 19 (cubic, or with pole terms: decided on the device from a2, a3)
    int n_params;
    int aux_off;               // sector: offset (in 8-byte words) of the compiled program in the aux area
    int aux_len;
    int out_index;             // index of the problem in the caller's arrays
    int gen;                   // the transform for the generic tile loop: GEN_* | r0 << 4 | r1 << 8
    int spec_case;             // specialised sector kernel (qmc_spec.cu): the problem's case in its kernel; else 0
};

// Per-problem tables derived on the device by prepare_kernel (one record per problem).
struct alignas(16) DevAux {
    unsigned long long z[QMC_MAX_DIM];     // z_j
    unsigned long long step[QMC_MAX_DIM];  // (kThreads * z_j) mod n : residue stride between a thread's points
    unsigned long long back[QMC_MAX_DIM];  // (steps * kThreads * z_j) mod n : rewinds a thread to its first point
    double fam_a[QMC_MAX_DIM];             // per-dimension integrand constants (family dependent)
    double fam_b[QMC_MAX_DIM];
    double fit[9][QMC_MAX_DIM];            // a4, a5, a6, 2*a5, 3*a6 of the cubic part; a0, a2 (a0-1), a1, a3 (a1-1) of the poles
    double fam0;                           // OSC: 2 pi u0
    double sec_c0[2];                      // sector: constant terms of U and F (real parts)
    double sec_c0i[2];                     // complex sector: their imaginary parts
    double sec_log[2];                     // sector: lu, lf of the optional log factor (lu log U + lf log F)^p
    int sec_a, sec_b;                      // sector: powers of U and F
    int sec_logp, sec_pad_;                // sector: p of the log factor, 0 = none
    int sec_nops[2];                       // sector: [0] = 32-bit step words of the program (U, end-of-U, F)
    int sec_ncoef[2];                      // sector: [0] = coefficients of the program
    int status;                            // 0 or a qmc_status found while preparing
    int fit_full;                          // 1 if any dimension of the fit map has a pole term (a2 or a3 non-zero)
    unsigned char nu[QMC_MAX_DIM];         // sector: nu_j
};

// One kernel variant queue: the problems (indices into DevProblem[]) it serves, in queue order.
struct VariantQueue {
    const int* plist;            // DEVICE: problem indices in queue order
    const long long* tile_prefix;// DEVICE: exclusive prefix of tiles over plist, plist_len+1 entries
    int plist_len;
    long long total_tiles;
    unsigned long long* counter; // DEVICE: tile queue head (zeroed before launch)
};

// Kernel parameter of every fused kernel and of the finalize kernel (passed by value).  Queue mode: the problems
// live in the workspace and CTAs pop tiles from vq.counter.  Single mode (one closed-form problem): the problem
// travels in the parameter itself, so the call needs no workspace upload and no prepare launch; when there are no
// more tiles than resident CTAs every CTA owns tile blockIdx.x and the queue (vq.counter == nullptr) is not used.  Result slots are per tile in both modes.
struct FusedLaunch {
    const DevProblem* probs;
    const DevAux* aux;                    // sector family only
    const unsigned long long* prog;       // sector family only
    double* partials;
    VariantQueue vq;
    int single;
    int pad_;
    DevProblem one;
};

}  // namespace qmc
