/* qmc_lattice.h -- C ABI of the B200-native rank-1 shifted lattice (R1SL) integrator.
 *
 * The library computes, on one CUDA device (sm_100a), the hot path of the `qmc` integrator of
 * arXiv:1811.11720 (PAPER.md = the paper text; cited as P:L<line>):
 *
 *   Q_s   = (1/n) sum_{k=0}^{n-1} W(u_{k,s}) f(x(u_{k,s})),  u_{k,s} = { k z / n + Delta_s }   Eq. 2
 *   Qbar  = (1/m) sum_s Q_s                                                                   Eq. 2
 *   err   = sqrt( sum_s (Q_s - Qbar)^2 / (m (m-1)) )   (per component for complex f)           Eq. 3
 *
 * with x = p(phi(u)) and W = prod_j omega(u_j) p'(phi(u_j)): phi/omega a periodizing transform
 * (Eq. 12-17), p an optional per-dimension fitted inverse-CDF map (Eq. 18-19,
 * P:L215-L223; composition order P:L338).  f is a member of a parameterised integrand family (a C
 * ABI cannot carry the paper's functors).
 *
 * Conventions
 *  - every function returns a qmc_status (0 = OK, negative = error); on an argument error no output
 *    is written and nothing is launched;
 *  - the caller owns every buffer passed in; the library may be called from several host threads on different
 *    streams and devices.  What it keeps between calls is (i) PER HOST THREAD: the text of the last CUDA error, the
 *    launch count and the profiling events of the measurement helpers, and the staging arena (one pinned host block,
 *    one device block, grown on demand) of the synchronous HOST-pointer entries -- all released by
 *    qmc_release_thread_resources() and at thread exit; (ii) per device ordinal: cached immutable attributes (SM count,
 *    resident CTAs of each kernel).  The stream-ordered entries allocate nothing and read no environment variables;
 *  - "HOST" / "DEVICE" beside a pointer says which address space it must point to;
 *  - there is no CPU fallback: without a CUDA device every compute entry returns QMC_ERR_CUDA.
 *
 * Layouts
 *  - z[j], j < dim: generating vector, 1 <= z_j < n, gcd(z_j, n) = 1 ("coprime to n");
 *  - shifts[s*dim + j] in [0,1): shift s, dimension j (Delta_k of Eq. 2);
 *  - fit_coeffs[j*6 + i] = a_i of Eq. 19 for dimension j, a_6 := 1-a_2-a_3-a_4-a_5
 *    (cubic map <=> a_2 = a_3 = 0; then a_0, a_1 are ignored; with pole terms a_0 >= 1.001, a_1 <= -0.001, a_2, a_3 >= 0,
 *    P:L231); the map must be increasing on [0,1]; NULL = no fit map;
 *  - complex results are interleaved (re, im);
 *  - params: packed per family, all doubles (small integers stored as exact doubles):
 *      QMC_FAMILY_GENZ_OSC      [u0, a_1..a_d]            f = cos(2 pi u0 + sum a_j x_j)
 *      QMC_FAMILY_GENZ_PRODPEAK [c_1..c_d, w_1..w_d]      f = prod 1/(c_j^-2 + (x_j-w_j)^2)
 *      QMC_FAMILY_CEXP_POLY     [a_1..a_d, b_1..b_d]      f = exp(i sum a_j x_j) prod(1+b_j x_j)  (complex)
 *      QMC_FAMILY_GENZ_CORNER   [c_1..c_d]                f = (1 + sum c_j x_j)^-(d+1)
 *      QMC_FAMILY_GENZ_GAUSSIAN [c_1..c_d, w_1..w_d]      f = exp(-sum c_j^2 (x_j-w_j)^2)
 *      QMC_FAMILY_GENZ_C0       [c_1..c_d, w_1..w_d]      f = exp(-sum c_j |x_j-w_j|)
 *      QMC_FAMILY_GENZ_DISCONT  [c_1..c_d, w_1, w_2]      f = 0 if x_1 > w_1 or x_2 > w_2, else exp(sum c_j x_j)
 *                               (d = 1: [c_1, w_1])
 *      QMC_FAMILY_SECTOR        [a, b, nU, nF, nu_1..nu_d, cU_1..cU_nU, eU_{1,1}..eU_{nU,d},
 *                                cF_1..cF_nF, eF_{1,1}..eF_{nF,d}]
 *                               f = prod x_j^nu_j * U(x)^a / F(x)^b, U = sum_t cU_t prod_j x_j^eU_{t,j}
 *                               (sector-decomposed shape); limits: dim <= QMC_MAX_SECTOR_DIM = 16 (the coordinates
 *                               of G points live in registers), 0 <= a,b <= 8, nu_j <= 8, nU,nF in 1..64,
 *                               exponents <= 8, total degree of a monomial <= 16 -- every block within these limits is
 *                               accepted (the interpreter program holds up to 128 monomials of degree 16).
 *                               Optional trailing block [lu, lf, p] (n_params = the above + 3):
 *                               f * (lu log U + lf log F)^p, p an integer in 1..4 -- the shape of the order-eps^p
 *                               term of U^(a + lu eps) / F^(b - lf eps) in the eps-expansion of a sector;
 *                               U, F > 0 is the caller's responsibility (a non-positive value gives NaN results).
 *                               Entry points that take n_params accept it; qmc_lattice_integrate, which derives
 *                               n_params from (family, dim, params), reads the block without it.
 *      QMC_FAMILY_SECTOR_COMPLEX [a, b, nU, nF, nu_1..nu_d, Re cU_1..nU, Im cU_1..nU, eU_{1,1}..eU_{nU,d},
 *                                 Re cF_1..nF, Im cF_1..nF, eF_{1,1}..eF_{nF,d}]     (complex results)
 *                               the same f with COMPLEX coefficients on the real cube: the shape of a sector after the
 *                               contour deformation x_j -> x_j - i lambda_j x_j (1 - x_j) dF/dx_j that handles integrable
 *                               singularities -- U, F and the Jacobian of the deformed integrand are polynomials
 *                               in the real x with complex coefficients (reading C-16).  Same limits as
 *                               QMC_FAMILY_SECTOR; F(x) != 0 on the cube is the caller's responsibility.  Optional
 *                               trailing [lu, lf, p]: f * (lu Log U + lf Log F)^p with the principal branch
 *                               Log z = log|z| + i arg z, arg in (-pi, pi].
 */
#ifndef QMC_LATTICE_H
#define QMC_LATTICE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    QMC_OK = 0,
    QMC_ERR_NULL = -1,       /* a required pointer is NULL */
    QMC_ERR_DIM = -2,        /* dim outside 1..QMC_MAX_DIM (1..QMC_MAX_SECTOR_DIM for QMC_FAMILY_SECTOR) */
    QMC_ERR_N = -3,          /* n outside 2 .. 2^53-1 (double(r) must be exact), or count/bins invalid */
    QMC_ERR_Z = -4,          /* z_j outside [1, n-1] or not coprime to n */
    QMC_ERR_SHIFT = -5,      /* a shift outside [0,1) or not finite */
    QMC_ERR_M = -6,          /* m < 2 (Eq. 3 divides by m-1) or m > QMC_MAX_M */
    QMC_ERR_TRANSFORM = -7,  /* unknown transform id / Korobov weight outside 1..6 */
    QMC_ERR_FAMILY = -8,     /* unknown family id */
    QMC_ERR_PARAMS = -9,     /* n_params does not match the family layout, or a value is out of range */
    QMC_ERR_FIT = -10,       /* fit map not monotone on [0,1] or parameters outside P:L231's bounds */
    QMC_ERR_WORKSPACE = -11, /* workspace NULL, misaligned (256 B) or too small */
    QMC_ERR_CUDA = -12,      /* CUDA runtime error (qmc_last_cuda_error() has the text) */
    QMC_ERR_NONFINITE = -13  /* a result is NaN/Inf (synchronous entry only; results are still written) */
} qmc_status;

enum { QMC_FAMILY_GENZ_OSC = 0, QMC_FAMILY_GENZ_PRODPEAK = 1, QMC_FAMILY_CEXP_POLY = 2, QMC_FAMILY_SECTOR = 3,
       /* the remaining functions of Genz' test suite: */
       QMC_FAMILY_GENZ_CORNER = 4, QMC_FAMILY_GENZ_GAUSSIAN = 5, QMC_FAMILY_GENZ_C0 = 6, QMC_FAMILY_GENZ_DISCONT = 7,
       /* sector polynomials with complex coefficients (complex results): */
       QMC_FAMILY_SECTOR_COMPLEX = 8 };

/* Periodizing transforms, Table A.2: none; baker Eq. 17;
 * Korobov with symmetric weight r, Eq. 15: QMC_TRANSFORM_KOROBOV + r, r = 1..6;
 * Sidi with weight r, Eq. 16: QMC_TRANSFORM_SIDI + r, r = 1..6;
 * Korobov with weights (r0, r1), Eq. 15: QMC_TRANSFORM_KOROBOV_ASYM + 16 r0 + r1, r0, r1 = 1..6 (Korobov<5,3>). */
enum { QMC_TRANSFORM_NONE = 0, QMC_TRANSFORM_BAKER = 1, QMC_TRANSFORM_KOROBOV = 100, QMC_TRANSFORM_SIDI = 200,
       QMC_TRANSFORM_KOROBOV_ASYM = 1000 };

enum { QMC_MAX_DIM = 32, QMC_MAX_M = 4096, QMC_MAX_SECTOR_DIM = 16 /* QMC_FAMILY_SECTOR only */ };

/* One integration problem.  In qmc_lattice_integrate_batch / qmc_lattice_project the four data
 * pointers are DEVICE pointers; the struct array itself is HOST memory. */
typedef struct {
    int family;               /* QMC_FAMILY_* */
    int dim;                  /* d, 1..QMC_MAX_DIM */
    int m;                    /* number of random shifts, >= 2 */
    int transform;            /* QMC_TRANSFORM_* */
    uint64_t n;               /* lattice size (need not be prime, Fig. 1 uses 55) */
    const double* params;     /* DEVICE, n_params doubles, family layout above */
    int n_params;
    const uint64_t* z;        /* DEVICE, dim entries */
    const double* shifts;     /* DEVICE, m*dim entries */
    const double* fit_coeffs; /* DEVICE, dim*6 entries, or NULL */
} qmc_problem;

/* Synchronous convenience call, HOST pointers only (north_star's argument list).  Validates all
 * values (including gcd(z_j,n) = 1, shifts in [0,1), monotone fit map), copies the inputs to the
 * device, runs the fused kernel + finalize on the default stream of the current device, copies the
 * results back and synchronises.  out_mean / out_err: 1 double (real families) or 2 (re, im).
 * n_params is implied by (family, dim, params).  Eq. 2-3. */
int qmc_lattice_integrate(int family, const double* params /*HOST*/, int dim, uint64_t n,
                          const uint64_t* z /*HOST*/, const double* shifts /*HOST [m][dim]*/, int m,
                          int transform, const double* fit_coeffs /*HOST [dim][6] or NULL*/,
                          double* out_mean /*HOST*/, double* out_err /*HOST*/);

/* As above, additionally returning the per-shift means Q_s (HOST, m*ncomp doubles, may be NULL). */
int qmc_lattice_integrate_ex(int family, const double* params, int n_params, int dim, uint64_t n,
                             const uint64_t* z, const double* shifts, int m, int transform,
                             const double* fit_coeffs, double* out_mean, double* out_err,
                             double* out_shift_means /*HOST or NULL*/);

/* Stream-ordered batched call: `count` problems of arbitrary, unequal cost in ONE persistent-grid
 * launch per kernel variant (device-side tile queue; the paper's host-side work queue is P:L388-L402) followed by
 * one finalize launch.  Never waits for the device: a call for one closed-form problem is kernel launches (and at most
 * one 8-byte memset) only and can be captured in a CUDA graph; a batch call also issues one cudaMemcpyAsync of its launch
 * plan (KBs) from pageable host memory, which the runtime stages before the call returns.  problems: HOST array whose data pointers are DEVICE
 * pointers (only the struct fields are validated here; the pointed-to values are the caller's
 * responsibility -- use qmc_validate_problem_host before uploading).
 *   out_means, out_errs : DEVICE, count*2 doubles: [p*2 + c], c = 0 (re) / 1 (im, 0 for real families)
 *   out_shift_means     : DEVICE or NULL, count*stride doubles, stride = 2*max_m:
 *                         [p*stride + s*ncomp + c]
 *   workspace           : DEVICE, 256-byte aligned, >= qmc_workspace_bytes(count, problems) bytes;
 *                         contents are scratch (per-tile partial sums in fixed slots: results do not
 *                         depend on the scheduling order, the grid size or the device's SM count).
 */
int qmc_lattice_integrate_batch(int count, const qmc_problem* problems /*HOST*/, double* out_means /*DEVICE*/,
                                double* out_errs /*DEVICE*/, double* out_shift_means /*DEVICE or NULL*/,
                                void* workspace /*DEVICE*/, size_t workspace_bytes, void* cuda_stream);

/* Bytes of workspace qmc_lattice_integrate_batch / qmc_lattice_project need (0 on invalid input). */
size_t qmc_workspace_bytes(int count, const qmc_problem* problems /*HOST*/);

/* Launch-plan options for tests and tuning (zero-initialise for the library's plan): the same calls with an options
 * struct.  tiles_target > 0: that many tiles per kernel variant instead of the planned count (S9; results are
 * bit-identical only for equal tilings); force_wide != 0: the 64-bit-residue kernels even for n < 2^31 (they are
 * otherwise reached only by n >= 2^31; results are bit-identical to the 32-bit kernels); group = 4 or 8: shifts evaluated per
 * lattice index by the product-peak kernels of <= 8 dimension slots (0: the plan chooses from m; other kernels ignore it; the
 * per-shift results do not depend on it bit for bit); generic_call != 0: Korobov r != 3, Korobov (r0, r1) and Sidi run the
 * generic loop inside the family's kernel even where a dedicated kernel exists (no fit map, n < 2^31, dim <= 16). */
typedef struct { int tiles_target; int force_wide; int group; int generic_call; } qmc_plan_options;
int qmc_lattice_integrate_batch_opts(int count, const qmc_problem* problems /*HOST*/, double* out_means /*DEVICE*/,
                                     double* out_errs /*DEVICE*/, double* out_shift_means /*DEVICE or NULL*/,
                                     void* workspace /*DEVICE*/, size_t workspace_bytes, void* cuda_stream,
                                     const qmc_plan_options* opts /*HOST or NULL*/);
size_t qmc_workspace_bytes_opts(int count, const qmc_problem* problems /*HOST*/, const qmc_plan_options* opts /*HOST or NULL*/);

/* Synchronous batched call, HOST pointers everywhere (problems[i].params / z / shifts / fit_coeffs included): full value
 * validation of every problem, ONE host-to-device copy of all inputs from the calling thread's pinned staging block, the
 * batched hot path on the default stream of the current device -- its last kernel writes the results into the same (mapped)
 * staging block -- synchronise, copy out of the staging block.
 *   out_means, out_errs : HOST, count*2 doubles [p*2 + c]
 *   out_shift_means     : HOST or NULL, count * 2*max_m doubles [p*(2 max_m) + s*ncomp + c], max_m = largest m of the batch
 * Returns QMC_ERR_NONFINITE (results still written) if a result is NaN/Inf. */
int qmc_lattice_integrate_batch_host(int count, const qmc_problem* problems /*HOST, HOST data pointers*/,
                                     double* out_means /*HOST*/, double* out_errs /*HOST*/, double* out_shift_means /*HOST or NULL*/);

/* Releases what the calling host thread holds (profiling events, staging arena); also done at thread exit. */
int qmc_release_thread_resources(void);

/* Full value validation of one problem whose data pointers are HOST pointers. */
int qmc_validate_problem_host(const qmc_problem* p /*HOST, HOST data pointers*/);

/* Projection pass for the variance-reduction fit (Eq. 20; reading C-8):
 * transform None, weight 1, the first shift of p only, all n lattice points:
 *   out_hist[j*bins + b] = sum_k |f(x_k)| [ floor(bins * x_{k,j}) == b ]     (|f| = modulus if complex)
 * Stream-ordered, deterministic.  p: HOST struct with DEVICE data pointers (p->m >= 1 here,
 * p->transform and p->fit_coeffs are ignored).  bins in 2..1024.  out_hist: DEVICE, dim*bins. */
int qmc_lattice_project(const qmc_problem* p /*HOST*/, int bins, double* out_hist /*DEVICE*/,
                        void* workspace /*DEVICE*/, size_t workspace_bytes, void* cuda_stream);
size_t qmc_project_workspace_bytes(const qmc_problem* p /*HOST*/, int bins);

/* Host-side closed-form least squares for the cubic sub-family of Eq. 19 (a_2 = a_3 = 0): with
 * c_b the CDF of hist at the bin edges e_b = b/bins, minimise sum_b (p(c_b) - e_b)^2 over (a_4, a_5);
 * identity map if the minimiser is not safely monotone (min p' <= 0.05).  hist, fit_coeffs: HOST. */
int qmc_fit_cubic(const double* hist /*HOST [dim][bins]*/, int dim, int bins, double* fit_coeffs /*HOST [dim][6]*/);

/* Host-side fit of the COMPLETE fit function of Eq. 19 (two pole terms + cubic) to the same data: bounded
 * Levenberg-Marquardt on (a_0..a_5) with a_0 >= 1.001, a_1 <= -0.001, a_2, a_3 >= 0 (the paper uses GSL), started from
 * the cubic solution; the cubic result is kept for a dimension unless the full function is a strictly better fit that is
 * increasing on [0,1].  bins in 8..1024.  hist, fit_coeffs: HOST.  The result is valid input for every compute entry. */
int qmc_fit_polysingular(const double* hist /*HOST [dim][bins]*/, int dim, int bins, double* fit_coeffs /*HOST [dim][6]*/);

/* The paper's own CDF sampling for the fit (`evaluate`; fitstepsize; DESIGN.md reading
 * C-8b): |f| on the n points of the lattice shifted by the first shift of p (transform None, weight 1); per dimension j the
 * samples sorted by x_j, the running sum of |f| over the sorted samples divided by the total, every fitstepsize-th sorted sample
 * kept: for t = 1..K, K = n / fitstepsize (qmc_cdf_sample_count),
 *   out_x[j*K + t-1]   = the (t * fitstepsize)-th smallest coordinate x_j of the lattice,
 *   out_cdf[j*K + t-1] = sum of |f| over the t * fitstepsize samples with the smallest x_j / sum over all samples.
 * No sort is performed: in one dimension the sorted order of a shifted rank-1 lattice is the cyclic order of its residues, so
 * every sample is scattered to its rank.  Stream-ordered, deterministic.  p: HOST struct with DEVICE data pointers (p->m >= 1;
 * transform and fit_coeffs ignored).  out_x, out_cdf: DEVICE, dim*K doubles.  A sector block that fails the device-side
 * validation gives NaN outputs. */
int qmc_lattice_cdf_samples(const qmc_problem* p /*HOST*/, int fitstepsize, double* out_x /*DEVICE*/, double* out_cdf /*DEVICE*/,
                            void* workspace /*DEVICE*/, size_t workspace_bytes, void* cuda_stream);
size_t qmc_cdf_workspace_bytes(const qmc_problem* p /*HOST*/, int fitstepsize);
long long qmc_cdf_sample_count(uint64_t n, int fitstepsize);        /* K; 0 if fitstepsize is outside 1..n */

/* Host-side fits from those samples: pairs (CDF_t, x_t), p(CDF_t) ~ x_t.  with_poles = 0: cubic sub-family, closed-form least
 * squares (identity map if not safely monotone); 1: the complete fit function of Eq. 19 by the bounded Levenberg-Marquardt of
 * qmc_fit_polysingular.  x, cdf: HOST [dim][count]; count >= 8. */
int qmc_fit_from_cdf(const double* x /*HOST*/, const double* cdf /*HOST*/, int dim, long long count, int with_poles,
                     double* fit_coeffs /*HOST [dim][6]*/);

/* Inspection: residues r = (k z_j) mod n and coordinates u = {r/n + shift_j} for k = k0..k0+count-1,
 * produced by the same device code the fused kernel uses (Eq. 2; fp64 realisation:
 * u = wrap(fma(double(r), 1/double(n), shift_j)), reading C-2).
 * z, shift: HOST.  out_r [count][dim], out_u [count][dim]: DEVICE (either may be NULL). */
int qmc_lattice_points(uint64_t n, int dim, const uint64_t* z /*HOST*/, const double* shift /*HOST [dim]*/,
                       uint64_t k0, uint64_t count, uint64_t* out_r /*DEVICE*/, double* out_u /*DEVICE*/,
                       void* cuda_stream);

/* Finalize stage alone (Eq. 2 outer mean + Eq. 3) on DEVICE per-shift means [m][ncomp]:
 * out_mean, out_err DEVICE, ncomp doubles each.  Stream-ordered. */
int qmc_finalize_means(const double* shift_means /*DEVICE*/, int m, int ncomp, double* out_mean /*DEVICE*/,
                       double* out_err /*DEVICE*/, void* cuda_stream);

/* The paper's `integrate` iteration (section 3.3.1; fields P:L887-L920; result P:L988-L995) around the
 * fused hot path (synchronous; device memory is allocated for the duration of the call only): sample min_m shifted copies of the smallest ladder lattice with n >= min_n; if the error goal
 *     err <= max(epsabs, epsrel * |E|)                                  (per component for complex)
 * is not met, DISCARD the result and take a larger lattice; stop when the goal is met or `maxeval`
 * evaluations have been spent; when the ladder is exhausted keep the largest lattice and add shifts
 * (Monte Carlo scaling) up to max_m.  The paper does not say how the next lattice is chosen (DESIGN.md reading
 * C-14): the smallest ladder n >= n * max(2, err / goal) (assumes >= 1/n error scaling), limited to what `maxeval` still
 * allows; a lattice is only tried if min_m samples of it fit the remaining budget (otherwise shifts are added to the current
 * lattice while they fit), so only the first lattice can take `evaluations` past maxeval.  All pointers HOST.
 *   ladder_n[i] ascending, ladder_z[i*dim + j] the generating vector of lattice i (an INPUT: P:L940-L942)
 *   shifts[max_m][dim]: the first m rows are used for a lattice sampled with m shifts
 *   errormode: 0 = all components, 1 = largest component (ignored for real families)
 * Returns QMC_OK when the goal was met, QMC_ERR_MAXEVAL (result still written) when it was not. */
typedef struct {
    double integral[2];       /* estimate (re, im); im = 0 for real families */
    double error[2];          /* error estimate per component (Eq. 3) */
    uint64_t n;               /* size of the last (largest) lattice used */
    int m;                    /* shifts of that lattice */
    int iterations;           /* lattices sampled + shift extensions */
    uint64_t evaluations;     /* integrand evaluations over all iterations */
} qmc_result;
enum { QMC_ERR_MAXEVAL = -14 };
int qmc_integrate(int family, const double* params /*HOST*/, int n_params, int dim, int transform,
                  const double* fit_coeffs /*HOST or NULL*/, int n_lattices, const uint64_t* ladder_n /*HOST*/,
                  const uint64_t* ladder_z /*HOST [n_lattices][dim]*/, const double* shifts /*HOST [max_m][dim]*/,
                  uint64_t min_n, int min_m, int max_m, double epsrel, double epsabs, uint64_t maxeval, int errormode,
                  qmc_result* out /*HOST*/);

/* The same iteration for MANY integrands at once (the batched counterpart of qmc_integrate; all pointers HOST, synchronous, default
 * stream of the current device).  Every integrand follows qmc_integrate's rules on its own -- first lattice, enlargement by the
 * error ratio, shift extension at the end of the ladder, maxeval per integrand -- but the lattice evaluations of one round, each
 * integrand on its own current lattice and shift range, share ONE batched launch of the fused kernels, and a round costs one
 * device-to-host copy and one synchronisation for all integrands.  With `module` (built from these integrands in this order:
 * qmc_sector_module_create reads family, dim, n_params, params of a qmc_problem) the sectors run as compiled code; NULL = the
 * default kernels.
 *   integrands[p]    : family, dim, transform, n_params, params (HOST), fit_coeffs (HOST [dim][6] or NULL)
 *   ladder_z, shifts : [n_lattices][ladder_dim] and [max_m][ladder_dim], ladder_dim >= every dim; an integrand of dimension d uses
 *                      the first d components of each (generating vectors built component by component are nested this way)
 *   out[p], out_status[p] : the result qmc_integrate would return for integrand p and its status (QMC_OK, QMC_ERR_MAXEVAL,
 *                      QMC_ERR_NONFINITE)
 * Returns QMC_OK if every integrand met its goal, else QMC_ERR_NONFINITE if one produced a non-finite value, else
 * QMC_ERR_MAXEVAL; argument and validation errors (nothing launched, out untouched) as qmc_integrate. */
typedef struct {
    int family, dim, transform, n_params;
    const double* params;      /* HOST */
    const double* fit_coeffs;  /* HOST [dim][6] or NULL */
} qmc_integrand;
typedef struct qmc_sector_module qmc_sector_module;
int qmc_integrate_batch(int count, const qmc_integrand* integrands /*HOST*/, qmc_sector_module* module /*or NULL*/, int n_lattices,
                        const uint64_t* ladder_n /*HOST*/, const uint64_t* ladder_z /*HOST*/, int ladder_dim,
                        const double* shifts /*HOST*/, uint64_t min_n, int min_m, int max_m, double epsrel, double epsabs,
                        uint64_t maxeval, int errormode, qmc_result* out /*HOST [count]*/, int* out_status /*HOST [count]*/);

/* Measurement helper: runs a DFMA-chain kernel (8 independent chains per thread, full occupancy)
 * for `iters` iterations on `cuda_stream`, synchronises, and returns the sustained thread-level
 * FP64 instruction rate in instructions/second through *out_rate (HOST) and the kernel time in ms
 * through *out_ms (HOST, may be NULL).  This is the denominator of the FP64 issue-rate roofline. */
int qmc_fp64_peak_probe(int iters, double* out_rate /*HOST*/, double* out_ms /*HOST or NULL*/, void* cuda_stream);

/* Number of fused-kernel launches + finalize launches the last batch call of this thread issued
 * (for the benchmark's gpu_launches accounting). */
int qmc_last_launch_count(void);

/* Measurement helper: with profiling enabled (per host thread), qmc_lattice_integrate_batch brackets its
 * fused-kernel launches (not prepare / finalize) with CUDA events on the caller's stream;
 * qmc_profile_last_fused_ms synchronises on the closing event of the LAST batch call of this thread and
 * returns the device time of the fused kernels in milliseconds (QMC_ERR_N if nothing was recorded). */
int qmc_profile_enable(int on);
int qmc_profile_last_fused_ms(double* out_ms /*HOST*/);

/* Launch geometry the library uses for a batch (for DESIGN.md / bench reporting): tiles, CTAs,
 * k indices per tile of problem 0.  Any pointer may be NULL. */
int qmc_plan_info(int count, const qmc_problem* problems /*HOST*/, long long* out_tiles, int* out_ctas,
                  long long* out_tile_len0);

/* Inspection: the interpreter program the device-side compiler makes of a QMC_FAMILY_SECTOR parameter block (all pointers
 * HOST; synchronous).  out_steps: n_steps one-byte step codes (0 no-op, 1 end of U, 2 end, 3 + 5 j + kind with kind
 * 0 SC: S = fma(A, x_j, S), 1 SL: S = fma(cf, x_j, S), 2 AL: A = fma(cf, x_j, A), 3 ALI: A = fma(cf, x_j, cf2), 4 AM: A = A x_j);
 * out_slots: n_slots pairs {cf, cf2}, one per SL / AL / ALI / end-of-U step in program order (the end-of-U slot holds F's
 * constant term) plus one of read-ahead; out_c0: constant terms of U and F.  out_steps / out_slots may be NULL (counts only);
 * QMC_ERR_WORKSPACE if a capacity is too small. */
int qmc_sector_compile(const double* params /*HOST*/, int n_params, int dim, unsigned char* out_steps /*HOST or NULL*/,
                       int steps_cap, int* out_n_steps /*HOST*/, double* out_slots /*HOST or NULL*/, int slots_cap,
                       int* out_n_slots /*HOST*/, double* out_c0 /*HOST [2]*/);

/* ---- modules of specialised sector kernels ------------------------------------------------------------------------------
 * The paper's integrands are compiled functions (every sector is C++ source compiled for the GPU before the
 * integration starts).  A C ABI carries parameter blocks instead, which the default kernels interpret step by step; a MODULE
 * gives the compiled route back: qmc_sector_module_create translates every QMC_FAMILY_SECTOR and QMC_FAMILY_SECTOR_COMPLEX
 * problem of a batch into
 * straight-line sm_100a code -- the same operations in the same order as the interpreting kernel, so both return the same bits --
 * inside copies of the fused kernel (up to `sectors_per_kernel` sectors per kernel; 0 = 32, doubled until the batch needs at most
 * 48 kernels; a batch call serves at most 64 kernel variants in all and returns QMC_ERR_WORKSPACE beyond),
 * assembled on the HOST with the CUDA toolkit's nvJitLink (opened at run time; QMC_ERR_CUDA with the assembler's text in
 * qmc_last_cuda_error if that fails), kernels in parallel on the host's cores.  It needs no GPU.  Used of each problem:
 * family, dim, n_params and params (HOST pointer; read during the call only); everything else is ignored, so one module
 * serves any lattice, shift set and sample count of the same integrands.  Problems of other families, and sector blocks the
 * validation rejects, simply stay on the default kernels.  The caller owns the module and destroys it (also unloads it from
 * every device it ran on); a module may be used from several host threads and on several devices.
 *
 * qmc_lattice_integrate_batch_module is qmc_lattice_integrate_batch (same arguments, stream-ordered; the workspace size comes
 * from qmc_sector_module_workspace_bytes: every kernel of the module has a tile queue of its own) with
 * the module's kernels for the problems that have code there AND run the default tile loop (transform Korobov r = 3, no fit map,
 * n < 2^31); the rest of the batch takes the default kernels in the same call.  `problems` must be the batch the module was
 * built from, in its order (count / family / dim / n_params are checked: QMC_ERR_N / QMC_ERR_PARAMS; the VALUES of params
 * are the caller's promise -- polynomials are read from the module, nu / a / b / log factors too).  The first launch on a
 * device loads the images there (a synchronous driver call). */
int qmc_sector_module_create(int count, const qmc_problem* problems /*HOST, HOST params*/, int sectors_per_kernel,
                             qmc_sector_module** out /*HOST*/);
void qmc_sector_module_destroy(qmc_sector_module* module);
/* what was built: specialised problems, kernels, host milliseconds of the create call, bytes of device code, host threads used
 * (any pointer may be NULL) */
int qmc_sector_module_info(const qmc_sector_module* module, int* n_specialised, int* n_kernels, double* build_ms, size_t* image_bytes,
                           int* host_threads);
/* kernel `kernel`'s device image (an ELF for cuobjdump -sass) and the assembler's report (registers, spills); sizes through
 * *image_bytes with image = NULL; QMC_ERR_WORKSPACE if image_cap is too small */
int qmc_sector_module_image(const qmc_sector_module* module, int kernel, void* image /*HOST or NULL*/, size_t image_cap,
                            size_t* image_bytes /*HOST or NULL*/, char* log /*HOST or NULL*/, size_t log_cap);
/* qmc_lattice_integrate_batch_host (synchronous, HOST data pointers) with a module; module = NULL is that entry itself */
int qmc_lattice_integrate_batch_host_module(qmc_sector_module* module /*or NULL*/, int count,
                                            const qmc_problem* problems /*HOST, HOST data pointers*/, double* out_means /*HOST*/,
                                            double* out_errs /*HOST*/, double* out_shift_means /*HOST or NULL*/);
size_t qmc_sector_module_workspace_bytes(const qmc_sector_module* module, int count, const qmc_problem* problems /*HOST*/);  /* 0 on invalid input */
int qmc_lattice_integrate_batch_module(qmc_sector_module* module, int count, const qmc_problem* problems /*HOST*/,
                                       double* out_means /*DEVICE*/, double* out_errs /*DEVICE*/,
                                       double* out_shift_means /*DEVICE or NULL*/, void* workspace /*DEVICE*/,
                                       size_t workspace_bytes, void* cuda_stream);

/* ---- prepared batches ---------------------------------------------------------------------------------------------------
 * qmc_lattice_integrate_batch plans the batch and uploads the plan on every call (from pageable host memory, which a CUDA graph
 * capture refuses).  A prepared batch does that ONCE: qmc_batch_create plans, uploads, runs the sector prepare kernel, loads the
 * kernels (synchronises `cuda_stream` before it returns); qmc_batch_launch is then one 512-byte memset of the tile-queue heads
 * plus the fused kernels and the finalize kernel -- nothing is read from host memory, nothing is allocated, no synchronisation --
 * and can be captured in a CUDA graph (with profiling off: qmc_profile_enable(0)).  Same kernels, same tiling, same bits as
 * qmc_lattice_integrate_batch (with `module`: as qmc_lattice_integrate_batch_module; workspace size from
 * qmc_workspace_bytes / qmc_sector_module_workspace_bytes).
 *   The workspace belongs to the batch until qmc_batch_destroy (which frees only host memory); launches of one batch that
 *   overlap on the GPU race on it.  Read at create: the problem structs, and of sector problems params, z and fit_coeffs (their
 *   programs and tables are compiled then).  Read at every launch, from the DEVICE pointers given at create: shifts of every
 *   problem, params / z / fit_coeffs of closed-form problems -- so fresh random shifts written into the same buffer need no new
 *   batch.  The module, if any, must outlive the batch. */
typedef struct qmc_batch qmc_batch;
int qmc_batch_create(int count, const qmc_problem* problems /*HOST*/, qmc_sector_module* module /*or NULL*/,
                     void* workspace /*DEVICE*/, size_t workspace_bytes, void* cuda_stream, qmc_batch** out /*HOST*/);
int qmc_batch_launch(qmc_batch* batch, double* out_means /*DEVICE*/, double* out_errs /*DEVICE*/,
                     double* out_shift_means /*DEVICE or NULL*/, void* cuda_stream);
void qmc_batch_destroy(qmc_batch* batch);

/* ---- an entry that allocates nothing --------------------------------------------------------------------------------------
 * For callers that cannot allocate device memory around a call (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): qmc_lattice_integrate_batch with the workspace in a device array that is part of the library image,
 * QMC_STATIC_SCRATCH_BYTES (4 MiB) per GPU that loads the library, held until the process exits.  Arguments, kernels and results
 * are those of qmc_lattice_integrate_batch (problems HOST structs with DEVICE data pointers, outputs DEVICE, stream-ordered, no
 * synchronisation); the call itself issues no cudaMalloc / cudaFree / allocating library routine.  (Under stream capture: a call
 * for ONE closed-form problem is kernel launches and an 8-byte memset and can be captured; a batch uploads its plan from pageable
 * host memory as qmc_lattice_integrate_batch does, which a capture refuses -- capture qmc_batch_launch instead.)
 *   Limit: qmc_workspace_bytes(count, problems) <= qmc_static_scratch_bytes(); a larger batch is rejected with QMC_ERR_WORKSPACE
 *   before anything is launched, and qmc_last_cuda_error() then says how many bytes the batch needs (configs[4] of the bench
 *   needs 0.15 MB, the 256-sector batch of configs[3] 1.3 MB).
 *   Sharing: every call on a device uses the same array, and the array keeps the last call's contents.  Nothing has to be
 *   cleared by the caller -- a call resets its tile queues itself and writes every partial sum before it reads it -- but two
 *   calls whose kernels OVERLAP on the GPU (different streams without an ordering between them, or two host threads on one
 *   device) race on it: order them, or use qmc_lattice_integrate_batch with separate workspaces. */
#define QMC_STATIC_SCRATCH_BYTES 4194304
size_t qmc_static_scratch_bytes(void);
int qmc_lattice_integrate_batch_static(int count, const qmc_problem* problems /*HOST*/, double* out_means /*DEVICE*/,
                                       double* out_errs /*DEVICE*/, double* out_shift_means /*DEVICE or NULL*/,
                                       void* cuda_stream);

int qmc_num_components(int family);          /* 1 or 2; <0 on unknown family */
const char* qmc_status_string(int status);
const char* qmc_last_cuda_error(void);       /* thread-local text of the last CUDA error ("" if none) */

#ifdef __cplusplus
}
#endif
#endif /* QMC_LATTICE_H */
