// qmc_sector_compile.h -- parameter block of a sector -> program of the two-accumulator Horner machine (qmc_sector.cuh has the
// machine).  Host and device: the interpreting kernels compile on the device (prepare_sector), the specialised kernels on the
// host (qmc_spec.cu), from the same function, so that both evaluate the same operations in the same order.
#pragma once
#include <cmath>

#include "qmc_internal.h"

#if defined(__CUDACC__)
#define QMC_HD __host__ __device__
#else
#define QMC_HD
#endif

namespace qmc {

constexpr int kSecKinds = 5;
// step codes (one byte each): 0 = no-op, 1 = end of a polynomial that is not the last, 2 = end of program, 3 + 5 j + kind
enum : int { SEC_NOP = 0, SEC_ENDP = 1, SEC_END = 2, SEC_BASE = 3 };
enum : int { SEC_SC = 0, SEC_SL = 1, SEC_AL = 2, SEC_ALI = 3, SEC_AM = 4 };

// ---- device-side compiler: params -> program (one thread per problem; runs once per call) ---------------------------
// Program area of a problem (8-byte words at prog_area + aux_off): sector_slot_words(nmono) words of coefficient slots,
// then the step bytes.  DevAux: sec_nops[0] = number of 32-bit step words, sec_ncoef[0] = number of slots.
// Full validation of a sector parameter block (on the device for the interpreting kernels and the projection pass, whose values
// live in DEVICE memory; on the host when a module of specialised kernels is built):
// a, b integers in 0..8; nU, nF integers in 1..kMaxSectorMono; n_params = 4 + d + (nU + nF)(1 + d) (+ 3 with the trailing
// [lu, lf, p], p an integer in 1..4; the complex family has (2 + d) per monomial); nu_j and every exponent integers in 0..8; degree <= 16
// (include/qmc_lattice.h).  Used by the device-side compiler and by the projection pass: nothing reads an exponent, a count
// or a power of a block that did not pass.  Returns 0 or QMC_ERR_PARAMS.
QMC_HD inline int sector_block_status(const double* p, int n_params, int d, bool cplx = false) {
    const int rec = (cplx ? 2 : 1) + d;                // monomial record: coefficient (re [, im]) + exponents
    if (n_params < 4 + d + 2 * rec) return QMC_ERR_PARAMS;
    const double av = p[0], bv = p[1], nUv = p[2], nFv = p[3];
    if (!(av >= 0.0 && av <= 8.0 && bv >= 0.0 && bv <= 8.0 && nUv >= 1.0 && nUv <= kMaxSectorMono && nFv >= 1.0 &&
          nFv <= kMaxSectorMono) ||
        av != floor(av) || bv != floor(bv) || nUv != floor(nUv) || nFv != floor(nFv))
        return QMC_ERR_PARAMS;
    const int cnt[2] = {(int)nUv, (int)nFv};
    const int n_base = 4 + d + (cnt[0] + cnt[1]) * rec;
    if (n_params == n_base + 3) {                      // trailing [lu, lf, p]: f (lu log U + lf log F)^p, p in 1..4
        const double pw = p[n_base + 2];
        if (!(pw >= 1.0 && pw <= 4.0) || pw != floor(pw)) return QMC_ERR_PARAMS;
    } else if (n_params != n_base) return QMC_ERR_PARAMS;
    for (int j = 0; j < d; ++j) {
        const double v = p[4 + j];
        if (!(v >= 0.0 && v <= 8.0) || v != floor(v)) return QMC_ERR_PARAMS;
    }
    const double* base = p + 4 + d;
    for (int pol = 0; pol < 2; ++pol) {
        const double* e = base + (cplx ? 2 : 1) * cnt[pol];
        for (int t = 0; t < cnt[pol]; ++t) {
            int deg = 0;
            for (int j = 0; j < d; ++j) {
                const double v = e[t * d + j];
                if (!(v >= 0.0 && v <= 8.0) || v != floor(v)) return QMC_ERR_PARAMS;
                deg += (int)v;
            }
            if (deg > 16) return QMC_ERR_PARAMS;
        }
        base += cnt[pol] * rec;
    }
    return 0;
}

struct SecEmit {                     // output cursor of the compiler
    double* slots;
    unsigned char* ops;
    int nslots, nops, max_slots, max_ops, status;
    bool cplx;                       // 32-byte slots {cf_re, cf_im, cf2_re, cf2_im}
    QMC_HD void op(int kind, int j) {
        if (nops >= max_ops) { status = QMC_ERR_PARAMS; return; }
        ops[nops++] = (unsigned char)(SEC_BASE + kSecKinds * j + kind);
    }
    QMC_HD void slot(double cf, double cfi, double cf2, double cf2i) {
        if (nslots >= max_slots) { status = QMC_ERR_PARAMS; return; }
        if (cplx) { slots[4 * nslots] = cf; slots[4 * nslots + 1] = cfi; slots[4 * nslots + 2] = cf2; slots[4 * nslots + 3] = cf2i; }
        else { slots[2 * nslots] = cf; slots[2 * nslots + 1] = cf2; }
        ++nslots;
    }
};

// One polynomial: `cnt` monomials, coefficients c[t], exponents e[t*d + j] (validated by the caller: integers 0..8, degree <= 16).
// Greedy Horner form.  A work item is a set of monomials (a range of idx[]) that share the prefix monomial they were reached
// by; rem[t][j] are the exponents still to be factored out, left[t] their sum.  From an item the variable that occurs in most of
// its monomials is factored out: the monomials that contain it form a child (processed as an item of its own unless it is a
// single finished monomial, a "leaf"), the others stay.  When the item is used up its group is emitted: prefix, the coefficient
// of the prefix monomial itself (own) and the leaves.  Returns the constant term.
// ci: imaginary parts of the coefficients (complex family) or nullptr; the constant term is returned through c0_re / c0_im.
QMC_HD inline void compile_polynomial(const double* c, const double* ci, const double* e, int cnt, int d, SecEmit& out,
                                          double* c0_re, double* c0_im) {
    unsigned char rem[kMaxSectorMono][16];
    unsigned char left[kMaxSectorMono];
    short idx[kMaxSectorMono];
    // work items: ranges of idx with the prefix they share (exponents) and the coefficient of the prefix monomial; items on the
    // stack are disjoint ranges with at least one unfinished monomial each, so there are never more than cnt of them
    short it_b[kMaxSectorMono + 1], it_e[kMaxSectorMono + 1];
    double it_own[kMaxSectorMono + 1], it_owni[kMaxSectorMono + 1];
    unsigned char it_prefix[kMaxSectorMono + 1][16];
    double c0 = 0.0, c0i = 0.0;
    int m = 0;
    for (int t = 0; t < cnt; ++t) {
        int deg = 0;
        for (int j = 0; j < d; ++j) { const int v = (int)e[t * d + j]; rem[t][j] = (unsigned char)v; deg += v; }
        for (int j = d; j < 16; ++j) rem[t][j] = 0;
        left[t] = (unsigned char)deg;
        if (deg == 0) { c0 += c[t]; if (ci) c0i += ci[t]; } else idx[m++] = (short)t;
    }
    int top = 0;
    it_b[0] = 0; it_e[0] = (short)m; it_own[0] = 0.0; it_owni[0] = 0.0;
    for (int j = 0; j < 16; ++j) it_prefix[0][j] = 0;
    top = 1;
    bool root = true;
    while (top > 0) {
        --top;
        const int b = it_b[top], en = it_e[top];
        const double own = it_own[top], owni = it_owni[top];
        unsigned char prefix[16];
        int pdeg = 0;
        for (int j = 0; j < 16; ++j) { prefix[j] = it_prefix[top][j]; pdeg += prefix[j]; }
        const bool is_root = root;
        root = false;
        double leaf_c[16], leaf_ci[16];
        int leaf_mask = 0;
        int cur = b;
        while (cur < en) {
            // the variable that occurs in most of the remaining monomials (lowest index on ties)
            int best = 0, best_cnt = -1;
            for (int j = 0; j < d; ++j) {
                int n = 0;
                for (int i = cur; i < en; ++i) n += rem[idx[i]][j] > 0;
                if (n > best_cnt) { best_cnt = n; best = j; }
            }
            // partition: monomials containing x_best to the front, the finished ones among them first
            int mid = cur;
            for (int i = cur; i < en; ++i)
                if (rem[idx[i]][best] > 0) { const short t = idx[i]; idx[i] = idx[mid]; idx[mid] = t; ++mid; }
            double child_own = 0.0, child_owni = 0.0;
            int fin = cur;
            for (int i = cur; i < mid; ++i) {
                const short t = idx[i];
                --rem[t][best]; --left[t];
                if (left[t] == 0) { child_own += c[t]; if (ci) child_owni += ci[t]; idx[i] = idx[fin]; idx[fin] = t; ++fin; }
            }
            if (fin == mid) {                                  // nothing below: a leaf of this item
                leaf_c[best] = (leaf_mask >> best & 1) ? leaf_c[best] + child_own : child_own;
                leaf_ci[best] = (leaf_mask >> best & 1) ? leaf_ci[best] + child_owni : child_owni;
                leaf_mask |= 1 << best;
            } else {                                           // a child item: prefix * x_best
                it_b[top] = (short)fin; it_e[top] = (short)mid; it_own[top] = child_own; it_owni[top] = child_owni;
                for (int j = 0; j < 16; ++j) it_prefix[top][j] = prefix[j];
                ++it_prefix[top][best];
                ++top;
            }
            cur = mid;
        }
        // emit the group of this item
        if (is_root) {
            for (int k = 0; k < d; ++k)
                if (leaf_mask >> k & 1) { out.op(SEC_SL, k); out.slot(leaf_c[k], leaf_ci[k], 0.0, 0.0); }
            continue;
        }
        int last = 0;
        for (int j = 0; j < d; ++j) if (prefix[j]) last = j;
        if (leaf_mask) {
            bool first = true;
            for (int k = 0; k < d; ++k)
                if (leaf_mask >> k & 1) {
                    out.op(first ? SEC_ALI : SEC_AL, k);
                    out.slot(leaf_c[k], leaf_ci[k], first ? own : 0.0, first ? owni : 0.0);
                    first = false;
                }
            for (int j = 0; j < d; ++j)
                for (int r = 0; r < prefix[j] - (j == last ? 1 : 0); ++r) out.op(SEC_AM, j);
            out.op(SEC_SC, last);
        } else if (own != 0.0 || owni != 0.0) {
            if (pdeg == 1) { out.op(SEC_SL, last); out.slot(own, owni, 0.0, 0.0); }
            else {
                int firstv = 0;
                for (int j = d - 1; j >= 0; --j) if (prefix[j]) firstv = j;
                out.op(SEC_ALI, firstv); out.slot(own, owni, 0.0, 0.0);
                for (int j = 0; j < d; ++j) {
                    const int reps = prefix[j] - (j == firstv ? 1 : 0) - (j == last ? 1 : 0);
                    for (int r = 0; r < reps; ++r) out.op(SEC_AM, j);
                }
                out.op(SEC_SC, last);
            }
        }
    }
    *c0_re = c0; *c0_im = c0i;
}

}  // namespace qmc
