"""Writes qmc_sector_interp.inc: the threaded-code interpreter of the sector family as inline PTX.

    python paper_1811_11720_b200/csrc/gen_sector_interp.py

Why PTX: the interpreter dispatches one byte-coded step at a time on the coordinates x[q][j], which must
stay in registers (shared memory cannot feed the FP64 pipe: 128 B/clk/SM against 2 fp64 warp
instructions/clk/SM).  Register operands can only be selected by control flow, and nvcc lowers a C++
`switch` to a tree of compare-and-branch pairs.  PTX `brx.idx` gives one indexed branch per step; every case
ends with its own dispatch (threaded code); step codes are fetched two steps ahead, so the index of the next
branch is known when a case is entered and its jump-table lookup overlaps the G fp64 instructions of the step.

The machine (qmc_sector.cuh has the device-side compiler that targets it): per point two accumulators, S (the value of
the polynomial) and A (the value of the current group).  A polynomial is a sum of groups
    x^P * (own + sum_k c_k x_k)          P a monomial (the shared prefix), own / c_k coefficients
found by factoring the most frequent variable out of the monomial set repeatedly (a greedy multivariate Horner
form: 30.6 steps instead of 44.4 for the flat monomial-by-monomial evaluation on the seeded sectors of configs[3]).
Step kinds, one fp64 instruction per point each:
    SC j : S = fma(A, x_j, S)            closes a group (last prefix variable)
    SL j : S = fma(cf, x_j, S)           a degree-1 monomial of the polynomial
    AL j : A = fma(cf, x_j, A)           a further leaf of the group
    ALI j: A = fma(cf, x_j, cf2)         first leaf of a group (cf2 = own), or cf * x_j for a plain monomial (cf2 = 0)
    AM j : A = A * x_j                   a prefix variable that is not the last
The complex family (sector polynomials with complex coefficients on real coordinates, reading C-16) runs the same five kinds
on paired accumulators (S_re, S_im), (A_re, A_im): two fp64 instructions per point and step, coefficient slots of 32 bytes
{cf_re, cf_im, cf2_re, cf2_im}.
Step code = 3 + 5 j + kind; 0 = no-op, 1 = end of a polynomial that is not the last (parks S in the thread's next
shared-memory column and restarts it with the next polynomial's constant term), 2 = end of program.  SL / AL / ALI and
the end-of-polynomial step read one 16-byte coefficient slot {cf, cf2} each, in program order.

What was measured on a B200 (one interpreter in isolation, G = 8, 6 coordinates, 12 warps per SM):
an indexed branch costs about 60 cycles that warps of one scheduler do not overlap well, so a step of 8 fp64
instructions per warp leaves the FP64 pipe at 35-45 %; the cases must stay resident in the ~6 KB L0 instruction
cache (48 cases of a three-accumulator Horner machine ran 50 % slower per step than 24, different programs on
co-resident CTAs 45 % slower than one program per SM -- hence one CTA per SM for this family); a tree of direct
branches on precomputed predicates was 20 % slower than brx.idx; moving the coefficient with or ahead of its use
made no difference.
"""
import os

# (DP, G, threads per CTA, complex) instantiated by qmc_fused_f3.cu (real sectors) and qmc_fused_f8.cu (complex sectors)
VARIANTS = [(4, 8, 384, False), (6, 8, 384, False), (8, 8, 256, False), (16, 4, 256, False),
            (4, 4, 384, True), (6, 4, 384, True), (8, 4, 384, True), (16, 2, 384, True)]
KINDS = 5
SC, SL, AL, ALI, AM = range(KINDS)


def gen(dp, g, nt, cplx):
    # operand numbering: S[q] = %q (complex: S_re[q] = %q, S_im[q] = %(g+q)), x[q][j] next, then steps address,
    # coefficient address, park address
    ns = 2 * g if cplx else g
    sr = lambda q: f"%{q}"
    si = lambda q: f"%{g + q}"
    x = lambda q, j: f"%{ns + q * dp + j}"
    steps, coefs, upark = (f"%{ns + g * dp + i}" for i in range(3))
    slot = 32 if cplx else 16
    L = []
    a = L.append
    a("{")
    if cplx:
        a(".reg .f64 " + ", ".join(f"A{q}, B{q}" for q in range(g)) + ", cfn, cfni, cf2n, cf2ni;")      # B = Im A
    else:
        a(".reg .f64 " + ", ".join(f"A{q}" for q in range(g)) + ", cfn, cf2n;")
    a(".reg .u32 pc, pk, pp, tgt, c0;")
    labels = ["T_NOP", "T_ENDU", "T_END"] + [f"T_{j}_{k}" for j in range(dp) for k in range(KINDS)]
    a("ts: .branchtargets " + ", ".join(labels) + ";")
    a(f"mov.u32 pc, {steps};")
    a(f"mov.u32 pk, {coefs};")
    a(f"mov.u32 pp, {upark};")
    for q in range(g):
        a(f"mov.f64 A{q}, 0d0000000000000000;")
        if cplx:
            a(f"mov.f64 B{q}, 0d0000000000000000;")

    def load_slot(off):
        if cplx:
            return [f"ld.shared.v2.f64 {{cfn, cfni}}, [pk+{off}];", f"ld.shared.v2.f64 {{cf2n, cf2ni}}, [pk+{off + 16}];"]
        return [f"ld.shared.v2.f64 {{cfn, cf2n}}, [pk+{off}];"]
    L.extend(load_slot(0))
    a("ld.shared.u8 tgt, [pc];")
    a("ld.shared.u8 c0, [pc+1];")
    leave = "brx.idx.uni tgt, ts;"
    a(leave)
    # on entry to the case of step i: c0 = code[i+1] has arrived; the branch index of step i+1 is known at entry
    fetch = ["mov.u32 tgt, c0;", "ld.shared.u8 c0, [pc+2];", "add.u32 pc, pc, 1;"]
    reload = load_slot(slot) + [f"add.u32 pk, pk, {slot};"]
    a("T_NOP:")
    L.extend(fetch)
    a(leave)
    a("T_ENDU:")
    L.extend(fetch)
    for q in range(g):
        if cplx:
            a(f"st.shared.f64 [pp+{8 * nt * (2 * q)}], {sr(q)};")
            a(f"st.shared.f64 [pp+{8 * nt * (2 * q + 1)}], {si(q)};")
            a(f"mov.f64 {sr(q)}, cfn;")
            a(f"mov.f64 {si(q)}, cfni;")
        else:
            a(f"st.shared.f64 [pp+{8 * nt * q}], {sr(q)};")
            a(f"mov.f64 {sr(q)}, cfn;")
    a(f"add.u32 pp, pp, {8 * nt * ns};")
    L.extend(reload)
    a(leave)
    for j in range(dp):
        for k in range(KINDS):
            a(f"T_{j}_{k}:")
            L.extend(fetch)
            for q in range(g):
                X = x(q, j)
                if k == SC:
                    a(f"fma.rn.f64 {sr(q)}, A{q}, {X}, {sr(q)};")
                    if cplx: a(f"fma.rn.f64 {si(q)}, B{q}, {X}, {si(q)};")
                elif k == SL:
                    a(f"fma.rn.f64 {sr(q)}, cfn, {X}, {sr(q)};")
                    if cplx: a(f"fma.rn.f64 {si(q)}, cfni, {X}, {si(q)};")
                elif k == AL:
                    a(f"fma.rn.f64 A{q}, cfn, {X}, A{q};")
                    if cplx: a(f"fma.rn.f64 B{q}, cfni, {X}, B{q};")
                elif k == ALI:
                    a(f"fma.rn.f64 A{q}, cfn, {X}, cf2n;")
                    if cplx: a(f"fma.rn.f64 B{q}, cfni, {X}, cf2ni;")
                else:
                    a(f"mul.rn.f64 A{q}, A{q}, {X};")
                    if cplx: a(f"mul.rn.f64 B{q}, B{q}, {X};")
            if k in (SL, AL, ALI):
                L.extend(reload)                      # after the last use of the slot: no register moves
            a(leave)
    a("T_END:")
    a("}")
    body = "\n".join(f'        "{line}\\n\\t"' for line in L)
    outs = ", ".join([f'"+d"(sum[{q}])' for q in range(g)] + ([f'"+d"(sum_im[{q}])' for q in range(g)] if cplx else []))
    ins = ", ".join([f'"d"(x[{q}][{j}])' for q in range(g) for j in range(dp)] +
                    ['"r"(steps_addr)', '"r"(coefs_addr)', '"r"(park_addr)'])
    if cplx:
        return f"""
template <> __device__ __forceinline__ void csector_interp<{dp}, {g}, {nt}>(const double (&x)[{g}][{dp}], unsigned steps_addr,
                                                                         unsigned coefs_addr, unsigned park_addr, double (&sum)[{g}],
                                                                         double (&sum_im)[{g}]) {{
    asm volatile(
{body}
        : {outs}
        : {ins}
        : "memory");
}}
"""
    return f"""
template <> __device__ __forceinline__ void sector_interp<{dp}, {g}, {nt}>(const double (&x)[{g}][{dp}], unsigned steps_addr,
                                                                        unsigned coefs_addr, unsigned park_addr, double (&sum)[{g}]) {{
    asm volatile(
{body}
        : {outs}
        : {ins}
        : "memory");
}}
"""


def gen_site(dp, g):
    """The place where a specialised kernel evaluates its sector (qmc_spec.cu splices straight-line PTX over the marker)."""
    ops = ([f'"=d"(num[{q}])' for q in range(g)] + [f'"=d"(den[{q}])' for q in range(g)] + [f'"=d"(F[{q}])' for q in range(g)])
    ins = ([f'"d"(x[{q}][{j}])' for q in range(g) for j in range(dp)] + [f'"d"(W[{q}])' for q in range(g)] + ['"r"(sel)', '"r"(park_addr)'])
    n = len(ops) + len(ins)
    text = "@@QMC_SITE " + " ".join(f"%{i}" for i in range(n)) + ";"
    return f"""
template <> __device__ __forceinline__ void sector_poly_site<{dp}, {g}>(const double (&x)[{g}][{dp}], const double (&W)[{g}], unsigned sel,
                                                                     unsigned park_addr, double (&num)[{g}], double (&den)[{g}],
                                                                     double (&F)[{g}]) {{
    asm volatile("{text}"
        : {", ".join(ops)}
        : {", ".join(ins)}
        : "memory");
}}
"""


def gen_csite(dp, g):
    """complex family: outputs n = W prod x^nu U^a, d = F^b, F and U as (re, im) pairs"""
    names = ["nr", "ni", "dr", "di", "Fr", "Fi", "Ur", "Ui"]
    ops = [f'"=d"({nm}[{q}])' for nm in names for q in range(g)]
    ins = ([f'"d"(x[{q}][{j}])' for q in range(g) for j in range(dp)] + [f'"d"(W[{q}])' for q in range(g)] + ['"r"(sel)'])
    text = "@@QMC_SITE " + " ".join(f"%{i}" for i in range(len(ops) + len(ins))) + ";"
    args = ", ".join(f"double (&{nm})[{g}]" for nm in names)
    return f"""
template <> __device__ __forceinline__ void csector_poly_site<{dp}, {g}>(const double (&x)[{g}][{dp}], const double (&W)[{g}], unsigned sel,
                                                                      {args}) {{
    asm volatile("{text}"
        : {", ".join(ops)}
        : {", ".join(ins)}
        : "memory");
}}
"""


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    out = ["// GENERATED by gen_sector_interp.py -- do not edit.  Threaded-code interpreter of the sector family",
           "// (inline PTX, one brx.idx.uni per step); included by qmc_sector.cuh inside namespace qmc.",
           "// sum[] must hold the first polynomial's constant term on entry; polynomial p < last is parked at",
           "// park_addr + 8 NT (G p + q) (shared memory, the thread's own column); on return sum[q] = the last polynomial at x_q.",
           "template <int DP, int G, int NT> __device__ __forceinline__ void sector_interp(const double (&x)[G][DP], unsigned steps_addr,",
           "                                                                               unsigned coefs_addr, unsigned park_addr,",
           "                                                                               double (&sum)[G]);"]
    out += ["// complex family: sum / sum_im hold the first polynomial's constant term (re, im) on entry; polynomial p < last is parked at",
            "// park_addr + 8 NT (2 G p + 2 q + c), c = 0 (re), 1 (im); on return (sum[q], sum_im[q]) = the last polynomial at x_q.",
            "template <int DP, int G, int NT> __device__ __forceinline__ void csector_interp(const double (&x)[G][DP], unsigned steps_addr,",
            "                                                                                unsigned coefs_addr, unsigned park_addr,",
            "                                                                                double (&sum)[G], double (&sum_im)[G]);"]
    real = [v for v in VARIANTS if not v[3]]
    cplx = [v for v in VARIANTS if v[3]]
    with open(os.path.join(here, "qmc_sector_interp.inc"), "w") as f:
        f.write("\n".join(out[:7] + [gen(*v) for v in real]))
    with open(os.path.join(here, "qmc_csector_interp.inc"), "w") as f:
        f.write("\n".join(out[:2] + out[7:] + [gen(*v) for v in cplx]))
    site = ["// GENERATED by gen_sector_interp.py -- do not edit.  The marker a specialised sector kernel carries where the code of its",
            "// sectors goes (qmc_spec_template.cu is compiled to PTX only; qmc_spec.cu replaces the marker line, whose operands are,",
            "// in this order: num[G], den[G], F[G] (outputs), x[G][DP], W[G], the case selector, the thread's park address).",
            "template <int DP, int G> __device__ __forceinline__ void sector_poly_site(const double (&x)[G][DP], const double (&W)[G], unsigned sel,",
            "                                                                          unsigned park_addr, double (&num)[G], double (&den)[G],",
            "                                                                          double (&F)[G]);"]
    with open(os.path.join(here, "qmc_sector_site.inc"), "w") as f:
        f.write("\n".join(site + [gen_site(dp, g) for dp, g, _, c in VARIANTS if not c]))
        f.write("\n".join(["", "// complex family: operands nr[G], ni[G], dr[G], di[G], Fr[G], Fi[G], Ur[G], Ui[G] (outputs), x[G][DP], W[G], the case selector",
                           "template <int DP, int G> __device__ __forceinline__ void csector_poly_site(const double (&x)[G][DP], const double (&W)[G], unsigned sel,",
                           "                                                                           double (&nr)[G], double (&ni)[G], double (&dr)[G], double (&di)[G],",
                           "                                                                           double (&Fr)[G], double (&Fi)[G], double (&Ur)[G], double (&Ui)[G]);"]
                          + [gen_csite(dp, g) for dp, g, _, c in VARIANTS if c]))


if __name__ == "__main__":
    main()
