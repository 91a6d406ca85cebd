"""Writes qmc_sector_interp.inc: the threaded-code interpreter of the sector family as inline PTX.

    python paper_1811_11720_b200/csrc/gen_sector_interp.py

Why PTX: the interpreter dispatches one byte-coded step at a time on the coordinates x[q][j], which must
stay in registers (shared memory cannot feed the FP64 pipe: 128 B/clk/SM against 2 fp64 warp
instructions/clk/SM).  Register operands can only be selected by control flow, and nvcc lowers a C++
`switch` to a tree of compare-and-branch pairs (5 dependent branches per step, which made the kernel
latency bound).  PTX `brx.idx` gives one indexed branch per step; every case ends with its own dispatch
(threaded code) and loads the next step code and the next coefficient before its fp64 work, so the
shared-memory latency hides behind the G fp64 instructions of the step.

Step codes (qmc_sector.cuh): 0 = no-op, 1 = end of U, 2 = end of program, 3 = dense linear form
(sum += sum_j c_j x_j with DP coefficients from the stream), 4 + 4*j + 2*FIRST + LAST:
    FIRST & LAST : sum  = fma(coef, x_j, sum)
    FIRST        : mon  = coef * x_j
    LAST         : sum  = fma(mon, x_j, sum)
    otherwise    : mon *= x_j
For DP <= 8 also pair steps, 4 + 4*DP + 2*pair_index(a, b) + FULL with a <= b: the first two variables of a
monomial in one dispatch,  mon = coef * x_a;  FULL ? sum = fma(mon, x_b, sum) : mon *= x_b.
"""
import os

VARIANTS = [(4, 8), (6, 8), (8, 8), (16, 4)]      # (DP, G) instantiated by qmc_fused_f3.cu
SETS = 1                                           # copies of the case table (register roles rotate, no moves)


def has_pairs(dp):
    """pair steps exist where all codes fit one byte (qmc_sector.cuh: sector_has_pairs)"""
    return dp <= 0


def pair_index(a, b, dp):
    return a * dp - a * (a - 1) // 2 + (b - a)


def gen(dp, g):
    # operand numbering: sum[q] = %q, U[q] = %(g+q), x[q][j] = %(2g + q*dp + j), then c0f, steps address, coefs address
    s = lambda q: f"%{q}"
    u = lambda q: f"%{g + q}"
    x = lambda q, j: f"%{2 * g + q * dp + j}"
    c0f, steps, coefs = (f"%{2 * g + g * dp + i}" for i in range(3))
    pairs = [(p, q) for p in range(dp) for q in range(p, dp)] if has_pairs(dp) else []
    L = []
    a = L.append
    a("{")
    a(".reg .f64 " + ", ".join(f"m{q}" for q in range(g)) + ", cf, cfn, " + ", ".join(f"l{j}" for j in range(1, dp)) + ";")
    a(".reg .u32 pc, pk, tgt, " + ", ".join(f"c{t}" for t in range(max(SETS, 2))) + ";")
    for t in range(SETS):
        labels = [f"T{t}_NOP", f"T{t}_ENDU", "LEND", f"T{t}_LIN"] + [f"T{t}_S{j}_{k}" for j in range(dp) for k in range(4)]
        labels += [f"T{t}_P{p}_{q}_{full}" for (p, q) in pairs for full in range(2)]
        a(f"ts{t}: .branchtargets " + ", ".join(labels) + ";")
    for q in range(g):
        a(f"mov.f64 m{q}, 0d0000000000000000;")
    a(f"mov.u32 pc, {steps};")
    a(f"mov.u32 pk, {coefs};")
    a("ld.shared.f64 cfn, [pk];")
    if SETS == 1:
        a("ld.shared.u8 tgt, [pc];")
        a("ld.shared.u8 c0, [pc+1];")
        a("ld.shared.u8 c1, [pc+2];")
        a("brx.idx.uni tgt, ts0;")
    else:
        for t in range(SETS):
            a(f"ld.shared.u8 c{t}, [pc+{t}];")
        a("brx.idx.uni c0, ts0;")
    for t in range(SETS):
        # case of step i in table t = i mod SETS: register c_t held code[i]; it is reloaded with code[i+SETS] and the
        # step leaves through c_{t+1} (loaded SETS-1 steps ago) into the next table
        nt = (t + 1) % SETS
        fetch = [f"ld.shared.u8 c{t}, [pc+{SETS}];", "add.u32 pc, pc, 1;"]
        leave = f"brx.idx.uni c{nt}, ts{nt};"
        if SETS == 1:
            # one table: c0 = code[i+1] (arrived), c1 = code[i+2] (in flight); the target of step i+1 is known at entry
            fetch = ["mov.u32 tgt, c0;", "mov.u32 c0, c1;", "ld.shared.u8 c1, [pc+3];", "add.u32 pc, pc, 1;"]
            leave = "brx.idx.uni tgt, ts0;"
        coef = ["mov.f64 cf, cfn;", "ld.shared.f64 cfn, [pk+8];", "add.u32 pk, pk, 8;"]
        a(f"T{t}_NOP:")
        L.extend(fetch)
        a(leave)
        a(f"T{t}_ENDU:")
        L.extend(fetch)
        for q in range(g):
            a(f"mov.f64 {u(q)}, {s(q)};")
            a(f"mov.f64 {s(q)}, {c0f};")
        a(leave)
        # dense linear form: DP coefficients from the stream (the first one is the prefetched cfn)
        a(f"T{t}_LIN:")
        L.extend(fetch)
        a("mov.f64 cf, cfn;")
        for j in range(1, dp):
            a(f"ld.shared.f64 l{j}, [pk+{8 * j}];")
        a(f"ld.shared.f64 cfn, [pk+{8 * dp}];")
        a(f"add.u32 pk, pk, {8 * dp};")
        for j in range(dp):
            for q in range(g):
                a(f"fma.rn.f64 {s(q)}, {'cf' if j == 0 else f'l{j}'}, {x(q, j)}, {s(q)};")
        a(leave)
        for j in range(dp):
            for k in range(4):
                first, last = k >> 1, k & 1
                a(f"T{t}_S{j}_{k}:")
                L.extend(fetch)
                if first:
                    L.extend(coef)
                for q in range(g):
                    if first and last:
                        a(f"fma.rn.f64 {s(q)}, cf, {x(q, j)}, {s(q)};")
                    elif first:
                        a(f"mul.rn.f64 m{q}, cf, {x(q, j)};")
                    elif last:
                        a(f"fma.rn.f64 {s(q)}, m{q}, {x(q, j)}, {s(q)};")
                    else:
                        a(f"mul.rn.f64 m{q}, m{q}, {x(q, j)};")
                a(leave)
        for (p, r) in pairs:
            for full in range(2):
                a(f"T{t}_P{p}_{r}_{full}:")
                L.extend(fetch)
                L.extend(coef)
                for q in range(g):
                    a(f"mul.rn.f64 m{q}, cf, {x(q, p)};")
                for q in range(g):
                    if full:
                        a(f"fma.rn.f64 {s(q)}, m{q}, {x(q, r)}, {s(q)};")
                    else:
                        a(f"mul.rn.f64 m{q}, m{q}, {x(q, r)};")
                a(leave)
    a("LEND:")
    a("}")
    body = "\n".join(f'        "{line}\\n\\t"' for line in L)
    outs = ", ".join([f'"+d"(sum[{q}])' for q in range(g)] + [f'"+d"(U[{q}])' for q in range(g)])
    ins = ", ".join([f'"d"(x[{q}][{j}])' for q in range(g) for j in range(dp)] + ['"d"(c0f)', '"r"(steps_addr)', '"r"(coefs_addr)'])
    return f"""
template <> __device__ __forceinline__ void sector_interp<{dp}, {g}>(const double (&x)[{g}][{dp}], unsigned steps_addr,
                                                                  unsigned coefs_addr, double c0f, double (&U)[{g}],
                                                                  double (&sum)[{g}]) {{
    asm volatile(
{body}
        : {outs}
        : {ins});
}}
"""


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    out = ["// GENERATED by gen_sector_interp.py -- do not edit.  Threaded-code interpreter of the sector family",
           "// (inline PTX, one brx.idx.uni per step); included by qmc_sector.cuh inside namespace qmc.",
           "// sum[] must hold U's constant term on entry; on return U[q] = U(x_q), sum[q] = F(x_q).",
           "template <int DP, int G> __device__ __forceinline__ void sector_interp(const double (&x)[G][DP], unsigned steps_addr,",
           "                                                                       unsigned coefs_addr, double c0f, double (&U)[G],",
           "                                                                       double (&sum)[G]);"]
    for dp, g in VARIANTS:
        out.append(gen(dp, g))
    with open(os.path.join(here, "qmc_sector_interp.inc"), "w") as f:
        f.write("\n".join(out))


if __name__ == "__main__":
    main()
