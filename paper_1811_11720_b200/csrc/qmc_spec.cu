// qmc_spec.cu -- modules of specialised sector kernels: the sector family as the paper runs it, compiled code per sector
// ("the integrand functions are compiled"), behind a C ABI that takes parameter blocks.
//
// qmc_sector_module_create compiles every real sector of a batch on the HOST into the Horner program of
// compile_polynomial (qmc_sector_compile.h -- the program the interpreting kernel would run), writes it out as straight-line
// PTX (one fp64 instruction per step and point, coefficients as immediates, nu_j / a / b unrolled), splices the cases of up to
// `sectors_per_kernel` sectors over the marker line of the kernel template (qmc_spec_template.cu, embedded as PTX text) and
// assembles each kernel for sm_100a with nvJitLink, kernels in parallel on the host's cores.  Nothing here touches a GPU;
// the assembled images are loaded on the device that is current when the module is first launched (driver API, entry points
// obtained through the runtime).  The arithmetic is that of the interpreting kernel, operation by operation, so that both
// return the same bits; what goes away is the dispatch of every step.
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include <cuda.h>
#include <dlfcn.h>

#include "qmc_kernels.h"
#include "qmc_sector.cuh"
#include "qmc_spec.h"

extern "C" const char qmc_spec_template_ptx[];          // build/qmc_spec_template_ptx.cpp, written by build.py

namespace qmc {
namespace {

// ---- the kernel template ---------------------------------------------------------------------------------------------
struct SlotKind { int dp, g, threads; bool cplx; const char* entry; size_t smem; };
constexpr int kSlotKindCount = 8;
const SlotKind kSlotKinds[kSlotKindCount] = {{4, 8, 384, false, "qmc_spec_dp4", sizeof(SectorShared<4, 8, 384>)},
                                             {6, 8, 384, false, "qmc_spec_dp6", sizeof(SectorShared<6, 8, 384>)},
                                             {8, 8, 256, false, "qmc_spec_dp8", sizeof(SectorShared<8, 8, 256>)},
                                             {16, 4, 256, false, "qmc_spec_dp16", sizeof(SectorShared<16, 4, 256>)},
                                             {4, 4, 384, true, "qmc_cspec_dp4", sizeof(SectorShared<4, 4, 384>)},
                                             {6, 4, 384, true, "qmc_cspec_dp6", sizeof(SectorShared<6, 4, 384>)},
                                             {8, 4, 384, true, "qmc_cspec_dp8", sizeof(SectorShared<8, 4, 384>)},
                                             {16, 2, 384, true, "qmc_cspec_dp16", sizeof(SectorShared<16, 2, 384>)}};
static_assert(sector_group(4) == 8 && sector_group(16) == 4 && sector_threads(6) == 384 && sector_threads(8) == 256 &&
                  csector_group(8) == 4 && csector_group(16) == 2 && kCSectorThreads == 384,
              "kSlotKinds must mirror the interpreting kernels' shapes (qmc_spec_template.cu has the same numbers)");
int slot_kind_of(int dp, bool cplx) { return (cplx ? 4 : 0) + (dp == 4 ? 0 : (dp == 6 ? 1 : (dp == 8 ? 2 : (dp == 16 ? 3 : -100)))); }

struct EntryText {
    std::string before, after;               // the entry's PTX around the marker line
    std::vector<std::string> operands;       // the marker's operands: num[G], den[G], F[G], x[G][DP], W[G], sel, park (complex:
                                             // nr, ni, dr, di, Fr, Fi, Ur, Ui [G] each, x[G][DP], W[G], sel)
};
struct Template {
    std::string header;                      // .version / .target / module-scope declarations
    EntryText entry[kSlotKindCount];
    bool ok = false;
};

const Template& kernel_template() {
    static const Template t = [] {
        Template r;
        const std::string text(qmc_spec_template_ptx);
        const std::string key = ".visible .entry ";
        std::vector<size_t> starts;
        for (size_t at = text.find(key); at != std::string::npos; at = text.find(key, at + 1)) starts.push_back(at);
        if (starts.size() != (size_t)kSlotKindCount) return r;
        r.header = text.substr(0, starts[0]);
        for (int k = 0; k < kSlotKindCount; ++k) {
            const size_t name_at = text.find(key + kSlotKinds[k].entry + "(");
            if (name_at == std::string::npos) return r;
            size_t end = text.size();
            for (size_t s : starts) if (s > name_at && s < end) end = s;
            const std::string body = text.substr(name_at, end - name_at);
            const size_t mark = body.find("@@QMC_SITE");
            if (mark == std::string::npos || body.find("@@QMC_SITE", mark + 1) != std::string::npos) return r;
            const size_t line_b = body.rfind('\n', mark) + 1, line_e = body.find('\n', mark);
            r.entry[k].before = body.substr(0, line_b);
            r.entry[k].after = body.substr(line_e);
            std::string ops = body.substr(mark + 10, line_e - mark - 10);
            size_t p = 0;
            while (p < ops.size()) {
                while (p < ops.size() && (ops[p] == ' ' || ops[p] == '\t' || ops[p] == ';')) ++p;
                size_t q = p;
                while (q < ops.size() && ops[q] != ' ' && ops[q] != '\t' && ops[q] != ';') ++q;
                if (q > p) r.entry[k].operands.push_back(ops.substr(p, q - p));
                p = q;
            }
            const int g = kSlotKinds[k].g, dp = kSlotKinds[k].dp;
            if ((int)r.entry[k].operands.size() != (kSlotKinds[k].cplx ? 8 * g + g * dp + g + 1 : 3 * g + g * dp + g + 2)) return r;
        }
        r.ok = true;
        return r;
    }();
    return t;
}

// ---- one sector on the host: the program of compile_polynomial, per polynomial ------------------------------------------
struct HostPoly {
    std::vector<unsigned char> ops;
    std::vector<double> slots;               // {cf, cf2} per coefficient-consuming step (complex: {cf_re, cf_im, cf2_re, cf2_im})
    double c0 = 0.0, c0i = 0.0;
};
struct HostSector {
    HostPoly U, F;
    int a = 0, b = 0, nu[16] = {0}, logp = 0;
};

bool compile_sector_host(const double* p, int n_params, int d, bool cplx, HostSector* out) {
    if (sector_block_status(p, n_params, d, cplx) != 0) return false;
    const int cnt[2] = {(int)p[2], (int)p[3]};
    const int rec = (cplx ? 2 : 1) + d, sw = cplx ? 4 : 2;
    const int n_base = 4 + d + (cnt[0] + cnt[1]) * rec;
    out->a = (int)p[0]; out->b = (int)p[1];
    for (int j = 0; j < d; ++j) out->nu[j] = (int)p[4 + j];
    out->logp = n_params == n_base + 3 ? (int)p[n_base + 2] : 0;
    const double* base = p + 4 + d;
    HostPoly* pol[2] = {&out->U, &out->F};
    for (int k = 0; k < 2; ++k) {
        HostPoly& hp = *pol[k];
        hp.ops.assign(16 * cnt[k] + 8, 0);
        hp.slots.assign(sw * (cnt[k] + 2), 0.0);
        SecEmit em;
        em.slots = hp.slots.data(); em.ops = hp.ops.data(); em.nslots = 0; em.nops = 0; em.status = 0; em.cplx = cplx;
        em.max_slots = cnt[k] + 1; em.max_ops = 16 * cnt[k];
        compile_polynomial(base, cplx ? base + cnt[k] : nullptr, base + (cplx ? 2 : 1) * cnt[k], cnt[k], d, em, &hp.c0, &hp.c0i);
        if (em.status) return false;
        hp.ops.resize(em.nops);
        hp.slots.resize(sw * em.nslots);
        base += cnt[k] * rec;
    }
    return true;
}

// ---- PTX of one case ---------------------------------------------------------------------------------------------------
struct Text {
    std::string s;
    void line(const char* fmt, ...) __attribute__((format(printf, 2, 3))) {
        char buf[256];
        va_list ap;
        va_start(ap, fmt);
        const int n = vsnprintf(buf, sizeof(buf), fmt, ap);
        va_end(ap);
        s.append(buf, (size_t)n);
        s.push_back('\n');
    }
};
std::string imm(double v) {
    unsigned long long u;
    std::memcpy(&u, &v, 8);
    char buf[24];
    snprintf(buf, sizeof(buf), "0d%016llX", u);
    return buf;
}

// The straight-line code of a sector for the G points of a thread; returns the number of temporaries t1.. it names.
int emit_case(const HostSector& hs, int d, const SlotKind& sk, const std::vector<std::string>& o, Text& out) {
    const int G = sk.g, DP = sk.dp;
    auto num = [&](int q) { return o[q].c_str(); };
    auto den = [&](int q) { return o[G + q].c_str(); };
    auto Fo = [&](int q) { return o[2 * G + q].c_str(); };
    auto x = [&](int q, int j) { return o[3 * G + q * DP + j].c_str(); };
    auto W = [&](int q) { return o[3 * G + G * DP + q].c_str(); };
    const char* park = o[3 * G + G * DP + G + 1].c_str();
    int nt = 0;
    auto fresh = [&]() { return "t" + std::to_string(++nt); };
    std::vector<std::string> val[2];                       // U, F at the G points
    const HostPoly* pol[2] = {&hs.U, &hs.F};
    // U and F are independent: their steps are written out alternately, so that the assembler's scheduling window always holds
    // two polynomials' worth of independent chains (each polynomial's own operations keep their order: the values do not change)
    std::vector<std::string> S[2], A[2];
    size_t at[2] = {0, 0};
    int si[2] = {0, 0};
    for (int k = 0; k < 2; ++k) { S[k].assign(G, imm(pol[k]->c0)); A[k].assign(G, imm(0.0)); }
    while (at[0] < hs.U.ops.size() || at[1] < hs.F.ops.size()) {
        for (int k = 0; k < 2; ++k) {
            const HostPoly& hp = *pol[k];
            if (at[k] >= hp.ops.size()) continue;
            const unsigned char code = hp.ops[at[k]++];
            const int j = (code - SEC_BASE) / kSecKinds, kind = (code - SEC_BASE) % kSecKinds;
            std::string cf, cf2;
            if (kind == SEC_SL || kind == SEC_AL || kind == SEC_ALI) { cf = imm(hp.slots[2 * si[k]]); cf2 = imm(hp.slots[2 * si[k] + 1]); ++si[k]; }
            for (int q = 0; q < G; ++q) {
                const std::string t = fresh();
                switch (kind) {
                    case SEC_SC: out.line("fma.rn.f64 %s, %s, %s, %s;", t.c_str(), A[k][q].c_str(), x(q, j), S[k][q].c_str()); S[k][q] = t; break;
                    case SEC_SL: out.line("fma.rn.f64 %s, %s, %s, %s;", t.c_str(), cf.c_str(), x(q, j), S[k][q].c_str()); S[k][q] = t; break;
                    case SEC_AL: out.line("fma.rn.f64 %s, %s, %s, %s;", t.c_str(), cf.c_str(), x(q, j), A[k][q].c_str()); A[k][q] = t; break;
                    case SEC_ALI: out.line("fma.rn.f64 %s, %s, %s, %s;", t.c_str(), cf.c_str(), x(q, j), cf2.c_str()); A[k][q] = t; break;
                    default: out.line("mul.rn.f64 %s, %s, %s;", t.c_str(), A[k][q].c_str(), x(q, j)); A[k][q] = t; break;
                }
            }
        }
    }
    val[0] = S[0]; val[1] = S[1];
    // num = W prod_j x_j^nu_j U^a, den = F^b: the multiplications of the interpreting kernel, in its order
    for (int q = 0; q < G; ++q) {
        std::string n = W(q);
        for (int j = 0; j < d; ++j)
            for (int e = 0; e < hs.nu[j]; ++e) { const std::string t = fresh(); out.line("mul.rn.f64 %s, %s, %s;", t.c_str(), n.c_str(), x(q, j)); n = t; }
        for (int e = 0; e < hs.a; ++e) { const std::string t = fresh(); out.line("mul.rn.f64 %s, %s, %s;", t.c_str(), n.c_str(), val[0][q].c_str()); n = t; }
        out.line("mov.f64 %s, %s;", num(q), n.c_str());
        std::string dn = hs.b > 0 ? val[1][q] : imm(1.0);
        for (int e = 1; e < hs.b; ++e) { const std::string t = fresh(); out.line("mul.rn.f64 %s, %s, %s;", t.c_str(), dn.c_str(), val[1][q].c_str()); dn = t; }
        out.line("mov.f64 %s, %s;", den(q), dn.c_str());
        out.line("mov.f64 %s, %s;", Fo(q), val[1][q].c_str());
        if (hs.logp) {                                     // the log factor reads U from park rows 8 + q (sector_log_factors)
            if (val[0][q][0] == '0') {                     // a constant U: through a register
                const std::string t = fresh();
                out.line("mov.f64 %s, %s;", t.c_str(), val[0][q].c_str());
                out.line("st.shared.f64 [%s+%d], %s;", park, 8 * sk.threads * (8 + q), t.c_str());
            } else {
                out.line("st.shared.f64 [%s+%d], %s;", park, 8 * sk.threads * (8 + q), val[0][q].c_str());
            }
        }
    }
    return nt;
}

// Complex family: the same programs on paired accumulators (two fp64 instructions per step and point); the products with U and F
// are CSectorEval's complex multiplications, t = fma(a, c, -(b d)), fma(a, d, b c), except that the first one, (w, 0) U and
// (1, 0) F, is written as what it evaluates to for finite values (w Ur, w Ui and F itself).
int emit_case_complex(const HostSector& hs, int d, const SlotKind& sk, const std::vector<std::string>& o, Text& out) {
    const int G = sk.g, DP = sk.dp;
    auto outp = [&](int which, int q) { return o[which * G + q].c_str(); };    // nr, ni, dr, di, Fr, Fi, Ur, Ui
    auto x = [&](int q, int j) { return o[8 * G + q * DP + j].c_str(); };
    auto W = [&](int q) { return o[8 * G + G * DP + q].c_str(); };
    int nt = 0;
    auto fresh = [&]() { return "t" + std::to_string(++nt); };
    auto op3 = [&](const char* ins, const std::string& a, const std::string& b, const std::string& c) {
        const std::string t = fresh();
        out.line("%s %s, %s, %s, %s;", ins, t.c_str(), a.c_str(), b.c_str(), c.c_str());
        return t;
    };
    auto mul = [&](const std::string& a, const std::string& b) {
        const std::string t = fresh();
        out.line("mul.rn.f64 %s, %s, %s;", t.c_str(), a.c_str(), b.c_str());
        return t;
    };
    auto neg = [&](const std::string& a) {
        const std::string t = fresh();
        out.line("neg.f64 %s, %s;", t.c_str(), a.c_str());
        return t;
    };
    std::vector<std::string> vr[2], vi[2];                  // U, F at the G points
    const HostPoly* pol[2] = {&hs.U, &hs.F};
    // U and F alternately, step by step (see emit_case)
    std::vector<std::string> Sr[2], Si[2], Ar[2], Ai[2];
    size_t at[2] = {0, 0};
    int si[2] = {0, 0};
    for (int k = 0; k < 2; ++k) { Sr[k].assign(G, imm(pol[k]->c0)); Si[k].assign(G, imm(pol[k]->c0i)); Ar[k].assign(G, imm(0.0)); Ai[k].assign(G, imm(0.0)); }
    while (at[0] < hs.U.ops.size() || at[1] < hs.F.ops.size()) {
        for (int k = 0; k < 2; ++k) {
            const HostPoly& hp = *pol[k];
            if (at[k] >= hp.ops.size()) continue;
            const unsigned char code = hp.ops[at[k]++];
            const int j = (code - SEC_BASE) / kSecKinds, kind = (code - SEC_BASE) % kSecKinds;
            std::string cr, ci, c2r, c2i;
            if (kind == SEC_SL || kind == SEC_AL || kind == SEC_ALI) {
                cr = imm(hp.slots[4 * si[k]]); ci = imm(hp.slots[4 * si[k] + 1]); c2r = imm(hp.slots[4 * si[k] + 2]); c2i = imm(hp.slots[4 * si[k] + 3]);
                ++si[k];
            }
            for (int q = 0; q < G; ++q) {
                const std::string X = x(q, j);
                switch (kind) {
                    case SEC_SC: Sr[k][q] = op3("fma.rn.f64", Ar[k][q], X, Sr[k][q]); Si[k][q] = op3("fma.rn.f64", Ai[k][q], X, Si[k][q]); break;
                    case SEC_SL: Sr[k][q] = op3("fma.rn.f64", cr, X, Sr[k][q]); Si[k][q] = op3("fma.rn.f64", ci, X, Si[k][q]); break;
                    case SEC_AL: Ar[k][q] = op3("fma.rn.f64", cr, X, Ar[k][q]); Ai[k][q] = op3("fma.rn.f64", ci, X, Ai[k][q]); break;
                    case SEC_ALI: Ar[k][q] = op3("fma.rn.f64", cr, X, c2r); Ai[k][q] = op3("fma.rn.f64", ci, X, c2i); break;
                    default: Ar[k][q] = mul(Ar[k][q], X); Ai[k][q] = mul(Ai[k][q], X); break;
                }
            }
        }
    }
    for (int k = 0; k < 2; ++k) { vr[k] = Sr[k]; vi[k] = Si[k]; }
    auto in_register = [&](const std::string& v) {           // a polynomial without steps is a constant: through a register
        if (v[0] != '0') return v;
        const std::string t = fresh();
        out.line("mov.f64 %s, %s;", t.c_str(), v.c_str());
        return t;
    };
    for (int q = 0; q < G; ++q) {
        const std::string Ur = in_register(vr[0][q]), Ui = in_register(vi[0][q]), Fr = in_register(vr[1][q]), Fi = in_register(vi[1][q]);
        std::string w = W(q);
        for (int j = 0; j < d; ++j)
            for (int e = 0; e < hs.nu[j]; ++e) w = mul(w, x(q, j));
        std::string nr = w, ni = imm(0.0);
        for (int e = 0; e < hs.a; ++e) {
            if (e == 0) { nr = mul(w, Ur); ni = mul(w, Ui); continue; }
            const std::string t = op3("fma.rn.f64", nr, Ur, neg(mul(ni, Ui)));
            ni = op3("fma.rn.f64", nr, Ui, mul(ni, Ur));
            nr = t;
        }
        std::string dr = imm(1.0), di = imm(0.0);
        for (int e = 0; e < hs.b; ++e) {
            if (e == 0) { dr = Fr; di = Fi; continue; }
            const std::string t = op3("fma.rn.f64", dr, Fr, neg(mul(di, Fi)));
            di = op3("fma.rn.f64", dr, Fi, mul(di, Fr));
            dr = t;
        }
        const std::string* vals[8] = {&nr, &ni, &dr, &di, &Fr, &Fi, &Ur, &Ui};
        for (int k = 0; k < 8; ++k) out.line("mov.f64 %s, %s;", outp(k, q), vals[k]->c_str());
    }
    return nt;
}

struct Kernel {                                 // one specialised kernel: up to sectors_per_kernel sectors of one slot kind
    int kind = 0;                               // index into kSlotKinds
    std::vector<int> problems;                  // indices into the batch, case order
    std::vector<char> image;                    // the assembled sm_100a image
    std::string log;                            // assembler messages (errors; with --verbose the register report)
    bool ok = false;
};

// ---- the assembler: nvJitLink (PTX -> sm_100a image), loaded at run time ---------------------------------------------------
// The toolkit's shared library is opened on first use -- linking the static PTX compiler would add 150 MB to this library.
// A PTX-only link runs the PTX assembler once per kernel; handles are independent, so kernels assemble in parallel.
struct Assembler {
    typedef void* Handle;
    int (*Create)(Handle*, uint32_t, const char**) = nullptr;
    int (*Destroy)(Handle*) = nullptr;
    int (*AddData)(Handle, int, const void*, size_t, const char*) = nullptr;
    int (*Complete)(Handle) = nullptr;
    int (*GetLinkedCubinSize)(Handle, size_t*) = nullptr;
    int (*GetLinkedCubin)(Handle, void*) = nullptr;
    int (*GetErrorLogSize)(Handle, size_t*) = nullptr;
    int (*GetErrorLog)(Handle, char*) = nullptr;
    int (*GetInfoLogSize)(Handle, size_t*) = nullptr;
    int (*GetInfoLog)(Handle, char*) = nullptr;
    std::string why;                                 // empty: usable
};
const Assembler& assembler() {
    static const Assembler a = [] {
        Assembler r;
        // the toolkit the template was compiled with first (its PTX version is the newest this nvcc writes)
        const char* names[] = {"/usr/local/cuda/lib64/libnvJitLink.so.12", "libnvJitLink.so.12", "libnvJitLink.so"};
        void* lib = nullptr;
        for (const char* n : names)
            if ((lib = dlopen(n, RTLD_NOW | RTLD_LOCAL))) break;
        if (!lib) { r.why = "libnvJitLink.so.12 (CUDA toolkit) could not be opened"; return r; }
        bool ok = true;
        auto get = [&](const char* name, void** fn) { *fn = dlsym(lib, name); if (!*fn) ok = false; };
        get("nvJitLinkCreate", reinterpret_cast<void**>(&r.Create));
        get("nvJitLinkDestroy", reinterpret_cast<void**>(&r.Destroy));
        get("nvJitLinkAddData", reinterpret_cast<void**>(&r.AddData));
        get("nvJitLinkComplete", reinterpret_cast<void**>(&r.Complete));
        get("nvJitLinkGetLinkedCubinSize", reinterpret_cast<void**>(&r.GetLinkedCubinSize));
        get("nvJitLinkGetLinkedCubin", reinterpret_cast<void**>(&r.GetLinkedCubin));
        get("nvJitLinkGetErrorLogSize", reinterpret_cast<void**>(&r.GetErrorLogSize));
        get("nvJitLinkGetErrorLog", reinterpret_cast<void**>(&r.GetErrorLog));
        get("nvJitLinkGetInfoLogSize", reinterpret_cast<void**>(&r.GetInfoLogSize));
        get("nvJitLinkGetInfoLog", reinterpret_cast<void**>(&r.GetInfoLog));
        if (!ok) r.why = "libnvJitLink.so.12 lacks an entry point";
        return r;
    }();
    return a;
}

bool assemble(const std::string& ptx, Kernel* k) {
    const Assembler& as = assembler();
    if (!as.why.empty()) { k->log = as.why; return false; }
    Assembler::Handle h = nullptr;
    const char* opts[] = {"-arch=sm_100a", "-verbose"};
    if (as.Create(&h, 2, opts) != 0) { k->log = "nvJitLinkCreate failed"; return false; }
    constexpr int kInputPtx = 2;                     // NVJITLINK_INPUT_PTX
    int rc = as.AddData(h, kInputPtx, ptx.c_str(), ptx.size() + 1, "qmc_spec");
    if (rc == 0) rc = as.Complete(h);
    size_t n = 0;
    if (rc != 0) {
        if (as.GetErrorLogSize(h, &n) == 0 && n) { k->log.resize(n + 1); as.GetErrorLog(h, &k->log[0]); }
        else k->log = "nvJitLink failed with code " + std::to_string(rc);
        as.Destroy(&h);
        return false;
    }
    if (as.GetInfoLogSize(h, &n) == 0 && n) { k->log.resize(n + 1); as.GetInfoLog(h, &k->log[0]); }
    bool ok = as.GetLinkedCubinSize(h, &n) == 0 && n > 0;
    if (ok) { k->image.resize(n); ok = as.GetLinkedCubin(h, k->image.data()) == 0; }
    as.Destroy(&h);
    return ok;
}

// ---- driver entry points, through the runtime (the library does not link libcuda) ---------------------------------------
struct Driver {
    CUresult (*ModuleLoadData)(CUmodule*, const void*) = nullptr;
    CUresult (*ModuleUnload)(CUmodule) = nullptr;
    CUresult (*ModuleGetFunction)(CUfunction*, CUmodule, const char*) = nullptr;
    CUresult (*FuncSetAttribute)(CUfunction, CUfunction_attribute, int) = nullptr;
    CUresult (*OccupancyMaxActiveBlocksPerMultiprocessor)(int*, CUfunction, int, size_t) = nullptr;
    CUresult (*LaunchKernel)(CUfunction, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, CUstream, void**, void**) = nullptr;
    CUresult (*GetErrorString)(CUresult, const char**) = nullptr;
    bool ok = false;
};
const Driver& driver() {
    static const Driver d = [] {
        Driver r;
        cudaFree(nullptr);                                  // the runtime's primary context becomes current
        bool ok = true;
        auto get = [&](const char* name, void** fn) {
            cudaDriverEntryPointQueryResult qr;
            if (cudaGetDriverEntryPoint(name, fn, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess || !*fn) ok = false;
        };
        get("cuModuleLoadData", reinterpret_cast<void**>(&r.ModuleLoadData));
        get("cuModuleUnload", reinterpret_cast<void**>(&r.ModuleUnload));
        get("cuModuleGetFunction", reinterpret_cast<void**>(&r.ModuleGetFunction));
        get("cuFuncSetAttribute", reinterpret_cast<void**>(&r.FuncSetAttribute));
        get("cuOccupancyMaxActiveBlocksPerMultiprocessor", reinterpret_cast<void**>(&r.OccupancyMaxActiveBlocksPerMultiprocessor));
        get("cuLaunchKernel", reinterpret_cast<void**>(&r.LaunchKernel));
        get("cuGetErrorString", reinterpret_cast<void**>(&r.GetErrorString));
        r.ok = ok;
        return r;
    }();
    return d;
}

struct Loaded {                                 // a kernel on one device
    CUmodule mod = nullptr;
    CUfunction fn = nullptr;
    int occ = 0;
};

}  // namespace
}  // namespace qmc

using namespace qmc;

struct qmc_sector_module {
    std::vector<SpecProblem> problems;
    std::vector<Kernel> kernels;
    double build_ms = 0.0;
    int threads_used = 0;
    std::mutex mu;
    std::map<int, std::vector<Loaded>> loaded;  // per device ordinal
};

namespace qmc {
namespace {

int driver_fail(CUresult rc, const char* where) {
    const char* msg = nullptr;
    if (driver().GetErrorString) driver().GetErrorString(rc, &msg);
    report_cuda_error(cudaErrorUnknown, (std::string(where) + ": " + (msg ? msg : "driver error")).c_str());
    return QMC_ERR_CUDA;
}

// the module's kernels on the current device, loaded on first use; nullptr after a failure (text in qmc_last_cuda_error)
const std::vector<Loaded>* loaded_on_current_device(qmc_sector_module* mod) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { report_cuda_error(cudaErrorNoDevice, "no CUDA device"); return nullptr; }
    std::lock_guard<std::mutex> lock(mod->mu);
    auto it = mod->loaded.find(dev);
    if (it != mod->loaded.end()) return &it->second;
    const Driver& drv = driver();
    if (!drv.ok) { report_cuda_error(cudaErrorNotSupported, "driver entry points for module loading unavailable"); return nullptr; }
    std::vector<Loaded> v(mod->kernels.size());
    auto unload = [&]() { for (Loaded& l : v) if (l.mod) drv.ModuleUnload(l.mod); };
    for (size_t i = 0; i < mod->kernels.size(); ++i) {
        const Kernel& k = mod->kernels[i];
        const SlotKind& sk = kSlotKinds[k.kind];
        CUresult rc = drv.ModuleLoadData(&v[i].mod, k.image.data());
        if (rc == CUDA_SUCCESS) rc = drv.ModuleGetFunction(&v[i].fn, v[i].mod, sk.entry);
        if (rc == CUDA_SUCCESS) rc = drv.FuncSetAttribute(v[i].fn, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)sk.smem);
        if (rc == CUDA_SUCCESS) rc = drv.OccupancyMaxActiveBlocksPerMultiprocessor(&v[i].occ, v[i].fn, sk.threads, sk.smem);
        if (rc != CUDA_SUCCESS) { driver_fail(rc, "loading a specialised sector kernel (is this an sm_100a device?)"); unload(); return nullptr; }
        if (v[i].occ < 1) { report_cuda_error(cudaErrorLaunchOutOfResources, "specialised sector kernel does not fit an SM"); unload(); return nullptr; }
    }
    return &(mod->loaded[dev] = std::move(v));
}

}  // namespace

int spec_problem_count(const qmc_sector_module* mod) { return (int)mod->problems.size(); }
const SpecProblem* spec_problems(const qmc_sector_module* mod) { return mod->problems.data(); }
int spec_kernel_dp(const qmc_sector_module* mod, int kernel) { return kSlotKinds[mod->kernels[kernel].kind].dp; }
int spec_kernel_threads(const qmc_sector_module* mod, int kernel) { return kSlotKinds[mod->kernels[kernel].kind].threads; }

int spec_occupancy(qmc_sector_module* mod, int kernel) {
    const std::vector<Loaded>* l = loaded_on_current_device(mod);
    return l ? (*l)[kernel].occ : -1;
}

int spec_launch(qmc_sector_module* mod, int kernel, int grid, cudaStream_t st, const FusedLaunch& a) {
    const std::vector<Loaded>* l = loaded_on_current_device(mod);
    if (!l) return QMC_ERR_CUDA;
    const SlotKind& sk = kSlotKinds[mod->kernels[kernel].kind];
    FusedLaunch arg = a;
    void* args[] = {&arg};
    const CUresult rc = driver().LaunchKernel((*l)[kernel].fn, (unsigned)grid, 1, 1, (unsigned)sk.threads, 1, 1, (unsigned)sk.smem,
                                              reinterpret_cast<CUstream>(st), args, nullptr);
    return rc == CUDA_SUCCESS ? QMC_OK : driver_fail(rc, "specialised sector kernel launch");
}

}  // namespace qmc

extern "C" {

int qmc_sector_module_create(int count, const qmc_problem* problems, int sectors_per_kernel, qmc_sector_module** out) {
    if (!problems || !out) return QMC_ERR_NULL;
    *out = nullptr;
    if (count < 1) return QMC_ERR_N;
    if (sectors_per_kernel < 0 || sectors_per_kernel > 1024) return QMC_ERR_N;
    const bool auto_size = sectors_per_kernel == 0;
    if (auto_size) sectors_per_kernel = 32;
    const Template& tpl = kernel_template();
    if (!tpl.ok) { report_cuda_error(cudaErrorUnknown, "the embedded kernel template has no usable marker"); return QMC_ERR_CUDA; }
    const auto t0 = std::chrono::steady_clock::now();
    qmc_sector_module* mod = new qmc_sector_module;
    mod->problems.resize(count);
    std::vector<HostSector> sectors(count);
    std::vector<int> by_kind[kSlotKindCount];
    for (int i = 0; i < count; ++i) {
        const qmc_problem& p = problems[i];
        SpecProblem& sp = mod->problems[i];
        sp.family = p.family; sp.dim = p.dim; sp.n_params = p.n_params; sp.kernel = -1; sp.kase = 0;
        if (!is_sector_family(p.family) || !p.params || p.dim < 1 || p.dim > QMC_MAX_SECTOR_DIM) continue;
        const bool cplx = p.family == QMC_FAMILY_SECTOR_COMPLEX;
        const int kind = slot_kind_of(sector_dim_slots(p.dim), cplx);
        if (kind < 0 || !compile_sector_host(p.params, p.n_params, p.dim, cplx, &sectors[i])) continue;   // the interpreting kernel reports a bad block
        by_kind[kind].push_back(i);
    }
    if (auto_size) {
        // a batch call serves at most 64 kernel variants: with many sectors, more of them share a kernel (at most kMaxAutoKernels
        // kernels, the rest of the variants is left to the batch's other families)
        constexpr size_t kMaxAutoKernels = 48;
        auto kernels_at = [&](size_t per) { size_t n = 0; for (auto& v : by_kind) n += (v.size() + per - 1) / per; return n; };
        while (kernels_at((size_t)sectors_per_kernel) > kMaxAutoKernels && sectors_per_kernel < 1024) sectors_per_kernel *= 2;
    }
    for (int kind = 0; kind < kSlotKindCount; ++kind)
        for (size_t b = 0; b < by_kind[kind].size(); b += (size_t)sectors_per_kernel) {
            Kernel k;
            k.kind = kind;
            const size_t e = std::min(by_kind[kind].size(), b + (size_t)sectors_per_kernel);
            k.problems.assign(by_kind[kind].begin() + b, by_kind[kind].begin() + e);
            for (size_t c = 0; c < k.problems.size(); ++c) {
                mod->problems[k.problems[c]].kernel = (int)mod->kernels.size();
                mod->problems[k.problems[c]].kase = (int)c;
            }
            mod->kernels.push_back(std::move(k));
        }
    // emit and assemble, one kernel per task
    std::atomic<size_t> next{0};
    auto work = [&]() {
        for (size_t i = next.fetch_add(1); i < mod->kernels.size(); i = next.fetch_add(1)) {
            Kernel& k = mod->kernels[i];
            const SlotKind& sk = kSlotKinds[k.kind];
            const EntryText& et = tpl.entry[k.kind];
            Text code;
            int max_t = 0;
            for (size_t c = 0; c < k.problems.size(); ++c) {
                code.line("QMC_CASE_%zu:", c);
                max_t = std::max(max_t, sk.cplx ? emit_case_complex(sectors[k.problems[c]], problems[k.problems[c]].dim, sk, et.operands, code)
                                                : emit_case(sectors[k.problems[c]], problems[k.problems[c]].dim, sk, et.operands, code));
                code.line("bra.uni QMC_SITE_DONE;");
            }
            std::string ptx;
            ptx.reserve(tpl.header.size() + et.before.size() + et.after.size() + code.s.size() + 64 * k.problems.size() + 256);
            ptx += tpl.header;
            ptx += et.before;
            ptx += "{\n.reg .f64 t<" + std::to_string(max_t + 1) + ">;\nqmc_cases: .branchtargets ";
            for (size_t c = 0; c < k.problems.size(); ++c) ptx += (c ? ", QMC_CASE_" : "QMC_CASE_") + std::to_string(c);
            ptx += ";\nbrx.idx.uni " + et.operands[et.operands.size() - (sk.cplx ? 1 : 2)] + ", qmc_cases;\n";
            ptx += code.s;
            ptx += "QMC_SITE_DONE:\n}";
            ptx += et.after;
            k.ok = assemble(ptx, &k);
        }
    };
    const unsigned hw = std::max(1u, std::thread::hardware_concurrency());
    const size_t nthreads = std::min<size_t>(mod->kernels.size(), hw);
    std::vector<std::thread> pool;
    for (size_t t = 1; t < nthreads; ++t) pool.emplace_back(work);
    work();
    for (auto& th : pool) th.join();
    mod->threads_used = (int)std::max<size_t>(nthreads, 1);
    for (const Kernel& k : mod->kernels)
        if (!k.ok) {
            report_cuda_error(cudaErrorInvalidPtx, ("assembling a specialised sector kernel: " + k.log).c_str());
            delete mod;
            return QMC_ERR_CUDA;
        }
    mod->build_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    *out = mod;
    return QMC_OK;
}

void qmc_sector_module_destroy(qmc_sector_module* mod) {
    if (!mod) return;
    for (auto& dev : mod->loaded)
        for (Loaded& l : dev.second)
            if (l.mod && driver().ModuleUnload) driver().ModuleUnload(l.mod);
    delete mod;
}

int qmc_sector_module_info(const qmc_sector_module* mod, int* n_specialised, int* n_kernels, double* build_ms, size_t* image_bytes,
                           int* host_threads) {
    if (!mod) return QMC_ERR_NULL;
    int ns = 0;
    size_t bytes = 0;
    for (const SpecProblem& p : mod->problems) ns += p.kernel >= 0;
    for (const Kernel& k : mod->kernels) bytes += k.image.size();
    if (n_specialised) *n_specialised = ns;
    if (n_kernels) *n_kernels = (int)mod->kernels.size();
    if (build_ms) *build_ms = mod->build_ms;
    if (image_bytes) *image_bytes = bytes;
    if (host_threads) *host_threads = mod->threads_used;
    return QMC_OK;
}

// kernel `kernel`'s assembled image (for cuobjdump / nvdisasm) and the assembler's report; sizes via null buffers
int qmc_sector_module_image(const qmc_sector_module* mod, int kernel, void* image, size_t image_cap, size_t* image_bytes, char* log,
                            size_t log_cap) {
    if (!mod) return QMC_ERR_NULL;
    if (kernel < 0 || kernel >= (int)mod->kernels.size()) return QMC_ERR_N;
    const Kernel& k = mod->kernels[kernel];
    if (image_bytes) *image_bytes = k.image.size();
    if (image) {
        if (image_cap < k.image.size()) return QMC_ERR_WORKSPACE;
        std::memcpy(image, k.image.data(), k.image.size());
    }
    if (log && log_cap) {
        const size_t n = std::min(log_cap - 1, std::strlen(k.log.c_str()));
        std::memcpy(log, k.log.c_str(), n);
        log[n] = 0;
    }
    return QMC_OK;
}

}  // extern "C"
