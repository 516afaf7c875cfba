// pm_codegen.cpp — build-time generator of the channel-specialised ket code of the fill kernel.
//
// Why: the ket side of eq. (22)'s angular part is, per quadrature node,
//   K[slot] = omega * sum_terms c * Y_{l' m}(p'^) * Y_{lam' mu}(q'^)
// with a few hundred terms fixed by the channel set.  Driven by tables it is bound by shared-memory loads
// (the paper's complaint about constants in global memory, L341, one level up); written out as straight-line
// code the harmonics live in registers, the coefficients are immediates and only FP64 instructions remain.
// This tool turns the host tables (pm_tables.cpp — the same ones the library builds at run time) of the channel
// sets listed in its input file into `gen/pm_spec_gen.cuh`; pm_fill picks a generated kernel when the hash of
// the lattice's tables equals the hash stored with it, and the table-driven kernel otherwise.
//
// Input (text): per set  "name J2 parity T2 statistics n_ch"  then n_ch lines  "l s j t lam I2".
// Usage: pm_codegen <sets.txt> <out.cuh>
#include <cinttypes>
#include <cstdio>
#include <fstream>
#include <map>
#include <set>
#include <sstream>
#include <string>
#include <vector>

#include "pm_tables.hpp"

using namespace pm;

namespace {

std::string num(double v)
{
    char buf[64];
    std::snprintf(buf, sizeof buf, "%.17g", v);
    std::string s(buf);
    if (s.find_first_of(".eEn") == std::string::npos) s += ".0";
    return s;
}

std::string yname(char side, int idx)
{
    int l = 0;
    while (ylm_index(l + 1, 0) <= idx) ++l;
    return std::string(1, side) + std::to_string(l) + "_" + std::to_string(idx - ylm_index(l, 0));
}

// scaled harmonics Q_lm of one direction, seed `seed` (omega for the p' side, 1 for the q' side)
void emit_q(std::ostringstream& o, char side, int lmax, const std::string& seed, const std::string& ux, const std::string& uz,
            const std::vector<double>& beta)
{
    o << "        const double " << yname(side, 0) << " = " << seed << ";\n";
    for (int m = 0; m <= lmax; ++m) {
        if (m > 0)
            o << "        const double " << yname(side, ylm_index(m, m)) << " = " << ux << " * " << yname(side, ylm_index(m - 1, m - 1)) << ";\n";
        for (int l = m + 1; l <= lmax; ++l) {
            o << "        const double " << yname(side, ylm_index(l, m)) << " = ";
            if (l == m + 1) o << uz << " * " << yname(side, ylm_index(l - 1, m)) << ";\n";
            else o << "fma(" << uz << ", " << yname(side, ylm_index(l - 1, m)) << ", " << num(-beta[(size_t)ylm_index(l, m)]) << " * "
                   << yname(side, ylm_index(l - 2, m)) << ");\n";
        }
    }
}

struct Stats { int n_prod = 0, n_fma = 0, n_mul = 0; };

std::string emit_spec(const std::string& name, const Tables& T, Stats& st)
{
    std::vector<double> ynorm, ybeta;
    scaled_harmonics(T.lmax, ynorm, ybeta);
    int la = 0, lb = 0;
    for (const Triple& t : T.tri) { la = std::max(la, t.l); lb = std::max(lb, t.lam); }
    std::ostringstream o;
    const int nf = (int)T.fun.size();
    o << "struct Spec_" << name << " {\n";
    o << "    static constexpr bool kStatic = true;\n";
    int maxm = 1, maxl1 = 1;                        // most M-terms of a function; number of L values (terms per output)
    for (const OrbFun& f : T.fun) { maxm = std::max(maxm, f.nM); maxl1 = std::max(maxl1, f.L + 1); }
    o << "    static constexpr int NS = " << T.n_slot << ", NF = " << nf << ", NCH = " << (nf + 31) / 32 << ", MAXM = " << maxm << ", MAXL1 = " << maxl1 << ";\n";
    char hb[32]; std::snprintf(hb, sizeof hb, "0x%016" PRIx64 "ull", tables_hash(T));
    o << "    static constexpr unsigned long long kHash = " << hb << ";\n";
    o << "    // K[s] = omega * (ket bipolar harmonic of slot s) at directions a = p'^ = (uxa,0,uza), b = q'^ = (uxb,0,uzb)\n";
    o << "    static __device__ __forceinline__ void ket(const DevLattice&, double om, double uxa, double uza, double uxb, double uzb,\n"
         "                                               double (&K)[NS])\n    {\n";
    emit_q(o, 'a', la, "om", "uxa", "uza", ybeta);
    emit_q(o, 'b', lb, "1.0", "uxb", "uzb", ybeta);
    // products shared by several terms
    std::map<std::pair<int, int>, int> uses;
    for (size_t t = 0; t < T.kt_c.size(); ++t) uses[{T.kt_ip[t], T.kt_iq[t]}]++;
    for (auto& kv : uses) {
        o << "        const double t" << kv.first.first << "_" << kv.first.second << " = " << yname('a', kv.first.first) << " * "
          << yname('b', kv.first.second) << ";\n";
        st.n_prod++;
    }
    for (int s = 0; s < T.n_slot; ++s) {
        const int b = T.kt_off[(size_t)s], e = T.kt_off[(size_t)s + 1];
        if (b == e) { o << "        K[" << s << "] = 0.0;\n"; continue; }
        std::string expr;
        for (int t = b; t < e; ++t) {
            const double c = T.kt_c[(size_t)t] * ynorm[(size_t)T.kt_ip[(size_t)t]] * ynorm[(size_t)T.kt_iq[(size_t)t]];
            const std::string p = "t" + std::to_string(T.kt_ip[(size_t)t]) + "_" + std::to_string(T.kt_iq[(size_t)t]);
            if (t == b) { expr = num(c) + " * " + p; st.n_mul++; }
            else { expr = "fma(" + num(c) + ", " + p + ", " + expr + ")"; st.n_fma++; }
        }
        o << "        K[" << s << "] = " << expr << ";\n";
    }
    o << "    }\n};\n\n";
    return o.str();
}

}  // namespace

int main(int argc, char** argv)
{
    if (argc != 3) { std::fprintf(stderr, "usage: pm_codegen <sets.txt> <out.cuh>\n"); return 2; }
    std::ifstream in(argv[1]);
    if (!in) { std::fprintf(stderr, "cannot read %s\n", argv[1]); return 2; }
    std::ostringstream out, reg;
    out << "// GENERATED by pm_codegen (csrc/pm_codegen.cpp) from the channel sets of csrc/build.py — do not edit.\n"
           "// One struct per channel set: the ket-side bipolar harmonics of eq. (22)'s angular part (DESIGN.md sec. 3.2)\n"
           "// as straight-line FP64 code; scaled harmonics Q_lm (pm_tables.hpp) with the norms folded into the coefficients,\n"
           "// omega folded into the seed of the p' side.\n#pragma once\n\nnamespace pm {\nnamespace gen {\n\n";
    std::string name;
    int J2, parity, T2, stat, n_ch, n_sets = 0;
    std::set<uint64_t> seen;
    while (in >> name >> J2 >> parity >> T2 >> stat >> n_ch) {
        std::vector<pm_channel> ch((size_t)n_ch);
        for (auto& c : ch) in >> c.l >> c.s >> c.j >> c.t >> c.lam >> c.I2;
        std::string msg = validate_channels(ch.data(), n_ch, J2, parity, T2, stat);
        Tables T;
        if (msg.empty()) msg = build_tables(ch.data(), n_ch, J2, T2, stat, T);
        if (!msg.empty()) { std::fprintf(stderr, "set %s: %s\n", name.c_str(), msg.c_str()); return 1; }
        if (!seen.insert(tables_hash(T)).second) {      // same ket tables as an earlier set: one kernel serves both
            out << "// " << name << ": same ket tables as an earlier set\n\n";
            continue;
        }
        Stats st;
        out << "// " << name << ": " << n_ch << " channels, " << T.n_slot << " slots, " << T.fun.size() << " orbital functions, "
            << T.kt_c.size() << " ket terms\n" << emit_spec(name, T, st);
        reg << "    PM_SPEC(Spec_" << name << ")\n";
        std::fprintf(stderr, "pm_codegen: %s  n_ch=%d slots=%d fun=%zu terms=%zu products=%d mul=%d fma=%d\n", name.c_str(), n_ch,
                     T.n_slot, T.fun.size(), T.kt_c.size(), st.n_prod, st.n_mul, st.n_fma);
        ++n_sets;
    }
    out << "}  // namespace gen\n}  // namespace pm\n\n// registry: expands PM_SPEC(S) once per generated struct\n#define PM_SPEC_LIST \\\n";
    std::string r = reg.str();
    for (size_t i = 0; i < r.size(); ++i) { if (r[i] == '\n') out << (i + 1 < r.size() ? " \\\n" : "\n"); else out << r[i]; }
    if (n_sets == 0) out << "\n";
    std::ofstream f(argv[2]);
    f << out.str();
    return f ? 0 : 1;
}
