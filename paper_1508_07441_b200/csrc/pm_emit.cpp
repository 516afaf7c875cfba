// pm_emit.cpp — emits the channel-specialised ket code of the fill kernel as CUDA source text (see pm_emit.hpp).
#include "pm_emit.hpp"

#include <cinttypes>
#include <cstdio>
#include <map>
#include <sstream>
#include <vector>

namespace pm {

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

}  // namespace

std::string emit_spec(const std::string& name, const KetView& V, EmitStats& st)
{
    struct { int n_slot; const std::vector<int32_t>&kt_off, &kt_ip, &kt_iq; const std::vector<double>& kt_c; const std::vector<OrbFun>& fun; }
        T{V.n_slot, *V.kt_off, *V.kt_ip, *V.kt_iq, *V.kt_c, *V.fun};
    auto l_of = [](int idx) { int l = 0; while (ylm_index(l + 1, 0) <= idx) ++l; return l; };
    int la = 0, lb = 0;
    for (size_t t = 0; t < T.kt_c.size(); ++t) { la = std::max(la, l_of(T.kt_ip[t])); lb = std::max(lb, l_of(T.kt_iq[t])); }
    std::vector<double> ynorm, ybeta;
    scaled_harmonics(std::max(la, lb), ynorm, ybeta);
    std::ostringstream o;
    const int nf = (int)T.fun.size();
    o << "struct Spec_" << name << " {\n";
    o << "    static constexpr bool kStatic = true;\n";
    int maxm = 1, maxl1 = 1;                        // most M-terms of a function; number of L values (terms per output)
    for (const OrbFun& f : T.fun) { maxm = std::max(maxm, f.nM); maxl1 = std::max(maxl1, f.L + 1); }
    if (V.n_bra > 254) maxm = std::max(maxm, 4);   // the packed descriptors (MAXM <= 3) hold bra slots in 8 bits
    o << "    static constexpr int NS = " << T.n_slot << ", NF = " << nf << ", NCH = " << (nf + 31) / 32 << ", MAXM = " << maxm << ", MAXL1 = " << maxl1 << ";\n";
    o << "    // most M-terms of the 32 functions step ch of the stage handles\n"
         "    static __device__ __forceinline__ constexpr int terms(int ch) { return ";
    for (int c = 0; c < (nf + 31) / 32; ++c) {
        int m = 1;
        for (int f = 32 * c; f < std::min(nf, 32 * c + 32); ++f) m = std::max(m, T.fun[(size_t)f].nM);
        if (c + 1 < (nf + 31) / 32) o << "ch == " << c << " ? " << m << " : ";
        else o << m;
    }
    o << "; }\n";
    o << "    static constexpr int NOT = " << V.n_oterm << ";            // terms per output kept in shared memory\n";
    o << "    static constexpr bool kOutTail = " << (V.oterm_tail ? "true" : "false") << ";     // some output has more terms than that\n";
    o << "    static constexpr bool kBraSmem = " << (V.bra_smem ? "true" : "false") << ";      // bra harmonics in shared / global memory\n";
    char hb[32]; std::snprintf(hb, sizeof hb, "0x%016" PRIx64 "ull", (uint64_t)V.hash);
    o << "    static constexpr unsigned long long kHash = " << hb << ";\n";
    o << "    // K[s] += omega * (ket bipolar harmonic of slot s) at directions a = p'^ = (uxa,0,uza), b = q'^ = (uxb,0,uzb)\n";
    o << "    static __device__ __forceinline__ void ket_acc(const DevLattice&, double om, double uxa, double uza, double uxb, double uzb,\n"
         "                                                   double (&K)[NS])\n    {\n";
    emit_q(o, 'a', la, "om", "uxa", "uza", ybeta);
    // The q' side harmonic by harmonic (m-major recurrence): each b_lm is multiplied into its products and those into the
    // running sums K[s] at once, so only the p' side harmonics and two or three b values are live at any point (the
    // accumulators K take 2*NS registers; short live ranges are what keeps the rest of the kernel out of local memory).
    std::map<std::pair<int, int>, std::vector<size_t>> terms;             // (iq, ip) -> ket terms
    for (int s = 0; s < T.n_slot; ++s)
        for (int t = T.kt_off[(size_t)s]; t < T.kt_off[(size_t)s + 1]; ++t) terms[{T.kt_iq[(size_t)t], T.kt_ip[(size_t)t]}].push_back((size_t)t);
    std::vector<int> slot_of(T.kt_c.size());
    for (int s = 0; s < T.n_slot; ++s)
        for (int t = T.kt_off[(size_t)s]; t < T.kt_off[(size_t)s + 1]; ++t) slot_of[(size_t)t] = s;
    for (int m = 0; m <= lb; ++m) {
        for (int l = m; l <= lb; ++l) {
            const int iq = ylm_index(l, m);
            const std::string bn = yname('b', iq);
            o << "        const double " << bn << " = ";
            if (l == 0) o << "1.0;\n";
            else if (l == m) o << "uxb * " << yname('b', ylm_index(m - 1, m - 1)) << ";\n";
            else if (l == m + 1) o << "uzb * " << yname('b', ylm_index(l - 1, m)) << ";\n";
            else o << "fma(uzb, " << yname('b', ylm_index(l - 1, m)) << ", " << num(-ybeta[(size_t)iq]) << " * " << yname('b', ylm_index(l - 2, m)) << ");\n";
            for (auto it = terms.lower_bound({iq, -1}); it != terms.end() && it->first.first == iq; ++it) {
                const int ip = it->first.second;
                const std::string p = "t" + std::to_string(ip) + "_" + std::to_string(iq);
                o << "        { const double " << p << " = " << yname('a', ip) << " * " << bn << ";";
                st.n_prod++;
                for (size_t t : it->second) {
                    const double c = T.kt_c[t] * ynorm[(size_t)T.kt_ip[t]] * ynorm[(size_t)T.kt_iq[t]];
                    const int s = slot_of[t];
                    o << " K[" << s << "] = fma(" << num(c) << ", " << p << ", K[" << s << "]);";
                    st.n_fma++;
                }
                o << " }\n";
            }
        }
    }
    o << "    }\n};\n\n";
    return o.str();
}


}  // namespace pm
