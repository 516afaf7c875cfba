// pm_tables.cpp — host precompute for libpm (see pm_tables.hpp).  Shares no code with oracle/.
#include "pm_tables.hpp"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <map>
#include <tuple>

#include "pm_ylm.h"

namespace pm {

namespace {

constexpr double kPi = 3.14159265358979323846;

// ln n! table: the Racah sums below are evaluated as exp(sum of logs) per term, which keeps
// every term O(1) regardless of the size of the momenta.
struct LogFact {
    std::vector<double> t;
    LogFact() : t(256, 0.0) { for (size_t i = 1; i < t.size(); ++i) t[i] = t[i - 1] + std::log((double)i); }
    double operator()(int n) const { return t[(size_t)n]; }
};
const LogFact& lf() { static LogFact f; return f; }

inline bool tri_ok(int a, int b, int c) { return ((a + b + c) % 2 == 0) && c >= std::abs(a - b) && c <= a + b; }

// ln of the triangle coefficient (doubled arguments)
inline double ln_delta(int a, int b, int c)
{
    return lf()((a + b - c) / 2) + lf()((a - b + c) / 2) + lf()((-a + b + c) / 2) - lf()((a + b + c) / 2 + 1);
}

}  // namespace

// <j1 m1 j2 m2 | j3 m3>, Racah's closed form
double clebsch(int j1, int m1, int j2, int m2, int j3, int m3)
{
    if (m1 + m2 != m3 || !tri_ok(j1, j2, j3)) return 0.0;
    if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(m3) > j3) return 0.0;
    if (((j1 + m1) | (j2 + m2) | (j3 + m3)) & 1) return 0.0;
    const double lnpref = 0.5 * (std::log((double)(j3 + 1)) + ln_delta(j1, j2, j3)
        + lf()((j1 + m1) / 2) + lf()((j1 - m1) / 2) + lf()((j2 + m2) / 2) + lf()((j2 - m2) / 2)
        + lf()((j3 + m3) / 2) + lf()((j3 - m3) / 2));
    const int a = (j1 + j2 - j3) / 2, b = (j1 - m1) / 2, c = (j2 + m2) / 2;
    const int d = (j3 - j2 + m1) / 2, e = (j3 - j1 - m2) / 2;
    const int kmin = std::max(0, std::max(-d, -e)), kmax = std::min(a, std::min(b, c));
    double sum = 0.0;
    for (int k = kmin; k <= kmax; ++k) {
        double ln = lnpref - (lf()(k) + lf()(a - k) + lf()(b - k) + lf()(c - k) + lf()(d + k) + lf()(e + k));
        sum += (k & 1) ? -std::exp(ln) : std::exp(ln);
    }
    return sum;
}

double sixj(int a, int b, int c, int d, int e, int f)
{
    if (!tri_ok(a, b, c) || !tri_ok(a, e, f) || !tri_ok(d, b, f) || !tri_ok(d, e, c)) return 0.0;
    const double lnpref = 0.5 * (ln_delta(a, b, c) + ln_delta(a, e, f) + ln_delta(d, b, f) + ln_delta(d, e, c));
    const int t1 = (a + b + c) / 2, t2 = (a + e + f) / 2, t3 = (d + b + f) / 2, t4 = (d + e + c) / 2;
    const int u1 = (a + b + d + e) / 2, u2 = (b + c + e + f) / 2, u3 = (c + a + f + d) / 2;
    const int kmin = std::max(std::max(t1, t2), std::max(t3, t4)), kmax = std::min(u1, std::min(u2, u3));
    double sum = 0.0;
    for (int k = kmin; k <= kmax; ++k) {
        double ln = lnpref + lf()(k + 1) - (lf()(k - t1) + lf()(k - t2) + lf()(k - t3) + lf()(k - t4)
                                            + lf()(u1 - k) + lf()(u2 - k) + lf()(u3 - k));
        sum += (k & 1) ? -std::exp(ln) : std::exp(ln);
    }
    return sum;
}

// { a b c ; d e f ; g h i } = sum_k (-1)^{2k} (2k+1) {a d g; h i k}{b e h; d k f}{c f i; k a b}
double ninej(int a, int b, int c, int d, int e, int f, int g, int h, int i)
{
    if (!tri_ok(a, b, c) || !tri_ok(d, e, f) || !tri_ok(g, h, i) || !tri_ok(a, d, g) || !tri_ok(b, e, h) || !tri_ok(c, f, i))
        return 0.0;
    const int kmin = std::max(std::abs(a - i), std::max(std::abs(d - h), std::abs(b - f)));
    const int kmax = std::min(a + i, std::min(d + h, b + f));
    double sum = 0.0;
    for (int k = kmin; k <= kmax; k += 2) {
        double t = (k + 1) * sixj(a, d, g, h, i, k) * sixj(b, e, h, d, k, f) * sixj(c, f, i, k, a, b);
        sum += (k & 1) ? -t : t;
    }
    return sum;
}

std::string validate_channels(const pm_channel* ch, int n_ch, int J2, int parity, int T2, int stat)
{
    if (stat != PM_FERMION_ISOSPIN && stat != PM_SPINLESS_BOSON) return "unknown statistics";
    if (parity != 1 && parity != -1) return "parity must be +1 or -1";
    if (J2 < 0 || T2 < 0) return "negative J2 or T2";
    for (int a = 0; a < n_ch; ++a) {
        const pm_channel& c = ch[a];
        if (c.l < 0 || c.lam < 0 || c.s < 0 || c.j < 0 || c.t < 0 || c.I2 < 0) return "negative quantum number";
        if (c.l > PM_MAX_L || c.lam > PM_MAX_L) return "orbital momentum above PM_MAX_L";
        if (((c.l + c.lam) & 1) != (parity == 1 ? 0 : 1)) return "channel parity differs from the lattice parity";
        if (stat == PM_SPINLESS_BOSON) {
            if (c.s != 0 || c.t != 0 || c.j != c.l || c.I2 != 2 * c.lam) return "spinless channel must have s=t=0, j=l, I2=2*lam";
            if (c.l & 1) return "identical bosons need even pair l";
            if (J2 & 1) return "boson J2 must be even";
            if (!tri_ok(2 * c.l, 2 * c.lam, J2)) return "triangle (l, lam, J) violated";
            if (T2 != 0) return "T2 must be 0 for spinless bosons";
        } else {
            if (c.s > 1 || c.t > 1) return "pair spin/isospin must be 0 or 1";
            if (((c.l + c.s + c.t) & 1) == 0) return "Pauli principle: (-1)^(l+s+t) must be -1";
            if (!tri_ok(2 * c.l, 2 * c.s, 2 * c.j)) return "triangle (l, s, j) violated";
            if (!tri_ok(2 * c.lam, 1, c.I2)) return "triangle (lam, 1/2, I) violated";
            if (!tri_ok(2 * c.j, c.I2, J2)) return "triangle (j, I, J) violated";
            if (!tri_ok(2 * c.t, 1, T2)) return "triangle (t, 1/2, T) violated";
        }
        for (int b = 0; b < a; ++b)
            if (ch[b].l == c.l && ch[b].s == c.s && ch[b].j == c.j && ch[b].t == c.t && ch[b].lam == c.lam && ch[b].I2 == c.I2)
                return "duplicate channel";
    }
    return "";
}

void gauss_legendre(int n, std::vector<double>& t, std::vector<double>& w)
{
    t.assign((size_t)n, 0.0); w.assign((size_t)n, 0.0);
    for (int k = 0; k < (n + 1) / 2; ++k) {
        long double z = std::cos(kPi * (k + 0.75) / (n + 0.5)), dp = 1.0L;
        for (int it = 0; it < 100; ++it) {
            long double p0 = 1.0L, p1 = z;
            for (int l = 2; l <= n; ++l) { long double p2 = ((2 * l - 1) * z * p1 - (l - 1) * p0) / l; p0 = p1; p1 = p2; }
            if (n == 1) { p0 = 1.0L; p1 = z; }
            dp = n * (z * p1 - p0) / (z * z - 1.0L);
            long double dz = p1 / dp;
            z -= dz;
            if (std::fabs((double)dz) < 1e-19) break;
        }
        {   // derivative at the converged root
            long double p0 = 1.0L, p1 = z;
            for (int l = 2; l <= n; ++l) { long double p2 = ((2 * l - 1) * z * p1 - (l - 1) * p0) / l; p0 = p1; p1 = p2; }
            dp = n * (z * p1 - p0) / (z * z - 1.0L);
        }
        long double wt = 2.0L / ((1.0L - z * z) * dp * dp);
        t[(size_t)(n - 1 - k)] = (double)z;  t[(size_t)k] = -(double)z;
        w[(size_t)(n - 1 - k)] = (double)wt; w[(size_t)k] = (double)wt;
    }
    if (n & 1) t[(size_t)(n / 2)] = 0.0;
}

namespace {

// LS(alpha) membership — integer logic only (reading R8)
bool has_LS(const pm_channel& c, int L, int S2, int J2, int stat)
{
    if (!tri_ok(2 * c.l, 2 * c.lam, 2 * L)) return false;
    if (stat == PM_SPINLESS_BOSON) return 2 * L == J2 && S2 == 0;
    if (S2 < std::abs(2 * c.s - 1) || S2 > 2 * c.s + 1 || !(S2 & 1)) return false;
    return tri_ok(2 * L, S2, J2);
}

// jI -> LS recoupling  C^{LS}_alpha
double recouple(const pm_channel& c, int L, int S2, int J2)
{
    return std::sqrt((double)((2 * c.j + 1) * (c.I2 + 1) * (2 * L + 1) * (S2 + 1)))
         * ninej(2 * c.l, 2 * c.s, 2 * c.j, 2 * c.lam, 1, c.I2, 2 * L, S2, J2);
}

// <((23)s,1)S | ((31)s',2)S> for three spin-1/2 particles
double spin_overlap(int s, int sp, int S2)
{
    double v = std::sqrt((double)((2 * s + 1) * (2 * sp + 1))) * sixj(1, 1, 2 * s, 1, S2, 2 * sp);
    return (sp & 1) ? -v : v;
}

}  // namespace

std::string build_tables(const pm_channel* ch, int n_ch, int J2, int T2, int stat, Tables& T)
{
    T = Tables();
    T.n_ch = n_ch;
    const int Lcap = (stat == PM_SPINLESS_BOSON) ? J2 / 2 : (J2 + 3) / 2;
    for (int a = 0; a < n_ch; ++a) T.lmax = std::max(T.lmax, std::max(ch[a].l, ch[a].lam));

    // coupled mask and coupled lists
    T.coupled.assign((size_t)n_ch * n_ch, 0);
    T.cl_off.assign((size_t)n_ch + 1, 0);
    for (int a = 0; a < n_ch; ++a) {
        for (int b = 0; b < n_ch; ++b) {
            bool c = false;
            for (int L = 0; L <= Lcap && !c; ++L)
                for (int S2 = 0; S2 <= 3 && !c; ++S2)
                    c = has_LS(ch[a], L, S2, J2, stat) && has_LS(ch[b], L, S2, J2, stat);
            T.coupled[(size_t)a * n_ch + b] = c;
            if (c) T.cl.push_back(b);
        }
        T.cl_off[(size_t)a + 1] = (int32_t)T.cl.size();
    }
    T.totcoup = (int)T.cl.size();

    // coefficients c^L (both cyclic terms: factor 2, reading R4), functions, triples
    std::map<std::tuple<int, int, int>, int> tri_id;
    std::map<std::tuple<int, int>, int> fun_id;
    auto get_tri = [&](int l, int lam, int L) {
        auto key = std::make_tuple(l, lam, L);
        auto it = tri_id.find(key);
        if (it != tri_id.end()) return it->second;
        Triple t{l, lam, L, (l + lam + L) & 1, 0, T.n_slot};
        t.nM = L - t.M0 + 1;
        T.n_slot += t.nM;
        T.tri.push_back(t);
        return tri_id[key] = (int)T.tri.size() - 1;
    };
    T.ot_off.assign(1, 0);
    for (int a = 0; a < n_ch; ++a)
        for (int idx = T.cl_off[(size_t)a]; idx < T.cl_off[(size_t)a + 1]; ++idx) {
            const int b = T.cl[(size_t)idx];
            for (int L = 0; L <= Lcap; ++L) {
                double c = 0.0;
                if (stat == PM_SPINLESS_BOSON) {
                    if (2 * L == J2 && tri_ok(2 * ch[a].l, 2 * ch[a].lam, 2 * L) && tri_ok(2 * ch[b].l, 2 * ch[b].lam, 2 * L)) c = 1.0;
                } else {
                    for (int S2 = 1; S2 <= 3; S2 += 2) {
                        if (!has_LS(ch[a], L, S2, J2, stat) || !has_LS(ch[b], L, S2, J2, stat)) continue;
                        c += recouple(ch[a], L, S2, J2) * recouple(ch[b], L, S2, J2)
                           * spin_overlap(ch[a].s, ch[b].s, S2) * spin_overlap(ch[a].t, ch[b].t, T2);
                    }
                }
                if (std::fabs(c) < 1e-15) continue;
                const int ta = get_tri(ch[a].l, ch[a].lam, L), tb = get_tri(ch[b].l, ch[b].lam, L);
                auto key = std::make_tuple(ta, tb);
                auto it = fun_id.find(key);
                int f;
                if (it == fun_id.end()) {
                    f = (int)T.fun.size();
                    T.fun.push_back(OrbFun{ta, tb, L, T.tri[(size_t)ta].slot0, T.tri[(size_t)tb].slot0, T.tri[(size_t)ta].nM});
                    fun_id[key] = f;
                } else f = it->second;
                T.ot_f.push_back(f);
                T.ot_c.push_back(16.0 * kPi * kPi * c);
            }
            T.ot_off.push_back((int32_t)T.ot_f.size());
        }

    // Triples renumbered by (L, l, lambda), so that the slots of all triples with one L are contiguous and evenly strided:
    // with the function order below, neighbouring lanes of the stage read evenly strided ket slots.
    {
        const int nt = (int)T.tri.size();
        std::vector<int> ord((size_t)nt), inv((size_t)nt);
        for (int t = 0; t < nt; ++t) ord[(size_t)t] = t;
        std::stable_sort(ord.begin(), ord.end(), [&](int x, int y) {
            const Triple &A = T.tri[(size_t)x], &B = T.tri[(size_t)y];
            return std::make_tuple(A.L, A.l, A.lam) < std::make_tuple(B.L, B.l, B.lam);
        });
        std::vector<Triple> sorted((size_t)nt);
        int slot = 0;
        for (int i = 0; i < nt; ++i) {
            sorted[(size_t)i] = T.tri[(size_t)ord[(size_t)i]];
            sorted[(size_t)i].slot0 = slot;
            slot += sorted[(size_t)i].nM;
            inv[(size_t)ord[(size_t)i]] = i;
        }
        T.tri.swap(sorted);
        for (OrbFun& f : T.fun) {
            f.ta = inv[(size_t)f.ta]; f.tb = inv[(size_t)f.tb];
            f.sa0 = T.tri[(size_t)f.ta].slot0; f.sb0 = T.tri[(size_t)f.tb].slot0;
        }
    }
    // Functions ordered by (number of M-terms, L, bra triple, ket triple): the fill kernel's stage handles 32 functions at
    // a time with as many terms as the largest of them has, neighbouring lanes then read the same bra slots and evenly
    // strided ket slots (few shared-memory bank conflicts), and the outputs of one row read neighbouring sums.
    {
        const int nf = (int)T.fun.size();
        std::vector<int> ord((size_t)nf), inv((size_t)nf);
        for (int f = 0; f < nf; ++f) ord[(size_t)f] = f;
        std::stable_sort(ord.begin(), ord.end(), [&](int x, int y) {
            const OrbFun &A = T.fun[(size_t)x], &B = T.fun[(size_t)y];
            return std::make_tuple(A.nM, A.L, A.ta, A.tb) < std::make_tuple(B.nM, B.L, B.ta, B.tb);
        });
        std::vector<OrbFun> sorted((size_t)nf);
        for (int i = 0; i < nf; ++i) { sorted[(size_t)i] = T.fun[(size_t)ord[(size_t)i]]; inv[(size_t)ord[(size_t)i]] = i; }
        T.fun.swap(sorted);
        for (int32_t& f : T.ot_f) f = inv[(size_t)f];
    }

    // per-slot bra weights and ket term lists
    T.slot_w.assign((size_t)T.n_slot, 0.0); T.slot_l.assign((size_t)T.n_slot, 0); T.slot_M.assign((size_t)T.n_slot, 0);
    T.kt_off.assign(1, 0);
    for (const Triple& t : T.tri)
        for (int i = 0; i < t.nM; ++i) {
            const int M = t.M0 + i, s = t.slot0 + i;
            T.slot_l[(size_t)s] = t.l; T.slot_M[(size_t)s] = M;
            if (M <= t.l)
                T.slot_w[(size_t)s] = (M == 0 ? 1.0 : 2.0) / (2 * t.L + 1)
                    * clebsch(2 * t.l, 2 * M, 2 * t.lam, 0, 2 * t.L, 2 * M) * std::sqrt((2 * t.lam + 1) / (4.0 * kPi));
            std::map<std::pair<int, int>, double> terms;           // (|m|, |mu|) -> coefficient with signs folded in
            for (int m = -t.l; m <= t.l; ++m) {
                const int mu = M - m;
                if (std::abs(mu) > t.lam) continue;
                double c = clebsch(2 * t.l, 2 * m, 2 * t.lam, 2 * mu, 2 * t.L, 2 * M);
                if (m < 0 && (m & 1)) c = -c;
                if (mu < 0 && (mu & 1)) c = -c;
                terms[{std::abs(m), std::abs(mu)}] += c;
            }
            for (auto& kv : terms) {
                if (std::fabs(kv.second) < 1e-15) continue;
                T.kt_ip.push_back(ylm_index(t.l, kv.first.first));
                T.kt_iq.push_back(ylm_index(t.lam, kv.first.second));
                T.kt_c.push_back(kv.second);
            }
            T.kt_off.push_back((int32_t)T.kt_c.size());
        }

    // recurrence constants
    const int ny = ylm_index(T.lmax, T.lmax) + 1;
    T.ya.assign((size_t)ny, 0.0); T.yb.assign((size_t)ny, 0.0); T.ydiag.assign((size_t)T.lmax + 1, 0.0);
    for (int m = 1; m <= T.lmax; ++m) T.ydiag[(size_t)m] = -std::sqrt((2.0 * m + 1.0) / (2.0 * m));
    for (int l = 1; l <= T.lmax; ++l)
        for (int m = 0; m < l; ++m) {
            T.ya[(size_t)ylm_index(l, m)] = std::sqrt((4.0 * l * l - 1.0) / ((double)l * l - (double)m * m));
            T.yb[(size_t)ylm_index(l, m)] = (l - 1 > m) ? std::sqrt((((double)l - 1) * (l - 1) - (double)m * m) / (4.0 * (l - 1) * (l - 1) - 1.0)) : 0.0;
        }
    if (T.fun.empty()) return "no coupled channel pair has a non-vanishing coefficient";
    return "";
}

void build_groups(const Tables& T, const pm_channel* ch, int max_slot, int max_fun, int max_out, std::vector<GroupTables>& groups)
{
    groups.clear();
    const int n_tri = (int)T.tri.size(), n_fun = (int)T.fun.size();
    // classes of ket triples by (l', lam'), in order of first appearance
    std::map<std::pair<int, int>, int> cls_id;
    std::vector<int> tri_cls((size_t)n_tri), cls_slots, cls_funs;
    for (int t = 0; t < n_tri; ++t) {
        auto key = std::make_pair(T.tri[(size_t)t].l, T.tri[(size_t)t].lam);
        auto it = cls_id.find(key);
        if (it == cls_id.end()) { it = cls_id.emplace(key, (int)cls_slots.size()).first; cls_slots.push_back(0); cls_funs.push_back(0); }
        tri_cls[(size_t)t] = it->second;
        cls_slots[(size_t)it->second] += T.tri[(size_t)t].nM;
    }
    for (const OrbFun& f : T.fun) cls_funs[(size_t)tri_cls[(size_t)f.tb]]++;
    const int n_cls = (int)cls_slots.size();
    std::vector<int> cls_outs((size_t)n_cls, 0);       // outputs (alpha, alpha') whose column channel has the class's orbital pair
    for (int o = 0; o < T.totcoup; ++o) {
        const auto it = cls_id.find(std::make_pair(ch[T.cl[(size_t)o]].l, ch[T.cl[(size_t)o]].lam));
        if (it != cls_id.end()) cls_outs[(size_t)it->second]++;
    }
    std::vector<int> cls_grp((size_t)n_cls, 0);
    int n_grp = 1;
    if (T.n_slot > max_slot || n_fun > max_fun || T.totcoup > max_out) {
        int gs = 0, gf = 0, go = 0;
        n_grp = 0;
        for (int c = 0; c < n_cls; ++c) {
            if (n_grp == 0 || gs + cls_slots[(size_t)c] > max_slot || gf + cls_funs[(size_t)c] > max_fun || go + cls_outs[(size_t)c] > max_out) {
                ++n_grp; gs = 0; gf = 0; go = 0;
            }
            cls_grp[(size_t)c] = n_grp - 1;
            gs += cls_slots[(size_t)c]; gf += cls_funs[(size_t)c]; go += cls_outs[(size_t)c];
        }
    }
    groups.resize((size_t)n_grp);
    std::vector<int> slot_local((size_t)T.n_slot, -1), fun_local((size_t)n_fun, -1);
    for (int g = 0; g < n_grp; ++g) groups[(size_t)g].kt_off.assign(1, 0);
    for (int t = 0; t < n_tri; ++t) {                  // local ket slots in triple order (one group: the global numbering)
        GroupTables& G = groups[(size_t)cls_grp[(size_t)tri_cls[(size_t)t]]];
        const Triple& tr = T.tri[(size_t)t];
        for (int i = 0; i < tr.nM; ++i) {
            const int s = tr.slot0 + i;
            slot_local[(size_t)s] = G.n_slot++;
            for (int k = T.kt_off[(size_t)s]; k < T.kt_off[(size_t)s + 1]; ++k) {
                G.kt_ip.push_back(T.kt_ip[(size_t)k]); G.kt_iq.push_back(T.kt_iq[(size_t)k]); G.kt_c.push_back(T.kt_c[(size_t)k]);
            }
            G.kt_off.push_back((int32_t)G.kt_c.size());
        }
    }
    for (int f = 0; f < n_fun; ++f) {
        const OrbFun& F = T.fun[(size_t)f];
        GroupTables& G = groups[(size_t)cls_grp[(size_t)tri_cls[(size_t)F.tb]]];
        fun_local[(size_t)f] = (int)G.fun.size();
        OrbFun L = F;
        L.sb0 = slot_local[(size_t)F.sb0];
        G.fun.push_back(L);
        G.f_global.push_back(f);
    }
    for (int g = 0; g < n_grp; ++g) groups[(size_t)g].ot_off.assign(1, 0);
    for (int a = 0; a < T.n_ch; ++a)
        for (int o = T.cl_off[(size_t)a]; o < T.cl_off[(size_t)a + 1]; ++o) {
            const int b = T.cl[(size_t)o];
            const auto it = cls_id.find(std::make_pair(ch[b].l, ch[b].lam));
            // a column channel whose orbital pair carries no triple at all has only structural zeros: any group may write them
            GroupTables& G = groups[(size_t)(it == cls_id.end() ? 0 : cls_grp[(size_t)it->second])];
            G.o_alpha.push_back(a); G.o_m.push_back(o - T.cl_off[(size_t)a]); G.o_ap.push_back(b);
            for (int k = T.ot_off[(size_t)o]; k < T.ot_off[(size_t)o + 1]; ++k) {
                G.ot_f.push_back(fun_local[(size_t)T.ot_f[(size_t)k]]); G.ot_c.push_back(T.ot_c[(size_t)k]);
            }
            G.ot_off.push_back((int32_t)G.ot_f.size());
        }
    // Whole rows (all outputs of one alpha, which the fill stores as one contiguous run per target) ordered by the largest
    // number of terms any of their outputs has (stable), so that the fill kernel's 32-output steps over the one-term
    // (two-term) rows load no padded terms while every store still covers consecutive entries of a row.
    for (GroupTables& G : groups) {
        const int n = (int)G.o_alpha.size();
        std::vector<int> ord((size_t)n);
        for (int o = 0; o < n; ++o) ord[(size_t)o] = o;
        auto nt = [&](int o) { return G.ot_off[(size_t)o + 1] - G.ot_off[(size_t)o]; };
        std::map<int, int> row_nt;                                     // alpha -> most terms of its outputs in this group
        for (int o = 0; o < n; ++o) row_nt[G.o_alpha[(size_t)o]] = std::max(row_nt[G.o_alpha[(size_t)o]], nt(o));
        std::stable_sort(ord.begin(), ord.end(), [&](int x, int y) { return row_nt[G.o_alpha[(size_t)x]] < row_nt[G.o_alpha[(size_t)y]]; });
        GroupTables R = G;
        R.ot_off.assign(1, 0); R.ot_f.clear(); R.ot_c.clear();
        G.n_out1 = G.n_out2 = G.n_out3 = 0;
        int max_nt = 0;
        for (int i = 0; i < n; ++i) {
            const int o = ord[(size_t)i];
            R.o_alpha[(size_t)i] = G.o_alpha[(size_t)o]; R.o_m[(size_t)i] = G.o_m[(size_t)o]; R.o_ap[(size_t)i] = G.o_ap[(size_t)o];
            for (int k = G.ot_off[(size_t)o]; k < G.ot_off[(size_t)o + 1]; ++k) { R.ot_f.push_back(G.ot_f[(size_t)k]); R.ot_c.push_back(G.ot_c[(size_t)k]); }
            R.ot_off.push_back((int32_t)R.ot_f.size());
            if (row_nt[G.o_alpha[(size_t)o]] <= 1) ++G.n_out1;
            if (row_nt[G.o_alpha[(size_t)o]] <= 2) ++G.n_out2;
            if (row_nt[G.o_alpha[(size_t)o]] <= 3) ++G.n_out3;
            max_nt = std::max(max_nt, nt(o));
        }
        R.n_out1 = G.n_out1; R.n_out2 = G.n_out2; R.n_out3 = G.n_out3;
        R.n_oterm = max_nt > 3 ? 4 : 3;
        R.oterm_tail = max_nt > 4;
        G = R;
        uint64_t h = 1469598103934665603ull;
        auto mix = [&](const void* p, size_t n) {
            const unsigned char* b = (const unsigned char*)p;
            for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ull; }
        };
        auto mixi = [&](int64_t v) { mix(&v, sizeof v); };
        mixi(G.n_slot); mixi((int64_t)G.fun.size()); mixi(G.n_oterm); mixi(G.oterm_tail ? 1 : 0);
        for (const OrbFun& f : G.fun) { mixi(f.sb0); mixi(f.nM); mixi(f.L); }
        mix(G.kt_off.data(), 4 * G.kt_off.size()); mix(G.kt_ip.data(), 4 * G.kt_ip.size());
        mix(G.kt_iq.data(), 4 * G.kt_iq.size()); mix(G.kt_c.data(), 8 * G.kt_c.size());
        G.hash = h;
    }
}

void build_bra(const Tables& T, const std::vector<double>& tx, std::vector<double>& bra)
{
    const int ny = ylm_index(T.lmax, T.lmax) + 1;
    std::vector<double> Y((size_t)ny);
    bra.assign(tx.size() * (size_t)T.n_slot, 0.0);
    for (size_t c = 0; c < tx.size(); ++c) {
        const double x = tx[c], sx = std::sqrt((1.0 - x) * (1.0 + x));
        ylm_fill(T.lmax, sx, x, T.ya.data(), T.yb.data(), T.ydiag.data(), Y.data());
        for (int s = 0; s < T.n_slot; ++s)
            if (T.slot_w[(size_t)s] != 0.0)
                bra[c * (size_t)T.n_slot + (size_t)s] = T.slot_w[(size_t)s] * Y[(size_t)ylm_index(T.slot_l[(size_t)s], T.slot_M[(size_t)s])];
    }
}

uint64_t tables_hash(const Tables& T)
{
    uint64_t h = 1469598103934665603ull;
    auto mix = [&](const void* p, size_t n) {
        const unsigned char* b = (const unsigned char*)p;
        for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ull; }
    };
    auto mixi = [&](int64_t v) { mix(&v, sizeof v); };
    mixi(T.lmax); mixi(T.n_slot); mixi((int64_t)T.tri.size()); mixi((int64_t)T.fun.size());
    for (const Triple& t : T.tri) { mixi(t.l); mixi(t.lam); mixi(t.L); mixi(t.M0); mixi(t.nM); mixi(t.slot0); }
    for (const OrbFun& f : T.fun) { mixi(f.sa0); mixi(f.sb0); mixi(f.nM); mixi(f.L); }
    mix(T.kt_off.data(), 4 * T.kt_off.size()); mix(T.kt_ip.data(), 4 * T.kt_ip.size());
    mix(T.kt_iq.data(), 4 * T.kt_iq.size()); mix(T.kt_c.data(), 8 * T.kt_c.size());
    return h;
}

KetView ket_view(const Tables& T)
{
    KetView v;
    v.n_slot = T.n_slot; v.n_bra = T.n_slot; v.kt_off = &T.kt_off; v.kt_ip = &T.kt_ip; v.kt_iq = &T.kt_iq; v.kt_c = &T.kt_c; v.fun = &T.fun;
    v.hash = tables_hash(T); v.bra_smem = true;
    for (size_t o = 0; o + 1 < T.ot_off.size(); ++o) {
        if (T.ot_off[o + 1] - T.ot_off[o] > 3) v.n_oterm = 4;
        if (T.ot_off[o + 1] - T.ot_off[o] > 4) v.oterm_tail = true;
    }
    return v;
}

KetView ket_view(const GroupTables& G, int n_bra, bool bra_smem)
{
    KetView v;
    v.n_bra = n_bra;
    v.n_slot = G.n_slot; v.kt_off = &G.kt_off; v.kt_ip = &G.kt_ip; v.kt_iq = &G.kt_iq; v.kt_c = &G.kt_c; v.fun = &G.fun;
    v.hash = G.hash; v.bra_smem = bra_smem; v.n_oterm = G.n_oterm; v.oterm_tail = G.oterm_tail;
    return v;
}

void scaled_harmonics(int lmax, std::vector<double>& ynorm, std::vector<double>& ybeta)
{
    const int ny = ylm_index(lmax, lmax) + 1;
    std::vector<long double> N((size_t)ny, 0.0L);
    ynorm.assign((size_t)ny, 0.0); ybeta.assign((size_t)ny, 0.0);
    auto ya = [](int l, int m) { return sqrtl((4.0L * l * l - 1.0L) / ((long double)l * l - (long double)m * m)); };
    auto yb = [](int l, int m) { return sqrtl((((long double)l - 1) * (l - 1) - (long double)m * m) / (4.0L * (l - 1) * (l - 1) - 1.0L)); };
    N[0] = 0.5L / sqrtl(3.14159265358979323846264338327950288L);
    for (int m = 0; m <= lmax; ++m) {
        if (m > 0) N[(size_t)ylm_index(m, m)] = -sqrtl((2.0L * m + 1.0L) / (2.0L * m)) * N[(size_t)ylm_index(m - 1, m - 1)];
        for (int l = m + 1; l <= lmax; ++l) {
            N[(size_t)ylm_index(l, m)] = ya(l, m) * N[(size_t)ylm_index(l - 1, m)];
            if (l - 2 >= m) ybeta[(size_t)ylm_index(l, m)] = (double)(yb(l, m) / ya(l - 1, m));
        }
    }
    for (int k = 0; k < ny; ++k) ynorm[(size_t)k] = (double)N[(size_t)k];
}

double ket_flops(const Tables& T)
{
    int la = 0, lb = 0;
    for (const Triple& t : T.tri) { la = std::max(la, t.l); lb = std::max(lb, t.lam); }
    auto rec = [](int lmax, bool unit_seed) {       // Q_mm: 1 mul; Q_{m+1,m}: 1 mul; Q_lm (l >= m+2): mul + FMA = 3
        double f = 0.0;
        for (int m = 0; m <= lmax; ++m) {
            if (m > 0) f += 1.0;
            for (int l = m + 1; l <= lmax; ++l) f += (l == m + 1) ? 1.0 : 3.0;
        }
        if (unit_seed && lmax >= 1) f -= 2.0;       // ux*1 and uz*1 are not operations
        return f;
    };
    std::map<std::pair<int, int>, int> prod;
    for (size_t t = 0; t < T.kt_c.size(); ++t) prod[{T.kt_ip[t], T.kt_iq[t]}]++;
    double f = rec(la, false) + rec(lb, true) + (double)prod.size();
    for (int s = 0; s < T.n_slot; ++s) {
        const int n = T.kt_off[(size_t)s + 1] - T.kt_off[(size_t)s];
        if (n > 0) f += 1.0 + 2.0 * (n - 1);
    }
    return f;
}

double sqrt_threshold(double e)
{
    if (!(e > 0.0)) return 0.0;                         // every y >= 0 has sqrt(y) >= 0
    double y = e * e;
    while (std::sqrt(y) >= e && y > 0.0) y = std::nextafter(y, 0.0);
    while (std::sqrt(y) < e) y = std::nextafter(y, std::numeric_limits<double>::infinity());
    return y;
}

void bucket_table(const std::vector<double>& thr, int n, int n_buckets, int& hmin, int& sh, std::vector<uint16_t>& start)
{
    auto hi32 = [](double x) { int64_t b; std::memcpy(&b, &x, 8); return (int)(b >> 32); };
    int first = 0;
    while (first < n - 1 && !(thr[(size_t)first] > 0.0)) ++first;      // smallest positive threshold (zero has its own bucket 0)
    hmin = hi32(thr[(size_t)first]);
    const int64_t span = (int64_t)hi32(thr[(size_t)n - 1]) - hmin;
    sh = 0;
    while ((span >> sh) >= n_buckets - 1) ++sh;
    auto bucket = [&](double x) { int64_t b = ((int64_t)hi32(x) - hmin) >> sh; return (int)std::max<int64_t>(0, std::min<int64_t>(n_buckets - 1, b)); };
    start.assign((size_t)n_buckets, 0);
    for (int b = 0; b < n_buckets; ++b) {
        int c = 0;
        while (c < n && bucket(thr[(size_t)c]) < b) ++c;
        start[(size_t)b] = (uint16_t)c;
    }
}

}  // namespace pm
