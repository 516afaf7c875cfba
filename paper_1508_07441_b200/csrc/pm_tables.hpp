// pm_tables.hpp — host-side channel / coefficient precompute of libpm (hot-path step a1).
// PAPER.md:L256 "calculation of algebraic coefficients g ... for recoupling between different spin-angular
// channels" (step 1), L341 "algebraic coefficients g, values of Legendre polynomials at the nodal points".
// The formulas are derived in DESIGN.md sec. 3.2.  No code is shared with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/pm.h"

namespace pm {

// index of Y_{l m}, m >= 0, in the packed per-direction table
inline int ylm_index(int l, int m) { return l * (l + 1) / 2 + m; }

// One bipolar harmonic family (l, lam, L).  Only M >= 0 is stored: for coplanar arguments
// Y^{L,-M} = (-1)^{l+lam-L+M} Y^{L,M}; families with l+lam+L odd have no M = 0 member.
struct Triple { int l, lam, L, M0, nM, slot0; };

// One distinct orbital function A^L_{l lam, l' lam'}: sum over nM slots of bra[sa0+i]*ket[sb0+i].
struct OrbFun { int ta, tb, L, sa0, sb0, nM; };

struct Tables {
    int n_ch = 0, lmax = 0, n_slot = 0, totcoup = 0;
    std::vector<uint8_t> coupled;          // [n_ch*n_ch]
    std::vector<int32_t> cl_off, cl;       // coupled lists: cl[cl_off[a] .. cl_off[a+1]) = alpha' ascending
    std::vector<Triple> tri;
    std::vector<OrbFun> fun;
    // ket side: slot s = sum over terms t in [kt_off[s], kt_off[s+1]) of kt_c[t]*Yp[kt_ip[t]]*Yq[kt_iq[t]]
    std::vector<int32_t> kt_off, kt_ip, kt_iq;
    std::vector<double> kt_c;
    // per output o = cl_off[a] + m: P = norm * sum_{t in [ot_off[o], ot_off[o+1])} ot_c[t]*acc[ot_f[t]]
    std::vector<int32_t> ot_off, ot_f;
    std::vector<double> ot_c;
    // bra weights per slot: wM/(2L+1) * <l M lam 0|L M> * sqrt((2 lam+1)/4pi); bra[c][s] = slot_w[s]*Y_{l M}(x_c)
    std::vector<double> slot_w;
    std::vector<int32_t> slot_l, slot_M;
    // normalised Legendre recurrence constants (see pm_ylm.h)
    std::vector<double> ya, yb, ydiag;
};

// A column-channel group: the channels alpha' whose orbital pair (l', lam') falls into one set of classes.  Every ket
// triple (l', lam', L), every orbital function and every output (alpha, alpha') belongs to exactly one group, so a group
// is a complete sub-problem of the fill: it writes its own columns of every row.  Channel sets whose ket tables exceed
// what one kernel holds (62 channels, J up to 17/2: 422 slots, 546 functions) are filled group by group.
struct GroupTables {
    int n_slot = 0;                                   // ket slots of the group, numbered locally
    std::vector<int32_t> kt_off, kt_ip, kt_iq;        // ket terms per local slot
    std::vector<double> kt_c;
    std::vector<OrbFun> fun;                          // sa0: GLOBAL bra slot, sb0: LOCAL ket slot
    std::vector<int32_t> f_global;                    // index in Tables::fun of each local function
    std::vector<int32_t> o_alpha, o_m, o_ap;          // outputs: row channel, position in the row's coupled list, column channel;
                                                      // rows ordered by the most terms of their outputs
    int n_out1 = 0, n_out2 = 0, n_out3 = 0;           // outputs in rows with at most one / two / three terms per output
    int n_oterm = 3;                                  // terms per output a specialised kernel keeps in shared memory: 3, or 4 when an output has more than 3
    bool oterm_tail = false;                          // some output has more terms than that (never for three spin-1/2 particles: at most four L per pair)
    std::vector<int32_t> ot_off, ot_f;                // terms per output, f numbered locally
    std::vector<double> ot_c;
    uint64_t hash = 0;                                // FNV-1a of what the group's ket code depends on (keys run-time compiled kernels)
};

// What the generated ket code of one kernel depends on: a whole channel set (Tables) or one column-channel group.
struct KetView {
    int n_slot = 0;
    int n_bra = 0;                                    // bra slots of the whole channel set (the functions' sa0 index them)
    const std::vector<int32_t> *kt_off = nullptr, *kt_ip = nullptr, *kt_iq = nullptr;
    const std::vector<double>* kt_c = nullptr;
    const std::vector<OrbFun>* fun = nullptr;
    uint64_t hash = 0;
    int n_oterm = 3;                                  // (GroupTables::n_oterm, oterm_tail)
    bool oterm_tail = false;
    bool bra_smem = true;                             // the kernel reads the bra harmonics from shared memory (else from global memory)
};
KetView ket_view(const Tables& T);
KetView ket_view(const GroupTables& G, int n_bra, bool bra_smem);

// One group holding everything when the set fits (max_slot, max_fun, max_out outputs), else a greedy packing of the
// (l', lam') classes under the three limits.
void build_groups(const Tables& T, const pm_channel* ch, int max_slot, int max_fun, int max_out, std::vector<GroupTables>& groups);

// Algebra (doubled arguments), exposed for host tests through the C ABI indirectly (pm_lattice_coupling).
double clebsch(int j1, int m1, int j2, int m2, int j3, int m3);
double sixj(int a, int b, int c, int d, int e, int f);
double ninej(int a, int b, int c, int d, int e, int f, int g, int h, int i);

// Validates the channel list against (J2, parity, T2, statistics); returns "" or a message.
std::string validate_channels(const pm_channel* ch, int n_ch, int J2, int parity, int T2, int stat);

// Builds every channel-dependent table.  Returns "" or a message.
std::string build_tables(const pm_channel* ch, int n_ch, int J2, int T2, int stat, Tables& T);

// Gauss-Legendre rule on [-1,1] by Newton iteration, ascending, exactly symmetric.
void gauss_legendre(int n, std::vector<double>& t, std::vector<double>& w);

// bra[c*n_slot + s] for the x-rule nodes
void build_bra(const Tables& T, const std::vector<double>& tx, std::vector<double>& bra);

// FNV-1a hash of everything the ket-side code of a fill kernel depends on (slot layout, ket term lists with
// the coefficient bit patterns, function list).  A kernel specialised at build time by pm_codegen carries the
// hash of the tables it was generated from; pm_fill uses it only when the lattice's tables hash equal.
uint64_t tables_hash(const Tables& T);

// Scaled harmonics used by generated code: Y_lm = ynorm[lm] * Q_lm with the constant-free recurrence
//   Q_00 = 1, Q_mm = ux*Q_{m-1,m-1}, Q_{m+1,m} = uz*Q_mm, Q_lm = uz*Q_{l-1,m} - ybeta[lm]*Q_{l-2,m}.
void scaled_harmonics(int lmax, std::vector<double>& ynorm, std::vector<double>& ybeta);

// FP64 flops (add = mul = 1, FMA = 2) of the ket code pm_codegen emits for these tables: the two scaled-harmonic
// recurrences, one product per distinct (Y_l'm, Y_lam'mu) pair, one multiply or FMA per ket term.
double ket_flops(const Tables& T);

// Smallest double y with sqrt(y) >= e (IEEE, correctly rounded): "e <= sqrt(y)" <=> "y >= sqrt_threshold(e)",
// so a node is located from p'^2 with the very decisions the oracle takes on p' = sqrt(p'^2) (reading R6).
double sqrt_threshold(double e);

// Bucket table over thresholds thr[0..n) (ascending, thr[0] >= 0) for the device-side locate (pm_device.cuh):
// bucket(v) = clamp((hi32(v) - hmin) >> sh, 0, n_buckets-1); start[b] = number of thresholds in buckets below b.
void bucket_table(const std::vector<double>& thr, int n, int n_buckets, int& hmin, int& sh, std::vector<uint16_t>& start);

}  // namespace pm
