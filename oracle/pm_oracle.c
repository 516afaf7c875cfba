/* pm_oracle.c — CPU ORACLE for the permutation-matrix build.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct implementation of what the hot path computes: the sparse
 * particle-permutation matrix P0 of the Faddeev equation in the three-body lattice (free
 * wave-packet) basis, PAPER.md:L206-215 (sec. 3.2, eq. 21-22), evaluated by the node-binning
 * quadrature of BASELINE.json `north_star` exactly as written out in DESIGN.md sec. 3
 * (= SURVEY.md sec. 8(c.1)).  It shares NO code with the CUDA path (paper_1508_07441_b200/csrc)
 * and neither includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it; the product never does.
 *
 * Parity status: the paper prints no value of any P0 element and no formula for g (eq. 22), so
 * parity WITH THE PAPER'S NUMBERS is "parity unpinned".  Every function below is pinned instead
 * by tests/test_oracle_*.py against things fixed by the mathematics:
 * library Wigner symbols (sympy), library spherical harmonics (scipy), the textbook triton
 * spin-isospin matrix, an explicit product-basis construction of the permutation kernel,
 * phase-space conservation, Monte-Carlo brute force, spectrum bounds, matrix symmetry.
 *
 * Value arithmetic is `real` (double, or long double with -DPO_LONG_DOUBLE); the node map and
 * the cell location are ALWAYS IEEE double in the exact operation order of DESIGN.md sec. 3.
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef PO_LONG_DOUBLE
typedef long double real;
#define RSQRT sqrtl
#else
typedef double real;
#define RSQRT sqrt
#endif

typedef struct { int32_t l, s, j, t, lam, I2; } po_channel;   /* I2 = 2*I */
enum { PO_FERMION_ISOSPIN = 0, PO_SPINLESS_BOSON = 1 };

#define PO_PI 3.14159265358979323846264338327950288L
#define PO_LMAX 12          /* largest orbital momentum handled by the Y tables */
#define PO_NFACT 80

/* ------------------------------------------------------------------------------------------
 * Angular-momentum algebra (standard Racah sums; arguments are DOUBLED integers: 2j, 2m).
 * Pinned against sympy.physics.wigner in tests/test_oracle_algebra.py.
 * ---------------------------------------------------------------------------------------- */
static long double po_fact(int n)
{
    static long double tab[PO_NFACT];
    static int ready = 0;
    if (!ready) {
        tab[0] = 1.0L;
        for (int i = 1; i < PO_NFACT; ++i) tab[i] = tab[i - 1] * (long double)i;
        ready = 1;
    }
    return (n < 0 || n >= PO_NFACT) ? 0.0L : tab[n];
}

static int po_triangle_ok(int a2, int b2, int c2)
{
    if ((a2 + b2 + c2) & 1) return 0;
    return (c2 >= abs(a2 - b2)) && (c2 <= a2 + b2);
}

/* triangle coefficient Delta(abc) = (a+b-c)!(a-b+c)!(-a+b+c)!/(a+b+c+1)! */
static long double po_delta(int a2, int b2, int c2)
{
    return po_fact((a2 + b2 - c2) / 2) * po_fact((a2 - b2 + c2) / 2) * po_fact((-a2 + b2 + c2) / 2)
         / po_fact((a2 + b2 + c2) / 2 + 1);
}

double po_wigner3j(int j1, int j2, int j3, int m1, int m2, int m3)
{
    if (m1 + m2 + m3 != 0) return 0.0;
    if (!po_triangle_ok(j1, j2, j3)) return 0.0;
    if (abs(m1) > j1 || abs(m2) > j2 || abs(m3) > j3) return 0.0;
    if (((j1 + m1) & 1) || ((j2 + m2) & 1) || ((j3 + m3) & 1)) return 0.0;
    long double pref = sqrtl(po_delta(j1, j2, j3)
        * po_fact((j1 + m1) / 2) * po_fact((j1 - m1) / 2)
        * po_fact((j2 + m2) / 2) * po_fact((j2 - m2) / 2)
        * po_fact((j3 + m3) / 2) * po_fact((j3 - m3) / 2));
    int kmin = 0;
    if ((j2 - j3 - m1) / 2 > kmin) kmin = (j2 - j3 - m1) / 2;
    if ((j1 - j3 + m2) / 2 > kmin) kmin = (j1 - j3 + m2) / 2;
    int kmax = (j1 + j2 - j3) / 2;
    if ((j1 - m1) / 2 < kmax) kmax = (j1 - m1) / 2;
    if ((j2 + m2) / 2 < kmax) kmax = (j2 + m2) / 2;
    long double sum = 0.0L;
    for (int k = kmin; k <= kmax; ++k) {
        long double den = po_fact(k) * po_fact((j1 + j2 - j3) / 2 - k) * po_fact((j1 - m1) / 2 - k)
            * po_fact((j2 + m2) / 2 - k) * po_fact((j3 - j2 + m1) / 2 + k) * po_fact((j3 - j1 - m2) / 2 + k);
        sum += ((k & 1) ? -1.0L : 1.0L) / den;
    }
    int ph = (j1 - j2 - m3) / 2;
    return (double)(((ph & 1) ? -1.0L : 1.0L) * pref * sum);
}

/* Clebsch-Gordan <j1 m1 j2 m2 | j3 m3> (Condon-Shortley) */
double po_cg(int j1, int m1, int j2, int m2, int j3, int m3)
{
    if (m1 + m2 != m3) return 0.0;
    int ph = (j1 - j2 + m3) / 2;
    double v = sqrt((double)(j3 + 1)) * po_wigner3j(j1, j2, j3, m1, m2, -m3);
    return (ph & 1) ? -v : v;
}

double po_wigner6j(int j1, int j2, int j3, int j4, int j5, int j6)
{
    if (!po_triangle_ok(j1, j2, j3) || !po_triangle_ok(j1, j5, j6) ||
        !po_triangle_ok(j4, j2, j6) || !po_triangle_ok(j4, j5, j3)) return 0.0;
    long double pref = sqrtl(po_delta(j1, j2, j3) * po_delta(j1, j5, j6) * po_delta(j4, j2, j6) * po_delta(j4, j5, j3));
    int a1 = (j1 + j2 + j3) / 2, a2 = (j1 + j5 + j6) / 2, a3 = (j4 + j2 + j6) / 2, a4 = (j4 + j5 + j3) / 2;
    int b1 = (j1 + j2 + j4 + j5) / 2, b2 = (j2 + j3 + j5 + j6) / 2, b3 = (j3 + j1 + j6 + j4) / 2;
    int kmin = a1; if (a2 > kmin) kmin = a2; if (a3 > kmin) kmin = a3; if (a4 > kmin) kmin = a4;
    int kmax = b1; if (b2 < kmax) kmax = b2; if (b3 < kmax) kmax = b3;
    long double sum = 0.0L;
    for (int k = kmin; k <= kmax; ++k) {
        long double den = po_fact(k - a1) * po_fact(k - a2) * po_fact(k - a3) * po_fact(k - a4)
            * po_fact(b1 - k) * po_fact(b2 - k) * po_fact(b3 - k);
        sum += ((k & 1) ? -1.0L : 1.0L) * po_fact(k + 1) / den;
    }
    return (double)(pref * sum);
}

/* 9j { j1 j2 j3 ; j4 j5 j6 ; j7 j8 j9 } as a sum over products of three 6j symbols */
double po_wigner9j(int j1, int j2, int j3, int j4, int j5, int j6, int j7, int j8, int j9)
{
    if (!po_triangle_ok(j1, j2, j3) || !po_triangle_ok(j4, j5, j6) || !po_triangle_ok(j7, j8, j9) ||
        !po_triangle_ok(j1, j4, j7) || !po_triangle_ok(j2, j5, j8) || !po_triangle_ok(j3, j6, j9)) return 0.0;
    int kmin = abs(j1 - j9); if (abs(j4 - j8) > kmin) kmin = abs(j4 - j8); if (abs(j2 - j6) > kmin) kmin = abs(j2 - j6);
    int kmax = j1 + j9; if (j4 + j8 < kmax) kmax = j4 + j8; if (j2 + j6 < kmax) kmax = j2 + j6;
    long double sum = 0.0L;
    for (int k = kmin; k <= kmax; k += 2) {
        long double t = (long double)(k + 1)
            * po_wigner6j(j1, j4, j7, j8, j9, k) * po_wigner6j(j2, j5, j8, j4, k, j6) * po_wigner6j(j3, j6, j9, k, j1, j2);
        sum += (k & 1) ? -t : t;       /* (-1)^(2k) with k doubled */
    }
    return (double)sum;
}

/* ------------------------------------------------------------------------------------------
 * Spherical harmonics of a unit vector u = (ux, 0, uz) lying in the xz-plane (all four
 * directions p^, q^, p'^, q'^ are coplanar).  Condon-Shortley phase.
 * The azimuth is 0 or pi; using the SIGNED ux in place of sin(theta) yields the factor
 * exp(i m pi) = (-1)^m automatically, so the value is real.   Y_{l,-m} = (-1)^m Y_{lm}.
 * Pinned against scipy.special.sph_harm_y in tests/test_oracle_algebra.py.
 * ---------------------------------------------------------------------------------------- */
static real po_ylm_r(int l, int m, real ux, real uz)
{
    int am = m < 0 ? -m : m;
    if (am > l) return 0;
    /* P_am^am = (-1)^am (2am-1)!! ux^am */
    real pmm = 1;
    for (int k = 1; k <= am; ++k) pmm *= -(real)(2 * k - 1) * ux;
    real plm;
    if (l == am) plm = pmm;
    else {
        real pm1 = uz * (real)(2 * am + 1) * pmm;      /* P_{am+1}^am */
        if (l == am + 1) plm = pm1;
        else {
            real pm2 = pmm; plm = 0;
            for (int ll = am + 2; ll <= l; ++ll) {
                plm = ((real)(2 * ll - 1) * uz * pm1 - (real)(ll + am - 1) * pm2) / (real)(ll - am);
                pm2 = pm1; pm1 = plm;
            }
        }
    }
    real norm = RSQRT((real)(2 * l + 1) / (4 * (real)PO_PI) * (real)(po_fact(l - am) / po_fact(l + am)));
    real y = norm * plm;
    if (m < 0 && (am & 1)) y = -y;
    return y;
}

double po_ylm(int l, int m, double ux, double uz) { return (double)po_ylm_r(l, m, (real)ux, (real)uz); }

/* ------------------------------------------------------------------------------------------
 * Recoupling coefficients (the paper only names them: g in eq. 22,
 * PAPER.md:L213-215, L256).
 *   jI -> LS:  C^{LS}_alpha = sqrt((2j+1)(2I+1)(2L+1)(2S+1)) 9j{ l s j ; lam 1/2 I ; L S J }
 *   spin:      R2(s,s';S) = <((23)s,1)S | ((31)s',2)S> = (-1)^{s'} sqrt((2s+1)(2s'+1)) 6j{1/2 1/2 s ; 1/2 S s'}
 *              R3(s,s';S) = <((23)s,1)S | ((12)s',3)S> = (-1)^{s+s'} R2(s,s';S)
 *   (same forms for isospin with t, T)
 * ---------------------------------------------------------------------------------------- */
double po_recoupling_C(const po_channel* a, int L, int S2, int J2)
{
    double n9 = po_wigner9j(2 * a->l, 2 * a->s, 2 * a->j, 2 * a->lam, 1, a->I2, 2 * L, S2, J2);
    return sqrt((double)((2 * a->j + 1) * (a->I2 + 1) * (2 * L + 1) * (S2 + 1))) * n9;
}

double po_spin_R(int s, int sp, int S2, int set)
{
    double v = sqrt((double)((2 * s + 1) * (2 * sp + 1))) * po_wigner6j(1, 1, 2 * s, 1, S2, 2 * sp);
    int ph = (set == 3) ? s : sp;       /* set 2: (-1)^{s'};  set 3: (-1)^{s+s'}(-1)^{s'} = (-1)^{s} */
    return (ph & 1) ? -v : v;
}

/* c^L_{alpha alpha'} = 8 pi^2 * sum_S C^{LS}_alpha C^{LS}_alpha' R(s,s';S) R(t,t';T)   (one cyclic term).
 * Spinless bosons: C = 1 iff L = J (j = l, I = lam, J = L), R = 1. */
double po_coef_L(const po_channel* a, const po_channel* b, int L, int J2, int T2, int stat, int set)
{
    const double pre = 8.0 * (double)(PO_PI * PO_PI);
    if (stat == PO_SPINLESS_BOSON) {
        if (2 * L != J2) return 0.0;
        if (!po_triangle_ok(2 * a->l, 2 * a->lam, 2 * L) || !po_triangle_ok(2 * b->l, 2 * b->lam, 2 * L)) return 0.0;
        return pre;
    }
    double sum = 0.0;
    for (int S2 = 1; S2 <= 3; S2 += 2) {
        double Ca = po_recoupling_C(a, L, S2, J2);
        double Cb = po_recoupling_C(b, L, S2, J2);
        if (Ca == 0.0 || Cb == 0.0) continue;
        sum += Ca * Cb * po_spin_R(a->s, b->s, S2, set) * po_spin_R(a->t, b->t, T2, set);
    }
    return pre * sum;
}

/* coupled(alpha, alpha') <=> LS(alpha) and LS(alpha') intersect — pure integer logic (reading R8):
 * LS(alpha) = {(L,S): |l-lam|<=L<=l+lam, |s-1/2|<=S<=s+1/2, |L-S|<=J<=L+S}. */
static int po_has_LS(const po_channel* a, int L, int S2, int J2, int stat)
{
    if (!po_triangle_ok(2 * a->l, 2 * a->lam, 2 * L)) return 0;
    if (stat == PO_SPINLESS_BOSON) return (2 * L == J2) && (S2 == 0);
    if (!(S2 >= abs(2 * a->s - 1) && S2 <= 2 * a->s + 1)) return 0;
    return po_triangle_ok(2 * L, S2, J2);
}

int po_coupled(const po_channel* a, const po_channel* b, int J2, int stat)
{
    int Lmax = a->l + a->lam;
    for (int L = 0; L <= Lmax; ++L)
        for (int S2 = 0; S2 <= 3; ++S2)
            if (po_has_LS(a, L, S2, J2, stat) && po_has_LS(b, L, S2, J2, stat)) return 1;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Jacobi momenta of the rotated sets, equal masses, in the frame q^ = z, p^ = (sqrt(1-x^2),0,x)
 * (DESIGN.md sec. 3.2):   set 2: p' = -p/2 - 3q/4,  q' =  p - q/2      (north_star's map)
 *                         set 3: p' = -p/2 + 3q/4,  q' = -p - q/2
 * Returns unit vectors (ux,uz) of p' and q' from the vector COMPONENTS (well conditioned).
 * ---------------------------------------------------------------------------------------- */
static void po_rotated_dirs(real p, real q, real x, int set, real* ppx, real* ppz, real* qpx, real* qpz)
{
    real sx = RSQRT((1 - x) * (1 + x));
    real ax, az, bx, bz;
    if (set == 3) { ax = -(real)0.5 * p * sx; az = -(real)0.5 * p * x + (real)0.75 * q; bx = -p * sx; bz = -p * x - (real)0.5 * q; }
    else          { ax = -(real)0.5 * p * sx; az = -(real)0.5 * p * x - (real)0.75 * q; bx =  p * sx; bz =  p * x - (real)0.5 * q; }
    real na = RSQRT(ax * ax + az * az), nb = RSQRT(bx * bx + bz * bz);
    *ppx = ax / na; *ppz = az / na; *qpx = bx / nb; *qpz = bz / nb;
}

/* bipolar harmonic  Y^{LM}_{l lam}(a^, b^) = sum_m <l m lam M-m | L M> Y_{lm}(a^) Y_{lam,M-m}(b^) */
static real po_bipolar(int l, int lam, int L, int M, real ax, real az, real bx, real bz)
{
    real sum = 0;
    for (int m = -l; m <= l; ++m) {
        int mu = M - m;
        if (mu < -lam || mu > lam) continue;
        double cg = po_cg(2 * l, 2 * m, 2 * lam, 2 * mu, 2 * L, 2 * M);
        if (cg == 0.0) continue;
        sum += (real)cg * po_ylm_r(l, m, ax, az) * po_ylm_r(lam, mu, bx, bz);
    }
    return sum;
}

/* orbital function A^L_{l lam, l' lam'}(p,q,x) = (2L+1)^-1 sum_M Y^{LM}_{l lam}(p^,q^) Y^{LM}_{l' lam'}(p'^,q'^) */
static real po_A_r(int l, int lam, int lp, int lamp, int L, real p, real q, real x, int set)
{
    real sx = RSQRT((1 - x) * (1 + x));
    real ppx, ppz, qpx, qpz;
    po_rotated_dirs(p, q, x, set, &ppx, &ppz, &qpx, &qpz);
    real sum = 0;
    for (int M = -L; M <= L; ++M)
        sum += po_bipolar(l, lam, L, M, sx, x, 0, 1) * po_bipolar(lp, lamp, L, M, ppx, ppz, qpx, qpz);
    return sum / (real)(2 * L + 1);
}

double po_A(int l, int lam, int lp, int lamp, int L, double p, double q, double x, int set)
{ return (double)po_A_r(l, lam, lp, lamp, L, (real)p, (real)q, (real)x, set); }

/* G^{(set)}_{alpha alpha'}(p,q,x) = sum_L c^L_{alpha alpha'} A^L_{l lam, l' lam'}(p,q,x): ONE cyclic term
 * (set = 2 or 3).  The matrix build uses 2*G^{(2)} (reading R4). */
double po_G(const po_channel* a, const po_channel* b, int J2, int T2, int stat, double p, double q, double x, int set)
{
    int Lmax = a->l + a->lam;
    real sum = 0;
    for (int L = 0; L <= Lmax; ++L) {
        double c = po_coef_L(a, b, L, J2, T2, stat, set);
        if (c == 0.0) continue;
        sum += (real)c * po_A_r(a->l, a->lam, b->l, b->lam, L, (real)p, (real)q, (real)x, set);
    }
    return (double)sum;
}

/* ------------------------------------------------------------------------------------------
 * Node map and cell location — DESIGN.md sec. 3.1, the exact IEEE-double operation order
 * (no FMA: compiled with -ffp-contract=off).  north_star: p'^2 = p^2/4 + 9q^2/16 + (3/4)pqx,
 * q'^2 = p^2 + q^2/4 - pqx.
 * ---------------------------------------------------------------------------------------- */
typedef struct { double p, q, x, w, pp, qq; int ic, jc; } po_node;   /* ic/jc = target cell or -1 */

/* largest k with e[k] <= v, i.e. (number of edges <= v) - 1; cells are half-open [e[k], e[k+1]) */
static int po_locate(const double* e, int N, double v)
{
    int cnt = 0;
    for (int k = 0; k <= N; ++k) if (e[k] <= v) ++cnt;
    return cnt - 1;
}

static void po_make_node(const double* pe, int Np, const double* qe, int Nq, int i, int j,
                         double ta, double wa, double tb, double wb, double tc, double wc, po_node* nd)
{
    double cp = 0.5 * (pe[i] + pe[i + 1]), hp = 0.5 * (pe[i + 1] - pe[i]);
    double cq = 0.5 * (qe[j] + qe[j + 1]), hq = 0.5 * (qe[j + 1] - qe[j]);
    double p = cp + hp * ta;
    double q = cq + hq * tb;
    double x = tc;
    double pq = p * q;
    double P2 = (0.25 * (p * p) + 0.5625 * (q * q)) + 0.75 * (pq * x);
    double Q2 = ((p * p) + 0.25 * (q * q)) - pq * x;
    if (P2 < 0.0) P2 = 0.0;
    if (Q2 < 0.0) Q2 = 0.0;
    double pp = sqrt(P2), qq = sqrt(Q2);
    int ic = po_locate(pe, Np, pp), jc = po_locate(qe, Nq, qq);
    if (ic < 0 || ic >= Np || jc < 0 || jc >= Nq || pp == 0.0 || qq == 0.0) { ic = -1; jc = -1; }
    nd->p = p; nd->q = q; nd->x = x; nd->pp = pp; nd->qq = qq; nd->ic = ic; nd->jc = jc;
    nd->w = ((hp * wa) * (hq * wb)) * wc;
}

/* Per-node table of one source cell, for the measure-conservation and invariant pins.
 * out arrays have n_p*n_q*n_x entries, lexicographic (a,b,c) order. */
int po_cell_nodes(const double* pe, int Np, const double* qe, int Nq, int cell,
                  const double* tp, const double* wp, int n_p, const double* tq, const double* wq, int n_q,
                  const double* tx, const double* wx, int n_x,
                  double* p, double* q, double* x, double* w, double* pp, double* qq, int32_t* target)
{
    int i = cell / Nq, j = cell % Nq, n = 0;
    for (int a = 0; a < n_p; ++a) for (int b = 0; b < n_q; ++b) for (int c = 0; c < n_x; ++c, ++n) {
        po_node nd;
        po_make_node(pe, Np, qe, Nq, i, j, tp[a], wp[a], tq[b], wq[b], tx[c], wx[c], &nd);
        p[n] = nd.p; q[n] = nd.q; x[n] = nd.x; w[n] = nd.w; pp[n] = nd.pp; qq[n] = nd.qq;
        target[n] = nd.ic < 0 ? -1 : nd.ic * Nq + nd.jc;
    }
    return n;
}

/* ------------------------------------------------------------------------------------------
 * Tables that depend on the channel list only (computed once per build): coupled mask, the
 * coefficients c^L, and Clebsch-Gordan tables of the bipolar harmonics that occur.
 * ---------------------------------------------------------------------------------------- */
#define PO_MAXL 10     /* max total orbital L kept in tables: L <= J + 3/2 = 10 for J = 17/2 (Table 1) */
typedef struct { int l, lam, L; double cg[2 * PO_MAXL + 1][2 * PO_LMAX + 1]; } po_triple;
typedef struct {
    int n_ch, n_tri, lmax;
    unsigned char* coupled;     /* n_ch*n_ch */
    double* coef;               /* [n_ch*n_ch][PO_MAXL+1]: 2 * c^L (both cyclic terms, reading R4) */
    int* tri_of;                /* [n_ch][PO_MAXL+1] -> triple index of (l,lam,L) or -1 */
    po_triple* tri;
} po_tables;

static int po_find_triple(po_tables* T, int l, int lam, int L)
{
    for (int k = 0; k < T->n_tri; ++k) if (T->tri[k].l == l && T->tri[k].lam == lam && T->tri[k].L == L) return k;
    po_triple* t = &T->tri[T->n_tri];
    t->l = l; t->lam = lam; t->L = L;
    for (int M = -L; M <= L; ++M) for (int m = -l; m <= l; ++m)
        t->cg[M + L][m + l] = (abs(M - m) <= lam) ? po_cg(2 * l, 2 * m, 2 * lam, 2 * (M - m), 2 * L, 2 * M) : 0.0;
    return T->n_tri++;
}

static int po_tables_init(po_tables* T, const po_channel* ch, int n_ch, int J2, int T2, int stat)
{
    memset(T, 0, sizeof(*T));
    T->n_ch = n_ch;
    T->coupled = (unsigned char*)calloc((size_t)n_ch * n_ch, 1);
    T->coef = (double*)calloc((size_t)n_ch * n_ch * (PO_MAXL + 1), sizeof(double));
    T->tri_of = (int*)malloc(sizeof(int) * n_ch * (PO_MAXL + 1));
    T->tri = (po_triple*)malloc(sizeof(po_triple) * n_ch * (PO_MAXL + 1));
    if (!T->coupled || !T->coef || !T->tri_of || !T->tri) return -1;
    if (stat != PO_SPINLESS_BOSON && (J2 + 3) / 2 > PO_MAXL) return -2;
    if (stat == PO_SPINLESS_BOSON && J2 / 2 > PO_MAXL) return -2;
    for (int a = 0; a < n_ch; ++a) {
        if (ch[a].l > PO_LMAX || ch[a].lam > PO_LMAX) return -2;
        if (ch[a].l > T->lmax) T->lmax = ch[a].l;
        if (ch[a].lam > T->lmax) T->lmax = ch[a].lam;
    }
    for (int a = 0; a < n_ch; ++a) for (int b = 0; b < n_ch; ++b) {
        T->coupled[a * n_ch + b] = (unsigned char)po_coupled(&ch[a], &ch[b], J2, stat);
        for (int L = 0; L <= PO_MAXL; ++L)
            T->coef[((size_t)a * n_ch + b) * (PO_MAXL + 1) + L] =
                2.0 * po_coef_L(&ch[a], &ch[b], L, J2, T2, stat, 2);
    }
    /* a triple (l,lam,L) is tabulated only if some coefficient with that channel and L is nonzero */
    for (int a = 0; a < n_ch; ++a) for (int L = 0; L <= PO_MAXL; ++L) {
        int used = 0;
        for (int b = 0; b < n_ch && !used; ++b)
            used = T->coef[((size_t)a * n_ch + b) * (PO_MAXL + 1) + L] != 0.0 ||
                   T->coef[((size_t)b * n_ch + a) * (PO_MAXL + 1) + L] != 0.0;
        T->tri_of[a * (PO_MAXL + 1) + L] = used ? po_find_triple(T, ch[a].l, ch[a].lam, L) : -1;
    }
    return 0;
}

static void po_tables_free(po_tables* T) { free(T->coupled); free(T->coef); free(T->tri_of); free(T->tri); }

/* all bipolar harmonics Y^{LM}_{l lam}(a^, b^) of the triple table at one pair of directions */
static void po_eval_bipolar(const po_tables* T, real ax, real az, real bx, real bz, real (*out)[2 * PO_MAXL + 1])
{
    real Ya[PO_LMAX + 1][2 * PO_LMAX + 1], Yb[PO_LMAX + 1][2 * PO_LMAX + 1];
    for (int l = 0; l <= T->lmax; ++l) for (int m = -l; m <= l; ++m) {
        Ya[l][m + l] = po_ylm_r(l, m, ax, az);
        Yb[l][m + l] = po_ylm_r(l, m, bx, bz);
    }
    for (int k = 0; k < T->n_tri; ++k) {
        const po_triple* t = &T->tri[k];
        for (int M = -t->L; M <= t->L; ++M) {
            real sum = 0;
            for (int m = -t->l; m <= t->l; ++m) {
                int mu = M - m;
                if (mu < -t->lam || mu > t->lam) continue;
                sum += (real)t->cg[M + t->L][m + t->l] * Ya[t->l][m + t->l] * Yb[t->lam][mu + t->lam];
            }
            out[k][M + t->L] = sum;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * The build (DESIGN.md sec. 3.1 = SURVEY.md sec. 8(c.1)), rows of source cells
 * [cell_begin, cell_end):
 *   row r = (cell - cell_begin)*n_ch + alpha, column c = cell'*n_ch + alpha' (GLOBAL), columns
 *   ascending; pattern = {hit cells} x {coupled(alpha,alpha')} — structural, never by value.
 *   P0[r][c] = ( sum_{nodes of (i,j) landing in (i',j')} omega * 2 G2_{alpha alpha'}(p,q,x) )
 *              / sqrt(d_i dbar_j d_i' dbar_j')
 * Call with colidx = vals = NULL to count (rowptr and *nnz_out are still filled).
 * Returns 0, or <0 on bad arguments / capacity overflow.
 * ---------------------------------------------------------------------------------------- */
/* Cell norm B_k of the radial basis (reading R2; eq. 21 is garbled in PAPER.md:L208):
 *   norm = 0, reading A: delta(p-p')-normalised radial states, f = 1, B_k = e[k+1] - e[k] (the width);
 *   norm = 1, reading B: states normalised in the p^2 dp measure,  B_k = (e[k+1]^3 - e[k]^3)/3.
 * Node weight: A  w * pq/(p'q') ;  B  w * p^2 q^2.  Prefactor (B_i Bbar_j B_i' Bbar_j')^(-1/2) in both. */
static real po_cell_norm(const double* e, int k, int norm)
{
    if (norm == 1) return ((real)e[k + 1] * (real)e[k + 1] * (real)e[k + 1] - (real)e[k] * (real)e[k] * (real)e[k]) / 3;
    return (real)e[k + 1] - (real)e[k];
}

int po_build_norm(const double* pe, int Np, const double* qe, int Nq,
             const po_channel* ch, int n_ch, int J2, int T2, int stat,
             const double* tp, const double* wp, int n_p, const double* tq, const double* wq, int n_q,
             const double* tx, const double* wx, int n_x,
             int cell_begin, int cell_end,
             int64_t* rowptr, int32_t* colidx, double* vals, int64_t cap, int64_t* nnz_out, int norm)
{
    const int n_cells = Np * Nq;
    if (cell_begin < 0 || cell_end > n_cells || cell_begin > cell_end) return -1;
    po_tables T;
    int rc = po_tables_init(&T, ch, n_ch, J2, T2, stat);
    if (rc) { po_tables_free(&T); return rc; }
    const int nblk = cell_end - cell_begin;
    const int nnode = n_p * n_q * n_x;

    /* pass 1: hit cells of every source cell -> row lengths */
    int* nhit = (int*)calloc((size_t)nblk + 1, sizeof(int));
    int* ncoup = (int*)calloc((size_t)n_ch, sizeof(int));
    for (int a = 0; a < n_ch; ++a) for (int b = 0; b < n_ch; ++b) ncoup[a] += T.coupled[a * n_ch + b];
#pragma omp parallel
    {
        unsigned char* flag = (unsigned char*)malloc((size_t)n_cells);
#pragma omp for schedule(dynamic, 8)
        for (int cb = 0; cb < nblk; ++cb) {
            int cell = cell_begin + cb, i = cell / Nq, j = cell % Nq;
            memset(flag, 0, (size_t)n_cells);
            for (int a = 0; a < n_p; ++a) for (int b = 0; b < n_q; ++b) for (int c = 0; c < n_x; ++c) {
                po_node nd;
                po_make_node(pe, Np, qe, Nq, i, j, tp[a], wp[a], tq[b], wq[b], tx[c], wx[c], &nd);
                if (nd.ic >= 0) flag[nd.ic * Nq + nd.jc] = 1;
            }
            int h = 0;
            for (int k = 0; k < n_cells; ++k) h += flag[k];
            nhit[cb] = h;
        }
        free(flag);
    }
    rowptr[0] = 0;
    for (int cb = 0; cb < nblk; ++cb)
        for (int a = 0; a < n_ch; ++a)
            rowptr[(int64_t)cb * n_ch + a + 1] = rowptr[(int64_t)cb * n_ch + a] + (int64_t)nhit[cb] * ncoup[a];
    const int64_t nnz = rowptr[(int64_t)nblk * n_ch];
    *nnz_out = nnz;
    if (!colidx && !vals) { free(nhit); free(ncoup); po_tables_free(&T); return 0; }
    if (nnz > cap) { free(nhit); free(ncoup); po_tables_free(&T); return -3; }

    /* pass 2: values */
#pragma omp parallel
    {
        unsigned char* flag = (unsigned char*)malloc((size_t)n_cells);
        int* local = (int*)malloc(sizeof(int) * (size_t)n_cells);     /* target cell -> hit rank */
        int* hitcell = (int*)malloc(sizeof(int) * (size_t)n_cells);
        po_node* nodes = (po_node*)malloc(sizeof(po_node) * (size_t)nnode);
        real (*bra)[2 * PO_MAXL + 1] = malloc(sizeof(real[2 * PO_MAXL + 1]) * (size_t)(T.n_tri + 1));
        real (*ket)[2 * PO_MAXL + 1] = malloc(sizeof(real[2 * PO_MAXL + 1]) * (size_t)(T.n_tri + 1));
        real* acc = NULL; size_t acc_cap = 0;
#pragma omp for schedule(dynamic, 4)
        for (int cb = 0; cb < nblk; ++cb) {
            int cell = cell_begin + cb, i = cell / Nq, j = cell % Nq;
            memset(flag, 0, (size_t)n_cells);
            int n = 0;
            for (int a = 0; a < n_p; ++a) for (int b = 0; b < n_q; ++b) for (int c = 0; c < n_x; ++c, ++n) {
                po_make_node(pe, Np, qe, Nq, i, j, tp[a], wp[a], tq[b], wq[b], tx[c], wx[c], &nodes[n]);
                if (nodes[n].ic >= 0) flag[nodes[n].ic * Nq + nodes[n].jc] = 1;
            }
            int H = 0;
            for (int k = 0; k < n_cells; ++k) if (flag[k]) { local[k] = H; hitcell[H++] = k; }
            size_t need = (size_t)H * n_ch * n_ch;
            if (need > acc_cap) { free(acc); acc = (real*)malloc(sizeof(real) * need); acc_cap = need; }
            for (size_t k = 0; k < need; ++k) acc[k] = 0;

            for (n = 0; n < nnode; ++n) {
                const po_node* nd = &nodes[n];
                if (nd->ic < 0) continue;
                real p = nd->p, q = nd->q, x = nd->x;
                real omega = norm == 1 ? (real)(nd->w * ((nd->p * nd->q) * (nd->p * nd->q)))
                                       : (real)(nd->w * ((nd->p * nd->q) / (nd->pp * nd->qq)));
                real sx = RSQRT((1 - x) * (1 + x));
                real ppx, ppz, qpx, qpz;
                po_rotated_dirs(p, q, x, 2, &ppx, &ppz, &qpx, &qpz);
                po_eval_bipolar(&T, sx, x, 0, 1, bra);
                po_eval_bipolar(&T, ppx, ppz, qpx, qpz, ket);
                real* A = acc + (size_t)local[nd->ic * Nq + nd->jc] * n_ch * n_ch;
                for (int a = 0; a < n_ch; ++a) for (int b = 0; b < n_ch; ++b) {
                    if (!T.coupled[a * n_ch + b]) continue;
                    real G = 0;
                    for (int L = 0; L <= PO_MAXL; ++L) {
                        double c = T.coef[((size_t)a * n_ch + b) * (PO_MAXL + 1) + L];
                        if (c == 0.0) continue;
                        int ta = T.tri_of[a * (PO_MAXL + 1) + L], tb = T.tri_of[b * (PO_MAXL + 1) + L];
                        real AL = 0;
                        for (int M = -L; M <= L; ++M) AL += bra[ta][M + L] * ket[tb][M + L];
                        G += (real)c * (AL / (real)(2 * L + 1));
                    }
                    A[a * n_ch + b] += omega * G;
                }
            }
            /* emit rows of this source cell */
            real di = po_cell_norm(pe, i, norm), dj = po_cell_norm(qe, j, norm);
            for (int a = 0; a < n_ch; ++a) {
                int64_t pos = rowptr[(int64_t)cb * n_ch + a];
                for (int h = 0; h < H; ++h) {
                    int ic = hitcell[h] / Nq, jc = hitcell[h] % Nq;
                    real dic = po_cell_norm(pe, ic, norm), djc = po_cell_norm(qe, jc, norm);
                    real norm = RSQRT(di * dj * dic * djc);
                    for (int b = 0; b < n_ch; ++b) {
                        if (!T.coupled[a * n_ch + b]) continue;
                        if (colidx) colidx[pos] = hitcell[h] * n_ch + b;
                        if (vals) vals[pos] = (double)(acc[((size_t)h * n_ch + a) * n_ch + b] / norm);
                        ++pos;
                    }
                }
            }
        }
        free(flag); free(local); free(hitcell); free(nodes); free(bra); free(ket); free(acc);
    }
    free(nhit); free(ncoup); po_tables_free(&T);
    return 0;
}

int po_build(const double* pe, int Np, const double* qe, int Nq,
             const po_channel* ch, int n_ch, int J2, int T2, int stat,
             const double* tp, const double* wp, int n_p, const double* tq, const double* wq, int n_q,
             const double* tx, const double* wx, int n_x,
             int cell_begin, int cell_end,
             int64_t* rowptr, int32_t* colidx, double* vals, int64_t cap, int64_t* nnz_out)
{
    return po_build_norm(pe, Np, qe, Nq, ch, n_ch, J2, T2, stat, tp, wp, n_p, tq, wq, n_q, tx, wx, n_x, cell_begin, cell_end,
                         rowptr, colidx, vals, cap, nnz_out, 0);
}

/* ------------------------------------------------------------------------------------------
 * Exact-overlap evaluation — the paper's own route: "a double integral with variable limits"
 * (sec. 3.2).  For a fixed outer node (p, q) of the source cell the image moves along
 *   p'^2 = A + B x ,  q'^2 = C - D x ,   A = p^2/4 + 9q^2/16, B = 3pq/4, C = p^2 + q^2/4, D = pq  (B, D > 0),
 * both linear in x, so the x-values landing in target cell (i', j') form ONE interval
 *   x_lo = max(-1, (pe[i']^2 - A)/B, (C - qe[j'+1]^2)/D) ,  x_hi = min(1, (pe[i'+1]^2 - A)/B, (C - qe[j']^2)/D),
 * and the smooth integrand is integrated over it with the n_x-point rule mapped to [x_lo, x_hi].  The outer (p, q)
 * rule is the tensor rule of the node-binning scheme.  Pattern: target cells with a non-empty interval (x_hi > x_lo)
 * for at least one outer node, times the coupled-channel mask.  Plain loops over ALL target cells — slow, obvious.
 * Same output conventions as po_build; norm as in po_build_norm.
 * ---------------------------------------------------------------------------------------- */
static int po_xo_interval(const double* pe, const double* qe, int ic, int jc, double A, double B, double C, double D,
                          double* x_lo, double* x_hi)
{
    double lo = -1.0, hi = 1.0, v;
    v = (pe[ic] * pe[ic] - A) / B;         if (v > lo) lo = v;
    v = (C - qe[jc + 1] * qe[jc + 1]) / D; if (v > lo) lo = v;
    v = (pe[ic + 1] * pe[ic + 1] - A) / B; if (v < hi) hi = v;
    v = (C - qe[jc] * qe[jc]) / D;         if (v < hi) hi = v;
    *x_lo = lo; *x_hi = hi;
    return hi > lo;
}

int po_build_xo(const double* pe, int Np, const double* qe, int Nq,
                const po_channel* ch, int n_ch, int J2, int T2, int stat,
                const double* tp, const double* wp, int n_p, const double* tq, const double* wq, int n_q,
                const double* tx, const double* wx, int n_x,
                int cell_begin, int cell_end,
                int64_t* rowptr, int32_t* colidx, double* vals, int64_t cap, int64_t* nnz_out, int norm)
{
    const int n_cells = Np * Nq;
    if (cell_begin < 0 || cell_end > n_cells || cell_begin > cell_end) return -1;
    po_tables T;
    int rc = po_tables_init(&T, ch, n_ch, J2, T2, stat);
    if (rc) { po_tables_free(&T); return rc; }
    const int nblk = cell_end - cell_begin;
    int* ncoup = (int*)calloc((size_t)n_ch, sizeof(int));
    for (int a = 0; a < n_ch; ++a) for (int b = 0; b < n_ch; ++b) ncoup[a] += T.coupled[a * n_ch + b];
    unsigned char* hit = (unsigned char*)calloc((size_t)nblk * n_cells + 1, 1);     /* [source][target] */
    /* pass 1: which targets have a non-empty interval */
#pragma omp parallel for schedule(dynamic, 4)
    for (int cb = 0; cb < nblk; ++cb) {
        int cell = cell_begin + cb, i = cell / Nq, j = cell % Nq;
        double cp = 0.5 * (pe[i] + pe[i + 1]), hp = 0.5 * (pe[i + 1] - pe[i]);
        double cq = 0.5 * (qe[j] + qe[j + 1]), hq = 0.5 * (qe[j + 1] - qe[j]);
        for (int a = 0; a < n_p; ++a) for (int b = 0; b < n_q; ++b) {
            double p = cp + hp * tp[a], q = cq + hq * tq[b];
            double A = 0.25 * (p * p) + 0.5625 * (q * q), B = 0.75 * (p * q), C = (p * p) + 0.25 * (q * q), D = p * q;
            for (int t = 0; t < n_cells; ++t) {
                double lo, hi;
                if (po_xo_interval(pe, qe, t / Nq, t % Nq, A, B, C, D, &lo, &hi)) hit[(size_t)cb * n_cells + t] = 1;
            }
        }
    }
    rowptr[0] = 0;
    for (int cb = 0; cb < nblk; ++cb) {
        int64_t h = 0;
        for (int t = 0; t < n_cells; ++t) h += hit[(size_t)cb * n_cells + t];
        for (int a = 0; a < n_ch; ++a) rowptr[(int64_t)cb * n_ch + a + 1] = rowptr[(int64_t)cb * n_ch + a] + h * ncoup[a];
    }
    const int64_t nnz = rowptr[(int64_t)nblk * n_ch];
    *nnz_out = nnz;
    if ((!colidx && !vals) || nnz > cap) { int r = (!colidx && !vals) ? 0 : -3; free(hit); free(ncoup); po_tables_free(&T); return r; }
    /* pass 2: values */
#pragma omp parallel
    {
        real (*bra)[2 * PO_MAXL + 1] = malloc(sizeof(real[2 * PO_MAXL + 1]) * (size_t)(T.n_tri + 1));
        real (*ket)[2 * PO_MAXL + 1] = malloc(sizeof(real[2 * PO_MAXL + 1]) * (size_t)(T.n_tri + 1));
        real* acc = (real*)malloc(sizeof(real) * (size_t)n_ch * n_ch);
#pragma omp for schedule(dynamic, 2)
        for (int cb = 0; cb < nblk; ++cb) {
            int cell = cell_begin + cb, i = cell / Nq, j = cell % Nq;
            double cp = 0.5 * (pe[i] + pe[i + 1]), hp = 0.5 * (pe[i + 1] - pe[i]);
            double cq = 0.5 * (qe[j] + qe[j + 1]), hq = 0.5 * (qe[j + 1] - qe[j]);
            int h = 0;
            for (int t = 0; t < n_cells; ++t) {
                if (!hit[(size_t)cb * n_cells + t]) continue;
                int ic = t / Nq, jc = t % Nq;
                for (int k = 0; k < n_ch * n_ch; ++k) acc[k] = 0;
                for (int a = 0; a < n_p; ++a) for (int b = 0; b < n_q; ++b) {
                    double p = cp + hp * tp[a], q = cq + hq * tq[b];
                    double A = 0.25 * (p * p) + 0.5625 * (q * q), B = 0.75 * (p * q), C = (p * p) + 0.25 * (q * q), D = p * q;
                    double lo, hi;
                    if (!po_xo_interval(pe, qe, ic, jc, A, B, C, D, &lo, &hi)) continue;
                    double xm = 0.5 * (lo + hi), xh = 0.5 * (hi - lo);
                    for (int c = 0; c < n_x; ++c) {
                        double x = xm + xh * tx[c];
                        double w = ((hp * wp[a]) * (hq * wq[b])) * (xh * wx[c]);
                        double P2 = A + B * x, Q2 = C - D * x;
                        real omega;
                        if (norm == 1) omega = (real)(w * ((p * q) * (p * q)));
                        else {
                            if (P2 <= 0.0 || Q2 <= 0.0) continue;       /* only at an interval end that touches p' = 0 or q' = 0 */
                            omega = (real)(w * ((p * q) / (sqrt(P2) * sqrt(Q2))));
                        }
                        real sx = RSQRT((1 - (real)x) * (1 + (real)x));
                        real ppx, ppz, qpx, qpz;
                        po_rotated_dirs((real)p, (real)q, (real)x, 2, &ppx, &ppz, &qpx, &qpz);
                        po_eval_bipolar(&T, sx, (real)x, 0, 1, bra);
                        po_eval_bipolar(&T, ppx, ppz, qpx, qpz, ket);
                        for (int al = 0; al < n_ch; ++al) for (int be = 0; be < n_ch; ++be) {
                            if (!T.coupled[al * n_ch + be]) continue;
                            real G = 0;
                            for (int L = 0; L <= PO_MAXL; ++L) {
                                double cL = T.coef[((size_t)al * n_ch + be) * (PO_MAXL + 1) + L];
                                if (cL == 0.0) continue;
                                int ta = T.tri_of[al * (PO_MAXL + 1) + L], tb = T.tri_of[be * (PO_MAXL + 1) + L];
                                real AL = 0;
                                for (int M = -L; M <= L; ++M) AL += bra[ta][M + L] * ket[tb][M + L];
                                G += (real)cL * (AL / (real)(2 * L + 1));
                            }
                            acc[al * n_ch + be] += omega * G;
                        }
                    }
                }
                real nrm = RSQRT(po_cell_norm(pe, i, norm) * po_cell_norm(qe, j, norm) * po_cell_norm(pe, ic, norm) * po_cell_norm(qe, jc, norm));
                for (int al = 0; al < n_ch; ++al) {
                    int64_t pos = rowptr[(int64_t)cb * n_ch + al] + (int64_t)h * ncoup[al];
                    for (int be = 0; be < n_ch; ++be) {
                        if (!T.coupled[al * n_ch + be]) continue;
                        if (colidx) colidx[pos] = t * n_ch + be;
                        if (vals) vals[pos] = (double)(acc[al * n_ch + be] / nrm);
                        ++pos;
                    }
                }
                ++h;
            }
        }
        free(bra); free(ket); free(acc);
    }
    free(hit); free(ncoup); po_tables_free(&T);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Pattern only (no values): the hit cells of every source cell in [cell_begin, cell_end), ascending —
 * the geometric half of the pattern  {hit cells} x {coupled(alpha,alpha')}  of DESIGN.md sec. 3.1
 * (the paper's step 2a 'pre-selection').  Same node loop and the same po_make_node as
 * po_build, nothing else.  hitptr[nblk+1] is always written; hitcell (capacity cap) may be NULL to count.
 * Returns 0, -1 on bad arguments, -3 when cap is too small.
 * ---------------------------------------------------------------------------------------- */
int po_hit_cells(const double* pe, int Np, const double* qe, int Nq,
                 const double* tp, const double* wp, int n_p, const double* tq, const double* wq, int n_q,
                 const double* tx, const double* wx, int n_x,
                 int cell_begin, int cell_end, int64_t* hitptr, int32_t* hitcell, int64_t cap)
{
    const int n_cells = Np * Nq;
    if (cell_begin < 0 || cell_end > n_cells || cell_begin > cell_end) return -1;
    const int nblk = cell_end - cell_begin;
    for (int pass = 0; pass < 2; ++pass) {
        if (pass == 1) {
            hitptr[0] = 0;
            for (int cb = 0; cb < nblk; ++cb) hitptr[cb + 1] += hitptr[cb];     /* counts -> offsets */
            if (!hitcell) return 0;
            if (hitptr[nblk] > cap) return -3;
        }
#pragma omp parallel
        {
            unsigned char* flag = (unsigned char*)malloc((size_t)n_cells);
#pragma omp for schedule(dynamic, 8)
            for (int cb = 0; cb < nblk; ++cb) {
                int cell = cell_begin + cb, i = cell / Nq, j = cell % Nq;
                memset(flag, 0, (size_t)n_cells);
                for (int a = 0; a < n_p; ++a) for (int b = 0; b < n_q; ++b) for (int c = 0; c < n_x; ++c) {
                    po_node nd;
                    po_make_node(pe, Np, qe, Nq, i, j, tp[a], wp[a], tq[b], wq[b], tx[c], wx[c], &nd);
                    if (nd.ic >= 0) flag[nd.ic * Nq + nd.jc] = 1;
                }
                if (pass == 0) {
                    int64_t h = 0;
                    for (int k = 0; k < n_cells; ++k) h += flag[k];
                    hitptr[cb + 1] = h;
                } else {
                    int64_t pos = hitptr[cb];
                    for (int k = 0; k < n_cells; ++k) if (flag[k]) hitcell[pos++] = k;
                }
            }
            free(flag);
        }
    }
    return 0;
}

int po_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void po_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
