/*
 * fp_oracle.c -- plain, slow CPU oracle of the FourPhonon scattering-rate hot path.   TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or call
 * this file.  It shares no code, header, table or constant with the CUDA path (paper_2510_00518_b200/csrc): the two
 * are written independently from the same text.  The product path never calls into it.
 *
 * What it computes: the definition itself -- Algorithm 1 of the paper (loops over q', j', j'', the
 * momentum modulo PAPER.md:155, compute_sigma PAPER.md:161, the |Delta| <= 2 sigma filter and the Gaussian weight
 * PAPER.md:163, WP accumulation PAPER.md:166, compute_Vp PAPER.md:168, Gamma += WP |V|^2 PAPER.md:170 and the final
 * /nptk and unit constant PAPER.md:187-189), written out for the five channels 3ph +,- and 4ph ++,+-,-- over the FULL
 * rectangular domain, with the formulas the paper defers to its references taken from SURVEY.md §8(c) steps 1-8
 * (readings listed in DESIGN.md §3).  No blocking, no pre-contraction, no symmetry reduction: every allowed process
 * evaluates its matrix element from the raw IFC list by the nested Cartesian loops of the definition.
 *
 * Arithmetic: IEEE binary64 throughout.  Compile with -ffp-contract=off: the filter decision (step 3) is a pinned
 * sequence of separately rounded operations.  Per-mode sums are Neumaier-compensated in loop order.  OpenMP only
 * distributes (target, q') pairs over threads; partial sums are combined in index order, so results do not depend on
 * the thread count.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force momentum enumeration and an independent dense-Fourier
 * evaluation on 2x2x2 / 3x2x1 meshes, the adaptive-sigma window of BOTH orders against brute-force process lists on
 * 3x3x3 / 3x2x1 / 3x3x2 meshes (3ph: sigma from v' - v''; 4ph: sigma from v'' - v''', the reading of SURVEY.md §8(c)
 * item 2) with the weighted phase space summed directly over those lists, closed-form counts with the filter disabled, the 1-atom single-entry |V|^2 closed
 * form, gauge / cell-offset invariance, permutation symmetry of |V|, vanishing |V| for Gamma-acoustic legs under the
 * sum rule, time reversal, dyadic window-edge cases, sigma closed form on a cubic cell, on-shell occupation identities,
 * high-T scaling, kappa limits, CODATA constants derived two ways.
 * PARITY UNPINNED: absolute magnitudes against the paper -- the paper prints no rate, kappa or |V| value (PAPER.md:86
 * gives only "< 0.1 %" agreement between its own builds) and its silicon inputs are not available.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t natoms;            /* atoms per cell; nb = 3*natoms                                         */
    int32_t mesh[3];           /* N1,N2,N3                                                              */
    double lattvec[9];         /* rows a1,a2,a3 (Angstrom)                                              */
    const double *masses;      /* natoms (u)                                                            */
    const double *omega;       /* N*nb (rad/ps), index iq*nb+j                                          */
    const double *eig;         /* N*nb*nb*2: [iq][j][3*atom+alpha][re,im]                               */
    const double *vg;          /* N*nb*3 (Angstrom/ps)                                                  */
    int64_t n3;                /* triplets                                                              */
    const int32_t *atoms3;     /* n3*3  (i,j,k)                                                         */
    const int32_t *cells3;     /* n3*2*3 integer cell offsets of j,k                                    */
    const double *phi3;        /* n3*27, alpha slowest, gamma fastest (eV/A^3)                          */
    int64_t n4;
    const int32_t *atoms4;     /* n4*4                                                                  */
    const int32_t *cells4;     /* n4*3*3                                                                */
    const double *phi4;        /* n4*81 (eV/A^4)                                                        */
    double T;                  /* K                                                                     */
    double scale;              /* broadening scale factor                                               */
    double ncut;               /* window half-width in sigma (2 = PAPER.md:163); INFINITY disables      */
    double sigma_const;        /* >0: fixed sigma (rad/ps) for every process  */
} orc_setup;

/* ---- constants, SURVEY.md §8(c) "Constants": derived from CODATA 2018 in code ------------------------------------ */
static const double HBAR = 1.054571817e-34;   /* J s  */
static const double KB   = 1.380649e-23;      /* J/K  */
static const double QE   = 1.602176634e-19;   /* C    */
static const double AMU  = 1.66053906660e-27; /* kg   */
static const double PI   = 3.14159265358979323846;

static double hbar_over_kb_psK(void) { return HBAR / KB * 1e12; }
/* (pi hbar/4) (eV/A^3)^2 / u^3 / (rad/ps)^4, in 1/ps */
static double const_c3(void) { double ev_a3 = QE / 1e-30; return PI * HBAR / 4.0 * ev_a3 * ev_a3 / (AMU * AMU * AMU) * 1e-48 * 1e-12; }
/* (pi hbar^2/8) (eV/A^4)^2 / u^4 / (rad/ps)^5, in 1/ps */
static double const_c4(void) { double ev_a4 = QE / 1e-40; return PI * HBAR * HBAR / 8.0 * ev_a4 * ev_a4 / (AMU * AMU * AMU * AMU) * 1e-60 * 1e-12; }
/* hbar^2/kB * (rad/ps)^2 (A/ps)^2 ps / A^3, in W/(m K) */
static double const_ckappa(void) { return HBAR * HBAR / KB * 1e24 * 1e4 * 1e-12 / 1e-30; }

void orc_constants(double out[4]) { out[0] = const_c3(); out[1] = const_c4(); out[2] = const_ckappa(); out[3] = hbar_over_kb_psK(); }

/* ---- mesh helpers ------------------------------------------------------------------------------------------------ */
static int nq_of(const orc_setup *s) { return s->mesh[0] * s->mesh[1] * s->mesh[2]; }
static void q_coords(const orc_setup *s, int iq, int c[3]) {
    c[0] = iq % s->mesh[0]; c[1] = (iq / s->mesh[0]) % s->mesh[1]; c[2] = iq / (s->mesh[0] * s->mesh[1]);
}
static int imod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }
/* step 1: q_out = qa + sb*qb + sc*qc, per component modulo the mesh */
static int q_combine(const orc_setup *s, int qa, int sb, int qb, int sc, int qc) {
    int a[3], b[3], c[3], r[3];
    q_coords(s, qa, a); q_coords(s, qb, b); q_coords(s, qc, c);
    for (int m = 0; m < 3; m++) r[m] = imod(a[m] + sb * b[m] + sc * c[m], s->mesh[m]);
    return r[0] + s->mesh[0] * (r[1] + s->mesh[1] * r[2]);
}

/* ---- step 3: reciprocal vectors B_mu = b_mu/N_mu, pinned operation order ------------------------------------------ */
void orc_recip(const double lattvec[9], const int32_t mesh[3], double B[9]) {
    const double *a1 = lattvec, *a2 = lattvec + 3, *a3 = lattvec + 6;
    double c1[3], c2[3], c3[3];
    c1[0] = (a2[1] * a3[2]) - (a2[2] * a3[1]); c1[1] = (a2[2] * a3[0]) - (a2[0] * a3[2]); c1[2] = (a2[0] * a3[1]) - (a2[1] * a3[0]);
    c2[0] = (a3[1] * a1[2]) - (a3[2] * a1[1]); c2[1] = (a3[2] * a1[0]) - (a3[0] * a1[2]); c2[2] = (a3[0] * a1[1]) - (a3[1] * a1[0]);
    c3[0] = (a1[1] * a2[2]) - (a1[2] * a2[1]); c3[1] = (a1[2] * a2[0]) - (a1[0] * a2[2]); c3[2] = (a1[0] * a2[1]) - (a1[1] * a2[0]);
    double vol = (a1[0] * c1[0] + a1[1] * c1[1]) + a1[2] * c1[2];
    double twopi = 2.0 * PI;
    for (int x = 0; x < 3; x++) {
        B[0 + x] = ((twopi * c1[x]) / vol) / (double)mesh[0];
        B[3 + x] = ((twopi * c2[x]) / vol) / (double)mesh[1];
        B[6 + x] = ((twopi * c3[x]) / vol) / (double)mesh[2];
    }
}

/* compute_sigma(v' - v''); pinned order of SURVEY.md §8(c) step 3 */
static double sigma_of(const orc_setup *s, const double B[9], const double *va, const double *vb) {
    if (s->sigma_const > 0.0) return s->sigma_const;
    double dv[3], t[3];
    for (int c = 0; c < 3; c++) dv[c] = va[c] - vb[c];
    for (int m = 0; m < 3; m++) t[m] = (B[3 * m + 0] * dv[0] + B[3 * m + 1] * dv[1]) + B[3 * m + 2] * dv[2];
    double ss = (t[0] * t[0] + t[1] * t[1]) + t[2] * t[2];
    return s->scale * sqrt(ss / 6.0);
}
double orc_sigma(const orc_setup *s, const double va[3], const double vb[3]) {
    double B[9]; orc_recip(s->lattvec, s->mesh, B); return sigma_of(s, B, va, vb);
}
/* the filter, "<= 2 sigma" (inclusive; sigma = 0 rejects, item 3) */
static int allowed(const orc_setup *s, double delta, double sigma) { return (sigma > 0.0) && (fabs(delta) <= s->ncut * sigma); }
int orc_allowed(const orc_setup *s, double delta, double sigma) { return allowed(s, delta, sigma); }

/* step 4: Bose-Einstein occupation */
double orc_be(double omega, double T) { double x = hbar_over_kb_psK() * omega / T; return 1.0 / expm1(x); }
/* step 5: normalised Gaussian */
static double gauss(double delta, double sigma) { double r = delta / sigma; return exp(-(r * r)) / (sigma * sqrt(PI)); }

/* ---- step 6: matrix elements from the definition ----------------------------------------------------------------- */
typedef struct { double re, im; } cplx;
static cplx cmul(cplx a, cplx b) { cplx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; return r; }
static cplx cconj(cplx a) { cplx r = { a.re, -a.im }; return r; }

/* phi(sign*q, R) = exp(sign * 2 pi i sum_mu i_mu n_mu / N_mu); the integer numerators are reduced modulo N_mu (exact) */
static cplx bloch_phase(const orc_setup *s, int iq, int sign, const int32_t *cell) {
    int c[3]; q_coords(s, iq, c);
    double x = 0.0;
    for (int m = 0; m < 3; m++) x += (double)imod(sign * c[m] * cell[m], s->mesh[m]) / (double)s->mesh[m];
    cplx r = { cos(2.0 * PI * x), sin(2.0 * PI * x) };
    return r;
}
/* mass-scaled eigenvector component e~_lam(atom, alpha) = e / sqrt(m_atom) */
static cplx etilde(const orc_setup *s, int lam, int atom, int alpha) {
    int nb = 3 * s->natoms;
    const double *p = s->eig + ((size_t)lam * nb + 3 * atom + alpha) * 2;
    double sm = sqrt(s->masses[atom]);
    cplx r = { p[0] / sm, p[1] / sm };
    return r;
}

/* V3^{sign}(lam; lam1, lam2), sign=+1: absorption (q2 = q + q1), sign=-1: emission (q2 = q - q1).  SURVEY.md §8(c) step 6:
 *   V3+ = sum_t sum_abc Phi_t^{abc} e~_lam(i,a) . e~_lam1(j,b) phi(q1,Rj)        . conj(e~_lam2(k,c)) phi(-q2,Rk)
 *   V3- = sum_t sum_abc Phi_t^{abc} e~_lam(i,a) . conj(e~_lam1(j,b)) phi(-q1,Rj) . conj(e~_lam2(k,c)) phi(-q2,Rk)      */
void orc_v3(const orc_setup *s, int lam, int lam1, int lam2, int sign, double out[2]) {
    int nb = 3 * s->natoms;
    int q1 = lam1 / nb, q2 = lam2 / nb;
    cplx V = { 0.0, 0.0 };
    for (int64_t t = 0; t < s->n3; t++) {
        int i = s->atoms3[3 * t], j = s->atoms3[3 * t + 1], k = s->atoms3[3 * t + 2];
        const int32_t *Rj = s->cells3 + 6 * t, *Rk = s->cells3 + 6 * t + 3;
        cplx pj = bloch_phase(s, q1, sign, Rj), pk = bloch_phase(s, q2, -1, Rk);
        cplx acc = { 0.0, 0.0 };
        for (int a = 0; a < 3; a++) {
            cplx ea = etilde(s, lam, i, a);
            for (int b = 0; b < 3; b++) {
                cplx eb = etilde(s, lam1, j, b);
                if (sign < 0) eb = cconj(eb);
                cplx eab = cmul(ea, eb);
                for (int c = 0; c < 3; c++) {
                    cplx ec = cconj(etilde(s, lam2, k, c));
                    cplx prod = cmul(eab, ec);
                    double f = s->phi3[27 * t + 9 * a + 3 * b + c];
                    acc.re += f * prod.re; acc.im += f * prod.im;
                }
            }
        }
        cplx term = cmul(acc, cmul(pj, pk));
        V.re += term.re; V.im += term.im;
    }
    out[0] = V.re; out[1] = V.im;
}

/* V4^{s1 s2}(lam; lam1, lam2, lam3), q3 = q + s1 q1 + s2 q2.  SURVEY.md §8(c) step 6:
 *   V4 = sum_c sum_abgd Phi_c^{abgd} e~_lam(i,a) . E^{s1}_lam1(j,b) . E^{s2}_lam2(k,g) . conj(e~_lam3(l,d)) phi(-q3,Rl)
 *   E^{+}_mu(x,b) = e~_mu(x,b) phi(q_mu,R_x),   E^{-} = conj(E^{+})                                                      */
void orc_v4(const orc_setup *s, int lam, int lam1, int lam2, int lam3, int s1, int s2, double out[2]) {
    int nb = 3 * s->natoms;
    int q1 = lam1 / nb, q2 = lam2 / nb, q3 = lam3 / nb;
    cplx V = { 0.0, 0.0 };
    for (int64_t c = 0; c < s->n4; c++) {
        int i = s->atoms4[4 * c], j = s->atoms4[4 * c + 1], k = s->atoms4[4 * c + 2], l = s->atoms4[4 * c + 3];
        const int32_t *Rj = s->cells4 + 9 * c, *Rk = s->cells4 + 9 * c + 3, *Rl = s->cells4 + 9 * c + 6;
        cplx pj = bloch_phase(s, q1, s1, Rj), pk = bloch_phase(s, q2, s2, Rk), pl = bloch_phase(s, q3, -1, Rl);
        cplx acc = { 0.0, 0.0 };
        for (int a = 0; a < 3; a++) {
            cplx ea = etilde(s, lam, i, a);
            for (int b = 0; b < 3; b++) {
                cplx eb = etilde(s, lam1, j, b);
                if (s1 < 0) eb = cconj(eb);
                cplx eab = cmul(ea, eb);
                for (int g = 0; g < 3; g++) {
                    cplx eg = etilde(s, lam2, k, g);
                    if (s2 < 0) eg = cconj(eg);
                    cplx eabg = cmul(eab, eg);
                    for (int d = 0; d < 3; d++) {
                        cplx ed = cconj(etilde(s, lam3, l, d));
                        cplx prod = cmul(eabg, ed);
                        double f = s->phi4[81 * c + 27 * a + 9 * b + 3 * g + d];
                        acc.re += f * prod.re; acc.im += f * prod.im;
                    }
                }
            }
        }
        cplx term = cmul(acc, cmul(cmul(pj, pk), pl));
        V.re += term.re; V.im += term.im;
    }
    out[0] = V.re; out[1] = V.im;
}

/* ---- Neumaier-compensated accumulator ---------------------------------------------------------------------------- */
typedef struct { double s, c; } ksum;
static void kadd(ksum *k, double x) {
    double t = k->s + x;
    if (fabs(k->s) >= fabs(x)) k->c += (k->s - t) + x; else k->c += (x - t) + k->s;
    k->s = t;
}
static double kval(const ksum *k) { return k->s + k->c; }

/* ---- three-phonon rates: Algorithm 1 for channels + (index 0) and - (index 1) ------------------- */
/* gamma, wp: nt*2 doubles; counts: nt*2 int64.  weights_only != 0 sets |V|^2 = 1 (pins the non-V part, A11).          */
int orc_rates3(const orc_setup *s, const int32_t *targets, int64_t nt, double *gamma, double *wp, int64_t *counts,
               int weights_only) {
    const int nb = 3 * s->natoms, N = nq_of(s);
    double B[9]; orc_recip(s->lattvec, s->mesh, B);
    const double C3 = const_c3();
    /* per (target, q') partials, combined in q' order afterwards: independent of the thread count */
    ksum *pg = calloc((size_t)nt * N * 2, sizeof(ksum)), *pw = calloc((size_t)nt * N * 2, sizeof(ksum));
    int64_t *pc = calloc((size_t)nt * N * 2, sizeof(int64_t));
    if (!pg || !pw || !pc) { free(pg); free(pw); free(pc); return -1; }
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t work = 0; work < nt * (int64_t)N; work++) {
        int64_t it = work / N; int q1 = (int)(work % N);
        int lam = targets[it], q = lam / nb;
        double w = s->omega[lam];
        if (w == 0.0) continue;                                             /* item 8 */
        for (int ch = 0; ch < 2; ch++) {
            int sign = ch == 0 ? +1 : -1;
            int q2 = q_combine(s, q, sign, q1, 0, 0);
            ksum *G = &pg[(it * N + q1) * 2 + ch], *W = &pw[(it * N + q1) * 2 + ch];
            for (int j1 = 0; j1 < nb; j1++) {
                int lam1 = q1 * nb + j1; double w1 = s->omega[lam1];
                if (w1 == 0.0) continue;
                double f1 = orc_be(w1, s->T);
                for (int j2 = 0; j2 < nb; j2++) {
                    int lam2 = q2 * nb + j2; double w2 = s->omega[lam2];
                    if (w2 == 0.0) continue;
                    double sigma = sigma_of(s, B, s->vg + 3 * (size_t)lam1, s->vg + 3 * (size_t)lam2);
                    double delta = sign > 0 ? (w + w1) - w2 : (w - w1) - w2;
                    if (!allowed(s, delta, sigma)) continue;
                    double f2 = orc_be(w2, s->T);
                    double occ = sign > 0 ? (f1 - f2) : (f1 + f2 + 1.0);
                    double WP = occ * gauss(delta, sigma) / (w * w1 * w2);
                    double v2 = 1.0;
                    if (!weights_only) { double V[2]; orc_v3(s, lam, lam1, lam2, sign, V); v2 = V[0] * V[0] + V[1] * V[1]; }
                    kadd(W, WP);
                    kadd(G, WP * v2);
                    pc[(it * N + q1) * 2 + ch]++;
                }
            }
        }
    }
    for (int64_t it = 0; it < nt; it++)
        for (int ch = 0; ch < 2; ch++) {
            ksum G = { 0, 0 }, W = { 0, 0 }; int64_t cnt = 0;
            for (int q1 = 0; q1 < N; q1++) {
                size_t o = (size_t)(it * N + q1) * 2 + ch;
                kadd(&G, pg[o].s); kadd(&G, pg[o].c); kadd(&W, pw[o].s); kadd(&W, pw[o].c); cnt += pc[o];
            }
            double sym = ch == 0 ? 1.0 : 0.5;                                /* item 4 */
            gamma[it * 2 + ch] = C3 / (double)N * sym * kval(&G);
            if (wp) wp[it * 2 + ch] = sym * kval(&W) / (double)N;
            counts[it * 2 + ch] = cnt;
        }
    free(pg); free(pw); free(pc);
    return 0;
}

/* process list of one target and channel, as (lam1, lam2) pairs in loop order; returns the count (may exceed cap) */
int64_t orc_list3(const orc_setup *s, int32_t lam, int ch, int32_t *pairs, int64_t cap) {
    const int nb = 3 * s->natoms, N = nq_of(s);
    double B[9]; orc_recip(s->lattvec, s->mesh, B);
    int q = lam / nb, sign = ch == 0 ? +1 : -1; double w = s->omega[lam];
    int64_t n = 0;
    if (w == 0.0) return 0;
    for (int q1 = 0; q1 < N; q1++) {
        int q2 = q_combine(s, q, sign, q1, 0, 0);
        for (int j1 = 0; j1 < nb; j1++) {
            int lam1 = q1 * nb + j1; double w1 = s->omega[lam1]; if (w1 == 0.0) continue;
            for (int j2 = 0; j2 < nb; j2++) {
                int lam2 = q2 * nb + j2; double w2 = s->omega[lam2]; if (w2 == 0.0) continue;
                double sigma = sigma_of(s, B, s->vg + 3 * (size_t)lam1, s->vg + 3 * (size_t)lam2);
                double delta = sign > 0 ? (w + w1) - w2 : (w - w1) - w2;
                if (!allowed(s, delta, sigma)) continue;
                if (n < cap) { pairs[2 * n] = lam1; pairs[2 * n + 1] = lam2; }
                n++;
            }
        }
    }
    return n;
}

/* ---- four-phonon rates: the same loop nest one level deeper, channels ++ (0), +- (1), -- (2) ----------------------- */
/* Only q' in [qp_begin, qp_end) is summed (the full definition is qp_begin=0, qp_end=N); the prefactor is always
 * C4/N^2, so partial sums over disjoint q' ranges add up to the full rate.                                            */
int orc_rates4(const orc_setup *s, const int32_t *targets, int64_t nt, int32_t qp_begin, int32_t qp_end, double *gamma,
               double *wp, int64_t *counts, int weights_only) {
    const int nb = 3 * s->natoms, N = nq_of(s);
    double B[9]; orc_recip(s->lattvec, s->mesh, B);
    const double C4 = const_c4();
    static const int S1[3] = { +1, +1, -1 }, S2[3] = { +1, -1, -1 };
    const int nqp = qp_end - qp_begin;
    if (qp_begin < 0 || qp_end > N) return -2;                               /* q' range outside the mesh */
    if (nqp <= 0) { for (int64_t i = 0; i < nt * 3; i++) { gamma[i] = 0; if (wp) wp[i] = 0; counts[i] = 0; } return 0; }
    ksum *pg = calloc((size_t)nt * nqp * 3, sizeof(ksum)), *pw = calloc((size_t)nt * nqp * 3, sizeof(ksum));
    int64_t *pc = calloc((size_t)nt * nqp * 3, sizeof(int64_t));
    if (!pg || !pw || !pc) { free(pg); free(pw); free(pc); return -1; }
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t work = 0; work < nt * (int64_t)nqp; work++) {
        int64_t it = work / nqp; int q1 = qp_begin + (int)(work % nqp);
        int lam = targets[it], q = lam / nb;
        double w = s->omega[lam];
        if (w == 0.0) continue;
        double f0 = orc_be(w, s->T);
        for (int ch = 0; ch < 3; ch++) {
            int s1 = S1[ch], s2 = S2[ch];
            size_t o = ((size_t)it * nqp + (q1 - qp_begin)) * 3 + ch;
            for (int j1 = 0; j1 < nb; j1++) {
                int lam1 = q1 * nb + j1; double w1 = s->omega[lam1];
                if (w1 == 0.0) continue;
                double f1 = orc_be(w1, s->T);
                for (int q2 = 0; q2 < N; q2++) {
                    int q3 = q_combine(s, q, s1, q1, s2, q2);                /* step 1 */
                    for (int j2 = 0; j2 < nb; j2++) {
                        int lam2 = q2 * nb + j2; double w2 = s->omega[lam2];
                        if (w2 == 0.0) continue;
                        double f2 = orc_be(w2, s->T);
                        for (int j3 = 0; j3 < nb; j3++) {
                            int lam3 = q3 * nb + j3; double w3 = s->omega[lam3];
                            if (w3 == 0.0) continue;
                            double sigma = sigma_of(s, B, s->vg + 3 * (size_t)lam2, s->vg + 3 * (size_t)lam3);   /* item 2 */
                            double delta = ch == 0 ? ((w + w1) + w2) - w3 : ch == 1 ? ((w + w1) - w2) - w3 : ((w - w1) - w2) - w3;
                            if (!allowed(s, delta, sigma)) continue;
                            double f3 = orc_be(w3, s->T);
                            double occ = ch == 0 ? (1.0 + f1) * (1.0 + f2) * f3 / f0
                                       : ch == 1 ? (1.0 + f1) * f2 * f3 / f0
                                                 : f1 * f2 * f3 / f0;       /* item 5 */
                            double WP = occ * gauss(delta, sigma) / (w * w1 * w2 * w3);
                            double v2 = 1.0;
                            if (!weights_only) { double V[2]; orc_v4(s, lam, lam1, lam2, lam3, s1, s2, V); v2 = V[0] * V[0] + V[1] * V[1]; }
                            kadd(&pw[o], WP);
                            kadd(&pg[o], WP * v2);
                            pc[o]++;
                        }
                    }
                }
            }
        }
    }
    for (int64_t it = 0; it < nt; it++)
        for (int ch = 0; ch < 3; ch++) {
            ksum G = { 0, 0 }, W = { 0, 0 }; int64_t cnt = 0;
            for (int iq = 0; iq < nqp; iq++) {
                size_t o = ((size_t)it * nqp + iq) * 3 + ch;
                kadd(&G, pg[o].s); kadd(&G, pg[o].c); kadd(&W, pw[o].s); kadd(&W, pw[o].c); cnt += pc[o];
            }
            double sym = ch == 2 ? 1.0 / 6.0 : 0.5;
            double nn = (double)N * (double)N;
            gamma[it * 3 + ch] = C4 / nn * sym * kval(&G);
            if (wp) wp[it * 3 + ch] = sym * kval(&W) / nn;
            counts[it * 3 + ch] = cnt;
        }
    free(pg); free(pw); free(pc);
    return 0;
}

/* process list of one target and channel over q' in [qp_begin, qp_end), as (lam1, lam2, lam3) triples in loop order:
 * the 4ph analogue of orc_list3 -- the loop nest, the sigma legs (v'' - v''') and the filter
 * are those of orc_rates4.  Returns the count (may exceed cap), -2 for a q' range outside the mesh.                   */
int64_t orc_list4(const orc_setup *s, int32_t lam, int ch, int32_t qp_begin, int32_t qp_end, int32_t *triples, int64_t cap) {
    const int nb = 3 * s->natoms, N = nq_of(s);
    double B[9]; orc_recip(s->lattvec, s->mesh, B);
    static const int S1[3] = { +1, +1, -1 }, S2[3] = { +1, -1, -1 };
    if (qp_begin < 0 || qp_end > N) return -2;
    int q = lam / nb, s1 = S1[ch], s2 = S2[ch]; double w = s->omega[lam];
    int64_t n = 0;
    if (w == 0.0) return 0;
    for (int q1 = qp_begin; q1 < qp_end; q1++)
        for (int j1 = 0; j1 < nb; j1++) {
            int lam1 = q1 * nb + j1; double w1 = s->omega[lam1]; if (w1 == 0.0) continue;
            for (int q2 = 0; q2 < N; q2++) {
                int q3 = q_combine(s, q, s1, q1, s2, q2);
                for (int j2 = 0; j2 < nb; j2++) {
                    int lam2 = q2 * nb + j2; double w2 = s->omega[lam2]; if (w2 == 0.0) continue;
                    for (int j3 = 0; j3 < nb; j3++) {
                        int lam3 = q3 * nb + j3; double w3 = s->omega[lam3]; if (w3 == 0.0) continue;
                        double sigma = sigma_of(s, B, s->vg + 3 * (size_t)lam2, s->vg + 3 * (size_t)lam3);
                        double delta = ch == 0 ? ((w + w1) + w2) - w3 : ch == 1 ? ((w + w1) - w2) - w3 : ((w - w1) - w2) - w3;
                        if (!allowed(s, delta, sigma)) continue;
                        if (n < cap) { triples[3 * n] = lam1; triples[3 * n + 1] = lam2; triples[3 * n + 2] = lam3; }
                        n++;
                    }
                }
            }
        }
    return n;
}

/* ---- step 8: RTA thermal conductivity ---------------------------------------------------------------------------- */
/* kappa^{ab} = C_kappa/(T^2 Omega N) sum_lam f(f+1) omega^2 v^a v^b / Gamma_lam, skipping zero modes and Gamma <= 0     */
void orc_kappa(const orc_setup *s, const double *gamma_total, double kappa[9]) {
    const int nb = 3 * s->natoms, N = nq_of(s);
    const double *a1 = s->lattvec, *a2 = s->lattvec + 3, *a3 = s->lattvec + 6;
    double vol = fabs(a1[0] * (a2[1] * a3[2] - a2[2] * a3[1]) + a1[1] * (a2[2] * a3[0] - a2[0] * a3[2]) + a1[2] * (a2[0] * a3[1] - a2[1] * a3[0]));
    ksum acc[9]; memset(acc, 0, sizeof(acc));
    for (int lam = 0; lam < N * nb; lam++) {
        double w = s->omega[lam], g = gamma_total[lam];
        if (w == 0.0 || !(g > 0.0)) continue;
        double f = orc_be(w, s->T);
        double pre = f * (f + 1.0) * w * w / g;
        const double *v = s->vg + 3 * (size_t)lam;
        for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) kadd(&acc[3 * a + b], pre * v[a] * v[b]);
    }
    double c = const_ckappa() / (s->T * s->T * vol * (double)N);
    for (int x = 0; x < 9; x++) kappa[x] = c * kval(&acc[x]);
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
