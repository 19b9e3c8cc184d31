/* oracle/oracle.c -- CPU fp64 oracle for the batched chemical-kinetics source term and its
 * analytical Jacobian (arxiv 1605.03262, "pyJac").
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the checker, not the product: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 * It shares no code with the CUDA library and never calls it.
 *
 * Two independent halves:
 *   (i)  the plain definition J = df/dPhi: the source term f (oracle_source.inc, Eqs. 1-43)
 *        instantiated for double complex and differentiated by complex step,
 *        J_ij = Im f_i(Phi + i h e_j)/h, h = 1e-30, with Y_Nsp moving through Eq. 2;
 *   (ii) the paper's analytical equations (Section 3, Eqs. 44-113) evaluated in the naive
 *        order of Algorithm 1 -- per element, summing over reactions, no reuse of the
 *        Theta products of Section 4.1.
 * GPU parity is checked against (ii); (ii) is pinned by (i) and by the invariants in
 * tests/test_oracle_pins.py.  Parity pins: every exported function is pinned there; none is
 * "parity unpinned" except value-level agreement with the paper's own runs, which print no
 * worked numeric example (PAPER.md has no table of rates or Jacobian entries).
 *
 * Output layout (readings C1-C2): dydt[n][Ns+1] = {dT/dt, dY_1/dt .. dY_Ns/dt};
 * jac[n][(Ns+1)^2], per state column-major with leading dimension Ns+1: element (r, c) at
 * r + c*(Ns+1); r, c = 0 <-> T; r, c = k <-> Y_k (k = 1..Ns).  Rows/cols 0..Ns-1 are the
 * paper's Jacobian (Eqs. 44-49); row Ns is the placeholder row of PAPER.md:570; column Ns is 0.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <tgmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#include "oracle_mech.h"

#define ORC_RU 8314.46261815324 /* J kmol^-1 K^-1 */
#define ORC_PATM 101325.0       /* Pa */

/* Eq. 43 */
static double orc_cheb_Pred(const double *lim, double P)
{
    return (2.0 * log10(P) - log10(lim[2]) - log10(lim[3])) / (log10(lim[3]) - log10(lim[2]));
}

/* ---- instantiate the source term for double and double complex ------------------------- */
#define S double
#define FN(name) name##_d
#define RE(x) (x)
#define LOG10(x) log10(x)
#include "oracle_source.inc"
#undef S
#undef FN
#undef RE
#undef LOG10

#define S double complex
#define FN(name) name##_z
#define RE(x) creal(x)
#define LOG10(x) (clog(x) / M_LN10)
#include "oracle_source.inc"
#undef S
#undef FN
#undef RE
#undef LOG10

/* ---- analytical Jacobian, naive order (Algorithm 1) ------------------- */

typedef struct {
    /* per reaction */
    double *L;      /* d ln k_f / dT: Eq. 65, Eq. 105, Eq. 110 (divided by k_f) */
    double *dRdT;   /* Eq. 69 / Eq. 75 (or Eq. 66 alone if irreversible) */
    double *dcdT;   /* Eqs. 77, 79, 82, 86 */
    double *dFdPr;  /* Eq. 94 (Troe), Eq. 98-99 form F dX/dPr ln(...) (SRI), 0 (Lindemann) */
    /* per species */
    double *cpk;    /* c_p,k   Eq. 12 */
    double *hk;     /* h_k     Eq. 12 */
    double *dcpkdT; /* Eq. 55 */
    /* species -> reactions with nu_ki != 0 (an index of "if nu != 0" in Algorithm 1) */
    const int *inc_ptr, *inc_rxn, *inc_nu;
    double *block;
} orc_jwork;

static int orc_jwork_alloc(orc_jwork *j, int ns, int nr)
{
    j->block = (double *)malloc(((size_t)4 * nr + (size_t)3 * ns) * sizeof(double));
    if (!j->block) return -1;
    double *p = j->block;
    j->L = p; p += nr; j->dRdT = p; p += nr; j->dcdT = p; p += nr; j->dFdPr = p; p += nr;
    j->cpk = p; p += ns; j->hk = p; p += ns; j->dcpkdT = p; p += ns;
    return 0;
}

/* net nu_ki = nu''_ki - nu'_ki (Eq. 15) */
static int orc_nu_net(const orc_mech *m, int i, int k)
{
    int nu = 0;
    for (int e = m->prod_ptr[i]; e < m->prod_ptr[i + 1]; ++e) if (m->prod_spec[e] == k) nu += m->prod_nu[e];
    for (int e = m->reac_ptr[i]; e < m->reac_ptr[i + 1]; ++e) if (m->reac_spec[e] == k) nu -= m->reac_nu[e];
    return nu;
}

/* species -> list of (reaction, nu_ki) with nu_ki != 0, reactions ascending */
static int orc_build_incidence(const orc_mech *m, int **ptr, int **rxn, int **nu)
{
    int ns = m->ns, nr = m->nr;
    int *cnt = (int *)calloc((size_t)ns + 1, sizeof(int));
    if (!cnt) return -1;
    for (int i = 0; i < nr; ++i)
        for (int k = 0; k < ns; ++k) {
            /* only species that appear in the reaction can have nu != 0 */
            int appears = 0;
            for (int e = m->reac_ptr[i]; e < m->reac_ptr[i + 1] && !appears; ++e) appears = m->reac_spec[e] == k;
            for (int e = m->prod_ptr[i]; e < m->prod_ptr[i + 1] && !appears; ++e) appears = m->prod_spec[e] == k;
            if (appears && orc_nu_net(m, i, k) != 0) cnt[k + 1]++;
        }
    for (int k = 0; k < ns; ++k) cnt[k + 1] += cnt[k];
    int total = cnt[ns];
    int *r = (int *)malloc((size_t)(total > 0 ? total : 1) * sizeof(int));
    int *n = (int *)malloc((size_t)(total > 0 ? total : 1) * sizeof(int));
    int *fill = (int *)calloc((size_t)ns, sizeof(int));
    if (!r || !n || !fill) return -1;
    for (int i = 0; i < nr; ++i)
        for (int k = 0; k < ns; ++k) {
            int appears = 0;
            for (int e = m->reac_ptr[i]; e < m->reac_ptr[i + 1] && !appears; ++e) appears = m->reac_spec[e] == k;
            for (int e = m->prod_ptr[i]; e < m->prod_ptr[i + 1] && !appears; ++e) appears = m->prod_spec[e] == k;
            if (!appears) continue;
            int v = orc_nu_net(m, i, k);
            if (v != 0) { r[cnt[k] + fill[k]] = i; n[cnt[k] + fill[k]] = v; fill[k]++; }
        }
    free(fill);
    *ptr = cnt; *rxn = r; *nu = n;
    return 0;
}

/* [X_l]^{nu_l - 1} prod_{n != l} [X_n]^{nu_n} over one side, entry `skip` losing one factor
 * (the product in Eqs. 64, 67, 76; never divides by a concentration) */
static double orc_prod_skip(const double *X, const int *spec, const int *nu, int b, int e, int skip)
{
    double p = 1.0;
    for (int q = b; q < e; ++q) {
        int pw = nu[q] - (q == skip ? 1 : 0);
        for (int t = 0; t < pw; ++t) p *= X[spec[q]];
    }
    return p;
}

/* Eq. 76 (with nu' / nu'' multiplying both terms, reading C11).  j is the 0-based
 * index of the species whose mass fraction is perturbed, j < ns-1. */
static double orc_dR_dYj(const orc_mech *m, const orc_work_d *w, int i, int j)
{
    const int last = m->ns - 1;
    const double dj = 1.0 / m->mw[j] - 1.0 / m->mw[last];
    double d = 0.0;
    for (int e = m->reac_ptr[i]; e < m->reac_ptr[i + 1]; ++e) {
        int l = m->reac_spec[e];
        double delta = (l == j ? 1.0 : 0.0) - (l == last ? 1.0 : 0.0);
        d += m->reac_nu[e] * (-w->Rf[i] * w->W * dj
             + delta * w->kf[i] * w->rho / m->mw[l]
               * orc_prod_skip(w->X, m->reac_spec, m->reac_nu, m->reac_ptr[i], m->reac_ptr[i + 1], e));
    }
    for (int e = m->prod_ptr[i]; e < m->prod_ptr[i + 1]; ++e) {
        int l = m->prod_spec[e];
        double delta = (l == j ? 1.0 : 0.0) - (l == last ? 1.0 : 0.0);
        d -= m->prod_nu[e] * (-w->Rr[i] * w->W * dj
             + delta * w->kr[i] * w->rho / m->mw[l]
               * orc_prod_skip(w->X, m->prod_spec, m->prod_nu, m->prod_ptr[i], m->prod_ptr[i + 1], e));
    }
    return d;
}

/* Eq. 85: dP_r/dY_j (mixture or single-species third body) */
static double orc_dPr_dYj(const orc_mech *m, const orc_work_d *w, int i, int j)
{
    const int last = m->ns - 1;
    const double dj = 1.0 / m->mw[j] - 1.0 / m->mw[last];
    const double ratio = w->k0[i] / w->kinf[i];
    int sp = m->tb_species[i];
    if (sp < 0)
        return -w->Pr[i] * w->W * dj
               + ratio * w->rho * (orc_alpha_d(m, i, j) / m->mw[j] - orc_alpha_d(m, i, last) / m->mw[last]);
    return -w->Pr[i] * w->W * dj
           + ratio * w->rho / m->mw[sp] * ((sp == j ? 1.0 : 0.0) - (sp == last ? 1.0 : 0.0));
}

/* Eqs. 78, 80-81, 83, 87 (with 89, 91, 98, 100): dc_i/dY_j */
static double orc_dc_dYj(const orc_mech *m, const orc_work_d *w, const orc_jwork *jw, int i, int j)
{
    const int last = m->ns - 1;
    const int type = m->rxn_type[i];
    const double dj = 1.0 / m->mw[j] - 1.0 / m->mw[last];
    if (type == 1) {
        int sp = m->tb_species[i];
        if (sp < 0)   /* Eq. 80 */
            return -w->W * w->c[i] * dj
                   + w->rho * (orc_alpha_d(m, i, j) / m->mw[j] - orc_alpha_d(m, i, last) / m->mw[last]);
        /* c_i = [X_m]: Eq. 62 */
        return -w->X[sp] * w->W * dj + ((sp == j ? 1.0 : 0.0) - (sp == last ? 1.0 : 0.0)) * w->rho / m->mw[sp];
    }
    if (type == 2 || type == 3) {
        double dPr = orc_dPr_dYj(m, w, i, j);
        double dF = jw->dFdPr[i] * dPr;                       /* Eqs. 89, 91, 98 + 100 */
        double Pr = w->Pr[i];
        if (type == 2) return w->c[i] * (dPr / (Pr * (1.0 + Pr)) + dF / w->F[i]);   /* Eq. 83 */
        return w->c[i] * (-dPr / (1.0 + Pr) + dF / w->F[i]);                          /* Eq. 87 */
    }
    return 0.0;   /* Eq. 78; PLOG and Chebyshev: PAPER.md:501 */
}

/* d ln k / dT for an Arrhenius set, Eq. 65 */
static double orc_arr_dlnk(const double *par, double T) { return (par[1] + par[2] / T) / T; }

static void orc_reaction_T_derivatives(const orc_mech *m, double T, double P, const orc_work_d *w,
                                       orc_jwork *jw)
{
    for (int i = 0; i < m->nr; ++i) {
        const int type = m->rxn_type[i];
        double L;
        if (type == 4) {                        /* Eq. 105 */
            int lo, hi; double wt;
            (void)orc_plog_d(m, i, T, P, &lo, &hi, &wt);
            const double *a1 = m->plog_arr + 3 * lo, *a2 = m->plog_arr + 3 * hi;
            L = (a1[1] + a1[2] / T + (a2[1] - a1[1] + (a2[2] - a1[2]) / T) * wt) / T;
        } else if (type == 5) {                 /* Eq. 110, U_n by recurrence */
            int nT = m->cheb_nT[i], nP = m->cheb_nP[i];
            const double *eta = m->cheb_eta + m->cheb_ptr[i];
            const double *lim = m->cheb_lim + 4 * i;
            double Tr = orc_cheb_Tred_d(lim, T), Pr = orc_cheb_Pred(lim, P);
            double sum = 0.0;
            double um2 = 1.0, um1 = 2.0 * Tr;     /* U_0, U_1 */
            for (int a = 1; a < nT; ++a) {        /* i-1 = a; needs U_{a-1} */
                int n = a - 1;
                double U = (n == 0) ? 1.0 : (n == 1) ? 2.0 * Tr : 2.0 * Tr * um1 - um2;
                if (n >= 2) { um2 = um1; um1 = U; }
                double pm2 = 1.0, pm1 = Pr;
                for (int b = 0; b < nP; ++b) {
                    double phiP = (b == 0) ? 1.0 : (b == 1) ? Pr : 2.0 * Pr * pm1 - pm2;
                    if (b >= 2) { pm2 = pm1; pm1 = phiP; }
                    sum += eta[a * nP + b] * a * U * phiP;
                }
            }
            L = M_LN10 / T * sum * (-2.0 / T) / (1.0 / lim[1] - 1.0 / lim[0]);
        } else if (type == 3) {
            L = orc_arr_dlnk(m->arr_lo + 3 * i, T);    /* k_f = k_0 for chem.-activated (C5) */
        } else {
            L = orc_arr_dlnk(m->arr_hi + 3 * i, T);
        }
        jw->L[i] = L;
        int snu_f = 0, snu_r = 0;
        for (int e = m->reac_ptr[i]; e < m->reac_ptr[i + 1]; ++e) snu_f += m->reac_nu[e];
        for (int e = m->prod_ptr[i]; e < m->prod_ptr[i + 1]; ++e) snu_r += m->prod_nu[e];
        double dRf = w->Rf[i] * (L - snu_f / T);                                   /* Eq. 66 */
        double dRr = 0.0;
        if (m->rev_type[i] == 1) {                                                  /* Eq. 75 */
            double sdB = 0.0;
            for (int e = m->prod_ptr[i]; e < m->prod_ptr[i + 1]; ++e) sdB += m->prod_nu[e] * w->dBdT[m->prod_spec[e]];
            for (int e = m->reac_ptr[i]; e < m->reac_ptr[i + 1]; ++e) sdB -= m->reac_nu[e] * w->dBdT[m->reac_spec[e]];
            dRr = w->Rr[i] * (L - snu_r / T - sdB);
        } else if (m->rev_type[i] == 2) {                                           /* Eq. 69 */
            dRr = w->Rr[i] * (orc_arr_dlnk(m->arr_rev + 3 * i, T) - snu_r / T);
        }
        jw->dRdT[i] = dRf - dRr;
        /* dc/dT */
        jw->dFdPr[i] = 0.0;
        if (type == 1) {
            jw->dcdT[i] = -w->c[i] / T;                                            /* Eq. 79 */
        } else if (type == 2 || type == 3) {
            const double *fp = m->falloff_par + 5 * i;
            const double *a0 = m->arr_lo + 3 * i, *ai = m->arr_hi + 3 * i;
            double Pr = w->Pr[i], F = w->F[i];
            double dPrdT = Pr / T * (a0[1] - ai[1] + (a0[2] - ai[2]) / T - 1.0);    /* Eq. 84 */
            double dFdT = 0.0;                                                      /* Eq. 88 */
            if (m->falloff_form[i] == 1) {
                double Fcent = (1 - fp[0]) * exp(-T / fp[1]) + fp[0] * exp(-T / fp[2]);
                double dFcent = -(1 - fp[0]) / fp[1] * exp(-T / fp[1]) - fp[0] / fp[2] * exp(-T / fp[2]);   /* Eq. 93 */
                if (fp[4] != 0.0) { Fcent += exp(-fp[3] / T); dFcent += fp[3] / (T * T) * exp(-fp[3] / T); }
                double lF = log10(Fcent), lP = log10(Pr);
                double A = lP - 0.67 * lF - 0.4, B = 0.806 - 1.1762 * lF - 0.14 * lP;
                double q = 1.0 + (A / B) * (A / B);
                double dA_dF = -0.67 / (Fcent * M_LN10), dB_dF = -1.1762 / (Fcent * M_LN10);   /* Eq. 95 */
                double dA_dP = 1.0 / (Pr * M_LN10), dB_dP = -0.14 / (Pr * M_LN10);             /* Eq. 96 */
                double dF_dFcent = F * (1.0 / (Fcent * q)
                                        - log(Fcent) * 2.0 * A / (B * B * B) * (dA_dF * B - A * dB_dF) / (q * q));   /* Eq. 92 */
                double dF_dPr = -F * log(Fcent) * 2.0 * A / (B * B * B) * (dA_dP * B - A * dB_dP) / (q * q);        /* Eq. 94 */
                dFdT = dF_dFcent * dFcent + dF_dPr * dPrdT;                                                         /* Eq. 90 */
                jw->dFdPr[i] = dF_dPr;
            } else if (m->falloff_form[i] == 2) {
                double lP = log10(Pr);
                double Xs = 1.0 / (1.0 + lP * lP);
                double dXdPr = -Xs * Xs * 2.0 * lP / (Pr * M_LN10);                                                 /* Eq. 99 */
                double base = fp[0] * exp(-fp[1] / T) + exp(-T / fp[2]);
                dFdT = F * (fp[4] / T
                            + Xs * (fp[0] * fp[1] / (T * T) * exp(-fp[1] / T) - exp(-T / fp[2]) / fp[2]) / base
                            + dXdPr * dPrdT * log(base));                                                           /* Eq. 97 */
                jw->dFdPr[i] = F * dXdPr * log(base);                                                               /* Eqs. 98, 100 */
            }
            if (type == 2) jw->dcdT[i] = w->c[i] * (dPrdT / (Pr * (1.0 + Pr)) + dFdT / F);   /* Eq. 82 */
            else           jw->dcdT[i] = w->c[i] * (-dPrdT / (1.0 + Pr) + dFdT / F);         /* Eq. 86 */
        } else {
            jw->dcdT[i] = 0.0;                                                      /* Eq. 77 */
        }
    }
}

static void orc_jacobian_state(const orc_mech *m, double T, double P, const double *Y,
                               orc_work_d *w, orc_jwork *jw, double *jac)
{
    const int ns = m->ns, LD = ns + 1, last = ns - 1;
    orc_source_d(m, T, P, Y, w);
    double dcpdT = 0.0;
    for (int k = 0; k < ns; ++k) {
        const double *a = (T <= m->t_mid[k]) ? m->nasa_lo + 7 * k : m->nasa_hi + 7 * k;
        jw->cpk[k] = ORC_RU * w->cpR[k] / m->mw[k];                                 /* Eq. 12 */
        jw->hk[k] = ORC_RU * w->hR[k] / m->mw[k];
        jw->dcpkdT[k] = ORC_RU / m->mw[k] * (a[1] + T * (2 * a[2] + T * (3 * a[3] + 4 * a[4] * T)));   /* Eq. 55 */
        dcpdT += Y[k] * jw->dcpkdT[k];                                              /* Eq. 54 */
    }
    orc_reaction_T_derivatives(m, T, P, w, jw);
    memset(jac, 0, (size_t)LD * LD * sizeof(double));
    /* species rows, including the placeholder row for the last species */
    for (int k = 0; k < ns; ++k) {
        const int b = jw->inc_ptr[k], e = jw->inc_ptr[k + 1];
        double s = 0.0;                                                             /* Eq. 111 */
        for (int q = b; q < e; ++q) {
            int i = jw->inc_rxn[q];
            double R = w->Rf[i] - w->Rr[i];
            s += jw->inc_nu[q] * (jw->dcdT[i] * R + w->c[i] * (jw->dRdT[i] + R / T));
        }
        jac[(k + 1) + 0 * LD] = m->mw[k] / w->rho * s;
        for (int j = 0; j < last; ++j) {                                            /* Eq. 112 */
            const double dj = 1.0 / m->mw[j] - 1.0 / m->mw[last];
            double sj = w->wdot[k] * w->W * dj;
            for (int q = b; q < e; ++q) {
                int i = jw->inc_rxn[q];
                double R = w->Rf[i] - w->Rr[i];
                sj += jw->inc_nu[q] * (orc_dc_dYj(m, w, jw, i, j) * R + w->c[i] * orc_dR_dYj(m, w, i, j));
            }
            jac[(k + 1) + (j + 1) * LD] = m->mw[k] / w->rho * sj;
        }
    }
    /* energy row, Eq. 113 (reading C10: Eq. 113, not Eqs. 46-47 as printed) */
    double sum_hg = 0.0;
    for (int k = 0; k < ns; ++k) sum_hg += jw->hk[k] * (m->mw[k] * w->wdot[k] / w->rho);
    double s11 = 0.0;
    for (int k = 0; k < ns; ++k) {
        double g = m->mw[k] * w->wdot[k] / w->rho;
        s11 += (jw->cpk[k] - jw->hk[k] / w->cp * dcpdT) * g + jw->hk[k] * jac[(k + 1) + 0 * LD];
    }
    jac[0] = -s11 / w->cp;
    for (int j = 0; j < last; ++j) {
        double sj = -(jw->cpk[j] - jw->cpk[last]) / w->cp * sum_hg;
        for (int k = 0; k < ns; ++k) sj += jw->hk[k] * jac[(k + 1) + (j + 1) * LD];
        jac[0 + (j + 1) * LD] = -sj / w->cp;
    }
}

/* complex-step Jacobian of the oracle's own source term (the plain definition) */
static void orc_jacobian_cs_state(const orc_mech *m, double T, double P, const double *Y,
                                  orc_work_z *w, double complex *Yz, double *jac)
{
    const int ns = m->ns, LD = ns + 1, last = ns - 1;
    const double h = 1e-30;
    memset(jac, 0, (size_t)LD * LD * sizeof(double));
    for (int k = 0; k < ns; ++k) Yz[k] = Y[k];
    orc_source_z(m, T + h * I, P, Yz, w);
    for (int r = 0; r < LD; ++r) jac[r] = cimag(w->dydt[r]) / h;
    for (int j = 0; j < last; ++j) {
        Yz[j] = Y[j] + h * I;
        Yz[last] = Y[last] - h * I;          /* Eq. 2 */
        orc_source_z(m, T, P, Yz, w);
        for (int r = 0; r < LD; ++r) jac[r + (j + 1) * LD] = cimag(w->dydt[r]) / h;
        Yz[j] = Y[j];
        Yz[last] = Y[last];
    }
}

/* ---- exported batch entry points ---------------------------------------------------------- */

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* any output may be NULL.  rf, rr, cmod: [n][nr]; wdot: [n][ns]; dydt: [n][ns+1] */
int orc_eval_source(const orc_mech *m, long n, const double *T, const double *P, const double *Y,
                    long ldy, double *rf, double *rr, double *cmod, double *wdot, double *dydt)
{
    int err = 0;
#pragma omp parallel
    {
        orc_work_d w;
        if (orc_work_alloc_d(&w, m->ns, m->nr) != 0) {
#pragma omp atomic write
            err = -1;
        } else {
#pragma omp for schedule(static)
            for (long s = 0; s < n; ++s) {
                orc_source_d(m, T[s], P[s], Y + s * ldy, &w);
                for (int i = 0; i < m->nr; ++i) {
                    if (rf) rf[s * m->nr + i] = w.Rf[i];
                    if (rr) rr[s * m->nr + i] = w.Rr[i];
                    if (cmod) cmod[s * m->nr + i] = w.c[i];
                }
                if (wdot) for (int k = 0; k < m->ns; ++k) wdot[s * m->ns + k] = w.wdot[k];
                if (dydt) for (int k = 0; k <= m->ns; ++k) dydt[s * (m->ns + 1) + k] = w.dydt[k];
            }
            orc_work_free_d(&w);
        }
    }
    return err;
}

/* per-reaction details for the pins: kf, kr, Kc, Pr, F, Xi, each [n][nr] (any may be NULL) */
int orc_eval_details(const orc_mech *m, long n, const double *T, const double *P, const double *Y,
                     long ldy, double *kf, double *kr, double *Kc, double *Pr, double *F, double *Xi)
{
    orc_work_d w;
    if (orc_work_alloc_d(&w, m->ns, m->nr) != 0) return -1;
    for (long s = 0; s < n; ++s) {
        orc_source_d(m, T[s], P[s], Y + s * ldy, &w);
        for (int i = 0; i < m->nr; ++i) {
            if (kf) kf[s * m->nr + i] = w.kf[i];
            if (kr) kr[s * m->nr + i] = w.kr[i];
            if (Kc) Kc[s * m->nr + i] = w.Kc[i];
            if (Pr) Pr[s * m->nr + i] = w.Pr[i];
            if (F) F[s * m->nr + i] = w.F[i];
            if (Xi) Xi[s * m->nr + i] = w.Xi[i];
        }
    }
    orc_work_free_d(&w);
    return 0;
}

/* species thermo at a complex temperature (Tre + i Tim): out[5][ns] real and imaginary parts of
 * Cp/R, H/R, S/R, B, dB/dT (Eqs. 9-11, 27, 74) */
int orc_species_thermo(const orc_mech *m, double Tre, double Tim, double *out_re, double *out_im)
{
    double complex T = Tre + Tim * I;
    for (int k = 0; k < m->ns; ++k) {
        double complex v[5];
        orc_species_thermo_z(m, k, T, &v[0], &v[1], &v[2], &v[3], &v[4]);
        for (int q = 0; q < 5; ++q) {
            out_re[q * m->ns + k] = creal(v[q]);
            if (out_im) out_im[q * m->ns + k] = cimag(v[q]);
        }
    }
    return 0;
}

static int orc_eval_jacobian_impl(const orc_mech *m, long n, const double *T, const double *P,
                                  const double *Y, long ldy, double *jac, int complex_step)
{
    int err = 0;
    int *iptr = NULL, *irxn = NULL, *inu = NULL;
    if (orc_build_incidence(m, &iptr, &irxn, &inu) != 0) return -1;
    const size_t stride = (size_t)(m->ns + 1) * (m->ns + 1);
#pragma omp parallel
    {
        orc_work_d w; orc_work_z wz; orc_jwork jw;
        double complex *Yz = (double complex *)malloc((size_t)m->ns * sizeof(double complex));
        int ok = Yz && orc_work_alloc_d(&w, m->ns, m->nr) == 0 && orc_work_alloc_z(&wz, m->ns, m->nr) == 0
                 && orc_jwork_alloc(&jw, m->ns, m->nr) == 0;
        if (!ok) {
#pragma omp atomic write
            err = -1;
        } else {
            jw.inc_ptr = iptr; jw.inc_rxn = irxn; jw.inc_nu = inu;
#pragma omp for schedule(static)
            for (long s = 0; s < n; ++s) {
                if (complex_step) orc_jacobian_cs_state(m, T[s], P[s], Y + s * ldy, &wz, Yz, jac + s * stride);
                else orc_jacobian_state(m, T[s], P[s], Y + s * ldy, &w, &jw, jac + s * stride);
            }
            orc_work_free_d(&w); orc_work_free_z(&wz); free(jw.block);
        }
        free(Yz);
    }
    free(iptr); free(irxn); free(inu);
    return err;
}

int orc_eval_jacobian(const orc_mech *m, long n, const double *T, const double *P, const double *Y,
                      long ldy, double *jac)
{
    return orc_eval_jacobian_impl(m, n, T, P, Y, ldy, jac, 0);
}

int orc_eval_jacobian_complex_step(const orc_mech *m, long n, const double *T, const double *P,
                                   const double *Y, long ldy, double *jac)
{
    return orc_eval_jacobian_impl(m, n, T, P, Y, ldy, jac, 1);
}

/* ---- first-order forward-difference Jacobian of the oracle's own source term ------------------------
 * The paper's comparison method ("a simple first-order forward difference adapted from
 * CVODE"; Tables 4-5).  The paper does not print the increment rule; DESIGN.md reading
 * C21 is followed step by step: with Phi = (T, Y_1 .. Y_{Ns-1}), N = N_s unknowns, f = dPhi/dt,
 *   w_j = 1 / (rtol |Phi_j| + atol),  D_j = max(sqrt(eps) |Phi_j|, sqrt(eps) / w_j),
 *   J(:,j) = (f(Phi + D_j e_j) - f(Phi)) / D_j,
 * a mass-fraction increment being taken from Y_Ns (Eq. 2).  Layout of orc_eval_jacobian; column N_s zero. */
int orc_eval_jacobian_fd(const orc_mech *m, long n, const double *T, const double *P, const double *Y,
                         long ldy, double rtol, double atol, double *jac)
{
    int err = 0;
    const int ns = m->ns, LD = ns + 1, last = ns - 1;
    const size_t stride = (size_t)LD * LD;
    const double eps = 2.220446049250313e-16, srur = sqrt(eps);
#pragma omp parallel
    {
        orc_work_d w;
        double *f0 = (double *)malloc((size_t)LD * sizeof(double));
        double *Yp = (double *)malloc((size_t)ns * sizeof(double));
        if (!f0 || !Yp || orc_work_alloc_d(&w, m->ns, m->nr) != 0) {
#pragma omp atomic write
            err = -1;
        } else {
#pragma omp for schedule(static)
            for (long s = 0; s < n; ++s) {
                const double *Ys = Y + s * ldy;
                double *J = jac + s * stride;
                memset(J, 0, stride * sizeof(double));
                orc_source_d(m, T[s], P[s], Ys, &w);
                for (int r = 0; r < LD; ++r) f0[r] = w.dydt[r];
                for (int j = 0; j < ns; ++j) {
                    const double phi = j == 0 ? T[s] : Ys[j - 1];
                    const double a = srur * fabs(phi), b = srur * (rtol * fabs(phi) + atol);
                    const double d = a > b ? a : b;
                    double Tp = T[s];
                    for (int k = 0; k < ns; ++k) Yp[k] = Ys[k];
                    if (j == 0) Tp = T[s] + d;
                    else { Yp[j - 1] = Ys[j - 1] + d; Yp[last] = Yp[last] - d; }
                    orc_source_d(m, Tp, P[s], Yp, &w);
                    for (int r = 0; r < LD; ++r) J[r + (size_t)j * LD] = (w.dydt[r] - f0[r]) / d;
                }
            }
            orc_work_free_d(&w);
        }
        free(f0); free(Yp);
    }
    return err;
}
