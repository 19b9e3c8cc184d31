// kernels.cu -- sm_100a kernels for the batched source term and analytical Jacobian.
//
// One CTA evaluates S thermochemical states per iteration of a persistent grid-stride loop; the S
// states are interleaved in shared memory (element i of a region for state q at (R + i) * S + q), so
// whatever does not depend on the state -- decoding a reaction, a gather entry, a column constant --
// is done once and applied to the S states with one vector load.  All work is assigned to the warps
// statically (item i of a phase goes to warp i mod NW; the items were sorted by cost at create
// time).  Per iteration:
//   P0    mixture (Eqs. 3-5) and species, warp <-> state: [X_k], c_pk, mixture c_p, d c_p / dT
//         (Eqs. 9-13, 54-55)
//   P1    reactions, lane <-> reaction, groups of 32: k_f, k_r (K_c from the per-reaction polynomial
//         of device_mech.h `th_data`), R_f, R_r, c_i and the reusable per-reaction products of
//         Section 4.1 into E: q_i, Theta_dT,i, a_i (the coefficient of d_j), the
//         sparse terms s'_ij, the enthalpy H_i.  Groups made only of plain elementary reactions take
//         a branch-free path that evaluates two states at a time.
//   AUX   fixed-order gathers over E: wdot_k (Eq. 14), alpha_r, gamma_r of Eq. 112, the T column
//         (Eq. 111), the column sums of the energy row (Eq. 113), the sums of long cell lists.
//         2^rshift neighbouring lanes share one sum (butterfly at the end).
//   FIX   the energy row, Eq. 113, per column into region Z
//   MAIN  the Jacobian as a flat column-major array: lane <-> output element.  Each element
//         gathers its short list from E and is stored straight from the register:
//           J(r, c) = alpha_r d_j + (W_k / W_j) sum_i nu_ki s'_ij - gamma_r        (r = k+1, c = j+1)
//         which is Eq. 112 with the per-reaction terms of Eqs. 118-127 regrouped by what they
//         multiply.  Row 0 and column 0 are lists of one finished entry
//         (Z_c, the T column), so the pass has no special cases.  A warp stores 256 contiguous bytes.
// There are no atomics and no Jacobian tile: every sum has an order fixed at pyjac_mech_create.
#include <cuda_runtime.h>

#include <cstdio>

#include "device_mech.h"
#include "kernels.h"

namespace pyjac {

namespace {

// -DPYJAC_PROF: CTA 0 prints the cycles warp 0 spends in each phase of its fourth iteration
#ifdef PYJAC_PROF
#define PROF_MARK(i) do { if (blockIdx.x == 0 && (tid & 31) == 0 && blk == blockIdx.x + 3 * (long long)gridDim.x) prof_t[i] = clock64(); } while (0)
#else
#define PROF_MARK(i) do { } while (0)
#endif

constexpr double kLn10 = 2.302585092994045684;
constexpr double kInvLn10 = 0.434294481903251828;

__device__ __forceinline__ double entry_coef(uint32_t e) { return __hiloint2double((int)(e & 0xFFFF0000u), 0); }

// exp(x) for the rate coefficients: Cody-Waite reduction by ln 2, degree-13 Taylor polynomial on
// |r| <= ln2/2 (truncation 4e-18), scaling by 2^n in two steps so that results underflow to 0
// and overflow to +inf like exp().  About 1 ulp; no special-case branches.  The coefficients sit
// in constant memory so that each Horner step is one DFMA with a constant-bank operand.
__constant__ double c_exp[14] = {
    1.6059043836821613e-10,  // 1/13!
    2.08767569878681e-09,    // 1/12!
    2.505210838544172e-08,   // 1/11!
    2.755731922398589e-07,   // 1/10!
    2.7557319223985893e-06,  // 1/9!
    2.48015873015873e-05,    // 1/8!
    1.984126984126984e-04,   // 1/7!
    1.388888888888889e-03,   // 1/6!
    8.333333333333333e-03,   // 1/5!
    4.1666666666666664e-02,  // 1/4!
    1.6666666666666666e-01,  // 1/3!
    0.5, 1.0, 1.0};
__constant__ double c_exp_red[4] = {1.4426950408889634074, 6755399441055744.0, -6.93147180369123816490e-01,
                                    -1.90821492927058770002e-10};

__device__ __forceinline__ double exp_rate(double x)
{
    const double s = fma(x, c_exp_red[0], c_exp_red[1]);
    int n = __double2loint(s);
    const double nd = s - c_exp_red[1];
    double r = fma(nd, c_exp_red[2], x);
    r = fma(nd, c_exp_red[3], r);
    double p = c_exp[0];
#pragma unroll
    for (int i = 1; i < 14; ++i) p = fma(p, r, c_exp[i]);
    n = max(-1080, min(1030, n));
    const int n1 = n >> 1, n2 = n - n1;
    p *= __hiloint2double((n1 + 1023) << 20, 0);
    return p * __hiloint2double((n2 + 1023) << 20, 0);
}

// x^nu and nu x^(nu-1) for nu in 0..3 by repeated multiplication (Eqs. 18-19, 120-121; never a
// division by a concentration)
__device__ __forceinline__ void int_pow(double x, int nu, double &p, double &pm)
{
    const double x2 = x * x;
    p = nu == 0 ? 1.0 : nu == 1 ? x : nu == 2 ? x2 : x2 * x;
    pm = nu == 0 ? 0.0 : nu == 1 ? 1.0 : nu == 2 ? 2.0 * x : 3.0 * x2;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

// the S interleaved values of one element: one vector load / store
template <int S>
__device__ __forceinline__ void ldv(const double *p, double (&v)[S])
{
    if (S == 2) {
        const double2 t = *reinterpret_cast<const double2 *>(p);
        v[0] = t.x; v[1] = t.y;
    } else if (S == 4) {
        const double2 t = *reinterpret_cast<const double2 *>(p), u = *reinterpret_cast<const double2 *>(p + 2);
        v[0] = t.x; v[1] = t.y; v[2] = u.x; v[3] = u.y;
    } else {
#pragma unroll
        for (int q = 0; q < S; ++q) v[q] = p[q];
    }
}
template <int S>
__device__ __forceinline__ void stv(double *p, const double (&v)[S])
{
    if (S == 2) {
        *reinterpret_cast<double2 *>(p) = make_double2(v[0], v[1]);
    } else if (S == 4) {
        *reinterpret_cast<double2 *>(p) = make_double2(v[0], v[1]);
        *reinterpret_cast<double2 *>(p + 2) = make_double2(v[2], v[3]);
    } else {
#pragma unroll
        for (int q = 0; q < S; ++q) p[q] = v[q];
    }
}

// ---- P1, plain path: 32 elementary reactions with at most three molecules per side (one slot per
// molecule), k_r from K_c or irreversible, one NASA breakpoint.  Two states at a time (q0, q0 + 1), no branches.
template <int LEVEL, int S>
__device__ __forceinline__ void plain_reactions(const DeviceMech &m, const SmemPlan &sp, double *E, const double *X,
                                                const double *sc, int s, int q0, const EvalOut &out, long long state0,
                                                long long n)
{
    constexpr int SP = S >= 2 ? 2 : 1;
    const int nr = m.nr;
    const uint4 sl = m.slots[s];
    const uint32_t meta = sl.w;
    const int x0 = (sl.x & 0xFFFF) * S, x1 = (sl.x >> 16) * S, x2 = (sl.y & 0xFFFF) * S,
              x3 = (sl.y >> 16) * S, x4 = (sl.z & 0xFFFF) * S, x5 = (sl.z >> 16) * S;
    const int nf = (meta & 0xF) + ((meta >> 4) & 0xF) + ((meta >> 8) & 0xF);
    const int nb = ((meta >> 12) & 0xF) + ((meta >> 16) & 0xF) + ((meta >> 20) & 0xF);
    const double snf = (double)nf, snr = (double)nb, dnu = (double)(nb - nf);
    const bool rev = meta_rev(meta) != PYJAC_IRREVERSIBLE;
    const double lnA = m.lnA[s], beta = m.beta[s], Ta = m.Ta[s];
    const double *th = m.th_soa + s;
    const double brk = th[0];
    int v0 = 0, v1 = 0, v2 = 0, v3 = 0, v4 = 0, v5 = 0;
    if (LEVEL == 2) {
        const uint4 vi = m.vidx[s];
        v0 = (vi.x & 0xFFFF) * S; v1 = (vi.x >> 16) * S; v2 = (vi.y & 0xFFFF) * S;
        v3 = (vi.y >> 16) * S; v4 = (vi.z & 0xFFFF) * S; v5 = (vi.z >> 16) * S;
    }
    const int orig = LEVEL == 0 ? m.rxn_orig[s] : 0;

    {
        double T[SP], lnT[SP], invT[SP], lnkf[SP], L[SP], sB[SP], sdB[SP], kf[SP], kr[SP];
#pragma unroll
        for (int u = 0; u < SP; ++u) {
            T[u] = sc[kT * S + q0 + u]; lnT[u] = sc[kLnT * S + q0 + u]; invT[u] = sc[kInvT * S + q0 + u];
            lnkf[u] = fma(beta, lnT[u], fma(-Ta, invT[u], lnA));                 // Eq. 21
            L[u] = fma(Ta, invT[u], beta) * invT[u];                             // Eq. 65
        }
        // sum_k nu_ki B_k (Eq. 27 over the reaction) and its T derivative (Eq. 74)
#pragma unroll
        for (int u = 0; u < SP; ++u) {
            const double *g = th + (size_t)(T[u] > brk ? 8 : 1) * nr;
            const double g0 = g[0], g1 = g[nr], g2 = g[2 * (size_t)nr], g3 = g[3 * (size_t)nr], g4 = g[4 * (size_t)nr],
                         g5 = g[5 * (size_t)nr], g6 = g[6 * (size_t)nr];
            const double t = T[u];
            sB[u] = fma(g1, lnT[u], g0) + fma(t, fma(t, fma(t, fma(t, g5, g4), g3), g2), g6 * invT[u]);
            sdB[u] = fma(fma(-g6, invT[u], g1), invT[u], g2) + t * fma(t, fma(4.0 * g5, t, 3.0 * g4), 2.0 * g3);
        }
#pragma unroll
        for (int u = 0; u < SP; ++u) kf[u] = exp_rate(lnkf[u]);
#pragma unroll
        for (int u = 0; u < SP; ++u) { kr[u] = exp_rate(lnkf[u] - sB[u]); kr[u] = rev ? kr[u] : 0.0; }   // Eqs. 23-27
#pragma unroll
        for (int u = 0; u < SP; ++u) {
            const int q = q0 + u;
            const double c0 = X[x0 + q], c1 = X[x1 + q], c2 = X[x2 + q], c3 = X[x3 + q], c4 = X[x4 + q], c5 = X[x5 + q];
            const double p01 = c0 * c1, p34 = c3 * c4;
            const double Rf = kf[u] * (p01 * c2), Rr = kr[u] * (p34 * c5);       // Eqs. 18-19
            const double R = Rf - Rr;
            E[(m.eQ + s) * S + q] = R;
            if (LEVEL >= 1) E[(m.eH + s) * S + q] = kRu * T[u] * fma(T[u], sdB[u], dnu);
            if (LEVEL == 0) {
                const long long st = state0 + q;
                if (st < n) {
                    const long long o = st * nr + orig;
                    if (out.rf) out.rf[o] = Rf;
                    if (out.rr) out.rr[o] = Rr;
                    if (out.cmod) out.cmod[o] = 1.0;
                }
            }
            if (LEVEL == 2) {
                const double W = sc[kW * S + q];
                const double iT = invT[u];
                // Theta_dT,i (Eq. 115) with Eqs. 66, 75; the d_j coefficient of Eq. 119 plus W q_i
                const double dRf = Rf * fma(-snf, iT, L[u]);
                const double dRr = Rr * (fma(-snr, iT, L[u]) - sdB[u]);
                E[(m.eTh + s) * S + q] = fma(R, iT, dRf - dRr);
                E[(m.eAr + s) * S + q] = W * (R - fma(Rf, snf, -Rr * snr));
                const double nkr = -kr[u];
                E[v0 + q] = kf[u] * (c1 * c2); E[v1 + q] = kf[u] * (c0 * c2); E[v2 + q] = kf[u] * p01;   // Eq. 120
                E[v3 + q] = nkr * (c4 * c5); E[v4 + q] = nkr * (c3 * c5); E[v5 + q] = nkr * p34;         // Eq. 121
            }
        }
    }
}

// ---- P1, general path: one reaction of any type, one state (q) ----------------------------------------
template <int LEVEL, int S>
__device__ __forceinline__ void reaction(const DeviceMech &m, const SmemPlan &sp, double *E, const double *X,
                                         const double *sc, int s, int q, const EvalOut &out, long long state0, long long n)
{
    const uint4 sl = m.slots[s];
    const uint32_t meta = sl.w;
    const int type = meta_type(meta), rev = meta_rev(meta);
    const int x0 = (sl.x & 0xFFFF) * S, x1 = (sl.x >> 16) * S, x2 = (sl.y & 0xFFFF) * S,
              x3 = (sl.y >> 16) * S, x4 = (sl.z & 0xFFFF) * S, x5 = (sl.z >> 16) * S;
    const bool unit_nu = (meta & 0x00EEEEEEu) == 0;          // every nu is 0 or 1
    const int snu_f = meta_nu(meta, 0) + meta_nu(meta, 1) + meta_nu(meta, 2);
    const int snu_r = meta_nu(meta, 3) + meta_nu(meta, 4) + meta_nu(meta, 5);
    const bool pdep = type == PYJAC_THIRD_BODY || type == PYJAC_FALLOFF || type == PYJAC_CHEM_ACTIVATED;
    const bool arrh = type != PYJAC_PLOG && type != PYJAC_CHEBYSHEV;
    double lnA = 0.0, beta = 0.0, Ta = 0.0;
    if (arrh) { lnA = m.lnA[s]; beta = m.beta[s]; Ta = m.Ta[s]; }
    const double dnu = (double)(snu_r - snu_f);
    const double *th = m.th_data + m.th_off[s];
    const int nint = (int)th[0];
    int v0 = 0, v1 = 0, v2 = 0, v3 = 0, v4 = 0, v5 = 0;
    if (LEVEL == 2) {
        const uint4 vi = m.vidx[s];
        v0 = (vi.x & 0xFFFF) * S; v1 = (vi.x >> 16) * S; v2 = (vi.y & 0xFFFF) * S;
        v3 = (vi.y >> 16) * S; v4 = (vi.z & 0xFFFF) * S; v5 = (vi.z >> 16) * S;
    }
    int eb = 0, ee = 0;
    if (pdep) { eb = m.eff_ptr[s]; ee = m.eff_ptr[s + 1]; }

    {
        const double T = sc[kT * S + q], lnT = sc[kLnT * S + q], invT = sc[kInvT * S + q];

        // ---- forward rate coefficient: ln k_f and L = d ln k_f / dT
        double lnkf, L;
        double lnk0 = 0.0, lnkinf = 0.0, lPrT = 0.0;
        if (arrh) {
            lnkinf = lnA + beta * lnT - Ta * invT;                  // Eq. 21
            lnkf = lnkinf;
            L = (beta + Ta * invT) * invT;                          // Eq. 65
            if (type == PYJAC_FALLOFF || type == PYJAC_CHEM_ACTIVATED) {
                const double b0 = m.lo_beta[s], Ta0 = m.lo_Ta[s];
                lnk0 = m.lo_lnA[s] + b0 * lnT - Ta0 * invT;
                lPrT = invT * (b0 - beta + (Ta0 - Ta) * invT - 1.0);   // Eq. 84 / P_r
                if (type == PYJAC_CHEM_ACTIVATED) { lnkf = lnk0; L = (b0 + Ta0 * invT) * invT; }
            }
        } else if (type == PYJAC_PLOG) {                            // Eqs. 37-39, 105
            const double P = sc[kP * S + q];
            const double *pk = m.pk_data + m.pk_ptr[s - m.n_pd];
            const int np = (int)pk[0];
            const double *row = pk + 1;                              // {p, ln p, ln A, beta, Ta}
            int lo = 0, hi = 0;
            double wt = 0.0;
            if (P <= row[0]) {
                lo = hi = 0;
            } else if (P >= row[5 * (np - 1)]) {
                lo = hi = np - 1;
            } else {
                int j = 0;
                while (!(row[5 * j] <= P && P < row[5 * (j + 1)])) ++j;
                lo = j; hi = j + 1;
                wt = (log(P) - row[5 * j + 1]) / (row[5 * (j + 1) + 1] - row[5 * j + 1]);
            }
            const double *a1 = row + 5 * lo, *a2 = row + 5 * hi;
            const double lnk1 = a1[2] + a1[3] * lnT - a1[4] * invT;
            const double lnk2 = a2[2] + a2[3] * lnT - a2[4] * invT;
            lnkf = lnk1 + (lnk2 - lnk1) * wt;
            L = (a1[3] + a1[4] * invT + (a2[3] - a1[3] + (a2[4] - a1[4]) * invT) * wt) * invT;
        } else {                                                    // Chebyshev, Eqs. 40-43, 110
            const double P = sc[kP * S + q];
            const double *pk = m.pk_data + m.pk_ptr[s - m.n_pd];
            const int nT = (int)pk[0], nP = (int)pk[1];
            const double iTmin = pk[2], iTmax = pk[3], lpmin = pk[4], lpmax = pk[5];
            const double *eta = pk + 6;
            const double Tr = (2.0 * invT - iTmin - iTmax) / (iTmax - iTmin);
            const double Pr = (2.0 * log10(P) - lpmin - lpmax) / (lpmax - lpmin);
            double sum = 0.0, dsum = 0.0;
            double tm2 = 1.0, tm1 = Tr;          // T_{a-2}, T_{a-1}
            double um2 = 1.0, um1 = 2.0 * Tr;    // U_{a-3}, U_{a-2}
            for (int a = 0; a < nT; ++a) {
                const double phiT = a == 0 ? 1.0 : a == 1 ? Tr : 2.0 * Tr * tm1 - tm2;
                if (a >= 2) { tm2 = tm1; tm1 = phiT; }
                double U = 0.0;                                       // U_{a-1}
                if (a >= 1) {
                    const int nn = a - 1;
                    U = nn == 0 ? 1.0 : nn == 1 ? 2.0 * Tr : 2.0 * Tr * um1 - um2;
                    if (nn >= 2) { um2 = um1; um1 = U; }
                }
                double pm2 = 1.0, pm1 = Pr, rowsum = 0.0;
                for (int b = 0; b < nP; ++b) {
                    const double phiP = b == 0 ? 1.0 : b == 1 ? Pr : 2.0 * Pr * pm1 - pm2;
                    if (b >= 2) { pm2 = pm1; pm1 = phiP; }
                    rowsum += eta[a * nP + b] * phiP;
                }
                sum += rowsum * phiT;
                dsum += rowsum * (double)a * U;
            }
            lnkf = sum * kLn10;
            L = kLn10 * invT * dsum * (-2.0 * invT) / (iTmax - iTmin);
        }
        const double kf = exp_rate(lnkf);

        // ---- sum_k nu_ki B_k (Eq. 27 over the reaction), its T derivative (Eq. 74) and the reaction
        //      enthalpy H_i = sum_k nu_ki h_k W_k = R T (T d(sum nu B)/dT + sum nu)
        int iv = 0;
        for (int b = 1; b < nint; ++b) iv += T > th[b] ? 1 : 0;
        const double *g = th + nint + 7 * iv;
        const double g1 = g[1], g2 = g[2], g3 = g[3], g4 = g[4], g5 = g[5], g6 = g[6];
        const double sB = fma(g1, lnT, g[0]) + fma(T, fma(T, fma(T, fma(T, g5, g4), g3), g2), g6 * invT);
        const double sdB = fma(fma(-g6, invT, g1), invT, g2) + T * fma(T, fma(4.0 * g5, T, 3.0 * g4), 2.0 * g3);
        const double H = kRu * T * fma(T, sdB, dnu);

        // ---- concentrations of the six slots (empty slots point at the dummy species [X] = 1)
        const double c0 = X[x0 + q], c1 = X[x1 + q], c2 = X[x2 + q], c3 = X[x3 + q], c4 = X[x4 + q], c5 = X[x5 + q];

        // ---- rates of progress (Eqs. 18-19) and the products that skip one factor (Eqs. 120-121)
        double Pf, Pr_, sk0, sk1, sk2, sk3, sk4, sk5;
        if (unit_nu) {
            const double p01 = c0 * c1, p34 = c3 * c4;
            Pf = p01 * c2; Pr_ = p34 * c5;
            sk0 = c1 * c2; sk1 = c0 * c2; sk2 = p01;
            sk3 = c4 * c5; sk4 = c3 * c5; sk5 = p34;
        } else {
            const int n0 = meta_nu(meta, 0), n1 = meta_nu(meta, 1), n2 = meta_nu(meta, 2),
                      n3 = meta_nu(meta, 3), n4 = meta_nu(meta, 4), n5 = meta_nu(meta, 5);
            double p0, p1, p2, p3, p4, p5, m0, m1, m2, m3, m4, m5;
            int_pow(c0, n0, p0, m0); int_pow(c1, n1, p1, m1); int_pow(c2, n2, p2, m2);
            int_pow(c3, n3, p3, m3); int_pow(c4, n4, p4, m4); int_pow(c5, n5, p5, m5);
            Pf = p0 * p1 * p2; Pr_ = p3 * p4 * p5;
            sk0 = m0 * p1 * p2; sk1 = p0 * m1 * p2; sk2 = p0 * p1 * m2;
            sk3 = m3 * p4 * p5; sk4 = p3 * m4 * p5; sk5 = p3 * p4 * m5;
        }

        // ---- reverse rate coefficient (Eqs. 23-27, 69, 75)
        double kr = 0.0, Lr = 0.0;
        if (rev == PYJAC_REV_FROM_KC) {
            kr = exp_rate(lnkf - sB);
            Lr = L - sdB;
        } else if (rev == PYJAC_REV_EXPLICIT) {
            const double rb = m.rev_beta[s], rTa = m.rev_Ta[s];
            kr = exp_rate(m.rev_lnA[s] + rb * lnT - rTa * invT);
            Lr = (rb + rTa * invT) * invT;
        }
        const double Rf = kf * Pf;
        const double Rr = kr * Pr_;
        const double R = Rf - Rr;

        // ---- pressure modification c_i (Eq. 20) and its derivatives (Eqs. 77-100)
        double c = 1.0, G = 0.0, fT = 0.0, b = 0.0, Xi = 0.0;
        if (pdep) {
            Xi = meta_single(meta) ? 0.0 : sc[kM * S + q];               // Eqs. 28-30
            for (int e = eb; e < ee; ++e) Xi += m.eff_eps[e] * X[(m.eff_spec[e] & 0xFFFF) * S + q];
            if (type == PYJAC_THIRD_BODY) {
                c = Xi; G = Xi; lPrT = -invT; b = R;                     // Eqs. 79-80
            } else {
                const double Pr = exp_rate(lnk0 - lnkinf) * Xi;          // Eq. 31
                const double *fp = m.fall_par + 5 * s;
                const int form = meta_form(meta);
                double F = 1.0, gF = 0.0;                                // gF = (P_r/F) dF/dP_r
                if (form == PYJAC_TROE) {                                // Eqs. 33-35, 90-96
                    const double a = fp[0];
                    const double e3 = exp_rate(-T / fp[1]), e1 = exp_rate(-T / fp[2]);
                    const double e2 = fp[4] != 0.0 ? exp_rate(-fp[3] * invT) : 0.0;
                    const double Fc = (1.0 - a) * e3 + a * e1 + e2;
                    const double dFc = -(1.0 - a) / fp[1] * e3 - a / fp[2] * e1 + fp[3] * invT * invT * e2;
                    const double lnFc = log(Fc);
                    const double lF = lnFc * kInvLn10, lP = log10(Pr);
                    const double At = lP - 0.67 * lF - 0.4;
                    const double Bt = 0.806 - 1.1762 * lF - 0.14 * lP;
                    const double AB = At / Bt, qq = 1.0 + AB * AB;
                    F = exp_rate(lnFc / qq);
                    const double k2 = lnFc * 2.0 * At / (Bt * Bt * Bt) / (kLn10 * qq * qq);
                    gF = -k2 * (Bt + 0.14 * At);
                    fT = (1.0 / (Fc * qq) - k2 * (1.1762 * At - 0.67 * Bt) / Fc) * dFc;
                } else if (form == PYJAC_SRI) {                          // Eqs. 36, 97-100
                    const double ea = exp_rate(-fp[1] * invT), ec = exp_rate(-T / fp[2]);
                    const double base = fp[0] * ea + ec, lnb = log(base);
                    const double lP = log10(Pr), Xs = 1.0 / (1.0 + lP * lP);
                    F = fp[3] * exp_rate(fp[4] * lnT + Xs * lnb);
                    gF = -Xs * Xs * 2.0 * lP * lnb * kInvLn10;
                    fT = fp[4] * invT + Xs * (fp[0] * fp[1] * invT * invT * ea - ec / fp[2]) / base;
                }
                const double i1p = 1.0 / (1.0 + Pr);
                double Theta;
                if (type == PYJAC_FALLOFF) { c = Pr * i1p * F; Theta = i1p; }       // Eqs. 82-83
                else                       { c = i1p * F;      Theta = -Pr * i1p; } // Eqs. 86-87
                G = c * (Theta + gF);
                b = R * G / Xi;
            }
        }
        const double qi = c * R;
        E[(m.eQ + s) * S + q] = qi;
        if (LEVEL >= 1) E[(m.eH + s) * S + q] = H;
        if (LEVEL == 0) {
            const long long st = state0 + q;
            if (st < n) {
                const long long o = st * m.nr + m.rxn_orig[s];
                if (out.rf) out.rf[o] = Rf;
                if (out.rr) out.rr[o] = Rr;
                if (out.cmod) out.cmod[o] = c;
            }
        }
        if (LEVEL == 2) {
            // Theta_dT,i of Eqs. 115-117: dc/dT R + c (dR/dT + R/T)
            const double dcdT = pdep ? G * lPrT + c * fT : 0.0;
            const double dRfdT = Rf * (L - (double)snu_f * invT);                 // Eq. 66
            const double dRrdT = Rr * (Lr - (double)snu_r * invT);                // Eqs. 69, 75
            E[(m.eTh + s) * S + q] = dcdT * R + c * (dRfdT - dRrdT + R * invT);
            // coefficient of d_j (Eqs. 119, 123, 127 regrouped), plus W q_i: the omega_k W d_j term of
            // Eq. 112 summed per reaction
            const double W = sc[kW * S + q];
            const double base = -W * (Rf * (double)snu_f - Rr * (double)snu_r);
            const double mix = (pdep && !meta_single(meta)) ? sc[kRho * S + q] : 0.0;
            E[(m.eAr + s) * S + q] = c * base + b * (mix - W * Xi) + W * qi;
            // sparse terms s'_ij = c (k_f S'_j - k_r S''_j) per slot, b (alpha_ij - 1) per efficiency
            const double ckf = c * kf, ckr = -c * kr;
            E[v0 + q] = ckf * sk0; E[v1 + q] = ckf * sk1; E[v2 + q] = ckf * sk2;
            E[v3 + q] = ckr * sk3; E[v4 + q] = ckr * sk4; E[v5 + q] = ckr * sk5;
            for (int e = eb; e < ee; ++e) E[(m.eff_spec[e] >> 16) * S + q] = b * m.eff_eps[e];
        }
    }
}

// next item of a phase's work queue (one shared counter per phase); plain ATOMS by lane 0
__device__ __forceinline__ int grab(int *ctr, int lane)
{
    int t = 0;
    if (lane == 0) {
        const unsigned a = (unsigned)__cvta_generic_to_shared(ctr);
        asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(t) : "r"(a) : "memory");
    }
    return __shfl_sync(0xFFFFFFFFu, t, 0);
}

// ---- P0: mixture (Eqs. 3-5) and species (Eqs. 5, 9, 12-13, 54-55) of one state, by one warp ----------
template <int LEVEL, int S>
__device__ __forceinline__ void mixture_and_species(const DeviceMech &m, double *X, double *Cp, double *sc, int q,
                                                    long long st, const double *__restrict__ Tg,
                                                    const double *__restrict__ Pg, const double *__restrict__ Yg,
                                                    long long ldy, int lane)
{
    const int ns = m.ns;
    const double *Ys = Yg + st * ldy;
    const double T = Tg[st], P = Pg[st];
    double s = 0.0;
    for (int k = lane; k < ns; k += 32) s += Ys[k] * m.inv_mw[k];
    s = warp_sum(s);
    const double W = 1.0 / s, M = P / (kRu * T), rho = M * W;
    double cp = 0.0, dcp = 0.0;
    for (int k = lane; k < ns; k += 32) {
        const double iw = m.inv_mw[k], y = Ys[k];
        X[k * S + q] = rho * (y * iw);
        if (LEVEL >= 1) {
            const double *a = m.nasa + (T <= m.t_mid[k] ? 0 : (size_t)5 * ns) + k;
            const double a0 = a[0], a1 = a[ns], a2 = a[2 * (size_t)ns], a3 = a[3 * (size_t)ns], a4 = a[4 * (size_t)ns];
            const double cpk = kRu * (a0 + T * (a1 + T * (a2 + T * (a3 + a4 * T)))) * iw;
            Cp[k * S + q] = cpk;
            cp += y * cpk;
            if (LEVEL == 2) dcp += y * (kRu * iw * (a1 + T * (2.0 * a2 + T * (3.0 * a3 + 4.0 * a4 * T))));
        }
    }
    if (LEVEL >= 1) { cp = warp_sum(cp); dcp = warp_sum(dcp); }
    if (lane == 0) {
        sc[kT * S + q] = T; sc[kLnT * S + q] = log(T); sc[kInvT * S + q] = 1.0 / T; sc[kP * S + q] = P;
        sc[kM * S + q] = M; sc[kW * S + q] = W; sc[kRho * S + q] = rho; sc[kIrho * S + q] = 1.0 / rho;
        sc[kCpMix * S + q] = cp; sc[kDcpDT * S + q] = dcp;
    }
}

// ---- the kernel ------------------------------------------------------------------------------------
// Shared memory: S interleaved state blocks of sp.total doubles, then the state-independent column
// and row constants.  The mixture block (X, Cp, scalars) is double-buffered: P0 of the NEXT batch is
// an item of this batch's P1 queue.
template <int LEVEL, int NT, int S, int MB>
__global__ void __launch_bounds__(NT, MB)
    eval_kernel(const DeviceMech m, const SmemPlan sp, long long n, const double *__restrict__ Tg,
                const double *__restrict__ Pg, const double *__restrict__ Yg, long long ldy, const EvalOut out)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ int ctr[2];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = NT / 32;
    constexpr int SP = S >= 2 ? 2 : 1;
    const int ns = m.ns, ld = m.ld, nr = m.nr;
    double *E = sm + sp.E * S;
    const double *colc = sm + (size_t)sp.total * S + sp.colc;
    double *wrow = sm + (size_t)sp.total * S + sp.wrow;
    {
        double *cw = sm + (size_t)sp.total * S + sp.colc;
        for (int i = tid; i < 4 * ld; i += NT) cw[i] = m.colc[i];
        for (int i = tid; i < ld; i += NT) wrow[i] = m.wrow[i];
    }
    if (tid < S) {   // the empty-slot dummy species, the zero slot, row 0 of alpha / gamma
        sm[(sp.P0 + sp.oX + ns) * S + tid] = 1.0;
        sm[(sp.P0 + sp.p0size + sp.oX + ns) * S + tid] = 1.0;
        E[m.eZero * S + tid] = 0.0;
        E[m.eAlpha * S + tid] = 0.0;
        E[m.eGamma * S + tid] = 0.0;
        if (nr == 0) { E[m.eS1 * S + tid] = 0.0; E[m.eA0 * S + tid] = 0.0; E[m.eS4 * S + tid] = 0.0; }
    }
    if (tid == 0) ctr[0] = 0;
    const long long nblk = (n + S - 1) / S;
    // work items of P1: the general groups one state at a time (most expensive first), P0 of the next
    // batch (one state each), then the plain groups SP states at a time
    const int n_gen = m.n_rchunk - m.n_plain;
    const int i_p0 = n_gen * S, i_plain = i_p0 + S;
    const int n_p1 = i_plain + m.n_plain * (S / SP);
    if (warp < S && (long long)blockIdx.x < nblk) {
        double *P0 = sm + sp.P0 * S;
        mixture_and_species<LEVEL, S>(m, P0 + sp.oX * S, P0 + sp.oCp * S, P0 + sp.oScal * S, warp,
                                      min((long long)blockIdx.x * S + warp, n - 1), Tg, Pg, Yg, ldy, lane);
    }
    int par = 0;
    for (long long blk = blockIdx.x; blk < nblk; blk += gridDim.x, par ^= 1) {
        const long long state0 = blk * S;
        double *P0 = sm + (sp.P0 + par * sp.p0size) * S, *P0n = sm + (sp.P0 + (par ^ 1) * sp.p0size) * S;
        const double *X = P0 + sp.oX * S, *Cp = P0 + sp.oCp * S, *sc = P0 + sp.oScal * S;
#ifdef PYJAC_PROF
        long long prof_t[12];
#endif
        PROF_MARK(0);
        __syncthreads();      // every warp has left the previous MAIN pass (and the first P0 is done)
        PROF_MARK(1);
        // ---- P1: reactions (+ the mixture of the next batch)
        for (int it = grab(&ctr[0], lane); it < n_p1; it = grab(&ctr[0], lane)) {
            if (it < i_p0) {
                const int c = it / S, q = it - c * S;
                reaction<LEVEL, S>(m, sp, E, X, sc, min(c * 32 + lane, nr - 1), q, out, state0, n);
            } else if (it < i_plain) {
                const int q = it - i_p0;
                if (blk + gridDim.x < nblk)
                    mixture_and_species<LEVEL, S>(m, P0n + sp.oX * S, P0n + sp.oCp * S, P0n + sp.oScal * S, q,
                                                  min((blk + gridDim.x) * S + q, n - 1), Tg, Pg, Yg, ldy, lane);
            } else {
                const int j = it - i_plain;
                const int c = n_gen + j / (S / SP), q0 = (j % (S / SP)) * SP;
                plain_reactions<LEVEL, S>(m, sp, E, X, sc, min(c * 32 + lane, nr - 1), q0, out, state0, n);
            }
        }
        PROF_MARK(2);
        __syncthreads();
        if (tid == 0) ctr[0] = 0;
        PROF_MARK(3);
        // ---- AUX gathers: chunk i of the list goes to warp i mod NW; the entries of a warp's next
        // chunk are fetched before the current one is summed
        {
            const int nch = LEVEL == 2 ? m.n_achunk : m.n_achunk01;
            const uint4 hz = make_uint4(0u, 0u, 0u, 0u);
            int t0 = warp;
            uint4 h0 = t0 < nch ? m.achunk[t0] : hz, h1 = t0 + NW < nch ? m.achunk[t0 + NW] : hz;
            const uint4 *ap = reinterpret_cast<const uint4 *>(m.a_ent);
            uint4 ea = hz, eb = hz;
            if (h0.y > 0 && (h0.z & 0xFF) != kAuxR3) { ea = ap[h0.x / 4 + lane * 2]; if (h0.y > 4) eb = ap[h0.x / 4 + lane * 2 + 1]; }
            for (; t0 < nch; t0 += NW) {
                const uint4 h2 = t0 + 2 * NW < nch ? m.achunk[t0 + 2 * NW] : hz;
                uint4 na = hz, nb = hz;
                if (h1.y > 0 && (h1.z & 0xFF) != kAuxR3) { na = ap[h1.x / 4 + lane * 2]; if (h1.y > 4) nb = ap[h1.x / 4 + lane * 2 + 1]; }
                // ---- chunk t0
                const uint4 ch = h0;
                const uint32_t kind = ch.z & 0xFF;
                const int rshift = (ch.z >> 8) & 0xFF, width = 1 << rshift;
                const bool head = (lane & (width - 1)) == 0;
                const uint32_t task = ch.w + (lane >> rshift);
                const uint32_t e0[8] = {ea.x, ea.y, ea.z, ea.w, eb.x, eb.y, eb.z, eb.w};
                if (kind == kAuxT3 || kind == kAuxR3) {
                    constexpr int NA = LEVEL == 2 ? 3 : 1;
                    constexpr int iA = NA > 1 ? 1 : 0, iT = NA > 2 ? 2 : 0;
                    double acc[NA][S];
#pragma unroll
                    for (int w = 0; w < NA; ++w)
#pragma unroll
                        for (int q = 0; q < S; ++q) acc[w][q] = 0.0;
                    if (kind == kAuxT3) {
                        auto step = [&](uint32_t e) {
                            const double cf = entry_coef(e);
                            const double *p = E + (e & 0xFFFF) * S;
#pragma unroll
                            for (int w = 0; w < NA; ++w) {
                                double a[S];
                                ldv<S>(p + (size_t)w * nr * S, a);
#pragma unroll
                                for (int q = 0; q < S; ++q) acc[w][q] = fma(cf, a[q], acc[w][q]);
                            }
                        };
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            if ((uint32_t)j < ch.y) step(e0[j]);
                        for (uint32_t t = 8; t < ch.y; ++t) step(m.a_ent[ch.x + (t >> 3) * 256 + lane * 8 + (t & 7)]);
                    } else {
                        for (int i = lane; i < nr; i += 32) {
                            double h[S];
                            ldv<S>(E + (m.eH + i) * S, h);
#pragma unroll
                            for (int w = 0; w < NA; ++w) {
                                double a[S];
                                ldv<S>(E + (m.eQ + w * nr + i) * S, a);
#pragma unroll
                                for (int q = 0; q < S; ++q) acc[w][q] = fma(h[q], a[q], acc[w][q]);
                            }
                        }
                    }
                    for (int o = 1; o < width; o <<= 1)
#pragma unroll
                        for (int w = 0; w < NA; ++w)
#pragma unroll
                            for (int q = 0; q < S; ++q) acc[w][q] += __shfl_xor_sync(0xFFFFFFFFu, acc[w][q], o);
                    if (head) {
                        if (kind == kAuxR3) {
                            stv<S>(E + m.eS1 * S, acc[0]);
                            if (LEVEL == 2) { stv<S>(E + m.eA0 * S, acc[iA]); stv<S>(E + m.eS4 * S, acc[iT]); }
                        } else {
                            const uint32_t k = m.a_out[task];
                            if (k != 0xFFFFFFFFu) {
                                stv<S>(E + (m.eWdot + k) * S, acc[0]);
                                if (LEVEL == 2) {
                                    const double wk = m.mw[k];
                                    double al[S], tc[S];
#pragma unroll
                                    for (int q = 0; q < S; ++q) {
                                        const double ir = sc[kIrho * S + q];
                                        al[q] = wk * ir * acc[iA][q];
                                        tc[q] = ir * acc[iT][q];
                                    }
                                    stv<S>(E + (m.eAlpha + k + 1) * S, al);
                                    stv<S>(E + (m.eTcol + k) * S, tc);
                                }
                            }
                        }
                    }
                } else if (LEVEL == 2) {
                    double acc[S];
#pragma unroll
                    for (int q = 0; q < S; ++q) acc[q] = 0.0;
                    if (kind == kAuxH2) {
                        auto step = [&](uint32_t e) {
                            double a[S], b[S];
                            ldv<S>(E + (e & 0xFFFF) * S, a);
                            ldv<S>(E + (e >> 16) * S, b);
#pragma unroll
                            for (int q = 0; q < S; ++q) acc[q] = fma(a[q], b[q], acc[q]);
                        };
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            if ((uint32_t)j < ch.y) step(e0[j]);
                        for (uint32_t t = 8; t < ch.y; ++t) step(m.a_ent[ch.x + (t >> 3) * 256 + lane * 8 + (t & 7)]);
                    } else {
                        auto step = [&](uint32_t e) {
                            const double cf = entry_coef(e);
                            double a[S];
                            ldv<S>(E + (e & 0xFFFF) * S, a);
#pragma unroll
                            for (int q = 0; q < S; ++q) acc[q] = fma(cf, a[q], acc[q]);
                        };
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            if ((uint32_t)j < ch.y) step(e0[j]);
                        for (uint32_t t = 8; t < ch.y; ++t) step(m.a_ent[ch.x + (t >> 3) * 256 + lane * 8 + (t & 7)]);
                    }
                    for (int o = 1; o < width; o <<= 1)
#pragma unroll
                        for (int q = 0; q < S; ++q) acc[q] += __shfl_xor_sync(0xFFFFFFFFu, acc[q], o);
                    const uint32_t slot = m.a_out[task];
                    if (head && slot != 0xFFFFFFFFu) {
                        if (kind == kAuxS1) {
                            const double cst = m.a_const[task];
#pragma unroll
                            for (int q = 0; q < S; ++q) acc[q] *= cst;
                        }
                        stv<S>(E + slot * S, acc);
                    }
                }
                h0 = h1; h1 = h2; ea = na; eb = nb;
            }
        }
        PROF_MARK(4);
        __syncthreads();
        PROF_MARK(5);
        // ---- outputs of the rates / source-term kernels (Eqs. 7-8, 14)
        if (LEVEL == 0 && out.wdot) {
            for (int k = tid; k < ns; k += NT)
#pragma unroll
                for (int q = 0; q < S; ++q)
                    if (state0 + q < n) out.wdot[(state0 + q) * ns + k] = E[(m.eWdot + k) * S + q];
        }
        if (LEVEL == 1) {
            for (int r = tid; r < ld; r += NT)
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    if (state0 + q >= n) continue;
                    const double irho = sc[kIrho * S + q];
                    const double v = r == 0 ? -E[m.eS1 * S + q] * irho / sc[kCpMix * S + q]
                                            : wrow[r] * E[(m.eWdot + r - 1) * S + q] * irho;
                    out.dydt[(state0 + q) * ld + r] = v;
                }
        }
        if (LEVEL == 2) {
            // ---- FIX: the energy row (Eq. 113).  Item 0 is J(0,0); item i >= 1 the columns 32(i-1)+1 ..
            const int nfix = 1 + (ns - 1 + 31) / 32;
            for (int it = warp; it < nfix; it += NW) {
                if (it == 0) {
                    double s3[S];       // sum_k c_pk W_k wdot_k
#pragma unroll
                    for (int q = 0; q < S; ++q) s3[q] = 0.0;
                    for (int k = lane; k < ns; k += 32) {
                        const double wk = wrow[k + 1];
                        double cp[S], wd[S];
                        ldv<S>(Cp + k * S, cp);
                        ldv<S>(E + (m.eWdot + k) * S, wd);
#pragma unroll
                        for (int q = 0; q < S; ++q) s3[q] = fma(cp[q] * wk, wd[q], s3[q]);
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                        for (int q = 0; q < S; ++q) s3[q] += __shfl_xor_sync(0xFFFFFFFFu, s3[q], o);
                    if (lane < S) {
                        const int q = lane;
                        double s = s3[0];
#pragma unroll
                        for (int u = 1; u < S; ++u) s = q == u ? s3[u] : s;
                        const double icp = 1.0 / sc[kCpMix * S + q];
                        E[m.eZ * S + q] = -icp * sc[kIrho * S + q] *
                                          (s - sc[kDcpDT * S + q] * icp * E[m.eS1 * S + q] + E[m.eS4 * S + q]);
                    }
                } else {
                    const int c = (it - 1) * 32 + lane + 1;
                    if (c < ns) {
                        const double dx = colc[4 * c];
                        const double wj = wrow[c], iwl = m.inv_mw[ns - 1];
#pragma unroll
                        for (int q = 0; q < S; ++q) {
                            const double icp = 1.0 / sc[kCpMix * S + q], irho = sc[kIrho * S + q];
                            const double a1 = irho * E[m.eS1 * S + q] * icp * icp;     // coefficient of c_pj - c_pNs
                            const double alpha0 = -(irho * icp) * E[m.eA0 * S + q];
                            const double gamma0 = -(iwl * icp) * E[(m.eG0 + ns - 1) * S + q];
                            const double dcp = Cp[(c - 1) * S + q] - Cp[(ns - 1) * S + q];
                            E[(m.eZ + c) * S + q] =
                                wj * (alpha0 * dx - gamma0 + a1 * dcp) - icp * E[(m.eG0 + c - 1) * S + q];
                        }
                    }
                }
            }
            PROF_MARK(6);
            __syncthreads();
            PROF_MARK(7);
            // ---- MAIN pass: warp <-> (slab of 32 rows, segment of columns); lane <-> row.  alpha_r,
            // gamma_r, W_r stay in registers; per column: one 16-byte load of the lane's entries (the
            // next column's is in flight), gather, Eq. 112, store (32 consecutive rows = 256 bytes).
            const long long Jstate = (long long)ld * ld;
            const int seg = m.m_seg, nseg = (ld + seg - 1) / seg;
            const int n_items = m.n_slab * nseg;
            const uint4 ez = make_uint4(0u, 0u, 0u, 0u);
            for (int it = warp; it < n_items; it += NW) {
                const int slab = it % m.n_slab, sg = it / m.n_slab;
                const int c0 = sg * seg, c1 = min(ld, c0 + seg);
                const int r = slab * 32 + lane;
                const bool rlive = r < ld;
                const int rr = rlive ? r : 0;
                const double wr = wrow[rr];
                double alpha[S], gamma[S];
                ldv<S>(E + (m.eAlpha + rr) * S, alpha);
                ldv<S>(E + (m.eGamma + rr) * S, gamma);
                const uint32_t hdrs = c0 + lane < c1 ? m.m_hdr[slab * ld + c0 + lane] : 0u;
                double *Jp = out.jac + state0 * Jstate + (long long)c0 * ld + rr;
                uint32_t h = __shfl_sync(0xFFFFFFFFu, hdrs, 0);
                uint4 e = (h & 7) ? m.m_ent[(h >> 3) * 32 + lane] : ez;
                for (int c = c0; c < c1; ++c, Jp += ld) {
                    const uint32_t hn = __shfl_sync(0xFFFFFFFFu, hdrs, (c + 1 - c0) & 31);
                    const uint4 en = (c + 1 < c1 && (hn & 7)) ? m.m_ent[(hn >> 3) * 32 + lane] : ez;
                    const uint32_t steps = h & 7;
                    double acc[S];
#pragma unroll
                    for (int q = 0; q < S; ++q) acc[q] = 0.0;
                    auto step = [&](uint32_t w) {
                        const double cf = entry_coef(w);
                        double a[S];
                        ldv<S>(E + (w & 0xFFFF) * S, a);
#pragma unroll
                        for (int q = 0; q < S; ++q) acc[q] = fma(cf, a[q], acc[q]);
                    };
                    if (steps > 0) step(e.x);
                    if (steps > 1) step(e.y);
                    if (steps > 2) step(e.z);
                    if (steps > 3) step(e.w);
                    const double2 c01 = *reinterpret_cast<const double2 *>(colc + 4 * c);
                    const double gz = colc[4 * c + 2];
                    const double wj = wr * c01.y;
#pragma unroll
                    for (int q = 0; q < S; ++q) {
                        const double v = fma(wj, acc[q], fma(alpha[q], c01.x, -(gamma[q] * gz)));
                        if (rlive && state0 + q < n) __stcs(Jp + q * Jstate, v);
                    }
                    h = hn; e = en;
                }
            }
            PROF_MARK(8);
#ifdef PYJAC_PROF
            if (blockIdx.x == 0 && (tid & 31) == 0 && blk == blockIdx.x + 3 * (long long)gridDim.x)
                printf("PROF w%d wait %lld | P1 %lld wait %lld | AUX %lld wait %lld | FIX %lld wait %lld | MAIN %lld\n",
                       warp, prof_t[1] - prof_t[0], prof_t[2] - prof_t[1], prof_t[3] - prof_t[2], prof_t[4] - prof_t[3],
                       prof_t[5] - prof_t[4], prof_t[6] - prof_t[5], prof_t[7] - prof_t[6], prof_t[8] - prof_t[7]);
#endif
        } else {
            __syncthreads();      // the outputs above read E and the scalars
        }
    }
}

template <int LEVEL, int NT, int S, int MB>
cudaError_t launch_t(const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem, long long n,
                     const double *T, const double *P, const double *Y, long long ldy, const EvalOut &out,
                     cudaStream_t stream)
{
    eval_kernel<LEVEL, NT, S, MB><<<grid, NT, smem, stream>>>(m, sp, n, T, P, Y, ldy, out);
    return cudaGetLastError();
}

}  // namespace

size_t eval_smem_bytes(const SmemPlan &sp, int S) { return ((size_t)S * sp.total + (size_t)sp.shared_total) * sizeof(double); }

// (threads, S, CTAs per SM the register budget is set for)
#define PYJAC_FOR_ALL(X) \
    X(128, 1, 4) X(128, 2, 4) X(128, 4, 4) X(256, 1, 2) X(256, 2, 2) X(256, 4, 2) X(512, 1, 1) X(512, 2, 1) X(512, 4, 1) \
    X(1024, 1, 1) X(1024, 2, 1) X(1024, 4, 1)

const void *eval_kernel_ptr(int level, int nt, int S)
{
#define PYJAC_PTR(N, SV, MB)                                                      \
    if (nt == N && S == SV)                                                       \
        return level == 0 ? (const void *)eval_kernel<0, N, SV, MB>               \
             : level == 1 ? (const void *)eval_kernel<1, N, SV, MB> : (const void *)eval_kernel<2, N, SV, MB>;
    PYJAC_FOR_ALL(PYJAC_PTR)
#undef PYJAC_PTR
    return nullptr;
}

cudaError_t launch_eval(int level, int nt, int S, const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem,
                        long long n, const double *T, const double *P, const double *Y, long long ldy,
                        const EvalOut &out, cudaStream_t stream)
{
#define PYJAC_CASE(N, SV, MB)                                                                                   \
    if (nt == N && S == SV) {                                                                                   \
        if (level == 0) return launch_t<0, N, SV, MB>(m, sp, grid, smem, n, T, P, Y, ldy, out, stream);         \
        if (level == 1) return launch_t<1, N, SV, MB>(m, sp, grid, smem, n, T, P, Y, ldy, out, stream);         \
        return launch_t<2, N, SV, MB>(m, sp, grid, smem, n, T, P, Y, ldy, out, stream);                         \
    }
    PYJAC_FOR_ALL(PYJAC_CASE)
#undef PYJAC_CASE
    return cudaErrorInvalidValue;
}

}  // namespace pyjac
