// kernels.cu -- sm_100a kernels for the batched source term and analytical Jacobian.
//
// One CTA evaluates S thermochemical states per iteration of a persistent grid-stride loop; the S
// states are interleaved in shared memory (element i of a region for state q at (R + i) * S + q), so
// whatever does not depend on the state -- decoding a reaction, a gather entry, a column constant --
// is done once and applied to the S states with one vector load.  Per iteration:
//   phase 0  mixture (Eqs. 3-5) and species: [X_k], c_pk, mixture c_p and d c_p / dT (Eqs. 9-13, 54-55)
//   phase 1  reactions, one thread per reaction, groups of 32 of one rate form taken from a queue:
//            k_f, k_r (K_c from the per-reaction polynomial of device_mech.h `th_data`), R_f, R_r, c_i
//            and the reusable per-reaction products of Section 4.1 into E:
//            q_i, Theta_dT,i, a_i (the coefficient of d_j), the sparse terms s'_ij, the enthalpy H_i
//   AUX      fixed-order gathers over E, 32 equally long lists per warp: wdot_k (Eq. 14), the row
//            vectors alpha_r, gamma_r of Eq. 112, the column sums of the energy row (Eq. 113) and the
//            sums of the long Jacobian cell lists
//   MAIN     the Jacobian as a flat column-major array: lane <-> output element.  Each element
//            gathers its short list from E and is stored straight from the register:
//              J(r, c) = alpha_r d_j + (W_k / W_j) sum_i nu_ki s'_ij - gamma_r        (r = k+1, c = j+1)
//            which is Eq. 112 with the per-reaction terms of Eqs. 118-127 regrouped by what they
//            multiply.  A warp stores 256 contiguous bytes.
// There are no atomics on data and no Jacobian tile: every sum has an order fixed at pyjac_mech_create.
#include <cuda_runtime.h>

#include "device_mech.h"
#include "kernels.h"

namespace pyjac {

namespace {

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

// next item of a phase's work queue (one shared counter per phase)
__device__ __forceinline__ int grab(int *ctr, int lane)
{
    int t = 0;
    if (lane == 0) t = atomicAdd(ctr, 1);
    return __shfl_sync(0xFFFFFFFFu, t, 0);
}

// ---- phase 1: one reaction, S states --------------------------------------------------------------
// Everything that does not depend on the state (slot decoding, Arrhenius parameters, table
// pointers) is read once; the loop over the S states of the CTA is inside.  `sm` is the CTA's
// shared memory, `sc` the scalar block of this iteration.
template <int LEVEL, int S>
__device__ __forceinline__ void reaction(const DeviceMech &m, const SmemPlan &sp, double *sm, const double *sc,
                                         int s, const EvalOut &out, long long state0, long long n)
{
    const uint4 sl = m.slots[s];
    const uint32_t meta = sl.w;
    const int type = meta_type(meta), rev = meta_rev(meta);
    const double *X = sm + sp.X * S;
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
    double *E = sm + sp.E * S;

#pragma unroll 1
    for (int q = 0; q < S; ++q) {
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
        const double sB = g[0] + g1 * lnT + T * (g2 + T * (g3 + T * (g4 + T * g5))) + g6 * invT;
        const double sdB = (g1 - g6 * invT) * invT + g2 + T * (2.0 * g3 + T * (3.0 * g4 + 4.0 * g5 * T));
        const double H = kRu * T * (T * sdB + dnu);

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
        int eb = 0, ee = 0;
        if (pdep) {
            eb = m.eff_ptr[s]; ee = m.eff_ptr[s + 1];
            Xi = meta_single(meta) ? 0.0 : sc[kM * S + q];               // Eqs. 28-30
            for (int e = eb; e < ee; ++e) Xi += m.eff_eps[e] * X[m.eff_spec[e] * S + q];
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
        E[(m.eH + s) * S + q] = H;
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
            double *V = E + m.vbase[s] * S + q;
            if (meta & 0x00000Fu) { *V = ckf * sk0; V += kVStride * S; }
            if (meta & 0x0000F0u) { *V = ckf * sk1; V += kVStride * S; }
            if (meta & 0x000F00u) { *V = ckf * sk2; V += kVStride * S; }
            if (meta & 0x00F000u) { *V = ckr * sk3; V += kVStride * S; }
            if (meta & 0x0F0000u) { *V = ckr * sk4; V += kVStride * S; }
            if (meta & 0xF00000u) { *V = ckr * sk5; V += kVStride * S; }
            if (pdep) {
                double *Ve = E + m.eff_vbase[s] * S + q;
                for (int e = eb; e < ee; ++e, Ve += kVStride * S) *Ve = b * m.eff_eps[e];
            }
        }
    }
}

// ---- the kernel ------------------------------------------------------------------------------------
// Shared memory: S interleaved state blocks of sp.total doubles, then kRedRows * S rows of 32 doubles
// of reduction scratch.  The scalar block is double-buffered by iteration parity: the mixture of the
// next batch is written while other warps still finish this batch's MAIN pass.
template <int LEVEL, int NT, int S>
__global__ void __launch_bounds__(NT, (NT <= 128 ? 4 : NT <= 256 ? 2 : 1))
    eval_kernel(const DeviceMech m, const SmemPlan sp, long long n, const double *__restrict__ Tg,
                const double *__restrict__ Pg, const double *__restrict__ Yg, long long ldy, const EvalOut out)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ int ctr[4];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = NT / 32;
    const int ns = m.ns, ld = m.ld;
    double *red = sm + (size_t)sp.total * S;
    double *E = sm + sp.E * S;
    double *X = sm + sp.X * S;
    double *Cp = sm + sp.Cp * S;
    if (tid < S) {   // the empty-slot dummy species, the zero slot and the constant scalar 1
        X[ns * S + tid] = 1.0;
        E[m.eZero * S + tid] = 0.0;
        sm[(sp.Scal + kOne) * S + tid] = 1.0;
        sm[(sp.Scal + kNScal + kOne) * S + tid] = 1.0;
    }
    const long long nblk = (n + S - 1) / S;
    int par = 0;
    for (long long blk = blockIdx.x; blk < nblk; blk += gridDim.x, par ^= 1) {
        const long long state0 = blk * S;
        double *sc = sm + (sp.Scal + par * kNScal) * S;
        // ---- phase 0a: mixture molecular weight, density (Eqs. 3-5); warp q <-> state q
        for (int q = warp; q < S; q += NW) {
            const long long st = min(state0 + q, n - 1);
            double s = 0.0;
            for (int k = lane; k < ns; k += 32) s += Yg[st * ldy + k] * m.inv_mw[k];
            s = warp_sum(s);
            if (lane == 0) {
                const double T = Tg[st], P = Pg[st];
                const double W = 1.0 / s, M = P / (kRu * T), rho = M * W;
                sc[kT * S + q] = T; sc[kLnT * S + q] = log(T); sc[kInvT * S + q] = 1.0 / T; sc[kP * S + q] = P;
                sc[kM * S + q] = M; sc[kW * S + q] = W; sc[kRho * S + q] = rho; sc[kIrho * S + q] = 1.0 / rho;
            }
        }
        __syncthreads();      // every warp has also left the previous iteration's last phase
        if (tid == 0) { ctr[0] = 0; ctr[1] = 0; ctr[2] = 0; }
        // ---- phase 0b: species (Eqs. 5, 9, 12-13, 54-55)
        {
            double part[2 * S];
#pragma unroll
            for (int i = 0; i < 2 * S; ++i) part[i] = 0.0;
            for (int k = tid; k < ns; k += NT) {
                const double iw = m.inv_mw[k], tm = m.t_mid[k];
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    const long long st = min(state0 + q, n - 1);
                    const double T = sc[kT * S + q];
                    const double y = Yg[st * ldy + k];
                    const double *a = m.nasa + (T <= tm ? 0 : (size_t)5 * ns) + k;
                    const double a0 = a[0], a1 = a[ns], a2 = a[2 * (size_t)ns], a3 = a[3 * (size_t)ns],
                                 a4 = a[4 * (size_t)ns];
                    X[k * S + q] = sc[kRho * S + q] * (y * iw);
                    if (LEVEL >= 1) {
                        const double cpk = kRu * (a0 + T * (a1 + T * (a2 + T * (a3 + a4 * T)))) * iw;
                        Cp[k * S + q] = cpk;
                        part[2 * q] += y * cpk;
                        if (LEVEL == 2) part[2 * q + 1] += y * (kRu * iw * (a1 + T * (2.0 * a2 + T * (3.0 * a3 + 4.0 * a4 * T))));
                    }
                }
            }
            if (LEVEL >= 1) {
#pragma unroll
                for (int i = 0; i < 2 * S; ++i) {
                    const double v = warp_sum(part[i]);
                    if (lane == 0) red[i * 32 + warp] = v;
                }
            }
        }
        __syncthreads();
        // ---- phase 1: reactions (the mixture heat capacity is finished on the side)
        if (LEVEL >= 1 && tid < S) {
            double cp = 0.0, dcp = 0.0;
            for (int w = 0; w < NW; ++w) { cp += red[(2 * tid) * 32 + w]; dcp += red[(2 * tid + 1) * 32 + w]; }
            const double icp = 1.0 / cp;
            sc[kCpMix * S + tid] = cp; sc[kDcpDT * S + tid] = dcp;
            sc[kNegIcp * S + tid] = -icp; sc[kNegIrhoIcp * S + tid] = -icp * sc[kIrho * S + tid];
        }
        for (int c = grab(&ctr[0], lane); c < m.n_rchunk; c = grab(&ctr[0], lane)) {
            const int s = c * 32 + lane;
            if (s < m.nr) reaction<LEVEL, S>(m, sp, sm, sc, s, out, state0, n);
        }
        __syncthreads();
        // ---- AUX gathers
        {
            const int nch = LEVEL == 2 ? m.n_achunk : m.n_achunk01;
            for (int c = grab(&ctr[1], lane); c < nch; c = grab(&ctr[1], lane)) {
                const uint4 ch = m.achunk[c];
                const uint32_t *ent = m.a_ent + ch.x + lane;
                double acc[S];
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] = 0.0;
                if (ch.z & kAuxTwoIndex) {
#pragma unroll 2
                    for (uint32_t t = 0; t < ch.y; ++t) {
                        const uint32_t e = ent[t * 32];
                        double a[S], b[S];
                        ldv<S>(E + (e & 0xFFFF) * S, a);
                        ldv<S>(E + (e >> 16) * S, b);
#pragma unroll
                        for (int q = 0; q < S; ++q) acc[q] = fma(a[q], b[q], acc[q]);
                    }
                } else {
#pragma unroll 2
                    for (uint32_t t = 0; t < ch.y; ++t) {
                        const uint32_t e = ent[t * 32];
                        const double cf = entry_coef(e);
                        double a[S];
                        ldv<S>(E + (e & 0xFFFF) * S, a);
#pragma unroll
                        for (int q = 0; q < S; ++q) acc[q] = fma(cf, a[q], acc[q]);
                    }
                }
                if (ch.z & kAuxReduce) {
#pragma unroll
                    for (int q = 0; q < S; ++q) acc[q] = warp_sum(acc[q]);
                }
                const uint32_t task = ch.w + ((ch.z & kAuxReduce) ? 0 : lane);
                const uint32_t slot = m.a_out[task];
                if (ch.z & kAuxScaled) {
                    const double cst = m.a_const[task];
                    const double *f = sc + ((ch.z >> 8) & 0xFF) * S;
#pragma unroll
                    for (int q = 0; q < S; ++q) acc[q] *= cst * f[q];
                }
                if (slot != 0xFFFFFFFFu && (!(ch.z & kAuxReduce) || lane == 0)) stv<S>(E + slot * S, acc);
            }
        }
        __syncthreads();
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
                                            : m.wrow[r] * E[(m.eWdot + r - 1) * S + q] * irho;
                    out.dydt[(state0 + q) * ld + r] = v;
                }
        }
        // ---- MAIN pass: lane <-> Jacobian element f = r + c * ld (column-major), gather + Eq. 112 / 113 + store
        if (LEVEL == 2) {
            const long long Jstate = (long long)ld * ld;
            double a1[S], irho[S];
#pragma unroll
            for (int q = 0; q < S; ++q) {
                const double icp = -sc[kNegIcp * S + q];
                irho[q] = sc[kIrho * S + q];
                a1[q] = irho[q] * E[m.eS1 * S + q] * icp * icp;    // energy row: coefficient of c_pj - c_pNs
            }
            for (int t = grab(&ctr[2], lane); t < m.n_mtask; t = grab(&ctr[2], lane)) {
                const uint4 mt = m.mtask[t];
                int r = (int)mt.z + lane, c = (int)mt.w;
                while (r >= ld) { r -= ld; ++c; }
                const bool live = c <= ns;
                const uint32_t *ent = m.m_ent + mt.x + lane;
                double acc[S];
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] = 0.0;
#pragma unroll 2
                for (uint32_t st = 0; st < mt.y; ++st) {
                    const uint32_t e = ent[st * 32];
                    const double cf = entry_coef(e);
                    double a[S];
                    ldv<S>(E + (e & 0xFFFF) * S, a);
#pragma unroll
                    for (int q = 0; q < S; ++q) acc[q] = fma(cf, a[q], acc[q]);
                }
                double j00[S];
                if (t == 0) {
                    // J(0,0) of Eq. 113: -(1/(rho c_p)) [sum_k c_pk W_k wdot_k - (dc_p/dT / c_p) S1 + S4]
#pragma unroll
                    for (int q = 0; q < S; ++q) {
                        double s3 = 0.0;
                        for (int k = lane; k < ns; k += 32) s3 += Cp[k * S + q] * m.wrow[k + 1] * E[(m.eWdot + k) * S + q];
                        s3 = warp_sum(s3);
                        const double nicp = sc[kNegIcp * S + q];
                        j00[q] = nicp * irho[q] * (s3 + sc[kDcpDT * S + q] * nicp * E[m.eS1 * S + q] + E[m.eS4 * S + q]);
                    }
                }
                const int cc_i = live ? c : 0;
                const double2 cc = m.colc[cc_i];
                const double wr = m.wrow[r];
                const double wj = wr * cc.y;
                double *Jp = out.jac + state0 * Jstate + (long long)t * 32 + lane;
                double alpha[S], gamma[S];
                ldv<S>(E + (m.eAlpha + r) * S, alpha);
                ldv<S>(E + (m.eGamma + r) * S, gamma);
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    double v = fma(alpha[q], cc.x, fma(wj, acc[q], -gamma[q]));
                    if (r == 0 && c > 0) v = fma(a1[q], Cp[(cc_i - 1) * S + q] - Cp[(ns - 1) * S + q], v);
                    if (c == 0) v = r == 0 ? (t == 0 ? j00[q] : 0.0) : wr * irho[q] * acc[q];
                    if (c == ns) v = 0.0;
                    if (live && state0 + q < n) __stcs(Jp + q * Jstate, v);
                }
            }
        }
    }
}

template <int LEVEL, int NT, int S>
cudaError_t launch_t(const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem, long long n,
                     const double *T, const double *P, const double *Y, long long ldy, const EvalOut &out,
                     cudaStream_t stream)
{
    eval_kernel<LEVEL, NT, S><<<grid, NT, smem, stream>>>(m, sp, n, T, P, Y, ldy, out);
    return cudaGetLastError();
}

}  // namespace

size_t eval_smem_bytes(const SmemPlan &sp, int S) { return ((size_t)S * sp.total + (size_t)kRedRows * S * 32) * sizeof(double); }

#define PYJAC_FOR_ALL(X) \
    X(128, 1) X(128, 2) X(128, 4) X(256, 1) X(256, 2) X(256, 4) X(512, 1) X(512, 2) X(512, 4)

const void *eval_kernel_ptr(int level, int nt, int S)
{
#define PYJAC_PTR(N, SV)                                                      \
    if (nt == N && S == SV)                                                   \
        return level == 0 ? (const void *)eval_kernel<0, N, SV>               \
             : level == 1 ? (const void *)eval_kernel<1, N, SV> : (const void *)eval_kernel<2, N, SV>;
    PYJAC_FOR_ALL(PYJAC_PTR)
#undef PYJAC_PTR
    return nullptr;
}

cudaError_t launch_eval(int level, int nt, int S, const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem,
                        long long n, const double *T, const double *P, const double *Y, long long ldy,
                        const EvalOut &out, cudaStream_t stream)
{
#define PYJAC_CASE(N, SV)                                                                                   \
    if (nt == N && S == SV) {                                                                               \
        if (level == 0) return launch_t<0, N, SV>(m, sp, grid, smem, n, T, P, Y, ldy, out, stream);         \
        if (level == 1) return launch_t<1, N, SV>(m, sp, grid, smem, n, T, P, Y, ldy, out, stream);         \
        return launch_t<2, N, SV>(m, sp, grid, smem, n, T, P, Y, ldy, out, stream);                         \
    }
    PYJAC_FOR_ALL(PYJAC_CASE)
#undef PYJAC_CASE
    return cudaErrorInvalidValue;
}

}  // namespace pyjac
