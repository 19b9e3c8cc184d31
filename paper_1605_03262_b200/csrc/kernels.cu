// kernels.cu -- sm_100a kernels for the batched source term and analytical Jacobian.
//
// One CTA evaluates S thermochemical states per iteration of a persistent grid-stride loop, each
// state in its own block of shared memory.  Whatever does not depend on the state -- decoding a
// reaction, a gather-list entry, a column constant -- is done once and applied to the S states.
// Per iteration:
//   phase 0  species: [X_k] (Eq. 5), NASA-7 c_pk, h_k W_k, B_k, dB_k/dT (Eqs. 9-12, 27, 74)
//   phase 1  reactions (one thread per reaction, sorted by type): k_f, k_r, R_f, R_r, c_i and the
//            reusable per-reaction products of Section 4.1: q_i, Theta_dT,i,
//            the d_j-proportional coefficient a_i and the sparse terms s'_ij
//   phase 2  fixed-order gathers: wdot_k, A_k, T-column sums and diagonal cells (kSpLanes lanes per
//            species); off-diagonal cells of the species block into a shared-memory tile, lists
//            sorted by length so that the 32 lanes of a warp run the same number of steps
//   phase 3  species finalisation + block reductions (dT/dt, energy row of Eq. 113)
//   phase 4  dense write-out, one coalesced column segment per warp: each element is
//            W_k ( A_k/rho d_j + sum_i nu_ki s'_ij / W_j - sum_i nu_ki s'_iNs / W_Ns )
//            which is Eq. 112 with the per-reaction terms of Eqs. 118-127 regrouped by what they
//            multiply.
// There are no atomics: every sum has an order fixed at pyjac_mech_create.
#include <cuda_runtime.h>

#include "device_mech.h"
#include "kernels.h"

namespace pyjac {

namespace {

constexpr double kLn10 = 2.302585092994045684;
constexpr double kInvLn10 = 0.434294481903251828;

// indices into the per-state scalar block
enum { kT = 0, kLnT, kInvT, kP, kRho, kW, kM, kCpMix, kDcpDT, kIrho };

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

// deterministic block reduction of NV values over the first `nwa` warps (the others hold zeros):
// xor-butterfly inside the warp, one partial per warp into `red` (NV rows of 32 doubles); after a
// __syncthreads, red_sum adds the partials of one row in warp order -- only the threads that need a
// sum pay for it.
template <int NV>
__device__ __forceinline__ void block_partials(double (&v)[NV], double *red, int lane, int warp, int nwa)
{
    if (warp < nwa) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xFFFFFFFFu, v[q], o);
            if (lane == 0) red[q * 32 + warp] = v[q];
        }
    }
}
__device__ __forceinline__ double red_sum(const double *red, int row, int nwa)
{
    double s = red[row * 32];
    for (int w = 1; w < nwa; ++w) s += red[row * 32 + w];
    return s;
}

// ---- phase 1: one reaction, S states --------------------------------------------------------------
// Everything that does not depend on the state (slot decoding, Arrhenius parameters, table
// pointers) is read once; the loop over the S states of the CTA is inside.
template <int LEVEL, int S>
__device__ __forceinline__ void reaction(const DeviceMech &m, const SmemPlan &sp, double *sm0, int SS, int s,
                                         const EvalOut &out, long long state0, long long n)
{
    const uint4 sl = m.slots[s];
    const uint32_t meta = sl.w;
    const int type = meta_type(meta), rev = meta_rev(meta);
    // offsets of the species blocks {X, B, dB, hW}
    const int sp0 = (sl.x & 0xFFFF) * 4, sp1 = (sl.x >> 16) * 4, sp2 = (sl.y & 0xFFFF) * 4,
              sp3 = (sl.y >> 16) * 4, sp4 = (sl.z & 0xFFFF) * 4, sp5 = (sl.z >> 16) * 4;
    const bool unit_nu = (meta & 0x00EEEEEEu) == 0;          // every nu is 0 or 1
    const int snu_f = meta_nu(meta, 0) + meta_nu(meta, 1) + meta_nu(meta, 2);
    const int snu_r = meta_nu(meta, 3) + meta_nu(meta, 4) + meta_nu(meta, 5);
    const bool pdep = type == PYJAC_THIRD_BODY || type == PYJAC_FALLOFF || type == PYJAC_CHEM_ACTIVATED;
    const bool arrh = type != PYJAC_PLOG && type != PYJAC_CHEBYSHEV;
    double lnA = 0.0, beta = 0.0, Ta = 0.0;
    if (arrh) { lnA = m.lnA[s]; beta = m.beta[s]; Ta = m.Ta[s]; }
    const double dnu_lnc = (double)(snu_r - snu_f) * m.ln_patm_over_R;
    const uint32_t vb = LEVEL == 2 ? m.vbase[s] : 0u;

#pragma unroll 1
    for (int q = 0; q < S; ++q) {
        double *sm = sm0 + q * SS;
        const double *S4 = sm + sp.Sp4;
        const double T = sm[sp.Scal + kT], lnT = sm[sp.Scal + kLnT], invT = sm[sp.Scal + kInvT];

        // ---- forward rate coefficient: ln k_f and L = d ln k_f / dT
        double lnkf, L;
        double lnk0 = 0.0, lnkinf = 0.0, lPrT = 0.0;
        if (arrh) {
            lnkinf = lnA + beta * lnT - Ta * invT;                  // Eq. 21
            lnkf = lnkinf;
            L = (beta + Ta * invT) * invT;                          // Eq. 65
            if (type == PYJAC_FALLOFF || type == PYJAC_CHEM_ACTIVATED) {
                const int pd = s - m.pd_begin;
                const double b0 = m.lo_beta[pd], Ta0 = m.lo_Ta[pd];
                lnk0 = m.lo_lnA[pd] + b0 * lnT - Ta0 * invT;
                lPrT = invT * (b0 - beta + (Ta0 - Ta) * invT - 1.0);   // Eq. 84 / P_r
                if (type == PYJAC_CHEM_ACTIVATED) { lnkf = lnk0; L = (b0 + Ta0 * invT) * invT; }
            }
        } else if (type == PYJAC_PLOG) {                            // Eqs. 37-39, 105
            const double P = sm[sp.Scal + kP];
            const double *pk = m.pk_data + m.pk_ptr[s - m.pk_begin];
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
            const double P = sm[sp.Scal + kP];
            const double *pk = m.pk_data + m.pk_ptr[s - m.pk_begin];
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

        // ---- species data of the six slots (empty slots point at the dummy species {1, 0, 0, 0})
        const double2 xb0 = *reinterpret_cast<const double2 *>(S4 + sp0);
        const double2 xb1 = *reinterpret_cast<const double2 *>(S4 + sp1);
        const double2 xb2 = *reinterpret_cast<const double2 *>(S4 + sp2);
        const double2 xb3 = *reinterpret_cast<const double2 *>(S4 + sp3);
        const double2 xb4 = *reinterpret_cast<const double2 *>(S4 + sp4);
        const double2 xb5 = *reinterpret_cast<const double2 *>(S4 + sp5);

        // ---- rates of progress (Eqs. 18-19) and the products that skip one factor (Eqs. 120-121)
        double Pf, Pr_, sk0, sk1, sk2, sk3, sk4, sk5, sB, sdB = 0.0;
        if (unit_nu) {
            const double p01 = xb0.x * xb1.x, p34 = xb3.x * xb4.x;
            Pf = p01 * xb2.x; Pr_ = p34 * xb5.x;
            sk0 = xb1.x * xb2.x; sk1 = xb0.x * xb2.x; sk2 = p01;
            sk3 = xb4.x * xb5.x; sk4 = xb3.x * xb5.x; sk5 = p34;
            sB = (xb3.y + xb4.y + xb5.y) - (xb0.y + xb1.y + xb2.y);
            if (LEVEL == 2)
                sdB = (S4[sp3 + 2] + S4[sp4 + 2] + S4[sp5 + 2]) - (S4[sp0 + 2] + S4[sp1 + 2] + S4[sp2 + 2]);
        } else {
            const int n0 = meta_nu(meta, 0), n1 = meta_nu(meta, 1), n2 = meta_nu(meta, 2),
                      n3 = meta_nu(meta, 3), n4 = meta_nu(meta, 4), n5 = meta_nu(meta, 5);
            double p0, p1, p2, p3, p4, p5, m0, m1, m2, m3, m4, m5;
            int_pow(xb0.x, n0, p0, m0); int_pow(xb1.x, n1, p1, m1); int_pow(xb2.x, n2, p2, m2);
            int_pow(xb3.x, n3, p3, m3); int_pow(xb4.x, n4, p4, m4); int_pow(xb5.x, n5, p5, m5);
            Pf = p0 * p1 * p2; Pr_ = p3 * p4 * p5;
            sk0 = m0 * p1 * p2; sk1 = p0 * m1 * p2; sk2 = p0 * p1 * m2;
            sk3 = m3 * p4 * p5; sk4 = p3 * m4 * p5; sk5 = p3 * p4 * m5;
            sB = ((double)n3 * xb3.y + (double)n4 * xb4.y + (double)n5 * xb5.y)
                 - ((double)n0 * xb0.y + (double)n1 * xb1.y + (double)n2 * xb2.y);
            if (LEVEL == 2)
                sdB = ((double)n3 * S4[sp3 + 2] + (double)n4 * S4[sp4 + 2] + (double)n5 * S4[sp5 + 2])
                      - ((double)n0 * S4[sp0 + 2] + (double)n1 * S4[sp1 + 2] + (double)n2 * S4[sp2 + 2]);
        }

        // ---- reverse rate coefficient (Eqs. 23-27, 69, 75)
        double kr = 0.0, Lr = 0.0;
        if (rev == PYJAC_REV_FROM_KC) {
            kr = exp_rate(lnkf - sB - dnu_lnc);
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
            const int pd = s - m.pd_begin;
            eb = m.eff_ptr[pd]; ee = m.eff_ptr[pd + 1];
            Xi = meta_single(meta) ? 0.0 : sm[sp.Scal + kM];             // Eqs. 28-30
            for (int e = eb; e < ee; ++e) Xi += m.eff_eps[e] * S4[4 * m.eff_spec[e]];
            if (type == PYJAC_THIRD_BODY) {
                c = Xi; G = Xi; lPrT = -invT; b = R;                     // Eqs. 79-80
            } else {
                const double Pr = exp_rate(lnk0 - lnkinf) * Xi;          // Eq. 31
                const double *fp = m.fall_par + 5 * pd;
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
        sm[sp.Q + s] = c * R;
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
            sm[sp.Th + s] = dcdT * R + c * (dRfdT - dRrdT + R * invT);
            // coefficient of d_j (Eqs. 119, 123, 127 regrouped)
            const double W = sm[sp.Scal + kW];
            const double base = -W * (Rf * (double)snu_f - Rr * (double)snu_r);
            const double mix = (pdep && !meta_single(meta)) ? sm[sp.Scal + kRho] : 0.0;
            sm[sp.Ar + s] = c * base + b * (mix - W * Xi);
            // sparse terms s'_ij = c (k_f S'_j - k_r S''_j) per slot, b (alpha_ij - 1) per efficiency
            const double ckf = c * kf, ckr = -c * kr;
            double *V = sm + sp.V + vb;
            if (meta & 0x00000Fu) *V++ = ckf * sk0;
            if (meta & 0x0000F0u) *V++ = ckf * sk1;
            if (meta & 0x000F00u) *V++ = ckf * sk2;
            if (meta & 0x00F000u) *V++ = ckr * sk3;
            if (meta & 0x0F0000u) *V++ = ckr * sk4;
            if (meta & 0xF00000u) *V++ = ckr * sk5;
            if (pdep) {
                double *Ve = sm + sp.V + m.eff_vbase[s - m.pd_begin] - eb;
                for (int e = eb; e < ee; ++e) Ve[e] = b * m.eff_eps[e];
            }
        }
    }
}

// ---- the kernel ------------------------------------------------------------------------------------
// Shared memory: S state blocks of sp.total doubles, then 7*S rows of 32 doubles of reduction scratch
// (3S rows for phase 0, 4S for phase 3).  The Jacobian tile of a state holds rows r = 0..ns of a
// panel of columns: r = 0 is the energy row (stored times W_j), r = k + 1 the raw species sums.
template <int LEVEL, int NT, int S>
__global__ void __launch_bounds__(NT, (NT <= 128 ? 4 : NT <= 256 ? 2 : 1))
    eval_kernel(const DeviceMech m, const SmemPlan sp, long long n, const double *__restrict__ Tg,
                const double *__restrict__ Pg, const double *__restrict__ Yg, long long ldy, const EvalOut out)
{
    extern __shared__ double sm_all[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = NT / 32;
    const int ns = m.ns, nr = m.nr, ld = m.ld, ldt = m.ldt;
    const int SS = sp.total;
    double *red0 = sm_all + S * SS, *red3 = red0 + 3 * S * 32;
    const int nwa = min(NW, (ns + 31) >> 5);     // warps that own species
#pragma unroll
    for (int q = 0; q < S; ++q) {
        double *sm = sm_all + q * SS;
        if (tid == 0) {   // the empty-slot dummy species {[X] = 1, B = dB = hW = 0} and the zero slots
            sm[sp.Sp4 + 4 * ns] = 1.0; sm[sp.Sp4 + 4 * ns + 1] = 0.0;
            sm[sp.Sp4 + 4 * ns + 2] = 0.0; sm[sp.Sp4 + 4 * ns + 3] = 0.0;
            sm[sp.Q + nr] = 0.0; sm[sp.Ar + nr] = 0.0; sm[sp.Th + nr] = 0.0; sm[sp.V + m.n_v] = 0.0;
            sm[sp.WA] = 0.0; sm[sp.WC] = 0.0; sm[sp.WA + ns + 1] = 0.0; sm[sp.WC + ns + 1] = 0.0;
        }
        if (LEVEL == 2)   // cells that collect no reaction stay zero for the whole launch (single panel)
            for (int i = tid; i < ldt * m.pw + 2; i += NT) sm[sp.Tile + i] = 0.0;
    }
    const long long nblk = (n + S - 1) / S;
    for (long long blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
        const long long state0 = blk * S;
        // ---- per-state scalars (one thread per state)
        if (tid < S) {
            const long long st = min(state0 + tid, n - 1);
            double *sc = sm_all + tid * SS + sp.Scal;
            const double T = Tg[st], P = Pg[st];
            sc[kT] = T; sc[kLnT] = log(T); sc[kInvT] = 1.0 / T; sc[kP] = P; sc[kM] = P / (kRu * T);
        }
        __syncthreads();
        // ---- phase 0: species (Eqs. 3-5, 9-13, 27, 54-55, 74)
        {
            double part[3 * S];
#pragma unroll
            for (int i = 0; i < 3 * S; ++i) part[i] = 0.0;
#pragma unroll
            for (int q = 0; q < S; ++q) {
                double *sm = sm_all + q * SS;
                const long long st = min(state0 + q, n - 1);
                const double T = sm[sp.Scal + kT], lnT = sm[sp.Scal + kLnT], invT = sm[sp.Scal + kInvT];
                for (int k = tid; k < ns; k += NT) {
                    const double y = Yg[st * ldy + k];
                    const double iw = m.inv_mw[k];
                    const double *a = m.nasa + (T <= m.t_mid[k] ? 0 : (size_t)7 * ns) + k;
                    const double a0 = a[0], a1 = a[ns], a2 = a[2 * (size_t)ns], a3 = a[3 * (size_t)ns],
                                 a4 = a[4 * (size_t)ns], a5 = a[5 * (size_t)ns], a6 = a[6 * (size_t)ns];
                    const double cpR = a0 + T * (a1 + T * (a2 + T * (a3 + a4 * T)));
                    const double hR = T * (a0 + T * (a1 * 0.5 + T * (a2 * (1.0 / 3.0) + T * (a3 * 0.25 + a4 * 0.2 * T)))) + a5;
                    const double cpk = kRu * cpR * iw;
                    double4 v;
                    v.x = y * iw;
                    v.y = a6 - a0 + (a0 - 1.0) * lnT
                          + T * (a1 * 0.5 + T * (a2 * (1.0 / 6.0) + T * (a3 * (1.0 / 12.0) + a4 * 0.05 * T))) - a5 * invT;
                    v.z = (a0 - 1.0 + a5 * invT) * invT + a1 * 0.5 + T * (a2 * (1.0 / 3.0) + T * (a3 * 0.25 + a4 * 0.2 * T));
                    v.w = kRu * hR;
                    *reinterpret_cast<double4 *>(sm + sp.Sp4 + 4 * k) = v;
                    part[3 * q] += y * iw;
                    if (LEVEL >= 1) { sm[sp.Cp + k] = cpk; part[3 * q + 1] += y * cpk; }
                    if (LEVEL == 2)
                        part[3 * q + 2] += y * (kRu * iw * (a1 + T * (2.0 * a2 + T * (3.0 * a3 + 4.0 * a4 * T))));
                }
            }
            block_partials<3 * S>(part, red0, lane, warp, nwa);
            __syncthreads();
            if (tid < ns) {
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    double *sm = sm_all + q * SS;
                    const double W = 1.0 / red_sum(red0, 3 * q, nwa);
                    const double rho = sm[sp.Scal + kM] * W;
                    if (tid == 0) {
                        sm[sp.Scal + kW] = W; sm[sp.Scal + kRho] = rho; sm[sp.Scal + kIrho] = 1.0 / rho;
                        if (LEVEL >= 1) sm[sp.Scal + kCpMix] = red_sum(red0, 3 * q + 1, nwa);
                        if (LEVEL == 2) sm[sp.Scal + kDcpDT] = red_sum(red0, 3 * q + 2, nwa);
                    }
                    for (int k = tid; k < ns; k += NT) sm[sp.Sp4 + 4 * k] *= rho;
                }
            }
        }
        __syncthreads();
        // ---- phase 1: reactions
        for (int s = tid; s < nr; s += NT) reaction<LEVEL, S>(m, sp, sm_all, SS, s, out, state0, n);
        __syncthreads();
        // ---- phase 2a: species sums over reactions, kSpLanes lanes per species (fixed order)
        for (int c = warp; c < m.n_spchunk; c += NW) {
            const uint2 ch = m.spchunk[c];
            const uint2 *ent = m.sp_ent + ch.x + lane;
            double wd[S], A[S], Tc[S], Dg[S];
#pragma unroll
            for (int q = 0; q < S; ++q) { wd[q] = 0.0; A[q] = 0.0; Tc[q] = 0.0; Dg[q] = 0.0; }
#pragma unroll 2
            for (uint32_t t = 0; t < ch.y; ++t) {
                const uint2 e = ent[t * 32];
                const int s = e.x & 0xFFFF, v = e.y & 0xFFFF;
                const double cf = entry_coef(e.x), cv = entry_coef(e.y);
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    const double *sm = sm_all + q * SS;
                    wd[q] += cf * sm[sp.Q + s];
                    if (LEVEL == 2) {
                        A[q] += cf * sm[sp.Ar + s];
                        Tc[q] += cf * sm[sp.Th + s];
                        Dg[q] += cv * sm[sp.V + v];
                    }
                }
            }
#pragma unroll
            for (int o = kSpLanes / 2; o > 0; o >>= 1) {
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    wd[q] += __shfl_xor_sync(0xFFFFFFFFu, wd[q], o);
                    if (LEVEL == 2) {
                        A[q] += __shfl_xor_sync(0xFFFFFFFFu, A[q], o);
                        Tc[q] += __shfl_xor_sync(0xFFFFFFFFu, Tc[q], o);
                        Dg[q] += __shfl_xor_sync(0xFFFFFFFFu, Dg[q], o);
                    }
                }
            }
            const int k = m.sptask_k[c * (32 / kSpLanes) + lane / kSpLanes];
            if ((lane % kSpLanes) == 0 && k >= 0) {
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    double *sm = sm_all + q * SS;
                    sm[sp.Wdot + k] = wd[q];
                    if (LEVEL == 2) {
                        sm[sp.A + k] = A[q]; sm[sp.Tc + k] = Tc[q];
                        if (m.n_panel == 1) sm[sp.Tile + k + 1 + k * ldt] = Dg[q]; else sm[sp.Diag + k] = Dg[q];
                    }
                }
            }
        }
        // ---- phase 2b: off-diagonal cells of the species block, longest lists first
        auto gather_cells = [&](int p) {
            const int2 pc = m.panel_chunks[p];
            for (int c = pc.x + warp; c < pc.y; c += NW) {
                const uint2 ch = m.cchunk[c];
                const uint32_t *ent = m.c_ent + ch.x + lane;
                const uint32_t addr = m.ctask_addr[c * 32 + lane];
                double acc[S];
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] = 0.0;
#pragma unroll 2
                for (uint32_t t = 0; t < ch.y; ++t) {
                    const uint32_t e = ent[t * 32];
                    const double cf = entry_coef(e);
                    const double *v = sm_all + sp.V + (e & 0xFFFF);
#pragma unroll
                    for (int q = 0; q < S; ++q) acc[q] += cf * v[q * SS];
                }
#pragma unroll
                for (int q = 0; q < S; ++q) sm_all[q * SS + sp.Tile + addr] = acc[q];
            }
        };
        if (LEVEL == 2 && m.n_panel == 1) gather_cells(0);
        __syncthreads();
        // ---- phase 3: species finalisation (Eqs. 7-8, 111, 113)
        {
            double part[4 * S];
#pragma unroll
            for (int i = 0; i < 4 * S; ++i) part[i] = 0.0;
#pragma unroll
            for (int q = 0; q < S; ++q) {
                double *sm = sm_all + q * SS;
                const bool live = state0 + q < n;
                const long long st = state0 + q;
                const double irho = sm[sp.Scal + kIrho], W = sm[sp.Scal + kW];
                for (int k = tid; k < ns; k += NT) {
                    const double wd = sm[sp.Wdot + k];
                    const double Wk = m.mw[k];
                    const double hw = sm[sp.Sp4 + 4 * k + 3];
                    if (LEVEL == 0) { if (out.wdot && live) out.wdot[st * ns + k] = wd; }
                    if (LEVEL == 1) { if (live) out.dydt[st * ld + k + 1] = Wk * wd * irho; }
                    part[4 * q] += hw * wd;
                    if (LEVEL == 2) {
                        const double Ap = wd * W + sm[sp.A + k];
                        const double Tc = sm[sp.Tc + k];
                        sm[sp.WA + k + 1] = Wk * Ap * irho;
                        sm[sp.Col0 + k + 1] = Wk * irho * Tc;
                        part[4 * q + 1] += hw * Ap;
                        part[4 * q + 2] += sm[sp.Cp + k] * Wk * wd;
                        part[4 * q + 3] += hw * Tc;
                    }
                }
            }
            if (LEVEL >= 1) {
                block_partials<4 * S>(part, red3, lane, warp, nwa);
                __syncthreads();
            }
        }
        if (LEVEL == 1 && tid < S && state0 + tid < n) {
            const double *sm = sm_all + tid * SS;
            out.dydt[(state0 + tid) * ld] = -red_sum(red3, 4 * tid, nwa) * sm[sp.Scal + kIrho] / sm[sp.Scal + kCpMix];
        }
        if (LEVEL == 2) {
            // sums needed by the energy row: only the threads that own a column (tid < ns) use them
            double shg[S], shA[S], icp[S], cpl[S], El[S];
#pragma unroll
            for (int q = 0; q < S; ++q) { shg[q] = 0.0; shA[q] = 0.0; icp[q] = 0.0; cpl[q] = 0.0; El[q] = 0.0; }
            const double iwl = m.inv_mw[ns - 1];
            const long long Jstate = (long long)ld * ld;
            if (tid < ns) {
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    double *sm = sm_all + q * SS;
                    const double irho = sm[sp.Scal + kIrho];
                    const double p0 = red_sum(red3, 4 * q, nwa);
                    icp[q] = 1.0 / sm[sp.Scal + kCpMix];
                    if (tid == 0)
                        sm[sp.Col0] = -icp[q] * irho * (red_sum(red3, 4 * q + 2, nwa) - sm[sp.Scal + kDcpDT] * icp[q] * p0
                                                        + red_sum(red3, 4 * q + 3, nwa));
                    shg[q] = p0 * irho; shA[q] = red_sum(red3, 4 * q + 1, nwa) * irho;
                    cpl[q] = sm[sp.Cp + ns - 1];
                    El[q] = 0.0;                      // energy-row sum of the virtual column Nsp
                }
            }
            // panels of columns; the one holding the virtual column Nsp goes first (its sums enter
            // every other column, Eqs. 119, 123, 127)
            for (int pi = 0; pi < m.n_panel; ++pi) {
                const int p = pi == 0 ? m.n_panel - 1 : pi - 1;
                const int j0 = p * m.pw, j1 = min(ns, j0 + m.pw), pwc = j1 - j0;
                if (m.n_panel > 1) {
                    if (pi > 0) __syncthreads();                  // previous panel's write-out done
#pragma unroll
                    for (int q = 0; q < S; ++q)
                        for (int i = tid; i < ldt * m.pw; i += NT) sm_all[q * SS + sp.Tile + i] = 0.0;
                    __syncthreads();
                    gather_cells(p);
#pragma unroll
                    for (int q = 0; q < S; ++q)
                        for (int j = j0 + tid; j < j1; j += NT)
                            sm_all[q * SS + sp.Tile + j + 1 + (j - j0) * ldt] = sm_all[q * SS + sp.Diag + j];
                    __syncthreads();
                }
                // energy-row partial sums E_j = sum_k h_k W_k cell(k, j), kEParts row ranges per column
                const int rows = (ns + kEParts - 1) / kEParts;
                for (int t = tid; t < pwc * kEParts; t += NT) {
                    const int pt = t / pwc, jl = t - pt * pwc;
                    const int k1 = min(ns, (pt + 1) * rows);
                    double e[S];
#pragma unroll
                    for (int q = 0; q < S; ++q) e[q] = 0.0;
                    const double *hw = sm_all + sp.Sp4 + 3, *tl = sm_all + sp.Tile + 1 + jl * ldt;
                    for (int k = pt * rows; k < k1; ++k) {
#pragma unroll
                        for (int q = 0; q < S; ++q) e[q] += hw[q * SS + 4 * k] * tl[q * SS + k];
                    }
#pragma unroll
                    for (int q = 0; q < S; ++q) sm_all[q * SS + sp.Ep + pt * (ns + 1) + jl] = e[q];
                }
                if (pi == 0) {
#pragma unroll
                    for (int q = 0; q < S; ++q)
                        for (int k = tid; k < ns; k += NT)
                            sm_all[q * SS + sp.WC + k + 1] = m.mw[k] * iwl * sm_all[q * SS + sp.Tile + k + 1 + (ns - 1 - j0) * ldt];
                }
                __syncthreads();
                if (tid < ns) {
                    if (pi == 0) {
                        const int jl = ns - 1 - j0;
#pragma unroll
                        for (int q = 0; q < S; ++q) {
                            for (int pt = 0; pt < kEParts; ++pt) El[q] += sm_all[q * SS + sp.Ep + pt * (ns + 1) + jl];
                            El[q] *= iwl;
                        }
                    }
                    // row 0 of the panel's columns, stored times W_j (phase 4 multiplies by 1/W_j)
                    for (int jl = tid; jl < pwc; jl += NT) {
                        const int j = j0 + jl;
                        if (j >= ns - 1) continue;
                        const double2 cc = m.colc[j];
                        const double Wj = m.mw[j];
#pragma unroll
                        for (int q = 0; q < S; ++q) {
                            double *sm = sm_all + q * SS;
                            double E = 0.0;
                            for (int pt = 0; pt < kEParts; ++pt) E += sm[sp.Ep + pt * (ns + 1) + jl];
                            sm[sp.Tile + jl * ldt] = -icp[q] * Wj * (-(sm[sp.Cp + j] - cpl[q]) * icp[q] * shg[q]
                                                                      + cc.x * shA[q] + cc.y * E - El[q]);
                        }
                    }
                }
                __syncthreads();
                // ---- phase 4: dense write-out (column-major, LD = ns + 1): element (r, j + 1) =
                //      WA[r] d_j + (wrow[r] / W_j) tile(r, j) - WC[r]; a warp writes one column segment
                const int pwo = min(j1, ns - 1) - j0;
                if ((ld & 1) == 0) {
                    // even LD: two rows per lane, 16-byte loads and stores
                    const int nrb = (ld + 63) >> 6;
                    int g = NW, h = nrb;                  // g = gcd(NW, nrb)
                    while (h) { const int t = g % h; g = h; h = t; }
                    const int cstep = NW / g, jl0 = warp / g;
                    for (int rb = warp % g; rb < nrb; rb += g) {
                        const int r0 = rb * 64 + 2 * lane;
                        const bool ok = r0 < ld;
                        const int rc = ok ? r0 : 0;
                        const double2 wk2 = *reinterpret_cast<const double2 *>(m.wrow + rc);
                        double2 wa2[S], wc2[S];
#pragma unroll
                        for (int q = 0; q < S; ++q) {
                            wa2[q] = *reinterpret_cast<const double2 *>(sm_all + q * SS + sp.WA + rc);
                            wc2[q] = *reinterpret_cast<const double2 *>(sm_all + q * SS + sp.WC + rc);
                        }
                        const double *src = sm_all + sp.Tile + rc + jl0 * ldt;
                        double *Jp = out.jac + state0 * Jstate + r0 + (long long)(j0 + 1 + jl0) * ld;
                        const double2 *cc = m.colc + j0 + jl0;
                        for (int jl = jl0; jl < pwo; jl += cstep) {
                            const double2 c2 = *cc;
                            const double wa_ = wk2.x * c2.y, wb_ = wk2.y * c2.y;
#pragma unroll
                            for (int q = 0; q < S; ++q) {
                                const double2 x = *reinterpret_cast<const double2 *>(src + q * SS);
                                double2 v;
                                v.x = fma(wa2[q].x, c2.x, fma(wa_, x.x, -wc2[q].x));
                                v.y = fma(wa2[q].y, c2.x, fma(wb_, x.y, -wc2[q].y));
                                if (ok && state0 + q < n) __stcs(reinterpret_cast<double2 *>(Jp + q * Jstate), v);
                            }
                            src += cstep * ldt; Jp += (long long)cstep * ld; cc += cstep;
                        }
                    }
                } else {
                    const int nrb = (ld + 31) >> 5;
                    int g = NW, h = nrb;
                    while (h) { const int t = g % h; g = h; h = t; }
                    const int cstep = NW / g, jl0 = warp / g;
                    for (int rb = warp % g; rb < nrb; rb += g) {
                        const int r = rb * 32 + lane;
                        const bool ok = r < ld;
                        const int rc = ok ? r : 0;
                        const double wk = m.wrow[rc];
                        double wa[S], wc[S];
#pragma unroll
                        for (int q = 0; q < S; ++q) { wa[q] = sm_all[q * SS + sp.WA + rc]; wc[q] = sm_all[q * SS + sp.WC + rc]; }
                        const double *src = sm_all + sp.Tile + rc + jl0 * ldt;
                        double *Jp = out.jac + state0 * Jstate + r + (long long)(j0 + 1 + jl0) * ld;
                        const double2 *cc = m.colc + j0 + jl0;
                        for (int jl = jl0; jl < pwo; jl += cstep) {
                            const double2 c2 = *cc;
                            const double wkiw = wk * c2.y;
#pragma unroll
                            for (int q = 0; q < S; ++q) {
                                const double val = fma(wa[q], c2.x, fma(wkiw, src[q * SS], -wc[q]));
                                if (ok && state0 + q < n) __stcs(Jp + q * Jstate, val);
                            }
                            src += cstep * ldt; Jp += (long long)cstep * ld; cc += cstep;
                        }
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < S; ++q) {
                if (state0 + q >= n) break;
                double *J = out.jac + (state0 + q) * Jstate;
                for (int r = tid; r < ld; r += NT) {
                    __stcs(J + r, sm_all[q * SS + sp.Col0 + r]);
                    __stcs(J + r + (long long)ns * ld, 0.0);
                }
            }
        }
        // the next iteration writes the scalars and the species arrays first: phase 4 reads neither,
        // and the three __syncthreads before phase 1 order everything else
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

size_t eval_smem_bytes(const SmemPlan &sp, int S) { return ((size_t)S * sp.total + 7 * S * 32) * sizeof(double); }

#define PYJAC_FOR_ALL(X) \
    X(128, 1) X(128, 2) X(128, 4) X(256, 1) X(256, 2) X(256, 4) X(512, 1) X(512, 2) X(512, 4) X(1024, 1) X(1024, 2)

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
