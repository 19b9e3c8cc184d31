// kernels.cu -- sm_100a kernels for the batched source term and analytical Jacobian.
//
// One CTA evaluates one thermochemical state at a time (persistent grid-stride loop over states);
// several CTAs are resident per SM so that the fp64-heavy reaction phase of one state overlaps the
// store-heavy write-out of another.  Per state, in shared memory:
//   phase 0  species: [X_k] (Eq. 5), NASA-7 c_pk, h_k W_k, B_k, dB_k/dT (Eqs. 9-12, 27, 74)
//   phase 1  reactions (one thread per reaction, sorted by type): k_f, k_r, R_f, R_r, c_i and the
//            reusable per-reaction products of Section 4.1: q_i, Theta_dT,i,
//            the d_j-proportional coefficient a_i and the sparse terms s'_ij
//   phase 2  fixed-order gathers: wdot_k, A_k, T-column sums, energy-row column sums, and the
//            Jacobian cells that collect more than kLongCell reactions
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

__device__ __forceinline__ double entry_coef(uint32_t e) { return __hiloint2double((int)(e & 0xFFFF0000u), 0); }

// x^nu and nu x^(nu-1) for nu in 0..3 by repeated multiplication (Eqs. 18-19, 120-121; never a
// division by a concentration)
__device__ __forceinline__ void int_pow(double x, int nu, double &p, double &pm)
{
    const double x2 = x * x;
    p = nu == 0 ? 1.0 : nu == 1 ? x : nu == 2 ? x2 : x2 * x;
    pm = nu == 0 ? 0.0 : nu == 1 ? 1.0 : nu == 2 ? 2.0 * x : 3.0 * x2;
}

struct StateScalars {
    double T, lnT, invT, P, rho, W, M, cp, dcpdT;
};

// deterministic block reduction of NV values: xor-butterfly inside the warp, then every thread sums
// the per-warp partials in warp order.  `red` holds NV rows of 32 doubles.  One __syncthreads.
template <int NV>
__device__ __forceinline__ void block_reduce(double (&v)[NV], double *red, int lane, int warp, int nwarps)
{
#pragma unroll
    for (int q = 0; q < NV; ++q) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xFFFFFFFFu, v[q], o);
        if (lane == 0) red[q * 32 + warp] = v[q];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NV; ++q) {
        double s = 0.0;
        for (int w = 0; w < nwarps; ++w) s += red[q * 32 + w];
        v[q] = s;
    }
}

// ---- phase 1: one reaction ------------------------------------------------------------------------
template <int LEVEL>
__device__ __forceinline__ void reaction(const DeviceMech &m, const SmemPlan &sp, double *sm, int s,
                                         const StateScalars &st, const EvalOut &out, long long state)
{
    const uint4 sl = m.slots[s];
    const uint32_t meta = sl.w;
    const int type = meta_type(meta), rev = meta_rev(meta);
    const int spec[6] = {(int)(sl.x & 0xFFFF), (int)(sl.x >> 16), (int)(sl.y & 0xFFFF),
                         (int)(sl.y >> 16), (int)(sl.z & 0xFFFF), (int)(sl.z >> 16)};
    int nu[6];
    double x[6];
#pragma unroll
    for (int e = 0; e < 6; ++e) {
        nu[e] = meta_nu(meta, e);
        x[e] = sm[sp.X + spec[e]];
    }
    const int snu_f = nu[0] + nu[1] + nu[2], snu_r = nu[3] + nu[4] + nu[5];
    const double T = st.T, lnT = st.lnT, invT = st.invT;

    // ---- forward rate coefficient: ln k_f and L = d ln k_f / dT
    double lnkf, L;
    double lnk0 = 0.0, lnkinf = 0.0, lPrT = 0.0;
    if (type == PYJAC_PLOG) {                                   // Eqs. 37-39, 105
        const double *pk = m.pk_data + m.pk_ptr[s - m.pk_begin];
        const int np = (int)pk[0];
        const double *row = pk + 1;                              // {p, ln p, ln A, beta, Ta}
        int lo = 0, hi = 0;
        double wt = 0.0;
        if (st.P <= row[0]) {
            lo = hi = 0;
        } else if (st.P >= row[5 * (np - 1)]) {
            lo = hi = np - 1;
        } else {
            int j = 0;
            while (!(row[5 * j] <= st.P && st.P < row[5 * (j + 1)])) ++j;
            lo = j; hi = j + 1;
            wt = (log(st.P) - row[5 * j + 1]) / (row[5 * (j + 1) + 1] - row[5 * j + 1]);
        }
        const double *a1 = row + 5 * lo, *a2 = row + 5 * hi;
        const double lnk1 = a1[2] + a1[3] * lnT - a1[4] * invT;
        const double lnk2 = a2[2] + a2[3] * lnT - a2[4] * invT;
        lnkf = lnk1 + (lnk2 - lnk1) * wt;
        L = (a1[3] + a1[4] * invT + (a2[3] - a1[3] + (a2[4] - a1[4]) * invT) * wt) * invT;
    } else if (type == PYJAC_CHEBYSHEV) {                       // Eqs. 40-43, 110
        const double *pk = m.pk_data + m.pk_ptr[s - m.pk_begin];
        const int nT = (int)pk[0], nP = (int)pk[1];
        const double iTmin = pk[2], iTmax = pk[3], lpmin = pk[4], lpmax = pk[5];
        const double *eta = pk + 6;
        const double Tr = (2.0 * invT - iTmin - iTmax) / (iTmax - iTmin);
        const double Pr = (2.0 * log10(st.P) - lpmin - lpmax) / (lpmax - lpmin);
        double sum = 0.0, dsum = 0.0;
        double tm2 = 1.0, tm1 = Tr;      // T_{a-2}, T_{a-1}
        double um2 = 1.0, um1 = 2.0 * Tr;   // U_{a-3}, U_{a-2}
        for (int a = 0; a < nT; ++a) {
            const double phiT = a == 0 ? 1.0 : a == 1 ? Tr : 2.0 * Tr * tm1 - tm2;
            if (a >= 2) { tm2 = tm1; tm1 = phiT; }
            double U = 0.0;                                       // U_{a-1}
            if (a >= 1) {
                const int n = a - 1;
                U = n == 0 ? 1.0 : n == 1 ? 2.0 * Tr : 2.0 * Tr * um1 - um2;
                if (n >= 2) { um2 = um1; um1 = U; }
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
    } else {
        lnkinf = m.lnA[s] + m.beta[s] * lnT - m.Ta[s] * invT;   // Eq. 21
        const double Linf = (m.beta[s] + m.Ta[s] * invT) * invT;   // Eq. 65
        lnkf = lnkinf; L = Linf;
        if (type == PYJAC_FALLOFF || type == PYJAC_CHEM_ACTIVATED) {
            const int pd = s - m.pd_begin;
            const double b0 = m.lo_beta[pd], Ta0 = m.lo_Ta[pd];
            lnk0 = m.lo_lnA[pd] + b0 * lnT - Ta0 * invT;
            lPrT = invT * (b0 - m.beta[s] + (Ta0 - m.Ta[s]) * invT - 1.0);   // Eq. 84 / P_r
            if (type == PYJAC_CHEM_ACTIVATED) { lnkf = lnk0; L = (b0 + Ta0 * invT) * invT; }
        }
    }
    const double kf = exp(lnkf);

    // ---- reverse rate coefficient (Eqs. 23-27, 69, 75)
    double kr = 0.0, Lr = 0.0;
    if (rev == PYJAC_REV_FROM_KC) {
        double sB = 0.0, sdB = 0.0;
#pragma unroll
        for (int e = 0; e < 6; ++e) {
            const double sgn = e < 3 ? -(double)nu[e] : (double)nu[e];
            sB += sgn * sm[sp.B + spec[e]];
            if (LEVEL == 2) sdB += sgn * sm[sp.dB + spec[e]];
        }
        kr = exp(lnkf - sB - (double)(snu_r - snu_f) * m.ln_patm_over_R);
        Lr = L - sdB;
    } else if (rev == PYJAC_REV_EXPLICIT) {
        kr = exp(m.rev_lnA[s] + m.rev_beta[s] * lnT - m.rev_Ta[s] * invT);
        Lr = (m.rev_beta[s] + m.rev_Ta[s] * invT) * invT;
    }

    // ---- rates of progress (Eqs. 18-19) and the products that skip one factor (Eqs. 120-121)
    double p[6], pm[6];
#pragma unroll
    for (int e = 0; e < 6; ++e) int_pow(x[e], nu[e], p[e], pm[e]);
    const double Rf = kf * (p[0] * p[1] * p[2]);
    const double Rr = kr * (p[3] * p[4] * p[5]);
    const double R = Rf - Rr;

    // ---- pressure modification c_i (Eq. 20) and its derivatives (Eqs. 77-100)
    double c = 1.0, G = 0.0, fT = 0.0, b = 0.0, Xi = 0.0;
    const bool pdep = type == PYJAC_THIRD_BODY || type == PYJAC_FALLOFF || type == PYJAC_CHEM_ACTIVATED;
    int eb = 0, ee = 0;
    if (pdep) {
        const int pd = s - m.pd_begin;
        eb = m.eff_ptr[pd]; ee = m.eff_ptr[pd + 1];
        Xi = meta_single(meta) ? 0.0 : st.M;                       // Eqs. 28-30
        for (int e = eb; e < ee; ++e) Xi += m.eff_eps[e] * sm[sp.X + m.eff_spec[e]];
        if (type == PYJAC_THIRD_BODY) {
            c = Xi; G = Xi; lPrT = -invT; b = R;                   // Eqs. 79-80
        } else {
            const double Pr = exp(lnk0 - lnkinf) * Xi;            // Eq. 31
            const double *fp = m.fall_par + 5 * pd;
            const int form = meta_form(meta);
            double F = 1.0, gF = 0.0;                             // gF = (P_r/F) dF/dP_r
            if (form == PYJAC_TROE) {                             // Eqs. 33-35, 90-96
                const double a = fp[0];
                const double e3 = exp(-T / fp[1]), e1 = exp(-T / fp[2]);
                const double e2 = fp[4] != 0.0 ? exp(-fp[3] * invT) : 0.0;
                const double Fc = (1.0 - a) * e3 + a * e1 + e2;
                const double dFc = -(1.0 - a) / fp[1] * e3 - a / fp[2] * e1 + fp[3] * invT * invT * e2;
                const double lnFc = log(Fc);
                const double lF = lnFc * kInvLn10, lP = log10(Pr);
                const double At = lP - 0.67 * lF - 0.4;
                const double Bt = 0.806 - 1.1762 * lF - 0.14 * lP;
                const double AB = At / Bt, q = 1.0 + AB * AB;
                F = exp(lnFc / q);
                const double k2 = lnFc * 2.0 * At / (Bt * Bt * Bt) / (kLn10 * q * q);
                gF = -k2 * (Bt + 0.14 * At);
                fT = (1.0 / (Fc * q) - k2 * (1.1762 * At - 0.67 * Bt) / Fc) * dFc;
            } else if (form == PYJAC_SRI) {                       // Eqs. 36, 97-100
                const double ea = exp(-fp[1] * invT), ec = exp(-T / fp[2]);
                const double base = fp[0] * ea + ec, lnb = log(base);
                const double lP = log10(Pr), Xs = 1.0 / (1.0 + lP * lP);
                F = fp[3] * exp(fp[4] * lnT + Xs * lnb);
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
    const double q = c * R;
    sm[sp.Q + s] = q;
    if (LEVEL == 0) {
        const long long o = state * m.nr + m.rxn_orig[s];
        if (out.rf) out.rf[o] = Rf;
        if (out.rr) out.rr[o] = Rr;
        if (out.cmod) out.cmod[o] = c;
    }
    if (LEVEL == 2) {
        // Theta_dT,i of Eqs. 115-117: dc/dT R + c (dR/dT + R/T)
        const double dcdT = pdep ? G * lPrT + c * fT : 0.0;
        const double dRfdT = Rf * (L - (double)snu_f * invT);                 // Eq. 66
        const double dRrdT = Rr * (Lr - (double)snu_r * invT);                // Eqs. 69, 75
        sm[sp.Th + s] = dcdT * R + c * (dRfdT - dRrdT + R * invT);
        // coefficient of d_j (Eqs. 119, 123, 127 regrouped)
        const double base = -st.W * (Rf * (double)snu_f - Rr * (double)snu_r);
        const double mix = (pdep && !meta_single(meta)) ? st.rho : 0.0;
        sm[sp.Ar + s] = c * base + b * (mix - st.W * Xi);
        // sparse terms s'_ij = c (k_f S'_j - k_r S''_j) per slot, b (alpha_ij - 1) per efficiency
        const double ckf = c * kf, ckr = -c * kr;
        double *V = sm + sp.V + m.vbase[s];
        int at = 0;
        if (nu[0]) V[at++] = ckf * (pm[0] * p[1] * p[2]);
        if (nu[1]) V[at++] = ckf * (p[0] * pm[1] * p[2]);
        if (nu[2]) V[at++] = ckf * (p[0] * p[1] * pm[2]);
        if (nu[3]) V[at++] = ckr * (pm[3] * p[4] * p[5]);
        if (nu[4]) V[at++] = ckr * (p[3] * pm[4] * p[5]);
        if (nu[5]) V[at++] = ckr * (p[3] * p[4] * pm[5]);
        if (pdep) {
            double *Ve = sm + sp.V + m.eff_vbase[s - m.pd_begin] - eb;
            for (int e = eb; e < ee; ++e) Ve[e] = b * m.eff_eps[e];
        }
    }
}

// ---- the kernel ------------------------------------------------------------------------------------
template <int LEVEL, int NT>
__global__ void __launch_bounds__(NT) eval_kernel(const DeviceMech m, const SmemPlan sp, long long n,
                                                  const double *__restrict__ Tg, const double *__restrict__ Pg,
                                                  const double *__restrict__ Yg, long long ldy, const EvalOut out)
{
    extern __shared__ double sm[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = NT / 32;
    const int ns = m.ns, nr = m.nr, ld = m.ld, ldt = m.ldt;
    double *tile = sm + sp.Tile;
    if (tid == 0) {   // the empty-slot dummy species ([X] = 1, B = dB = hW = 0) and the zero slots
        sm[sp.X + ns] = 1.0; sm[sp.B + ns] = 0.0; sm[sp.dB + ns] = 0.0; sm[sp.HW + ns] = 0.0;
        sm[sp.Q + nr] = 0.0; sm[sp.Ar + nr] = 0.0; sm[sp.Th + nr] = 0.0; sm[sp.V + m.n_v] = 0.0;
    }
    if (LEVEL == 2)   // cells that collect no reaction stay zero for the whole launch (single panel)
        for (int i = tid; i < ldt * m.pw + 2; i += NT) tile[i] = 0.0;
    double *red = sm + sp.Red;
    for (long long state = blockIdx.x; state < n; state += gridDim.x) {
        StateScalars st;
        st.T = Tg[state]; st.P = Pg[state];
        st.lnT = log(st.T); st.invT = 1.0 / st.T;
        // ---- phase 0: species (Eqs. 3-5, 9-13, 27, 54-55, 74)
        {
            const double T = st.T;
            double part[3] = {0.0, 0.0, 0.0};
            for (int k = tid; k < ns; k += NT) {
                const double y = Yg[state * ldy + k];
                const double iw = m.inv_mw[k];
                const double *a = m.nasa + (T <= m.t_mid[k] ? 0 : (size_t)7 * ns) + k;
                const double a0 = a[0], a1 = a[ns], a2 = a[2 * (size_t)ns], a3 = a[3 * (size_t)ns],
                             a4 = a[4 * (size_t)ns], a5 = a[5 * (size_t)ns], a6 = a[6 * (size_t)ns];
                const double cpR = a0 + T * (a1 + T * (a2 + T * (a3 + a4 * T)));
                const double hR = T * (a0 + T * (a1 * 0.5 + T * (a2 * (1.0 / 3.0) + T * (a3 * 0.25 + a4 * 0.2 * T)))) + a5;
                const double cpk = kRu * cpR * iw;
                sm[sp.X + k] = y * iw;
                sm[sp.B + k] = a6 - a0 + (a0 - 1.0) * st.lnT
                               + T * (a1 * 0.5 + T * (a2 * (1.0 / 6.0) + T * (a3 * (1.0 / 12.0) + a4 * 0.05 * T)))
                               - a5 * st.invT;
                sm[sp.HW + k] = kRu * hR;
                part[0] += y * iw;
                if (LEVEL >= 1) { sm[sp.Cp + k] = cpk; part[1] += y * cpk; }
                if (LEVEL == 2) {
                    sm[sp.dB + k] = (a0 - 1.0 + a5 * st.invT) * st.invT + a1 * 0.5
                                    + T * (a2 * (1.0 / 3.0) + T * (a3 * 0.25 + a4 * 0.2 * T));
                    part[2] += y * (kRu * iw * (a1 + T * (2.0 * a2 + T * (3.0 * a3 + 4.0 * a4 * T))));
                }
            }
            block_reduce<3>(part, red, lane, warp, NW);
            st.W = 1.0 / part[0];
            st.M = st.P / (kRu * st.T);
            st.rho = st.M * st.W;
            st.cp = part[1]; st.dcpdT = part[2];
            for (int k = tid; k < ns; k += NT) sm[sp.X + k] *= st.rho;
        }
        __syncthreads();
        // ---- phase 1: reactions
        for (int s = tid; s < nr; s += NT) reaction<LEVEL>(m, sp, sm, s, st, out, state);
        __syncthreads();
        // ---- phase 2a: species sums over reactions, kSpLanes lanes per species (fixed order)
        for (int c = warp; c < m.n_spchunk; c += NW) {
            const uint2 ch = m.spchunk[c];
            const uint2 *ent = m.sp_ent + ch.x + lane;
            double wd = 0.0, A = 0.0, Tc = 0.0, Dg = 0.0;
            for (uint32_t t = 0; t < ch.y; ++t) {
                const uint2 e = ent[t * 32];
                const int s = e.x & 0xFFFF;
                const double cf = entry_coef(e.x);
                wd += cf * sm[sp.Q + s];
                if (LEVEL == 2) {
                    A += cf * sm[sp.Ar + s];
                    Tc += cf * sm[sp.Th + s];
                    Dg += entry_coef(e.y) * sm[sp.V + (e.y & 0xFFFF)];
                }
            }
#pragma unroll
            for (int o = kSpLanes / 2; o > 0; o >>= 1) {
                wd += __shfl_xor_sync(0xFFFFFFFFu, wd, o);
                if (LEVEL == 2) {
                    A += __shfl_xor_sync(0xFFFFFFFFu, A, o);
                    Tc += __shfl_xor_sync(0xFFFFFFFFu, Tc, o);
                    Dg += __shfl_xor_sync(0xFFFFFFFFu, Dg, o);
                }
            }
            const int k = m.sptask_k[c * (32 / kSpLanes) + lane / kSpLanes];
            if ((lane % kSpLanes) == 0 && k >= 0) {
                sm[sp.Wdot + k] = wd;
                if (LEVEL == 2) {
                    sm[sp.A + k] = A; sm[sp.Tc + k] = Tc;
                    if (m.n_panel == 1) tile[k + k * ldt] = Dg; else sm[sp.Diag + k] = Dg;
                }
            }
        }
        // ---- phase 2b: off-diagonal cells of the species block, longest lists first (single panel)
        auto gather_cells = [&](int p) {
            const int2 pc = m.panel_chunks[p];
            for (int c = pc.x + warp; c < pc.y; c += NW) {
                const uint2 ch = m.cchunk[c];
                const uint32_t *ent = m.c_ent + ch.x + lane;
                double acc = 0.0;
                for (uint32_t t = 0; t < ch.y; ++t) {
                    const uint32_t e = ent[t * 32];
                    acc += entry_coef(e) * sm[sp.V + (e & 0xFFFF)];
                }
                tile[m.ctask_addr[c * 32 + lane]] = acc;
            }
        };
        if (LEVEL == 2 && m.n_panel == 1) gather_cells(0);
        __syncthreads();
        // ---- phase 3: species finalisation (Eqs. 7-8, 111, 113)
        const double irho = 1.0 / st.rho;
        double part[4] = {0.0, 0.0, 0.0, 0.0};
        for (int k = tid; k < ns; k += NT) {
            const double wd = sm[sp.Wdot + k];
            const double Wk = m.mw[k];
            const double hw = sm[sp.HW + k];
            if (LEVEL == 0) { if (out.wdot) out.wdot[state * ns + k] = wd; }
            if (LEVEL == 1) { out.dydt[state * ld + k + 1] = Wk * wd * irho; }
            part[0] += hw * wd;
            if (LEVEL == 2) {
                const double Ap = wd * st.W + sm[sp.A + k];
                const double Tc = sm[sp.Tc + k];
                sm[sp.WA + k] = Wk * Ap * irho;
                sm[sp.Col0 + k + 1] = Wk * irho * Tc;
                part[1] += hw * Ap;
                part[2] += sm[sp.Cp + k] * Wk * wd;
                part[3] += hw * Tc;
            }
        }
        if (LEVEL >= 1) {
            block_reduce<4>(part, red + 3 * 32, lane, warp, NW);
            if (LEVEL == 1 && tid == 0) out.dydt[state * ld] = -part[0] * irho / st.cp;
        }
        if (LEVEL == 2) {
            const double icp = 1.0 / st.cp;
            if (tid == 0) sm[sp.Col0] = -icp * irho * (part[2] - st.dcpdT * icp * part[0] + part[3]);
            const double shg = part[0] * irho, shA = part[1] * irho;
            const double cpl = sm[sp.Cp + ns - 1];
            const double iwl = m.inv_mw[ns - 1];
            double *J = out.jac + state * (long long)ld * ld;
            const int nrb = (ld + 31) >> 5;
            int g = NW, h = nrb;            // g = gcd(NW, nrb)
            while (h) { const int t = g % h; g = h; h = t; }
            double El = 0.0;                // energy-row sum of the virtual column Nsp
            // panels of columns; the one holding the virtual column Nsp goes first (its sums enter
            // every other column, Eqs. 119, 123, 127)
            for (int pi = 0; pi < m.n_panel; ++pi) {
                const int p = pi == 0 ? m.n_panel - 1 : pi - 1;
                const int j0 = p * m.pw, j1 = min(ns, j0 + m.pw), pwc = j1 - j0;
                if (m.n_panel > 1) {
                    if (pi > 0) __syncthreads();                  // previous panel's write-out done
                    for (int i = tid; i < ldt * m.pw; i += NT) tile[i] = 0.0;
                    __syncthreads();
                    gather_cells(p);
                    for (int j = j0 + tid; j < j1; j += NT) tile[j + (j - j0) * ldt] = sm[sp.Diag + j];
                    __syncthreads();
                }
                // energy-row partial sums E_j = sum_k h_k W_k cell(k, j), kEParts row ranges per column
                const int rows = (ns + kEParts - 1) / kEParts;
                for (int t = tid; t < pwc * kEParts; t += NT) {
                    const int jl = t % pwc, pt = t / pwc;
                    const int k1 = min(ns, (pt + 1) * rows);
                    double e = 0.0;
                    for (int k = pt * rows; k < k1; ++k) e += sm[sp.HW + k] * tile[k + jl * ldt];
                    sm[sp.Ep + pt * (ns + 1) + jl] = e;
                }
                if (pi == 0)
                    for (int k = tid; k < ns; k += NT) sm[sp.WC + k] = m.mw[k] * iwl * tile[k + (ns - 1 - j0) * ldt];
                __syncthreads();
                if (pi == 0) {
                    const int jl = ns - 1 - j0;
                    for (int pt = 0; pt < kEParts; ++pt) El += sm[sp.Ep + pt * (ns + 1) + jl];
                    El *= iwl;
                }
                for (int jl = tid; jl < pwc; jl += NT) {
                    const int j = j0 + jl;
                    if (j >= ns - 1) continue;
                    double E = 0.0;
                    for (int pt = 0; pt < kEParts; ++pt) E += sm[sp.Ep + pt * (ns + 1) + jl];
                    sm[sp.Row0 + j + 1] = -icp * (-(sm[sp.Cp + j] - cpl) * icp * shg + m.dcol[j] * shA
                                                  + m.inv_mw[j] * E - El);
                }
                __syncthreads();
                // ---- phase 4: dense write-out (column-major, LD = ns + 1), one column segment per warp
                const int pwo = min(j1, ns - 1) - j0;
                for (int rb = warp % g; rb < nrb; rb += g) {
                    const int r = rb * 32 + lane;
                    const bool row_ok = r < ld;
                    const int k = r - 1;
                    double wa = 0.0, wk = 0.0, wc = 0.0;
                    if (row_ok && r >= 1) { wa = sm[sp.WA + k]; wk = m.mw[k]; wc = sm[sp.WC + k]; }
                    for (int jl = warp / g; jl < pwo; jl += NW / g) {
                        const int j = j0 + jl;
                        const double dj = m.dcol[j], iwj = m.inv_mw[j];
                        if (row_ok) {
                            double val;
                            if (r == 0) val = sm[sp.Row0 + j + 1];
                            else val = wa * dj + (wk * iwj * tile[k + jl * ldt] - wc);
                            __stcs(J + r + (long long)(j + 1) * ld, val);
                        }
                    }
                }
            }
            for (int r = tid; r < ld; r += NT) {
                __stcs(J + r, sm[sp.Col0 + r]);
                __stcs(J + r + (long long)ns * ld, 0.0);
            }
        }
        // the next state's phase 0 writes only arrays that phase 4 does not read; its
        // __syncthreads (two before the tile is written again) order everything else
    }
}

template <int LEVEL, int NT>
cudaError_t launch_t(const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem, long long n,
                     const double *T, const double *P, const double *Y, long long ldy, const EvalOut &out,
                     cudaStream_t stream)
{
    eval_kernel<LEVEL, NT><<<grid, NT, smem, stream>>>(m, sp, n, T, P, Y, ldy, out);
    return cudaGetLastError();
}

template <int LEVEL>
const void *kernel_ptr(int nt)
{
    switch (nt) {
        case 64: return (const void *)eval_kernel<LEVEL, 64>;
        case 128: return (const void *)eval_kernel<LEVEL, 128>;
        case 256: return (const void *)eval_kernel<LEVEL, 256>;
        case 512: return (const void *)eval_kernel<LEVEL, 512>;
        default: return (const void *)eval_kernel<LEVEL, 1024>;
    }
}

}  // namespace

const void *eval_kernel_ptr(int level, int nt)
{
    return level == 0 ? kernel_ptr<0>(nt) : level == 1 ? kernel_ptr<1>(nt) : kernel_ptr<2>(nt);
}

cudaError_t launch_eval(int level, int nt, const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem,
                        long long n, const double *T, const double *P, const double *Y, long long ldy,
                        const EvalOut &out, cudaStream_t stream)
{
#define PYJAC_CASE(L, N) \
    if (level == L && nt == N) return launch_t<L, N>(m, sp, grid, smem, n, T, P, Y, ldy, out, stream)
    PYJAC_CASE(0, 64); PYJAC_CASE(0, 128); PYJAC_CASE(0, 256); PYJAC_CASE(0, 512); PYJAC_CASE(0, 1024);
    PYJAC_CASE(1, 64); PYJAC_CASE(1, 128); PYJAC_CASE(1, 256); PYJAC_CASE(1, 512); PYJAC_CASE(1, 1024);
    PYJAC_CASE(2, 64); PYJAC_CASE(2, 128); PYJAC_CASE(2, 256); PYJAC_CASE(2, 512); PYJAC_CASE(2, 1024);
#undef PYJAC_CASE
    return cudaErrorInvalidValue;
}

}  // namespace pyjac
