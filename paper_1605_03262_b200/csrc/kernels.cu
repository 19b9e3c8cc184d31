// kernels.cu -- sm_100a kernels for the batched source term and analytical Jacobian.
//
// One CTA evaluates S thermochemical states per iteration of a persistent grid-stride loop.  The S states
// are interleaved in shared memory (element i of a region for state q at (R + i) * S + q), so whatever does
// not depend on the state -- decoding a reaction, a gather entry, a column constant -- is done once per lane
// and applied to the S states.  Per iteration, separated by CTA barriers:
//   P1  one dynamic queue.  Its first S items are the mixtures of the NEXT batch (Eqs. 3-5, 9-13, 54-55;
//       warp <-> state: [X_k], c_pk, mixture c_p, d c_p / dT; for the Jacobian-vector product also the
//       vector), written into the other of two mixture parts.  The others are groups of 32 reactions,
//       lane <-> reaction: k_f, k_r (K_c from the per-reaction polynomial of device_mech.h `th_data`), R_f,
//       R_r, c_i and the reusable per-reaction products of Section 4.1 into E: q_i,
//       Theta_dT,i, a_i (the coefficient of d_j), the sparse terms s'_ij, the enthalpy H_i.  The reaction's
//       constants are read once per item and stay in registers over its states; the common part of every
//       rate form is branch-free, pressure-dependent lanes add the c_i tail.
//   A   fixed-order gathers over E, lane <-> sum (or a share of one): wdot_k (Eq. 14), alpha'_r, gamma'_r
//       of Eq. 112, the T column (Eq. 111), the column sums of the energy row (Eq. 113), and the long
//       Jacobian-cell lists piece by piece
//   B   the Jacobian, column by column, lane <-> two rows: every cell gathers its (at most three) entries
//       on top of alpha'_r u_c - gamma'_r v_c, which is Eq. 112 with the per-reaction terms of Eqs.
//       118-127 regrouped by what they multiply, and is stored at once: a warp
//       stores up to 512 contiguous bytes per state and column, nothing is staged.  FIX items of the same
//       phase finish and store the energy row (Eq. 113).  The rates, source-term and Jacobian-vector-product
//       kernels (LEVEL 0, 1, 3) write their outputs here instead: they need the per-species sums only.
// There are no atomics on data: every sum has an order fixed at pyjac_mech_create.
#include <cuda_runtime.h>

#include "device_mech.h"
#include "kernels.h"

// -DPYJAC_CHECKED builds the kernels with a bounds check on every table-driven shared-memory access and
// every gather-table read (the shipped build relies on the self-check of mech_pack.cu instead); a violation
// traps, which the next synchronisation reports as a launch failure.  Used by tests/test_gpu_parity.py's
// checked-build run (profiles/r2_checked_build.md): compute-sanitizer is closed on the measurement pool.
#ifdef PYJAC_CHECKED
#define PYJAC_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define PYJAC_CHECK(cond) do { } while (0)
#endif

namespace pyjac {

namespace {

constexpr double kLn10 = 2.302585092994045684;
constexpr double kInvLn10 = 0.434294481903251828;

__device__ __forceinline__ double entry_coef(uint32_t e) { return __hiloint2double((int)(e & ~kEntOffMask), 0); }

// exp(x) for the rate coefficients: x = (32 k + j) ln2/32 + r with |r| <= ln2/64, so that
// exp(x) = 2^k 2^(j/32) exp(r): a 32-entry table (staged in shared memory; the index differs per lane), a
// degree-6 polynomial (truncation 4e-18) and the power of two added to the exponent field.  About 1.5 ulp;
// x <= -708 gives 0 and x >= 708 gives +inf (the rate is outside the normal range either way).
__constant__ double c_exp2_32[32] = {
    0x1.0000000000000p+0, 0x1.059b0d3158574p+0, 0x1.0b5586cf9890fp+0, 0x1.11301d0125b51p+0,
    0x1.172b83c7d517bp+0, 0x1.1d4873168b9aap+0, 0x1.2387a6e756238p+0, 0x1.29e9df51fdee1p+0,
    0x1.306fe0a31b715p+0, 0x1.371a7373aa9cbp+0, 0x1.3dea64c123422p+0, 0x1.44e086061892dp+0,
    0x1.4bfdad5362a27p+0, 0x1.5342b569d4f82p+0, 0x1.5ab07dd485429p+0, 0x1.6247eb03a5585p+0,
    0x1.6a09e667f3bcdp+0, 0x1.71f75e8ec5f74p+0, 0x1.7a11473eb0187p+0, 0x1.82589994cce13p+0,
    0x1.8ace5422aa0dbp+0, 0x1.93737b0cdc5e5p+0, 0x1.9c49182a3f090p+0, 0x1.a5503b23e255dp+0,
    0x1.ae89f995ad3adp+0, 0x1.b7f76f2fb5e47p+0, 0x1.c199bdd85529cp+0, 0x1.cb720dcef9069p+0,
    0x1.d5818dcfba487p+0, 0x1.dfc97337b9b5fp+0, 0x1.ea4afa2a490dap+0, 0x1.f50765b6e4540p+0};
// {32/ln2, 1.5 2^52, -(ln2/32) high part (29 bits), -(ln2/32) low part}
__constant__ double c_exp_red[4] = {0x1.71547652b82fep+5, 6755399441055744.0, -0x1.62e42fe000000p-6,
                                    -0x1.f473de6af278fp-35};
// 1/6!, 1/5!, 1/4!, 1/3!, 1/2
__constant__ double c_exp[5] = {1.388888888888889e-03, 8.333333333333333e-03, 4.1666666666666664e-02,
                                1.6666666666666666e-01, 0.5};

__device__ __forceinline__ double exp_rate(double x, const double *etab)
{
    const double s = fma(x, c_exp_red[0], c_exp_red[1]);
    const int n = __double2loint(s);
    const double nd = s - c_exp_red[1];
    double r = fma(nd, c_exp_red[2], x);
    r = fma(nd, c_exp_red[3], r);
    const double t = etab[n & 31];
    double p = fma(c_exp[0], r, c_exp[1]);
    p = fma(p, r, c_exp[2]);
    p = fma(p, r, c_exp[3]);
    p = fma(p, r, c_exp[4]);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    p *= t;                                            // in [1, 2)
    const int hx = __double2hiint(x), ax = hx & 0x7FFFFFFF;
    double v = __hiloint2double(__double2hiint(p) + ((n >> 5) << 20), __double2loint(p));
    // |x| >= 708 (2^k would leave the normal range), infinities and NaN
    if (ax >= 0x40862000) v = ax > 0x7FF00000 ? x : hx < 0 ? 0.0 : __longlong_as_double(0x7FF0000000000000ll);
    return v;
}

// x^nu and nu x^(nu-1) for nu in 0..3 by repeated multiplication (Eqs. 18-19, 120-121; never a
// division by a concentration)
__device__ __forceinline__ void int_pow(double x, int nu, double &p, double &pm)
{
    const double x2 = x * x;
    p = nu == 0 ? 1.0 : nu == 1 ? x : nu == 2 ? x2 : x2 * x;
    pm = nu == 0 ? 0.0 : nu == 1 ? 1.0 : nu == 2 ? 2.0 * x : 3.0 * x2;
}

template <int N>
struct IntC { static constexpr int value = N; };

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

// the S interleaved values of one element: 16-byte vector loads / stores
template <int S>
__device__ __forceinline__ void ldv(const double *p, double (&v)[S])
{
    if (S % 2 == 0) {
#pragma unroll
        for (int q = 0; q < S; q += 2) {
            const double2 t = *reinterpret_cast<const double2 *>(p + q);
            v[q] = t.x; v[q + 1 < S ? q + 1 : q] = t.y;
        }
    } else {
#pragma unroll
        for (int q = 0; q < S; ++q) v[q] = p[q];
    }
}
template <int S>
__device__ __forceinline__ void stv(double *p, const double (&v)[S])
{
    if (S % 2 == 0) {
#pragma unroll
        for (int q = 0; q < S; q += 2) *reinterpret_cast<double2 *>(p + q) = make_double2(v[q], v[q + 1 < S ? q + 1 : q]);
    } else {
#pragma unroll
        for (int q = 0; q < S; ++q) p[q] = v[q];
    }
}

// ---- rate coefficient of a PLOG or Chebyshev reaction (Eqs. 37-43) and L = d ln k_f / dT (Eqs. 105, 110)
__device__ __forceinline__ void special_rate(const DeviceMech &m, int s, int type, double P, double lnP, double lnT,
                                             double invT, double &lnkf, double &L)
{
    const double *pk = m.pk_data + m.pk_ptr[s - m.n_pd];
    if (type == PYJAC_PLOG) {                                       // Eqs. 37-39, 105
        const int np = (int)pk[0];
        const double *row = pk + 1;                              // {p, ln p, ln A, beta, Ta}
        int lo = 0, hi = 0;
        double wt = 0.0;
        if (P <= row[0]) {
            lo = hi = 0;
        } else if (P >= row[5 * (np - 1)]) {
            lo = hi = np - 1;
        } else {
            int j = 0;                                           // p_j <= P < p_{j+1}
            for (int k = 1; k < np - 1; ++k) j += P >= row[5 * k] ? 1 : 0;
            lo = j; hi = j + 1;
            wt = (lnP - row[5 * j + 1]) / (row[5 * (j + 1) + 1] - row[5 * j + 1]);
        }
        const double *a1 = row + 5 * lo, *a2 = row + 5 * hi;
        const double lnk1 = a1[2] + a1[3] * lnT - a1[4] * invT;
        const double lnk2 = a2[2] + a2[3] * lnT - a2[4] * invT;
        lnkf = lnk1 + (lnk2 - lnk1) * wt;
        L = (a1[3] + a1[4] * invT + (a2[3] - a1[3] + (a2[4] - a1[4]) * invT) * wt) * invT;
    } else {                                                        // Chebyshev, Eqs. 40-43, 110
        const int nT = (int)pk[0], nP = (int)pk[1];
        const double iTmin = pk[2], iTmax = pk[3], lpmin = pk[4], lpmax = pk[5];
        const double *eta = pk + 6;
        const double Tr = (2.0 * invT - iTmin - iTmax) / (iTmax - iTmin);
        const double Pr = (2.0 * (lnP * kInvLn10) - lpmin - lpmax) / (lpmax - lpmin);
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
}

// ---- P1, fast path: 32 reactions with at most three molecules per side (one slot per molecule), k_r from
// K_c or irreversible, one NASA breakpoint; the states [q0, q1) of the block one after the other.  Everything
// that does not depend on the state -- the reaction's constants, its slots' addresses -- is read once and
// kept in registers over the states.
// GEN = false: plain elementary reactions only.  GEN = true: any rate form -- PLOG / Chebyshev lanes
// replace ln k_f and L, pressure-dependent lanes (third body, falloff, chemically activated) scale the
// products of the common part by c_i and add the derivative terms of c_i (Eqs. 77-100).
template <int LEVEL, int S, bool GEN>
__device__ __forceinline__ void p1_group(const DeviceMech &m, double *E, const double *X, const double *Vw, const double *sc,
                                         const double *etab, int s, int q0, int q1, const EvalOut &out,
                                         long long state0, long long n)
{
    constexpr bool DER = LEVEL >= 2;       // the derivative terms: Jacobian (2) and Jacobian-vector product (3)
    const int nr = m.nr;
    const uint4 sl = m.slots[s];
    const uint32_t meta = sl.w;
    const int x0 = (sl.x & 0xFFFF) * S, x1 = (sl.x >> 16) * S, x2 = (sl.y & 0xFFFF) * S,
              x3 = (sl.y >> 16) * S, x4 = (sl.z & 0xFFFF) * S, x5 = (sl.z >> 16) * S;
    const int nf = (meta & 0xF) + ((meta >> 4) & 0xF) + ((meta >> 8) & 0xF);
    const int nb = ((meta >> 12) & 0xF) + ((meta >> 16) & 0xF) + ((meta >> 20) & 0xF);
    const double snf = (double)nf, snr = (double)nb, dnu = (double)(nb - nf);
    const bool rev = meta_rev(meta) != PYJAC_IRREVERSIBLE;
    const int type = GEN ? meta_type(meta) : PYJAC_ELEMENTARY;
    const bool pdep = GEN && (type == PYJAC_THIRD_BODY || type == PYJAC_FALLOFF || type == PYJAC_CHEM_ACTIVATED);
    const bool fall = GEN && (type == PYJAC_FALLOFF || type == PYJAC_CHEM_ACTIVATED);
    const bool special = GEN && (type == PYJAC_PLOG || type == PYJAC_CHEBYSHEV);
    const bool mixM = pdep && !meta_single(meta);
    double lnA = m.lnA[s], beta = m.beta[s], Ta = m.Ta[s];
    double dlnA = 0.0, dbeta = 0.0, dTa = 0.0, fp[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (GEN) {
        // k_0 - k_inf of the falloff forms (Eq. 31); a chemically activated reaction multiplies its
        // concentrations by k_0 (reading C5)
        const int s_pd = min(s, max(m.n_pd, 1) - 1);
        const double l0 = m.lo_lnA[s_pd], b0 = m.lo_beta[s_pd], t0 = m.lo_Ta[s_pd];
#pragma unroll
        for (int i = 0; i < 5; ++i) fp[i] = m.fall_par[5 * s_pd + i];
        if (fall) { dlnA = l0 - lnA; dbeta = b0 - beta; dTa = t0 - Ta; }
        if (type == PYJAC_CHEM_ACTIVATED) { lnA = l0; beta = b0; Ta = t0; }
    }
    // sum_k nu_ki B_k (Eq. 27 over the reaction): both intervals
    const double *th = m.th_soa + (size_t)(s >> 5) * (2 * 7 * 32) + (s & 31);
    const double brk = m.brk_common == m.brk_common ? m.brk_common : m.th_brk[s];
    int v0 = 0, v1 = 0, v2 = 0, v3 = 0, v4 = 0, v5 = 0;
    const uint4 vi = m.vidx[s];
    if (LEVEL == 2) {
        v0 = (vi.x & 0xFFFF) * S; v1 = (vi.x >> 16) * S; v2 = (vi.y & 0xFFFF) * S;
        v3 = (vi.y >> 16) * S; v4 = (vi.z & 0xFFFF) * S; v5 = (vi.z >> 16) * S;
    }
    const int orig = LEVEL == 0 ? m.rxn_orig[s] : 0;
    // efficiencies of the group's reactions, entry e of lane l at eff_ent[eff_base[group] + 32 e + l]
    // (padded with eps = 0 on the dummy species, so the trip count is the group's)
    const uint4 *ef = nullptr;
    int n_eff = 0;
    if (GEN) {
        const int grp = s >> 5;
        ef = m.eff_ent + m.eff_base[grp] + (s & 31);
        n_eff = m.eff_base[grp + 1] - m.eff_base[grp];
    }
    const int eq = (m.eQ + 3 * (int)vi.w) * S, eh = (m.eH + (int)vi.w) * S;
    PYJAC_CHECK(x0 <= m.ns * S && x1 <= m.ns * S && x2 <= m.ns * S && x3 <= m.ns * S && x4 <= m.ns * S && x5 <= m.ns * S);
    PYJAC_CHECK(v0 < m.n_e * S && v1 < m.n_e * S && v2 < m.n_e * S && v3 < m.n_e * S && v4 < m.n_e * S && v5 < m.n_e * S);
    PYJAC_CHECK(eq + 3 * S <= m.n_e * S && eh + S <= m.n_e * S && q0 >= 0 && q1 <= S);

    // NQ states at a time (independent chains: the fp64 pipe sees several of them)
    auto body = [&](auto nq_c, const int q) {
        constexpr int NQ = decltype(nq_c)::value;
        double T[NQ], lnT[NQ], invT[NQ], lnkf[NQ], L[NQ], sB[NQ], sdB[NQ], kf[NQ], kr[NQ];
#pragma unroll
        for (int u = 0; u < NQ; ++u) {
            T[u] = sc[kT * S + q + u]; lnT[u] = sc[kLnT * S + q + u]; invT[u] = sc[kInvT * S + q + u];
            lnkf[u] = fma(beta, lnT[u], fma(-Ta, invT[u], lnA));                  // Eq. 21
            L[u] = fma(Ta, invT[u], beta) * invT[u];                              // Eq. 65
        }
        if (GEN && special) {
#pragma unroll
            for (int u = 0; u < NQ; ++u)
                special_rate(m, s, type, sc[kP * S + q + u], sc[kLnP * S + q + u], lnT[u], invT[u], lnkf[u], L[u]);
        }
        // sum_k nu_ki B_k and its T derivative (Eq. 74)
#pragma unroll
        for (int u = 0; u < NQ; ++u) {
            const double *g = th + (T[u] > brk ? 7 * 32 : 0);
            const double g0 = g[0], g1 = g[32], g2 = g[64], g3 = g[96], g4 = g[128], g5 = g[160], g6 = g[192];
            const double t = T[u];
            sB[u] = fma(g1, lnT[u], g0) + fma(t, fma(t, fma(t, fma(t, g5, g4), g3), g2), g6 * invT[u]);
            sdB[u] = fma(fma(-g6, invT[u], g1), invT[u], g2) + t * fma(t, fma(4.0 * g5, t, 3.0 * g4), 2.0 * g3);
        }
#pragma unroll
        for (int u = 0; u < NQ; ++u) kf[u] = exp_rate(lnkf[u], etab);
#pragma unroll
        for (int u = 0; u < NQ; ++u) { kr[u] = exp_rate(lnkf[u] - sB[u], etab); kr[u] = rev ? kr[u] : 0.0; }   // Eqs. 23-27
        double Rf[NQ], Rr[NQ], W[NQ], vq0[NQ], vq1[NQ], vq2[NQ], vh[NQ], vs[6][NQ], cm[NQ];
#pragma unroll
        for (int u = 0; u < NQ; ++u) {
            const double c0 = X[x0 + q + u], c1 = X[x1 + q + u], c2 = X[x2 + q + u], c3 = X[x3 + q + u],
                         c4 = X[x4 + q + u], c5 = X[x5 + q + u];
            const double p01 = c0 * c1, p34 = c3 * c4;
            Rf[u] = kf[u] * (p01 * c2); Rr[u] = kr[u] * (p34 * c5);           // Eqs. 18-19
            const double R = Rf[u] - Rr[u];
            vq0[u] = R; vq1[u] = 0.0; vq2[u] = 0.0; W[u] = 0.0; cm[u] = 1.0;
            vh[u] = kRu * T[u] * fma(T[u], sdB[u], dnu);
            if (DER) {
                W[u] = sc[kW * S + q + u];
                const double iT = invT[u];
                // Theta_dT,i (Eq. 115) with Eqs. 66, 75; the d_j coefficient of Eq. 119 plus W q_i
                const double dRf = Rf[u] * fma(-snf, iT, L[u]);
                const double dRr = Rr[u] * (fma(-snr, iT, L[u]) - sdB[u]);
                vq2[u] = fma(R, iT, dRf - dRr);
                vq1[u] = W[u] * (R - fma(Rf[u], snf, -Rr[u] * snr));
                const double nkr = -kr[u];
                vs[0][u] = kf[u] * (c1 * c2); vs[1][u] = kf[u] * (c0 * c2); vs[2][u] = kf[u] * p01;     // Eq. 120
                vs[3][u] = nkr * (c4 * c5); vs[4][u] = nkr * (c3 * c5); vs[5][u] = nkr * p34;           // Eq. 121
            }
        }
        double sig[NQ];                   // level 3: the efficiency part of sigma_i = sum_j s'_ij v_j / W_j
#pragma unroll
        for (int u = 0; u < NQ; ++u) sig[u] = 0.0;
        if (GEN) {
            // ---- pressure modification c_i (Eq. 20) and its derivatives (Eqs. 77-100): q_i = c R,
            // Theta = dc/dT R + c Theta0, a = c a0 + b (rho - W [X]_i), s'_ij = c s0_ij, and b (alpha_ij - 1)
            // per efficiency; lanes without a pressure dependence keep c = 1, b = 0
            double Xi[NQ], bb[NQ], dcdT[NQ];
#pragma unroll
            for (int u = 0; u < NQ; ++u) { Xi[u] = mixM ? sc[kM * S + q + u] : 0.0; bb[u] = 0.0; dcdT[u] = 0.0; }
            for (int e = 0; e < n_eff; e += 128) {                       // Eqs. 28-30, four entries at a time
                uint4 w[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) w[k] = e + 32 * k < n_eff ? ef[e + 32 * k] : make_uint4((uint32_t)m.ns, 0u, 0u, 0u);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double eps = __hiloint2double((int)w[k].w, (int)w[k].z);
                    const int xo = (w[k].x & 0xFFFF) * S + q;
                    PYJAC_CHECK((int)(w[k].x & 0xFFFF) <= m.ns);
#pragma unroll
                    for (int u = 0; u < NQ; ++u) Xi[u] = fma(eps, X[xo + u], Xi[u]);
                }
            }
            if (pdep) {
#pragma unroll
                for (int u = 0; u < NQ; ++u) {
                    const double R = vq0[u], iT = invT[u], Tu = T[u];
                    double cc, G, lPrT, fT = 0.0;
                    if (type == PYJAC_THIRD_BODY) {
                        cc = Xi[u]; G = Xi[u]; lPrT = -iT; bb[u] = R;            // Eqs. 79-80
                    } else {
                        const double Pr = exp_rate(fma(dbeta, lnT[u], fma(-dTa, iT, dlnA)), etab) * Xi[u];   // Eq. 31
                        lPrT = iT * (dbeta + dTa * iT - 1.0);                    // Eq. 84 / P_r
                        const int form = meta_form(meta);
                        double F = 1.0, gF = 0.0;                                // gF = (P_r/F) dF/dP_r
                        if (form == PYJAC_TROE) {                                // Eqs. 33-35, 90-96
                            // fp[1], fp[2] hold 1/T***, 1/T* (mech_pack.cu); three reciprocals serve every quotient
                            const double a = fp[0], i3 = fp[1], i1 = fp[2];
                            const double e3 = exp_rate(-Tu * i3, etab), e1 = exp_rate(-Tu * i1, etab);
                            const double e2 = fp[4] != 0.0 ? exp_rate(-fp[3] * iT, etab) : 0.0;
                            const double Fc = (1.0 - a) * e3 + a * e1 + e2;
                            const double dFc = -(1.0 - a) * i3 * e3 - a * i1 * e1 + fp[3] * iT * iT * e2;
                            const double lnFc = log(Fc);
                            const double lF = lnFc * kInvLn10, lP = log10(Pr);
                            const double At = lP - 0.67 * lF - 0.4;
                            const double Bt = 0.806 - 1.1762 * lF - 0.14 * lP;
                            const double rB = 1.0 / Bt, rF = 1.0 / Fc;
                            const double AB = At * rB, rq = 1.0 / (1.0 + AB * AB);
                            F = exp_rate(lnFc * rq, etab);
                            const double k2 = lnFc * 2.0 * At * (rB * rB * rB) * (kInvLn10 * rq * rq);
                            gF = -k2 * (Bt + 0.14 * At);
                            fT = (rq - k2 * (1.1762 * At - 0.67 * Bt)) * rF * dFc;
                        } else if (form == PYJAC_SRI) {                          // Eqs. 36, 97-100
                            const double ea = exp_rate(-fp[1] * iT, etab), ec = exp_rate(-Tu * fp[2], etab);   // fp[2] holds 1/c
                            const double base = fp[0] * ea + ec, lnb = log(base);
                            const double lP = log10(Pr), Xs = 1.0 / (1.0 + lP * lP);
                            F = fp[3] * exp_rate(fp[4] * lnT[u] + Xs * lnb, etab);
                            gF = -Xs * Xs * 2.0 * lP * lnb * kInvLn10;
                            fT = fp[4] * iT + Xs * (fp[0] * fp[1] * iT * iT * ea - ec * fp[2]) / base;
                        }
                        const double i1p = 1.0 / (1.0 + Pr);
                        double Theta;
                        if (type == PYJAC_FALLOFF) { cc = Pr * i1p * F; Theta = i1p; }       // Eqs. 82-83
                        else                       { cc = i1p * F;      Theta = -Pr * i1p; } // Eqs. 86-87
                        G = cc * (Theta + gF);
                        bb[u] = R * G / Xi[u];
                    }
                    cm[u] = cc;
                    dcdT[u] = G * lPrT + cc * fT;
                }
            }
            if (DER) {
#pragma unroll
                for (int u = 0; u < NQ; ++u) {
                    const double mixW = mixM ? sc[kRho * S + q + u] - W[u] * Xi[u] : -W[u] * Xi[u];
                    const double R = vq0[u];
                    vq2[u] = fma(dcdT[u], R, cm[u] * vq2[u]);
                    vq1[u] = fma(bb[u], mixW, cm[u] * vq1[u]);
#pragma unroll
                    for (int k = 0; k < 6; ++k) vs[k][u] *= cm[u];
                }
                for (int e = 0; e < n_eff; e += 128) {
                    uint4 w[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        w[k] = e + 32 * k < n_eff ? ef[e + 32 * k] : make_uint4((uint32_t)m.ns | (uint32_t)m.eDump << 16, 0u, 0u, 0u);
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const double eps = __hiloint2double((int)w[k].w, (int)w[k].z);
                        if (LEVEL == 2) {
                            const int eo = (w[k].x >> 16) * S + q;
                            PYJAC_CHECK((int)(w[k].x >> 16) < m.n_e);
#pragma unroll
                            for (int u = 0; u < NQ; ++u) E[eo + u] = bb[u] * eps;
                        } else {        // level 3: b (alpha_ij - 1) v_j / W_j into sigma_i
                            const int xo = (w[k].x & 0xFFFF) * S + q;
#pragma unroll
                            for (int u = 0; u < NQ; ++u) sig[u] = fma(bb[u] * eps, Vw[xo + u], sig[u]);
                        }
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < NQ; ++u) vq0[u] *= cm[u];
        }
#pragma unroll
        for (int u = 0; u < NQ; ++u) {
            if (LEVEL == 0) {
                const long long st = state0 + q + u;
                if (st < n) {
                    const long long o = st * nr + orig;
                    if (out.rf) out.rf[o] = Rf[u];
                    if (out.rr) out.rr[o] = Rr[u];
                    if (out.cmod) out.cmod[o] = cm[u];
                }
            }
            E[eq + q + u] = vq0[u];
            if (LEVEL >= 1) E[eh + q + u] = vh[u];
            if (LEVEL == 3) {
                // tau_i = sum_j s'_ij v_j / W_j + (U / rho) a_i + (v_0 / rho) Theta_i: the one per-reaction
                // scalar of the Jacobian-vector product, (J v)_{k+1} = W_k sum_i nu_ki tau_i
                double t = sig[u];
                t = fma(vs[0][u], Vw[x0 + q + u], t); t = fma(vs[1][u], Vw[x1 + q + u], t); t = fma(vs[2][u], Vw[x2 + q + u], t);
                t = fma(vs[3][u], Vw[x3 + q + u], t); t = fma(vs[4][u], Vw[x4 + q + u], t); t = fma(vs[5][u], Vw[x5 + q + u], t);
                t = fma(sc[kUrho * S + q + u], vq1[u], t);
                t = fma(sc[kV0rho * S + q + u], vq2[u], t);
                E[eq + S + q + u] = t;
            }
            if (LEVEL == 2) {
                E[eq + S + q + u] = vq1[u];
                E[eq + 2 * S + q + u] = vq2[u];
                E[v0 + q + u] = vs[0][u]; E[v1 + q + u] = vs[1][u]; E[v2 + q + u] = vs[2][u];
                E[v3 + q + u] = vs[3][u]; E[v4 + q + u] = vs[4][u]; E[v5 + q + u] = vs[5][u];
            }
        }
    };
    int q = q0;
#pragma unroll 1
    for (; !GEN && q + 2 <= q1; q += 2) body(IntC<2>{}, q);
#pragma unroll 1
    for (; GEN && q + 1 < q1; ++q) body(IntC<1>{}, q);
    if (q < q1) body(IntC<1>{}, q);
}

// ---- P1, general path: one reaction of any type, one state (q) ----------------------------------------
template <int LEVEL, int S>
__device__ __forceinline__ void reaction(const DeviceMech &m, const SmemPlan &sp, double *E, const double *X, const double *Vw,
                                         const double *sc, const double *etab, int s, int q, const EvalOut &out,
                                         long long state0, long long n)
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
    // every table read of the reaction is issued here, before the first use, so that the reads
    // overlap (one L2 round trip instead of one per parameter group); indices are clamped, the values
    // of reactions that do not use them are ignored
    const double brk = m.brk_common == m.brk_common ? m.brk_common : m.th_brk[s];   // NaN: more than two intervals, see th_data
    const double lnA = m.lnA[s], beta = m.beta[s], Ta = m.Ta[s];
    const int s_pd = min(s, max(m.n_pd, 1) - 1);
    const double lo_lnA = m.lo_lnA[s_pd], lo_beta = m.lo_beta[s_pd], lo_Ta = m.lo_Ta[s_pd];
    double fp[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) fp[i] = m.fall_par[5 * s_pd + i];
    const double dnu = (double)(snu_r - snu_f);
    int v0 = 0, v1 = 0, v2 = 0, v3 = 0, v4 = 0, v5 = 0;
    const uint4 vi = m.vidx[s];
    const int rq = (m.eQ + 3 * (int)vi.w) * S, rh = (m.eH + (int)vi.w) * S;     // the reaction's places in Q and H
    if (LEVEL == 2) {
        v0 = (vi.x & 0xFFFF) * S; v1 = (vi.x >> 16) * S; v2 = (vi.y & 0xFFFF) * S;
        v3 = (vi.y >> 16) * S; v4 = (vi.z & 0xFFFF) * S; v5 = (vi.z >> 16) * S;
    }
    // efficiencies of the group's reactions, entry e of lane l at eff_ent[eff_base[group] + 32 e + l]
    // (padded with eps = 0 on the dummy species, so the trip count is the group's)
    const int grp = s >> 5;
    const uint4 *ef = m.eff_ent + m.eff_base[grp] + (s & 31);
    const int n_eff = m.eff_base[grp + 1] - m.eff_base[grp];        // 32 x entries per lane

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
                const double b0 = lo_beta, Ta0 = lo_Ta;
                lnk0 = lo_lnA + b0 * lnT - Ta0 * invT;
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
                int j = 0;                                           // p_j <= P < p_{j+1}
                for (int k = 1; k < np - 1; ++k) j += P >= row[5 * k] ? 1 : 0;
                lo = j; hi = j + 1;
                wt = (sc[kLnP * S + q] - row[5 * j + 1]) / (row[5 * (j + 1) + 1] - row[5 * j + 1]);
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
            const double Pr = (2.0 * (sc[kLnP * S + q] * kInvLn10) - lpmin - lpmax) / (lpmax - lpmin);
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
        const double kf = exp_rate(lnkf, etab);

        // ---- sum_k nu_ki B_k (Eq. 27 over the reaction), its T derivative (Eq. 74) and the reaction
        //      enthalpy H_i = sum_k nu_ki h_k W_k = R T (T d(sum nu B)/dT + sum nu)
        double g0, g1, g2, g3, g4, g5, g6;
        if (brk == brk) {
            const double *g = m.th_soa + (size_t)((s >> 5) * 2 + (T > brk ? 1 : 0)) * (7 * 32) + (s & 31);
            g0 = g[0]; g1 = g[32]; g2 = g[64]; g3 = g[96]; g4 = g[128]; g5 = g[160]; g6 = g[192];
        } else {
            const double *th = m.th_data + m.th_off[s];
            const int nint = (int)th[0];
            int iv = 0;
            for (int b = 1; b < nint; ++b) iv += T > th[b] ? 1 : 0;
            const double *g = th + nint + 7 * iv;
            g0 = g[0]; g1 = g[1]; g2 = g[2]; g3 = g[3]; g4 = g[4]; g5 = g[5]; g6 = g[6];
        }
        const double sB = fma(g1, lnT, g0) + fma(T, fma(T, fma(T, fma(T, g5, g4), g3), g2), g6 * invT);
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
            kr = exp_rate(lnkf - sB, etab);
            Lr = L - sdB;
        } else if (rev == PYJAC_REV_EXPLICIT) {
            const double rb = m.rev_beta[s], rTa = m.rev_Ta[s];
            kr = exp_rate(m.rev_lnA[s] + rb * lnT - rTa * invT, etab);
            Lr = (rb + rTa * invT) * invT;
        }
        const double Rf = kf * Pf;
        const double Rr = kr * Pr_;
        const double R = Rf - Rr;

        // ---- pressure modification c_i (Eq. 20) and its derivatives (Eqs. 77-100)
        double c = 1.0, G = 0.0, fT = 0.0, b = 0.0, Xi = 0.0;
        if (pdep) {
            Xi = meta_single(meta) ? 0.0 : sc[kM * S + q];               // Eqs. 28-30
            for (int e = 0; e < n_eff; e += 256) {                       // eight entries at a time, all reads first
                uint4 w[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) w[u] = e + 32 * u < n_eff ? ef[e + 32 * u] : make_uint4((uint32_t)m.ns, 0u, 0u, 0u);
                double xa = 0.0, xb = 0.0;
#pragma unroll
                for (int u = 0; u < 8; u += 2) {
                    xa = fma(__hiloint2double((int)w[u].w, (int)w[u].z), X[(w[u].x & 0xFFFF) * S + q], xa);
                    xb = fma(__hiloint2double((int)w[u + 1].w, (int)w[u + 1].z), X[(w[u + 1].x & 0xFFFF) * S + q], xb);
                }
                Xi += xa + xb;
            }
            if (type == PYJAC_THIRD_BODY) {
                c = Xi; G = Xi; lPrT = -invT; b = R;                     // Eqs. 79-80
            } else {
                const double Pr = exp_rate(lnk0 - lnkinf, etab) * Xi;          // Eq. 31
                const int form = meta_form(meta);
                double F = 1.0, gF = 0.0;                                // gF = (P_r/F) dF/dP_r
                if (form == PYJAC_TROE) {                                // Eqs. 33-35, 90-96
                    // fp[1], fp[2] hold 1/T***, 1/T* (mech_pack.cu); three reciprocals serve every quotient
                    const double a = fp[0], i3 = fp[1], i1 = fp[2];
                    const double e3 = exp_rate(-T * i3, etab), e1 = exp_rate(-T * i1, etab);
                    const double e2 = fp[4] != 0.0 ? exp_rate(-fp[3] * invT, etab) : 0.0;
                    const double Fc = (1.0 - a) * e3 + a * e1 + e2;
                    const double dFc = -(1.0 - a) * i3 * e3 - a * i1 * e1 + fp[3] * invT * invT * e2;
                    const double lnFc = log(Fc);
                    const double lF = lnFc * kInvLn10, lP = log10(Pr);
                    const double At = lP - 0.67 * lF - 0.4;
                    const double Bt = 0.806 - 1.1762 * lF - 0.14 * lP;
                    const double rB = 1.0 / Bt, rF = 1.0 / Fc;
                    const double AB = At * rB, rq = 1.0 / (1.0 + AB * AB);
                    F = exp_rate(lnFc * rq, etab);
                    const double k2 = lnFc * 2.0 * At * (rB * rB * rB) * (kInvLn10 * rq * rq);
                    gF = -k2 * (Bt + 0.14 * At);
                    fT = (rq - k2 * (1.1762 * At - 0.67 * Bt)) * rF * dFc;
                } else if (form == PYJAC_SRI) {                          // Eqs. 36, 97-100
                    const double ea = exp_rate(-fp[1] * invT, etab), ec = exp_rate(-T * fp[2], etab);       // fp[2] holds 1/c
                    const double base = fp[0] * ea + ec, lnb = log(base);
                    const double lP = log10(Pr), Xs = 1.0 / (1.0 + lP * lP);
                    F = fp[3] * exp_rate(fp[4] * lnT + Xs * lnb, etab);
                    gF = -Xs * Xs * 2.0 * lP * lnb * kInvLn10;
                    fT = fp[4] * invT + Xs * (fp[0] * fp[1] * invT * invT * ea - ec * fp[2]) / base;
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
        E[rq + q] = qi;
        if (LEVEL >= 1) E[rh + q] = H;
        if (LEVEL == 0) {
            const long long st = state0 + q;
            if (st < n) {
                const long long o = st * m.nr + m.rxn_orig[s];
                if (out.rf) out.rf[o] = Rf;
                if (out.rr) out.rr[o] = Rr;
                if (out.cmod) out.cmod[o] = c;
            }
        }
        if (LEVEL >= 2) {
            // Theta_dT,i of Eqs. 115-117: dc/dT R + c (dR/dT + R/T)
            const double dcdT = pdep ? G * lPrT + c * fT : 0.0;
            const double dRfdT = Rf * (L - (double)snu_f * invT);                 // Eq. 66
            const double dRrdT = Rr * (Lr - (double)snu_r * invT);                // Eqs. 69, 75
            const double theta = dcdT * R + c * (dRfdT - dRrdT + R * invT);
            // coefficient of d_j (Eqs. 119, 123, 127 regrouped), plus W q_i: the omega_k W d_j term of
            // Eq. 112 summed per reaction
            const double W = sc[kW * S + q];
            const double base = -W * (Rf * (double)snu_f - Rr * (double)snu_r);
            const double mix = (pdep && !meta_single(meta)) ? sc[kRho * S + q] : 0.0;
            const double ai = c * base + b * (mix - W * Xi) + W * qi;
            // sparse terms s'_ij = c (k_f S'_j - k_r S''_j) per slot, b (alpha_ij - 1) per efficiency
            const double ckf = c * kf, ckr = -c * kr;
            if (LEVEL == 2) {
                E[rq + 2 * S + q] = theta;
                E[rq + S + q] = ai;
                E[v0 + q] = ckf * sk0; E[v1 + q] = ckf * sk1; E[v2 + q] = ckf * sk2;
                E[v3 + q] = ckr * sk3; E[v4 + q] = ckr * sk4; E[v5 + q] = ckr * sk5;
            }
            // level 3: tau_i = sum_j s'_ij v_j / W_j + (U / rho) a_i + (v_0 / rho) Theta_i (see p1_group)
            double tau = fma(sc[kUrho * S + q], ai, sc[kV0rho * S + q] * theta);
            if (LEVEL == 3) {
                tau = fma(ckf * sk0, Vw[x0 + q], tau); tau = fma(ckf * sk1, Vw[x1 + q], tau); tau = fma(ckf * sk2, Vw[x2 + q], tau);
                tau = fma(ckr * sk3, Vw[x3 + q], tau); tau = fma(ckr * sk4, Vw[x4 + q], tau); tau = fma(ckr * sk5, Vw[x5 + q], tau);
            }
            if (pdep)
                for (int e = 0; e < n_eff; e += 256) {
                    uint4 w[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        w[u] = e + 32 * u < n_eff ? ef[e + 32 * u] : make_uint4((uint32_t)m.ns | (uint32_t)m.eDump << 16, 0u, 0u, 0u);
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const double be = b * __hiloint2double((int)w[u].w, (int)w[u].z);
                        if (LEVEL == 2) E[(w[u].x >> 16) * S + q] = be;
                        else tau = fma(be, Vw[(w[u].x & 0xFFFF) * S + q], tau);
                    }
                }
            if (LEVEL == 3) E[rq + S + q] = tau;
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
__device__ __forceinline__ void mixture_and_species(const DeviceMech &m, double *X, double *Cp, double *Vw, double *sc, int q,
                                                    long long st, const double *__restrict__ Tg,
                                                    const double *__restrict__ Pg, const double *__restrict__ Yg,
                                                    long long ldy, int lane, const double *__restrict__ vg, long long ldv)
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
            if (LEVEL >= 2) dcp += y * (kRu * iw * (a1 + T * (2.0 * a2 + T * (3.0 * a3 + 4.0 * a4 * T))));
        }
    }
    if (LEVEL >= 1) { cp = warp_sum(cp); dcp = warp_sum(dcp); }
    if (LEVEL == 3) {
        // the vector of the Jacobian-vector product: v_0 (T), v_{j+1} (Y_j), the last species' entry unused
        // (Eq. 2).  Vw_j = v_{j+1} / W_j; the last species takes -sum_j v_{j+1} / W_Ns, which folds the
        // gamma_r term of Eq. 112 into the per-reaction sums
        const double *vs = vg + st * ldv;
        const double iwl = m.inv_mw[ns - 1];
        double U = 0.0, Vs = 0.0, Cv = 0.0;
        __syncwarp();
        for (int k = lane; k < ns - 1; k += 32) {
            const double vk = vs[k + 1], iw = m.inv_mw[k];
            Vw[k * S + q] = vk * iw;
            U = fma(iw - iwl, vk, U);
            Vs += vk;
            Cv = fma(Cp[k * S + q], vk, Cv);
        }
        U = warp_sum(U); Vs = warp_sum(Vs); Cv = warp_sum(Cv);
        __syncwarp();
        if (lane == 0) {
            const double rho_ = rho, v0 = vs[0];
            Vw[(ns - 1) * S + q] = -Vs * iwl;
            Vw[ns * S + q] = 0.0;
            sc[kV0 * S + q] = v0; sc[kUrho * S + q] = U / rho_; sc[kV0rho * S + q] = v0 / rho_;
            sc[kCv * S + q] = Cv - Cp[(ns - 1) * S + q] * Vs;
        }
    }
    if (lane == 0) {
        sc[kT * S + q] = T; sc[kLnT * S + q] = log(T); sc[kInvT * S + q] = 1.0 / T; sc[kP * S + q] = P; sc[kLnP * S + q] = log(P);
        sc[kM * S + q] = M; sc[kW * S + q] = W; sc[kRho * S + q] = rho; sc[kIrho * S + q] = 1.0 / rho;
        sc[kCpMix * S + q] = cp; sc[kDcpDT * S + q] = dcp; sc[kIcp * S + q] = 1.0 / cp;
    }
}

// 16-byte streaming store of two consecutive Jacobian rows
__device__ __forceinline__ void st_cs_v2(double *p, double a, double b)
{
    __stcs(reinterpret_cast<double2 *>(p), make_double2(a, b));     // st.global.cs.v2.f64; no compiler barrier
}

// ---- phase A, one chunk: 32 lanes, 32 >> rshift sums (device_mech.h).  An entry is decoded once and
// applied to the S states; whole blocks of four steps run without a branch, the chunk's last block by
// its step count.
template <int LEVEL, int S>
__device__ __forceinline__ void a_chunk(const DeviceMech &m, const uint4 *a_ent, double *E, const double *sc, const uint2 ch, int lane,
                                        const uint4 r0_pre, const uint4 w0_pre)
{
    // one state per CTA (S = 1): the chunk's first two table blocks were fetched while the previous chunk was summed
    constexpr bool PRE = S == 1;
    const uint32_t kind = (ch.y >> 8) & 0xF;
    const int steps = (int)(ch.y & 0xFF), rshift = (int)(ch.y >> 12) & 0xF, width = 1 << rshift;
    const uint4 *ep = a_ent + ch.x + lane;
    PYJAC_CHECK((int)ch.x + 32 * (2 + ((int)((ch.y >> 8) & 0xF) == (int)kAll3 ? 0 : ((int)(ch.y & 0xFF) + 3) / 4)) <= m.n_aent);
    const uint4 r0 = PRE ? r0_pre : ep[0];
    const bool head = (lane & (width - 1)) == 0 && r0.x != 0xFFFFFFFFu;
    const char *Eb = reinterpret_cast<const char *>(E);
    const int nr = m.nr;
    const int nfull = steps >> 2, rem = steps & 3;

    // walks the chunk's blocks: `step` is applied to every entry of the lane
#define PYJAC_WALK(step)                                                   \
    {                                                                      \
        const uint4 *bp = ep + 32;                                         \
        uint4 w = PRE ? w0_pre : *bp;                                      \
        for (int b = 0; b < nfull; ++b) {                                  \
            bp += 32;                                                      \
            const uint4 wn = *bp; /* one block ahead (the table is padded) */ \
            step(w.x); step(w.y); step(w.z); step(w.w);                    \
            w = wn;                                                        \
        }                                                                  \
        if (rem > 0) {                                                     \
            step(w.x);                                                     \
            if (rem > 1) {                                                 \
                step(w.y);                                                 \
                if (rem > 2) step(w.z);                                    \
            }                                                              \
        }                                                                  \
    }

    if (kind == kSum1) {
        if (LEVEL == 2) {
            double acc[S];
#pragma unroll
            for (int q = 0; q < S; ++q) acc[q] = 0.0;
            auto step = [&](uint32_t w) {
                const double cf = entry_coef(w);
                double a[S];
                PYJAC_CHECK((w & kEntOffMask) + 8u * S <= 8u * S * (uint32_t)m.n_e);
                ldv<S>(reinterpret_cast<const double *>(Eb + (w & kEntOffMask)), a);
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] = fma(cf, a[q], acc[q]);
            };
            PYJAC_WALK(step)
            for (int o = 1; o < width; o <<= 1)
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] += __shfl_xor_sync(0xFFFFFFFFu, acc[q], o);
            PYJAC_CHECK(!head || (int)r0.x < m.n_e);
            if (head) {
                const double cst = __hiloint2double((int)r0.z, (int)r0.y);
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] *= cst;
                stv<S>(E + r0.x * S, acc);
            }
        }
    } else if (kind == kProd) {
        if (LEVEL == 2) {
            double acc[S];
#pragma unroll
            for (int q = 0; q < S; ++q) acc[q] = 0.0;
            auto step = [&](uint32_t w) {
                double a[S], b[S];
                PYJAC_CHECK((int)(w & 0xFFFF) < m.n_e && (int)(w >> 16) < m.n_e);
                ldv<S>(reinterpret_cast<const double *>(Eb + (w & 0xFFFF) * (S * 8)), a);
                ldv<S>(reinterpret_cast<const double *>(Eb + (w >> 16) * (S * 8)), b);
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] = fma(a[q], b[q], acc[q]);
            };
            PYJAC_WALK(step)
            for (int o = 1; o < width; o <<= 1)
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] += __shfl_xor_sync(0xFFFFFFFFu, acc[q], o);
            PYJAC_CHECK(!head || (int)r0.x < m.n_e);
            if (head) stv<S>(E + r0.x * S, acc);
        }
    } else {
        // kSum3 / kAll3: three sums at once (one for the rates / source-term kernels)
        constexpr int NA = LEVEL == 2 ? 3 : LEVEL == 3 ? 2 : 1;        // level 3: q_i and tau_i
        double acc[NA][S];
#pragma unroll
        for (int w = 0; w < NA; ++w)
#pragma unroll
            for (int q = 0; q < S; ++q) acc[w][q] = 0.0;
        if (kind == kSum3) {
            auto step = [&](uint32_t w_) {
                const double cf = entry_coef(w_);
                PYJAC_CHECK((w_ & kEntOffMask) + 8u * S * NA <= 8u * S * (uint32_t)m.n_e);
                const double *src = reinterpret_cast<const double *>(Eb + (w_ & kEntOffMask));
#pragma unroll
                for (int w = 0; w < NA; ++w) {
                    double a[S];
                    ldv<S>(src + w * S, a);
#pragma unroll
                    for (int q = 0; q < S; ++q) acc[w][q] = fma(cf, a[q], acc[w][q]);
                }
            };
            PYJAC_WALK(step)
        } else {
            for (int i = lane; i < nr; i += 32) {
                double h[S];
                ldv<S>(E + (m.eH + i) * S, h);
#pragma unroll
                for (int w = 0; w < NA; ++w) {
                    double a[S];
                    ldv<S>(E + (m.eQ + 3 * i + w) * S, a);
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
        constexpr int iA = NA > 1 ? 1 : 0, iT = NA > 2 ? 2 : 0;
        if (kind == kAll3) {
            if (lane == 0) {
                stv<S>(E + m.eS1 * S, acc[0]);
                if (LEVEL == 2) { stv<S>(E + m.eA0 * S, acc[iA]); stv<S>(E + m.eS4 * S, acc[iT]); }
                if (LEVEL == 3) stv<S>(E + m.eA0 * S, acc[iA]);          // sum_i H_i tau_i
            }
        } else if (head) {
            const uint32_t k = r0.x;
            PYJAC_CHECK((int)k < m.ns);
            stv<S>(E + (m.eWdot + k) * S, acc[0]);
            if (LEVEL == 3) stv<S>(E + (m.eAlpha + k + 1) * S, acc[iA]);    // sum_i nu_ki tau_i = (J v)_{k+1} / W_k
            if (LEVEL == 2) {
                // alpha'_{k+1} of Eq. 112 regrouped and the T column (Eq. 111), both without W_k
                double ir[S], al[S], tc[S];
                ldv<S>(sc + kIrho * S, ir);
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    al[q] = ir[q] * acc[iA][q];
                    tc[q] = ir[q] * acc[iT][q];
                }
                stv<S>(E + (m.eAlpha + k + 1) * S, al);
                stv<S>(E + (m.eTc + k + 1) * S, tc);
            }
        }
    }
#undef PYJAC_WALK
}

// ---- FIX item `it`: the energy row (Eq. 113), stored by the lanes that finish it (phase B skips row 0).
// Item 0 is J(0,0); item i >= 1 the columns 32(i-1)+1 .. (column ns is zero)
template <int S>
__device__ __forceinline__ void fix_item(const DeviceMech &m, const double *E, const double *Cp, const double *sc,
                                         const double *colc, const double *wrow, int it, int lane, double *J0, int nq)
{
    const int ns = m.ns, ld = m.ld;
    const long long Jstate = (long long)ld * ld;
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
            const double icp = sc[kIcp * S + q];
            const double z = -icp * sc[kIrho * S + q] *
                             (s - sc[kDcpDT * S + q] * icp * E[m.eS1 * S + q] + E[m.eS4 * S + q]);
            if (q < nq) J0[q * Jstate] = z;
        }
        return;
    }
    const int c = (it - 1) * 32 + lane + 1;
    if (c < ns) {
        const double uc = colc[4 * c], wj = colc[4 * c + 1], iwj = colc[4 * c + 2], iwl = m.inv_mw[ns - 1];
        double icp[S], irho[S], s1[S], a0[S], gl[S], cpj[S], cpl[S], g0[S];
        ldv<S>(sc + kIcp * S, icp);
        ldv<S>(sc + kIrho * S, irho);
        ldv<S>(E + m.eS1 * S, s1);
        ldv<S>(E + m.eA0 * S, a0);
        ldv<S>(E + (m.eG0 + ns - 1) * S, gl);
        ldv<S>(Cp + (c - 1) * S, cpj);
        ldv<S>(Cp + (ns - 1) * S, cpl);
        ldv<S>(E + (m.eG0 + c - 1) * S, g0);
#pragma unroll
        for (int q = 0; q < S; ++q) {
            const double a1 = irho[q] * s1[q] * icp[q] * icp[q];     // coefficient of c_pj - c_pNs
            const double alpha0 = -(irho[q] * icp[q]) * a0[q];
            const double gamma0 = -(iwl * icp[q]) * gl[q];
            const double z = (alpha0 * uc + wj * (a1 * (cpj[q] - cpl[q]) - gamma0) - icp[q] * g0[q]) * iwj;
            if (q < nq) J0[q * Jstate + (long long)c * ld] = z;
        }
    } else if (c == ns) {
#pragma unroll
        for (int q = 0; q < S; ++q)
            if (q < nq) J0[q * Jstate + (long long)c * ld] = 0.0;
    }
}

// ---- phase B: the items [it0, it1) of one warp (one item = one Jacobian column for one slab of rows).
// J(r, c) = W_r / W_j (sum of the cell's entries + alpha'_r u_c - gamma'_r v_c)  (Eq. 112 regrouped), RP rows
// per lane; alpha', gamma' and W_r stay in registers while the slab does not change.  A cell has three
// entry words (padded with the zero slot) and the item's step count; the entries of the next item are
// fetched while this one is summed.  FAST: all S states are stored and the output is 16-byte aligned.
template <int S, int RP, bool FAST>
__device__ __forceinline__ void b_run(const DeviceMech &m, const uint4 *b_ent, const double *E, const double *colc, const double *wrow,
                                      int it0, int it1, int lane, double *J0, int nvalid, bool aligned16)
{
    const int ld = m.ld;
    const uint32_t j_state = (uint32_t)(ld * ld);
    const char *Eb = reinterpret_cast<const char *>(E);
    const uint4 *ebase = b_ent + lane;
    int it = it0;
    while (it < it1) {
        const int slab = it / ld, c0 = it - slab * ld;
        const int c1 = min(ld, c0 + (it1 - it));
        const int r = RP * (32 * slab + lane);
        const bool rowok = r < ld;
        const int rr = rowok ? r : 0;
        double al[RP * S], ga[RP * S], wr[RP];
        ldv<RP * S>(E + (m.eAlpha + rr) * S, al);
        ldv<RP * S>(E + (m.eGamma + rr) * S, ga);
#pragma unroll
        for (int hh = 0; hh < RP; ++hh) wr[hh] = wrow[rr + hh];
        const uint4 *ep = ebase + (size_t)it * (32 * RP);
        PYJAC_CHECK(it >= 0 && c1 <= ld && (it + (c1 - c0) + kBPad) * (32 * RP) <= m.n_bent && slab >= 0 && slab < m.n_slab);
        const double *cc = colc + 4 * c0;
        // element (r, c) of the batch's first state: a running pointer when there is one state (measured: 360
        // species 2.63 -> 2.40 ms per 4,096 states), a 32-bit offset otherwise (S pointers cost registers: 53
        // species 2.14 -> 2.16 ms)
        double *dq0 = J0 + (size_t)(c0 * ld + r);
        uint32_t off = (uint32_t)(c0 * ld + r);
        auto dst_of = [&](int q) { return S == 1 ? dq0 : J0 + (off + (uint32_t)q * j_state); };
        // the entries of the next D items are in flight while this one is summed (the table is padded by kBPad
        // items).  One state per CTA makes an item short against the L2 latency of its table words: three items
        // ahead there (360 species, 4,096 states: 2.37 ms with one, 2.05 with two); with S > 1 the registers cost
        // more than the latency (53 species 2.13 -> 2.17 ms with two)
        constexpr int D = S == 1 ? kBPad : 1;
        uint4 qA[D + 1], qB[D + 1];
        uint4 cA = ep[0], cB = cA;                                // D = 1: the current and the next item only
        if (RP == 2) cB = ep[32];
        if (D > 1) {
#pragma unroll
            for (int k = 0; k <= D; ++k) {
                qA[k] = ep[(size_t)k * 32 * RP];
                qB[k] = RP == 2 ? ep[(size_t)k * 32 * RP + 32] : qA[k];
            }
            ep += (size_t)D * 32 * RP;
        }
        for (int c = c0; c < c1; ++c, cc += 4) {
            ep += 32 * RP;
            uint4 wA = cA, wB = cB;
            if (D > 1) {
                wA = qA[0]; wB = qB[0];
#pragma unroll
                for (int k = 0; k < D; ++k) { qA[k] = qA[k + 1]; qB[k] = qB[k + 1]; }
                qA[D] = ep[0];
                qB[D] = RP == 2 ? ep[32] : qA[D];
            } else {
                cA = ep[0];
                cB = RP == 2 ? ep[32] : cA;
            }
            const double2 uv = *reinterpret_cast<const double2 *>(cc);
            const double iw = cc[2];
            double acc[RP * S];
#pragma unroll
            for (int e = 0; e < RP * S; ++e) acc[e] = fma(-ga[e], uv.y, al[e] * uv.x);
            auto step = [&](uint32_t w, int hh) {
                const double cf = entry_coef(w);
                double a[S];
                PYJAC_CHECK((w & kEntOffMask) + 8u * S <= 8u * S * (uint32_t)m.n_e);
                ldv<S>(reinterpret_cast<const double *>(Eb + (w & kEntOffMask)), a);
#pragma unroll
                for (int q = 0; q < S; ++q) acc[hh * S + q] = fma(cf, a[q], acc[hh * S + q]);
            };
            if (wA.w != 0u) {
                step(wA.x, 0);
                if (wA.w > 1u) { step(wA.y, 0); step(wA.z, 0); }
            }
            if (RP == 2 && wB.w != 0u) {
                step(wB.x, RP - 1);
                if (wB.w > 1u) { step(wB.y, RP - 1); step(wB.z, RP - 1); }
            }
            double f[RP];
#pragma unroll
            for (int hh = 0; hh < RP; ++hh) f[hh] = wr[hh] * iw;
            if (FAST) {
                if (rowok) {
#pragma unroll
                    for (int q = 0; q < S; ++q) {
                        double *dst = dst_of(q);
                        if (RP == 2) {
                            const double v0 = acc[q] * f[0], v1 = acc[S + q] * f[RP - 1];
                            if (r != 0) st_cs_v2(dst, v0, v1);
                            else __stcs(dst + 1, v1);
                        } else {
                            if (r != 0) __stcs(dst, acc[q] * f[0]);
                        }
                    }
                }
            } else if (rowok) {
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    if (q >= nvalid) continue;
                    double *dst = dst_of(q);
                    if (RP == 2) {
                        const double v0 = acc[q] * f[0], v1 = acc[S + q] * f[RP - 1];
                        if (r != 0 && aligned16) st_cs_v2(dst, v0, v1);
                        else {
                            if (r != 0) __stcs(dst, v0);
                            __stcs(dst + 1, v1);
                        }
                    } else {
                        if (r != 0) __stcs(dst, acc[q] * f[0]);
                    }
                }
            }
            if (S == 1) dq0 += ld; else off += (uint32_t)ld;
        }
        it += c1 - c0;
    }
}

// ---- the kernel ------------------------------------------------------------------------------------
// Shared memory: S interleaved states of sp.total doubles each (E, two mixture parts), then the
// state-independent column and row constants.
template <int LEVEL, int S, bool STAGE>
__global__ void __launch_bounds__(kMaxThreads, 1)
    eval_kernel(const DeviceMech m, const SmemPlan sp, long long n, const double *__restrict__ Tg,
                const double *__restrict__ Pg, const double *__restrict__ Yg, long long ldy, const EvalOut out)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ int ctr[2];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NT = blockDim.x, NW = NT >> 5;
    const int ns = m.ns, ld = m.ld, nr = m.nr;
    double *E = sm + sp.E * S;
    const double *colc = sm + (size_t)sp.total * S + sp.colc;
    double *wrow = sm + (size_t)sp.total * S + sp.wrow;
    const double *etab = sm + (size_t)sp.total * S + sp.etab;
    {
        if (tid < 32) sm[(size_t)sp.total * S + sp.etab + tid] = c_exp2_32[tid];
        double *cw = sm + (size_t)sp.total * S + sp.colc;
        for (int i = tid; i < 4 * ld; i += NT) cw[i] = m.colc[i];
        for (int i = tid; i < ld; i += NT) wrow[i] = m.wrow[i];
        // E starts as zeros: sums without a list, the zero slots and row 0 of alpha' / gamma' stay zero
        for (int i = tid; i < m.n_e * S; i += NT) E[i] = 0.0;
    }
    // the gather tables of phases A and B: from global memory (L1 / L2), or staged here once per CTA
    const uint2 *achunk = m.achunk;
    const uint4 *a_ent = m.a_ent, *b_ent = m.b_ent;
    if (STAGE) {
        uint4 *base = reinterpret_cast<uint4 *>(sm + (size_t)sp.total * S);
        uint4 *d0 = base + sp.t_achunk / 2, *d1 = base + sp.t_aent / 2, *d2 = base + sp.t_bent / 2;
        const uint4 *s0 = reinterpret_cast<const uint4 *>(m.achunk);
        for (int i = tid; i < sp.n_achunk16; i += NT) d0[i] = s0[i];
        for (int i = tid; i < sp.n_aent16; i += NT) d1[i] = m.a_ent[i];
        for (int i = tid; i < sp.n_bent16; i += NT) d2[i] = m.b_ent[i];
        achunk = reinterpret_cast<const uint2 *>(d0); a_ent = d1; b_ent = d2;
    }
    if (tid < S) {     // the empty-slot dummy species of both mixture parts
        sm[(sp.P0 + sp.oX + ns) * S + tid] = 1.0;
        sm[(sp.P0 + sp.p0size + sp.oX + ns) * S + tid] = 1.0;
    }
    if (tid == 0) ctr[0] = 0;
    const long long nbatch = (n + S - 1) / S;
    const int n_p1 = m.n_p1item;
    const int arows = LEVEL == 2 ? m.n_arow : m.n_arow01;      // levels 0, 1, 3: the per-species sums only
    const int it0 = m.bsplit[warp], it1 = m.bsplit[warp + 1];
    const int nfix = 1 + (ns + 31) / 32;
    const bool aligned16 = (reinterpret_cast<uintptr_t>(out.jac) & 15) == 0;
    int par = 0;
    if ((long long)blockIdx.x < nbatch && warp < S) {
        double *P0 = sm + sp.P0 * S;
        mixture_and_species<LEVEL, S>(m, P0 + sp.oX * S, P0 + sp.oCp * S, P0 + sp.oVw * S, P0 + sp.oScal * S, warp,
                                      min((long long)blockIdx.x * S + warp, n - 1), Tg, Pg, Yg, ldy, lane, out.v, out.ldv);
    }
    __syncthreads();
    for (long long b = blockIdx.x; b < nbatch; b += gridDim.x, par ^= 1) {
        const long long state0 = b * S;
        double *P0 = sm + (sp.P0 + par * sp.p0size) * S;
        const double *X = P0 + sp.oX * S, *sc = P0 + sp.oScal * S, *Vw = P0 + sp.oVw * S;
        // ---- P1: reactions
        // the queue starts with the mixtures of the NEXT batch (into the other mixture part, which nobody reads
        // during this iteration): their input reads from HBM overlap the reactions
        const bool more = b + gridDim.x < nbatch;
        for (int it = grab(&ctr[0], lane); it < n_p1 + S; it = grab(&ctr[0], lane)) {
            if (it < S) {
                if (more) {
                    double *Pn = sm + (sp.P0 + (par ^ 1) * sp.p0size) * S;
                    mixture_and_species<LEVEL, S>(m, Pn + sp.oX * S, Pn + sp.oCp * S, Pn + sp.oVw * S, Pn + sp.oScal * S, it,
                                                  min((b + gridDim.x) * S + it, n - 1), Tg, Pg, Yg, ldy, lane, out.v, out.ldv);
                }
                continue;
            }
            // item = {group of 32 reactions, path, first state}: most expensive first (device_mech.h `p1item`)
            PYJAC_CHECK(it - S < m.n_p1item);
            const uint32_t w = m.p1item[it - S];
            const int c = (int)(w & 0xFFFF), kind = (int)(w >> 16) & 0xF, q = (int)(w >> 20) & 0xF, nq = (int)(w >> 24);
            const int s = min(c * 32 + lane, nr - 1);
            if (kind == 1) p1_group<LEVEL, S, false>(m, E, X, Vw, sc, etab, s, q, q + nq, out, state0, n);
            else if (kind == 2) p1_group<LEVEL, S, true>(m, E, X, Vw, sc, etab, s, q, q + nq, out, state0, n);
            else reaction<LEVEL, S>(m, sp, E, X, Vw, sc, etab, s, q, out, state0, n);
        }
        __syncthreads();
        if (tid == 0) ctr[0] = 0;
        // ---- A: sums over the reactions per species / per column, pieces of the long cell lists
        {
            const uint2 *hp = achunk + warp;
            uint2 h = *hp;
            uint4 r0 = make_uint4(0u, 0u, 0u, 0u), w0 = r0;
            if (S == 1) { r0 = a_ent[h.x + lane]; w0 = a_ent[h.x + 32 + lane]; }
            for (int row = 0; row < arows; ++row) {
                hp += NW;
                PYJAC_CHECK((row + 1) * NW + warp < m.n_achunk);
                const uint2 hn = *hp;                 // the header table is padded by one row
                uint4 r0n = r0, w0n = w0;
                if (S == 1) {                         // both tables are padded for the reads behind the last chunk
                    PYJAC_CHECK((int)hn.x + 64 <= m.n_aent);
                    r0n = a_ent[hn.x + lane]; w0n = a_ent[hn.x + 32 + lane];
                }
                a_chunk<LEVEL, S>(m, a_ent, E, sc, h, lane, r0, w0);
                h = hn; r0 = r0n; w0 = w0n;
            }
        }
        __syncthreads();
        const int nvalid = (int)min((long long)S, n - state0);
        if (LEVEL == 2) {
            // ---- B: the Jacobian column by column, the energy row
            double *J0 = out.jac + state0 * ((long long)ld * ld);
            if (nvalid == S && aligned16) {
                if (m.rp == 2) b_run<S, 2, true>(m, b_ent, E, colc, wrow, it0, it1, lane, J0, nvalid, true);
                else b_run<S, 1, true>(m, b_ent, E, colc, wrow, it0, it1, lane, J0, nvalid, true);
            } else {
                if (m.rp == 2) b_run<S, 2, false>(m, b_ent, E, colc, wrow, it0, it1, lane, J0, nvalid, aligned16);
                else b_run<S, 1, false>(m, b_ent, E, colc, wrow, it0, it1, lane, J0, nvalid, aligned16);
            }
            for (int it = NW - 1 - warp; it < nfix; it += NW)
                fix_item<S>(m, E, P0 + sp.oCp * S, sc, colc, wrow, it, lane, J0, nvalid);
        }
        // ---- outputs of the rates / source-term kernels (Eqs. 7-8, 14)
        if (LEVEL == 0 && out.wdot) {
            for (int k = tid; k < ns; k += NT)
#pragma unroll
                for (int q = 0; q < S; ++q)
                    if (q < nvalid) out.wdot[(state0 + q) * ns + k] = E[(m.eWdot + k) * S + q];
        }
        if (LEVEL == 1) {
            for (int r = tid; r < ld; r += NT)
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    if (q >= nvalid) continue;
                    const double irho = sc[kIrho * S + q];
                    const double v = r == 0 ? -E[m.eS1 * S + q] * irho / sc[kCpMix * S + q]
                                            : wrow[r] * E[(m.eWdot + r - 1) * S + q] * irho;
                    out.dydt[(state0 + q) * ld + r] = v;
                }
        }
        if (LEVEL == 3) {
            // ---- Jacobian-vector product without the matrix: (J v)_{k+1} = W_k sum_i nu_ki tau_i (Eq. 112
            // times v, summed over the columns per reaction first); the energy row (Eq. 113) the same way
            for (int r = 1 + tid; r < ld; r += NT)
#pragma unroll
                for (int q = 0; q < S; ++q)
                    if (q < nvalid) out.jv[(state0 + q) * ld + r] = wrow[r] * E[(m.eAlpha + r) * S + q];
            if (warp == NW - 1) {
                const double *Cp = P0 + sp.oCp * S;
                double s3[S];       // sum_k c_pk W_k wdot_k
#pragma unroll
                for (int q = 0; q < S; ++q) s3[q] = 0.0;
                for (int k = lane; k < ns; k += 32) {
                    const double wk = wrow[k + 1];
#pragma unroll
                    for (int q = 0; q < S; ++q) s3[q] = fma(Cp[k * S + q] * wk, E[(m.eWdot + k) * S + q], s3[q]);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                    for (int q = 0; q < S; ++q) s3[q] += __shfl_xor_sync(0xFFFFFFFFu, s3[q], o);
                if (lane < S && lane < nvalid) {
                    const int q = lane;
                    double sq = s3[0];
#pragma unroll
                    for (int u = 1; u < S; ++u) sq = q == u ? s3[u] : sq;
                    const double icp = sc[kIcp * S + q], irho = sc[kIrho * S + q], S1 = E[m.eS1 * S + q];
                    out.jv[(state0 + q) * ld] = -icp * E[m.eA0 * S + q]
                                                - icp * irho * (sq - sc[kDcpDT * S + q] * icp * S1) * sc[kV0 * S + q]
                                                + irho * S1 * icp * icp * sc[kCv * S + q];
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace

// This file is compiled once per S (states a CTA interleaves): -DPYJAC_S=<1|2|3|4|6> (build.py);
// dispatch.cu switches over them.
#if !defined(PYJAC_S)
#error "compile with -DPYJAC_S=<1|2|3|4|6>"
#endif
#define PYJAC_CAT2(a, b) a##b
#define PYJAC_NAME(a, s) PYJAC_CAT2(a, s)

const void *PYJAC_NAME(eval_kernel_ptr_, PYJAC_S)(int level, bool stage)
{
    if (stage)
        return level == 0 ? (const void *)eval_kernel<0, PYJAC_S, true>
             : level == 1 ? (const void *)eval_kernel<1, PYJAC_S, true>
             : level == 2 ? (const void *)eval_kernel<2, PYJAC_S, true>
                          : (const void *)eval_kernel<3, PYJAC_S, true>;
    return level == 0 ? (const void *)eval_kernel<0, PYJAC_S, false>
         : level == 1 ? (const void *)eval_kernel<1, PYJAC_S, false>
         : level == 2 ? (const void *)eval_kernel<2, PYJAC_S, false>
                      : (const void *)eval_kernel<3, PYJAC_S, false>;
}

cudaError_t PYJAC_NAME(launch_eval_, PYJAC_S)(int level, int threads, const DeviceMech &m, const SmemPlan &sp, int grid,
                                               size_t smem, long long n, const double *T, const double *P,
                                               const double *Y, long long ldy, const EvalOut &out, cudaStream_t stream)
{
#define PYJAC_LAUNCH(L, ST) eval_kernel<L, PYJAC_S, ST><<<grid, threads, smem, stream>>>(m, sp, n, T, P, Y, ldy, out)
    if (sp.staged) {
        if (level == 0) PYJAC_LAUNCH(0, true);
        else if (level == 1) PYJAC_LAUNCH(1, true);
        else if (level == 2) PYJAC_LAUNCH(2, true);
        else PYJAC_LAUNCH(3, true);
    } else {
        if (level == 0) PYJAC_LAUNCH(0, false);
        else if (level == 1) PYJAC_LAUNCH(1, false);
        else if (level == 2) PYJAC_LAUNCH(2, false);
        else PYJAC_LAUNCH(3, false);
    }
#undef PYJAC_LAUNCH
    return cudaGetLastError();
}

}  // namespace pyjac
