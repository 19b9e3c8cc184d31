// device_mech.h -- device-resident tables of one kinetic model and the shared-memory plan of the
// evaluation kernels.  Built by mech_pack.cu (host), consumed by kernels.cu (device).
//
// Notation follows the paper (PAPER.md Sections 2-4): species k, reaction i, nu' / nu'' the
// reactant / product coefficients (Eq. 15), [X_k] concentrations (Eq. 5), c_i the pressure
// modification (Eq. 20).  Reactions are stored in a SORTED order (most expensive rate form first,
// the plain elementary ones last); `rxn_orig` maps back to the caller's order.
//
// One CTA evaluates S states at a time, interleaved in one array `E` in shared memory (element e of
// state q at (e * S + q) doubles); the evaluation is a chain of fixed-order gathers over it:
//   P1  writes, per reaction, the reusable products of Section 4.1: the sparse
//       derivative terms s'_ij (region V), q_i, a_i, Theta_dT,i (region Q, interleaved per reaction)
//       and the reaction enthalpy H_i (region H);
//   A   sums them into per-species / per-column quantities (wdot_k, alpha'_r, gamma'_r, the T column,
//       the column sums of the energy row) and sums the long Jacobian-cell lists piecewise (region Hs);
//   B   walks the Jacobian column by column, lane <-> two rows: each cell gathers its (short) list,
//       adds the rank-two part of Eq. 112 and is streamed to HBM; the energy row (Eq. 113) is finished
//       and stored by the FIX items of the same phase.
#pragma once
#include <cstdint>

namespace pyjac {

constexpr double kRu = 8314.46261815324;   // J kmol^-1 K^-1
constexpr double kPatm = 101325.0;         // Pa
constexpr int kMaxSide = 3;                // species per reaction side
constexpr int kMaxThreads = 512;           // threads per CTA the kernels are compiled for
constexpr int kBPad = 3;                   // items of padding behind the phase-B table (the kernel reads that far ahead)

// meta word of a reaction: bits 0..23 six 4-bit nu (slots 0-2 reactants, 3-5 products; 0 = empty
// slot), 24..26 rxn_type, 27..28 rev_type, 29..30 falloff_form, 31 third body is a single species.
// A reaction with at most three molecules per side is stored with one slot per MOLECULE (nu = 1,
// a species may repeat): then R_f = k_f [X_a][X_b][X_c] and every S'_j of Eq. 120 is a product of
// the other slots -- no powers, and the repeated slots' list entries add up to nu [X]^(nu-1).
__host__ __device__ inline int meta_nu(uint32_t m, int slot) { return (m >> (4 * slot)) & 0xF; }
__host__ __device__ inline int meta_type(uint32_t m) { return (m >> 24) & 7; }
__host__ __device__ inline int meta_rev(uint32_t m) { return (m >> 27) & 3; }
__host__ __device__ inline int meta_form(uint32_t m) { return (m >> 29) & 3; }
__host__ __device__ inline int meta_single(uint32_t m) { return (m >> 31) & 1; }

// A gather entry of the kSum1 / kSum3 lists and of the Jacobian cells: bits 0..17 = byte offset of the
// source element in the CTA's E array (E index * S * 8, below 256 KB), bits 18..31 = the top 14 bits
// of the fp64 coefficient (sign, exponent, two mantissa bits: exact for every integer up to 8 in
// magnitude; larger ones are split into two entries).  Coefficient bits 0 = the padding entry.
constexpr uint32_t kEntOffMask = 0x3FFFFu;
__host__ __device__ inline uint32_t coef_hi14(int coef)
{
    uint32_t a = coef < 0 ? uint32_t(-coef) : uint32_t(coef);
    // high word of the double a, for 1 <= a <= 8
    static const uint32_t hi[9] = {0u,          0x3FF00000u, 0x40000000u, 0x40080000u, 0x40100000u,
                                   0x40140000u, 0x40180000u, 0x401C0000u, 0x40200000u};
    uint32_t h = a <= 8 ? hi[a] : 0u;
    if (coef < 0) h |= 0x80000000u;
    return h & ~kEntOffMask;
}

// kinds of phase-A chunks (32 lanes, 32 >> rshift sums each)
enum : uint32_t {
    kSum3 = 0,     // entries {q_i of reaction i, nu_ki}: sums of nu q_i, nu a_i, nu Theta_i -> wdot_k, alpha'_{k+1}, T column
    kSum1 = 1,     // entries {source, coef}: one sum, times a task constant -> E slot
    kProd = 2,     // entries {index a | index b << 16}: sum of E[a] * E[b] -> E slot
    kAll3 = 3,     // no entries: sums over all reactions of H_i {q_i, a_i, Theta_i} -> S1, A0, S4
};

struct DeviceMech {
    int ns, nr;                 // N_sp, N_reac
    int ld;                     // N_sp + 1
    // ---- species tables
    const double *inv_mw;       // [ns]
    const double *mw;           // [ns]
    const double *colc;         // [ns+1][4] column constants by Jacobian column c: {u_c, v_c, 1/W_j, 0}, j = c - 1:
                                //        u_c = W_j d_j with d_j = 1/W_j - 1/W_Ns (the d rho / d Y_j factor, Eq. 51);
                                //        v_c = W_j where gamma_r applies (1 <= c < ns); c = 0: {0, 0, 1}; c = ns: zeros
    const double *wrow;         // [ns+1] row factors by Jacobian row r: {1, W_0 .. W_{ns-1}}
    const double *nasa;         // [2][5][ns] a_0..a_4, range-major, coefficient-major (coalesced over k)
    const double *t_mid;        // [ns]
    // ---- reaction tables, sorted order
    int n_pd;                   // pressure-dependent reactions (third body, falloff, chem. activated): [0, n_pd)
    int n_pk;                   // PLOG / Chebyshev reactions: [n_pd, n_pd + n_pk)
    int n_rchunk;               // groups of 32 reactions
    int n_plain;                // the last n_plain groups hold only plain reactions
    int n_p1item;
    const uint32_t *p1item;     // work items of P1, most expensive first: group | path << 16 | first state << 20 |
                                // states << 24; path 0 = any reaction (one state); 1 = plain elementary reactions,
                                // 2 = any rate form with at most three molecules per side, k_r from K_c and one NASA
                                // breakpoint: the item's states one after the other, the reaction's constants in registers
    const uint4 *slots;         // [nr] {spec0|spec1<<16, spec2|spec3<<16, spec4|spec5<<16, meta}
    const uint4 *vidx;          // [nr] E indices of the slots' s'_ij: {v0|v1<<16, v2|v3<<16, v4|v5<<16, rpos}
                                //      (empty slots point at the dump slot); rpos = the reaction's position in the
                                //      regions Q and H (a permutation within its store wavefront, mech_pack.cu)
    const double *lnA, *beta, *Ta;               // [nr] forward Arrhenius (k_inf for falloff forms)
    const int32_t *rxn_orig;    // [nr] caller's reaction index
    const double *rev_lnA, *rev_beta, *rev_Ta;   // [nr] explicit reverse parameters
    const uint32_t *th_off;     // [nr] offset into th_data
    const double *th_data;      // per reaction: n_int, (n_int - 1) ascending breakpoints, n_int x {g_0..g_6}:
                                // sum_k nu_ki B_k(T) = g0 + g1 ln T + T (g2 + T (g3 + T (g4 + T g5))) + g6 / T
                                // (Eq. 27 summed over the reaction, one set per interval between the t_mid of
                                // its species; g0 includes (sum nu) ln(p_atm / R) of Eq. 26)
    double brk_common;          // the breakpoint every reaction shares (all n_int <= 2, one t_mid), else NaN
    const double *th_soa;       // the same for reactions with n_int <= 2, per group of 32 reactions and interval:
                                // g_c of reaction s at [(((s >> 5) * 2 + interval) * 7 + c) * 32 + (s & 31)], so that a
                                // lane reads its seven coefficients at constant offsets from one address (coalesced)
    const double *th_brk;       // [nr] the breakpoint (+inf if n_int = 1, NaN if n_int > 2)
    const double *lo_lnA, *lo_beta, *lo_Ta;      // [n_pd] k_0
    const double *fall_par;                      // [n_pd][5]; Troe: {a, 1/T***, 1/T*, T**, has T**}; SRI: {a, b, 1/c, d, e}
    const int32_t *eff_base;    // [general groups + 1] first efficiency entry of a group of 32 reactions
    const uint4 *eff_ent;       // entry e of lane l of group c at [eff_base[c] + 32 e + l]: {species of alpha_ij != 1
                                // (or the single species) | E index of its term << 16, 0, alpha_ij - 1 (fp64 bits;
                                // 1 for the single species)}; padded with {dummy species | dump slot << 16, 0, 0.0}
    const int32_t *pk_ptr;      // [n_pk+1] offsets into pk_data
    const double *pk_data;      // PLOG: n, then n x {p, ln p, ln A, beta, Ta};
                                // Chebyshev: nT, nP, 1/Tmin, 1/Tmax, log10 pmin, log10 pmax, eta[nT*nP]
    // ---- phase A: chunks of 32 lanes, 32 >> rshift sums each, sorted by length at create time and
    // arranged in rows of NW chunks (warp w takes chunk row * NW + w); rows [0, n_arow01) serve the
    // rates / source-term kernels too
    int n_arow, n_arow01;
    const uint2 *achunk;        // {first block of a_ent, steps | kind << 8 | rshift << 12}
    const uint4 *a_ent;         // block 0 of a chunk = a_ent[first + lane] = {output E index (kSum3: species k;
                                // ~0 = none), constant factor (fp64 bits, 2 words), 0}; block b >= 1 =
                                // a_ent[first + 32 b + lane] = the lane's entries of steps 4b-4 .. 4b-1
    // ---- phase B: one item per (slab of rows, Jacobian column), slab-major.  A lane owns `rp` rows
    // (rp = 2: rows 64 slab + 2 lane, + 1, stored with one 16-byte store; rp = 1 when ld is odd).
    int rp, n_slab;
    const uint4 *b_ent;         // item it = slab * ld + c: b_ent[(it * rp + h) * 32 + lane] = {three entries of the lane's
                                // cell h (padded with the zero slot), steps of the item's cells h: 0 none, 1 one, 2 three}
    const int32_t *bsplit;      // [NW + 1] the items of warp w are [bsplit[w], bsplit[w + 1])
    // ---- regions of E (indices in elements per state)
    int eQ;                     // [nr][3] {q_i, a_i + W q_i, Theta_dT,i} of the reaction at position rpos
    int eH;                     // [nr] reaction enthalpy H_i, same positions
    int eAlpha, eGamma;         // [ns+1] alpha'_r = A_k / rho, gamma'_r = Gamma_k / W_Ns by Jacobian row r = k + 1
    int eTc;                    // [ns+1] the T column by row: sum_i nu_ki Theta_i / rho (Eq. 111 without W_k)
    int eWdot;                  // [ns]
    int eG0;                    // [ns]   sum_i H_i s'_ij per column species j
    int eS1, eA0, eS4;          // scalars: sum_i H_i q_i, sum_i H_i a_i, sum_i H_i Theta_i
    int eZero;                  // slots that stay 0 (padding of the lists)
    int eDump;                  // a slot nobody reads (stores of empty reaction slots)
    int eHs;                    // partial sums of the long Jacobian-cell lists
    int n_e;                    // size of E
    int n_aent, n_bent, n_achunk;   // sizes of a_ent, b_ent (16-byte units) and achunk (8-byte units): the checked build
};

// per-state scalars (region Scal of the shared-memory plan)
enum {
    kT = 0, kLnT, kInvT, kP, kLnP, kRho, kIrho, kW, kM, kCpMix, kDcpDT, kIcp,
    // Jacobian-vector product (level 3): v_0, U / rho and v_0 / rho with U = sum_j d_j v_j, and
    // C_v = sum_j (c_pj - c_pNs) v_j (the vector's entries for T and the species, Eq. 1)
    kV0, kUrho, kV0rho, kCv, kNScal = 16
};

// Shared-memory plan (offsets in doubles PER STATE).  The S states of a CTA iteration are interleaved:
// element i of region R of state q lives at (R + i) * S + q.  The mixture part (X, Cp, Scal) exists
// twice: the one of the next iteration is filled while this one is in use.  After the S states come the
// state-independent tables (colc, wrow), loaded once per CTA.
struct SmemPlan {
    int E;                              // [n_e]
    int P0;                             // two mixture parts of p0size doubles
    int p0size;
    int oX;                             // within a mixture part: [ns+1] concentrations; slot ns = 1 (empty reaction slots)
    int oCp;                            // [ns] c_pk (mass based)
    int oVw;                            // [ns+1] level 3: v_j / W_j per species (the last one: -sum_j v_j / W_Ns; slot ns = 0)
    int oScal;                          // [kNScal]
    int total;                          // doubles per state
    int colc;                           // [ld][4], offset in doubles from the end of the state part
    int wrow;                           // [ld]
    int etab;                           // [32] 2^(j/32), the table of exp_rate (kernels.cu)
    int staged;                         // 1: the gather tables of phases A and B are copied to shared memory once per CTA
    int t_achunk, t_aent, t_bent;       // their offsets (doubles from the end of the state part), sizes in 16-byte units
    int n_achunk16, n_aent16, n_bent16;
    int shared_total;                   // doubles of the state-independent part
};

inline SmemPlan make_smem_plan(int ns, int n_e, int n_achunk16 = 0, int n_aent16 = 0, int n_bent16 = 0)
{
    SmemPlan p{};
    int o = 0;
    auto take = [&](int n) { int r = o; o += (n + 1) & ~1; return r; };
    p.E = take(n_e);
    p.P0 = o;
    {
        const int base = o;
        p.oX = take(ns + 1) - base;
        p.oCp = take(ns) - base;
        p.oVw = take(ns + 1) - base;
        p.oScal = take(kNScal) - base;
        p.p0size = o - base;
        o += p.p0size;
    }
    p.total = o;
    o = 0;
    p.colc = take(4 * (ns + 1));
    p.wrow = take(ns + 1);
    p.etab = take(32);
    p.staged = n_bent16 > 0 ? 1 : 0;
    p.n_achunk16 = n_achunk16; p.n_aent16 = n_aent16; p.n_bent16 = n_bent16;
    p.t_achunk = take(2 * n_achunk16);
    p.t_aent = take(2 * n_aent16);
    p.t_bent = take(2 * n_bent16);
    p.shared_total = o;
    return p;
}

}  // namespace pyjac
