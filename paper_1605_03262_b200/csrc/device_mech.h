// device_mech.h -- device-resident tables of one kinetic model and the shared-memory plan of the
// evaluation kernels.  Built by mech_pack.cu (host), consumed by kernels.cu (device).
//
// Notation follows the paper (PAPER.md Sections 2-4): species k, reaction i, nu' / nu'' the
// reactant / product coefficients (Eq. 15), [X_k] concentrations (Eq. 5), c_i the pressure
// modification (Eq. 20).  Reactions are stored in a SORTED order (most expensive rate form first,
// the plain elementary ones last); `rxn_orig` maps back to the caller's order.
//
// The evaluation is a chain of fixed-order gathers over one per-state array `E` in shared memory:
//   phase 1 writes, per reaction, the reusable products of Section 4.1:
//           the sparse derivative terms s'_ij (region V), q_i, a_i, Theta_dT,i (region Q,
//           interleaved per reaction) and the reaction enthalpy H_i (region H);
//   the A1 gathers sum them into per-species / per-column quantities (wdot_k, alpha_r, gamma_r,
//           the T column, the column sums of the energy row);
//   a short FIX step finishes the energy row (Eq. 113);
//   the CELL gathers sum, for every structurally non-zero Jacobian entry, its list of s'_ij into a
//           tile (a panel of Jacobian columns) that follows E in shared memory;
//   the DENSE pass adds the rank-two part of Eq. 112 to the tile and streams it to HBM.
#pragma once
#include <cstdint>

namespace pyjac {

constexpr double kRu = 8314.46261815324;   // J kmol^-1 K^-1
constexpr double kPatm = 101325.0;         // Pa
constexpr int kMaxSide = 3;                // species per reaction side

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

// A gather entry of the kAuxS1 / kAuxT3 lists: bits 0..18 = byte offset of the source element in
// the CTA's interleaved E array (E index * S * 8), bits 19..31 = the top 13 bits of the fp64
// coefficient (exact for +-1, 2, 3, 4, 6, 8; other small integers are split into two entries).
constexpr uint32_t kEntOffMask = 0x7FFFFu;
__host__ __device__ inline uint32_t coef_hi13(int coef)
{
    uint32_t a = coef < 0 ? uint32_t(-coef) : uint32_t(coef);
    uint32_t hi = a == 1 ? 0x3FF0u : a == 2 ? 0x4000u : a == 3 ? 0x4008u : a == 4 ? 0x4010u
                : a == 6 ? 0x4018u : a == 8 ? 0x4020u : 0u;
    if (coef < 0) hi |= 0x8000u;
    return (hi >> 3) << 19;
}

// kinds of gather chunks
enum : uint32_t {
    kAuxT3 = 0,    // entries {q_i of reaction i, nu_ki}: sums of nu q_i, nu a_i, nu Theta_i -> wdot_k, alpha_{k+1}, T column
    kAuxS1 = 1,    // entries {source, coef}: one sum, times a task constant -> E / tile slot
    kAuxH2 = 2,    // entries {index a | index b << 16}: sum of E[a] * E[b] -> E slot
    kAuxR3 = 3,    // no entries: sums over all reactions of H_i {q_i, a_i, Theta_i} -> S1, A0, S4
};

struct DeviceMech {
    int ns, nr;                 // N_sp, N_reac
    int ld;                     // N_sp + 1
    // ---- species tables
    const double *inv_mw;       // [ns]
    const double *mw;           // [ns]
    const double *colc;         // [ns+1][2] column constants by Jacobian column c: {d_j, g_c}, j = c - 1;
                                //        d_j = 1/W_j - 1/W_Ns (the d rho / d Y_j factor, Eq. 51); g_c = 1 where
                                //        gamma_r applies (1 <= c < ns), else 0; c = 0 and c = ns: zeros
    const double *wrow;         // [ns+1] row factors by Jacobian row r: {1, W_0 .. W_{ns-1}}
    const double *nasa;         // [2][5][ns] a_0..a_4, range-major, coefficient-major (coalesced over k)
    const double *t_mid;        // [ns]
    // ---- reaction tables, sorted order
    int n_pd;                   // pressure-dependent reactions (third body, falloff, chem. activated): [0, n_pd)
    int n_pk;                   // PLOG / Chebyshev reactions: [n_pd, n_pd + n_pk)
    int n_rchunk;               // groups of 32 reactions
    int split_general;          // 1: the group that holds reaction n_pd is two work items (pressure-dependent lanes /
                                // the others).  Shortens the longest item; set when one CTA per SM leaves the
                                // reaction queue latency-bound (cfg2: 10.51 -> 10.23 ms), not otherwise (cfg1:
                                // 2.69 -> 2.83 ms, the extra item costs issue slots the other CTA would use)
    int n_plain;                // the last n_plain groups hold only plain reactions
    const uint32_t *rchunk;     // [n_rchunk] 1 = every reaction of the group takes the plain path
    const uint4 *slots;         // [nr] {spec0|spec1<<16, spec2|spec3<<16, spec4|spec5<<16, meta}
    const uint4 *vidx;          // [nr] E indices of the slots' s'_ij: {v0|v1<<16, v2|v3<<16, v4|v5<<16, 0}
                                //      (empty slots point at the dump slot)
    const double *lnA, *beta, *Ta;               // [nr] forward Arrhenius (k_inf for falloff forms)
    const int32_t *rxn_orig;    // [nr] caller's reaction index
    const double *rev_lnA, *rev_beta, *rev_Ta;   // [nr] explicit reverse parameters
    const uint32_t *th_off;     // [nr] offset into th_data
    const double *th_data;      // per reaction: n_int, (n_int - 1) ascending breakpoints, n_int x {g_0..g_6}:
                                // sum_k nu_ki B_k(T) = g0 + g1 ln T + T (g2 + T (g3 + T (g4 + T g5))) + g6 / T
                                // (Eq. 27 summed over the reaction, one set per interval between the t_mid of
                                // its species; g0 includes (sum nu) ln(p_atm / R) of Eq. 26)
    double brk_common;          // the breakpoint every reaction shares (all n_int <= 2, one t_mid), else NaN
    const double *th_soa;       // [15][nr] the same for reactions with n_int <= 2, coalesced over reactions:
                                // row 0 the breakpoint (+inf if n_int = 1), rows 1..7 g of the lower interval,
                                // rows 8..14 g of the upper one
    const double *lo_lnA, *lo_beta, *lo_Ta;      // [n_pd] k_0
    const double *fall_par;                      // [n_pd][5]; Troe: {a, 1/T***, 1/T*, T**, has T**}; SRI: {a, b, 1/c, d, e}
    const int32_t *eff_base;    // [general groups + 1] first efficiency entry of a group of 32 reactions
    const uint4 *eff_ent;       // entry e of lane l of group c at [eff_base[c] + 32 e + l]: {species of alpha_ij != 1
                                // (or the single species) | E index of its term << 16, 0, alpha_ij - 1 (fp64 bits;
                                // 1 for the single species)}; padded with {dummy species | dump slot << 16, 0, 0.0}
    const int32_t *pk_ptr;      // [n_pk+1] offsets into pk_data
    const double *pk_data;      // PLOG: n, then n x {p, ln p, ln A, beta, Ta};
                                // Chebyshev: nT, nP, 1/Tmin, 1/Tmax, log10 pmin, log10 pmax, eta[nT*nP]
    // ---- gathers: chunks of 32 lanes, 32 >> rshift sums each, sorted by length at create time.
    // Chunks [0, n_a1) are the A1 phase (the first n_a1_01 of them serve rates / dydt too); the
    // chunks of the cells of column panel p are [panel_ptr[p], panel_ptr[p+1]).
    int n_a1, n_a1_01;
    const uint2 *achunk;        // {first block of a_ent, steps | kind << 16 | rshift << 20 | sums per lane << 24}
    const uint4 *a_ent;         // block r of a chunk = a_ent[first + 32 r + lane].  One sum per lane: block 0 =
                                // {output E index (kAuxT3: species k; ~0 = none), constant factor (fp64 bits, 2
                                // words), entry of step 0}; block r >= 1: the entries of steps 4r-3 .. 4r.  Two
                                // sums A, B per lane (kAuxS1 only): blocks 0 and 1 are the records of A and B,
                                // block r >= 2 = {A, B of step 2r-3, A, B of step 2r-2}
    const int32_t *panel_ptr;   // [n_panel + 1]
    // ---- the tile: column panels of the Jacobian, state-interleaved like E, element (r, c) of
    // panel p at E index eTile + (p % nbuf) * pw * ld + (c - p * pw) * ld + r
    int n_panel, pw, nbuf;
    int eTile;
    int pair;                   // 1: ld is even, the DENSE pass owns two rows per lane (16-byte stores)
    int d_seg;                  // columns per DENSE work item
    int n_slab;                 // slabs of rows of the DENSE pass: 64 rows each if pair, else 32
    // ---- regions of E (indices in doubles per state)
    int eQ;                     // [nr][3] {q_i, a_i + W q_i, Theta_dT,i}
    int eH;                     // [nr] reaction enthalpy H_i
    int eAlpha, eGamma;         // [ns+1] by Jacobian row; row 0 stays 0
    int eWdot;                  // [ns]
    int eG0;                    // [ns]   sum_i H_i s'_ij per column species j
    int eZ;                     // [ns+1] finished energy row J(0, c)
    int eS1, eA0, eS4;          // scalars: sum_i H_i q_i, sum_i H_i a_i, sum_i H_i Theta_i
    int eZero;                  // a slot that stays 0 (padding of the lists)
    int eDump;                  // a slot nobody reads (stores of empty reaction slots)
    int n_e;                    // size of E without the tile
};

// per-state scalars (region Scal of the shared-memory plan)
enum {
    kT = 0, kLnT, kInvT, kP, kLnP, kRho, kIrho, kW, kM, kCpMix, kDcpDT, kIcp, kNScal = 12
};

// Shared-memory plan (offsets in doubles PER STATE).  A CTA evaluates S states at a time and
// interleaves them: element i of region R of state q lives at (R + i) * S + q.  The mixture block
// (X, Cp, Scal) exists twice: the block of the next batch is filled while this one is in use.  After
// the S interleaved state blocks come the state-independent tables (colc, wrow), loaded once per CTA.
struct SmemPlan {
    int E;                              // [n_e + tile]
    int P0;                             // three mixture blocks of p0size doubles
    int p0size;
    int oX;                             // within a mixture block: [ns+1] concentrations; slot ns = 1 (empty reaction slots)
    int oCp;                            // [ns] c_pk (mass based)
    int oScal;                          // [kNScal]
    int total;                          // doubles per state
    int colc;                           // [ld][2], offset in doubles from the end of the state blocks
    int wrow;                           // [ld]
    int shared_total;                   // doubles of the state-independent part
};

inline SmemPlan make_smem_plan(int ns, int n_e)
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
        p.oScal = take(kNScal) - base;
        p.p0size = o - base;
        o += 2 * p.p0size;
    }
    p.total = o;
    o = 0;
    p.colc = take(2 * (ns + 1));
    p.wrow = take(ns + 1);
    p.shared_total = o;
    return p;
}

}  // namespace pyjac
