// device_mech.h -- device-resident SoA tables of one kinetic model and the shared-memory plan of
// the evaluation kernels.  Built by mech_pack.cpp (host), consumed by kernels.cu (device).
//
// Notation follows the paper (PAPER.md Sections 2-4): species k, reaction i, nu' / nu'' the
// reactant / product coefficients (Eq. 15), [X_k] concentrations (Eq. 5), c_i the pressure
// modification (Eq. 20).  Reactions are stored in a SORTED order (grouped by type so that a warp
// evaluates one rate form); `rxn_orig` maps back to the caller's order.
#pragma once
#include <cstdint>

namespace pyjac {

constexpr double kRu = 8314.46261815324;   // J kmol^-1 K^-1
constexpr double kPatm = 101325.0;         // Pa
constexpr int kMaxSide = 3;                // species per reaction side
constexpr int kSpLanes = 4;                // lanes that share one species task

// meta word of a reaction: bits 0..23 six 4-bit nu (slots 0-2 reactants, 3-5 products; 0 = empty
// slot), 24..26 rxn_type, 27..28 rev_type, 29..30 falloff_form, 31 third body is a single species.
__host__ __device__ inline int meta_nu(uint32_t m, int slot) { return (m >> (4 * slot)) & 0xF; }
__host__ __device__ inline int meta_type(uint32_t m) { return (m >> 24) & 7; }
__host__ __device__ inline int meta_rev(uint32_t m) { return (m >> 27) & 3; }
__host__ __device__ inline int meta_form(uint32_t m) { return (m >> 29) & 3; }
__host__ __device__ inline int meta_single(uint32_t m) { return (m >> 31) & 1; }

// A gather entry: low 16 bits = source index, high 16 bits = the top 16 bits of the fp64
// coefficient (exact for +-1, +-2, +-3: the only stoichiometric factors that occur).
__host__ __device__ inline uint32_t pack_entry(uint32_t src, int coef)
{
    // 1.0 = 0x3FF0.., 2.0 = 0x4000.., 3.0 = 0x4008..; sign in bit 15
    uint32_t a = coef < 0 ? uint32_t(-coef) : uint32_t(coef);
    uint32_t hi = a == 1 ? 0x3FF0u : a == 2 ? 0x4000u : a == 3 ? 0x4008u
                : a == 4 ? 0x4010u : a == 5 ? 0x4014u : a == 6 ? 0x4018u : 0u;
    if (coef < 0) hi |= 0x8000u;
    return (hi << 16) | (src & 0xFFFFu);
}

struct DeviceMech {
    int ns, nr;                 // N_sp, N_reac
    int ld;                     // N_sp + 1
    double ln_patm_over_R;      // ln(p_atm / R) of Eq. 26
    // ---- species tables
    const double *mw;           // [ns]
    const double *inv_mw;       // [ns]
    const double *dcol;         // [ns] d_j = 1/W_j - 1/W_Ns  (the d rho / d Y_j factor, Eq. 51)
    const double2 *colc;        // [ns] {d_j, 1/W_j}: the two column constants of phase 4
    const double *wrow;         // [ns+2] row factors of phase 4: {1, W_0 .. W_{ns-1}, 1}
    const double *nasa;         // [2][7][ns]  range-major, coefficient-major (coalesced over k)
    const double *t_mid;        // [ns]
    // ---- reaction tables, sorted order
    const double *lnA, *beta, *Ta;        // [nr] forward Arrhenius (k_inf for falloff forms)
    const uint4 *slots;                   // [nr] {spec0|spec1<<16, spec2|spec3<<16, spec4|spec5<<16, meta}
    const uint32_t *vbase;                // [nr] first V entry (reactant slots, then product slots)
    const int32_t *rxn_orig;              // [nr] caller's reaction index
    const double *rev_lnA, *rev_beta, *rev_Ta;   // [nr] explicit reverse parameters
    // pressure-dependent reactions occupy sorted indices [pd_begin, nr); tables indexed by s - pd_begin
    int pd_begin, n_pd;
    const double *lo_lnA, *lo_beta, *lo_Ta;      // [n_pd] k_0
    const double *fall_par;                      // [n_pd][5]
    const int32_t *tb_spec;                      // [n_pd] single species or -1
    const int32_t *eff_ptr;                      // [n_pd+1]
    const int32_t *eff_spec;                     // species of alpha_ij != 1 (or the single species)
    const double *eff_eps;                       // alpha_ij - 1      (1 for the single species)
    const uint32_t *eff_vbase;                   // [n_pd] first V entry of the efficiency terms
    // PLOG / Chebyshev reactions occupy sorted indices [pk_begin, pk_begin + n_pk)
    int pk_begin, n_pk;
    const int32_t *pk_ptr;      // [n_pk+1] offsets into pk_data
    const double *pk_data;      // PLOG: n, then n x {p, ln p, ln A, beta, Ta};
                                // Chebyshev: nT, nP, 1/Tmin, 1/Tmax, log10 pmin, log10 pmax, eta[nT*nP]
    // ---- species tasks: wdot_k, A_k, Tcol_k and the diagonal cell (k, k) are sums over the
    // reactions that contain k.  kSpLanes lanes share one species; a chunk is 32 / kSpLanes species.
    int n_spchunk;
    const uint2 *spchunk;       // [n_spchunk] {first entry, steps}; entries at [first + step*32 + lane]
    const int32_t *sptask_k;    // [n_spchunk * 32 / kSpLanes] species or -1
    const uint2 *sp_ent;        // {reaction (sorted) | coef16, V index | coef16}
    // ---- cell tasks: the off-diagonal cells (k, j) of the species block that collect at least
    // one reaction, per column panel, sorted by list length (descending); 32 tasks per chunk.
    int n_panel, pw, ldt;       // panels of pw columns; tile leading dimension (even, rows r = k + 1)
    const int2 *panel_chunks;   // [n_panel] {first chunk, one past last}
    const uint2 *cchunk;        // {first entry, steps}; entries at [first + step*32 + lane]
    const uint32_t *ctask_addr; // [n_chunk*32] tile offset (k + 1) + (j - j0)*ldt (pad: ldt*pw)
    const uint32_t *c_ent;      // V index | coef16 (pad: zero slot n_v, coefficient 0)
    int n_v;                    // per-reaction derivative entries s'_ij; V[n_v] is a zero slot
};

// Shared-memory plan of ONE state (offsets in doubles).  A CTA that evaluates S states at a time
// holds S such blocks back to back (stride `total`).
struct SmemPlan {
    int Sp4;                            // [ns+1][4] {[X_k], B_k, dB_k/dT, h_k W_k}; slot ns = {1, 0, 0, 0}
    int Cp;                             // [ns+1] c_pk
    int Wdot, A, Tc, Diag;              // [ns+1] indexed by species k
    int WA, WC;                         // [ns+2] indexed by row r = k + 1; slot 0 is zero (energy row)
    int Ep;                             // [kEParts][ns+1] partial energy-row column sums
    int Col0;                           // [ns+1] column 0 (d/dT) by row
    int Q, Ar, Th;                      // [nr+1] (slot nr stays zero: padding of the gather lists)
    int V;                              // [n_v+1]
    int Tile;                           // [ldt*pw + 2]
    int Scal;                           // [16] per-state scalars, see kernels.cu
    int total;                          // doubles per state
};

constexpr int kEParts = 4;

inline SmemPlan make_smem_plan(int ns, int nr, int n_v, int ldt, int pw)
{
    SmemPlan p{};
    int o = 0;
    auto take = [&](int n) { int r = o; o += (n + 1) & ~1; return r; };
    const int s1 = ns + 1;
    p.Sp4 = take(4 * s1); p.Cp = take(s1);
    p.Wdot = take(s1); p.A = take(s1); p.Tc = take(s1); p.Diag = take(s1); p.WA = take(s1 + 1); p.WC = take(s1 + 1);
    p.Ep = take(kEParts * s1);
    p.Col0 = take(s1);
    p.Q = take(nr + 1); p.Ar = take(nr + 1); p.Th = take(nr + 1);
    p.V = take(n_v + 1);
    p.Tile = take(ldt * pw + 2);
    p.Scal = take(16);
    p.total = o;
    return p;
}

}  // namespace pyjac
