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
constexpr int kLongCell = 3;               // cells with more contributions are pre-reduced (phase 2)

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
    // ---- phase-2 gather tasks (fixed summation order)
    int n_sp_task;              // = ns: species sums over reactions (wdot, A, Tcol)
    const int32_t *sp_ptr;      // [ns+1]
    const uint32_t *sp_ent;     // entries: reaction (sorted) | coef16 (net nu_ki)
    const int32_t *col_ptr;     // [ns+1] energy-row column sums: entries (V index | reaction<<16)
    const uint32_t *col_ent;
    int n_long;                 // pre-reduced cells (incl. every cell of the virtual column Ns)
    const int32_t *long_ptr;    // [n_long+1]
    const uint32_t *long_ent;   // entries: V index | coef16
    // ---- phase-4 cell lists: cell (r, c), r, c in 0..ns, at r + c*ld
    const uint32_t *cell_info;  // [ld*ld] offset<<3 | count (count <= kLongCell)
    const uint32_t *cell_ent;   // entries: V index | coef16
    // ---- sizes of the per-state shared-memory arrays
    int n_v;                    // per-reaction derivative entries s'_ij (phase 1 output)
    int n_vext;                 // n_v + n_long + 1 (a zero slot)
    int spns_base;              // V-ext index of the (k, Ns) sums, k = 0..ns-1
};

// Shared-memory plan of one CTA (doubles).  Every array is per state.
struct SmemPlan {
    int X, B, dB, HW, Cp, dCp;          // [ns+1] species arrays (slot ns is the empty-slot dummy)
    int Wdot, A, Tc, E, WA, Row0, Col0; // [ns+1]
    int Q, Ar, Th, H;                   // [nr]
    int V;                              // [n_vext]
    int Red;                            // [8][32] reduction scratch
    int Scal;                           // [16] per-state scalars
    int total;                          // doubles
};

inline SmemPlan make_smem_plan(int ns, int nr, int n_vext)
{
    SmemPlan p{};
    int o = 0;
    auto take = [&](int n) { int r = o; o += (n + 1) & ~1; return r; };
    const int s1 = ns + 1;
    p.X = take(s1); p.B = take(s1); p.dB = take(s1); p.HW = take(s1); p.Cp = take(s1); p.dCp = take(s1);
    p.Wdot = take(s1); p.A = take(s1); p.Tc = take(s1); p.E = take(s1); p.WA = take(s1);
    p.Row0 = take(s1); p.Col0 = take(s1);
    p.Q = take(nr); p.Ar = take(nr); p.Th = take(nr); p.H = take(nr);
    p.V = take(n_vext);
    p.Red = take(8 * 32);
    p.Scal = take(16);
    p.total = o;
    return p;
}

}  // namespace pyjac
