// mech_pack.h -- host-side packing of a pyjac_mech_desc into the tables of device_mech.h.
#pragma once
#include <cstdint>
#include <utility>
#include <vector>

#include "../../include/pyjac_b200.h"

namespace pyjac {

struct HostPack {
    int ns = 0, nr = 0;
    std::vector<double> inv_mw, mw, colc, wrow, nasa, t_mid;
    int n_pd = 0, n_pk = 0;
    std::vector<uint32_t> rchunk;         // per group of 32 reactions: the P1 path (device_mech.h `p1item`)
    std::vector<uint32_t> p1item;
    std::vector<uint32_t> slots;          // 4 words per reaction
    std::vector<uint32_t> vidx;           // 4 words per reaction
    std::vector<double> lnA, beta, Ta, rev_lnA, rev_beta, rev_Ta;
    std::vector<int32_t> rxn_orig;
    std::vector<uint32_t> th_off;
    std::vector<double> th_data, th_soa, th_brk;
    double brk_common = 0.0;              // NaN unless every reaction has at most two intervals and one breakpoint
    std::vector<double> lo_lnA, lo_beta, lo_Ta, fall_par;
    std::vector<int32_t> eff_ptr;
    std::vector<uint32_t> eff_spec;
    std::vector<double> eff_eps;
    std::vector<int32_t> eff_base;        // per general group
    std::vector<uint32_t> eff_ent;        // uint4 flattened
    std::vector<int32_t> pk_ptr;
    std::vector<double> pk_data;
    int n_rchunk = 0;
    // phase A chunks in rows of NW (device_mech.h); rows [0, n_arow01) serve the rates / dydt kernels too
    int n_arow = 0, n_arow01 = 0;
    std::vector<uint32_t> achunk;         // uint2 flattened
    std::vector<uint32_t> a_ent;          // uint4 flattened
    // phase B items, one per (slab, column)
    int rp = 1, n_slab = 1;
    std::vector<uint32_t> b_ent;          // uint4 flattened
    std::vector<int32_t> bsplit;          // [NW + 1]
    int eQ = 0, eH = 0, eAlpha = 0, eGamma = 0, eTc = 0, eWdot = 0, eG0 = 0;
    int eS1 = 0, eA0 = 0, eS4 = 0, eZero = 0, eDump = 0, eHs = 0, n_e = 0;
    // launch shape chosen with the tables: S states per CTA iteration, threads per CTA, the CTAs per SM
    // the shared-memory footprint was sized for
    int S = 1, threads = 128, ctas_target = 1;
    bool stage = false;                   // gather tables staged in shared memory
    // only with ShapeHints::keep_cells: per flat cell index r + c * ld the (E index, integer coefficient) pairs summed into
    // the cell, before any splitting or piecewise summing (the gather probe of tools.cu deals them out its own way)
    std::vector<std::vector<std::pair<uint32_t, int>>> raw_cells;
    // statistics (pyjac_pack_stats)
    long long n_cell_entries = 0, n_cells = 0, n_heavy_cells = 0, n_heavy_pieces = 0, n_a_steps = 0, n_b_steps = 0;
    long long n_plain_chunks = 0;
    long long n_a_steps_kind[4] = {0, 0, 0, 0};     // phase-A steps by chunk kind
    long long n_layout_excess[2] = {0, 0};          // bank-group excess of the gather groups before / after the layout search
    long long n_conflict_wf[2] = {0, 0};            // shared-memory wavefronts beyond one per lane group and step that the
                                                    // placement leaves (phase A, phase B; model of mech_pack.cu `place`)
};

// What the launch-shape choice may use (filled from the device properties and a pyjac_launch_shape;
// 0 = choose).
struct ShapeHints {
    long long smem_bytes = 227 * 1024 - 1024;   // dynamic shared memory one CTA may use
    int S = 0, threads = 0, ctas = 0;
    int cap = 0;        // longest list one lane walks in phase A
    int cell_cap = 0;   // longest Jacobian-cell list gathered in phase B (1..3); longer ones are summed piecewise in phase A
    int rp = 0;         // rows per lane in phase B (1 or 2)
    int p1_states = 0;  // states per work item of the fast reaction path (0: all S)
    int stage = 0;      // 1: copy the gather tables of phases A and B to shared memory once per CTA
    int layout = 0;     // 2: keep the s' values in allocation order (no bank-aware layout of E)
    int keep_cells = 0; // 1: also return the raw contribution lists of the Jacobian cells (HostPack::raw_cells; probes only)
};

// The hints of an explicit launch shape (NULL: all zeros = choose); `smem_optin` = the device's opt-in
// shared memory per CTA (0: the architecture's 227 KB).
ShapeHints hints_from_shape(const pyjac_launch_shape *shape, long long smem_optin);

// Returns PYJAC_OK, PYJAC_EINVAL or PYJAC_ELIMIT.  `why` (optional) receives a static message.
int pack_mechanism(const pyjac_mech_desc *d, HostPack &out, const ShapeHints &hints, const char **why);

}  // namespace pyjac
