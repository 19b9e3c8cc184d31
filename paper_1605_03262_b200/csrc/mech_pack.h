// mech_pack.h -- host-side packing of a pyjac_mech_desc into the tables of device_mech.h.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/pyjac_b200.h"

namespace pyjac {

struct HostPack {
    int ns = 0, nr = 0;
    std::vector<double> inv_mw, mw, colc, wrow, nasa, t_mid;
    int n_pd = 0, n_pk = 0;
    std::vector<uint32_t> rchunk;
    std::vector<uint32_t> slots;          // 4 words per reaction
    std::vector<uint32_t> vidx;           // 4 words per reaction
    std::vector<double> lnA, beta, Ta, rev_lnA, rev_beta, rev_Ta;
    std::vector<int32_t> rxn_orig;
    std::vector<uint32_t> th_off;
    std::vector<double> th_data, th_soa;
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
    // gathers (device_mech.h): A1 chunks first, then the cell chunks panel by panel
    int n_a1 = 0, n_a1_01 = 0;
    std::vector<uint32_t> achunk;         // uint2 flattened
    std::vector<uint32_t> a_ent;          // uint4 flattened
    std::vector<int32_t> panel_ptr;       // [n_panel + 1]
    int n_panel = 1, pw = 0, nbuf = 1, eTile = 0, pair = 0, d_seg = 3;
    int eQ = 0, eH = 0, eAlpha = 0, eGamma = 0, eWdot = 0, eG0 = 0, eZ = 0;
    int eS1 = 0, eA0 = 0, eS4 = 0, eZero = 0, eDump = 0, n_e = 0;
    // launch shape chosen with the tables: S states per CTA iteration, threads per CTA, the CTAs
    // per SM the shared-memory footprint was sized for
    int S = 1, threads = 128, ctas_target = 1;
    // statistics (pyjac_pack_stats)
    long long n_cell_entries = 0, n_cell_steps = 0, n_a1_steps = 0, n_cells = 0, n_plain_chunks = 0;
};

// What the launch-shape choice may use (api.cu fills it from the device properties and the
// PYJAC_S / PYJAC_THREADS / PYJAC_PW / PYJAC_CTAS tuning hooks; 0 = choose).
struct ShapeHints {
    long long smem_bytes = 227 * 1024 - 1024;   // dynamic shared memory one CTA may use
    int S = 0, threads = 0, pw = 0, ctas = 0, cap = 0, seg = 0;      // cap: longest list one lane walks; seg: columns per DENSE item
};

// Returns PYJAC_OK, PYJAC_EINVAL or PYJAC_ELIMIT.  `why` (optional) receives a static message.
int pack_mechanism(const pyjac_mech_desc *d, HostPack &out, const ShapeHints &hints, const char **why);

}  // namespace pyjac
