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
    std::vector<double> lo_lnA, lo_beta, lo_Ta, fall_par;
    std::vector<int32_t> eff_ptr;
    std::vector<uint32_t> eff_spec;
    std::vector<double> eff_eps;
    std::vector<int32_t> pk_ptr;
    std::vector<double> pk_data;
    int n_rchunk = 0;
    int n_achunk = 0, n_achunk01 = 0;
    std::vector<uint32_t> achunk;         // uint4 flattened
    std::vector<uint32_t> a_ent, a_out;
    std::vector<double> a_const;
    int n_slab = 0;
    std::vector<uint32_t> m_hdr;          // [n_slab][ns+1]
    std::vector<uint32_t> m_ent;          // blocks of 32 lanes x 4 entries
    int eQ = 0, eAr = 0, eTh = 0, eH = 0, eAlpha = 0, eGamma = 0, eWdot = 0, eTcol = 0, eG0 = 0, eZ = 0;
    int eS1 = 0, eA0 = 0, eS4 = 0, eZero = 0, eDump = 0, n_e = 0;
    // statistics (pyjac_pack_stats)
    long long n_main_entries = 0, n_aux_entries = 0, n_list_entries = 0, n_plain_chunks = 0;
};

// Returns PYJAC_OK, PYJAC_EINVAL or PYJAC_ELIMIT.  `why` (optional) receives a static message.
// smem_doubles: doubles of shared memory one state may use for E (decides how many of the
// Jacobian's cell lists are summed by AUX tasks instead of inline in the MAIN pass).
int pack_mechanism(const pyjac_mech_desc *d, HostPack &out, long long smem_doubles, const char **why);

}  // namespace pyjac
