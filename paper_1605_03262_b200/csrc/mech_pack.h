// mech_pack.h -- host-side packing of a pyjac_mech_desc into the SoA tables of device_mech.h.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/pyjac_b200.h"

namespace pyjac {

struct HostPack {
    int ns = 0, nr = 0;
    std::vector<double> mw, inv_mw, dcol, colc, wrow, nasa, t_mid;
    std::vector<double> lnA, beta, Ta, rev_lnA, rev_beta, rev_Ta;
    std::vector<uint32_t> slots;          // 4 words per reaction
    std::vector<uint32_t> vbase;
    std::vector<int32_t> rxn_orig;
    int pd_begin = 0, n_pd = 0;
    std::vector<double> lo_lnA, lo_beta, lo_Ta, fall_par;
    std::vector<int32_t> tb_spec, eff_ptr, eff_spec;
    std::vector<double> eff_eps;
    std::vector<uint32_t> eff_vbase;
    int pk_begin = 0, n_pk = 0;
    std::vector<int32_t> pk_ptr;
    std::vector<double> pk_data;
    int n_spchunk = 0;
    std::vector<uint32_t> spchunk, sp_ent;      // uint2 pairs flattened
    std::vector<int32_t> sptask_k;
    int n_panel = 1, pw = 0, ldt = 0;
    std::vector<int32_t> panel_chunks;          // int2 pairs flattened
    std::vector<uint32_t> cchunk, ctask_addr, c_ent;
    int n_v = 0;
};

// Returns PYJAC_OK, PYJAC_EINVAL or PYJAC_ELIMIT.  `why` (optional) receives a static message.
// smem_budget: bytes of shared memory one CTA may use (decides the column-panel width);
// panel_override > 0 forces that many column panels (tuning).
int pack_mechanism(const pyjac_mech_desc *d, HostPack &out, size_t smem_budget, int panel_override,
                   const char **why);

}  // namespace pyjac
