// mech_pack.h -- host-side packing of a pyjac_mech_desc into the SoA tables of device_mech.h.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/pyjac_b200.h"

namespace pyjac {

struct HostPack {
    int ns = 0, nr = 0;
    std::vector<double> mw, inv_mw, dcol, nasa, t_mid;
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
    std::vector<int32_t> sp_ptr, col_ptr, long_ptr;
    std::vector<uint32_t> sp_ent, col_ent, long_ent, cell_info, cell_ent;
    int n_long = 0, n_v = 0, n_vext = 0, spns_base = 0;
};

// Returns PYJAC_OK, PYJAC_EINVAL or PYJAC_ELIMIT.  `why` (optional) receives a static message.
int pack_mechanism(const pyjac_mech_desc *d, HostPack &out, const char **why);

}  // namespace pyjac
