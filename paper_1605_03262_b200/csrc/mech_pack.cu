// mech_pack.cu -- validate a pyjac_mech_desc and pack it into the device table layout (host code).
//
// What is precomputed here is state-independent bookkeeping of the paper's restructured evaluation
// order (Algorithm 2): which per-reaction products feed which Jacobian entries.
// No thermodynamic or kinetic quantity is evaluated on the host except ln A and ln p of the tables.
#include <algorithm>
#include <cmath>
#include <numeric>

#include "device_mech.h"
#include "mech_pack.h"

namespace pyjac {

namespace {

struct Fail {
    int code;
    const char *why;
};

#define REQUIRE(cond, msg)                        \
    do {                                          \
        if (!(cond)) throw Fail{PYJAC_EINVAL, msg}; \
    } while (0)

struct ColEntry {
    int spec;      // column species j
    uint32_t vi;   // V index of s'_ij
};

}  // namespace

static void pack_impl(const pyjac_mech_desc *d, HostPack &o, size_t smem_budget, int panel_override)
{
    REQUIRE(d != nullptr, "description is NULL");
    const int ns = d->n_species, nr = d->n_reactions;
    REQUIRE(ns >= 1 && nr >= 0, "n_species must be >= 1 and n_reactions >= 0");
    if (ns > 65534 || nr > 65534) throw Fail{PYJAC_ELIMIT, "more than 65534 species or reactions"};
    REQUIRE(d->mol_wt && d->nasa_lo && d->nasa_hi && d->t_mid, "species arrays missing");
    if (nr > 0) {
        REQUIRE(d->reac_ptr && d->prod_ptr && d->rxn_type && d->rev_type && d->arr_hi && d->arr_lo &&
                    d->arr_rev && d->falloff_form && d->falloff_par && d->tb_species && d->eff_ptr &&
                    d->plog_ptr && d->cheb_ptr && d->cheb_nT && d->cheb_nP && d->cheb_lim,
                "per-reaction arrays missing");
    }
    o.ns = ns;
    o.nr = nr;
    // ---- species
    o.mw.assign(d->mol_wt, d->mol_wt + ns);
    o.inv_mw.resize(ns);
    o.dcol.resize(ns);
    o.t_mid.assign(d->t_mid, d->t_mid + ns);
    o.nasa.resize((size_t)14 * ns);
    for (int k = 0; k < ns; ++k) {
        REQUIRE(d->mol_wt[k] > 0.0 && std::isfinite(d->mol_wt[k]), "molecular weight must be positive");
        o.inv_mw[k] = 1.0 / d->mol_wt[k];
        for (int c = 0; c < 7; ++c) {
            o.nasa[(size_t)(0 * 7 + c) * ns + k] = d->nasa_lo[7 * k + c];
            o.nasa[(size_t)(1 * 7 + c) * ns + k] = d->nasa_hi[7 * k + c];
        }
    }
    for (int k = 0; k < ns; ++k) o.dcol[k] = 1.0 / d->mol_wt[k] - 1.0 / d->mol_wt[ns - 1];
    o.wrow.assign((size_t)ns + 2, 1.0);
    for (int k = 0; k < ns; ++k) o.wrow[k + 1] = d->mol_wt[k];
    o.colc.resize((size_t)2 * ns);
    for (int k = 0; k < ns; ++k) { o.colc[2 * k] = o.dcol[k]; o.colc[2 * k + 1] = o.inv_mw[k]; }

    // ---- validate reactions and choose the sorted order
    std::vector<int> key(nr);
    for (int i = 0; i < nr; ++i) {
        const int t = d->rxn_type[i], rv = d->rev_type[i];
        REQUIRE(t >= 0 && t <= 5, "rxn_type out of range");
        REQUIRE(rv >= 0 && rv <= 2, "rev_type out of range");
        for (int side = 0; side < 2; ++side) {
            const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
            const int32_t *sp = side ? d->prod_spec : d->reac_spec;
            const int32_t *nu = side ? d->prod_nu : d->reac_nu;
            const int b = ptr[i], e = ptr[i + 1];
            REQUIRE(b >= 0 && e >= b, "stoichiometry CSR pointers must be non-decreasing");
            REQUIRE(e - b <= kMaxSide, "more than 3 species on one side of a reaction");
            REQUIRE(e == b || (sp && nu), "stoichiometry arrays missing");
            for (int q = b; q < e; ++q) {
                REQUIRE(sp[q] >= 0 && sp[q] < ns, "species index out of range");
                REQUIRE(nu[q] >= 1 && nu[q] <= 3, "stoichiometric coefficient outside 1..3");
                for (int q2 = b; q2 < q; ++q2) REQUIRE(sp[q2] != sp[q], "species repeated within a side");
            }
        }
        int form = 0;
        if (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED) {
            form = d->falloff_form[i];
            REQUIRE(form >= 0 && form <= 2, "falloff_form out of range");
            REQUIRE(d->arr_lo[3 * i] > 0.0 && d->arr_hi[3 * i] > 0.0, "falloff pre-exponentials must be > 0");
        }
        if (t == PYJAC_ELEMENTARY || t == PYJAC_THIRD_BODY)
            REQUIRE(d->arr_hi[3 * i] > 0.0, "pre-exponential factor must be > 0");
        if (rv == PYJAC_REV_EXPLICIT) REQUIRE(d->arr_rev[3 * i] > 0.0, "reverse pre-exponential must be > 0");
        if (t == PYJAC_THIRD_BODY || t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED) {
            const int m = d->tb_species[i];
            REQUIRE(m >= -1 && m < ns, "tb_species out of range");
            const int b = d->eff_ptr[i], e = d->eff_ptr[i + 1];
            REQUIRE(b >= 0 && e >= b, "efficiency CSR pointers must be non-decreasing");
            REQUIRE(e == b || (d->eff_spec && d->eff_val), "efficiency arrays missing");
            for (int q = b; q < e; ++q) {
                REQUIRE(d->eff_spec[q] >= 0 && d->eff_spec[q] < ns, "efficiency species out of range");
                for (int q2 = b; q2 < q; ++q2)
                    REQUIRE(d->eff_spec[q2] != d->eff_spec[q], "efficiency species repeated");
            }
        }
        if (t == PYJAC_PLOG) {
            const int b = d->plog_ptr[i], e = d->plog_ptr[i + 1];
            REQUIRE(e - b >= 2 && d->plog_p && d->plog_arr, "PLOG reaction needs >= 2 pressures");
            for (int q = b; q < e; ++q) {
                REQUIRE(d->plog_p[q] > 0.0 && d->plog_arr[3 * q] > 0.0, "PLOG pressure and A must be > 0");
                if (q > b) REQUIRE(d->plog_p[q] > d->plog_p[q - 1], "PLOG pressures must ascend");
            }
        }
        if (t == PYJAC_CHEBYSHEV) {
            const int nT = d->cheb_nT[i], nP = d->cheb_nP[i];
            REQUIRE(nT >= 1 && nP >= 1 && d->cheb_eta, "Chebyshev table empty");
            REQUIRE(d->cheb_ptr[i + 1] - d->cheb_ptr[i] >= nT * nP, "Chebyshev table too short");
            const double *lim = d->cheb_lim + 4 * i;
            REQUIRE(lim[0] > 0 && lim[1] > lim[0] && lim[2] > 0 && lim[3] > lim[2], "Chebyshev limits invalid");
        }
        // group: elementary, PLOG, Chebyshev | third body, falloff forms (Lindemann, Troe, SRI)
        int group = t == PYJAC_ELEMENTARY ? 0 : t == PYJAC_PLOG ? 1 : t == PYJAC_CHEBYSHEV ? 2
                  : t == PYJAC_THIRD_BODY ? 3 : 4 + form;
        bool unit = true;
        for (int q = d->reac_ptr[i]; q < d->reac_ptr[i + 1]; ++q) unit = unit && d->reac_nu[q] == 1;
        for (int q = d->prod_ptr[i]; q < d->prod_ptr[i + 1]; ++q) unit = unit && d->prod_nu[q] == 1;
        int neff = 0;
        if (group >= 3) neff = d->tb_species[i] >= 0 ? 1 : d->eff_ptr[i + 1] - d->eff_ptr[i];
        // warps evaluate one rate form, one stoichiometry path and equally long efficiency lists
        key[i] = ((group * 2 + (unit ? 0 : 1)) * 4 + rv) * 64 + std::min(neff, 63);
    }
    std::vector<int> order(nr);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return key[a] < key[b]; });

    // ---- per-reaction tables in sorted order
    o.lnA.resize(nr); o.beta.resize(nr); o.Ta.resize(nr);
    o.rev_lnA.assign(nr, 0.0); o.rev_beta.assign(nr, 0.0); o.rev_Ta.assign(nr, 0.0);
    o.slots.assign((size_t)4 * nr, 0u);
    o.vbase.resize(nr);
    o.rxn_orig.resize(nr);
    o.pd_begin = nr; o.n_pd = 0; o.pk_begin = nr; o.n_pk = 0;
    o.pk_ptr.assign(1, 0);
    o.eff_ptr.assign(1, 0);
    std::vector<std::vector<ColEntry>> cols(nr);          // column entries of each reaction
    std::vector<std::vector<std::pair<int, int>>> net(nr);  // (species, net nu) of each reaction
    uint32_t nv = 0;
    for (int s = 0; s < nr; ++s) {
        const int i = order[s];
        const int t = d->rxn_type[i], rv = d->rev_type[i];
        o.rxn_orig[s] = i;
        const bool pk = (t == PYJAC_PLOG || t == PYJAC_CHEBYSHEV);
        const bool pd = (t == PYJAC_THIRD_BODY || t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED);
        if (pk && o.n_pk++ == 0) o.pk_begin = s;
        if (pd && o.n_pd++ == 0) o.pd_begin = s;
        if (!pk) {
            o.lnA[s] = std::log(d->arr_hi[3 * i]);
            o.beta[s] = d->arr_hi[3 * i + 1];
            o.Ta[s] = d->arr_hi[3 * i + 2];
        }
        if (rv == PYJAC_REV_EXPLICIT) {
            o.rev_lnA[s] = std::log(d->arr_rev[3 * i]);
            o.rev_beta[s] = d->arr_rev[3 * i + 1];
            o.rev_Ta[s] = d->arr_rev[3 * i + 2];
        }
        uint32_t spec[6] = {(uint32_t)ns, (uint32_t)ns, (uint32_t)ns, (uint32_t)ns, (uint32_t)ns, (uint32_t)ns};
        uint32_t meta = 0;
        o.vbase[s] = nv;
        for (int side = 0; side < 2; ++side) {
            const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
            const int32_t *sp = side ? d->prod_spec : d->reac_spec;
            const int32_t *nu = side ? d->prod_nu : d->reac_nu;
            for (int q = ptr[i], e = 0; q < ptr[i + 1]; ++q, ++e) {
                const int slot = 3 * side + e;
                spec[slot] = (uint32_t)sp[q];
                meta |= (uint32_t)nu[q] << (4 * slot);
                cols[s].push_back({sp[q], nv++});
                const int signed_nu = side ? nu[q] : -nu[q];
                bool found = false;
                for (auto &pr : net[s])
                    if (pr.first == sp[q]) { pr.second += signed_nu; found = true; }
                if (!found) net[s].push_back({sp[q], signed_nu});
            }
        }
        const int form = (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED) ? d->falloff_form[i] : 0;
        const int single = pd && d->tb_species[i] >= 0;
        meta |= (uint32_t)t << 24 | (uint32_t)rv << 27 | (uint32_t)form << 29 | (uint32_t)single << 31;
        o.slots[4 * s + 0] = spec[0] | spec[1] << 16;
        o.slots[4 * s + 1] = spec[2] | spec[3] << 16;
        o.slots[4 * s + 2] = spec[4] | spec[5] << 16;
        o.slots[4 * s + 3] = meta;
        if (pk) {
            if (t == PYJAC_PLOG) {
                const int b = d->plog_ptr[i], e = d->plog_ptr[i + 1];
                o.pk_data.push_back((double)(e - b));
                for (int q = b; q < e; ++q) {
                    o.pk_data.push_back(d->plog_p[q]);
                    o.pk_data.push_back(std::log(d->plog_p[q]));
                    o.pk_data.push_back(std::log(d->plog_arr[3 * q]));
                    o.pk_data.push_back(d->plog_arr[3 * q + 1]);
                    o.pk_data.push_back(d->plog_arr[3 * q + 2]);
                }
            } else {
                const int nT = d->cheb_nT[i], nP = d->cheb_nP[i];
                const double *lim = d->cheb_lim + 4 * i;
                o.pk_data.push_back((double)nT);
                o.pk_data.push_back((double)nP);
                o.pk_data.push_back(1.0 / lim[0]);
                o.pk_data.push_back(1.0 / lim[1]);
                o.pk_data.push_back(std::log10(lim[2]));
                o.pk_data.push_back(std::log10(lim[3]));
                for (int q = 0; q < nT * nP; ++q) o.pk_data.push_back(d->cheb_eta[d->cheb_ptr[i] + q]);
            }
            o.pk_ptr.push_back((int32_t)o.pk_data.size());
        }
    }
    // pressure-dependent tables (third-body efficiencies get their V entries after all slots)
    for (int s = o.pd_begin; s < o.pd_begin + o.n_pd; ++s) {
        const int i = order[s];
        const int t = d->rxn_type[i];
        const bool fall = (t != PYJAC_THIRD_BODY);
        o.lo_lnA.push_back(fall ? std::log(d->arr_lo[3 * i]) : 0.0);
        o.lo_beta.push_back(fall ? d->arr_lo[3 * i + 1] : 0.0);
        o.lo_Ta.push_back(fall ? d->arr_lo[3 * i + 2] : 0.0);
        for (int c = 0; c < 5; ++c) o.fall_par.push_back(fall ? d->falloff_par[5 * i + c] : 0.0);
        const int m = d->tb_species[i];
        o.tb_spec.push_back(m);
        o.eff_vbase.push_back(nv);
        if (m >= 0) {       // Eq. 30: [X]_i = [X_m]; one entry with "alpha - 1" = 1 and no [M] term
            o.eff_spec.push_back(m);
            o.eff_eps.push_back(1.0);
            cols[s].push_back({m, nv++});
        } else {            // Eq. 28 written as [M] + sum_j (alpha_ij - 1)[X_j]
            for (int q = d->eff_ptr[i]; q < d->eff_ptr[i + 1]; ++q) {
                if (d->eff_val[q] == 1.0) continue;
                o.eff_spec.push_back(d->eff_spec[q]);
                o.eff_eps.push_back(d->eff_val[q] - 1.0);
                cols[s].push_back({d->eff_spec[q], nv++});
            }
        }
        o.eff_ptr.push_back((int32_t)o.eff_spec.size());
    }
    if (o.n_pd == 0) o.pd_begin = nr;
    if (o.n_pk == 0) o.pk_begin = nr;
    o.n_v = (int)nv;

    if (o.n_v + 1 > 65535) throw Fail{PYJAC_ELIMIT, "more than 65534 per-reaction derivative entries"};
    const uint32_t zero_slot = (uint32_t)o.n_v;

    // ---- cells of the species block: (k, j) += nu_ki s'_ij  (Eqs. 112, 118-127); j = ns-1 is the
    // virtual column of the terms proportional to 1/W_Nsp
    std::vector<std::vector<uint32_t>> cell((size_t)ns * ns);   // [j][k]
    for (int s = 0; s < nr; ++s)
        for (auto &pr : net[s]) {
            if (pr.second == 0) continue;
            for (auto &ce : cols[s]) cell[(size_t)ce.spec * ns + pr.first].push_back(pack_entry(ce.vi, pr.second));
        }

    // ---- species tasks: wdot_k, A_k, Tcol_k = sum_i nu_ki {q_i, a_i, thetaT_i} (Eqs. 14, 111,
    // 115-117) and the diagonal cell (k, k); kSpLanes lanes per species, longest lists first
    {
        std::vector<std::vector<std::pair<uint32_t, uint32_t>>> lists(ns);
        for (int s = 0; s < nr; ++s)
            for (auto &pr : net[s]) {
                if (pr.second == 0) continue;
                const int k = pr.first;
                bool first = true;
                for (auto &ce : cols[s]) {
                    if (ce.spec != k) continue;
                    lists[k].push_back({first ? pack_entry((uint32_t)s, pr.second) : (uint32_t)nr,
                                        pack_entry(ce.vi, pr.second)});
                    first = false;
                }
                if (first) lists[k].push_back({pack_entry((uint32_t)s, pr.second), zero_slot});
            }
        std::vector<int> ord(ns);
        std::iota(ord.begin(), ord.end(), 0);
        std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return lists[a].size() > lists[b].size(); });
        const int per = 32 / kSpLanes;
        const int nchunk = (ns + per - 1) / per;
        o.sptask_k.assign((size_t)nchunk * per, -1);
        for (int c = 0; c < nchunk; ++c) {
            int steps = 0;
            for (int i = 0; i < per && c * per + i < ns; ++i) {
                const int k = ord[c * per + i];
                o.sptask_k[(size_t)c * per + i] = k;
                steps = std::max(steps, (int)((lists[k].size() + kSpLanes - 1) / kSpLanes));
            }
            const uint32_t base = (uint32_t)(o.sp_ent.size() / 2);
            o.spchunk.push_back(base);
            o.spchunk.push_back((uint32_t)steps);
            o.sp_ent.resize(o.sp_ent.size() + (size_t)2 * steps * 32, 0u);
            for (int st = 0; st < steps; ++st)
                for (int lane = 0; lane < 32; ++lane) {
                    const int i = lane / kSpLanes, sub = lane % kSpLanes;
                    uint32_t w0 = (uint32_t)nr, w1 = zero_slot;   // coefficient 0 on the zero slots
                    if (c * per + i < ns) {
                        const auto &lst = lists[ord[c * per + i]];
                        const size_t e = (size_t)st * kSpLanes + sub;
                        if (e < lst.size()) { w0 = lst[e].first; w1 = lst[e].second; }
                    }
                    o.sp_ent[2 * ((size_t)base + (size_t)st * 32 + lane) + 0] = w0;
                    o.sp_ent[2 * ((size_t)base + (size_t)st * 32 + lane) + 1] = w1;
                }
        }
        o.n_spchunk = nchunk;
    }

    // ---- cell tasks per column panel
    o.ldt = (ns + 1 + 1) & ~1;                 // rows r = 0..ns (r = k + 1), even
    if ((o.ldt & 3) == 0) o.ldt += 2;            // 2 (mod 4): 2-way instead of 4-way bank conflicts across columns
    {
        // shared memory that does not depend on the panel width (doubles), see make_smem_plan
        const SmemPlan fixed = make_smem_plan(ns, nr, o.n_v, o.ldt, 0);
        long long room = (long long)smem_budget / 8 - fixed.total;
        int pw = ns;
        if ((long long)o.ldt * ns > room) pw = (int)(room / o.ldt);
        if (panel_override > 0) pw = std::min(ns, (ns + panel_override - 1) / panel_override);
        if (pw < 1) throw Fail{PYJAC_ELIMIT, "per-state tables exceed the shared memory of one CTA"};
        if (pw < ns && pw > 8) pw &= ~3;
        o.pw = pw;
        o.n_panel = (ns + pw - 1) / pw;
    }
    const uint32_t pad_addr = (uint32_t)(o.ldt * o.pw);
    for (int p = 0; p < o.n_panel; ++p) {
        const int j0 = p * o.pw, j1 = std::min(ns, j0 + o.pw);
        std::vector<std::pair<int, int>> tasks;   // (j, k) with a non-empty list, off the diagonal
        for (int j = j0; j < j1; ++j)
            for (int k = 0; k < ns; ++k)
                if (k != j && !cell[(size_t)j * ns + k].empty()) tasks.push_back({j, k});
        std::stable_sort(tasks.begin(), tasks.end(), [&](const std::pair<int, int> &a, const std::pair<int, int> &b) {
            return cell[(size_t)a.first * ns + a.second].size() > cell[(size_t)b.first * ns + b.second].size();
        });
        o.panel_chunks.push_back((int32_t)(o.cchunk.size() / 2));
        for (size_t t0 = 0; t0 < tasks.size(); t0 += 32) {
            const int steps = (int)cell[(size_t)tasks[t0].first * ns + tasks[t0].second].size();
            const uint32_t base = (uint32_t)o.c_ent.size();
            o.cchunk.push_back(base);
            o.cchunk.push_back((uint32_t)steps);
            o.c_ent.resize(o.c_ent.size() + (size_t)steps * 32, zero_slot);
            for (int lane = 0; lane < 32; ++lane) {
                if (t0 + lane >= tasks.size()) { o.ctask_addr.push_back(pad_addr); continue; }
                const int j = tasks[t0 + lane].first, k = tasks[t0 + lane].second;
                o.ctask_addr.push_back((uint32_t)(k + 1 + (j - j0) * o.ldt));
                const auto &lst = cell[(size_t)j * ns + k];
                for (size_t e = 0; e < lst.size(); ++e) o.c_ent[(size_t)base + e * 32 + lane] = lst[e];
            }
        }
        o.panel_chunks.push_back((int32_t)(o.cchunk.size() / 2));
    }
    if (o.c_ent.empty()) o.c_ent.push_back(zero_slot);
    if (o.cchunk.empty()) { o.cchunk.push_back(0u); o.cchunk.push_back(0u); }
    if (o.ctask_addr.empty()) o.ctask_addr.push_back(pad_addr);
    if (o.sp_ent.empty()) { o.sp_ent.push_back((uint32_t)nr); o.sp_ent.push_back(zero_slot); }
}

int pack_mechanism(const pyjac_mech_desc *d, HostPack &out, size_t smem_budget, int panel_override,
                   const char **why)
{
    try {
        pack_impl(d, out, smem_budget, panel_override);
    } catch (const Fail &f) {
        if (why) *why = f.why;
        return f.code;
    } catch (...) {
        if (why) *why = "host allocation failed";
        return PYJAC_ENOMEM;
    }
    if (why) *why = "";
    return PYJAC_OK;
}

}  // namespace pyjac
