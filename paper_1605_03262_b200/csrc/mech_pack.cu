// mech_pack.cu -- validate a pyjac_mech_desc and pack it into the device table layout (host code).
//
// What is precomputed here is state-independent bookkeeping of the paper's restructured evaluation
// order (Algorithm 2): which per-reaction products feed which Jacobian entries,
// and in which fixed order they are summed.  No kinetic quantity is evaluated on the host except
// ln A, ln p of the tables and the per-reaction sums of NASA coefficients (Eq. 27 summed over a
// reaction, see device_mech.h `th_data`).
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
    uint32_t vi;   // E index of s'_ij
};

// one gathered sum of the AUX phase
struct Task {
    std::vector<uint32_t> ent;
    uint32_t flags = 0;     // kAuxTwoIndex | kAuxScaled | scalar << 8
    uint32_t out = 0;       // E slot
    double cst = 0.0;
    bool reduce = false;    // spread over the 32 lanes of its own chunk
    bool lvl01 = false;     // needed by the rates / dydt kernels too
};

void validate(const pyjac_mech_desc *d)
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
    for (int k = 0; k < ns; ++k)
        REQUIRE(d->mol_wt[k] > 0.0 && std::isfinite(d->mol_wt[k]), "molecular weight must be positive");
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
        if (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED) {
            const int form = d->falloff_form[i];
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
    }
}

bool is_pd(int t) { return t == PYJAC_THIRD_BODY || t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED; }
bool is_pk(int t) { return t == PYJAC_PLOG || t == PYJAC_CHEBYSHEV; }

// number of efficiency terms the kernel sums for reaction i (Eq. 28 written as [M] + sum (alpha - 1)[X_j])
int n_eff_terms(const pyjac_mech_desc *d, int i)
{
    if (!is_pd(d->rxn_type[i])) return 0;
    if (d->tb_species[i] >= 0) return 1;
    int n = 0;
    for (int q = d->eff_ptr[i]; q < d->eff_ptr[i + 1]; ++q) n += d->eff_val[q] != 1.0;
    return n;
}

}  // namespace

static void pack_impl(const pyjac_mech_desc *d, HostPack &o, long long smem_doubles)
{
    validate(d);
    const int ns = d->n_species, nr = d->n_reactions, ld = ns + 1;
    o.ns = ns;
    o.nr = nr;
    // ---- species
    o.inv_mw.resize(ns);
    o.t_mid.assign(d->t_mid, d->t_mid + ns);
    o.nasa.resize((size_t)10 * ns);
    for (int k = 0; k < ns; ++k) {
        o.inv_mw[k] = 1.0 / d->mol_wt[k];
        for (int c = 0; c < 5; ++c) {
            o.nasa[(size_t)(0 * 5 + c) * ns + k] = d->nasa_lo[7 * k + c];
            o.nasa[(size_t)(1 * 5 + c) * ns + k] = d->nasa_hi[7 * k + c];
        }
    }
    const double iw_last = 1.0 / d->mol_wt[ns - 1];
    o.wrow.assign((size_t)ld, 1.0);
    for (int k = 0; k < ns; ++k) o.wrow[k + 1] = d->mol_wt[k];
    o.colc.assign((size_t)2 * ld, 0.0);
    o.colc[1] = 1.0;
    for (int k = 0; k < ns; ++k) {
        o.colc[2 * (k + 1)] = 1.0 / d->mol_wt[k] - iw_last;
        o.colc[2 * (k + 1) + 1] = 1.0 / d->mol_wt[k];
    }

    // ---- sorted order: most expensive rate form first; one form, one stoichiometry path and
    // equally many V entries per group of 32
    std::vector<int> key(nr);
    for (int i = 0; i < nr; ++i) {
        const int t = d->rxn_type[i], rv = d->rev_type[i];
        const int form = (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED) ? d->falloff_form[i] : 0;
        int rank;
        if (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED)
            rank = form == PYJAC_TROE ? 0 : form == PYJAC_SRI ? 1 : 2;
        else
            rank = t == PYJAC_THIRD_BODY ? 3 : t == PYJAC_CHEBYSHEV ? 4 : t == PYJAC_PLOG ? 5 : 6;
        bool unit = true;
        for (int q = d->reac_ptr[i]; q < d->reac_ptr[i + 1]; ++q) unit = unit && d->reac_nu[q] == 1;
        for (int q = d->prod_ptr[i]; q < d->prod_ptr[i + 1]; ++q) unit = unit && d->prod_nu[q] == 1;
        const int nslot = (d->reac_ptr[i + 1] - d->reac_ptr[i]) + (d->prod_ptr[i + 1] - d->prod_ptr[i]);
        const int neff = std::min(n_eff_terms(d, i), 63);
        key[i] = ((((rank * 2 + (unit ? 0 : 1)) * 4 + rv) * 8 + nslot) * 64) + neff;
    }
    std::vector<int> order(nr);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return key[a] < key[b]; });
    o.n_rchunk = (nr + 31) / 32;

    // ---- E indices of the V entries: per group of 32 reactions, slot-major (lane-contiguous)
    o.vbase.assign(nr, 0u);
    std::vector<uint32_t> eff_vb(nr, 0u);
    uint32_t nv = 0;
    for (int c = 0; c < o.n_rchunk; ++c) {
        int maxslot = 0, maxeff = 0;
        for (int s = 32 * c; s < std::min(nr, 32 * c + 32); ++s) {
            const int i = order[s];
            maxslot = std::max(maxslot, (d->reac_ptr[i + 1] - d->reac_ptr[i]) + (d->prod_ptr[i + 1] - d->prod_ptr[i]));
            maxeff = std::max(maxeff, n_eff_terms(d, i));
        }
        for (int s = 32 * c; s < std::min(nr, 32 * c + 32); ++s) {
            o.vbase[s] = nv + (uint32_t)(s - 32 * c);
            eff_vb[s] = nv + (uint32_t)(kVStride * maxslot + (s - 32 * c));
        }
        nv += (uint32_t)(kVStride * (maxslot + maxeff));
    }
    const int eQ = (int)nv, eAr = eQ + nr, eTh = eAr + nr, eH = eTh + nr;
    const int eAlpha = eH + nr, eGamma = eAlpha + ld, eWdot = eGamma + ld;
    const int eS1 = eWdot + ns, eS4 = eS1 + 1;
    int next_slot = eS4 + 1;          // further AUX results
    o.eQ = eQ; o.eAr = eAr; o.eTh = eTh; o.eH = eH; o.eAlpha = eAlpha; o.eGamma = eGamma; o.eWdot = eWdot;
    o.eS1 = eS1; o.eS4 = eS4;

    // ---- per-reaction tables in sorted order
    o.lnA.assign(nr, 0.0); o.beta.assign(nr, 0.0); o.Ta.assign(nr, 0.0);
    o.rev_lnA.assign(nr, 0.0); o.rev_beta.assign(nr, 0.0); o.rev_Ta.assign(nr, 0.0);
    o.slots.assign((size_t)4 * nr, 0u);
    o.rxn_orig.resize(nr);
    o.th_off.resize(nr);
    o.n_pd = 0; o.n_pk = 0;
    o.pk_ptr.assign(1, 0);
    o.eff_ptr.assign(1, 0);
    std::vector<std::vector<ColEntry>> cols(nr);            // column entries of each reaction
    std::vector<std::vector<std::pair<int, int>>> net(nr);  // (species, net nu) of each reaction
    const double ln_patm_R = std::log(kPatm / kRu);
    for (int s = 0; s < nr; ++s) {
        const int i = order[s];
        const int t = d->rxn_type[i], rv = d->rev_type[i];
        o.rxn_orig[s] = i;
        if (is_pd(t)) { REQUIRE(s == o.n_pd, "internal: sort order"); ++o.n_pd; }
        if (is_pk(t)) { REQUIRE(s == o.n_pd + o.n_pk, "internal: sort order"); ++o.n_pk; }
        if (!is_pk(t)) {
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
        uint32_t vi = o.vbase[s];
        int dnu = 0;
        for (int side = 0; side < 2; ++side) {
            const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
            const int32_t *sp = side ? d->prod_spec : d->reac_spec;
            const int32_t *nu = side ? d->prod_nu : d->reac_nu;
            for (int q = ptr[i], e = 0; q < ptr[i + 1]; ++q, ++e) {
                const int slot = 3 * side + e;
                spec[slot] = (uint32_t)sp[q];
                meta |= (uint32_t)nu[q] << (4 * slot);
                cols[s].push_back({sp[q], vi});
                vi += kVStride;
                const int signed_nu = side ? nu[q] : -nu[q];
                dnu += signed_nu;
                bool found = false;
                for (auto &pr : net[s])
                    if (pr.first == sp[q]) { pr.second += signed_nu; found = true; }
                if (!found) net[s].push_back({sp[q], signed_nu});
            }
        }
        const int form = (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED) ? d->falloff_form[i] : 0;
        const int single = is_pd(t) && d->tb_species[i] >= 0;
        meta |= (uint32_t)t << 24 | (uint32_t)rv << 27 | (uint32_t)form << 29 | (uint32_t)single << 31;
        o.slots[4 * s + 0] = spec[0] | spec[1] << 16;
        o.slots[4 * s + 1] = spec[2] | spec[3] << 16;
        o.slots[4 * s + 2] = spec[4] | spec[5] << 16;
        o.slots[4 * s + 3] = meta;

        // sum_k nu_ki B_k(T) as one polynomial per interval between the t_mid of the species
        {
            std::vector<double> brk;
            for (auto &pr : net[s]) brk.push_back(d->t_mid[pr.first]);
            std::sort(brk.begin(), brk.end());
            brk.erase(std::unique(brk.begin(), brk.end()), brk.end());
            const int nint = (int)brk.size() + 1;
            o.th_off[s] = (uint32_t)o.th_data.size();
            o.th_data.push_back((double)nint);
            for (double b : brk) o.th_data.push_back(b);
            for (int iv = 0; iv < nint; ++iv) {
                // interval iv: brk[iv-1] < T <= brk[iv]; species k is in its low range iff T <= t_mid[k]
                double da[7] = {0, 0, 0, 0, 0, 0, 0};
                for (auto &pr : net[s]) {
                    const int k = pr.first;
                    const int m = (int)(std::lower_bound(brk.begin(), brk.end(), d->t_mid[k]) - brk.begin());  // 0-based
                    const bool low = m >= iv;
                    const double *a = (low ? d->nasa_lo : d->nasa_hi) + 7 * k;
                    for (int c = 0; c < 7; ++c) da[c] += (double)pr.second * a[c];
                }
                o.th_data.push_back(da[6] - da[0] + (double)dnu * ln_patm_R);   // g0
                o.th_data.push_back(da[0] - (double)dnu);                        // g1
                o.th_data.push_back(da[1] * 0.5);                                // g2
                o.th_data.push_back(da[2] * (1.0 / 6.0));                        // g3
                o.th_data.push_back(da[3] * (1.0 / 12.0));                       // g4
                o.th_data.push_back(da[4] * 0.05);                               // g5
                o.th_data.push_back(-da[5]);                                     // g6
            }
        }
        if (is_pd(t)) {
            const bool fall = (t != PYJAC_THIRD_BODY);
            o.lo_lnA.push_back(fall ? std::log(d->arr_lo[3 * i]) : 0.0);
            o.lo_beta.push_back(fall ? d->arr_lo[3 * i + 1] : 0.0);
            o.lo_Ta.push_back(fall ? d->arr_lo[3 * i + 2] : 0.0);
            for (int c = 0; c < 5; ++c) o.fall_par.push_back(fall ? d->falloff_par[5 * i + c] : 0.0);
            o.eff_vbase.push_back(eff_vb[s]);
            uint32_t ve = eff_vb[s];
            const int m = d->tb_species[i];
            if (m >= 0) {       // Eq. 30: [X]_i = [X_m]; one entry with "alpha - 1" = 1 and no [M] term
                o.eff_spec.push_back(m);
                o.eff_eps.push_back(1.0);
                cols[s].push_back({m, ve});
            } else {            // Eq. 28 written as [M] + sum_j (alpha_ij - 1)[X_j]
                for (int q = d->eff_ptr[i]; q < d->eff_ptr[i + 1]; ++q) {
                    if (d->eff_val[q] == 1.0) continue;
                    o.eff_spec.push_back(d->eff_spec[q]);
                    o.eff_eps.push_back(d->eff_val[q] - 1.0);
                    cols[s].push_back({d->eff_spec[q], ve});
                    ve += kVStride;
                }
            }
            o.eff_ptr.push_back((int32_t)o.eff_spec.size());
        }
        if (is_pk(t)) {
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

    // ---- AUX tasks that always exist
    std::vector<Task> tasks;
    auto scaled = [](uint32_t scalar) { return (uint32_t)kAuxScaled | scalar << 8; };
    // (a) wdot_k = sum_i nu_ki q_i (Eq. 14) and S1 = sum_i H_i q_i: the rates / dydt kernels need them too
    for (int k = 0; k < ns; ++k) {
        Task t;
        t.out = (uint32_t)(eWdot + k);
        t.lvl01 = true;
        tasks.push_back(t);
    }
    const size_t tS1 = tasks.size();
    { Task t; t.flags = kAuxTwoIndex; t.out = (uint32_t)eS1; t.reduce = true; t.lvl01 = true; tasks.push_back(t); }
    // (b) alpha_r = (W_k / rho) sum_i nu_ki (a_i + W q_i), the coefficient of d_j in row r = k + 1
    //     (Eqs. 112, 119, 123, 127 regrouped); gamma_r = (W_k / W_Ns) sum_i nu_ki s'_iNs
    const size_t tAlpha = tasks.size();
    for (int k = 0; k < ns; ++k) {
        Task t;
        t.out = (uint32_t)(eAlpha + k + 1); t.flags = scaled(kIrho); t.cst = d->mol_wt[k];
        tasks.push_back(t);
    }
    const size_t tGamma = tasks.size();
    for (int k = 0; k < ns; ++k) {
        Task t;
        t.out = (uint32_t)(eGamma + k + 1); t.flags = scaled(kOne); t.cst = d->mol_wt[k] * iw_last;
        tasks.push_back(t);
    }
    // (c) energy row (Eq. 113): G0_j = sum_i H_i s'_ij per column, scaled by -1/c_p
    const size_t tG0 = tasks.size();
    std::vector<uint32_t> g0_slot(ns, 0u);
    for (int j = 0; j < ns; ++j) {
        Task t;
        t.flags = kAuxTwoIndex | scaled(kNegIcp);
        if (j == ns - 1) { t.out = (uint32_t)eGamma; t.cst = iw_last; }
        else { t.out = (uint32_t)next_slot++; t.cst = 1.0; g0_slot[j] = t.out; }
        tasks.push_back(t);
    }
    //     alpha_0 = -(1 / (rho c_p)) sum_i H_i (a_i + W q_i);  S4 = sum_i H_i Theta_i
    const size_t tA0 = tasks.size();
    { Task t; t.flags = kAuxTwoIndex | scaled(kNegIrhoIcp); t.out = (uint32_t)eAlpha; t.cst = 1.0; t.reduce = true; tasks.push_back(t); }
    const size_t tS4 = tasks.size();
    { Task t; t.flags = kAuxTwoIndex; t.out = (uint32_t)eS4; t.reduce = true; tasks.push_back(t); }

    // ---- lists of the Jacobian cells, flat column-major index f = r + c * ld
    std::vector<std::vector<uint32_t>> cell((size_t)ld * ld);
    for (int s = 0; s < nr; ++s) {
        const uint32_t hs = (uint32_t)(eH + s);
        tasks[tS1].ent.push_back((uint32_t)(eQ + s) | hs << 16);
        tasks[tA0].ent.push_back((uint32_t)(eAr + s) | hs << 16);
        tasks[tS4].ent.push_back((uint32_t)(eTh + s) | hs << 16);
        for (auto &ce : cols[s]) tasks[tG0 + ce.spec].ent.push_back(ce.vi | hs << 16);
        for (auto &pr : net[s]) {
            if (pr.second == 0) continue;
            const int k = pr.first;
            tasks[k].ent.push_back(pack_entry((uint32_t)(eQ + s), pr.second));
            tasks[tAlpha + k].ent.push_back(pack_entry((uint32_t)(eAr + s), pr.second));
            cell[(size_t)(k + 1)].push_back(pack_entry((uint32_t)(eTh + s), pr.second));        // column 0 (d/dT)
            for (auto &ce : cols[s]) {
                if (ce.spec == ns - 1) tasks[tGamma + k].ent.push_back(pack_entry(ce.vi, pr.second));
                else cell[(size_t)(k + 1) + (size_t)(ce.spec + 1) * ld].push_back(pack_entry(ce.vi, pr.second));
            }
        }
    }
    for (int j = 0; j < ns - 1; ++j) cell[(size_t)(j + 1) * ld].push_back(pack_entry(g0_slot[j], 1));   // row 0
    for (auto &c : cell) o.n_list_entries += (long long)c.size();

    // ---- MAIN tasks: 32 consecutive cells; lists longer than the task's cap are summed by an AUX
    // task and enter as one entry.  The cap minimises (steps of the task) + (steps of the AUX
    // chunks it causes); `lambda` prices the extra E slots and grows until E fits the shared memory.
    const size_t ncell = (size_t)ld * ld;
    o.n_mtask = (int)((ncell + 31) / 32);
    const size_t fixed_tasks = tasks.size();
    std::vector<int> cap(o.n_mtask, 0);
    for (double lambda = 0.15;; lambda *= 2.0) {
        tasks.resize(fixed_tasks);
        int slots = next_slot;
        bool any_overflow = false;
        for (int t = 0; t < o.n_mtask; ++t) {
            int len[32], mx = 0;
            for (int l = 0; l < 32; ++l) {
                const size_t f = (size_t)t * 32 + l;
                len[l] = f < ncell ? (int)cell[f].size() : 0;
                mx = std::max(mx, len[l]);
            }
            double best = 1e300;
            int bestc = mx;
            for (int c = (mx > 0 ? 1 : 0); c <= mx; ++c) {
                double cost = (double)c;
                for (int l = 0; l < 32; ++l)
                    if (len[l] > c) cost += 1.25 * len[l] / 32.0 + lambda;
                if (cost < best) { best = cost; bestc = c; }
            }
            cap[t] = bestc;
            for (int l = 0; l < 32; ++l)
                if (len[l] > bestc) { ++slots; any_overflow = true; }
        }
        if (slots + 1 <= std::min<long long>(smem_doubles, 65535)) break;
        if (!any_overflow) throw Fail{PYJAC_ELIMIT, "per-state tables exceed the shared memory of one CTA"};
        if (lambda > 1e6) {   // no overflow at all: every list inline
            for (int t = 0; t < o.n_mtask; ++t) {
                int mx = 0;
                for (int l = 0; l < 32; ++l) {
                    const size_t f = (size_t)t * 32 + l;
                    if (f < ncell) mx = std::max(mx, (int)cell[f].size());
                }
                cap[t] = mx;
            }
            if (next_slot + 1 > std::min<long long>(smem_doubles, 65535))
                throw Fail{PYJAC_ELIMIT, "per-state tables exceed the shared memory of one CTA"};
            break;
        }
    }
    for (int t = 0; t < o.n_mtask; ++t)
        for (int l = 0; l < 32; ++l) {
            const size_t f = (size_t)t * 32 + l;
            if (f >= ncell || (int)cell[f].size() <= cap[t]) continue;
            Task a;
            a.out = (uint32_t)next_slot++;
            a.ent.swap(cell[f]);
            tasks.push_back(a);
            cell[f].push_back(pack_entry(tasks.back().out, 1));
        }
    const int eZero = next_slot++;
    o.eZero = eZero;
    o.n_e = next_slot;
    if (o.n_e > 65535) throw Fail{PYJAC_ELIMIT, "more than 65535 per-state table entries"};
    const uint32_t pad1 = pack_entry((uint32_t)eZero, 0);
    const uint32_t pad2 = (uint32_t)eZero | (uint32_t)eZero << 16;

    // ---- MAIN entries
    o.mtask.assign((size_t)4 * o.n_mtask, 0u);
    for (int t = 0; t < o.n_mtask; ++t) {
        const uint32_t base = (uint32_t)o.m_ent.size();
        o.mtask[4 * t + 0] = base;
        o.mtask[4 * t + 1] = (uint32_t)cap[t];
        o.mtask[4 * t + 2] = (uint32_t)(((size_t)t * 32) % ld);
        o.mtask[4 * t + 3] = (uint32_t)(((size_t)t * 32) / ld);
        o.m_ent.resize(o.m_ent.size() + (size_t)cap[t] * 32, pad1);
        for (int l = 0; l < 32; ++l) {
            const size_t f = (size_t)t * 32 + l;
            if (f >= ncell) continue;
            for (size_t e = 0; e < cell[f].size(); ++e) o.m_ent[(size_t)base + e * 32 + l] = cell[f][e];
        }
        o.n_main_entries += (long long)cap[t] * 32;
    }
    if (o.m_ent.empty()) o.m_ent.push_back(pad1);

    // ---- AUX chunks: tasks with equal flags and similar length share a chunk of 32 lanes
    struct Chunk { std::vector<size_t> t; int steps; bool lvl01; bool reduce; };
    std::vector<Chunk> chunks;
    {
        std::vector<size_t> idx;
        for (size_t t = 0; t < tasks.size(); ++t) {
            if (tasks[t].reduce) chunks.push_back({{t}, (int)((tasks[t].ent.size() + 31) / 32), tasks[t].lvl01, true});
            else idx.push_back(t);
        }
        std::stable_sort(idx.begin(), idx.end(), [&](size_t a, size_t b) {
            if (tasks[a].lvl01 != tasks[b].lvl01) return tasks[a].lvl01;
            if (tasks[a].flags != tasks[b].flags) return tasks[a].flags < tasks[b].flags;
            return tasks[a].ent.size() > tasks[b].ent.size();
        });
        for (size_t p = 0; p < idx.size();) {
            Chunk c{{}, 0, tasks[idx[p]].lvl01, false};
            const uint32_t fl = tasks[idx[p]].flags;
            while (p < idx.size() && c.t.size() < 32 && tasks[idx[p]].lvl01 == c.lvl01 && tasks[idx[p]].flags == fl) {
                c.steps = std::max(c.steps, (int)tasks[idx[p]].ent.size());
                c.t.push_back(idx[p++]);
            }
            chunks.push_back(c);
        }
        // longest first (the warps take chunks from a queue); the rates / dydt subset in front
        std::stable_sort(chunks.begin(), chunks.end(), [&](const Chunk &a, const Chunk &b) {
            if (a.lvl01 != b.lvl01) return a.lvl01;
            return a.steps > b.steps;
        });
    }
    o.n_achunk = (int)chunks.size();
    o.n_achunk01 = 0;
    for (auto &c : chunks) o.n_achunk01 += c.lvl01 ? 1 : 0;
    for (auto &c : chunks) {
        const Task &t0 = tasks[c.t[0]];
        const uint32_t base = (uint32_t)o.a_ent.size();
        const bool two = (t0.flags & kAuxTwoIndex) != 0;
        o.a_ent.resize(o.a_ent.size() + (size_t)c.steps * 32, two ? pad2 : pad1);
        o.achunk.push_back(base);
        o.achunk.push_back((uint32_t)c.steps);
        o.achunk.push_back(t0.flags | (c.reduce ? (uint32_t)kAuxReduce : 0u));
        o.achunk.push_back((uint32_t)o.a_out.size());
        if (c.reduce) {
            for (size_t e = 0; e < t0.ent.size(); ++e) o.a_ent[(size_t)base + (e / 32) * 32 + (e % 32)] = t0.ent[e];
            o.a_out.push_back(t0.out);
            o.a_const.push_back(t0.cst);
            for (int l = 1; l < 32; ++l) { o.a_out.push_back(0xFFFFFFFFu); o.a_const.push_back(0.0); }
        } else {
            for (int l = 0; l < 32; ++l) {
                if (l >= (int)c.t.size()) { o.a_out.push_back(0xFFFFFFFFu); o.a_const.push_back(0.0); continue; }
                const Task &t = tasks[c.t[l]];
                o.a_out.push_back(t.out);
                o.a_const.push_back(t.cst);
                for (size_t e = 0; e < t.ent.size(); ++e) o.a_ent[(size_t)base + e * 32 + l] = t.ent[e];
            }
        }
        o.n_aux_entries += (long long)c.steps * 32;
    }
    if (o.a_ent.empty()) o.a_ent.push_back(pad1);
    if (o.achunk.empty()) { o.achunk.assign(4, 0u); }
    if (o.a_out.empty()) { o.a_out.push_back(0xFFFFFFFFu); o.a_const.push_back(0.0); }
}

int pack_mechanism(const pyjac_mech_desc *d, HostPack &out, long long smem_doubles, const char **why)
{
    try {
        pack_impl(d, out, smem_doubles);
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
