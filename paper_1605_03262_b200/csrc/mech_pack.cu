// mech_pack.cu -- validate a pyjac_mech_desc and pack it into the device table layout (host code).
//
// What is precomputed here is state-independent bookkeeping of the paper's restructured evaluation
// order (Algorithm 2): which per-reaction products feed which Jacobian entries,
// and in which fixed order they are summed.  No kinetic quantity is evaluated on the host except
// ln A, ln p of the tables and the per-reaction sums of NASA coefficients (Eq. 27 summed over a
// reaction, see device_mech.h `th_data`).
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <utility>
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

// one gathered sum (A1 phase or one Jacobian cell)
struct Task {
    std::vector<std::pair<uint32_t, int>> ent;   // kSum1 / kSum3: (E index, coefficient); kProd: (a | b << 16, 0)
    uint32_t kind = kSum1;
    uint32_t out = 0;       // E index of the result (kSum3: species k)
    double cst = 1.0;
    int rshift = 0;         // 2^rshift lanes share the sum
    bool lvl01 = false;     // needed by the rates / dydt kernels too
    size_t n_words = 0;     // entries after splitting coefficients
    int steps() const { return (int)((n_words + (size_t(1) << rshift) - 1) >> rshift); }
};

// lanes that share one sum: enough that no lane walks more than `cap` entries.  Long lists on one
// lane cost the fewest instructions (no padding, no shuffle reduction) but make long chunks: with two
// CTAs per SM the other CTA fills the tail, with one CTA per SM and a barrier per column panel it does
// not.  Measured (PYJAC_CAP sweep): cfg1 2.60 / 2.55 / 2.68 / 2.91 ms at cap 16 / 24 / 32 / 48; cfg2
// 9.80 / 9.41 / 9.50 / 9.54 / 11.16 ms at cap 6 / 8 / 12 / 16 / 24.  So the cap follows the shape: 24 / 10.
int pick_rshift(size_t len, size_t cap)
{
    for (int r = 0; r < 5; ++r)
        if (((len + (size_t(1) << r) - 1) >> r) <= cap) return r;
    return 5;
}
constexpr int kZeroSlots = 18;     // >= lanes of one shared-memory wavefront (16 at S = 1) + 2

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

static void pack_impl(const pyjac_mech_desc *d, HostPack &o, const ShapeHints &hints)
{
    validate(d);
    const int ns = d->n_species, nr = d->n_reactions, ld = ns + 1;
    o.ns = ns;
    o.nr = nr;
    // ---- species
    o.inv_mw.resize(ns);
    o.mw.assign(d->mol_wt, d->mol_wt + ns);
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
    o.colc.assign((size_t)4 * ld, 0.0);       // {u_c, v_c, 1/W_j, 0} (device_mech.h); column ns: zeros
    o.colc[2] = 1.0;
    for (int k = 0; k + 1 < ns; ++k) {
        o.colc[4 * (k + 1) + 0] = d->mol_wt[k] * (1.0 / d->mol_wt[k] - iw_last);
        o.colc[4 * (k + 1) + 1] = d->mol_wt[k];
        o.colc[4 * (k + 1) + 2] = 1.0 / d->mol_wt[k];
    }

    // ---- per reaction: molecules per side, breakpoints of its species' NASA ranges
    std::vector<int> mol_f(nr, 0), mol_r(nr, 0), n_brk(nr, 0);
    for (int i = 0; i < nr; ++i) {
        for (int q = d->reac_ptr[i]; q < d->reac_ptr[i + 1]; ++q) mol_f[i] += d->reac_nu[q];
        for (int q = d->prod_ptr[i]; q < d->prod_ptr[i + 1]; ++q) mol_r[i] += d->prod_nu[q];
        std::vector<double> brk;
        for (int q = d->reac_ptr[i]; q < d->reac_ptr[i + 1]; ++q) brk.push_back(d->t_mid[d->reac_spec[q]]);
        for (int q = d->prod_ptr[i]; q < d->prod_ptr[i + 1]; ++q) brk.push_back(d->t_mid[d->prod_spec[q]]);
        std::sort(brk.begin(), brk.end());
        n_brk[i] = (int)(std::unique(brk.begin(), brk.end()) - brk.begin());
    }
    auto expandable = [&](int i) { return mol_f[i] <= kMaxSide && mol_r[i] <= kMaxSide; };
    auto plain = [&](int i) {
        return d->rxn_type[i] == PYJAC_ELEMENTARY && d->rev_type[i] != PYJAC_REV_EXPLICIT && expandable(i) &&
               n_brk[i] <= 1;
    };

    // ---- sorted order: most expensive rate form first, the plain elementary reactions last
    std::vector<int> key(nr);
    for (int i = 0; i < nr; ++i) {
        const int t = d->rxn_type[i], rv = d->rev_type[i];
        const int form = (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED) ? d->falloff_form[i] : 0;
        int rank;
        if (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED)
            rank = form == PYJAC_TROE ? 0 : form == PYJAC_SRI ? 1 : 2;
        else
            rank = t == PYJAC_THIRD_BODY ? 3 : t == PYJAC_CHEBYSHEV ? 4 : t == PYJAC_PLOG ? 5 : plain(i) ? 7 : 6;
        const int nslot = expandable(i) ? mol_f[i] + mol_r[i]
                                        : (d->reac_ptr[i + 1] - d->reac_ptr[i]) + (d->prod_ptr[i + 1] - d->prod_ptr[i]);
        const int neff = std::min(n_eff_terms(d, i), 63);
        key[i] = (((rank * 4 + rv) * 8 + nslot) * 64) + neff;
    }
    std::vector<int> order(nr);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return key[a] < key[b]; });
    // A group of 32 lanes runs every code path one of its reactions needs, one after the other, and the
    // longest group is the critical path of the reaction queue.  The expensive falloff forms (Troe, SRI)
    // therefore never share a group: after each of them the group is filled up with third-body /
    // Lindemann reactions, which add almost nothing to a falloff group (same common part).
    {
        auto rank_of = [&](int i) { return key[i] / (4 * 8 * 64); };
        std::vector<int> troe, sri, fill, rest;
        for (int i : order) {
            const int r = rank_of(i);
            (r == 0 ? troe : r == 1 ? sri : (r == 2 || r == 3) ? fill : rest).push_back(i);
        }
        std::vector<int> out;
        size_t f = 0;
        for (auto *blk : {&troe, &sri}) {
            if (blk->empty()) continue;
            out.insert(out.end(), blk->begin(), blk->end());
            while (out.size() % 32 != 0 && f < fill.size()) out.push_back(fill[f++]);
        }
        while (f < fill.size()) out.push_back(fill[f++]);
        out.insert(out.end(), rest.begin(), rest.end());
        order.swap(out);
    }
    // ---- P1 path of every group of 32 reactions (device_mech.h `p1item`)
    auto fastgen = [&](int i) { return d->rev_type[i] != PYJAC_REV_EXPLICIT && expandable(i) && n_brk[i] <= 1; };
    o.n_rchunk = (nr + 31) / 32;
    o.rchunk.assign(std::max(o.n_rchunk, 1), 0u);
    for (int c = 0; c < o.n_rchunk; ++c) {
        bool all_plain = true, all_fast = true;
        for (int s = 32 * c; s < std::min(nr, 32 * c + 32); ++s) {
            all_plain = all_plain && plain(order[s]);
            all_fast = all_fast && fastgen(order[s]);
        }
        o.rchunk[c] = all_plain ? 1u : all_fast ? 2u : 0u;
    }
    // the plain groups are the last ones (sorted order); a plain group in front of a non-plain one takes path 2
    for (int c = o.n_rchunk - 1, tail = 1; c >= 0; --c) {
        if (o.rchunk[c] != 1u) tail = 0;
        else if (!tail) o.rchunk[c] = 2u;
        o.n_plain_chunks += o.rchunk[c] == 1u ? 1 : 0;
    }

    // ---- slots of every reaction (sorted order): species and nu per slot
    struct Slots { int spec[6]; int nu[6]; };
    std::vector<Slots> sl(nr);
    for (int s = 0; s < nr; ++s) {
        const int i = order[s];
        for (int p = 0; p < 6; ++p) { sl[s].spec[p] = ns; sl[s].nu[p] = 0; }
        for (int side = 0; side < 2; ++side) {
            const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
            const int32_t *sp = side ? d->prod_spec : d->reac_spec;
            const int32_t *nu = side ? d->prod_nu : d->reac_nu;
            int p = 3 * side;
            for (int q = ptr[i]; q < ptr[i + 1]; ++q) {
                if (expandable(i)) {
                    for (int r = 0; r < nu[q]; ++r, ++p) { sl[s].spec[p] = sp[q]; sl[s].nu[p] = 1; }
                } else {
                    sl[s].spec[p] = sp[q]; sl[s].nu[p] = nu[q]; ++p;
                }
            }
        }
    }

    // ---- E indices of the V entries, compact: per group of 32 reactions, slot position by slot
    // position, the lanes that use the position in lane order (neighbouring lanes, neighbouring words)
    std::vector<std::array<uint32_t, 6>> vslot(nr);
    std::vector<std::vector<uint32_t>> veff(nr);
    uint32_t nv = 0;
    // v_run[v] = (group, position, lane) of the store instruction that writes V entry v (the layout
    // optimisation below permutes indices among the lanes of one shared-memory wavefront of such a store)
    std::vector<std::array<int, 3>> v_run;
    for (int c = 0; c < o.n_rchunk; ++c) {
        const int s0 = 32 * c, s1 = std::min(nr, 32 * c + 32);
        for (int p = 0; p < 6; ++p)
            for (int s = s0; s < s1; ++s) {
                vslot[s][p] = sl[s].nu[p] ? nv++ : 0xFFFFFFFFu;
                if (sl[s].nu[p]) v_run.push_back({c, p, s - s0});
            }
        int maxeff = 0;
        for (int s = s0; s < s1; ++s) maxeff = std::max(maxeff, n_eff_terms(d, order[s]));
        for (int s = s0; s < s1; ++s) veff[s].clear();
        for (int e = 0; e < maxeff; ++e)
            for (int s = s0; s < s1; ++s)
                if (n_eff_terms(d, order[s]) > e) { veff[s].push_back(nv++); v_run.push_back({c, 6 + e, s - s0}); }
    }
    int next_slot = (int)nv;
    auto take = [&](int n) { int r = next_slot; next_slot += n; return r; };
    const int eQ = take(3 * nr), eH = take(nr);
    auto take2 = [&](int n) { next_slot = (next_slot + 1) & ~1; return take(n); };      // even: read in pairs of rows
    const int eAlpha = take2(ld), eGamma = take2(ld), eTc = take2(ld), eWdot = take(ns), eG0 = take(ns);
    const int eS1 = take(1), eA0 = take(1), eS4 = take(1), eZero = take(kZeroSlots), eDump = take(1);   // zero slots: one per bank group, plus two (kSum3 pads read q, a, Theta)
    o.eQ = eQ; o.eH = eH; o.eAlpha = eAlpha; o.eGamma = eGamma; o.eTc = eTc; o.eWdot = eWdot;
    o.eG0 = eG0; o.eS1 = eS1; o.eA0 = eA0; o.eS4 = eS4; o.eZero = eZero; o.eDump = eDump;
    const int eHs = next_slot;          // the partial sums of the long cell lists follow (sized below)

    // ---- per-reaction tables in sorted order
    o.lnA.assign(nr, 0.0); o.beta.assign(nr, 0.0); o.Ta.assign(nr, 0.0);
    o.rev_lnA.assign(nr, 0.0); o.rev_beta.assign(nr, 0.0); o.rev_Ta.assign(nr, 0.0);
    o.slots.assign((size_t)4 * std::max(nr, 1), 0u);
    o.vidx.assign((size_t)4 * std::max(nr, 1), 0u);
    o.rxn_orig.resize(nr);
    o.th_off.resize(nr);
    o.th_brk.assign(std::max(nr, 1), 0.0);
    o.th_soa.assign((size_t)((nr + 31) / 32 + 1) * 2 * 7 * 32, 0.0);
    auto th_at = [&](int sr, int iv, int c) -> double & { return o.th_soa[((size_t)((sr >> 5) * 2 + iv) * 7 + c) * 32 + (sr & 31)]; };
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
        uint32_t meta = 0, vi[6];
        int dnu = 0;
        for (int p = 0; p < 6; ++p) {
            vi[p] = (uint32_t)eDump;
            if (!sl[s].nu[p]) continue;
            const int k = sl[s].spec[p];
            meta |= (uint32_t)sl[s].nu[p] << (4 * p);
            vi[p] = vslot[s][p];
            cols[s].push_back({k, vi[p]});
            const int signed_nu = p >= 3 ? sl[s].nu[p] : -sl[s].nu[p];
            dnu += signed_nu;
            bool found = false;
            for (auto &pr : net[s])
                if (pr.first == k) { pr.second += signed_nu; found = true; }
            if (!found) net[s].push_back({k, signed_nu});
        }
        const int form = (t == PYJAC_FALLOFF || t == PYJAC_CHEM_ACTIVATED) ? d->falloff_form[i] : 0;
        const int single = is_pd(t) && d->tb_species[i] >= 0;
        meta |= (uint32_t)t << 24 | (uint32_t)rv << 27 | (uint32_t)form << 29 | (uint32_t)single << 31;
        o.slots[4 * s + 0] = (uint32_t)sl[s].spec[0] | (uint32_t)sl[s].spec[1] << 16;
        o.slots[4 * s + 1] = (uint32_t)sl[s].spec[2] | (uint32_t)sl[s].spec[3] << 16;
        o.slots[4 * s + 2] = (uint32_t)sl[s].spec[4] | (uint32_t)sl[s].spec[5] << 16;
        o.slots[4 * s + 3] = meta;
        o.vidx[4 * s + 0] = vi[0] | vi[1] << 16;
        o.vidx[4 * s + 1] = vi[2] | vi[3] << 16;
        o.vidx[4 * s + 2] = vi[4] | vi[5] << 16;

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
            o.th_brk[s] = nint == 2 ? brk[0] : nint == 1 ? HUGE_VAL : std::nan("");
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
                const double g[7] = {da[6] - da[0] + (double)dnu * ln_patm_R, da[0] - (double)dnu, da[1] * 0.5,
                                     da[2] * (1.0 / 6.0), da[3] * (1.0 / 12.0), da[4] * 0.05, -da[5]};
                for (int c = 0; c < 7; ++c) o.th_data.push_back(g[c]);
                if (nint <= 2)
                    for (int c = 0; c < 7; ++c) {
                        th_at(s, iv, c) = g[c];
                        if (nint == 1) th_at(s, 1, c) = g[c];
                    }
            }
        }
        if (is_pd(t)) {
            const bool fall = (t != PYJAC_THIRD_BODY);
            o.lo_lnA.push_back(fall ? std::log(d->arr_lo[3 * i]) : 0.0);
            o.lo_beta.push_back(fall ? d->arr_lo[3 * i + 1] : 0.0);
            o.lo_Ta.push_back(fall ? d->arr_lo[3 * i + 2] : 0.0);
            for (int c = 0; c < 5; ++c) {
                double v = fall ? d->falloff_par[5 * i + c] : 0.0;
                // the temperatures that only ever divide are stored as reciprocals: Troe T***, T* (Eq. 33),
                // SRI c (Eq. 36)
                if (fall && ((d->falloff_form[i] == PYJAC_TROE && (c == 1 || c == 2)) ||
                             (d->falloff_form[i] == PYJAC_SRI && c == 2)))
                    v = 1.0 / v;
                o.fall_par.push_back(v);
            }
            size_t e = 0;
            const int m = d->tb_species[i];
            if (m >= 0) {       // Eq. 30: [X]_i = [X_m]; one entry with "alpha - 1" = 1 and no [M] term
                o.eff_spec.push_back((uint32_t)m | veff[s][0] << 16);
                o.eff_eps.push_back(1.0);
                cols[s].push_back({m, veff[s][0]});
            } else {            // Eq. 28 written as [M] + sum_j (alpha_ij - 1)[X_j]
                for (int q = d->eff_ptr[i]; q < d->eff_ptr[i + 1]; ++q) {
                    if (d->eff_val[q] == 1.0) continue;
                    o.eff_spec.push_back((uint32_t)d->eff_spec[q] | veff[s][e] << 16);
                    o.eff_eps.push_back(d->eff_val[q] - 1.0);
                    cols[s].push_back({d->eff_spec[q], veff[s][e]});
                    ++e;
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


    // ---- one breakpoint for all reactions?  (reactions with a single interval carry the same
    // coefficients for both intervals in th_soa, so any breakpoint is right for them)
    {
        double common = HUGE_VAL;
        bool ok = true;
        for (int sr = 0; sr < nr && ok; ++sr) {
            const double b = o.th_brk[sr];
            if (b != b) ok = false;
            else if (b != HUGE_VAL) {
                if (common == HUGE_VAL) common = b;
                else if (common != b) ok = false;
            }
        }
        o.brk_common = ok ? common : std::nan("");
    }

    // ---- efficiencies, regrouped per group of 32 reactions (device_mech.h `eff_ent`)
    {
        const int n_gen = o.n_rchunk - (int)o.n_plain_chunks;
        o.eff_base.assign(1, 0);
        for (int c = 0; c < n_gen; ++c) {
            int gmax = 0;
            for (int l = 0; l < 32; ++l) {
                const int sr = 32 * c + l;
                if (sr < o.n_pd) gmax = std::max(gmax, o.eff_ptr[sr + 1] - o.eff_ptr[sr]);
            }
            for (int e = 0; e < gmax; ++e)
                for (int l = 0; l < 32; ++l) {
                    const int sr = 32 * c + l;
                    uint32_t w0 = (uint32_t)ns | (uint32_t)eDump << 16;
                    double eps = 0.0;
                    if (sr < o.n_pd && e < o.eff_ptr[sr + 1] - o.eff_ptr[sr]) {
                        w0 = o.eff_spec[o.eff_ptr[sr] + e];
                        eps = o.eff_eps[o.eff_ptr[sr] + e];
                    }
                    uint64_t bits;
                    std::memcpy(&bits, &eps, 8);
                    o.eff_ent.push_back(w0);
                    o.eff_ent.push_back(0u);
                    o.eff_ent.push_back((uint32_t)bits);
                    o.eff_ent.push_back((uint32_t)(bits >> 32));
                }
            o.eff_base.push_back((int32_t)(o.eff_ent.size() / 4));
        }
    }

    // ---- which per-reaction products feed which sums: Algorithm 2's scatter written
    // as fixed-order gathers
    std::vector<Task> sums;
    // (a) per species k: sums of nu_ki {q_i, a_i, Theta_i} (Eq. 14; the d_j coefficient of Eqs. 112, 119,
    //     123, 127 regrouped; the T column, Eq. 111).  The rates / dydt kernels need wdot too.
    const size_t tS3 = sums.size();
    for (int k = 0; k < ns; ++k) { Task t; t.kind = kSum3; t.out = (uint32_t)k; t.lvl01 = true; sums.push_back(t); }
    // (b) gamma'_r = (1 / W_Ns) sum_i nu_ki s'_iNs
    const size_t tGamma = sums.size();
    for (int k = 0; k < ns; ++k) {
        Task t; t.kind = kSum1; t.out = (uint32_t)(eGamma + k + 1); t.cst = iw_last;
        sums.push_back(t);
    }
    // (c) energy row (Eq. 113): G0_j = sum_i H_i s'_ij per column species
    const size_t tG0 = sums.size();
    for (int j = 0; j < ns; ++j) { Task t; t.kind = kProd; t.out = (uint32_t)(eG0 + j); sums.push_back(t); }

    // ---- lists of the Jacobian cells, flat column-major index f = r + c * ld.  Column 0 (the T column,
    // Eq. 111) reads the finished sum of its row; row 0 (the energy row) and column ns have no list.
    std::vector<std::vector<std::pair<uint32_t, int>>> cell((size_t)ld * ld);
    for (int s = 0; s < nr; ++s) {
        const uint32_t hs = (uint32_t)(eH + s);
        for (auto &ce : cols[s]) sums[tG0 + ce.spec].ent.push_back({ce.vi | hs << 16, 0});
        for (auto &pr : net[s]) {
            if (pr.second == 0) continue;
            const int k = pr.first;
            sums[tS3 + k].ent.push_back({(uint32_t)(eQ + 3 * s), pr.second});
            for (auto &ce : cols[s]) {
                if (ce.spec == ns - 1) sums[tGamma + k].ent.push_back({ce.vi, pr.second});
                else cell[(size_t)(k + 1) + (size_t)(ce.spec + 1) * ld].push_back({ce.vi, pr.second});
            }
        }
    }
    for (int r = 1; r < ld; ++r) cell[(size_t)r].push_back({(uint32_t)(eTc + r), 1});
    if (hints.keep_cells == 1) o.raw_cells = cell;

    // ---- entries after splitting coefficients beyond +-8 (device_mech.h); E indices, not yet offsets
    auto split = [&](const std::vector<std::pair<uint32_t, int>> &ent, std::vector<std::pair<uint32_t, int>> &w) {
        w.clear();
        for (auto &e : ent) {
            int c = e.second;
            const int sg = c < 0 ? -1 : 1;
            c = c < 0 ? -c : c;
            while (c > 0) { const int pz = std::min(c, 8); w.push_back({e.first, sg * pz}); c -= pz; }
        }
    };

    // ---- long cell lists are summed piecewise in phase A (balanced over the lanes: lists sorted by
    // length); phase B then reads at most `cell_cap` entries per cell, all lanes of a warp alike
    REQUIRE(hints.cell_cap >= 0 && hints.cell_cap <= 3, "cell_cap must be 0 (choose) or 1..3");
    REQUIRE(hints.cap >= 0 && hints.rp >= 0 && hints.rp <= 2 && hints.ctas >= 0 && hints.ctas <= 4 && hints.threads >= 0 && hints.S >= 0,
            "launch shape out of range");
    REQUIRE(hints.p1_states >= 0 && hints.p1_states <= 255, "p1_states out of range");
    const int cell_cap = hints.cell_cap >= 1 ? hints.cell_cap : 3;
    constexpr int kPiece = 8;
    std::vector<std::vector<std::pair<uint32_t, int>>> cell_w((size_t)ld * ld);
    {
        std::vector<std::pair<uint32_t, int>> w;
        int n_hs = 0;
        for (size_t f = 0; f < cell.size(); ++f) {
            if (cell[f].empty()) continue;
            split(cell[f], w);
            o.n_cells += 1;
            o.n_cell_entries += (long long)w.size();
            if ((int)w.size() <= cell_cap) { cell_w[f] = w; continue; }
            const int np = std::min(cell_cap, ((int)w.size() + kPiece - 1) / kPiece);
            o.n_heavy_cells += 1;
            size_t at = 0;
            for (int p = 0; p < np; ++p) {
                const size_t len = (w.size() - at + (np - p) - 1) / (np - p);
                Task t; t.kind = kSum1; t.out = (uint32_t)(eHs + n_hs); t.cst = 1.0;
                t.ent.assign(w.begin() + at, w.begin() + at + len);
                at += len;
                sums.push_back(t);
                cell_w[f].push_back({(uint32_t)(eHs + n_hs), 1});
                ++n_hs;
            }
        }
        o.n_heavy_pieces = n_hs;
        o.eHs = eHs;
        o.n_e = (eHs + n_hs + 1) & ~1;
        if (o.n_e > 65535) throw Fail{PYJAC_ELIMIT, "more than 65535 per-state table entries"};
    }

    // ---- launch shape: S states per CTA iteration, threads per CTA, CTAs per SM.  Everything lives in
    // shared memory: S x (E + two mixture parts) + the column / row constants.  S = 6 (48-byte elements)
    // and S = 2 (16-byte elements) let the 16-byte loads of a quarter warp fall into eight different bank
    // groups; S = 4 cannot (its elements cover only every other bank group), S = 3 uses 8-byte loads.
    {
        const long long sm_bytes = 228 * 1024;                       // shared memory of one sm_100 SM
        const SmemPlan pl = make_smem_plan(ns, o.n_e);
        auto bytes_for = [&](int S) { return ((long long)S * pl.total + pl.shared_total) * 8; };
        // each resident CTA also takes a 1 KB system reserve and the kernel's few static bytes
        auto limit_for = [&](int ctas) { return std::min<long long>(sm_bytes / ctas - 1024 - 128, hints.smem_bytes); };
        int S = hints.S, ctas = hints.ctas;
        if (S == 0) {
            // measured on B200 (profiles/): three interleaved states beat two, four and six on every
            // benchmark mechanism they fit (finer work items of the reaction queue, conflict-free 8-byte
            // gathers over sixteen bank pairs); then two, then one
            for (int cand : {3, 2, 1})
                if (S == 0 && bytes_for(cand) <= limit_for(ctas > 0 ? ctas : 1)) S = cand;
            if (S == 0) throw Fail{PYJAC_ELIMIT, "per-state tables exceed the shared memory of one CTA"};
        }
        if (S != 1 && S != 2 && S != 3 && S != 4 && S != 6) throw Fail{PYJAC_EINVAL, "states per CTA iteration must be 1, 2, 3, 4 or 6"};
        if (bytes_for(S) > limit_for(1)) throw Fail{PYJAC_ELIMIT, "per-state tables exceed the shared memory of one CTA"};
        if (ctas == 0) {
            ctas = 1;
            while (ctas < 4 && bytes_for(S) <= limit_for(ctas + 1)) ++ctas;
        }
        if (bytes_for(S) > limit_for(ctas)) throw Fail{PYJAC_ELIMIT, "the requested launch shape exceeds shared memory"};
        // measured on B200 (profiles/r2_shape_sweeps.md): with one state per CTA (the 360-species mechanism)
        // 384 threads beat 512 (1.55 M against 1.40 M states/s): fewer warps share the one-state queue tails
        int threads = hints.threads > 0 ? hints.threads : S == 1 && ctas == 1 ? 384 : (kMaxThreads / ctas) & ~31;
        // an explicit value outside the contract is an error (a sweep must not record a shape that never ran);
        // only the library's own choice is raised to the minimum
        if (hints.threads < 0 || (hints.threads > 0 && (threads < 32 * S || threads < 64)))
            throw Fail{PYJAC_EINVAL, "threads per CTA must be at least 64 and 32 per interleaved state"};
        if (threads < 32 * S) threads = 32 * S;
        if (threads < 64) threads = 64;
        if (threads > kMaxThreads || threads % 32) throw Fail{PYJAC_EINVAL, "threads per CTA must be a multiple of 32 up to kMaxThreads"};
        o.S = S; o.threads = threads; o.ctas_target = ctas;
        if ((long long)o.n_e * S * 8 > (long long)kEntOffMask + 1)
            throw Fail{PYJAC_ELIMIT, "per-CTA tables exceed the 256 KB offset range of a gather entry"};
    }
    const int S = o.S, NW = o.threads / 32;
    if (hints.rp == 2 && ld % 2 != 0)
        throw Fail{PYJAC_EINVAL, "two rows per lane need an odd number of species (even leading dimension)"};
    if (hints.p1_states < 0) throw Fail{PYJAC_EINVAL, "p1_states must not be negative"};
    o.rp = (hints.rp == 1 || hints.rp == 2) ? hints.rp : (ld % 2 == 0 ? 2 : 1);
    const int rp = o.rp;
    o.n_slab = (ld + 32 * rp - 1) / (32 * rp);

    // ---- work items of P1: the groups that need the one-state path first, then the pressure-dependent
    // groups, then the plain ones, each for every state (pair)
    {
        // states per fast-path item.  Plain groups (nine of eleven on 53 species) take all S states in one item:
        // the reaction's constants are read once per batch and stay in registers.  Groups with pressure-dependent
        // or PLOG / Chebyshev lanes cost two to three times as much per state and are the long items of the queue:
        // one state per item, so that the queue balances over the warps.  Measured with the bank-aware layout in
        // place (profiles/r2_shape_sweeps.md), 53 species S = 3: 2.16 ms against 2.29 (one state per item
        // everywhere) and 2.44 (three everywhere); 111 species 5.72 against 6.02 ms.
        // shape.p1_states: 0 = this rule; else states per plain item + 16 * states per general item (0: the same)
        const int per = hints.p1_states > 0 ? std::max(1, std::min(hints.p1_states % 16, S)) : S;
        const int per_gen = hints.p1_states >= 16 ? std::min(hints.p1_states / 16, S) : hints.p1_states > 0 ? per : 1;
        for (uint32_t kind : {0u, 2u, 1u})
            for (int c = 0; c < o.n_rchunk; ++c) {
                if (o.rchunk[c] != kind) continue;
                const int step = kind == 0u ? 1 : kind == 2u ? per_gen : per;
                for (int q = 0; q < S; q += step)
                    o.p1item.push_back((uint32_t)c | kind << 16 | (uint32_t)q << 20 | (uint32_t)std::min(step, S - q) << 24);
            }
    }

    // ---- encoding (device_mech.h) and bank-aware placement.  Which step of a lane reads which of its
    // entries, and which zero slot a padding entry reads, is free: both are chosen greedily so that the
    // lanes of one shared-memory wavefront hit different bank groups at every step.
    auto enc = [&](const std::pair<uint32_t, int> &e) { return coef_hi14(e.second) | (uint32_t)(e.first * S * 8); };
    const int gsz = S % 2 == 0 ? 16 : 8, LP = 128 / gsz, nq = 32 / LP;     // bytes per lane access, lanes per wavefront
    // lists[slot] sits on lanes [perm[slot] * width, (perm[slot] + 1) * width); returns grid[lane * steps + step].
    // Local search over two kinds of moves: two steps of one lane trade places; two sums of a chunk trade
    // lanes (`swap_slots`; not for phase B, whose lanes are tied to Jacobian rows).  The cost of a (step,
    // wavefront group of LP lanes) is the number of wavefronts beyond the first: the largest number of
    // different addresses in one bank group.
    auto place = [&](const std::vector<std::vector<uint32_t>> &lists, int width, int steps, uint32_t kind,
                     bool swap_slots, std::vector<int> *perm_out) {
        const int nstream = kind == kProd ? 2 : 1;
        const int nslot = 32 / width;
        std::vector<uint32_t> grid((size_t)32 * std::max(steps, 1), 0u);
        std::vector<int> perm(nslot);
        for (int i = 0; i < nslot; ++i) perm[i] = i;
        if (perm_out) *perm_out = perm;
        if (steps == 0) return grid;
        constexpr uint32_t kPad = 0xFFFFFFFFu;                 // a padding position (reads a zero slot chosen at the end)
        std::fill(grid.begin(), grid.end(), kPad);
        auto granule = [&](uint32_t w, int k) -> uint32_t {
            if (kind == kProd) return (k == 0 ? (w & 0xFFFF) : (w >> 16)) * (uint32_t)(S * 8 / gsz);
            return (w & kEntOffMask) / (uint32_t)gsz;
        };
        // initial layout: the words of a list go round its lanes
        for (size_t sl = 0; sl < lists.size(); ++sl) {
            REQUIRE((int)lists[sl].size() <= width * steps, "internal: a gather list does not fit its lanes");
            for (size_t e = 0; e < lists[sl].size(); ++e)
                grid[(size_t)((int)sl * width + (int)(e % width)) * steps + e / width] = lists[sl][e];
        }
        auto cell_cost = [&](int step, int quarter) {
            int cost = 0;
            for (int k = 0; k < nstream; ++k) {
                uint32_t seen[32];
                int nseen = 0, cnt[32] = {0};
                int worst = 1;
                for (int j = 0; j < LP; ++j) {
                    const uint32_t w = grid[(size_t)(quarter * LP + j) * steps + step];
                    if (w == kPad) continue;
                    const uint32_t g = granule(w, k);
                    bool dup = false;
                    for (int i = 0; i < nseen; ++i) dup = dup || seen[i] == g;
                    if (dup) continue;
                    seen[nseen++] = g;
                    worst = std::max(worst, ++cnt[g % LP]);
                }
                cost += worst - 1;
            }
            return cost;
        };
        // single-stream lists: an exact start.  Within one wavefront group (LP lanes) the entries are the edges of
        // a bipartite multigraph lanes x bank groups; `steps` colours (= steps) colour it without two edges of
        // one colour at a vertex iff no bank group is read more often than `steps` times (Koenig) -- then every
        // step reads LP different bank groups.  Alternating-path edge colouring; an edge whose bank group is
        // over capacity takes a step that is free at its lane and stays a conflict for the search below.
        {       // (two streams: the colouring takes the first stream, the search below sees both)
            for (int q = 0; q < nq; ++q) {
                std::vector<std::array<int, 3>> edges;                 // lane (within the group), bank group, word
                for (int j = 0; j < LP; ++j)
                    for (int st = 0; st < steps; ++st) {
                        const uint32_t w = grid[(size_t)(q * LP + j) * steps + st];
                        if (w != kPad) edges.push_back({j, (int)(granule(w, 0) % (uint32_t)LP), (int)w});
                    }
                std::vector<int> at_lane((size_t)LP * steps, -1), at_res((size_t)LP * steps, -1), colour(edges.size(), -1);
                for (size_t e = 0; e < edges.size(); ++e) {
                    const int u = edges[e][0], r = edges[e][1];
                    int a = -1, b = -1;
                    for (int c = 0; c < steps && a < 0; ++c) if (at_lane[(size_t)u * steps + c] < 0) a = c;
                    for (int c = 0; c < steps && b < 0; ++c) if (at_res[(size_t)r * steps + c] < 0) b = c;
                    REQUIRE(a >= 0, "internal: a lane holds more gather entries than steps");
                    if (b < 0) { colour[e] = a; at_lane[(size_t)u * steps + a] = (int)e; continue; }   // over capacity
                    if (at_res[(size_t)r * steps + a] >= 0) {
                        // flip the a / b alternating path that starts at bank group r with colour a
                        std::vector<int> path;
                        int cur_res = r, col = a;
                        for (;;) {
                            const int e1 = at_res[(size_t)cur_res * steps + col];
                            if (e1 < 0) break;
                            path.push_back(e1);
                            const int lane1 = edges[e1][0], other = col == a ? b : a;
                            const int e2 = at_lane[(size_t)lane1 * steps + other];
                            if (e2 < 0) break;
                            path.push_back(e2);
                            cur_res = edges[e2][1];
                            if (at_res[(size_t)cur_res * steps + other] != e2) break;     // e2 was an over-capacity edge
                        }
                        for (int pe : path) {
                            const int c0 = colour[pe];
                            if (at_lane[(size_t)edges[pe][0] * steps + c0] == pe) at_lane[(size_t)edges[pe][0] * steps + c0] = -1;
                            if (at_res[(size_t)edges[pe][1] * steps + c0] == pe) at_res[(size_t)edges[pe][1] * steps + c0] = -1;
                        }
                        for (int pe : path) {
                            const int c1 = colour[pe] == a ? b : a;
                            colour[pe] = c1;
                            at_lane[(size_t)edges[pe][0] * steps + c1] = pe;
                            if (at_res[(size_t)edges[pe][1] * steps + c1] < 0) at_res[(size_t)edges[pe][1] * steps + c1] = pe;
                        }
                    }
                    if (at_lane[(size_t)u * steps + a] >= 0 || at_res[(size_t)r * steps + a] >= 0) {
                        // the flip could not free colour a here (an over-capacity edge cut the path): any free step
                        a = -1;
                        for (int c = 0; c < steps && a < 0; ++c) if (at_lane[(size_t)u * steps + c] < 0) a = c;
                        colour[e] = a; at_lane[(size_t)u * steps + a] = (int)e;
                        if (at_res[(size_t)r * steps + a] < 0) at_res[(size_t)r * steps + a] = (int)e;
                        continue;
                    }
                    colour[e] = a;
                    at_lane[(size_t)u * steps + a] = (int)e;
                    at_res[(size_t)r * steps + a] = (int)e;
                }
                // write the group's lanes back: entry of colour c at step c, the rest pads
                std::vector<uint32_t> fresh((size_t)LP * steps, kPad);
                bool ok = true;
                for (size_t e = 0; e < edges.size(); ++e) {
                    uint32_t &slot = fresh[(size_t)edges[e][0] * steps + colour[e]];
                    if (slot != kPad) ok = false;
                    slot = (uint32_t)edges[e][2];
                }
                if (ok)
                    for (int j = 0; j < LP; ++j)
                        for (int st = 0; st < steps; ++st) grid[(size_t)(q * LP + j) * steps + st] = fresh[(size_t)j * steps + st];
            }
        }
        for (int pass = 0; pass < 6; ++pass) {
            bool improved = false;
            for (int lane = 0; lane < 32; ++lane) {
                const int q = lane / LP;
                for (int s1 = 0; s1 < steps; ++s1)
                    for (int s2 = s1 + 1; s2 < steps; ++s2) {
                        uint32_t &a = grid[(size_t)lane * steps + s1], &b = grid[(size_t)lane * steps + s2];
                        if (a == b) continue;
                        const int before = cell_cost(s1, q) + cell_cost(s2, q);
                        if (before == 0) continue;
                        std::swap(a, b);
                        const int after = cell_cost(s1, q) + cell_cost(s2, q);
                        if (after < before) improved = true;
                        else std::swap(a, b);
                    }
            }
            if (swap_slots && width <= LP)
                for (int a = 0; a < nslot; ++a)
                    for (int b = a + 1; b < nslot; ++b) {
                        const int qa = a * width / LP, qb = b * width / LP;
                        if (qa == qb) continue;
                        int before = 0;
                        for (int st = 0; st < steps; ++st) before += cell_cost(st, qa) + cell_cost(st, qb);
                        if (before == 0) continue;
                        auto swap_all = [&]() {
                            for (int j = 0; j < width; ++j)
                                for (int st = 0; st < steps; ++st)
                                    std::swap(grid[(size_t)(a * width + j) * steps + st], grid[(size_t)(b * width + j) * steps + st]);
                        };
                        swap_all();
                        int after = 0;
                        for (int st = 0; st < steps; ++st) after += cell_cost(st, qa) + cell_cost(st, qb);
                        if (after < before) { improved = true; std::swap(perm[a], perm[b]); }
                        else swap_all();
                    }
            if (!improved) break;
        }
        for (int st = 0; st < steps; ++st)
            for (int q = 0; q < nq; ++q) o.n_conflict_wf[swap_slots ? 0 : 1] += cell_cost(st, q);
        // perm[position] = list that sits there; callers want list -> position
        if (perm_out) {
            perm_out->assign(nslot, 0);
            for (int pos = 0; pos < nslot; ++pos) (*perm_out)[perm[pos]] = pos;
        }
        // pads: coefficient 0 (kProd: zero times zero) on a zero slot whose bank group is free
        for (int st = 0; st < steps; ++st)
            for (int q = 0; q < nq; ++q) {
                bool used[2][32] = {{false}};
                for (int j = 0; j < LP; ++j) {
                    const uint32_t w = grid[(size_t)(q * LP + j) * steps + st];
                    if (w == kPad) continue;
                    for (int k = 0; k < nstream; ++k) used[k][granule(w, k) % LP] = true;
                }
                int z = 0;
                for (int t = 0; t < LP; ++t) {
                    const uint32_t g = (uint32_t)(eZero + t) * (uint32_t)(S * 8 / gsz);
                    bool ok = true;
                    for (int k = 0; k < nstream; ++k) ok = ok && !used[k][g % LP];
                    if (ok) { z = t; break; }
                }
                const uint32_t zi = (uint32_t)(eZero + z);
                for (int j = 0; j < LP; ++j) {
                    uint32_t &w = grid[(size_t)(q * LP + j) * steps + st];
                    if (w == kPad) w = kind == kProd ? (zi | zi << 16) : zi * (uint32_t)(S * 8);
                }
            }
        return grid;
    };

    // ---- phase A chunks: sums of one kind, shared by equally many lanes and of similar length, fill the
    // 32 lanes of a chunk; the warps take the chunks row by row, most expensive first.
    {
        std::vector<std::pair<uint32_t, int>> w;
        for (auto &t : sums) {
            if (t.kind == kProd) t.n_words = t.ent.size();
            else { split(t.ent, w); t.n_words = w.size(); }
            // longest list one lane walks: 12, and 20 when a CTA holds one state (360 species 1.94 -> 1.88 ms per 4,096 states)
            t.rshift = pick_rshift(t.n_words, hints.cap > 0 ? (size_t)hints.cap : S == 1 ? 20 : 12);
        }
        struct Chunk { std::vector<Task *> t; uint32_t kind; int rshift; int steps; bool lvl01; double cost; };
        std::vector<Chunk> chunks;
        if (nr > 0) chunks.push_back({{}, kAll3, 5, (nr + 31) / 32, true, 0.0});
        std::vector<Task *> idx;
        for (auto &t : sums)
            if (t.kind == kSum3 || !t.ent.empty()) idx.push_back(&t);
        std::stable_sort(idx.begin(), idx.end(), [&](const Task *a, const Task *b) {
            if (a->kind != b->kind) return a->kind < b->kind;
            if (a->rshift != b->rshift) return a->rshift > b->rshift;
            return a->steps() > b->steps();
        });
        for (size_t p = 0; p < idx.size();) {
            const Task &t0 = *idx[p];
            Chunk c{{}, t0.kind, t0.rshift, 0, t0.lvl01, 0.0};
            const size_t per = (size_t)32 >> t0.rshift;
            while (p < idx.size() && c.t.size() < per && idx[p]->kind == c.kind && idx[p]->rshift == c.rshift) {
                c.steps = std::max(c.steps, idx[p]->steps());
                c.t.push_back(idx[p++]);
            }
            chunks.push_back(c);
        }
        // cost in loads per block: a chunk's fixed part, its steps, its shuffle reduction
        for (auto &c : chunks) {
            const double per_step = c.kind == kSum3 ? 3.0 : c.kind == kAll3 ? 4.0 : c.kind == kProd ? 2.0 : 1.0;
            const double nsum = (c.kind == kSum3 || c.kind == kAll3) ? 3.0 : 1.0;
            c.cost = 4.0 + per_step * c.steps + 1.5 * nsum * c.rshift;
        }
        // the warps take chunk (row * NW + w): arrange the chunks so that every warp gets about the same
        // cost (longest first onto the least loaded warp; rows padded with empty chunks).  The chunks the
        // rates / source-term kernels need too come first, in rows of their own.
        std::vector<Chunk> arranged;
        std::vector<double> load(NW, 0.0);
        int rows01 = 0;
        for (int pass = 0; pass < 2; ++pass) {
            std::vector<Chunk *> grp;
            for (auto &c : chunks)
                if (c.lvl01 == (pass == 0)) grp.push_back(&c);
            if (grp.empty()) continue;
            std::stable_sort(grp.begin(), grp.end(), [](const Chunk *a, const Chunk *b) { return a->cost > b->cost; });
            std::vector<std::vector<Chunk *>> mine(NW);
            for (Chunk *c : grp) {
                int wmin = 0;
                for (int i = 1; i < NW; ++i)
                    if (load[i] < load[wmin]) wmin = i;
                mine[wmin].push_back(c);
                load[wmin] += c->cost;
            }
            size_t rows = 0;
            for (auto &v : mine) rows = std::max(rows, v.size());
            for (size_t k = 0; k < rows; ++k)
                for (int wi = 0; wi < NW; ++wi) {
                    if (k < mine[wi].size()) arranged.push_back(*mine[wi][k]);
                    else arranged.push_back(Chunk{{}, kSum1, 0, 0, pass == 0, 0.0});      // empty chunk
                }
            if (pass == 0) rows01 = (int)rows;
        }
        o.n_arow = (int)(arranged.size() / NW);
        o.n_arow01 = rows01;

        // the partial sums of the long cell lists (region Hs) in the order in which the chunks' lanes produce them:
        // the 32 results of a chunk go to 32 consecutive elements (their stores meet few bank conflicts)
        if (hints.layout != 2 && o.n_heavy_pieces > 0) {
            std::vector<uint32_t> renum((size_t)o.n_heavy_pieces, 0xFFFFFFFFu);
            uint32_t next = 0;
            for (auto &c : arranged)
                if (c.kind == kSum1)
                    for (Task *t : c.t)
                        if (t->out >= (uint32_t)eHs && t->out < (uint32_t)(eHs + o.n_heavy_pieces)) {
                            renum[t->out - (uint32_t)eHs] = next;
                            t->out = (uint32_t)eHs + next++;
                        }
            REQUIRE(next == (uint32_t)o.n_heavy_pieces, "internal: a partial sum of a cell list is in no chunk");
            for (auto &cl : cell_w)
                for (auto &e : cl)
                    if (e.first >= (uint32_t)eHs && e.first < (uint32_t)(eHs + o.n_heavy_pieces))
                        e.first = (uint32_t)eHs + renum[e.first - (uint32_t)eHs];
        }

        // ---- bank-aware LAYOUT of the s' values.  Where a value sits in E decides its bank; the lanes of one
        // shared-memory wavefront of a gather (LP lanes) should read LP different bank groups at every step.  The
        // reaction phase writes the values of one slot position of 32 reactions to consecutive indices, so any
        // permutation of the indices AMONG the lanes of one of its store wavefronts keeps those stores
        // conflict-free.  That freedom is used here: a gather group (the LP lanes of a chunk or of a phase-B
        // cell column, `cap` steps) is conflict-free iff no bank group is read more than `cap` times (the
        // lane x bank-group multigraph is then cap-edge-colourable, Koenig; `place` below finds the steps), and
        // pairs of values of one store wavefront trade indices while that lowers the total excess.
        if (hints.layout != 2 && nv > 0) {
            const uint32_t unit = (uint32_t)(S * 8 / gsz);
            auto res_of = [&](uint32_t e) { return (int)((e * unit) % (uint32_t)LP); };
            struct Grp { int cap; std::array<int, 16> cnt; };
            std::vector<Grp> groups;
            std::vector<std::vector<int>> member(nv);                  // V entry -> groups (with multiplicity)
            auto add_entry = [&](int g, uint32_t e) {
                if (e < nv) member[e].push_back(g);
                groups[g].cnt[res_of(e)] += 1;
            };
            for (auto &c : arranged) {
                if (c.kind != kSum1 && c.kind != kProd) continue;
                const int width = 1 << c.rshift;
                const int g0 = (int)groups.size();
                for (int h = 0; h < nq; ++h) groups.push_back(Grp{c.steps, {}});
                for (size_t i = 0; i < c.t.size(); ++i) {
                    std::vector<std::pair<uint32_t, int>> ww;
                    if (c.kind == kProd) ww = c.t[i]->ent; else split(c.t[i]->ent, ww);
                    for (size_t e = 0; e < ww.size(); ++e) {
                        const int lane = (int)i * width + (int)(e % width);
                        add_entry(g0 + lane / LP, c.kind == kProd ? (ww[e].first & 0xFFFF) : ww[e].first);
                    }
                }
            }
            for (int slab = 0; slab < o.n_slab; ++slab)
                for (int c = 0; c < ld; ++c)
                    for (int h = 0; h < rp; ++h) {
                        int nst = 0;
                        for (int lane = 0; lane < 32; ++lane) {
                            const int r = rp * (32 * slab + lane) + h;
                            if (r < ld) nst = std::max(nst, (int)cell_w[(size_t)r + (size_t)c * ld].size());
                        }
                        if (nst == 0) continue;
                        const int g0 = (int)groups.size();
                        for (int hh = 0; hh < nq; ++hh) groups.push_back(Grp{nst == 1 ? 1 : 3, {}});
                        for (int lane = 0; lane < 32; ++lane) {
                            const int r = rp * (32 * slab + lane) + h;
                            if (r >= ld) continue;
                            for (auto &e : cell_w[(size_t)r + (size_t)c * ld]) add_entry(g0 + lane / LP, e.first);
                        }
                    }
            auto excess = [&](int g) {
                int x = 0;
                for (int k = 0; k < LP; ++k) x += std::max(0, groups[g].cnt[k] - groups[g].cap);
                return x;
            };
            // store wavefronts: V entries with the same (group, position, lane / LP), consecutive in v_run
            std::vector<uint32_t> where(nv);                          // where[v] = index v's value now sits at
            for (uint32_t v = 0; v < nv; ++v) where[v] = v;
            long long before = 0, after = 0;
            for (size_t g = 0; g < groups.size(); ++g) before += excess((int)g);
            for (int sweep = 0; sweep < 12; ++sweep) {
                bool improved = false;
                for (uint32_t a0 = 0; a0 < nv;) {
                    uint32_t a1 = a0 + 1;
                    while (a1 < nv && v_run[a1][0] == v_run[a0][0] && v_run[a1][1] == v_run[a0][1] &&
                           v_run[a1][2] / LP == v_run[a0][2] / LP)
                        ++a1;
                    for (uint32_t x = a0; x < a1; ++x)
                        for (uint32_t y = x + 1; y < a1; ++y) {
                            // values x and y trade places: every group of x moves one count from res(where[x]) to
                            // res(where[y]) and vice versa
                            const int rx = res_of(where[x]), ry = res_of(where[y]);
                            if (rx == ry) continue;
                            int cost0 = 0, cost1 = 0;
                            for (int g : member[x]) cost0 += excess(g);
                            for (int g : member[y]) cost0 += excess(g);
                            for (int g : member[x]) { groups[g].cnt[rx] -= 1; groups[g].cnt[ry] += 1; }
                            for (int g : member[y]) { groups[g].cnt[ry] -= 1; groups[g].cnt[rx] += 1; }
                            for (int g : member[x]) cost1 += excess(g);
                            for (int g : member[y]) cost1 += excess(g);
                            if (cost1 < cost0) {
                                std::swap(where[x], where[y]);
                                improved = true;
                            } else {
                                for (int g : member[x]) { groups[g].cnt[rx] += 1; groups[g].cnt[ry] -= 1; }
                                for (int g : member[y]) { groups[g].cnt[ry] += 1; groups[g].cnt[rx] -= 1; }
                            }
                        }
                    a0 = a1;
                }
                if (!improved) break;
            }
            for (size_t g = 0; g < groups.size(); ++g) after += excess((int)g);
            o.n_layout_excess[0] = before; o.n_layout_excess[1] = after;
            // apply: every reference to V entry v now names where[v]
            auto mv = [&](uint32_t e) { return e < nv ? where[e] : e; };
            for (int sr = 0; sr < nr; ++sr) {
                for (int w = 0; w < 3; ++w) {
                    const uint32_t lo = o.vidx[4 * sr + w] & 0xFFFF, hi = o.vidx[4 * sr + w] >> 16;
                    o.vidx[4 * sr + w] = mv(lo) | mv(hi) << 16;
                }
            }
            for (size_t k = 0; k < o.eff_ent.size(); k += 4) {
                const uint32_t sp = o.eff_ent[k] & 0xFFFF, vi = o.eff_ent[k] >> 16;
                o.eff_ent[k] = sp | mv(vi) << 16;
            }
            for (auto &t : sums) {
                if (t.kind == kSum1) for (auto &e : t.ent) e.first = mv(e.first);
                if (t.kind == kProd) for (auto &e : t.ent) e.first = mv(e.first & 0xFFFF) | (e.first & 0xFFFF0000u);
            }
            for (auto &cl : cell_w)
                for (auto &e : cl) e.first = mv(e.first);
        }
        // The same for the per-reaction blocks {q_i, a_i, Theta_i} (region Q, three elements per reaction) and H_i:
        // reaction s keeps both at position rpos[s]; positions are traded among the reactions of one store
        // wavefront (LP lanes of a group of 32) against the gather groups of the per-species sums (they read Q)
        // and of the energy-row column sums (their second stream reads H).
        std::vector<uint32_t> rpos(std::max(nr, 1));
        for (int sr = 0; sr < nr; ++sr) rpos[sr] = (uint32_t)sr;
        if (hints.layout != 2 && nr > 0) {
            const uint32_t unit = (uint32_t)(S * 8 / gsz);
            auto res_t = [&](int type, uint32_t pos) {
                return (int)(((type == 0 ? (uint32_t)eQ + 3u * pos : (uint32_t)eH + pos) * unit) % (uint32_t)LP);
            };
            struct Grp { int cap; std::array<int, 16> cnt; };
            std::vector<Grp> groups;
            std::vector<std::vector<std::pair<int, int>>> member(nr);      // reaction -> (group, type)
            for (auto &c : arranged) {
                if (c.kind != kSum3 && c.kind != kProd) continue;
                const int width = 1 << c.rshift, type = c.kind == kSum3 ? 0 : 1;
                const int g0 = (int)groups.size();
                for (int h = 0; h < nq; ++h) groups.push_back(Grp{c.steps, {}});
                for (size_t i = 0; i < c.t.size(); ++i) {
                    std::vector<std::pair<uint32_t, int>> ww;
                    if (c.kind == kProd) ww = c.t[i]->ent; else split(c.t[i]->ent, ww);
                    for (size_t e = 0; e < ww.size(); ++e) {
                        const int lane = (int)i * width + (int)(e % width);
                        const int sr = c.kind == kSum3 ? (int)(ww[e].first - (uint32_t)eQ) / 3 : (int)((ww[e].first >> 16) - (uint32_t)eH);
                        member[sr].push_back({g0 + lane / LP, type});
                        groups[g0 + lane / LP].cnt[res_t(type, (uint32_t)sr)] += 1;
                    }
                }
            }
            auto excess = [&](int g) {
                int x = 0;
                for (int k = 0; k < LP; ++k) x += std::max(0, groups[g].cnt[k] - groups[g].cap);
                return x;
            };
            auto move = [&](int sr, uint32_t from, uint32_t to) {
                for (auto &mg : member[sr]) {
                    groups[mg.first].cnt[res_t(mg.second, from)] -= 1;
                    groups[mg.first].cnt[res_t(mg.second, to)] += 1;
                }
            };
            for (int sweep = 0; sweep < 12; ++sweep) {
                bool improved = false;
                for (int a0 = 0; a0 < nr; a0 += LP) {
                    const int a1 = std::min(nr, std::min(a0 + LP, (a0 / 32 + 1) * 32));
                    for (int x = a0; x < a1; ++x)
                        for (int y = x + 1; y < a1; ++y) {
                            int cost0 = 0, cost1 = 0;
                            for (auto &mg : member[x]) cost0 += excess(mg.first);
                            for (auto &mg : member[y]) cost0 += excess(mg.first);
                            const uint32_t px = rpos[x], py = rpos[y];
                            move(x, px, py); move(y, py, px);
                            for (auto &mg : member[x]) cost1 += excess(mg.first);
                            for (auto &mg : member[y]) cost1 += excess(mg.first);
                            if (cost1 < cost0) { std::swap(rpos[x], rpos[y]); improved = true; }
                            else { move(x, py, px); move(y, px, py); }
                        }
                }
                if (!improved) break;
            }
            for (auto &t : sums) {
                if (t.kind == kSum3)
                    for (auto &e : t.ent) e.first = (uint32_t)eQ + 3u * rpos[(e.first - (uint32_t)eQ) / 3];
                if (t.kind == kProd)
                    for (auto &e : t.ent) e.first = (e.first & 0xFFFF) | ((uint32_t)eH + rpos[(e.first >> 16) - (uint32_t)eH]) << 16;
            }
        }
        for (int sr = 0; sr < nr; ++sr) o.vidx[4 * sr + 3] = rpos[sr];

        for (auto &c : arranged) {
            const uint32_t base = (uint32_t)(o.a_ent.size() / 4);       // in uint4 units
            const int width = 1 << c.rshift, per_row = 32 / width;
            o.achunk.push_back(base);
            o.achunk.push_back((uint32_t)c.steps | c.kind << 8 | (uint32_t)c.rshift << 12);
            REQUIRE(c.steps < 256, "internal: a phase-A chunk has more than 255 steps");
            const int nblk = 1 + (c.kind == kAll3 ? 0 : (c.steps + 3) / 4);
            o.a_ent.resize(o.a_ent.size() + (size_t)nblk * 128, 0u);
            uint32_t *blk = o.a_ent.data() + (size_t)base * 4;
            std::vector<std::vector<uint32_t>> lists((size_t)per_row);
            if (c.kind != kAll3)
                for (size_t i = 0; i < c.t.size(); ++i) {
                    if (c.kind == kProd) {
                        for (auto &e : c.t[i]->ent) lists[i].push_back(e.first);
                    } else {
                        split(c.t[i]->ent, w);
                        for (auto &e : w) lists[i].push_back(enc(e));
                    }
                }
            // blocks of four steps; the words behind the chunk's last step are never read
            std::vector<int> pos;
            const std::vector<uint32_t> grid = place(lists, width, c.kind == kAll3 ? 0 : c.steps, c.kind, true, &pos);
            for (int lane = 0; lane < 32; ++lane) {
                blk[(size_t)lane * 4 + 0] = 0xFFFFFFFFu;
                blk[(size_t)lane * 4 + 1] = 0u;
                blk[(size_t)lane * 4 + 2] = 0u;
            }
            if (c.kind != kAll3)
                for (size_t i = 0; i < c.t.size(); ++i) {
                    uint64_t bits;
                    std::memcpy(&bits, &c.t[i]->cst, 8);
                    for (int j = 0; j < width; ++j) {
                        const size_t lane = (size_t)pos[i] * width + j;
                        blk[lane * 4 + 0] = c.t[i]->out;
                        blk[lane * 4 + 1] = (uint32_t)bits;
                        blk[lane * 4 + 2] = (uint32_t)(bits >> 32);
                    }
                }
            o.n_a_steps_kind[c.kind] += c.steps;
            if (c.kind == kAll3) { o.n_a_steps += c.steps; continue; }
            for (int lane = 0; lane < 32; ++lane)
                for (int st = 0; st < c.steps; ++st)
                    blk[((size_t)(1 + st / 4) * 32 + lane) * 4 + st % 4] = grid[(size_t)lane * c.steps + st];
            o.n_a_steps += c.steps;
        }
        o.a_ent.resize(o.a_ent.size() + 128, 0u);        // the kernels read one block past a chunk's last
        o.achunk.resize(o.achunk.size() + (size_t)2 * 2 * NW, 0u);  // ... and the headers two rows ahead
    }

    // ---- phase B items: one per (slab, column); a lane's cells are rows rp * (32 slab + lane) .. + rp - 1.
    // Every cell has three entry words (padded with a zero slot); the fourth word of every lane is the
    // step count of the item's cells h: 0 (no lane has an entry), 1 (one step), 2 (three steps).
    {
        const size_t n_item = (size_t)o.n_slab * ld;
        o.b_ent.assign((n_item + kBPad) * rp * 128, (uint32_t)(eZero * S * 8));     // padding items: read ahead
        std::vector<double> cost(n_item, 0.0);
        for (int slab = 0; slab < o.n_slab; ++slab)
            for (int c = 0; c < ld; ++c) {
                const size_t it = (size_t)slab * ld + c;
                cost[it] = 8.0 + 3.0 * rp;
                for (int h = 0; h < rp; ++h) {
                    std::vector<std::vector<uint32_t>> lists(32);
                    int nst = 0;
                    for (int lane = 0; lane < 32; ++lane) {
                        const int r = rp * (32 * slab + lane) + h;
                        if (r >= ld) continue;
                        for (auto &e : cell_w[(size_t)r + (size_t)c * ld]) lists[lane].push_back(enc(e));
                        nst = std::max(nst, (int)lists[lane].size());
                    }
                    REQUIRE(nst <= 3, "internal: a phase-B cell list is longer than three entries");
                    const int run = nst == 0 ? 0 : nst == 1 ? 1 : 3;          // steps the kernel executes (1 or 3)
                    const std::vector<uint32_t> grid = place(lists, 1, std::max(run, 1), kSum1, false, nullptr);
                    uint32_t *blk = o.b_ent.data() + (it * rp + h) * 128;
                    for (int lane = 0; lane < 32; ++lane) {
                        for (int st = 0; st < std::max(run, 1); ++st) blk[lane * 4 + st] = grid[(size_t)lane * std::max(run, 1) + st];
                        blk[lane * 4 + 3] = nst == 0 ? 0u : nst == 1 ? 1u : 2u;
                    }
                    cost[it] += run;
                    o.n_b_steps += run;
                }
            }
        for (size_t k = n_item * rp * 128 + 3; k < o.b_ent.size(); k += 4) o.b_ent[k] = 0u;
        // contiguous ranges of items per warp, balanced by cost
        double total = 0.0;
        for (double c : cost) total += c;
        o.bsplit.assign(NW + 1, 0);
        double acc = 0.0;
        int wi = 1;
        for (size_t it = 0; it < cost.size(); ++it) {
            acc += cost[it];
            while (wi < NW && acc >= total * wi / NW) o.bsplit[wi++] = (int32_t)(it + 1);
        }
        while (wi <= NW) o.bsplit[wi++] = (int32_t)cost.size();
    }

    // ---- gather tables in shared memory?  (one copy per CTA, read with 16-byte shared loads instead of
    // through L1 / L2 for every batch)
    if (hints.stage == 1) {
        const SmemPlan pl = make_smem_plan(ns, o.n_e, (int)((o.achunk.size() / 2 + 1) / 2), (int)(o.a_ent.size() / 4),
                                           (int)(o.b_ent.size() / 4));
        const long long bytes = ((long long)S * pl.total + pl.shared_total) * 8;
        if (bytes > std::min<long long>(228 * 1024 / o.ctas_target - 1024 - 128, hints.smem_bytes))
            throw Fail{PYJAC_ELIMIT, "the gather tables do not fit the shared memory of this launch shape"};
        o.stage = true;
    }

    // ---- self-check of what the kernels rely on without bounds checks: every source offset and every
    // output index inside the block's E array, every block a chunk or an item reads inside its table
    {
        auto bad = [](const char *wh) { throw Fail{PYJAC_ELIMIT, wh}; };
        const uint32_t e_total = (uint32_t)o.n_e;
        const size_t na_blocks = o.a_ent.size() / 4;
        if (o.achunk.size() / 2 != (size_t)(o.n_arow + 2) * NW) bad("internal: phase A is not whole rows of chunks");
        for (size_t c = 0; c < (size_t)o.n_arow * NW; ++c) {
            const uint32_t base = o.achunk[2 * c], meta = o.achunk[2 * c + 1];
            const int steps = (int)(meta & 0xFF), kind = (int)((meta >> 8) & 0xF);
            const int nblk = 1 + (kind == (int)kAll3 ? 0 : (steps + 3) / 4);
            if ((size_t)base + 32 * (size_t)(nblk + 1) > na_blocks) bad("internal: a chunk reads past the entry table");
            if (kind == (int)kAll3) continue;
            const uint32_t *blk = o.a_ent.data() + (size_t)base * 4;
            for (int lane = 0; lane < 32; ++lane) {
                const uint32_t out = blk[(size_t)lane * 4];
                if (out != 0xFFFFFFFFu && out >= (kind == (int)kSum3 ? (uint32_t)ns : e_total))
                    bad("internal: a gather result lies outside E");
                for (int st = 0; st < steps; ++st) {
                    const uint32_t wd = blk[((size_t)(1 + st / 4) * 32 + lane) * 4 + st % 4];
                    const bool ok = kind == (int)kProd
                                        ? ((wd & 0xFFFF) < e_total && (wd >> 16) < e_total)
                                        : ((wd & kEntOffMask) % (8u * S) == 0 &&
                                           (wd & kEntOffMask) / (8u * S) + (kind == (int)kSum3 ? 2u : 0u) < e_total);
                    if (!ok) bad("internal: a gather entry points outside E");
                }
            }
        }
        if (o.b_ent.size() != ((size_t)o.n_slab * ld + kBPad) * rp * 128) bad("internal: phase B table has the wrong size");
        for (size_t k = 0; k < o.b_ent.size(); ++k) {
            const uint32_t wd = o.b_ent[k];
            if (k % 4 == 3) { if (wd > 2u) bad("internal: a phase-B step count is out of range"); continue; }
            if ((wd & kEntOffMask) % (8u * S) != 0 || (wd & kEntOffMask) / (8u * S) >= e_total)
                bad("internal: a cell entry points outside E");
        }
        if (o.bsplit[0] != 0 || o.bsplit[NW] != o.n_slab * ld) bad("internal: phase B ranges do not cover the items");
    }
}

ShapeHints hints_from_shape(const pyjac_launch_shape *shape, long long smem_optin)
{
    ShapeHints h;
    if (smem_optin > 0) h.smem_bytes = smem_optin - 128;
    if (shape) {
        h.S = shape->states_per_cta; h.threads = shape->threads; h.ctas = shape->ctas_per_sm;
        h.cap = shape->list_cap; h.cell_cap = shape->cell_cap; h.rp = shape->rows_per_lane;
        h.p1_states = shape->p1_states; h.stage = shape->stage_tables; h.layout = shape->layout;
    }
    return h;
}

int pack_mechanism(const pyjac_mech_desc *d, HostPack &out, const ShapeHints &hints, const char **why)
{
    try {
        pack_impl(d, out, hints);
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
