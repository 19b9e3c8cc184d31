"""Seeded synthetic kinetic models and thermochemical states (input generators only).

The paper measured on four published kinetic models with PaSR-generated states
(PAPER.md:746-753 Table 1, :761, Table 2 :767-778); neither is available here, so
BASELINE.json's synthetic configurations stand in for them.  This module draws
those inputs.  It contains none of the method's arithmetic (no rates, no
thermodynamic evaluation of the model, no Jacobian): only random parameters, the
element bookkeeping needed to write balanced reactions, and a least-squares fit
that *produces* NASA-7 coefficients.  Both the oracle tests and the CUDA path get
their inputs from here; neither side's results ever feed back into it.

Recipe (DESIGN.md "Synthetic inputs" has the full statement):
  species   distinct element compositions with 1..max_atoms atoms; the bare atoms
            and N2 always present; N2 last (the paper puts the abundant inert
            species last) and inert in the benchmark mechanisms
  thermo    NASA-7, two ranges 300-t_mid-5000 K fitted to a smooth
            cp/R = c_lo + (c_hi-c_lo)(1-exp(-T/theta)); a5 from a bond-additive h_f/R
            (element terms - 2.2e4 K per bond + U(-1e4,1e4) K) at 298.15 K, a6 from
            s/R = 12 + 3.5 ln W + U(-2,2); upper range continuous in H and S
  reactions element-balanced, 1-3 reactants and 1-3 products, reversible through K_c;
            ln A ~ U(10,35), beta ~ U(-2,3), Ea ~ U(0,50) kcal/mol
  states    T ~ U(800,2500) K, P ~ logU(1,50) atm, Y ~ Dirichlet(0.5) floored at
            1e-20, renormalised, largest component swapped into the last slot
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass

import numpy as np

from .mechanism import (CHEBYSHEV, CHEM_ACTIVATED, ELEMENTARY, FALLOFF, IRREVERSIBLE, LINDEMANN,
                        PLOG, REV_EXPLICIT, REV_FROM_KC, SRI, THIRD_BODY, TROE, Mechanism,
                        MechanismBuilder)

ATOMIC_WEIGHT = {"H": 1.008, "O": 15.999, "N": 14.007, "C": 12.011}
P_ATM = 101325.0                       # Pa
R_KCAL = 1.98720425864083e-3           # kcal mol^-1 K^-1 (Ea -> Ta conversion only)
BASE_SEED = 1605032620


@dataclass(frozen=True)
class Config:
    name: str
    n_species: int
    n_reactions: int
    elements: tuple
    max_atoms: int
    n_third_body: int
    n_troe: int
    n_lindemann: int
    n_sri: int
    n_chem_act: int
    n_plog: int
    n_cheb: int
    n_states: int
    seed: int


CONFIGS = {
    0: Config("cfg0_13sp_27rx", 13, 27, ("H", "O", "N"), 4, 6, 2, 0, 0, 0, 0, 0, 1024, BASE_SEED + 0),
    1: Config("cfg1_53sp_325rx", 53, 325, ("C", "H", "O", "N"), 4, 30, 20, 5, 0, 0, 2, 0, 100_000,
              BASE_SEED + 1),
    2: Config("cfg2_111sp_784rx", 111, 784, ("C", "H", "O", "N"), 5, 60, 50, 0, 5, 5, 0, 4, 100_000,
              BASE_SEED + 2),
    3: Config("cfg3_360sp_2172rx", 360, 2172, ("C", "H", "O", "N"), 8, 120, 90, 0, 20, 0, 5, 5,
              32_768, BASE_SEED + 3),
}
# config 4 of BASELINE.json is the state-count sweep on the config-1 mechanism
SWEEP_STATES = [4 ** k for k in range(5, 11)]


# ----------------------------------------------------------------------------- species + thermo
def _formula(elements, counts):
    return "".join(e + (str(c) if c > 1 else "") for e, c in zip(elements, counts) if c > 0)


def _all_compositions(n_el, max_atoms):
    out = []
    for n in range(1, max_atoms + 1):
        for c in itertools.combinations_with_replacement(range(n_el), n):
            v = [0] * n_el
            for i in c:
                v[i] += 1
            out.append(tuple(v))
    return out


# h_f/R = sum_e n_e*ETA_e - BOND*(n_atoms-1) + noise: balanced exchange reactions then have a
# reaction enthalpy set by the noise alone and recombinations are exothermic by about one bond,
# as in real mechanisms, so equilibrium constants stay within physically plausible ranges.
ETA_ELEMENT = {"H": 2.6e4, "O": 3.0e4, "N": 5.7e4, "C": 8.6e4}      # K
BOND = 2.2e4                                                         # K per bond


def _fit_nasa(rng, n_atoms, t_mid, hf_base, mol_wt):
    """Least-squares NASA-7 coefficients for one synthetic species (generator, not method)."""
    if n_atoms == 1:
        c_lo, c_hi = 2.5, 2.5
    else:
        c_lo = 3.5 if n_atoms == 2 else 4.0
        c_hi = c_lo + (3 * n_atoms - (5 if n_atoms == 2 else 6)) * rng.uniform(0.7, 1.0)
    theta = rng.uniform(800.0, 2000.0)
    cp = lambda T: c_lo + (c_hi - c_lo) * (1.0 - np.exp(-T / theta))
    coef = []
    for lo, hi in ((300.0, t_mid), (t_mid, 5000.0)):
        T = np.linspace(lo, hi, 64)
        x = T / 1000.0                               # scaled for conditioning
        V = np.vander(x, 5, increasing=True)
        a, *_ = np.linalg.lstsq(V, cp(T), rcond=None)
        coef.append(a / (1000.0 ** np.arange(5)))
    hf = hf_base - BOND * (n_atoms - 1) + rng.uniform(-1.0e4, 1.0e4)   # H/R at 298.15 K, in K
    s0 = 12.0 + 3.5 * np.log(mol_wt) + rng.uniform(-2.0, 2.0)          # S/R at 298.15 K

    def h_poly(a, T):                                # T(a0 + a1 T/2 + ...), the a5-free part
        return T * (a[0] + T * (a[1] / 2 + T * (a[2] / 3 + T * (a[3] / 4 + T * a[4] / 5))))

    def s_poly(a, T):
        return a[0] * np.log(T) + T * (a[1] + T * (a[2] / 2 + T * (a[3] / 3 + T * a[4] / 4)))

    lo, hi = coef
    a5_lo = hf - h_poly(lo, 298.15)
    a6_lo = s0 - s_poly(lo, 298.15)
    a5_hi = h_poly(lo, t_mid) + a5_lo - h_poly(hi, t_mid)
    a6_hi = s_poly(lo, t_mid) + a6_lo - s_poly(hi, t_mid)
    return np.concatenate([lo, [a5_lo, a6_lo]]), np.concatenate([hi, [a5_hi, a6_hi]])


def _make_species(rng, elements, max_atoms, n_species, t_mid_choices=(1000.0,), n2_last=True):
    n_el = len(elements)
    comps = _all_compositions(n_el, max_atoms)
    forced = [tuple(1 if i == j else 0 for i in range(n_el)) for j in range(n_el)]
    n2 = None
    if "N" in elements and n2_last:
        n2 = tuple(2 if e == "N" else 0 for e in elements)
        forced.append(n2)
    rest = [c for c in comps if c not in forced]
    if n_species < len(forced) or n_species > len(comps):
        raise ValueError("cannot draw %d distinct compositions" % n_species)
    pick = rng.choice(len(rest), size=n_species - len(forced), replace=False)
    chosen = forced + [rest[i] for i in sorted(pick)]
    order = list(rng.permutation(len(chosen)))
    chosen = [chosen[i] for i in order]
    if n2 is not None:
        chosen.remove(n2)
        chosen.append(n2)
    comp = np.array(chosen, dtype=np.int32)
    w = comp @ np.array([ATOMIC_WEIGHT[e] for e in elements])
    lo, hi, tm = [], [], []
    eta = np.array([ETA_ELEMENT[e] for e in elements])
    for c, wk in zip(chosen, w):
        t_mid = float(rng.choice(t_mid_choices))
        a_lo, a_hi = _fit_nasa(rng, int(sum(c)), t_mid, float(np.dot(c, eta)), float(wk))
        lo.append(a_lo); hi.append(a_hi); tm.append(t_mid)
    names = [_formula(elements, c) for c in chosen]
    return names, comp, w, np.array(lo), np.array(hi), np.array(tm)


# ----------------------------------------------------------------------------- balanced reactions
def _multiset_buckets(rng, comp, reactive, max_triples=400_000):
    """{composition: {size: [multiset, ...]}} for species multisets of size 1..3."""
    buckets = {}

    def put(ms):
        key = tuple(int(v) for v in comp[list(ms)].sum(axis=0))
        buckets.setdefault(key, {}).setdefault(len(ms), []).append(ms)

    for a in reactive:
        put((a,))
    for ms in itertools.combinations_with_replacement(reactive, 2):
        put(ms)
    n = len(reactive)
    n_tri = n * (n + 1) * (n + 2) // 6
    if n_tri <= max_triples:
        for ms in itertools.combinations_with_replacement(reactive, 3):
            put(ms)
    else:
        seen = set()
        r = np.asarray(reactive)
        draws = r[rng.integers(0, n, size=(max_triples, 3))]
        for row in draws:
            ms = tuple(sorted(int(v) for v in row))
            if ms not in seen:
                seen.add(ms)
                put(ms)
    return buckets


def _draw_reactions(rng, comp, reactive, n_rx, size_prob=(0.15, 0.65, 0.20)):
    buckets = _multiset_buckets(rng, comp, reactive)
    by_size = {1: [], 2: [], 3: []}
    for key, d in buckets.items():
        if sum(len(v) for v in d.values()) >= 2:
            for s, lst in d.items():
                for ms in lst:
                    by_size[s].append((key, ms))
    out, seen = [], set()
    tries = 0
    while len(out) < n_rx:
        tries += 1
        if tries > 400 * n_rx + 10_000:
            raise RuntimeError("could not draw %d balanced reactions (got %d)" % (n_rx, len(out)))
        sl = int(rng.choice(3, p=size_prob)) + 1
        sr = int(rng.choice(3, p=size_prob)) + 1
        if not by_size[sl]:
            continue
        key, lhs = by_size[sl][int(rng.integers(len(by_size[sl])))]
        cands = buckets[key].get(sr, [])
        if not cands:
            continue
        rhs = cands[int(rng.integers(len(cands)))]
        if set(lhs) & set(rhs):
            continue
        tag = frozenset((lhs, rhs))
        if tag in seen:
            continue
        seen.add(tag)
        out.append((lhs, rhs))
    return out


def _side(ms):
    return [(s, ms.count(s)) for s in sorted(set(ms))]


def _arrhenius(rng):
    ln_a = rng.uniform(10.0, 35.0)
    beta = rng.uniform(-2.0, 3.0)
    ta = rng.uniform(0.0, 50.0) / R_KCAL
    return float(np.exp(ln_a)), float(beta), float(ta)


def _low_pressure(rng, arr):
    a, b, ta = arr
    return (float(a * np.exp(rng.uniform(0.0, 8.0))), float(b + rng.uniform(-1.0, 1.0)),
            float(ta + rng.uniform(-2000.0, 2000.0)))


def _troe_par(rng):
    has = rng.uniform() < 0.7
    return (rng.uniform(0.2, 0.9), rng.uniform(50.0, 500.0), rng.uniform(500.0, 3000.0),
            rng.uniform(2000.0, 8000.0) if has else 0.0, 1.0 if has else 0.0)


def _sri_par(rng):
    return (rng.uniform(0.5, 2.0), rng.uniform(100.0, 1000.0), rng.uniform(500.0, 3000.0),
            rng.uniform(0.5, 1.5), rng.uniform(-0.3, 0.3))


def _efficiencies(rng, n_species):
    k = int(rng.integers(3, 7))
    k = min(k, n_species)
    sp = sorted(int(s) for s in rng.choice(n_species, size=k, replace=False))
    return [(s, float(rng.uniform(0.5, 5.0))) for s in sp]


def _plog_table(rng, arr, pressures_atm=(0.1, 1.0, 10.0, 100.0)):
    a, b, ta = arr
    rows = []
    for p in pressures_atm:
        rows.append((p * P_ATM, float(a * np.exp(rng.uniform(-2.0, 2.0))),
                     float(b + rng.uniform(-0.5, 0.5)),
                     float(max(0.0, ta + rng.uniform(-1000.0, 1000.0)))))
    return rows


def _cheb_table(rng, n_t=7, n_p=3):
    eta = np.empty((n_t, n_p))
    for i in range(n_t):
        for j in range(n_p):
            eta[i, j] = rng.uniform(-1.0, 1.0) / ((i + 1) * (j + 1))
    eta[0, 0] = rng.uniform(6.0, 12.0)
    lim = (300.0, 3000.0, 0.01 * P_ATM, 100.0 * P_ATM)
    return (n_t, n_p, lim, eta)


def make_mechanism(cfg) -> Mechanism:
    """One of BASELINE.json's synthetic mechanisms (cfg = 0..3 or a `Config`)."""
    if not isinstance(cfg, Config):
        cfg = CONFIGS[int(cfg)]
    rng = np.random.default_rng(cfg.seed)
    names, comp, w, lo, hi, tm = _make_species(rng, cfg.elements, cfg.max_atoms, cfg.n_species)
    ns = cfg.n_species
    reactive = list(range(ns - 1))                   # N2 (last) is inert
    rx = _draw_reactions(rng, comp, reactive, cfg.n_reactions)
    kinds = ([THIRD_BODY] * cfg.n_third_body + ["troe"] * cfg.n_troe + ["lind"] * cfg.n_lindemann
             + ["sri"] * cfg.n_sri + ["chem"] * cfg.n_chem_act + [PLOG] * cfg.n_plog
             + [CHEBYSHEV] * cfg.n_cheb)
    kinds += [ELEMENTARY] * (cfg.n_reactions - len(kinds))
    kinds = [kinds[i] for i in rng.permutation(len(kinds))]
    b = MechanismBuilder(names, cfg.elements, comp, w, lo, hi, tm, label=cfg.name)
    for (lhs, rhs), kind in zip(rx, kinds):
        arr = _arrhenius(rng)
        kw = {}
        if kind == THIRD_BODY:
            kw = dict(rxn_type=THIRD_BODY, eff=_efficiencies(rng, ns))
        elif kind in ("troe", "lind", "sri", "chem"):
            kw = dict(rxn_type=CHEM_ACTIVATED if kind == "chem" else FALLOFF,
                      arr_lo=_low_pressure(rng, arr), eff=_efficiencies(rng, ns))
            if kind in ("troe", "chem"):
                kw.update(falloff_form=TROE, falloff_par=_troe_par(rng))
            elif kind == "sri":
                kw.update(falloff_form=SRI, falloff_par=_sri_par(rng))
            else:
                kw.update(falloff_form=LINDEMANN)
        elif kind == PLOG:
            kw = dict(rxn_type=PLOG, plog=_plog_table(rng, arr))
        elif kind == CHEBYSHEV:
            kw = dict(rxn_type=CHEBYSHEV, cheb=_cheb_table(rng))
        b.add(_side(lhs), _side(rhs), arr, **kw)
    return b.build()


def make_tiny_mechanism(seed=0, n_species=9, last_reacts=True) -> Mechanism:
    """Small mechanism that exercises every reaction type, falloff form, reverse
    treatment and third-body variant of the paper at least once (test input)."""
    rng = np.random.default_rng(977 + seed)
    elements = ("H", "O")
    names, comp, w, lo, hi, tm = _make_species(rng, elements, 3, n_species,
                                               t_mid_choices=(900.0, 1000.0, 1300.0),
                                               n2_last=False)
    reactive = list(range(n_species if last_reacts else n_species - 1))
    plan = []
    for form, par in ((LINDEMANN, None), (TROE, "troe"), (TROE, "troe_no_t2"), (SRI, "sri")):
        for rtype in (FALLOFF, CHEM_ACTIVATED):
            for tb in ("mix", "single"):
                plan.append(("fall", rtype, form, par, tb))
    plan += [("tb", "mix"), ("tb", "single"), ("tb", "unit"), ("plog",), ("plog",), ("cheb",),
             ("cheb",), ("elem", REV_FROM_KC), ("elem", REV_FROM_KC), ("elem", REV_EXPLICIT),
             ("elem", IRREVERSIBLE), ("elem", REV_FROM_KC)]
    rx = _draw_reactions(rng, comp, reactive, len(plan), size_prob=(0.25, 0.5, 0.25))
    b = MechanismBuilder(names, elements, comp, w, lo, hi, tm, label="tiny%d" % seed)
    rev_cycle = itertools.cycle([REV_FROM_KC, REV_FROM_KC, REV_EXPLICIT, IRREVERSIBLE])
    for (lhs, rhs), item in zip(rx, plan):
        arr = _arrhenius(rng)
        kw = {}
        if item[0] == "fall":
            _, rtype, form, par, tb = item
            kw = dict(rxn_type=rtype, falloff_form=form, arr_lo=_low_pressure(rng, arr),
                      rev_type=next(rev_cycle))
            if par == "troe":
                p = list(_troe_par(rng)); p[3], p[4] = rng.uniform(2000.0, 8000.0), 1.0
                kw["falloff_par"] = tuple(p)
            elif par == "troe_no_t2":
                p = list(_troe_par(rng)); p[3], p[4] = 0.0, 0.0
                kw["falloff_par"] = tuple(p)
            elif par == "sri":
                kw["falloff_par"] = _sri_par(rng)
            if tb == "mix":
                kw["eff"] = _efficiencies(rng, n_species)
            else:
                kw["tb_species"] = int(rng.integers(n_species))
        elif item[0] == "tb":
            kw = dict(rxn_type=THIRD_BODY, rev_type=next(rev_cycle))
            if item[1] == "mix":
                eff = _efficiencies(rng, n_species)
                if not any(s == n_species - 1 for s, _ in eff):   # exercise alpha_{i,Ns} != 1
                    eff.append((n_species - 1, float(rng.uniform(0.5, 5.0))))
                kw["eff"] = sorted(eff)
            elif item[1] == "single":
                kw["tb_species"] = int(rng.integers(n_species))
        elif item[0] == "plog":
            kw = dict(rxn_type=PLOG, plog=_plog_table(rng, arr), rev_type=next(rev_cycle))
        elif item[0] == "cheb":
            kw = dict(rxn_type=CHEBYSHEV, cheb=_cheb_table(rng, 5, 4), rev_type=next(rev_cycle))
        else:
            kw = dict(rev_type=item[1])
        if kw.get("rev_type", REV_FROM_KC) == REV_EXPLICIT:
            kw["arr_rev"] = _arrhenius(rng)
        b.add(_side(lhs), _side(rhs), arr, **kw)
    return b.build()


# ----------------------------------------------------------------------------- states
def make_states(n_species, n_states, seed, t_range=(800.0, 2500.0), p_range_atm=(1.0, 50.0),
                alpha=0.5, floor=1e-20):
    """(T[n], P[n] in Pa, Y[n][n_species]) drawn as BASELINE.json config 0 states."""
    rng = np.random.default_rng(seed)
    T = rng.uniform(t_range[0], t_range[1], size=n_states)
    P = P_ATM * np.exp(rng.uniform(np.log(p_range_atm[0]), np.log(p_range_atm[1]), size=n_states))
    Y = rng.gamma(alpha, 1.0, size=(n_states, n_species))      # Dirichlet via normalised gammas
    Y /= Y.sum(axis=1, keepdims=True)
    Y = np.maximum(Y, floor)
    Y /= Y.sum(axis=1, keepdims=True)
    big = np.argmax(Y, axis=1)
    rows = np.arange(n_states)
    last = Y[:, -1].copy()
    Y[:, -1] = Y[rows, big]
    Y[rows, big] = last
    # the swap is a no-op where the last slot already holds the maximum
    return np.ascontiguousarray(T), np.ascontiguousarray(P), np.ascontiguousarray(Y)


def config_states(cfg, n_states=None):
    if not isinstance(cfg, Config):
        cfg = CONFIGS[int(cfg)]
    n = cfg.n_states if n_states is None else int(n_states)
    return make_states(cfg.n_species, n, cfg.seed + 1000)
