"""Plain data container for a kinetic model (species, NASA-7 thermo, reactions).

This module holds NO arithmetic of the method: it is only the description that
both the CUDA library (through ``binding.py``) and the CPU oracle (through
``oracle/oracle.py``) are handed.  Field meaning follows the paper's notation
(Sections 2.2-2.3):

  mol_wt[k]                 W_k, kg/kmol                        (Eq. 4)
  nasa_lo/hi[k][0..6]       a_{0..6,k} below / above t_mid[k]   (Eqs. 9-11)
  reac_* / prod_*           CSR lists of (species, nu') / (species, nu'')  (Eq. 15)
  rxn_type[i]               which case of Eq. 20 / Eqs. 37-43 applies
  rev_type[i]               irreversible / k_r = k_f/K_c (Eq. 23) / explicit Arrhenius
  arr_hi[i] = (A, beta, Ta) Eq. 21; the only set for non-falloff reactions,
                            k_inf for FALLOFF and CHEM_ACTIVATED
  arr_lo[i]                 k_0 (falloff / chemically activated only)
  arr_rev[i]                explicit reverse parameters (REV_EXPLICIT only)
  falloff_form[i], falloff_par[i][0..4]
                            Lindemann / Troe (a, T***, T*, T**, has_T**) /
                            SRI (a, b, c, d, e)                 (Eqs. 32-36)
  tb_species[i]             m >= 0: single species third body (Eq. 30); -1: mixture
  eff_*                     CSR list of (species, alpha_ij) for alpha_ij != 1 (Eq. 28)
  plog_*                    CSR list of (p [Pa], A, beta, Ta), ascending p (Eqs. 37-39)
  cheb_*                    N_T, N_p, (Tmin, Tmax, pmin, pmax), eta row-major (Eqs. 40-43)

Units: SI with kmol (J, kmol, m^3, K, Pa).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List

import numpy as np

# reaction types (Eq. 20 cases + Eqs. 37-43)
ELEMENTARY, THIRD_BODY, FALLOFF, CHEM_ACTIVATED, PLOG, CHEBYSHEV = range(6)
# reverse-rate treatment
IRREVERSIBLE, REV_FROM_KC, REV_EXPLICIT = range(3)
# falloff forms (Eq. 32)
LINDEMANN, TROE, SRI = range(3)


@dataclass
class Mechanism:
    species_names: List[str]
    element_names: List[str]
    composition: np.ndarray      # [ns][ne] int32, atoms of each element
    mol_wt: np.ndarray           # [ns]
    nasa_lo: np.ndarray          # [ns][7]
    nasa_hi: np.ndarray          # [ns][7]
    t_mid: np.ndarray            # [ns]
    reac_ptr: np.ndarray         # [nr+1] int32
    reac_spec: np.ndarray        # int32
    reac_nu: np.ndarray          # int32
    prod_ptr: np.ndarray
    prod_spec: np.ndarray
    prod_nu: np.ndarray
    rxn_type: np.ndarray         # [nr] int32
    rev_type: np.ndarray         # [nr] int32
    arr_hi: np.ndarray           # [nr][3]
    arr_lo: np.ndarray           # [nr][3]
    arr_rev: np.ndarray          # [nr][3]
    falloff_form: np.ndarray     # [nr] int32
    falloff_par: np.ndarray      # [nr][5]
    tb_species: np.ndarray       # [nr] int32
    eff_ptr: np.ndarray          # [nr+1] int32
    eff_spec: np.ndarray         # int32
    eff_val: np.ndarray          # float64
    plog_ptr: np.ndarray         # [nr+1] int32
    plog_p: np.ndarray           # float64, Pa
    plog_arr: np.ndarray         # [n][3]
    cheb_ptr: np.ndarray         # [nr+1] int32 offsets into cheb_eta
    cheb_nT: np.ndarray          # [nr] int32
    cheb_nP: np.ndarray          # [nr] int32
    cheb_lim: np.ndarray         # [nr][4] Tmin, Tmax, pmin, pmax
    cheb_eta: np.ndarray         # float64
    label: str = ""
    _keep: list = field(default_factory=list, repr=False)

    @property
    def n_species(self) -> int:
        return int(self.mol_wt.shape[0])

    @property
    def n_reactions(self) -> int:
        return int(self.rxn_type.shape[0])

    def normalized(self) -> "Mechanism":
        """Contiguous arrays of the dtypes the C interfaces expect."""
        f8 = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        i4 = lambda a: np.ascontiguousarray(a, dtype=np.int32)
        for name in ("mol_wt", "nasa_lo", "nasa_hi", "t_mid", "arr_hi", "arr_lo", "arr_rev",
                     "falloff_par", "eff_val", "plog_p", "plog_arr", "cheb_lim", "cheb_eta"):
            setattr(self, name, f8(getattr(self, name)))
        for name in ("composition", "reac_ptr", "reac_spec", "reac_nu", "prod_ptr", "prod_spec",
                     "prod_nu", "rxn_type", "rev_type", "falloff_form", "tb_species", "eff_ptr",
                     "eff_spec", "plog_ptr", "cheb_ptr", "cheb_nT", "cheb_nP"):
            setattr(self, name, i4(getattr(self, name)))
        self.plog_arr = self.plog_arr.reshape(-1, 3)
        return self


class MechanismBuilder:
    """Accumulates reactions one by one and emits the CSR arrays of `Mechanism`."""

    def __init__(self, species_names, element_names, composition, mol_wt, nasa_lo, nasa_hi, t_mid,
                 label=""):
        self.sp = dict(species_names=list(species_names), element_names=list(element_names),
                       composition=np.asarray(composition, dtype=np.int32),
                       mol_wt=np.asarray(mol_wt, dtype=np.float64),
                       nasa_lo=np.asarray(nasa_lo, dtype=np.float64),
                       nasa_hi=np.asarray(nasa_hi, dtype=np.float64),
                       t_mid=np.asarray(t_mid, dtype=np.float64))
        self.label = label
        self.rx = []

    def add(self, reactants, products, arr, rxn_type=ELEMENTARY, rev_type=REV_FROM_KC,
            arr_lo=(1.0, 0.0, 0.0), arr_rev=(1.0, 0.0, 0.0), falloff_form=LINDEMANN,
            falloff_par=(0, 0, 0, 0, 0), tb_species=-1, eff=(), plog=(), cheb=None):
        """reactants/products: lists of (species index, integer nu >= 1), distinct species."""
        self.rx.append(dict(reactants=list(reactants), products=list(products), arr=tuple(arr),
                            rxn_type=rxn_type, rev_type=rev_type, arr_lo=tuple(arr_lo),
                            arr_rev=tuple(arr_rev), falloff_form=falloff_form,
                            falloff_par=tuple(falloff_par), tb_species=tb_species,
                            eff=list(eff), plog=list(plog), cheb=cheb))
        return len(self.rx) - 1

    def build(self) -> Mechanism:
        nr = len(self.rx)

        def csr(key, width):
            ptr = [0]
            cols = [[] for _ in range(width)]
            for r in self.rx:
                for item in r[key]:
                    for c, v in zip(cols, item):
                        c.append(v)
                ptr.append(len(cols[0]))
            return ptr, cols

        rptr, (rs, rn) = csr("reactants", 2)
        pptr, (ps, pn) = csr("products", 2)
        eptr, (es, ev) = csr("eff", 2)
        lptr, (lp, la, lb, lt) = csr("plog", 4)
        cptr, eta = [0], []
        cnT, cnP, clim = [], [], []
        for r in self.rx:
            if r["cheb"] is None:
                cnT.append(0); cnP.append(0); clim.append((0.0, 0.0, 0.0, 0.0))
            else:
                nT, nP, lim, e = r["cheb"]
                e = np.asarray(e, dtype=np.float64).reshape(nT, nP)
                cnT.append(nT); cnP.append(nP); clim.append(tuple(lim)); eta.extend(e.ravel())
            cptr.append(len(eta))
        m = Mechanism(
            **self.sp,
            reac_ptr=np.array(rptr), reac_spec=np.array(rs, dtype=np.int32),
            reac_nu=np.array(rn, dtype=np.int32),
            prod_ptr=np.array(pptr), prod_spec=np.array(ps, dtype=np.int32),
            prod_nu=np.array(pn, dtype=np.int32),
            rxn_type=np.array([r["rxn_type"] for r in self.rx]),
            rev_type=np.array([r["rev_type"] for r in self.rx]),
            arr_hi=np.array([r["arr"] for r in self.rx], dtype=np.float64).reshape(nr, 3),
            arr_lo=np.array([r["arr_lo"] for r in self.rx], dtype=np.float64).reshape(nr, 3),
            arr_rev=np.array([r["arr_rev"] for r in self.rx], dtype=np.float64).reshape(nr, 3),
            falloff_form=np.array([r["falloff_form"] for r in self.rx]),
            falloff_par=np.array([r["falloff_par"] for r in self.rx],
                                 dtype=np.float64).reshape(nr, 5),
            tb_species=np.array([r["tb_species"] for r in self.rx]),
            eff_ptr=np.array(eptr), eff_spec=np.array(es, dtype=np.int32),
            eff_val=np.array(ev, dtype=np.float64),
            plog_ptr=np.array(lptr), plog_p=np.array(lp, dtype=np.float64),
            plog_arr=np.array(list(zip(la, lb, lt)), dtype=np.float64).reshape(-1, 3),
            cheb_ptr=np.array(cptr), cheb_nT=np.array(cnT), cheb_nP=np.array(cnP),
            cheb_lim=np.array(clim, dtype=np.float64).reshape(nr, 4),
            cheb_eta=np.array(eta, dtype=np.float64),
            label=self.label,
        )
        return m.normalized()
