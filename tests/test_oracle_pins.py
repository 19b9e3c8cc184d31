"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

The paper prints no worked numeric example (no table of rates or Jacobian entries), so
every pin here is a closed form, an invariant, a special case that reduces to a textbook
or library routine, or the plain definition J = df/dPhi by complex step.  Each test names
the passage it checks.  Nothing here re-types the oracle's own formula and nothing comes
from the CUDA path.
"""
import numpy as np
import pytest

from oracle.oracle import Oracle, as_matrix
from paper_1605_03262_b200 import synth
from paper_1605_03262_b200.mechanism import (CHEBYSHEV, CHEM_ACTIVATED, ELEMENTARY, FALLOFF,
                                             IRREVERSIBLE, LINDEMANN, PLOG, REV_EXPLICIT,
                                             REV_FROM_KC, SRI, THIRD_BODY, TROE, MechanismBuilder)

RU = 8314.46261815324
PATM = 101325.0


def const_cp_species(names, weights, cp_over_R, a5, a6, t_mid=1000.0):
    """Species with constant C_p/R (a1..a4 = 0), identical in both ranges."""
    ns = len(names)
    a = np.zeros((ns, 7))
    a[:, 0], a[:, 5], a[:, 6] = cp_over_R, a5, a6
    comp = np.eye(ns, dtype=np.int32)
    return dict(species_names=names, element_names=["E%d" % i for i in range(ns)],
                composition=comp, mol_wt=np.asarray(weights, float), nasa_lo=a, nasa_hi=a.copy(),
                t_mid=np.full(ns, t_mid))


# ------------------------------------------------------------------ P2 thermo (Eqs. 9-11, 27, 74)
def test_thermo_derivative_identities(tiny_mechs):
    """dH/dT = Cp and dS/dT = Cp/T (thermodynamics), dB/dT of Eq. 74 = d/dT of Eq. 27, all by
    complex step of the oracle's own polynomials; B = S/R - H/(RT) - ln T (Eqs. 24-27)."""
    h = 1e-30
    for m in tiny_mechs:
        o = Oracle(m)
        for T in (350.0, 899.0, 901.0, 1000.0, 1450.0, 3000.0):
            re, im = o.species_thermo(T, h)
            cp, H, S, B, dB = re
            np.testing.assert_allclose(im[1] / h, cp, rtol=1e-13)          # dH/dT = Cp
            np.testing.assert_allclose(im[2] / h, cp / T, rtol=1e-13)      # dS/dT = Cp/T
            np.testing.assert_allclose(im[3] / h, dB, rtol=1e-12, atol=1e-18)
            np.testing.assert_allclose(B, S - H / T - np.log(T), rtol=1e-13, atol=1e-12)


def test_thermo_constant_cp_textbook():
    """Constant-cp species: H/R = c T + a5, S/R = c ln T + a6 (textbook ideal gas)."""
    sp = const_cp_species(["A", "B"], [10.0, 20.0], [2.5, 3.5], [100.0, -2000.0], [3.0, 5.0])
    b = MechanismBuilder(**sp)
    b.add([(0, 2)], [(1, 1)], (1.0, 0.0, 0.0))
    o = Oracle(b.build())
    for T in (400.0, 1500.0):
        re, _ = o.species_thermo(T)
        np.testing.assert_allclose(re[0], [2.5, 3.5], rtol=0)
        np.testing.assert_allclose(re[1], [2.5 * T + 100.0, 3.5 * T - 2000.0], rtol=1e-15)
        np.testing.assert_allclose(re[2], [2.5 * np.log(T) + 3.0, 3.5 * np.log(T) + 5.0], rtol=1e-15)


def test_enthalpy_is_integral_of_cp(tiny_mechs):
    """h(Tb) - h(Ta) = int cp dT by Gauss-Legendre quadrature (inside one NASA range)."""
    m = tiny_mechs[0]
    o = Oracle(m)
    x, wq = np.polynomial.legendre.leggauss(12)
    for Ta, Tb in ((300.0, 850.0), (1400.0, 4000.0)):
        Tq = 0.5 * (Tb - Ta) * x + 0.5 * (Tb + Ta)
        cpq = np.array([o.species_thermo(t)[0][0] for t in Tq])          # [q][ns]
        integral = 0.5 * (Tb - Ta) * (wq[:, None] * cpq).sum(0)
        dH = o.species_thermo(Tb)[0][1] - o.species_thermo(Ta)[0][1]
        np.testing.assert_allclose(dH, integral, rtol=1e-12)


# ------------------------------------------------------------------ P3 equilibrium constant
def test_Kc_from_gibbs(tiny_mechs):
    """K_c of Eqs. 26-27 equals K_p (p_atm/RT)^sum(nu) with K_p = exp(dS/R - dH/RT), Eqs. 24-25,
    assembled here from S/R and H/R (Eqs. 10-11)."""
    for m in tiny_mechs:
        o = Oracle(m)
        T, P, Y = synth.make_states(m.n_species, 6, 11)
        d = o.details(T, P, Y)
        for s in range(len(T)):
            re, _ = o.species_thermo(T[s])
            g = re[2] - re[1] / T[s]                                        # S/R - H/(RT)
            for i in range(m.n_reactions):
                if m.rev_type[i] != REV_FROM_KC:
                    assert d["Kc"][s, i] == 0.0
                    continue
                nu = np.zeros(m.n_species)
                for e in range(m.prod_ptr[i], m.prod_ptr[i + 1]):
                    nu[m.prod_spec[e]] += m.prod_nu[e]
                for e in range(m.reac_ptr[i], m.reac_ptr[i + 1]):
                    nu[m.reac_spec[e]] -= m.reac_nu[e]
                Kp = np.exp(np.dot(nu, g))
                Kc = Kp * (PATM / (RU * T[s])) ** nu.sum()
                assert d["Kc"][s, i] == pytest.approx(Kc, rel=1e-12)
                assert d["kr"][s, i] == pytest.approx(d["kf"][s, i] / Kc, rel=1e-12)


# ------------------------------------------------------------------ P4 Arrhenius (Eqs. 21-22)
def test_arrhenius_variants():
    """The five evaluation variants of Eq. 22 against A*T**beta*exp(-Ta/T) in numpy."""
    sp = const_cp_species(["A", "B"], [10.0, 10.0], [2.5, 2.5], [0.0, 0.0], [1.0, 1.0])
    pars = [(3.0e5, 0.0, 0.0), (2.0e3, 1.7, 0.0), (5.0e9, -1.2, 8000.0), (7.0e12, 0.0, 15000.0),
            (4.0, 2.0, 0.0), (9.0e7, -1.0, 0.0)]
    b = MechanismBuilder(**sp)
    for p in pars:
        b.add([(0, 1)], [(1, 1)], p, rev_type=IRREVERSIBLE)
    o = Oracle(b.build())
    T = np.array([300.0, 1234.5, 2500.0])
    d = o.details(T, np.full(3, PATM), np.tile([0.4, 0.6], (3, 1)))
    for i, (A, beta, Ta) in enumerate(pars):
        ref = A * T ** beta * np.exp(-Ta / T)
        np.testing.assert_allclose(d["kf"][:, i], ref, rtol=1e-13)
        if Ta == 0.0 and beta == 2.0:
            np.testing.assert_allclose(d["kf"][:, i], A * T * T, rtol=1e-13)   # A prod^beta T
    assert np.all(d["kr"] == 0.0)


# ------------------------------------------------------------------ P5 PLOG (Eqs. 37-39, 105)
def _two_species_builder():
    return MechanismBuilder(**const_cp_species(["A", "B", "I"], [10.0, 10.0, 28.0],
                                               [3.0, 4.0, 3.5], [1000.0, -500.0, 0.0],
                                               [20.0, 22.0, 23.0]))


def test_plog_reduces_and_interpolates():
    arr = (3.0e8, 0.7, 6000.0)
    arr2 = (9.0e9, -0.3, 9000.0)
    p = [0.1 * PATM, 1.0 * PATM, 10.0 * PATM]
    b = _two_species_builder()
    b.add([(0, 1)], [(1, 1)], arr, rxn_type=PLOG, plog=[(pp,) + arr for pp in p])      # same k at all p
    b.add([(0, 1)], [(1, 1)], arr)                                                     # elementary twin
    b.add([(0, 1)], [(1, 1)], arr, rxn_type=PLOG, plog=[(p[0],) + arr, (p[1],) + arr2, (p[2],) + arr])
    o = Oracle(b.build())
    T = np.array([900.0, 1600.0])
    Y = np.tile([0.3, 0.2, 0.5], (2, 1))
    k = lambda a, T: a[0] * T ** a[1] * np.exp(-a[2] / T)
    # identical Arrhenius at every pressure == elementary reaction, at any pressure
    for P in (0.05 * PATM, 0.5 * PATM, 3.0 * PATM, 50.0 * PATM):
        d = o.details(T, np.full(2, P), Y)
        np.testing.assert_allclose(d["kf"][:, 0], d["kf"][:, 1], rtol=1e-13)
    J = as_matrix(o.jacobian(T, np.full(2, 0.5 * PATM), Y), 3)
    # P = p_k returns k_k; continuity across the interval boundary
    d = o.details(T, np.full(2, p[1]), Y)
    np.testing.assert_allclose(d["kf"][:, 2], k(arr2, T), rtol=1e-13)
    lo = o.details(T, np.full(2, p[1] * (1 - 1e-12)), Y)["kf"][:, 2]
    hi = o.details(T, np.full(2, p[1] * (1 + 1e-12)), Y)["kf"][:, 2]
    np.testing.assert_allclose(lo, hi, rtol=1e-10)
    # geometric mean of pressures -> geometric mean of rates (Eq. 39 with weight 1/2)
    d = o.details(T, np.full(2, np.sqrt(p[0] * p[1])), Y)
    np.testing.assert_allclose(d["kf"][:, 2], np.sqrt(k(arr, T) * k(arr2, T)), rtol=1e-12)
    # outside the table the end value is held (reading C6)
    d = o.details(T, np.full(2, 1e-3 * PATM), Y)
    np.testing.assert_allclose(d["kf"][:, 2], k(arr, T), rtol=1e-13)
    assert np.isfinite(J).all()


# ------------------------------------------------------------------ P6 Chebyshev (Eqs. 40-43, 110)
def test_chebyshev_against_numpy_chebval2d():
    """Eq. 40 with the recurrence for Eq. 41 against numpy's Chebyshev evaluation."""
    rng = np.random.default_rng(3)
    nT, nP = 6, 4
    eta = rng.uniform(-1, 1, size=(nT, nP)); eta[0, 0] = 8.0
    lim = (300.0, 3000.0, 0.01 * PATM, 100.0 * PATM)
    b = _two_species_builder()
    b.add([(0, 1)], [(1, 1)], (1.0, 0.0, 0.0), rxn_type=CHEBYSHEV, cheb=(nT, nP, lim, eta))
    o = Oracle(b.build())
    T = np.array([300.0, 777.0, 1500.0, 3000.0])
    P = np.array([0.01, 0.3, 7.0, 100.0]) * PATM
    d = o.details(T, P, np.tile([0.3, 0.2, 0.5], (4, 1)))
    Tr = (2.0 / T - 1 / lim[0] - 1 / lim[1]) / (1 / lim[1] - 1 / lim[0])
    Pr = (2 * np.log10(P) - np.log10(lim[2]) - np.log10(lim[3])) / (np.log10(lim[3]) - np.log10(lim[2]))
    ref = 10.0 ** np.polynomial.chebyshev.chebval2d(Tr, Pr, eta)
    np.testing.assert_allclose(d["kf"][:, 0], ref, rtol=1e-12)
    # Eq. 41 itself at interior points: cos((n-1) arccos x)
    x = Tr[1]
    direct = sum(eta[a, bb] * np.cos(a * np.arccos(x)) * np.cos(bb * np.arccos(Pr[1]))
                 for a in range(nT) for bb in range(nP))
    assert d["kf"][1, 0] == pytest.approx(10.0 ** direct, rel=1e-12)


def test_chebyshev_2x1_is_arrhenius():
    """N_T = 2, N_p = 1: T~ is affine in 1/T, so Eq. 40 is an Arrhenius rate with beta = 0;
    rates AND Jacobian (Eq. 110 vs Eq. 65) must equal those of the elementary twin."""
    lim = (300.0, 3000.0, 0.01 * PATM, 100.0 * PATM)
    e11, e21 = 7.5, -1.3
    a = 2.0 / (1 / lim[1] - 1 / lim[0])
    bb = -(1 / lim[0] + 1 / lim[1]) / (1 / lim[1] - 1 / lim[0])
    A = 10.0 ** (e11 + e21 * bb)
    Ta = -np.log(10.0) * e21 * a
    J = []
    for kind in ("cheb", "arr"):
        b = _two_species_builder()
        if kind == "cheb":
            b.add([(0, 1)], [(1, 1)], (1.0, 0.0, 0.0), rxn_type=CHEBYSHEV,
                  cheb=(2, 1, lim, [[e11], [e21]]))
        else:
            b.add([(0, 1)], [(1, 1)], (A, 0.0, Ta))
        o = Oracle(b.build())
        T = np.array([650.0, 1800.0]); P = np.array([2.0, 30.0]) * PATM
        Y = np.tile([0.3, 0.2, 0.5], (2, 1))
        J.append((o.source(T, P, Y), o.jacobian(T, P, Y)))
    np.testing.assert_allclose(J[0][0]["rf"], J[1][0]["rf"], rtol=1e-12)
    np.testing.assert_allclose(J[0][1], J[1][1], rtol=1e-9, atol=1e-9 * np.abs(J[1][1]).max())


# ------------------------------------------------------------------ P7 third body (Eqs. 28-30, 81)
def test_third_body_unit_efficiencies_and_single_species():
    b = _two_species_builder()
    b.add([(0, 1)], [(1, 1)], (1e6, 0.0, 1000.0), rxn_type=THIRD_BODY)                  # all alpha = 1
    b.add([(0, 1)], [(1, 1)], (1e6, 0.0, 1000.0), rxn_type=THIRD_BODY, tb_species=2)    # [X]_i = [X_I]
    b.add([(0, 1)], [(1, 1)], (1e6, 0.0, 1000.0), rxn_type=THIRD_BODY, eff=[(0, 2.5), (2, 0.4)])
    m = b.build()
    o = Oracle(m)
    T, P, Y = synth.make_states(3, 5, 2)
    src = o.source(T, P, Y)
    W = 1.0 / (Y / m.mol_wt).sum(1)
    rho = P * W / (RU * T)
    X = rho[:, None] * Y / m.mol_wt
    np.testing.assert_allclose(src["cmod"][:, 0], P / (RU * T), rtol=1e-13)              # Eq. 29
    np.testing.assert_allclose(src["cmod"][:, 1], X[:, 2], rtol=1e-13)                   # Eq. 30
    np.testing.assert_allclose(src["cmod"][:, 2], 2.5 * X[:, 0] + X[:, 1] + 0.4 * X[:, 2], rtol=1e-13)


def test_unit_efficiency_third_body_has_no_Y_dependence_in_c():
    """Eq. 81 / Appendix B: with all alpha = 1, c = p/(RT) does not depend on Y, so the Jacobian
    Y-columns equal those of the elementary reaction scaled by p/(RT)."""
    def jac(rtype, A):
        b = _two_species_builder()
        b.add([(0, 1)], [(1, 1)], (A, 0.5, 2000.0), rxn_type=rtype)
        o = Oracle(b.build())
        return as_matrix(o.jacobian([1100.0], [3 * PATM], [[0.3, 0.2, 0.5]]), 3)[0]
    M = 3 * PATM / (RU * 1100.0)
    Jtb = jac(THIRD_BODY, 1e5)
    Jel = jac(ELEMENTARY, 1e5 * M)
    np.testing.assert_allclose(Jtb[:, 1:], Jel[:, 1:], rtol=1e-12, atol=1e-12 * np.abs(Jel).max())


# ------------------------------------------------------------------ P8 falloff (Eqs. 20, 31-36)
def _falloff_mech(form, par, rtype=FALLOFF):
    b = _two_species_builder()
    b.add([(0, 2)], [(1, 1)], (4.0e10, 0.3, 3000.0), rxn_type=rtype, falloff_form=form,
          falloff_par=par, arr_lo=(6.0e13, -0.5, 2500.0), eff=[(1, 3.0)])
    return b.build()


def test_falloff_forms_against_standard_expressions():
    T, P, Y = synth.make_states(3, 12, 4, p_range_atm=(0.01, 200.0))
    troe = (0.6, 120.0, 1500.0, 5000.0, 1.0)
    sri = (1.2, 500.0, 1800.0, 0.9, 0.15)
    for rtype in (FALLOFF, CHEM_ACTIVATED):
        # Lindemann: F = 1
        o = Oracle(_falloff_mech(LINDEMANN, (0, 0, 0, 0, 0), rtype))
        d, s = o.details(T, P, Y), o.source(T, P, Y)
        np.testing.assert_array_equal(d["F"][:, 0], 1.0)
        Pr = d["Pr"][:, 0]
        ref = Pr / (1 + Pr) if rtype == FALLOFF else 1 / (1 + Pr)
        np.testing.assert_allclose(s["cmod"][:, 0], ref, rtol=1e-13)
        k0 = 6.0e13 * T ** -0.5 * np.exp(-2500.0 / T)
        kinf = 4.0e10 * T ** 0.3 * np.exp(-3000.0 / T)
        np.testing.assert_allclose(Pr, k0 / kinf * d["Xi"][:, 0], rtol=1e-12)          # Eq. 31
        np.testing.assert_allclose(d["kf"][:, 0], kinf if rtype == FALLOFF else k0, rtol=1e-12)
        # Troe in the standard (c, n, d) form: Eq. 35's constants are 0.75 + 0.14*0.4 and 1.27 - 0.14*0.67
        o = Oracle(_falloff_mech(TROE, troe, rtype))
        d = o.details(T, P, Y)
        a, T3, T1, T2, _ = troe
        Fc = (1 - a) * np.exp(-T / T3) + a * np.exp(-T / T1) + np.exp(-T2 / T)
        c = -0.4 - 0.67 * np.log10(Fc)
        n = 0.75 - 1.27 * np.log10(Fc)
        f1 = (np.log10(d["Pr"][:, 0]) + c) / (n - 0.14 * (np.log10(d["Pr"][:, 0]) + c))
        np.testing.assert_allclose(d["F"][:, 0], 10.0 ** (np.log10(Fc) / (1 + f1 ** 2)), rtol=1e-12)
        # Troe without T**: last term of Eq. 33 omitted
        o = Oracle(_falloff_mech(TROE, (a, T3, T1, 0.0, 0.0), rtype))
        d = o.details(T, P, Y)
        Fc = (1 - a) * np.exp(-T / T3) + a * np.exp(-T / T1)
        c = -0.4 - 0.67 * np.log10(Fc); n = 0.75 - 1.27 * np.log10(Fc)
        f1 = (np.log10(d["Pr"][:, 0]) + c) / (n - 0.14 * (np.log10(d["Pr"][:, 0]) + c))
        np.testing.assert_allclose(d["F"][:, 0], 10.0 ** (np.log10(Fc) / (1 + f1 ** 2)), rtol=1e-12)
        # SRI, Eqs. 32, 36
        o = Oracle(_falloff_mech(SRI, sri, rtype))
        d = o.details(T, P, Y)
        Xs = 1 / (1 + np.log10(d["Pr"][:, 0]) ** 2)
        ref = sri[3] * T ** sri[4] * (sri[0] * np.exp(-sri[1] / T) + np.exp(-T / sri[2])) ** Xs
        np.testing.assert_allclose(d["F"][:, 0], ref, rtol=1e-12)


def test_falloff_pressure_limits():
    """P_r -> infinity: c -> F (k -> k_inf F); P_r -> 0: c -> P_r F (k -> k_0 [M] F)  (Eq. 20)."""
    m = _falloff_mech(LINDEMANN, (0, 0, 0, 0, 0))
    o = Oracle(m)
    Y = [[0.3, 0.2, 0.5]]
    hi = o.source([1200.0], [1e12 * PATM], Y)["cmod"][0, 0]
    assert hi == pytest.approx(1.0, rel=1e-6)
    d = o.details([1200.0], [1e-9 * PATM], Y)
    lo = o.source([1200.0], [1e-9 * PATM], Y)["cmod"][0, 0]
    assert lo == pytest.approx(d["Pr"][0, 0], rel=1e-6)


def test_sri_blending_by_its_special_cases():
    """Eq. 36 pinned by what it reduces to, not by re-typing it:
      P_r = 1       =>  X = 1 and F = d T^e (a e^{-b/T} + e^{-T/c}), no exponent left;
      P_r -> 0, oo  =>  X -> 0 and F -> d T^e;
      a = 1, b = 0, c -> oo, d = 1, e = 0  =>  F = 2^X, so 1/log2(F) - 1 = (log10 P_r)^2, which fixes
                        the form of X and that its logarithm is base 10 (reading C13)."""
    sri = (1.2, 500.0, 1800.0, 0.9, 0.15)
    a, b, c, d, e = sri
    Y = [[0.3, 0.2, 0.5]]
    for rtype in (FALLOFF, CHEM_ACTIVATED):
        o = Oracle(_falloff_mech(SRI, sri, rtype))
        for T in (700.0, 1300.0, 2400.0):
            P0 = 2.0 * PATM
            Pr0 = o.details([T], [P0], Y)["Pr"][0, 0]
            det = o.details([T], [P0 / Pr0], Y)                     # P_r is linear in P at fixed T, Y
            assert det["Pr"][0, 0] == pytest.approx(1.0, rel=1e-13)
            assert det["F"][0, 0] == pytest.approx(d * T ** e * (a * np.exp(-b / T) + np.exp(-T / c)), rel=1e-12)
            for P in (1e-200, 1e200):                               # |log10 P_r| ~ 200: X ~ 2.5e-5
                det = o.details([T], [P], Y)
                X = 1.0 / (1.0 + np.log10(det["Pr"][0, 0]) ** 2)
                assert X < 1e-4
                assert det["F"][0, 0] == pytest.approx(d * T ** e, rel=2e-4)
        o = Oracle(_falloff_mech(SRI, (1.0, 0.0, 1e300, 1.0, 0.0), rtype))
        T, P, Yr = synth.make_states(3, 16, 9, p_range_atm=(1e-3, 1e3))
        det = o.details(T, P, Yr)
        F, Pr = det["F"][:, 0], det["Pr"][:, 0]
        np.testing.assert_allclose(1.0 / np.log2(F) - 1.0, np.log10(Pr) ** 2, rtol=1e-9, atol=1e-11)



# ------------------------------------------------------------------ P9 conservation
@pytest.mark.parametrize("cfg", [0, 1])
def test_mass_and_element_conservation(cfg):
    """sum_k W_k wdot_k = 0 and sum_k n_ek wdot_k = 0 to 1e-12 relative (north_star);
    sum_k dY_k/dt = 0; c_p dT/dt + sum_k h_k dY_k/dt = 0 (Eq. 7 rearranged)."""
    m = synth.make_mechanism(cfg)
    o = Oracle(m)
    T, P, Y = synth.config_states(cfg, 64)
    s = o.source(T, P, Y)
    wd = s["wdot"]
    # the bound is on each reaction's contribution: per-reaction rates are balanced exactly,
    # so the residual is rounding of the sum, measured against sum |terms|
    mass = (wd * m.mol_wt).sum(1)
    assert np.all(np.abs(mass) <= 1e-12 * np.abs(wd * m.mol_wt).sum(1))
    for e in range(m.composition.shape[1]):
        el = (wd * m.composition[:, e]).sum(1)
        assert np.all(np.abs(el) <= 1e-12 * np.abs(wd * m.composition[:, e]).sum(1) + 1e-300)
    ydot = s["dydt"][:, 1:]
    assert np.all(np.abs(ydot.sum(1)) <= 1e-12 * np.abs(ydot).sum(1))
    for i in range(8):
        re, _ = o.species_thermo(T[i])
        cpk = RU * re[0] / m.mol_wt
        hk = RU * re[1] / m.mol_wt
        cp = (Y[i] * cpk).sum()
        resid = cp * s["dydt"][i, 0] + (hk * ydot[i]).sum()
        assert abs(resid) <= 1e-11 * np.abs(hk * ydot[i]).sum()


def test_conservation_all_reaction_types(tiny_mechs):
    for m in tiny_mechs:
        o = Oracle(m)
        T, P, Y = synth.make_states(m.n_species, 32, 9)
        wd = o.source(T, P, Y)["wdot"]
        assert np.all(np.abs((wd * m.mol_wt).sum(1)) <= 1e-12 * np.abs(wd * m.mol_wt).sum(1))
        for e in range(m.composition.shape[1]):
            assert np.all(np.abs((wd * m.composition[:, e]).sum(1))
                          <= 1e-12 * np.abs(wd * m.composition[:, e]).sum(1))


def test_wdot_is_stoichiometric_sum_of_rates(tiny_mechs):
    """Eq. 14-17 assembled here from the exported R_f, R_r, c with a dense nu matrix."""
    m = tiny_mechs[1]
    o = Oracle(m)
    T, P, Y = synth.make_states(m.n_species, 8, 1)
    s = o.source(T, P, Y)
    nu = np.zeros((m.n_species, m.n_reactions))
    for i in range(m.n_reactions):
        for e in range(m.prod_ptr[i], m.prod_ptr[i + 1]):
            nu[m.prod_spec[e], i] += m.prod_nu[e]
        for e in range(m.reac_ptr[i], m.reac_ptr[i + 1]):
            nu[m.reac_spec[e], i] -= m.reac_nu[e]
    q = s["cmod"] * (s["rf"] - s["rr"])
    ref = q @ nu.T
    scale = (np.abs(q)[:, None, :] * np.abs(nu)[None]).sum(2)
    assert np.all(np.abs(s["wdot"] - ref) <= 1e-13 * scale)


# ------------------------------------------------------------------ P10 equilibrium
def test_equilibrium_composition_gives_zero_net_rate():
    """A <=> B with [B]/[A] = K_c  =>  R_f = R_r (Eqs. 17-19, 23)."""
    b = MechanismBuilder(**const_cp_species(["A", "B", "I"], [10.0, 10.0, 28.0], [3.0, 4.0, 3.5],
                                            [1000.0, -500.0, 0.0], [20.0, 22.0, 23.0]))
    b.add([(0, 1)], [(1, 1)], (2.0e7, 0.4, 3000.0))
    o = Oracle(b.build())
    T = 1300.0
    Kc = o.details([T], [PATM], [[0.2, 0.2, 0.6]])["Kc"][0, 0]
    yA = 0.4 / (1 + Kc)
    s = o.source([T], [5 * PATM], [[yA, 0.4 - yA, 0.6]])
    assert abs(s["rf"][0, 0] - s["rr"][0, 0]) <= 1e-13 * s["rf"][0, 0]
    assert np.all(np.abs(s["dydt"][0]) <= 1e-12 * s["rf"][0, 0] * 10.0 / 1.0)


# ------------------------------------------------------------------ P13 closed-form Jacobian
def test_isomerisation_jacobian_by_hand():
    """A <=> B (explicit constant k_f, k_r), inert I last, constant-cp thermo.  With W_A = W_B:
    dY_A/dt = -k_f Y_A + k_r Y_B exactly, so all nine entries of the paper's Jacobian
    (Phi = {T, Y_A, Y_B}) follow by hand from Eqs. 7-8 and 44-49."""
    cA, cB, cI = 3.0, 4.5, 3.5
    hA5, hB5, hI5 = 1200.0, -800.0, 50.0
    WA, WI = 16.0, 28.0
    sp = const_cp_species(["A", "B", "I"], [WA, WA, WI], [cA, cB, cI], [hA5, hB5, hI5], [20., 21., 22.])
    kf, kr = 37.0, 11.0
    b = MechanismBuilder(**sp)
    b.add([(0, 1)], [(1, 1)], (kf, 0.0, 0.0), rev_type=REV_EXPLICIT, arr_rev=(kr, 0.0, 0.0))
    o = Oracle(b.build())
    T, P = 1234.0, 2.5 * PATM
    YA, YB, YI = 0.25, 0.15, 0.60
    J = as_matrix(o.jacobian([T], [P], [[YA, YB, YI]]), 3)[0]
    f = o.source([T], [P], [[YA, YB, YI]])["dydt"][0]
    cpA, cpB, cpI = RU * cA / WA, RU * cB / WA, RU * cI / WI
    hA, hB = RU * (cA * T + hA5) / WA, RU * (cB * T + hB5) / WA
    cp = YA * cpA + YB * cpB + YI * cpI
    YAdot = -kf * YA + kr * YB
    Tdot = -(hA - hB) * YAdot / cp
    np.testing.assert_allclose(f, [Tdot, YAdot, -YAdot, 0.0], rtol=1e-13, atol=1e-13 * abs(YAdot))
    ref = np.zeros((3, 3))
    ref[0, 0] = -(cpA - cpB) * YAdot / cp
    ref[0, 1] = -(hA - hB) * (-kf) / cp + (hA - hB) * YAdot * (cpA - cpI) / cp ** 2
    ref[0, 2] = -(hA - hB) * (kr) / cp + (hA - hB) * YAdot * (cpB - cpI) / cp ** 2
    ref[1] = [0.0, -kf, kr]
    ref[2] = [0.0, kf, -kr]
    scale = np.abs(ref).max()
    np.testing.assert_allclose(J[:3, :3], ref, rtol=1e-12, atol=1e-13 * scale)
    np.testing.assert_allclose(J[3, :3], 0.0, atol=1e-13 * scale)       # inert placeholder row
    np.testing.assert_array_equal(J[:, 3], 0.0)                         # column Ns is zero (C1)


# ------------------------------------------------------------------ P11, P12, P14 whole Jacobian
def _erel_paper(J, Jref):
    """Eq. 131 over the elements the paper keeps, |J_ij| >= ||J||_F / 1e20."""
    mask = np.abs(Jref) >= np.linalg.norm(Jref) / 1e20
    return np.linalg.norm((Jref[mask] - J[mask]) / Jref[mask]), int(mask.sum())


def _erel_filtered(J, Jref):
    """Eq. 131 over the elements the paper keeps AND that carry significant digits at all:
    |J_ij| >= 1e-8 max_j' |J_ij'| (reading C19b).  Every element of row i is a
    sum of terms of the size of that row's largest entries, so an element 1e-8 below them has lost 8
    of fp64's 16 digits to cancellation in BOTH Jacobians; on the seeded far-from-equilibrium states
    (norms ~1e24) the paper's filter alone keeps such noise (elements ~1e6 in rows ~1e21) and E_rel
    then measures rounding, not the formulas."""
    mask = np.abs(Jref) >= np.linalg.norm(Jref) / 1e20
    mask &= np.abs(Jref) >= 1e-8 * np.abs(Jref).max(axis=1, keepdims=True)
    return np.linalg.norm((Jref[mask] - J[mask]) / Jref[mask]), int(mask.sum())


def _assert_rows_and_columns(Ja, Jc, tol):
    """Per ROW and per COLUMN relative 2-norms (the whole-matrix norm is the energy row: it carries
    0.9999998 of ||J||_F on these states, so it says nothing about the species block, Eqs. 111-112).
    The column check leaves the energy row out.  A row or column of the reference that is exactly
    zero (inert species, the dependent column N_sp) must be exactly zero: no floor applies to it."""
    row_den = np.linalg.norm(Jc, axis=1)
    row_num = np.linalg.norm(Ja - Jc, axis=1)
    assert np.all(row_num <= tol * row_den), (row_num / np.maximum(row_den, 1e-300)).max()
    # element-wise against the largest entry of the element's row: an element is a rounded sum of terms
    # of the size of its row's largest entries (the alpha_k d_j part of Eq. 112 is in every column), so
    # this is what rounding allows; observed 7e-15 over all configurations
    rowmax = np.abs(Jc).max(axis=1, keepdims=True)
    assert np.all(np.abs(Ja - Jc) <= tol * rowmax)
    # columns of the species block: a column can consist of cancelled elements only (each far below its
    # row's scale), so the floor is the rounding of its elements, 64 eps ||rowmax||_2
    col_den = np.linalg.norm(Jc[1:], axis=0)
    col_num = np.linalg.norm(Ja[1:] - Jc[1:], axis=0)
    floor = 64 * 2.220446049250313e-16 * np.linalg.norm(rowmax[1:])
    assert np.all(col_num <= tol * col_den + floor), ((col_num - floor) / np.maximum(col_den, 1e-300)).max()


def test_jacobian_vs_complex_step_tiny(tiny_mechs):
    """Every reaction type / falloff form / reverse treatment: analytic columns match the
    complex-step derivative within 1e-8 relative (north_star; observed ~1e-14).  Per row and per
    column (energy row excluded) within 1e-12, so that the explicit-reverse (Eq. 69), irreversible and
    single-species third-body (Eq. 85) terms -- which only these mechanisms contain -- are pinned in the
    species rows themselves and not through their weight in the energy row."""
    for m in tiny_mechs:
        o = Oracle(m)
        T, P, Y = synth.make_states(m.n_species, 24, 21, t_range=(500.0, 2800.0),
                                    p_range_atm=(0.05, 80.0))
        Ja = as_matrix(o.jacobian(T, P, Y), m.n_species)
        Jc = as_matrix(o.jacobian_complex_step(T, P, Y), m.n_species)
        for s in range(len(T)):
            for c in range(m.n_species):
                den = np.linalg.norm(Jc[s][:, c])
                assert np.linalg.norm(Ja[s][:, c] - Jc[s][:, c]) <= 1e-8 * den + 1e-300
            assert np.linalg.norm(Ja[s] - Jc[s]) <= 1e-12 * np.linalg.norm(Jc[s])
            _assert_rows_and_columns(Ja[s], Jc[s], 1e-12)
            assert np.all(Ja[s][:, -1] == 0.0) and np.all(Jc[s][:, -1] == 0.0)


@pytest.mark.parametrize("cfg,n", [(0, 32), (1, 8), (2, 4), (3, 2)])
def test_jacobian_paper_criterion_on_configs(cfg, n):
    """agreement within 0.001 % (E_rel <= 1e-5) between the analytical Jacobian
    and the reference derivative, on every benchmark configuration -- under reading C19b's filter;
    under the paper's filter alone the cancelled elements' rounding noise dominates E_rel (observed up
    to 3.5e-5 on single states), so that figure is only bounded loosely here and the per-row,
    per-column and per-element checks carry the weight (observed < 1e-14)."""
    m = synth.make_mechanism(cfg)
    o = Oracle(m)
    T, P, Y = synth.config_states(cfg, n)
    Ja = as_matrix(o.jacobian(T, P, Y), m.n_species)
    Jc = as_matrix(o.jacobian_complex_step(T, P, Y), m.n_species)
    for s in range(n):
        assert np.linalg.norm(Ja[s] - Jc[s]) <= 1e-11 * np.linalg.norm(Jc[s])
        _assert_rows_and_columns(Ja[s], Jc[s], 1e-12)
        e_c19b, _ = _erel_filtered(Ja[s], Jc[s])
        e_paper, _ = _erel_paper(Ja[s], Jc[s])
        assert e_c19b <= 1e-5
        assert e_paper <= 1e-3


def test_jacobian_species_columns_sum_to_zero(tiny_mechs):
    """sum over all N_sp species rows (incl. the placeholder row) of dYdot_k/dPhi_j = 0, because
    sum_k Ydot_k = 0 identically (sum_k W_k nu_ki = 0)."""
    for m in tiny_mechs[:2] + [synth.make_mechanism(0)]:
        o = Oracle(m)
        T, P, Y = synth.make_states(m.n_species, 8, 33)
        J = as_matrix(o.jacobian(T, P, Y), m.n_species)
        for s in range(len(T)):
            sp = J[s][1:, :]
            # each element of row k is a rounded sum of terms as large as that row's largest
            # entries, so the residual is measured against sum_k max_j |J_kj| (a wrong sign or
            # index anywhere leaves a residual of that size, 13 orders above this bound)
            scale = np.abs(sp).max(axis=1).sum()
            assert np.all(np.abs(sp.sum(0)) <= 1e-13 * scale + 1e-300)


def test_batch_independence_and_threads(tiny_mechs):
    """Appendix D's thread-safety lesson: results do not depend on batch split or thread count."""
    m = tiny_mechs[0]
    T, P, Y = synth.make_states(m.n_species, 16, 7)
    a = Oracle(m).jacobian(T, P, Y)
    o1 = Oracle(m, threads=1)
    b = np.concatenate([o1.jacobian(T[:5], P[:5], Y[:5]), o1.jacobian(T[5:], P[5:], Y[5:])])
    np.testing.assert_array_equal(a, b)


def test_oracle_regression_fixture():
    """tests/golden/oracle_tiny_jacobian.txt (written by tests/golden/make_golden.py, which calls only
    oracle/) freezes the oracle's arithmetic: an accidental change of oracle.c shows up here.  It is not
    a pin to the paper (which prints no worked example)."""
    import os
    from paper_1605_03262_b200 import synth as _synth
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_tiny_jacobian.txt")
    rows = [l for l in open(path).read().splitlines() if l and not l.startswith("#")]
    i = 0
    while i < len(rows):
        tag, seed, n, ns = rows[i].split()
        assert tag == "case"
        seed, n, ns = int(seed), int(n), int(ns)
        m = _synth.make_tiny_mechanism(seed)
        assert m.n_species == ns
        T, P, Y = _synth.make_states(ns, n, 4242 + seed)
        o = Oracle(m)
        src, J = o.source(T, P, Y), o.jacobian(T, P, Y)
        for s in range(n):
            dy = np.array([float(x) for x in rows[i + 1 + 2 * s].split()])
            Js = np.array([float(x) for x in rows[i + 2 + 2 * s].split()])
            assert np.allclose(src["dydt"][s], dy, rtol=1e-12, atol=1e-12 * np.abs(dy).max())
            assert np.linalg.norm(J[s] - Js) <= 1e-12 * np.linalg.norm(Js)
        i += 1 + 2 * n


# ---------------------------------------------------------------- forward-difference Jacobian (f2)
def test_fd_jacobian_approximates_the_derivative(tiny_mechs):
    """PAPER.md:817 (the paper's comparison method, Tables 4-5): the oracle's first-order forward
    difference (reading C21) against the plain definition J = df/dPhi by complex step.  A
    forward difference with increment D carries a truncation error D f''/2; here the measure is the
    paper's own (Eq. 132) plus a per-element bound at the row scale, loose enough for a
    first-order quotient (the paper reports FD errors that prevented its use as the reference,
    PAPER.md:765-780) and far too tight for a wrong sign, index, transposition or a missed Eq. 2
    compensation.  Column N_s is exactly zero; a mechanism without reactions gives exactly zero."""
    for m in tiny_mechs:
        o = Oracle(m)
        ns = m.n_species
        T, P, Y = synth.make_states(ns, 16, 33, t_range=(700.0, 2500.0), p_range_atm=(0.5, 20.0))
        Jf = as_matrix(o.jacobian_fd(T, P, Y, rtol=1e-8, atol=1e-12), ns)
        Jc = as_matrix(o.jacobian_complex_step(T, P, Y), ns)
        for s in range(len(T)):
            assert np.all(Jf[s][:, -1] == 0.0)
            assert np.linalg.norm(Jf[s] - Jc[s]) <= 2e-2 * np.linalg.norm(Jc[s])
            rowmax = np.abs(Jc[s]).max(axis=1, keepdims=True)
            assert np.all(np.abs(Jf[s] - Jc[s]) <= 0.2 * rowmax + 1e-300)
    # the Eq. 2 compensation: the mass-fraction columns differentiate along Y_j - Y_Ns.  Without it the
    # quotient would be the unconstrained partial derivative, which differs at first order
    m = tiny_mechs[0]
    o = Oracle(m)
    # C21: atol = 0 would give an absent species the increment 0 (a column of 0/0): refused; with atol > 0 a
    # state with a zero mass fraction has a finite forward difference
    with pytest.raises(ValueError):
        o.jacobian_fd(*synth.make_states(m.n_species, 2, 1), atol=0.0)
    Tz, Pz, Yz = synth.make_states(m.n_species, 3, 35)
    Yz[:, -1] += Yz[:, 0]
    Yz[:, 0] = 0.0
    assert np.all(np.isfinite(o.jacobian_fd(Tz, Pz, Yz, atol=1e-15)))
    ns = m.n_species
    T, P, Y = synth.make_states(ns, 4, 34)
    Jf = as_matrix(o.jacobian_fd(T, P, Y, rtol=1e-8, atol=1e-12), ns)
    for s in range(len(T)):
        f0 = o.source(T[s:s + 1], P[s:s + 1], Y[s:s + 1])["dydt"][0]
        j = int(np.argmax(Y[s, :-1]))
        d = np.sqrt(2.220446049250313e-16) * Y[s, j]
        Yp = Y[s].copy(); Yp[j] += d                       # no compensation
        g = (o.source(T[s:s + 1], P[s:s + 1], Yp[None])["dydt"][0] - f0) / d
        assert np.linalg.norm(g - Jf[s][:, j + 1]) > 1e-3 * np.linalg.norm(Jf[s][:, j + 1])
    # no reactions: f = 0 identically
    b = MechanismBuilder(["A", "B"], ["X"], np.array([[1], [1]], dtype=np.int32), np.array([10.0, 20.0]),
                         np.tile(np.array([3.5, 0, 0, 0, 0, 0, 0.0]), (2, 1)), np.tile(np.array([3.5, 0, 0, 0, 0, 0, 0.0]), (2, 1)),
                         np.array([1000.0, 1000.0]))
    m0 = b.build()
    J0 = Oracle(m0).jacobian_fd(np.array([1200.0]), np.array([101325.0]), np.array([[0.3, 0.7]]))
    assert np.all(J0 == 0.0)


def test_element_potential_composition_is_at_equilibrium():
    """Eqs. 18-19, 23-27 together, by a construction the oracle does not use: for ANY element potentials
    lambda the concentrations ln[X_k] = B_k + ln(p_atm/R) + sum_e lambda_e a_ke put every element-balanced
    reaction with k_r = k_f / K_c at equilibrium, R_f = R_r (tests/trajectory.py builds such states from the
    species B_k alone).  A wrong sign in B_k, a wrong power of p_atm/R in K_c (Eq. 26) or a wrong
    stoichiometric exponent in R_f / R_r breaks it for every reaction with sum nu != 0."""
    from trajectory import equilibrium_states
    m = synth.make_mechanism(1)
    o = Oracle(m)
    T, P, Y = equilibrium_states(m, [900.0, 1400.0, 2300.0], p_target_atm=3.0)
    src = o.source(T, P, Y)
    rev = np.asarray(m.rev_type) == REV_FROM_KC
    rf, rr = src["rf"][:, rev], src["rr"][:, rev]
    assert rev.sum() > 200
    assert np.all(np.abs(rf - rr) <= 1e-11 * (rf + rr))
