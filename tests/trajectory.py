"""Ignition-trajectory states for the parity tests.

The seeded workload states of synth.py are independent Dirichlet draws, far from equilibrium.  The
paper's states come from reactor trajectories (PaSR) and it singles out states near
equilibrium as the ones where difference quotients fail -- there R_f - R_r cancels.
This helper marches the constant-pressure source term dPhi/dt = f(Phi) (Eqs. 6-8) from a seeded state
towards equilibrium with the linearly implicit Euler method, (I - h J) dPhi = h f, and returns the
states it passes through.  It is test infrastructure: f and J come from the CPU oracle, nothing from
the CUDA path, and nothing here is used by the product.
"""
import numpy as np

from oracle.oracle import Oracle, as_matrix


def march_to_equilibrium(mech, T0, P0, Y0, n_steps=120, growth=1.6, max_rel_change=0.2):
    """Returns (T[k], P[k], Y[k][ns], cancel[k]) for k = 0 .. n_steps: the trajectory and, per state, the
    cancellation measure max_i |R_f - R_r| / max_i (R_f + R_r) (1 = far from equilibrium, -> 0 at it)."""
    o = Oracle(mech, threads=1)
    ns = mech.n_species
    T, Y = float(T0), np.array(Y0, dtype=np.float64)
    P = float(P0)
    Ts, Ys, cs = [], [], []
    h = None
    for _ in range(n_steps + 1):
        src = o.source(np.array([T]), np.array([P]), Y[None])
        rf, rr, c = src["rf"][0], src["rr"][0], src["cmod"][0]
        Ts.append(T); Ys.append(Y.copy())
        cs.append(float(np.abs(c * (rf - rr)).max() / max(np.abs(c * (rf + rr)).max(), 1e-300)))
        f = src["dydt"][0][:ns]                                   # unknowns: T, Y_1 .. Y_{Ns-1}
        J = as_matrix(o.jacobian(np.array([T]), np.array([P]), Y[None]), ns)[0][:ns, :ns]
        phi = np.concatenate([[T], Y[:ns - 1]])
        scale = np.maximum(np.abs(phi), 1e-6)
        if h is None:
            h = 1e-3 / max(np.abs(f / scale).max(), 1e-300)
        for _try in range(60):
            try:
                d = np.linalg.solve(np.eye(ns) - h * J, h * f)
            except np.linalg.LinAlgError:
                h *= 0.5
                continue
            if np.all(np.isfinite(d)) and np.abs(d / scale).max() <= max_rel_change:
                break
            h *= 0.5
        phi = phi + d
        T = float(min(max(phi[0], 300.0), 4500.0))
        Yn = np.maximum(phi[1:], 0.0)
        last = max(1.0 - Yn.sum(), 0.0)
        Y = np.concatenate([Yn, [last]])
        Y = np.maximum(Y / Y.sum(), 1e-30)
        Y /= Y.sum()
        h *= growth
    n = len(Ts)
    return np.array(Ts), np.full(n, P), np.array(Ys), np.array(cs)


def equilibrium_states(mech, temperatures, p_target_atm=10.0, floor=1e-30, perturb=0.0, seed=0):
    """States AT chemical equilibrium of every K_c-reversible reaction, from element potentials: for any
    vector lambda (one entry per element) the concentrations
        ln [X_k] = B_k(T) + ln(p_atm / R) + sum_e lambda_e a_ke     (B_k of Eq. 27 carries the -ln T of Eq. 26)
    satisfy prod_k [X_k]^nu_ki = K_c,i (Eq. 26) for every element-balanced reaction, i.e. R_f = R_r
    exactly: the cancellation the paper warns about.  lambda is chosen by least squares so
    that as many species as possible are of comparable size, then shifted along the atom count to the
    target pressure.  Mass fractions below `floor` are raised to it (those species leave equilibrium, the
    others stay); `perturb` multiplies every Y_k by (1 + perturb * U(-1, 1)) to step off the manifold.
    B_k comes from the oracle (test infrastructure)."""
    o = Oracle(mech, threads=1)
    ns = mech.n_species
    a = np.asarray(mech.composition, dtype=np.float64)                 # [ns][ne]
    rng = np.random.default_rng(seed)
    Ts, Ps, Ys = [], [], []
    for T in temperatures:
        B = o.species_thermo(float(T))[0][3]
        base = B + np.log(101325.0 / 8314.46261815324)
        # least squares: base + a lambda ~ const
        A1 = np.concatenate([a, -np.ones((ns, 1))], axis=1)
        sol = np.linalg.lstsq(A1, -base, rcond=None)[0]
        lam = sol[:-1]
        natoms = a.sum(axis=1)
        lo, hi = -200.0, 200.0
        for _ in range(200):                                            # bisection on the total concentration
            t = 0.5 * (lo + hi)
            lnX = base + a @ lam + t * natoms
            ctot = np.exp(np.minimum(lnX, 700.0)).sum()
            if ctot * 8314.46261815324 * T > p_target_atm * 101325.0:
                hi = t
            else:
                lo = t
        X = np.exp(base + a @ lam + 0.5 * (lo + hi) * natoms)
        Y = X * mech.mol_wt
        Y = Y / Y.sum()
        if perturb:
            Y = Y * (1.0 + perturb * rng.uniform(-1.0, 1.0, ns))
        Y = np.maximum(Y, floor)
        Y = Y / Y.sum()
        W = 1.0 / (Y / mech.mol_wt).sum()
        Ts.append(float(T)); Ys.append(Y)
        # the pressure that belongs to these concentrations: rho = sum_k [X_k] W_k with the unfloored X
        rho = (X * mech.mol_wt).sum()
        Ps.append(float(rho * 8314.46261815324 * T / W))
    return np.array(Ts), np.array(Ps), np.array(Ys)
