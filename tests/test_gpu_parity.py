"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Tolerances (BASELINE.json north_star):
  rates R_f, R_r, c_i      element-wise relative 1e-12 (north_star), R_r included: the conditioning bound
                           of k_r = k_f / K_c, `kr_bound`, is several 1e-12, but the observed maximum is
                           3e-13, so the plain 1e-12 holds and is what is asserted
  wdot, dPhi/dt            1e-12 of the largest term summed, per state (C19: do not judge cancellation)
  Jacobian                 Frobenius-norm relative error per state <= 1e-10 (Eq. 132)
"""
import numpy as np
import pytest

from oracle.oracle import Oracle
from paper_1605_03262_b200 import synth
from paper_1605_03262_b200.mechanism import (CHEBYSHEV, ELEMENTARY, FALLOFF, PLOG, REV_FROM_KC, THIRD_BODY,
                                             TROE, MechanismBuilder)

pytestmark = pytest.mark.gpu

RATE_TOL = 1e-12
JAC_TOL = 1e-10
EPS = 2.220446049250313e-16


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.skip("no CUDA device")
    return t


@pytest.fixture(scope="module")
def PyJac():
    from paper_1605_03262_b200 import build
    build.build()
    from paper_1605_03262_b200.binding import PyJac as P
    return P


def dev(torch, *arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def kr_bound(oracle, T):
    """Conditioning of k_r = k_f / K_c with K_c from exp(sum_k nu_ki B_k) (Eqs. 23-27): each B_k is
    rounded at eps |B_k| (its a_5/T term reaches several hundred for large species), so two correct
    evaluation orders may differ by up to ~eps * sum|nu| * max|B_k| in the exponent.  Reported beside
    the observed error; NOT the tolerance (that is RATE_TOL)."""
    bmax = max(np.abs(oracle.species_thermo(float(t))[0][3]).max() for t in (T.min(), T.max()))
    return max(RATE_TOL, 8.0 * 6 * EPS * bmax)


RATES_OBSERVED = {}     # label -> largest relative errors of the rate arrays, next to the tolerance in force


def check_rates(torch, pj, o, T, P, Y, label=None):
    dT, dP, dY = dev(torch, T, P, Y)
    got = {k: v.cpu().numpy() for k, v in pj.eval_rates(dT, dP, dY).items()}
    dy = pj.eval_dydt(dT, dP, dY).cpu().numpy()
    ref = o.source(T, P, Y)
    tiny = 1e-300
    tol_r = RATE_TOL
    rel = lambda a, b: float((np.abs(a - b) / np.maximum(np.abs(b), tiny))[np.abs(b) > 0].max(initial=0.0))
    # production rates and source term: against the size of what was summed (C19); with reverse
    # rates entering, the bound is the reverse-rate one
    q = np.abs(ref["cmod"]) * (np.abs(ref["rf"]) + np.abs(ref["rr"]))
    scale_w = q.max(axis=1, keepdims=True)
    seen = dict(rf=rel(got["rf"], ref["rf"]), rr=rel(got["rr"], ref["rr"]), cmod=rel(got["cmod"], ref["cmod"]),
                wdot=float((np.abs(got["wdot"] - ref["wdot"]) / np.maximum(scale_w, tiny)).max(initial=0.0)),
                kr_bound=kr_bound(o, T))
    assert np.all(np.abs(got["rf"] - ref["rf"]) <= RATE_TOL * np.abs(ref["rf"]) + tiny)
    assert np.all(np.abs(got["rr"] - ref["rr"]) <= tol_r * np.abs(ref["rr"]) + tiny)
    assert np.all(np.abs(got["cmod"] - ref["cmod"]) <= RATE_TOL * np.abs(ref["cmod"]) + tiny)
    assert np.all(np.abs(got["wdot"] - ref["wdot"]) <= tol_r * scale_w + tiny)
    for name, part in (("dTdt", slice(0, 1)), ("dYdt", slice(1, None))):
        scale = np.abs(ref["dydt"][:, part]).max(axis=1, keepdims=True)
        term = np.maximum(scale, _dydt_term_scale(o, ref, T, P, Y, part))
        bound = max(tol_r, RATE_TOL) * term
        seen[name] = float((np.abs(dy[:, part] - ref["dydt"][:, part]) / np.maximum(term, tiny)).max(initial=0.0))
        assert np.all(np.abs(dy[:, part] - ref["dydt"][:, part]) <= bound + tiny)
    if label is not None:
        best = RATES_OBSERVED.setdefault(label, dict(seen))
        for k, v in seen.items():
            best[k] = max(best[k], v)
    return got, dy


def _dydt_term_scale(o, ref, T, P, Y, part):
    """size of the terms summed into dT/dt (Eq. 7) or dY_k/dt (Eq. 8), per state"""
    m = o.mech
    W = 1.0 / (Y / m.mol_wt).sum(1)
    rho = P * W / (8314.46261815324 * T)
    q = (np.abs(ref["cmod"]) * (np.abs(ref["rf"]) + np.abs(ref["rr"]))).max(axis=1)
    if part.start == 1:
        return (m.mol_wt.max() * q / rho)[:, None]
    out = np.empty(len(T))
    for s in range(len(T)):
        re, _ = o.species_thermo(float(T[s]))
        cp = (Y[s] * 8314.46261815324 * re[0] / m.mol_wt).sum()
        out[s] = np.abs(8314.46261815324 * re[1]).max() * q[s] / (rho[s] * cp)
    return out[:, None]


JVP_OBSERVED = {}   # config -> largest error of (J v)_r over max_c |J_rc| sum_c |v_c|
FD_OBSERVED = {}    # config -> largest forward-difference error over its bound (test_fd_jacobian_matches_oracle_fd)
OBSERVED = {}       # label -> largest errors seen, printed at the end of the module (pytest -s) and written to gpurun_out/


def jacobian_errors(J, Jr, ns):
    """Errors of a batch of GPU Jacobians against the oracle's, each as a maximum over the batch:
      fro   ||J - Jr||_F / ||Jr||_F per state (Eq. 132, north_star's wording).  On the seeded states the
            energy row carries 0.9999998 of ||Jr||_F, so this alone says nothing about the species block;
      row   per row r: ||J[r,:] - Jr[r,:]||_2 / ||Jr[r,:]||_2 (rows of the reference that are exactly
            zero -- an inert species, Eq. 112 with nu_ki = 0 -- must be exactly zero: counted in `zero_bad`);
      elem  per element: |J_rc - Jr_rc| / max_c' |Jr_rc'|.  An element of row r is a rounded sum of terms of
            the size of the row's largest entries (the alpha_r d_c part of Eq. 112 is in every column), so
            the row's largest entry is the scale rounding works at; elements far below it are cancelled
            sums that no evaluation order reproduces to a relative 1e-10;
      col   per column c with the energy row EXCLUDED: (||dJ[1:,c]||_2 - floor) / ||Jr[1:,c]||_2, floor =
            1e-13 ||rowmax[1:]||_2: a column can consist of cancelled elements only, the floor is their
            rounding (450 eps times the row scales)."""
    ld = ns + 1
    A = np.asarray(J).reshape(-1, ld, ld).transpose(0, 2, 1)      # [n][row][col]
    B = np.asarray(Jr).reshape(-1, ld, ld).transpose(0, 2, 1)
    D = A - B
    tiny = 1e-300
    fro = np.linalg.norm(D, axis=(1, 2)) / np.maximum(np.linalg.norm(B, axis=(1, 2)), tiny)
    row_den = np.linalg.norm(B, axis=2)
    row_num = np.linalg.norm(D, axis=2)
    zero_rows = row_den == 0.0
    zero_bad = int(np.count_nonzero(zero_rows & (np.abs(A).max(axis=2) != 0.0)))
    row = np.where(zero_rows, 0.0, row_num / np.maximum(row_den, tiny))
    rowmax = np.abs(B).max(axis=2, keepdims=True)
    elem = np.abs(D) / np.maximum(rowmax, tiny)
    elem = np.where(rowmax == 0.0, 0.0, elem)
    col_den = np.linalg.norm(B[:, 1:, :], axis=1)
    col_num = np.linalg.norm(D[:, 1:, :], axis=1)
    floor = 1e-13 * np.linalg.norm(rowmax[:, 1:, 0], axis=1)[:, None]
    col = np.maximum(col_num - floor, 0.0) / np.maximum(col_den, tiny)
    col = np.where(col_den == 0.0, np.where(col_num > floor, np.inf, 0.0), col)
    tcol = np.linalg.norm(D[:, 1:, 0], axis=1) / np.maximum(np.linalg.norm(B[:, 1:, 0], axis=1), tiny)
    return dict(fro=float(fro.max(initial=0.0)), row=float(row.max(initial=0.0)), elem=float(elem.max(initial=0.0)),
                col=float(col.max(initial=0.0)), tcol=float(tcol.max(initial=0.0)), zero_bad=zero_bad)


def assert_jacobian(J, Jr, ns, tol=JAC_TOL, label=None):
    """North_star's bound (Frobenius, 1e-10 per state) AND the same bound per row, per element against
    its row's scale, per species-block column and on the T column (Eq. 111) alone."""
    e = jacobian_errors(J, Jr, ns)
    if label is not None:
        best = OBSERVED.setdefault(label, dict(e))
        for k, v in e.items():
            best[k] = max(best[k], v)
    assert e["zero_bad"] == 0, e
    for k in ("fro", "row", "elem", "col", "tcol"):
        assert e[k] <= tol, (k, e)
    return e


def check_jacobian(torch, pj, o, T, P, Y, tol=JAC_TOL, label=None):
    dT, dP, dY = dev(torch, T, P, Y)
    J = pj.eval_jacobian(dT, dP, dY).cpu().numpy()
    Jr = o.jacobian(T, P, Y)
    assert np.all(np.isfinite(J))
    e = assert_jacobian(J, Jr, o.ns, tol, label)
    ld = o.ns + 1
    assert np.all(J.reshape(-1, ld, ld)[:, ld - 1, :] == 0.0)      # column Nsp is zero (C1)
    return J, e["fro"]


@pytest.fixture(scope="module", autouse=True)
def _report_observed():
    yield
    if not OBSERVED and not RATES_OBSERVED and not JVP_OBSERVED and not FD_OBSERVED:
        return
    import json
    import os
    if RATES_OBSERVED:
        print("\nobserved maxima of the rate arrays, GPU vs oracle (tolerance 1e-12; kr_bound = conditioning bound of k_r):")
        for k, v in sorted(RATES_OBSERVED.items()):
            print("%-28s " % k + " ".join("%s=%.2e" % (n, x) for n, x in sorted(v.items())))
    lines = ["%-28s " % k + " ".join("%s=%.2e" % (n, v[n]) for n in ("fro", "row", "elem", "col", "tcol"))
             for k, v in sorted(OBSERVED.items())]
    print("\nobserved maxima, GPU vs oracle (tolerance %.0e):\n" % JAC_TOL + "\n".join(lines))
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_observed.json"), "w") as f:
            json.dump(dict(jacobian=OBSERVED, rates=RATES_OBSERVED, fd_error_over_bound=FD_OBSERVED,
                           jvp_error_over_scale=JVP_OBSERVED), f, indent=1,
                      sort_keys=True)
    except OSError:
        pass


# ---------------------------------------------------------------------------------- small cases
def test_tiny_mechanisms_all_reaction_types(torch, PyJac, tiny_mechs):
    """Every reaction type, falloff form, reverse treatment and third-body variant (C17)."""
    for m in tiny_mechs:
        o, pj = Oracle(m), PyJac(m)
        T, P, Y = synth.make_states(m.n_species, 257, 5, t_range=(500.0, 2800.0), p_range_atm=(0.05, 80.0))
        check_rates(torch, pj, o, T, P, Y, label="tiny")
        check_jacobian(torch, pj, o, T, P, Y, label="tiny")


def test_tiny_mechanism_last_species_inert(torch, PyJac):
    m = synth.make_tiny_mechanism(3, n_species=8, last_reacts=False)
    o, pj = Oracle(m), PyJac(m)
    T, P, Y = synth.make_states(m.n_species, 64, 6)
    check_rates(torch, pj, o, T, P, Y)
    check_jacobian(torch, pj, o, T, P, Y)


def test_config0_all_states(torch, PyJac):
    m = synth.make_mechanism(0)
    o, pj = Oracle(m), PyJac(m)
    T, P, Y = synth.config_states(0)
    assert len(T) == 1024
    check_rates(torch, pj, o, T, P, Y, label="cfg0_all")
    check_jacobian(torch, pj, o, T, P, Y, label="cfg0_all")


@pytest.mark.parametrize("cfg,n", [(1, 1500), (2, 300), (3, 24)])
def test_config_prefix(torch, PyJac, cfg, n):
    """Sizes the oracle finishes in seconds, spanning several CTAs' worth of states and a ragged tail."""
    m = synth.make_mechanism(cfg)
    o, pj = Oracle(m), PyJac(m)
    T, P, Y = synth.config_states(cfg, n)
    check_rates(torch, pj, o, T, P, Y, label="cfg%d_prefix" % cfg)
    check_jacobian(torch, pj, o, T, P, Y, label="cfg%d_prefix" % cfg)


# ---------------------------------------------------------------------------------- full sizes
def named_states(n, S, grid):
    """States of a launch of n states worth looking at by name (the kernel is a persistent grid-stride loop over
    batches of S consecutive states, CTA c taking batches c, c + grid, ..; it rotates two mixture blocks and
    prefetches the next batch while the current one runs): every state of the first three and last three batches
    of the first and of the last CTA -- both parities of the rotating blocks, the prologue without a predecessor
    and the epilogue without a successor -- and the ragged last batch of the launch."""
    nb = (n + S - 1) // S
    batches = {nb - 1}
    for cta in {0, min(grid, nb) - 1}:
        it = list(range(cta, nb, grid))
        batches.update(it[:3] + it[-3:])
    return np.array(sorted({s for b in batches for s in range(b * S, min(n, (b + 1) * S))}))


@pytest.mark.parametrize("cfg,chunk,n_sample", [(1, 100_000, 8192), (2, 100_000, 2048), (3, 8192, 64)])
def test_config_full_size_sampled(torch, PyJac, cfg, chunk, n_sample):
    """BASELINE.json's full state counts in the launch configuration bench.py times (one launch per
    chunk); sampled states against the oracle -- the named ones of `named_states` plus uniform draws up to
    n_sample per launch (8,192 / 2,048 / 4 x 64 states: about a second of oracle time each on the box's cores) --
    and invariants on every state."""
    m = synth.make_mechanism(cfg)
    o, pj = Oracle(m), PyJac(m)
    T, P, Y = synth.config_states(cfg)
    n, ns, ld = len(T), m.n_species, m.n_species + 1
    rng = np.random.default_rng(100 + cfg)
    mw = torch.from_numpy(m.mol_wt).cuda()
    buf = torch.empty((min(chunk, n), ld * ld), dtype=torch.float64, device="cuda")
    for s0 in range(0, n, chunk):
        s1 = min(n, s0 + chunk)
        dT, dP, dY = dev(torch, T[s0:s1], P[s0:s1], Y[s0:s1])
        J = pj.eval_jacobian(dT, dP, dY, out=buf)[: s1 - s0].view(-1, ld, ld)   # [n][col][row]
        assert bool(torch.isfinite(J).all())
        assert bool((J[:, ld - 1, :] == 0).all())
        # P12: species rows (incl. placeholder) of every column sum to zero; checked on all states
        sp = J[:, :, 1:]
        resid = sp.sum(dim=2).abs().amax(dim=1)
        scale = sp.abs().amax(dim=1).sum(dim=1)
        assert bool((resid <= 1e-12 * scale).all())
        lc = pj.launch_config(s1 - s0)
        named = named_states(s1 - s0, lc["states_per_cta"], lc["grid"])
        assert len(named) <= 13 * lc["states_per_cta"] and named[-1] == s1 - s0 - 1 and named[0] == 0
        drawn = rng.choice(s1 - s0, size=min(n_sample, s1 - s0), replace=False)
        pick = np.unique(np.concatenate([named, drawn]))[: max(n_sample, len(named))]
        pick = np.unique(np.concatenate([named, pick]))
        Jr = o.jacobian(T[s0:s1][pick], P[s0:s1][pick], Y[s0:s1][pick])
        Jg = J.reshape(-1, ld * ld)[torch.from_numpy(pick).cuda()].cpu().numpy()
        assert_jacobian(Jg, Jr, ns, label="cfg%d_full_sampled" % cfg)
    del buf


def test_state_count_sweep_rates_and_dydt(torch, PyJac):
    """Config 4: the 53-species mechanism at 4^5 .. 4^8 states (larger counts are bench-only);
    the three kernels agree with the oracle on sampled states at each count."""
    m = synth.make_mechanism(1)
    o, pj = Oracle(m), PyJac(m)
    for n in (4 ** 5, 4 ** 6, 4 ** 7, 4 ** 8):
        T, P, Y = synth.make_states(m.n_species, n, synth.CONFIGS[1].seed + 2000 + n)
        dT, dP, dY = dev(torch, T, P, Y)
        dy = pj.eval_dydt(dT, dP, dY).cpu().numpy()
        J = pj.eval_jacobian(dT, dP, dY)
        pick = np.sort(np.random.default_rng(n).choice(n, size=48, replace=False))
        ref = o.source(T[pick], P[pick], Y[pick])
        scale = np.abs(ref["dydt"][:, 1:]).max(axis=1, keepdims=True)
        tol = RATE_TOL
        bound = tol * np.maximum(scale, _dydt_term_scale(o, ref, T[pick], P[pick], Y[pick], slice(1, None)))
        assert np.all(np.abs(dy[pick][:, 1:] - ref["dydt"][:, 1:]) <= bound)
        Jr = o.jacobian(T[pick], P[pick], Y[pick])
        Jg = J[torch.from_numpy(pick).cuda()].cpu().numpy()
        assert_jacobian(Jg, Jr, m.n_species, label="cfg4_sweep")


# ---------------------------------------------------------------------------------- edge cases
def test_empty_and_single_state(torch, PyJac, tiny_mechs):
    m = tiny_mechs[0]
    o, pj = Oracle(m), PyJac(m)
    T, P, Y = synth.make_states(m.n_species, 1, 8)
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    eY = torch.empty((0, m.n_species), dtype=torch.float64, device="cuda")
    assert pj.eval_jacobian(e, e, eY).shape == (0, (m.n_species + 1) ** 2)
    assert pj.eval_dydt(e, e, eY).shape == (0, m.n_species + 1)
    check_jacobian(torch, pj, o, T, P, Y)


@pytest.mark.parametrize("cfg,n", [(0, 777), (1, 1999), (2, 1000), (3, 130)])
def test_padded_leading_dimension_and_batch_split_bit_identical(torch, PyJac, cfg, n):
    """ldy > Nsp; results do not depend on n, batch split, stream or repetition (header contract; App. D).  A
    batch split changes which CTA evaluates which state and with which neighbours in its batch, and so the
    timing of every phase: a race between the phases would show as a difference (compute-sanitizer's racecheck
    is closed on the pool, profiles/r2_checked_build.md).  All four mechanisms: one and several resident CTAs,
    S = 1 and 3, one and two rows per lane."""
    m = synth.make_mechanism(cfg)
    pj = PyJac(m)
    T, P, Y = synth.config_states(cfg, n)
    dT, dP, dY = dev(torch, T, P, Y)
    J = pj.eval_jacobian(dT, dP, dY)
    for _ in range(3):
        assert torch.equal(pj.eval_jacobian(dT, dP, dY), J)
    Ypad = torch.full((n, m.n_species + 5), 7.0, dtype=torch.float64, device="cuda")
    Ypad[:, : m.n_species] = dY
    assert torch.equal(pj.eval_jacobian(dT, dP, Ypad), J)
    cuts = (0, 1, n // 3 + 1, n)
    parts = [pj.eval_jacobian(dT[a:b].contiguous(), dP[a:b].contiguous(), dY[a:b].contiguous())
             for a, b in zip(cuts[:-1], cuts[1:])]
    assert torch.equal(torch.cat(parts), J)
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        J2 = pj.eval_jacobian(dT, dP, dY)
    s.synchronize()
    assert torch.equal(J2, J)
    r1 = pj.eval_rates(dT, dP, dY)
    r2 = pj.eval_rates(dT[:100].contiguous(), dP[:100].contiguous(), dY[:100].contiguous())
    for k in r1:
        assert torch.equal(r1[k][:100], r2[k])


def test_zero_mass_fractions(torch, PyJac, tiny_mechs):
    """Y_k = 0 exactly for several species (no division by a concentration)."""
    m = tiny_mechs[1]
    o, pj = Oracle(m), PyJac(m)
    T, P, Y = synth.make_states(m.n_species, 40, 12)
    rng = np.random.default_rng(4)
    for s in range(len(T)):
        z = rng.choice(m.n_species - 1, size=3, replace=False)
        Y[s, z] = 0.0
        Y[s] /= Y[s].sum()
    # falloff reactions need a non-zero third-body concentration (header precondition): keep the
    # single-species third bodies present
    for i in range(m.n_reactions):
        if m.tb_species[i] >= 0:
            Y[:, m.tb_species[i]] = np.maximum(Y[:, m.tb_species[i]], 1e-6)
    Y /= Y.sum(axis=1, keepdims=True)
    check_rates(torch, pj, o, T, P, Y)
    check_jacobian(torch, pj, o, T, P, Y)


def test_branch_points(torch, PyJac, tiny_mechs):
    """T exactly at a NASA midpoint, P exactly at and outside PLOG table pressures (C4, C6)."""
    m = tiny_mechs[0]
    o, pj = Oracle(m), PyJac(m)
    T, P, Y = synth.make_states(m.n_species, 12, 13)
    T[:3] = [900.0, 1000.0, 1300.0]
    P[3:8] = np.array([0.1, 1.0, 10.0, 100.0, 1e-3]) * 101325.0
    P[8] = 500.0 * 101325.0
    check_rates(torch, pj, o, T, P, Y)
    check_jacobian(torch, pj, o, T, P, Y)


def test_degenerate_mechanisms(torch, PyJac):
    """No reactions at all; a single species; a reaction whose net stoichiometry cancels."""
    sp = synth._make_species(np.random.default_rng(1), ("H", "O"), 2, 4, n2_last=False)
    names, comp, w, lo, hi, tm = sp
    b = MechanismBuilder(names, ("H", "O"), comp, w, lo, hi, tm)
    m0 = b.build()
    o, pj = Oracle(m0), PyJac(m0)
    T, P, Y = synth.make_states(4, 9, 1)
    J, _ = check_jacobian(torch, pj, o, T, P, Y, tol=0.0)
    assert np.all(J == 0.0)
    b1 = MechanismBuilder(names[:1], ("H", "O"), comp[:1], w[:1], lo[:1], hi[:1], tm[:1])
    m1 = b1.build()
    o, pj = Oracle(m1), PyJac(m1)
    T, P, Y = synth.make_states(1, 3, 1)
    check_jacobian(torch, pj, o, T, P, Y, tol=0.0)


def test_host_buffer_variant_matches_device_variant(torch, PyJac):
    m = synth.make_mechanism(0)
    pj = PyJac(m)
    T, P, Y = synth.config_states(0, 1000)
    dT, dP, dY = dev(torch, T, P, Y)
    J = pj.eval_jacobian(dT, dP, dY).cpu()
    ld = m.n_species + 1
    out = torch.empty((1000, ld * ld), dtype=torch.float64).pin_memory()
    hT, hP, hY = (torch.from_numpy(a).pin_memory() for a in (T, P, Y))
    pj.eval_jacobian_host(hT, hP, hY, out, chunk_states=333)      # ragged chunks, both buffers reused
    assert torch.equal(out, J)
    out2 = np.empty((1000, ld * ld))
    pj.eval_jacobian_host(T, P, Y, out2)                           # pageable numpy buffers
    assert np.array_equal(out2, J.numpy())
    dy = np.empty((1000, ld))
    pj.eval_dydt_host(T, P, Y, dy, chunk_states=512)
    assert np.array_equal(dy, pj.eval_dydt(dT, dP, dY).cpu().numpy())
    before = pj.kernel_launches()
    pj.eval_jacobian(dT, dP, dY)
    assert pj.kernel_launches() == before + 1


def test_host_variant_keeps_a_bounded_footprint_and_trim_returns_it(torch, PyJac):
    """the staging buffers a *_host call leaves with the handle are capped by bytes (one output buffer
    of at most 512 MiB, ~1.1 GiB in all), an explicit larger chunk goes through temporary buffers, and
    pyjac_mech_trim gives the kept ones back.  111 species: 100,352 B per state, 5,349 states per default chunk."""
    m = synth.make_mechanism(2)
    pj = PyJac(m)
    ld = m.n_species + 1
    n = 6000
    T, P, Y = synth.config_states(2, n)
    dT, dP, dY = dev(torch, T, P, Y)
    J = pj.eval_jacobian(dT, dP, dY).cpu().numpy()
    torch.cuda.synchronize()
    out = np.empty((n, ld * ld))
    free0 = torch.cuda.mem_get_info()[0]
    pj.eval_jacobian_host(T, P, Y, out)                            # default chunk: two chunks, buffers kept
    assert np.array_equal(out, J)
    kept = free0 - torch.cuda.mem_get_info()[0]
    assert (512 << 20) <= kept <= int(1.2 * (1 << 30)), kept
    pj.trim()
    assert free0 - torch.cuda.mem_get_info()[0] < (64 << 20)       # the streams' few KB may stay
    out[:] = 0.0
    pj.eval_jacobian_host(T, P, Y, out, chunk_states=n)            # 602 MB per output buffer: above the cap, not kept
    assert np.array_equal(out, J)
    assert free0 - torch.cuda.mem_get_info()[0] < (64 << 20)
    pj.trim()                                                      # nothing to free: still fine


def test_tile_store_probe_writes_every_element(torch, PyJac):
    """Helper library, not the product: the tile-store probe behind profiles/r3_tile_store_probe.md (per-state tiles
    filled in shared memory, then one cp.async.bulk per tile, or a read-back and streaming stores) must write tile t,
    element i = t + i for every tile, including counts that are no multiple of the grid and both tile sizes."""
    from paper_1605_03262_b200 import binding
    sp = torch.cuda.current_stream().cuda_stream
    for td, nt in ((54 * 54, 1000), (112 * 112, 301), (14 * 14, 5)):
        want = (torch.arange(nt, dtype=torch.float64, device="cuda")[:, None]
                + torch.arange(td, dtype=torch.float64, device="cuda")[None, :])
        for mode in (0, 1):
            for ctas in (1, 2):
                buf = torch.full((nt + 1, td), -1.0, dtype=torch.float64, device="cuda")
                binding.peak_tile_store(buf, nt, td, mode, ctas, sp)
                torch.cuda.synchronize()
                assert torch.equal(buf[:nt], want) and bool((buf[nt] == -1.0).all())
    with pytest.raises(binding.PyJacError):
        binding.peak_tile_store(torch.empty(2 * 127 * 127 + 1, dtype=torch.float64, device="cuda")[1:], 2, 127 * 127 - 1, 0, 1, sp)


def test_gather_probe_sums_the_real_cell_lists(torch, PyJac):
    """Helper library, not the product: the gather timing prototype behind profiles/r3_gather_probe.md must really sum
    the mechanism's cell lists (its timing means nothing otherwise): every state's tile equals the tile the host
    computes from the same lists and stand-in values, for every S, both buffer counts and a ragged last batch."""
    from paper_1605_03262_b200 import binding
    sp = torch.cuda.current_stream().cuda_stream
    for cfg, n in ((0, 1000), (1, 500)):
        m = synth.make_mechanism(cfg)
        ld = m.n_species + 1
        st0 = binding.pack_stats(m)
        for S, threads, ctas, nbuf in ((1, 128, 2, 2), (2, 256, 1, 2), (3, 512, 1, 1), (3, 96, 1, 2)):
            out = torch.full((n + 1, ld * ld), -1.0, dtype=torch.float64, device="cuda")
            r = binding.gather_probe(m, out, n, S, threads, ctas, nbuf, 1, sp)
            torch.cuda.synchronize()
            exp = torch.from_numpy(r["expected"]).cuda()
            assert bool(((out[:n] - exp[None, :]).abs() <= 1e-13 * exp.abs().max()).all())
            assert bool((out[n] == -1.0).all())
            assert r["cells"] == ld * ld and r["nonempty_cells"] == st0["cells"] and r["entries"] <= r["entries_padded"]
            assert r["entries_padded"] <= 1.25 * r["entries"] + 32 * 16          # sorted by length: little padding


# ---------------------------------------------------------------------------------- launch shapes
@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n,shape", [
    (1, 301, dict(states_per_cta=1, ctas_per_sm=4)),                                # one state per CTA iteration
    (1, 301, dict(states_per_cta=2, ctas_per_sm=3, threads=160)),                   # three small CTAs per SM
    (1, 301, dict(states_per_cta=3, ctas_per_sm=1, threads=512)),                   # odd S: 8-byte shared loads
    (1, 301, dict(states_per_cta=4, threads=256)),
    (1, 301, dict(states_per_cta=6, threads=384)),
    (1, 301, dict(cell_cap=1, list_cap=4)),                    # everything summed in the summing phase, short lane lists
    (1, 301, dict(states_per_cta=2, cell_cap=2, list_cap=30)),
    (1, 301, dict(rows_per_lane=1)),                                                # one row per lane, 8-byte stores
    (1, 301, dict(p1_states=1)),                                      # one state per reaction work item
    (1, 301, dict(p1_states=3)),                                      # all states in one item, every rate form
    (1, 301, dict(p1_states=2 + 16 * 2)),                             # two per item, plain and general groups
    (1, 301, dict(layout=2)),                                         # per-reaction terms in allocation order
    (2, 65, dict(layout=2, p1_states=3)),
    (3, 9, dict(layout=2)),
    (3, 211, dict(threads=512)),                                      # 360 species, one state per CTA: read-ahead paths over
                                                                      # two grid-stride iterations and a ragged last one
    (1, 301, dict(states_per_cta=6, threads=512, ctas_per_sm=1, p1_states=2)),   # pairs of states, constants in registers
    (1, 301, dict(states_per_cta=2, threads=512, ctas_per_sm=1, stage_tables=1)),  # gather tables staged in shared memory
    (0, 1024, dict(stage_tables=1)),
    (0, 1024, dict(states_per_cta=1, threads=64)),
    (2, 65, dict(states_per_cta=2)),
])
def test_launch_shapes(torch, PyJac, cfg, n, shape):
    """Every launch shape pyjac_mech_create_shaped accepts (states per CTA iteration, CTAs per SM, CTA
    size, list lengths of the two gather phases, rows per lane) evaluates the same Jacobian: parity with
    the oracle within the same tolerance, ragged last batch included."""
    m = synth.make_mechanism(cfg)
    T, P, Y = synth.config_states(cfg, n)
    pj = PyJac(m, shape=shape)
    o = Oracle(m)
    check_jacobian(torch, pj, o, T, P, Y, label="launch_shapes")
    check_rates(torch, pj, o, T[:64], P[:64], Y[:64])


# ---------------------------------------------------------------------------------- near-equilibrium states (f4)
@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_equilibrium_and_trajectory_states(torch, PyJac, cfg):
    """States the paper singles out: at chemical equilibrium of every K_c-reversible
    reaction (element potentials, tests/trajectory.py: R_f = R_r to rounding, so q_i is a cancelled
    difference), a step of 1e-8 and of 1e-3 off it, and -- for the two smaller mechanisms -- along a
    linearly implicit Euler march of the source term from a seeded state.  Same tolerances as everywhere:
    R_f, R_r, c_i element-wise, the production rates against the size of what was summed (C19), the
    Jacobian per state, row, element and column."""
    from trajectory import equilibrium_states, march_to_equilibrium
    m = synth.make_mechanism(cfg)
    o, pj = Oracle(m), PyJac(m)
    temps = np.linspace(850.0, 2400.0, 12)
    parts = [equilibrium_states(m, temps, p_target_atm=p, perturb=d, seed=7)
             for p, d in ((1.0, 0.0), (20.0, 0.0), (5.0, 1e-8), (5.0, 1e-3))]
    if cfg <= 1:
        T0, P0, Y0 = synth.config_states(cfg, 2)
        for k in range(2):
            Tt, Pt, Yt, _ = march_to_equilibrium(m, T0[k], P0[k], Y0[k], n_steps=60, growth=2.0)
            parts.append((Tt, Pt, Yt))
    T = np.concatenate([p[0] for p in parts]); P = np.concatenate([p[1] for p in parts])
    Y = np.concatenate([p[2] for p in parts])
    ref = o.source(T[:24], P[:24], Y[:24])
    rel = np.abs(ref["rf"] - ref["rr"]) / np.maximum(ref["rf"] + ref["rr"], 1e-300)
    assert np.median(rel) < 1e-10 or cfg == 0          # the first 24 states really are at equilibrium
    check_rates(torch, pj, o, T, P, Y, label="cfg%d_equilibrium" % cfg)
    check_jacobian(torch, pj, o, T, P, Y, label="cfg%d_equilibrium" % cfg)


# ---------------------------------------------------------------------------------- Jacobian-vector product (f1)

@pytest.mark.parametrize("cfg,n", [(0, 1024), (1, 700), (2, 200), (3, 20)])
def test_jvp_matches_oracle_jacobian_times_vector(torch, PyJac, cfg, n):
    """pyjac_eval_jvp (the Jacobian consumed on chip) against the plain
    definition: the oracle's analytical Jacobian (Eqs. 44-113) times the vector, in numpy.  An element J_rc is
    a rounded sum of terms of the size of its row's largest entry (the alpha_r d_c part of Eq. 112 is in every
    column: see `jacobian_errors`), and the product sums those terms per reaction before it sums over the
    columns, so entry r of J v is judged at max_c |J_rc| * sum_c |v_c|: tolerance JAC_TOL of it, observed
    maxima recorded.  Vectors: seeded normal entries scaled to the state (T-sized first entry, mass-fraction
    sized others), a unit vector per state (one column of J), and padded ldv."""
    m = synth.make_mechanism(cfg)
    o, pj = Oracle(m), PyJac(m)
    ns, ld = m.n_species, m.n_species + 1
    T, P, Y = synth.config_states(cfg, n)
    rng = np.random.default_rng(77 + cfg)
    v = np.zeros((n, ld + 3))
    v[:, 0] = T * 1e-3 * rng.standard_normal(n)
    v[:, 1:ld] = Y * rng.standard_normal((n, ns))
    v[:, ld:] = 1e300                                   # padding of ldv: never read
    unit = np.zeros((n, ld)); unit[np.arange(n), rng.integers(0, ns, n)] = 1.0
    Jr = o.jacobian(T, P, Y).reshape(n, ld, ld).transpose(0, 2, 1)        # [n][row][col]
    dT, dP, dY = dev(torch, T, P, Y)
    worst = 0.0
    for vec in (v, unit):
        dv = torch.from_numpy(vec).cuda()
        got = pj.eval_jvp(dT, dP, dY, dv).cpu().numpy()
        ref = np.einsum("nrc,nc->nr", Jr, vec[:, :ld])
        scale = np.abs(Jr).max(axis=2) * np.abs(vec[:, :ns]).sum(axis=1, keepdims=True)
        err = np.abs(got - ref)
        worst = max(worst, float((err / np.maximum(scale, 1e-300))[scale > 0].max(initial=0.0)))
        assert np.all(err <= JAC_TOL * scale + 1e-300), worst
        assert np.all(got[scale == 0.0] == 0.0)
    JVP_OBSERVED["cfg%d" % cfg] = worst


def test_jvp_tiny_mechanisms_and_arguments(torch, PyJac, tiny_mechs):
    """Every reaction type (one-state general path included), a single state, n = 0, and the argument checks."""
    from paper_1605_03262_b200.binding import PyJacError
    for m in tiny_mechs:
        o, pj = Oracle(m), PyJac(m)
        ns, ld = m.n_species, m.n_species + 1
        T, P, Y = synth.make_states(ns, 130, 9, t_range=(500.0, 2800.0), p_range_atm=(0.05, 80.0))
        rng = np.random.default_rng(3)
        v = np.concatenate([(T * rng.standard_normal(len(T)))[:, None], rng.standard_normal((len(T), ns))], axis=1)
        Jr = o.jacobian(T, P, Y).reshape(len(T), ld, ld).transpose(0, 2, 1)
        dT, dP, dY = dev(torch, T, P, Y)
        got = pj.eval_jvp(dT, dP, dY, torch.from_numpy(v).cuda()).cpu().numpy()
        ref = np.einsum("nrc,nc->nr", Jr, v)
        scale = np.abs(Jr).max(axis=2) * np.abs(v[:, :ns]).sum(axis=1, keepdims=True)
        assert np.all(np.abs(got - ref) <= JAC_TOL * scale + 1e-300)
        one = pj.eval_jvp(dT[:1], dP[:1], dY[:1], torch.from_numpy(v[:1]).cuda()).cpu().numpy()
        assert np.array_equal(one[0], got[0])
        assert pj.eval_jvp(dT[:0], dP[:0], dY[:0], torch.from_numpy(v[:0]).cuda()).shape == (0, ld)
        with pytest.raises(ValueError):
            pj.eval_jvp(dT, dP, dY, torch.from_numpy(v[:, :ns]).cuda())       # vector too short
    assert isinstance(PyJacError(-1, "x"), Exception)


# ---------------------------------------------------------------------------------- forward differences (f2)

@pytest.mark.parametrize("cfg,n,chunk", [(0, 1024, 100), (1, 300, 64), (2, 40, 7), (3, 6, 4)])
def test_fd_jacobian_matches_oracle_fd(torch, PyJac, cfg, n, chunk):
    """pyjac_eval_jacobian_fd (the paper's comparison method; C21) against the
    oracle's forward difference with the same increments.  Both subtract two source terms and divide by
    D_j = sqrt(eps) max(|Phi_j|, rtol |Phi_j| + atol), so a disagreement of the source terms of t times
    the size of the terms they sum (RATE_TOL, asserted in check_rates) becomes 2 t (term size) / D_j in
    column j: that is the element-wise tolerance.  Column N_s is exactly zero; chunks smaller than the
    batch (ragged last chunk) give bit-identical results to one chunk."""
    m = synth.make_mechanism(cfg)
    o, pj = Oracle(m), PyJac(m)
    ns, ld = m.n_species, m.n_species + 1
    T, P, Y = synth.config_states(cfg, n)
    rtol, atol = 1e-8, 1e-12
    dT, dP, dY = dev(torch, T, P, Y)
    J = pj.eval_jacobian_fd(dT, dP, dY, rtol=rtol, atol=atol, chunk_states=chunk).cpu().numpy()
    J1 = pj.eval_jacobian_fd(dT, dP, dY, rtol=rtol, atol=atol, chunk_states=n).cpu().numpy()
    assert np.array_equal(J, J1)
    Jr = o.jacobian_fd(T, P, Y, rtol=rtol, atol=atol)
    A = J.reshape(n, ld, ld).transpose(0, 2, 1)
    B = Jr.reshape(n, ld, ld).transpose(0, 2, 1)
    assert np.all(A[:, :, ns] == 0.0)
    ref = o.source(T, P, Y)
    phi = np.concatenate([T[:, None], Y[:, :ns - 1]], axis=1)
    inc = np.sqrt(EPS) * np.maximum(np.abs(phi), rtol * np.abs(phi) + atol)              # [n][ns]
    term = np.empty((n, ld))
    term[:, :1] = np.maximum(np.abs(ref["dydt"][:, :1]), _dydt_term_scale(o, ref, T, P, Y, slice(0, 1)))
    term[:, 1:] = np.maximum(np.abs(ref["dydt"][:, 1:]).max(axis=1, keepdims=True),
                             _dydt_term_scale(o, ref, T, P, Y, slice(1, None)))
    bound = 2.0 * RATE_TOL * term[:, :, None] / inc[:, None, :]                          # [n][row][col]
    err = np.abs(A[:, :, :ns] - B[:, :, :ns])
    FD_OBSERVED["cfg%d" % cfg] = float((err / bound).max())
    assert np.all(err <= bound), float((err / bound).max())


def test_fd_jacobian_argument_errors(torch, PyJac):
    m = synth.make_mechanism(0)
    pj = PyJac(m)
    T, P, Y = synth.config_states(0, 8)
    dT, dP, dY = dev(torch, T, P, Y)
    from paper_1605_03262_b200.binding import PyJacError
    with pytest.raises(PyJacError):       # scratch for less than one state
        pj.eval_jacobian_fd(dT, dP, dY, work=torch.empty(8, dtype=torch.float64, device="cuda"))
    with pytest.raises(PyJacError):
        pj.eval_jacobian_fd(dT, dP, dY, rtol=0.0)
    with pytest.raises(PyJacError):       # atol = 0 would give an absent species the increment 0 and a column of 0/0
        pj.eval_jacobian_fd(dT, dP, dY, atol=0.0)
    Y0 = Y.copy()
    Y0[:, -1] += Y0[:, 2]
    Y0[:, 2] = 0.0                        # an unknown that is exactly zero: finite with the smallest positive atol in use
    J0 = pj.eval_jacobian_fd(dT, dP, torch.from_numpy(Y0).cuda(), atol=1e-15).cpu().numpy()
    Jr0 = Oracle(m).jacobian_fd(T, P, Y0, atol=1e-15)
    assert np.all(np.isfinite(J0)) and np.all(np.isfinite(Jr0))
    # (the zero unknown's column is a quotient of rounding noise by 1.5e-23 on both sides: only finiteness is
    # asserted there; the temperature column has a sane increment and must agree)
    ld = m.n_species + 1
    assert np.allclose(J0[:, :ld], Jr0[:, :ld], rtol=1e-6, atol=1e-6 * np.abs(Jr0[:, :ld]).max())
    assert pj.fd_workspace_doubles(0) == -1
    l0 = pj.kernel_launches()
    pj.eval_jacobian_fd(dT, dP, dY, chunk_states=4)
    assert pj.kernel_launches() - l0 == 8             # two chunks of four launches


@pytest.mark.gpu
def test_two_live_handles_share_a_kernel(torch, PyJac):
    """A handle is immutable after creation: creating a second, smaller mechanism that uses the same kernel
    function must not disturb the first one's launches (the kernel's dynamic shared-memory limit is set to
    what the device allows, never to one handle's size)."""
    big, small = synth.make_mechanism(1), synth.make_mechanism(0)
    shape = dict(states_per_cta=2, ctas_per_sm=1, threads=256)
    T, P, Y = synth.config_states(1, 130)
    dT, dP, dY = dev(torch, T, P, Y)
    pj_big = PyJac(big, shape=shape)
    J0 = pj_big.eval_jacobian(dT, dP, dY).clone()
    pj_small = PyJac(small, shape=shape)                      # same kernel function, 8 KB instead of 67 KB
    Ts, Ps, Ys = synth.config_states(0, 64)
    check_jacobian(torch, pj_small, Oracle(small), Ts, Ps, Ys)
    assert torch.equal(pj_big.eval_jacobian(dT, dP, dY), J0)
    check_jacobian(torch, pj_big, Oracle(big), T, P, Y)


@pytest.mark.gpu
def test_later_handle_does_not_take_shared_memory_from_an_earlier_one(torch, PyJac):
    """the preferred shared-memory carve-out is an attribute of the kernel FUNCTION, which every handle
    of the same S shares.  The 53-species handle needs ~90 % of the SM's memory as shared memory for its two resident
    CTAs; the 13-species handle created after it would ask for a few per cent.  The library keeps the largest value
    ever asked for, so the first handle still runs with the CTAs per SM its grid was sized for: same launch time
    (a drop from two resident CTAs to one costs far more than the 15 % allowed here) and the same bits."""
    big, small = synth.make_mechanism(1), synth.make_mechanism(0)
    T, P, Y = synth.config_states(1, 30_000)
    dT, dP, dY = dev(torch, T, P, Y)
    pj_big = PyJac(big)
    out = torch.empty((len(T), (big.n_species + 1) ** 2), dtype=torch.float64, device="cuda")

    def launch_ms():
        for _ in range(3):
            pj_big.eval_jacobian(dT, dP, dY, out=out)
        torch.cuda.synchronize()
        times = []
        for _ in range(7):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            pj_big.eval_jacobian(dT, dP, dY, out=out)
            b.record()
            torch.cuda.synchronize()
            times.append(a.elapsed_time(b))
        return sorted(times)[3]

    before = launch_ms()
    J0 = out.clone()
    cfg_before = pj_big.launch_config(len(T))
    pj_small = PyJac(small)
    assert pj_small.launch_config(64)["states_per_cta"] == cfg_before["states_per_cta"]      # the same kernel function
    Ts, Ps, Ys = synth.config_states(0, 256)
    pj_small.eval_jacobian(*dev(torch, Ts, Ps, Ys))
    after = launch_ms()
    assert torch.equal(out, J0)
    assert after <= 1.15 * before, (before, after)


@pytest.mark.gpu
def test_one_handle_from_two_host_threads(torch, PyJac):
    """Evaluation on a handle is re-entrant (the paper's complaint about TChem): two host
    threads evaluate on the same handle at once, each on its own stream, device-pointer and host-buffer
    calls mixed; every result is bit-identical to the serial one."""
    import threading
    m = synth.make_mechanism(0)
    pj = PyJac(m)
    ld = m.n_species + 1
    T, P, Y = synth.config_states(0, 1024)
    dT, dP, dY = dev(torch, T, P, Y)
    ref = pj.eval_jacobian(dT, dP, dY).cpu()
    torch.cuda.synchronize()
    errors = []

    def work(k):
        try:
            torch.cuda.set_device(0)
            s = torch.cuda.Stream()
            for it in range(6):
                with torch.cuda.stream(s):
                    J = pj.eval_jacobian(dT, dP, dY)
                s.synchronize()
                assert torch.equal(J.cpu(), ref)
                out = np.empty((1024, ld * ld))
                pj.eval_jacobian_host(T, P, Y, out, chunk_states=300 + 37 * k)
                assert np.array_equal(out, ref.numpy())
        except Exception as e:                                  # noqa: BLE001
            errors.append(repr(e))

    threads = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


@pytest.mark.gpu
def test_binding_rejects_bad_output_tensors(torch, PyJac):
    m = synth.make_mechanism(0)
    pj = PyJac(m)
    ld = m.n_species + 1
    T, P, Y = synth.config_states(0, 8)
    dT, dP, dY = dev(torch, T, P, Y)
    for bad in (torch.empty((8, ld * ld), dtype=torch.float32, device="cuda"),
                torch.empty((8, ld * ld - 1), dtype=torch.float64, device="cuda"),
                torch.empty((8, 2 * ld * ld), dtype=torch.float64, device="cuda")[:, ::2],
                torch.empty((8, ld * ld), dtype=torch.float64)):
        with pytest.raises(ValueError):
            pj.eval_jacobian(dT, dP, dY, out=bad)
    with pytest.raises(ValueError):
        pj.eval_dydt(dT, dP, dY, out=torch.empty((8, ld - 1), dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):
        pj.eval_jacobian_host(T, P, Y, np.empty((8, ld * ld), dtype=np.float32))


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n", [(0, 257), (1, 301), (2, 100)])
def test_output_pointer_not_16_byte_aligned(torch, PyJac, cfg, n):
    """An output pointer that is only 8-byte aligned takes the 8-byte store path; same numbers (one and two
    slabs of rows, one and two resident CTAs)."""
    m = synth.make_mechanism(cfg)
    pj = PyJac(m)
    T, P, Y = synth.config_states(cfg, n)
    dT, dP, dY = dev(torch, T, P, Y)
    J = pj.eval_jacobian(dT, dP, dY)
    ld = m.n_species + 1
    buf = torch.zeros(n * ld * ld + 1, dtype=torch.float64, device="cuda")
    view = buf[1:]
    assert view.data_ptr() % 16 == 8
    pj.eval_jacobian(dT, dP, dY, out=view)
    assert torch.equal(view.reshape(n, ld * ld), J)
    assert float(buf[0]) == 0.0


@pytest.mark.gpu
def test_peak_probes(torch):
    """The roofline probes of the helper library: the store stream writes every element
    once, the FMA probe reports the flops it ran; bad arguments are refused."""
    from paper_1605_03262_b200 import binding
    sp = torch.cuda.current_stream().cuda_stream
    buf = torch.full((1 << 16,), -1.0, dtype=torch.float64, device="cuda")
    binding.peak_store_stream(buf, sp)
    torch.cuda.synchronize()
    assert torch.equal(buf[0::2], torch.arange(1 << 15, dtype=torch.float64, device="cuda"))
    assert bool((buf[1::2] == 1.0).all())
    out = torch.zeros(148 * 4096, dtype=torch.float64, device="cuda")
    flops = binding.peak_dfma(out, 128, sp)
    torch.cuda.synchronize()
    assert flops > 0 and flops % (2 * 8 * 128) == 0 and bool(torch.isfinite(out).all())
    lib = binding.load_tools()
    assert lib.pyjac_tools_peak_store_stream(None, 16, None) == binding.PYJAC_EINVAL
    assert lib.pyjac_tools_peak_store_stream(buf.data_ptr() + 8, 16, None) == binding.PYJAC_EINVAL
