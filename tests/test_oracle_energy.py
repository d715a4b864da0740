"""Pins of the oracle's NEXT-1 part (temperature right-hand side and the energy row of the (N+1) x (N+1) Jacobian, PAPER.md
Eq. 7) and of its zero-QSS Jacobian mode (L232) against things other than the oracle: a closed form on a
three-species toy with heat release (mpmath), conservation of the internal energy along an explicit Euler step with the
thermodynamics restated in mpmath, mechanical derivatives of the right-hand side (dual numbers, complex step), the float128
referee, and for the simplified Jacobians the cases in which they must coincide with the exact one.  No GPU involved."""
import mpmath as mp
import numpy as np
import pytest

import oracle
from qss_synth import config_mechanism, config_states, make_states, toy_dag, toy_nonqss
from qss_synth.mechanism import assemble, T_LOW, T_MID, T_HIGH

mp.mp.dps = 40
R = mp.mpf("8.31446261815324")
P0 = mp.mpf(101325)


def _nasa(a, T):
    """h/RT, s/R, cp/R of one NASA-7 set, written out in mpmath (independent of the oracle)."""
    T = mp.mpf(T); a = [mp.mpf(float(x)) for x in a]
    h = a[0] + a[1] * T / 2 + a[2] * T ** 2 / 3 + a[3] * T ** 3 / 4 + a[4] * T ** 4 / 5 + a[5] / T
    s = a[0] * mp.log(T) + a[1] * T + a[2] * T ** 2 / 2 + a[3] * T ** 3 / 3 + a[4] * T ** 4 / 4 + a[6]
    cp = a[0] + a[1] * T + a[2] * T ** 2 + a[3] * T ** 3 + a[4] * T ** 4
    return h, s, cp


def _set(m, s, T):
    return m.nasa_lo[s] if T < m.nasa_T[s, 1] else m.nasa_hi[s]


def _heat_toy():
    """A <=> Q, Q <=> B with DIFFERENT enthalpies of formation and heat capacities (the toys of qss_synth share them, so that
    their heat release vanishes identically)."""
    lo = np.array([[3.6, 1.1e-3, -2.0e-7, 0.0, 0.0, -1.0e3, 1.0],          # A
                   [4.4, 0.7e-3, -1.0e-7, 0.0, 0.0, -9.0e3, 0.4],          # B
                   [4.0, 1.0e-3, -2.0e-7, 0.0, 0.0, -3.0e3, 2.2]])         # Q
    nasa_T = np.tile(np.array([T_LOW, T_MID, T_HIGH]), (3, 1))
    rx = [dict(reac=[(0, 1)], prod=[(2, 1)], arr=(3.0e3, 0.7, 3.0e4)), dict(reac=[(2, 1)], prod=[(1, 1)], arr=(7.0e2, -1.1, 1.2e4))]
    return assemble(2, 1, [[1], [1], [1]], nasa_T, lo, lo.copy(), rx, elem_weight=[12.011])


def test_heat_release_toy_closed_form():
    """Tdot = -T (h_A - h_B)/(RT) wdot_A / (A (cp_A/R - 1) + B (cp_B/R - 1)) with wdot_A = -(k1f k2f A - k1b k2b B)/(k1b + k2f);
    the energy row by differentiating that closed form (mpmath) in A, B and T."""
    m = _heat_toy()
    A0, B0, T0 = 2.0, 0.5, 1234.5

    def tdot(A, B, T):
        T = mp.mpf(T)
        (hA, sA, cA), (hB, sB, cB), (hQ, sQ, cQ) = (_nasa(m.nasa_lo[i], T) for i in range(3))
        k1f = mp.mpf(3.0e3) * T ** mp.mpf("0.7") * mp.e ** (-mp.mpf(3.0e4) / (R * T))
        k2f = mp.mpf(7.0e2) * T ** mp.mpf("-1.1") * mp.e ** (-mp.mpf(1.2e4) / (R * T))
        k1b = k1f / mp.e ** (-((hQ - sQ) - (hA - sA)))          # Kc = exp(-sum nu g/RT), sum nu = 0
        k2b = k2f / mp.e ** (-((hB - sB) - (hQ - sQ)))
        wA = -(k1f * k2f * A - k1b * k2b * B) / (k1b + k2f)
        return -T * (hA - hB) * wA / (A * (cA - 1) + B * (cB - 1))

    om = oracle.OracleMech(m)
    C = np.array([[A0], [B0]]); T = np.array([T0])
    o = oracle.evaluate_energy(om, C, T)
    ref = tdot(A0, B0, T0)
    assert abs(float(ref)) > 1.0                                       # (there is heat release in this toy)
    assert o["tdot"][0] == pytest.approx(float(ref), rel=1e-11)
    drow = [mp.diff(lambda a: tdot(a, B0, T0), A0), mp.diff(lambda b: tdot(A0, b, T0), B0), mp.diff(lambda t: tdot(A0, B0, t), T0)]
    for k in range(3):
        assert abs(o["erow"][k, 0] - float(drow[k])) <= 1e-10 * abs(float(drow[k])) + 1e-13 * o["escale"][k, 0], k


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "dag", "nonqss"])
def test_internal_energy_is_conserved_to_second_order(name):
    """Adiabatic constant-volume reactor (reading G17): U = sum_i C_i (H_i(T) - R T) over the transported species is conserved, so
    along one explicit Euler step (C + dt wdot, T + dt Tdot) its change is O(dt^2): halving dt divides it by four, and it is tiny
    against dt sum |u_i wdot_i|.  U is written out here in mpmath from the NASA-7 coefficients."""
    m = {"cfg1": lambda: config_mechanism(1), "cfg2": lambda: config_mechanism(2), "dag": toy_dag, "nonqss": toy_nonqss}[name]()
    n = 6
    C, T = (config_states(int(name[3]), n) if name.startswith("cfg") else make_states(m.n_nqss, n, 77))
    om = oracle.OracleMech(m)
    o = oracle.evaluate(om, C, T, n, want_jac=False)
    e = oracle.evaluate_energy(om, C, T, n)
    N = m.n_nqss

    def U(Cc, Tc):
        return sum(Cc[i] * R * Tc * (_nasa(_set(m, i, float(Tc)), Tc)[0] - 1) for i in range(N))

    for c in range(n):
        if abs(T[c] - m.nasa_T[0, 1]) < 5.0:
            continue                                                   # (a step across Tmid would mix the two NASA sets)
        Cc = [mp.mpf(C[i, c]) for i in range(N)]; Tc = mp.mpf(T[c])
        w = [mp.mpf(o["wdot"][i, c]) for i in range(N)]; td = mp.mpf(e["tdot"][c])
        heat = sum(abs(R * Tc * (_nasa(_set(m, i, T[c]), Tc)[0] - 1) * w[i]) for i in range(N))
        rate = max(max(abs(w[i]) / Cc[i] for i in range(N)), abs(td) / Tc)
        dt = mp.mpf("1e-4") / rate
        d1 = U([Cc[i] + dt * w[i] for i in range(N)], Tc + dt * td) - U(Cc, Tc)
        d2 = U([Cc[i] + dt / 2 * w[i] for i in range(N)], Tc + dt / 2 * td) - U(Cc, Tc)
        assert abs(d1) <= 1e-3 * dt * heat + mp.mpf("1e-9") * abs(U(Cc, Tc)), (c, d1, dt * heat)
        if abs(d1) > 1e-12 * dt * heat:                                # (the first-order term is gone to the oracle's rounding)
            assert 3.0 < abs(d1 / d2) < 5.0 or abs(d1) <= 1e-9 * dt * heat, (c, d1 / d2)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "dag"])
def test_energy_row_against_mechanical_derivatives_and_float128(name):
    """The explicit energy row (hand-differentiated -T E / Cv on top of the species block) against the SAME right-hand side
    differentiated mechanically (dual numbers, complex step), and the fp64 evaluation against float128."""
    m = {"cfg1": lambda: config_mechanism(1), "cfg2": lambda: config_mechanism(2), "dag": toy_dag}[name]()
    n = 24
    C, T = (config_states(int(name[3]), n) if name.startswith("cfg") else make_states(m.n_nqss, n, 77))
    om = oracle.OracleMech(m)
    e = oracle.evaluate_energy(om, C, T, n)
    q = oracle.evaluate_energy(om, C, T, n, mode=oracle.EXPLICIT_F128)
    assert np.all(np.abs(e["tdot"][:n] - q["tdot"][:n]) <= 1e-10 * np.abs(q["tdot"][:n]) + 1e-13 * q["escale"][-1, :n] * T[:n])
    for mode in (oracle.JAC_DUAL, oracle.JAC_CSTEP, oracle.EXPLICIT_F128):
        o = oracle.evaluate_energy(om, C, T, n, mode=mode)
        d = np.abs(o["erow"][:, :n] - e["erow"][:, :n])
        assert np.all(d <= 1e-9 * np.abs(e["erow"][:, :n]) + 1e-12 * e["escale"][:, :n]), (mode, float(np.max(d / (e["escale"][:, :n] + 1e-300))))
    # the row is not trivially small: |row| is within a few decades of its scale in most entries
    assert np.median(np.abs(e["erow"][:, :n]) / e["escale"][:, :n]) > 1e-6


def test_simplified_jacobians_coincide_with_the_exact_one_where_they_must():
    """Constant-QSS AJ = exact AJ without the chain term, zero-QSS AJ = additionally C_QSS := 0 in the partials.
    Without QSS species all three coincide; with QSS species the zero-QSS matrix equals the exact matrix of the mechanism in
    which every reaction that CONSUMES a QSS species in a direction has that direction disabled and the chain term dropped --
    restated here through the const-QSS mode on such a stripped mechanism -- and both approximations are far from the exact
    matrix in some columns of the synthetic mechanisms (Table 5a shape, L240-244)."""
    import dataclasses
    m0 = toy_nonqss()
    C, T = make_states(m0.n_nqss, 8, 3)
    om0 = oracle.OracleMech(m0)
    ex = oracle.evaluate(om0, C, T, 8)["jac"]
    for mode in (oracle.JAC_CONST_QSS, oracle.JAC_ZERO_QSS):
        assert np.array_equal(oracle.evaluate(om0, C, T, 8, mode=mode)["jac"], ex)
    m = config_mechanism(1)
    n = 32
    C, T = config_states(1, n)
    om = oracle.OracleMech(m)
    ex = oracle.evaluate(om, C, T, n)["jac"][:, :, :n]
    cq = oracle.evaluate(om, C, T, n, mode=oracle.JAC_CONST_QSS)["jac"][:, :, :n]
    zq = oracle.evaluate(om, C, T, n, mode=oracle.JAC_ZERO_QSS)["jac"][:, :, :n]
    # stripped mechanism: directions with a QSS reactant disabled (their rates vanish at C_QSS = 0)
    mask = m.dir_mask.copy()
    for j in range(m.n_reac):
        re, pr = m.reaction_sides(j)
        if any(s >= m.n_nqss for s, _ in re):
            mask[j] &= 2
        if any(s >= m.n_nqss for s, _ in pr):
            mask[j] &= 1
    # the rate constants of the remaining directions do not depend on the stripped ones, so W_x at y = 0 is the stripped
    # mechanism's W_x; its own (different) closure only enters the chain term, which the const-QSS mode drops
    ms = dataclasses.replace(m, dir_mask=mask)
    with np.errstate(all="ignore"):
        st = oracle.evaluate(oracle.OracleMech(ms), C, T, n, mode=oracle.JAC_CONST_QSS)["jac"][:, :, :n]
    assert np.isfinite(st).all() and np.allclose(zq, st, rtol=1e-12, atol=0.0)

    def eps(a):                                                        # PAPER.md Eq. 10
        return float(np.mean(np.sqrt(((a - ex) ** 2).sum((0, 1))) / np.sqrt((ex ** 2).sum((0, 1)))))

    def worst_col(a):                                                  # the whole-matrix norm is dominated by a few huge columns
        return float(np.max(np.sqrt(((a - ex) ** 2).sum(0)) / np.sqrt((ex ** 2).sum(0))))

    print("Eq.-10 error on cfg1: constant-QSS %.3g, zero-QSS %.3g; worst column %.3g / %.3g" % (eps(cq), eps(zq), worst_col(cq), worst_col(zq)))
    assert worst_col(cq) > 1e-2 and worst_col(zq) > 1e-2 and not np.allclose(cq, zq)


@pytest.mark.parametrize("cfg", [1, 2])
def test_finite_difference_temperature_column_against_the_analytic_one(cfg):
    """NEXT-3 (reading G22): the central difference with dT = 1e-4 T has a truncation error of
    (dT^2 / 6) w''' -- about 1e-8..1e-6 of the column -- and really is a difference (not the analytic column copied)."""
    m = config_mechanism(cfg); n = 64
    om = oracle.OracleMech(m)
    C, T = config_states(cfg, n)
    fd = oracle.evaluate_fdT(om, C, T, n); ex = oracle.evaluate(om, C, T, n, want_scale=True)
    N = m.n_nqss
    assert np.array_equal(fd["jac"][:, :N, :n], ex["jac"][:, :N, :n])
    a, b, s = fd["jac"][:, N, :n], ex["jac"][:, N, :n], ex["jscale"][:, N, :n]
    well = s <= 1e3 * np.abs(b)
    rel = np.abs(a - b)[well] / np.abs(b)[well]
    print("cfg%d FD-in-T column vs analytic: median %.2e, 99th percentile %.2e, well-conditioned %.2f" % (cfg, np.median(rel), np.quantile(rel, 0.99), well.mean()))
    assert well.mean() > 0.5 and np.median(rel) < 1e-6 and np.quantile(rel, 0.9) < 1e-4
    assert np.median(rel) > 1e-13                                        # a finite difference, not the analytic column
    # the perturbed temperatures are symmetric to rounding and the divisor is their exact difference
    assert np.allclose((fd["Tp"][:n] - fd["Tm"][:n]) / T[:n], 2e-4, rtol=1e-10)
