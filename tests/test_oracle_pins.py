"""Pins of the CPU oracle against things OTHER than itself (SURVEY.md section 8(c) "Pins").

Closed forms on toy mechanisms (sympy-derived in the survey, restated here and evaluated with mpmath),
closed-form equilibrium constants, Troe special cases, conservation laws, detailed-balance equilibrium,
closure residuals, mechanical derivatives (dual numbers, complex step), a float128 referee, the element
null space of every Jacobian column, and first-order convergence of one-sided finite differences
(App. C). No GPU is involved anywhere in this file.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import gates
import oracle
from qss_synth import (config_mechanism, config_states, make_states, toy1, toy2, toy3, toy_dag, toy_nonqss)
from qss_synth.mechanism import assemble
from qss_synth.toys import _toy_thermo

mp.mp.dps = 40
R = mp.mpf("8.31446261815324")
P0 = mp.mpf(101325)


def _one_cell(C, T):
    C = np.asarray(C, dtype=np.float64).reshape(-1, 1)
    return np.ascontiguousarray(C), np.array([float(T)])


def _arr(A, b, Ea, T):
    T = mp.mpf(T)
    return mp.mpf(A) * T ** mp.mpf(b) * mp.e ** (-mp.mpf(Ea) / (R * T))


# --------------------------------------------------------------------------------------------------
# toys: hand-derived closed forms
# --------------------------------------------------------------------------------------------------
def test_toy1_closed_form_with_T_column():
    """A <=> Q, Q <=> B, Q QSS:  Q = (k1f A + k2b B)/(k1b + k2f),
    wdot_A = -(k1f k2f A - k1b k2b B)/(k1b + k2f) = -wdot_B; the T column by differentiating the k's."""
    a7 = (1.0, 0.4, 2.2); beta = (0.7, -1.1); Ea = (3.0e4, 1.2e4)
    m = toy1(3.0e3, 7.0e2, a7, beta, Ea)
    A, B, T0 = 2.0, 0.5, 1234.5

    def wA(T):
        k1f = _arr(3.0e3, beta[0], Ea[0], T); k2f = _arr(7.0e2, beta[1], Ea[1], T)
        k1b = k1f / mp.e ** mp.mpf(a7[2] - a7[0]); k2b = k2f / mp.e ** mp.mpf(a7[1] - a7[2])
        return -(k1f * k2f * A - k1b * k2b * B) / (k1b + k2f), (k1f * A + k2b * B) / (k1b + k2f), (k1f, k2f, k1b, k2b)

    w, Q, (k1f, k2f, k1b, k2b) = wA(T0)
    dwdT = mp.diff(lambda t: wA(t)[0], T0)
    o = oracle.evaluate(oracle.OracleMech(m), *_one_cell([A, B], T0))
    assert o["cqss"][0, 0] == pytest.approx(float(Q), rel=1e-13)
    S = o["S"][0, 0]                                   # running-error scale: the two terms of wdot_A cancel
    assert abs(o["wdot"][0, 0] - float(w)) <= 1e-12 * abs(float(w)) + 1e-14 * S
    assert abs(o["wdot"][1, 0] + float(w)) <= 1e-12 * abs(float(w)) + 1e-14 * S
    J = o["jac"][:, :, 0]
    Js = oracle.evaluate(oracle.OracleMech(m), *_one_cell([A, B], T0), want_scale=True)["jscale"][:, :, 0]

    def near(val, ref, scale):      # entries are differences of large terms: guard with the running-error scale
        return abs(val - float(ref)) <= 1e-12 * abs(float(ref)) + 1e-14 * scale

    assert near(J[0, 0], -k1f * k2f / (k1b + k2f), Js[0, 0])
    assert near(J[0, 1], k1b * k2b / (k1b + k2f), Js[0, 1])
    assert near(J[1, 0], k1f * k2f / (k1b + k2f), Js[1, 0])
    assert near(J[0, 2], dwdT, Js[0, 2]) and near(J[1, 2], -dwdT, Js[1, 2])
    assert Js[0, 0] < 1e6 * abs(J[0, 0])               # ... and the guard is not what makes it pass


def test_toy2_coupled_group_closed_form():
    """A <=> Q1, Q1 <=> Q2, Q2 <=> B:  Delta = k1b k2b + k1b k3f + k2f k3f."""
    a7 = (1.0, 0.4, 2.2, 1.7)
    k1f, k2f, k3f = 3.0e3, 5.0e4, 7.0e2
    m = toy2(k1f, k2f, k3f, a7)                       # species order A, B, Q1, Q2
    k1b = k1f / math.exp(a7[2] - a7[0]); k2b = k2f / math.exp(a7[3] - a7[2]); k3b = k3f / math.exp(a7[1] - a7[3])
    A, B = 0.3, 4.0
    D = k1b * k2b + k1b * k3f + k2f * k3f
    o = oracle.evaluate(oracle.OracleMech(m), *_one_cell([A, B], 900.0))
    assert o["cqss"][0, 0] == pytest.approx((k1f * A * (k2b + k3f) + k2b * k3b * B) / D, rel=1e-13)
    assert o["cqss"][1, 0] == pytest.approx((k1f * k2f * A + (k1b + k2f) * k3b * B) / D, rel=1e-13)
    wA = -(k1f * k2f * k3f * A - k1b * k2b * k3b * B) / D
    assert o["wdot"][0, 0] == pytest.approx(wA, rel=1e-12)
    assert o["wdot"][1, 0] == pytest.approx(-wA, rel=1e-12)
    J = o["jac"][:, :, 0]
    assert J[0, 0] == pytest.approx(-k1f * k2f * k3f / D, rel=1e-12)
    assert J[0, 1] == pytest.approx(k1b * k2b * k3b / D, rel=1e-12)
    assert abs(J[0, 2]) <= 1e-9 * abs(wA)            # constant k's, Delta nu = 0: no T dependence


def test_toy3_bimolecular_closed_form():
    """A + B <=> Q + D, Q <=> E:  Q = (k1f A B + k2b E)/(k1b D + k2f),
    d wdot_A / dD = k1b k2f (k1f A B + k2b E)/(k1b D + k2f)^2."""
    a7 = (1.0, 0.4, 0.9, 1.3, 2.0)                     # A B D E Q
    k1f, k2f = 4.0e2, 9.0e3
    m = toy3(k1f, k2f, a7)
    k1b = k1f / math.exp(a7[4] + a7[2] - a7[0] - a7[1]); k2b = k2f / math.exp(a7[3] - a7[4])
    A, B, D, E = 1.5, 0.2, 3.0, 0.05
    o = oracle.evaluate(oracle.OracleMech(m), *_one_cell([A, B, D, E], 1500.0))
    den = k1b * D + k2f
    assert o["cqss"][0, 0] == pytest.approx((k1f * A * B + k2b * E) / den, rel=1e-13)
    wA = -(k1f * k2f * A * B - k1b * k2b * D * E) / den
    assert o["wdot"][0, 0] == pytest.approx(wA, rel=1e-12)
    assert o["wdot"][1, 0] == pytest.approx(wA, rel=1e-12)
    assert o["wdot"][2, 0] == pytest.approx(-wA, rel=1e-12)
    assert o["wdot"][3, 0] == pytest.approx(-wA, rel=1e-12)
    J = o["jac"][:, :, 0]
    assert J[0, 2] == pytest.approx(k1b * k2f * (k1f * A * B + k2b * E) / den ** 2, rel=1e-12)
    assert J[0, 0] == pytest.approx(-k1f * k2f * B / den, rel=1e-12)
    assert J[0, 3] == pytest.approx(k1b * k2b * D / den, rel=1e-12)


# --------------------------------------------------------------------------------------------------
# rate constants
# --------------------------------------------------------------------------------------------------
def _nasa_mp(a, T):
    T = mp.mpf(T); a = [mp.mpf(float(x)) for x in a]
    h = a[0] + a[1] * T / 2 + a[2] * T ** 2 / 3 + a[3] * T ** 3 / 4 + a[4] * T ** 4 / 5 + a[5] / T
    s = a[0] * mp.log(T) + a[1] * T + a[2] * T ** 2 / 2 + a[3] * T ** 3 / 3 + a[4] * T ** 4 / 4 + a[6]
    return h, s


@pytest.mark.parametrize("T", [650.0, 1000.0, 2210.0])
def test_arrhenius_and_kc_hand_calculation(T):
    """kf = A T^beta exp(-Ea/RT); Kc = exp(-sum nu g/RT) (P0/RT)^(sum nu); kb = kf/Kc -- evaluated
    independently with 40-digit mpmath on cfg1's mechanism (both NASA ranges and T == Tmid)."""
    m = config_mechanism(1)
    om = oracle.OracleMech(m)
    C = np.full(m.n_nqss, 1.0)
    kf, kb = oracle.rate_constants(om, C, T)
    for j in range(m.n_reac):
        A, b, Ea = m.arr[j]
        kref = _arr(A, b, Ea, T)
        assert kf[j] == pytest.approx(float(kref), rel=2e-13)
        re, pr = m.reaction_sides(j)
        lnKc = mp.mpf(0); dnu = 0
        for sp, nu in pr + [(s, -n) for s, n in re]:
            a = m.nasa_lo[sp] if T < m.nasa_T[sp, 1] else m.nasa_hi[sp]
            h, s = _nasa_mp(a, T)
            lnKc -= nu * (h - s); dnu += nu
        lnKc += dnu * mp.log(P0 / (R * mp.mpf(T)))
        assert kb[j] == pytest.approx(float(kref / mp.e ** lnKc), rel=5e-12)


def test_kc_closed_form_identical_thermo():
    """Identical NASA sets on both sides => Kc = (P0/RT)^(dnu); with only a7 differing and dnu = 0,
    Kc = exp(sum nu a7) and kb = kf/Kc."""
    T, lo, hi = _toy_thermo(np.array([0.0, 0.0, 0.0]))
    rx = [dict(reac=[(0, 1)], prod=[(1, 2)], arr=(5.0e3, 0.0, 0.0)),          # A <=> 2B, dnu = +1
          dict(reac=[(0, 1)], prod=[(2, 1)], arr=(2.0e3, 0.0, 0.0))]          # A <=> C,  dnu = 0
    m = assemble(3, 0, [[2], [1], [2]], T, lo, hi, rx, elem_weight=[1.0])
    Tc = 1111.0
    kf, kb = oracle.rate_constants(oracle.OracleMech(m), np.ones(3), Tc)
    # sum nu g/RT = (2-1) * g_common for reaction 0 -> not a pure power; use dnu = 0 reaction for exactness
    assert kb[1] == pytest.approx(kf[1], rel=1e-14)
    # reaction 0 with dnu = 1: Kc = exp(-g_common) * P0/(R T); g_common from mpmath
    h, s = _nasa_mp(lo[0], Tc)
    Kc0 = mp.e ** (-(h - s)) * P0 / (R * mp.mpf(Tc))
    assert kb[0] == pytest.approx(float(mp.mpf(5.0e3) / Kc0), rel=1e-12)


def _falloff_mech(troe, A_inf=1.0e10, A0=1.0e12):
    T, lo, hi = _toy_thermo(np.array([0.3, 0.9, 0.1]))
    rx = [dict(reac=[(0, 1)], prod=[(1, 1)], arr=(A_inf, 0.5, 2.0e4), type=2, arr_low=(A0, -0.5, 1.0e4),
               troe=troe, eff=[(2, 2.5)])]
    return assemble(3, 0, [[1], [1], [1]], T, lo, hi, rx, elem_weight=[1.0])


def test_troe_lindemann_special_case():
    """Fcent = 1 (alpha = 1, T* -> inf, T** -> inf) => F = 1 and k = k_inf Pr/(1+Pr), M = sum alpha_k C_k."""
    m = _falloff_mech((1.0, 100.0, 1e300, 1e300))
    C = np.array([0.7, 1.3, 4.0]); T = 1350.0
    kf, _ = oracle.rate_constants(oracle.OracleMech(m), C, T)
    kinf = _arr(1.0e10, 0.5, 2.0e4, T); k0 = _arr(1.0e12, -0.5, 1.0e4, T)
    M = mp.mpf(0.7) + mp.mpf(1.3) + mp.mpf(2.5) * 4
    Pr = k0 * M / kinf
    assert kf[0] == pytest.approx(float(kinf * Pr / (1 + Pr)), rel=1e-13)


def test_troe_blending_and_limits():
    """Troe F restated with mpmath at an intermediate Pr (a retyping check only; the pins of the blending function
    are the hand-derived points of test_troe_blending_hand_derived_points below), plus the high-pressure limit
    f1 -> -1/0.14 => F -> Fcent^(1/(1+0.14^-2)) (approached like 1/log10 Pr, hence the loose tolerance; the 0.14 itself
    is pinned at the pole of f1 below)."""
    troe = (0.6, 120.0, 1500.0, 5000.0)
    m = _falloff_mech(troe)
    om = oracle.OracleMech(m)
    T = 1400.0

    def k_ref(C):
        kinf = _arr(1.0e10, 0.5, 2.0e4, T); k0 = _arr(1.0e12, -0.5, 1.0e4, T)
        M = mp.mpf(C[0]) + mp.mpf(C[1]) + mp.mpf(2.5) * mp.mpf(C[2])
        Pr = k0 * M / kinf
        Tm = mp.mpf(T)
        Fc = (1 - mp.mpf(troe[0])) * mp.e ** (-Tm / troe[1]) + mp.mpf(troe[0]) * mp.e ** (-Tm / troe[2]) + mp.e ** (-mp.mpf(troe[3]) / Tm)
        L = mp.log10(Pr); Lc = mp.log10(Fc)
        c = mp.mpf("-0.4") - mp.mpf("0.67") * Lc; n = mp.mpf("0.75") - mp.mpf("1.27") * Lc
        f1 = (L + c) / (n - mp.mpf("0.14") * (L + c))
        F = mp.mpf(10) ** (Lc / (1 + f1 ** 2))
        return kinf * Pr / (1 + Pr) * F, kinf, Fc

    for C in ([0.7, 1.3, 4.0], [1e-3, 2e-3, 1e-4], [300.0, 20.0, 90.0]):
        kf, _ = oracle.rate_constants(om, np.array(C), T)
        assert kf[0] == pytest.approx(float(k_ref(C)[0]), rel=1e-12)
    Chuge = [1e200, 1e200, 1e200]
    kf, _ = oracle.rate_constants(om, np.array(Chuge), T)
    _, kinf, Fc = k_ref(Chuge)
    expo = 1.0 / (1.0 + (1.0 / 0.14) ** 2)
    assert kf[0] == pytest.approx(float(kinf * Fc ** expo), rel=2e-2)     # approached like 1/log10(Pr)


def _fcent_pinned(T, alpha, e3, e1, e2):
    """Troe parameters for which the three exponentials of Fcent take the given VALUES at temperature T
    (T*** = T/ln(1/e3), T* = T/ln(1/e1), T** = T ln(1/e2)), so that Fcent = (1-alpha) e3 + alpha e1 + e2 is a
    number fixed by hand, not by any code."""
    return (alpha, T / math.log(1.0 / e3), T / math.log(1.0 / e1), T * math.log(1.0 / e2))


# (alpha, e3, e1, e2) -> Fcent by hand: 0.4*0.5 + 0.6*0.25 + 0.25 = 0.6 ; 0.75*0.125 + 0.25*0.5 + 0.0625 = 0.28125.
# Swapping the roles of T*** and T* gives 0.65 / 0.46875, dropping the T** term 0.35 / 0.21875.
_FCENT_CASES = [((0.6, 0.5, 0.25, 0.25), 0.6), ((0.25, 0.125, 0.5, 0.0625), 0.28125)]


@pytest.mark.parametrize("case", [0, 1])
@pytest.mark.parametrize("point", ["f1=0", "f1=+1", "f1=-1", "f1=inf"])
def test_troe_blending_hand_derived_points(case, point):
    """Pins the Troe blending F(Pr, Fcent) at intermediate Pr with values no code supplies (the rate forms are not in
    the paper: the pins come from the mathematics).  With c = -0.4 - 0.67 log10 Fcent,
    n = 0.75 - 1.27 log10 Fcent and f1 = (log10 Pr + c)/(n - 0.14 (log10 Pr + c)), log10 F = log10 Fcent/(1 + f1^2):
      log10 Pr = -c             => f1 = 0    => F = Fcent
      log10 Pr = n/1.14 - c     => f1 = +1   => F = Fcent^(1/2)
      log10 Pr = -n/0.86 - c    => f1 = -1   => F = Fcent^(1/2)
      log10 Pr = n/0.14 - c     => f1 = inf  => F = 1            (the pole of f1: pins the 0.14)
    Each at two values of Fcent, so that every one of the five constants is separated: any single wrong or swapped
    constant moves f1 away from the special value at one of these points and F changes in the 2nd-3rd digit."""
    (alpha, e3, e1, e2), Fc = _FCENT_CASES[case]
    T = 1400.0
    m = _falloff_mech(_fcent_pinned(T, alpha, e3, e1, e2))
    om = oracle.OracleMech(m)
    kinf = _arr(1.0e10, 0.5, 2.0e4, T); k0 = _arr(1.0e12, -0.5, 1.0e4, T)
    Lc = mp.log10(mp.mpf(Fc))
    c = mp.mpf("-0.4") - mp.mpf("0.67") * Lc
    n = mp.mpf("0.75") - mp.mpf("1.27") * Lc
    L, F = {"f1=0": (-c, mp.mpf(Fc)), "f1=+1": (n / mp.mpf("1.14") - c, mp.sqrt(mp.mpf(Fc))),
            "f1=-1": (-n / mp.mpf("0.86") - c, mp.sqrt(mp.mpf(Fc))), "f1=inf": (n / mp.mpf("0.14") - c, mp.mpf(1))}[point]
    Pr = mp.mpf(10) ** L
    M = Pr * kinf / k0                                  # third-body concentration that gives this Pr
    C = np.array([float(M) * 0.25, float(M) * 0.25, 0.0])
    C[2] = float((M - mp.mpf(C[0]) - mp.mpf(C[1])) / mp.mpf("2.5"))          # M = C0 + C1 + 2.5 C2
    assert C[2] > 0
    kf, _ = oracle.rate_constants(om, C, T)
    tol = 1e-12 if point != "f1=inf" else 1e-10        # at the pole f1 ~ 1e15, F = Fcent^(1e-30)
    assert kf[0] == pytest.approx(float(kinf * Pr / (1 + Pr) * F), rel=tol)
    # the pin separates the constants: the neighbouring "wrong" values differ by far more than the tolerance
    assert abs(float(mp.mpf(Fc) ** mp.mpf("0.5")) - Fc) > 1e-2


def test_troe_chemkin_placeholder_parameters():
    """CHEMKIN files use T*** ~ 1e-30 and T*, T** ~ 1e30 as placeholders for an absent term: the exponentials are then
    exactly 0 / 1 / 0 and Fcent = alpha (the arguments -T/T*** = -1e33 are far outside any polynomial exp)."""
    alpha = 0.37
    m = _falloff_mech((alpha, 1.0e-30, 1.0e30, 1.0e30))
    T = 1400.0
    kinf = _arr(1.0e10, 0.5, 2.0e4, T); k0 = _arr(1.0e12, -0.5, 1.0e4, T)
    Lc = mp.log10(mp.mpf(alpha))
    c = mp.mpf("-0.4") - mp.mpf("0.67") * Lc
    M = mp.mpf(10) ** (-c) * kinf / k0                  # f1 = 0 => F = Fcent = alpha
    C = np.array([float(M) * 0.5, float(M) * 0.5, 0.0])
    kf, _ = oracle.rate_constants(oracle.OracleMech(m), C, T)
    Pr = k0 * (mp.mpf(C[0]) + mp.mpf(C[1])) / kinf
    assert np.isfinite(kf[0])
    assert kf[0] == pytest.approx(float(kinf * Pr / (1 + Pr) * alpha), rel=1e-12)


# --------------------------------------------------------------------------------------------------
# invariants on the BASELINE-shaped mechanisms
# --------------------------------------------------------------------------------------------------
MECHS = {"cfg1": lambda: config_mechanism(1), "cfg2": lambda: config_mechanism(2), "dag": toy_dag}


def _states_for(name, m, n):
    if name == "cfg1":
        return config_states(1, n)
    if name == "cfg2":
        return config_states(2, n)
    return make_states(m.n_nqss, n, 77)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "dag"])
def test_mass_and_element_conservation(name):
    """sum_i a_ie wdot_i = 0 for every element (QSS species included implicitly: their rates are the
    closure residuals, zero), hence sum_i W_i wdot_i = 0 (Eq. 3-4)."""
    m = MECHS[name](); n = 96
    C, T = _states_for(name, m, n)
    o = oracle.evaluate(oracle.OracleMech(m), C, T, n, want_jac=False)
    a = m.comp[:m.n_nqss].astype(np.float64)                        # [N, n_elem]
    for e in range(m.n_elem):
        tot = (a[:, e, None] * o["wdot"][:, :n]).sum(0)
        scale = (a[:, e, None] * o["S"][:, :n]).sum(0)
        assert np.all(np.abs(tot) <= 2e-14 * scale + 1e-300), f"element {e}: {np.max(np.abs(tot) / scale)}"
    W = m.species_weight()[:m.n_nqss]
    tot = (W[:, None] * o["wdot"][:, :n]).sum(0); scale = (W[:, None] * o["S"][:, :n]).sum(0)
    assert np.all(np.abs(tot) <= 2e-14 * scale)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "dag"])
def test_closure_residual_and_positivity(name):
    """Eq. 4: the net production rate of every QSS species vanishes at the closure solution; y >= 0."""
    m = MECHS[name](); n = 48
    C, T = _states_for(name, m, n)
    om = oracle.OracleMech(m)
    for c in range(n):
        y, res, sc = oracle.closure_check(om, C[:, c], T[c])
        assert np.all(y >= 0)
        assert np.all(np.abs(res) <= 1e-14 * sc), np.max(np.abs(res) / sc)


def _g_RT_numpy(m, T):
    a = np.where((T < m.nasa_T[:, 1])[:, None], m.nasa_lo, m.nasa_hi)
    h = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T ** 2 / 3 + a[:, 3] * T ** 3 / 4 + a[:, 4] * T ** 4 / 5 + a[:, 5] / T
    s = a[:, 0] * np.log(T) + a[:, 1] * T + a[:, 2] * T ** 2 / 2 + a[:, 3] * T ** 3 / 3 + a[:, 4] * T ** 4 / 4 + a[:, 6]
    return h - s


@pytest.mark.parametrize("cfg", [1, 2])
def test_detailed_balance_equilibrium(cfg):
    """For any element potentials mu and T, C_s = (P0/RT) exp(-g_s/RT + sum_e a_se mu_e) makes every
    reversible reaction's net rate zero: wdot = 0 (relative to S) AND the closure must return
    y_m = C_m^eq. All reactions of the generated configs are reversible and element-conserving."""
    m = config_mechanism(cfg)
    rng = np.random.default_rng(5)
    n = 24
    N = m.n_nqss
    C = np.zeros((N, 32)); T = np.full(32, 1000.0); yeq = np.zeros((m.n_qss, 32))
    for c in range(32):
        Tc = rng.uniform(900.0, 2400.0)
        mu = rng.uniform(-3.0, 0.0, size=m.n_elem)
        Ceq = (101325.0 / (8.31446261815324 * Tc)) * np.exp(-_g_RT_numpy(m, Tc) + m.comp @ mu)
        scale = 50.0 / Ceq[:N].sum()                       # keep total concentration moderate: rescale via mu shift
        # a uniform scale is NOT an equilibrium unless sum(nu)=0, so fold it into the potentials instead:
        lam = math.log(scale) / max(m.comp.sum(1).max(), 1)
        Ceq = (101325.0 / (8.31446261815324 * Tc)) * np.exp(-_g_RT_numpy(m, Tc) + m.comp @ (mu + lam))
        C[:, c] = Ceq[:N]; T[c] = Tc; yeq[:, c] = Ceq[N:]
    o = oracle.evaluate(oracle.OracleMech(m), C, T, n, want_jac=False)
    assert np.all(np.abs(o["wdot"][:, :n]) <= 2e-12 * o["S"][:, :n])
    assert np.allclose(o["cqss"][:, :n], yeq[:, :n], rtol=2e-12, atol=0)


# --------------------------------------------------------------------------------------------------
# Jacobian
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["cfg1", "cfg2", "dag"])
def test_jacobian_vs_dual_and_complex_step(name):
    """The hand-derived explicit formulas agree with mechanical differentiation of the wdot routine."""
    m = MECHS[name](); n = 64
    C, T = _states_for(name, m, n)
    om = oracle.OracleMech(m)
    ref = oracle.evaluate(om, C, T, n, want_scale=True)
    for mode in (oracle.JAC_DUAL, oracle.JAC_CSTEP):
        o = oracle.evaluate(om, C, T, n, mode=mode)
        gates.assert_jac(o["jac"], ref["jac"], ref["jscale"], n, what=f"{name} mode {mode}")


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "dag"])
def test_double_oracle_meets_gates_against_float128(name):
    """The oracle itself must meet both tiers against its own __float128 instantiation."""
    m = MECHS[name](); n = 128
    C, T = _states_for(name, m, n)
    om = oracle.OracleMech(m)
    d = oracle.evaluate(om, C, T, n, want_scale=True)
    q = oracle.evaluate(om, C, T, n, want_scale=True, mode=oracle.EXPLICIT_F128)
    cfg = {"cfg1": 1, "cfg2": 2}.get(name)              # floors under the well-conditioned filter (gates.WELLCOND_FLOOR)
    gw = gates.assert_wdot(d["wdot"], q["wdot"], q["S"], n, what=name, cfg=cfg)
    gj = gates.assert_jac(d["jac"], q["jac"], q["jscale"], n, what=name, cfg=cfg)
    # reading G16 as evidence: what the fp64 ORACLE itself reaches on the unfiltered strict tier against float128
    print(f"[gates] oracle fp64 vs float128, {name}: wdot tier-1 unfiltered {gw['tier1_frac_unfiltered']:.4f} (filtered {gw['tier1_frac']:.4f}, "
          f"well-conditioned {gw['wellcond_frac']:.4f}); columns unfiltered {gj['col_tier1_frac_unfiltered']:.4f} (filtered {gj['col_tier1_frac']:.4f}, "
          f"well-conditioned {gj['col_wellcond_frac']:.4f})")
    assert np.allclose(d["cqss"][:, :n], q["cqss"][:, :n], rtol=1e-12)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "dag"])
def test_jacobian_element_null_space(name):
    """sum_i a_ie J_ik = 0 for every element e and every column k incl. T. Holds ONLY with the chain
    term W_y*Y_x (Eq. 9 second parenthesis): the constant-QSS matrix (L232) violates it."""
    m = MECHS[name](); n = 64
    C, T = _states_for(name, m, n)
    om = oracle.OracleMech(m)
    o = oracle.evaluate(om, C, T, n, want_scale=True)
    oc = oracle.evaluate(om, C, T, n, mode=oracle.JAC_CONST_QSS)
    a = m.comp[:m.n_nqss].astype(np.float64)
    worst_exact, worst_const = 0.0, 0.0
    for e in range(m.n_elem):
        if not a[:, e].any():
            continue
        tot = np.einsum("i,ikc->kc", a[:, e], o["jac"][:, :, :n])
        sc = np.einsum("i,ikc->kc", a[:, e], o["jscale"][:, :, :n])
        ok = sc > 0
        worst_exact = max(worst_exact, float(np.max(np.abs(tot[ok]) / sc[ok])))
        totc = np.einsum("i,ikc->kc", a[:, e], oc["jac"][:, :, :n])
        worst_const = max(worst_const, float(np.max(np.abs(totc[ok]) / sc[ok])))
    assert worst_exact <= 1e-13, worst_exact
    assert worst_const >= 1e-6, worst_const            # the approximation breaks the invariant grossly


@pytest.mark.parametrize("cfg", [1, 2])
def test_constant_qss_jacobian_error_is_order_one(cfg):
    """Dropping the chain term gives an O(0.1-1) error (Table 5a shape, L240-244), not ~0.
    Column-wise on both configs (cfg1's whole-matrix norm is dominated by one non-QSS entry and cannot see
    it); whole-matrix Eq. 10 with the paper's sampling (L234) on the 35+18-shaped cfg2."""
    m = config_mechanism(cfg); n = 100
    om = oracle.OracleMech(m)
    C, T = config_states(cfg, n)
    ex = oracle.evaluate(om, C, T, n)["jac"][:, :, :n]; co = oracle.evaluate(om, C, T, n, mode=oracle.JAC_CONST_QSS)["jac"][:, :, :n]
    errc = np.sqrt(((ex - co) ** 2).sum(0)) / np.sqrt((ex ** 2).sum(0))
    assert np.median(errc) > 0.05, np.median(errc)
    if cfg == 2:
        rng = np.random.default_rng(3)
        C = np.ascontiguousarray(rng.uniform(1e-4, 1.0, size=(m.n_nqss, n))); T = rng.uniform(300.0, 1300.0, size=n)
        ex = oracle.evaluate(om, C, T)["jac"]; co = oracle.evaluate(om, C, T, mode=oracle.JAC_CONST_QSS)["jac"]
        err = np.sqrt(((ex - co) ** 2).sum((0, 1))) / np.sqrt((ex ** 2).sum((0, 1)))
        assert 0.05 < np.median(err) < 100.0, np.median(err)


def test_no_qss_species_reduces_to_textbook_jacobian():
    """N_q = 0: J_ik = sum_j nu_ij dQ_j/dx_k (ref [37]) written out densely in numpy with
    per-reaction complex-step derivatives of the rate-of-progress (no closure anywhere)."""
    m = toy_nonqss(); n = 16
    C, T = make_states(m.n_nqss, n, 9)
    om = oracle.OracleMech(m)
    o = oracle.evaluate(om, C, T, n, want_scale=True)
    assert o["cqss"].shape[0] == 0
    N = m.n_nqss
    for c in range(4):
        J = np.zeros((N, N + 1))
        # C columns from the product rule with rate constants at the base point; the dependence of k on
        # C_k through the third-body concentration M by central differences of the rate constants
        kf, kb = oracle.rate_constants(om, C[:, c], T[c])
        for k in range(N):
            dC = C[:, c].sum() * 1e-6
            Cp = C[:, c].copy(); Cp[k] += dC
            Cm = C[:, c].copy(); Cm[k] -= dC
            kfp, kbp = oracle.rate_constants(om, Cp, T[c]); kfm, kbm = oracle.rate_constants(om, Cm, T[c])
            for j in range(m.n_reac):
                re, pr = m.reaction_sides(j)
                def prod_and_partial(side, kk):
                    val = 1.0; part = 0.0
                    for s, nu in side:
                        val *= C[s, c] ** nu
                    for s, nu in side:
                        if s == k:
                            others = 1.0
                            for s2, nu2 in side:
                                if s2 != k:
                                    others *= C[s2, c] ** nu2
                            part = nu * C[k, c] ** (nu - 1) * others
                    return val, part
                vf, pf = prod_and_partial(re, k); vb, pb = prod_and_partial(pr, k)
                dQ = kf[j] * pf - kb[j] * pb + (kfp[j] - kfm[j]) / (2 * dC) * vf - (kbp[j] - kbm[j]) / (2 * dC) * vb
                for s, nu in pr:
                    J[s, k] += nu * dQ
                for s, nu in re:
                    J[s, k] -= nu * dQ
        ref = o["jac"][:, :N, c]
        assert np.linalg.norm(J[:, :N] - ref) <= 1e-6 * np.linalg.norm(ref)
    # and the mechanical derivative agrees to rounding
    d = oracle.evaluate(om, C, T, n, mode=oracle.JAC_CSTEP)
    gates.assert_jac(d["jac"], o["jac"], o["jscale"], n)


def test_finite_difference_converges_at_first_order():
    """PAPER.md App. C (L477-481): a one-sided FD Jacobian converges to the analytical one at first order
    in Delta C; sampling C ~ U[0.1, 1.1] mol/m^3, T ~ U[300, 1300] K as in the paper."""
    m = config_mechanism(1); n = 40
    rng = np.random.default_rng(12)
    C = np.ascontiguousarray(rng.uniform(0.1, 1.1, size=(m.n_nqss, n))); T = rng.uniform(300.0, 1300.0, size=n)
    om = oracle.OracleMech(m)
    base = oracle.evaluate(om, C, T)
    N = m.n_nqss
    errs = []
    for dC in (1e-2, 1e-3, 1e-4):
        Jfd = np.zeros((N, N, n))
        for k in range(N):
            Cp = C.copy(); Cp[k] += dC
            wp = oracle.evaluate(om, Cp, T, want_jac=False)["wdot"]
            Jfd[:, k, :] = (wp - base["wdot"]) / dC
        ref = base["jac"][:, :N, :]
        e = np.sqrt(((Jfd - ref) ** 2).sum((0, 1))) / np.sqrt((ref ** 2).sum((0, 1)))
        errs.append(np.mean(e))
    assert 5.0 < errs[0] / errs[1] < 20.0, errs
    assert 5.0 < errs[1] / errs[2] < 20.0, errs


def test_golden_regression():
    """tests/golden/oracle_toys.txt (written by tests/golden/make_golden.py from the oracle alone): the oracle reproduces its stored
    values; a change of its arithmetic has to come with a regenerated fixture and the passage that justifies it."""
    import importlib.util
    here = os.path.dirname(os.path.abspath(__file__))
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "golden", "make_golden.py"))
    mg = importlib.util.module_from_spec(spec); spec.loader.exec_module(mg)
    stored = np.loadtxt(os.path.join(here, "golden", "oracle_toys.txt"), comments="#")
    now = np.concatenate([mg.values(name, n) for name, n in mg.CASES])
    assert stored.shape == now.shape
    scale = np.maximum(np.abs(stored), 1e-300)
    assert np.all(np.abs(now - stored) <= 1e-12 * scale + 1e-280), float(np.max(np.abs(now - stored) / scale))
