"""Pins of the oracle's 0-D integrator (NEXT-4; oracle.bdf1_advance, reading G21: backward-Euler substeps, full Newton
iterations with the exact (N+1) x (N+1) Jacobian) against what the mathematics fixes: first-order convergence to an independent
high-accuracy solution of the same ODE (scipy's Radau on the oracle's right-hand side), quadratic convergence of the Newton
iteration (which needs the EXACT Jacobian, energy row included), element conservation to rounding after every substep (a linear
invariant: needs a^T J = 0 and a consistent solve), fixed point at h = 0."""
from __future__ import annotations

import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from qss_synth import config_mechanism, config_states, make_states, toy3, toy_dag


def _rhs(om, N):
    def f(t, y):
        C = np.ascontiguousarray(np.maximum(y[:N], 0.0)[:, None]); T = np.array([y[N]])
        w = oracle.evaluate(om, C, T, 1, want_jac=False, nthreads=1)["wdot"][:, 0]          # (one cell: no thread team)
        td = oracle.evaluate_energy(om, C, T, 1, nthreads=1)["tdot"][0]
        return np.concatenate([w, [td]])
    return f


def _time_scale(om, C, T):
    ev = oracle.evaluate(om, C, T); en = oracle.evaluate_energy(om, C, T)
    return 1.0 / np.maximum(np.abs(ev["jac"]).max((0, 1)), np.abs(en["erow"]).max(0))


@pytest.mark.parametrize("mk", [toy3, toy_dag])
def test_first_order_convergence_to_radau(mk):
    m = mk(); om = oracle.OracleMech(m); N = m.n_nqss
    C, T = make_states(N, 2, seed=4)
    tau = _time_scale(om, C, T)
    tend = 2.0 * tau                                                    # a couple of the fastest time scales: the state moves visibly
    errs = []
    ref = []
    for c in range(2):
        sol = solve_ivp(_rhs(om, N), (0.0, tend[c]), np.concatenate([C[:, c], [T[c]]]), method="Radau", rtol=1e-11, atol=1e-14 * np.abs(C[:, c]).max())
        assert sol.success
        ref.append(sol.y[:, -1])
    ref = np.array(ref).T
    for nsub in (8, 16, 32, 64):
        Cn, Tn = oracle.bdf1_advance(om, C, T, tend / nsub, nsub, 6, 2)
        y = np.vstack([Cn, Tn[None]])[:, :2]
        errs.append(np.abs(y - ref).max(0) / np.abs(ref).max(0))
    errs = np.array(errs)
    assert (np.abs(ref[:N] - C[:, :2]).max(0) > 1e-3 * np.abs(C[:, :2]).max(0)).all(), "the state did not move: the test would be vacuous"
    ratio = errs[:-1] / errs[1:]
    print("backward Euler error vs Radau:", errs.T, "ratios", ratio.T)
    assert (errs[-1] < 0.05).all() and (ratio[-1] > 1.6).all() and (ratio[-1] < 2.5).all(), ratio


def test_newton_iteration_converges_quadratically_with_the_exact_jacobian():
    m = config_mechanism(1); om = oracle.OracleMech(m); N = m.n_nqss
    C, T = config_states(1, 8)
    h = 3.0 * _time_scale(om, C, T)
    sols = []
    for it in (1, 2, 3, 4, 8):
        Cn, Tn = oracle.bdf1_advance(om, C, T, h, 1, it, 8)
        sols.append(np.vstack([Cn, Tn[None]])[:, :8])
    ref = sols[-1]
    e = np.array([np.abs(s - ref).max(0) / np.abs(ref).max(0) for s in sols[:-1]])
    print("Newton error after 1..4 iterations:", e.max(1))
    ok = e[0] > 1e-9                                                    # cells that needed more than one iteration
    assert ok.any()
    # quadratic: e_{m+1} ~ K e_m^2 (checked as e_{m+1} <= 10 e_m^1.5: a linearly converging iteration, e.g. with an approximate
    # Jacobian or a wrong energy row, gives e_{m+1} ~ rho e_m and fails)
    for mm in (1, 2):
        assert (e[mm + 1][ok] <= np.maximum(1e-13, 10.0 * e[mm][ok] ** 1.5)).all(), e
    assert (e[3] <= 1e-8).all(), e


@pytest.mark.parametrize("cfg", [1, 2])
def test_elements_are_conserved_to_rounding(cfg):
    m = config_mechanism(cfg); om = oracle.OracleMech(m); N = m.n_nqss
    n = 6
    C, T = config_states(cfg, n)
    h = 10.0 * _time_scale(om, C, T)
    a = m.comp[:N].astype(np.float64)                                   # [N, n_elem]
    Cn, Tn = oracle.bdf1_advance(om, C, T, h, 3, 3, n)
    e0 = a.T @ C[:, :n]; e1 = a.T @ Cn[:, :n]
    scale = np.abs(a).T @ np.maximum(np.abs(C[:, :n]), np.abs(Cn[:, :n]))
    assert (np.abs(Cn[:, :n] - C[:, :n]).max(0) > 1e-6 * np.abs(C[:, :n]).max(0)).sum() >= 2, "the state did not move"
    assert np.abs(e1 - e0).max() <= 1e-11 * scale.max(), np.abs(e1 - e0).max() / scale.max()


def test_zero_step_is_the_identity():
    m = config_mechanism(1); om = oracle.OracleMech(m)
    C, T = config_states(1, 4)
    Cn, Tn = oracle.bdf1_advance(om, C, T, np.zeros(C.shape[1]), 2, 2)
    assert np.array_equal(Cn, C) and np.array_equal(Tn, T)


def test_adaptive_integrator_reaches_t_end_and_matches_radau():
    """oracle.ignition_advance (reading G23): every cell reaches t_end exactly (the last step is clipped), rejected attempts leave the
    state untouched and shrink the step, and the result agrees with scipy's Radau on the oracle's right-hand side to the order of the
    method's error at the accepted step sizes (backward Euler: first order; the Newton tolerance only controls the solve)."""
    m = toy_dag(); om = oracle.OracleMech(m); N = m.n_nqss
    C, T = make_states(N, 4, seed=4)
    tau = _time_scale(om, C, T)
    t_end = float(2.0 * tau[:4].min())
    out = oracle.ignition_advance(om, C, T, 0.02 * tau, np.zeros(C.shape[1]), t_end, 400, 3, 4, rtol=1e-9, atol_C=1e-14 * np.abs(C).max(), atol_T=1e-9)
    assert np.all(out["t"][:4] == t_end)                                # reached exactly: h = min(dt, t_end - t), then h = 0
    assert (out["accepted"][:4] >= 5).all()
    for c in range(4):
        sol = solve_ivp(_rhs(om, N), (0.0, t_end), np.concatenate([C[:, c], [T[c]]]), method="Radau", rtol=1e-11, atol=1e-14 * np.abs(C[:, c]).max())
        y = np.concatenate([out["C"][:, c], [out["T"][c]]])
        assert np.abs(y - sol.y[:, -1]).max() / np.abs(sol.y[:, -1]).max() < 0.05
    # a step far too large for three Newton iterations is rejected: state unchanged, step shrunk, nothing accepted, time not advanced
    big = oracle.ignition_advance(om, C, T, 1e6 * tau, np.zeros(C.shape[1]), 1e9 * float(tau.max()), 1, 1, 4, rtol=1e-12, atol_C=0.0, atol_T=0.0)
    assert (big["accepted"][:4] == 0).all() and np.array_equal(big["C"], C) and np.array_equal(big["T"], T)
    assert np.allclose(big["dt"][:4], 0.25e6 * tau[:4]) and (big["t"][:4] == 0).all()
    # with everything accepted and no growth the adaptive form IS the fixed-step integrator
    fix = oracle.bdf1_advance(om, C, T, 0.01 * tau, 5, 4, 4)
    ada = oracle.ignition_advance(om, C, T, 0.01 * tau, np.zeros(C.shape[1]), 1e9, 5, 4, 4, rtol=1.0, atol_C=1e300, atol_T=1e300, grow=1.0)
    assert np.array_equal(ada["C"][:, :4], fix[0][:, :4]) and np.array_equal(ada["T"][:4], fix[1][:4]) and (ada["accepted"][:4] == 5).all()


def test_ignition_time_is_the_first_accepted_time_above_the_threshold():
    m = config_mechanism(1); om = oracle.OracleMech(m)
    C, T = config_states(1, 8)
    tau = _time_scale(om, C, T)
    out = oracle.ignition_advance(om, C, T, 0.5 * tau, np.zeros(C.shape[1]), 1e9, 30, 3, 8, dT_ign=1e-3, rtol=1e-6)
    moved = np.abs(out["T"][:8] - T[:8]) > 0
    assert moved.any()
    up = out["T"][:8] - T[:8] >= 1e-3
    assert np.all(np.isnan(out["t_ign"][:8]) | (out["t_ign"][:8] <= out["t"][:8])) and np.all(np.isfinite(out["t_ign"][:8])[up])
    assert np.isfinite(out["t_ign"][:8]).any()
    # replay with a trace of T: t_ign is the time of the first accepted state at or above T0 + dT_ign
    t = np.zeros(C.shape[1]); dt = 0.5 * tau; Cc, Tc = C, T; tig = None; first = np.full(8, np.nan)
    for a in range(30):
        o = oracle.ignition_advance(om, Cc, Tc, dt, t, 1e9, 1, 3, 8, dT_ign=1e-3, rtol=1e-6, T0=T, t_ign=tig)
        Cc, Tc, dt, t, tig = o["C"], o["T"], o["dt"], o["t"], o["t_ign"]
        hit = np.isnan(first) & (Tc[:8] - T[:8] >= 1e-3)
        first[hit] = t[:8][hit]
    assert np.array_equal(first, out["t_ign"][:8], equal_nan=True) and np.array_equal(Tc[:8], out["T"][:8])
