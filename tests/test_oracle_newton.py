"""Pins of the Newton-solve oracle (NEXT-2; oracle/qss_newton_oracle.cpp, reading G20) against what the mathematics
fixes: exact cases (gamma = 0, scaled permutations, integer systems), Cramer's rule, LAPACK (numpy.linalg.solve re-derives the
matrix from the SoA arrays in numpy: an independent assembly AND an independent elimination), the float128 run, the backward
error in extended precision.  Each pin names the mistake it catches."""
from __future__ import annotations

import numpy as np
import pytest

import gates
import oracle
from qss_synth import config_mechanism, config_states, newton_inputs


def soa(Js, gam, bs):
    """List of (n x n J, gamma, b) -> SoA arrays with the energy row split off (n = N + 1)."""
    m, n = len(Js), Js[0].shape[0]
    N = n - 1
    jac = np.zeros((N, N + 1, m)); erow = np.zeros((N + 1, m)); b = np.zeros((n, m))
    for c, (J, rhs) in enumerate(zip(Js, bs)):
        jac[:, :, c] = J[:N, :]; erow[:, c] = J[N, :]; b[:, c] = rhs
    return jac, erow, np.ascontiguousarray(np.asarray(gam, dtype=np.float64)), b


def test_gamma_zero_returns_b_exactly():
    d = newton_inputs(7, 9, 3)
    g0 = np.zeros_like(d["gamma"])
    o = oracle.newton_solve(d["jac"], d["erow"], g0, d["b"])
    assert np.array_equal(o["x"], d["b"]) and not o["info"].any()


def test_scaled_permutation_is_solved_exactly_and_needs_row_interchanges():
    """I - gamma J = P D with a zero diagonal: elimination WITHOUT pivoting divides by zero; with it the result is exact."""
    rng = np.random.default_rng(5); n = 6
    Js, bs, xs = [], [], []
    for _ in range(8):
        perm = np.roll(np.arange(n), rng.integers(1, n))            # a derangement: every diagonal entry of P is zero
        dscale = 2.0 ** rng.integers(-6, 7, size=n)
        A = np.zeros((n, n)); A[np.arange(n), perm] = dscale         # A x = b  ->  x[perm[i]] = b[i] / d[i]
        Js.append((np.eye(n) - A) / 0.5)                              # gamma = 0.5: I - 0.5 J = A exactly (powers of two)
        b = rng.integers(-9, 10, size=n).astype(np.float64); bs.append(b)
        x = np.zeros(n); x[perm] = b / dscale; xs.append(x)
    jac, erow, gam, b = soa(Js, [0.5] * 8, bs)
    o = oracle.newton_solve(jac, erow, gam, b)
    assert np.array_equal(o["x"].T, np.array(xs)) and not o["info"].any()


def test_two_by_two_against_cramer_and_tiny_pivot():
    """N = 1 (one species + T).  The second system has |a11| = 1e-20 << |a21|: without partial pivoting x1 comes out as 0 or 2."""
    cases = [(np.array([[3.0, -2.0], [1.0, 4.0]]), np.array([1.0, 5.0])),
             (np.array([[1e-20, 1.0], [1.0, 1.0]]), np.array([1.0, 2.0])),
             (np.array([[-7.0, 0.5], [2.0, 1e3]]), np.array([0.25, -3.0]))]
    Js = [(np.eye(2) - A) / 0.25 for A, _ in cases]
    jac, erow, gam, b = soa(Js, [0.25] * 3, [r for _, r in cases])
    o = oracle.newton_solve(jac, erow, gam, b)
    for c, (A0, r) in enumerate(cases):
        A = np.eye(2) - 0.25 * Js[c]                                 # what the oracle sees (rounded once)
        det = A[0, 0] * A[1, 1] - A[0, 1] * A[1, 0]
        cram = np.array([r[0] * A[1, 1] - A[0, 1] * r[1], A[0, 0] * r[1] - r[0] * A[1, 0]]) / det
        assert np.allclose(o["x"][:, c], cram, rtol=1e-14, atol=0.0), (c, o["x"][:, c], cram)
    assert np.allclose(o["x"][:, 1], [1.0, 1.0], rtol=1e-15)


def test_integer_system_with_known_solution_catches_a_transposed_operand():
    """Small integers: A x* = b exactly representable; a non-symmetric A, so J^T or a swapped (row, column) index fails."""
    rng = np.random.default_rng(11); n = 9
    Js, bs, xs = [], [], []
    for _ in range(16):
        A = rng.integers(-4, 5, size=(n, n)).astype(np.float64) + np.diag(rng.integers(1, 4, size=n) * 8.0)
        xstar = rng.integers(-5, 6, size=n).astype(np.float64)
        Js.append(np.eye(n) - A); bs.append(A @ xstar); xs.append(xstar)        # gamma = 1
    jac, erow, gam, b = soa(Js, [1.0] * 16, bs)
    o = oracle.newton_solve(jac, erow, gam, b)
    assert np.allclose(o["x"].T, np.array(xs), rtol=0.0, atol=1e-12)
    Jt = [J.T.copy() for J in Js]
    jt, et, _, _ = soa(Jt, [1.0] * 16, bs)
    assert not np.allclose(oracle.newton_solve(jt, et, gam, b)["x"].T, np.array(xs), atol=1e-3)


@pytest.mark.parametrize("N,with_energy", [(8, True), (35, True), (35, False), (1, True), (40, True)])
def test_against_lapack_float128_and_backward_error(N, with_energy):
    m = 48
    d = newton_inputs(N, m, 100 + N, ld=m + 5, with_energy=with_energy)
    o = oracle.newton_solve(d["jac"], d["erow"], d["gamma"], d["b"], m)
    q = oracle.newton_solve(d["jac"], d["erow"], d["gamma"], d["b"], m, quad=True)
    cells = np.arange(m)
    A = gates.newton_matrix(d["jac"], d["erow"], d["gamma"], cells)
    b = d["b"][:, :m].T
    lap = np.stack([np.linalg.solve(A[c], b[c]) for c in cells])
    for ref in (lap, q["x"][:, :m].T):
        g = gates.newton_gates(A, b, o["x"][:, :m].T, ref)
        gates.assert_newton(g)
    assert gates.newton_gates(A, b, q["x"][:, :m].T)["eta_worst"] < 2e-16            # the float128 run is the better solution
    assert np.isnan(o["x"][:, m:]).all() or (o["x"][:, m:] == 0).all()                # padding untouched
    assert not o["info"].any()


def test_species_block_ignores_temperature_column_and_energy_row():
    d = newton_inputs(6, 10, 8)
    o = oracle.newton_solve(d["jac"], None, d["gamma"], np.ascontiguousarray(d["b"][:6]))
    for c in range(10):
        A = np.eye(6) - d["gamma"][c] * d["jac"][:, :6, c]
        assert np.allclose(o["x"][:, c], np.linalg.solve(A, d["b"][:6, c]), rtol=1e-10)


def test_exactly_singular_matrix_is_reported():
    J = np.eye(3) - np.array([[1.0, 2.0, 3.0], [2.0, 4.0, 6.0], [1.0, 0.0, 1.0]])     # rows 0 and 1 of A proportional
    jac, erow, gam, b = soa([J], [1.0], [np.array([1.0, 2.0, 3.0])])
    o = oracle.newton_solve(jac, erow, gam, b)
    assert o["info"][0] == 3                                            # zero pivot at the last step (k = 2)


@pytest.mark.parametrize("cfg", [1, 2])
def test_on_jacobians_of_the_synthetic_mechanisms(cfg):
    """The matrices the solve meets in the path: oracle Jacobian + energy row on config states, b = (wdot, Tdot)."""
    m = config_mechanism(cfg); n_cells = 24
    om = oracle.OracleMech(m)
    C, T = config_states(cfg, n_cells)
    ev = oracle.evaluate(om, C, T, n_cells); en = oracle.evaluate_energy(om, C, T, n_cells)
    jac = np.ascontiguousarray(ev["jac"]); erow = np.ascontiguousarray(en["erow"])
    b = np.ascontiguousarray(np.vstack([ev["wdot"], en["tdot"][None]]))
    Jmax = np.maximum(np.abs(jac).max((0, 1)), np.abs(erow).max(0))
    rng = np.random.default_rng(cfg)
    gamma = 10.0 ** rng.uniform(-2.0, 3.0, size=jac.shape[2]) / np.where(Jmax > 0, Jmax, 1.0)
    o = oracle.newton_solve(jac, erow, gamma, b, n_cells); q = oracle.newton_solve(jac, erow, gamma, b, n_cells, quad=True)
    cells = np.arange(n_cells)
    A = gates.newton_matrix(jac, erow, gamma, cells)
    g = gates.newton_gates(A, b[:, :n_cells].T, o["x"][:, :n_cells].T, q["x"][:, :n_cells].T)
    print("cfg%d Newton solve: worst backward error %.2e, well-conditioned %.2f, worst forward error there %.2e, error / bound %.2e"
          % (cfg, g["eta_worst"], g["wellcond_frac"], g["fwd_worst_wellcond"], g["fwd_worst_over_bound"]))
    gates.assert_newton(g, floor=0.0)
