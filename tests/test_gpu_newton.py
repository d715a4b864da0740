"""GPU parity of NEXT-2: the batched dense direct solve of the Newton system, qss_newton_solve
(Eq. 7; reading G20), against the CPU oracle (oracle/qss_newton_oracle.cpp: Gaussian
elimination with partial pivoting) on the same seeded inputs.  Gates: gates.newton_gates (backward error of every cell in
extended precision; forward agreement 1e-9 on the well-conditioned cells, cond-scaled bound on all)."""
import numpy as np
import pytest

import gates
import oracle
import qss_synth
from qss_synth import newton_inputs, newton_inputs_torch

pytestmark = pytest.mark.gpu

_MECH = {}


def _mech(cfg):
    import paper_2405_05974_b200 as qss
    if cfg not in _MECH:
        _MECH[cfg] = qss.QssMech(qss_synth.config_mechanism(cfg), 0)
    return _MECH[cfg]


def _solve(qm, d, n, inplace=False):
    import torch
    t = {k: (torch.from_numpy(v).cuda() if v is not None else None) for k, v in d.items()}
    nrow = d["b"].shape[0]
    if inplace:
        x = t["b"]
    else:
        x = torch.full((nrow, d["b"].shape[1]), float("nan"), dtype=torch.float64, device="cuda")
    qm.newton_solve(t["jac"], t["erow"], t["gamma"], t["b"], n, x=x)
    torch.cuda.synchronize()
    return x.cpu().numpy()


@pytest.mark.parametrize("cfg,n,with_energy", [(2, 1, True), (2, 3, True), (2, 4, True), (2, 5, True), (2, 33, True), (2, 1024 + 3, True),
                                               (2, 130, False), (1, 4096, True), (1, 257, False)])
def test_newton_solve_against_oracle(cfg, n, with_energy):
    """Jacobian-shaped synthetic matrices (qss_synth.newton), cell counts around the block size (4 cells) with ragged tails and
    a padded leading dimension; n = 36 (two register rows per lane), 35, 9, 8."""
    qm = _mech(cfg)
    d = newton_inputs(qm.N, n, seed=40 + n, ld=n + 6, with_energy=with_energy)
    x = _solve(qm, d, n)
    ref = oracle.newton_solve(d["jac"], d["erow"], d["gamma"], d["b"], n)
    assert np.isnan(x[:, n:]).all(), "padding was written"
    cells = np.arange(n) if n <= 512 else np.random.default_rng(0).choice(n, 512, replace=False)
    A = gates.newton_matrix(d["jac"], d["erow"], d["gamma"], cells)
    g = gates.newton_gates(A, d["b"][:, cells].T, x[:, cells].T, ref["x"][:, cells].T)
    print("cfg%d n=%d energy=%d: eta %.2e, well-conditioned %.2f, forward error there %.2e, error / bound %.2e"
          % (cfg, n, with_energy, g["eta_worst"], g["wellcond_frac"], g["fwd_worst_wellcond"], g["fwd_worst_over_bound"]))
    gates.assert_newton(g, floor=0.5 if n >= 33 else 0.0)
    # every cell against the oracle with the cond-free part of the gate: the solutions agree to 1e-6 normwise even on the worst cell
    err = np.abs(x[:, :n] - ref["x"][:, :n]).max(0) / np.abs(ref["x"][:, :n]).max(0)
    assert np.isfinite(x[:, :n]).all() and err.max() < 1e-6, err.max()


def test_in_place_and_zero_cells():
    qm = _mech(2)
    d = newton_inputs(qm.N, 77, seed=3)
    x0 = _solve(qm, d, 77)
    x1 = _solve(qm, d, 77, inplace=True)
    assert np.array_equal(x0, x1)
    import torch
    e = torch.empty((qm.N + 1, 0), dtype=torch.float64, device="cuda")
    qm.newton_solve(torch.empty((qm.N, qm.N + 1, 0), dtype=torch.float64, device="cuda"), e, torch.empty(0, dtype=torch.float64, device="cuda"), e, 0)


def test_scaled_permutations_are_solved_exactly():
    """I - gamma J = P D with a zero diagonal (powers of two): every step needs an interchange, rows 32..35 (the second register
    row of lanes 0..3) included; the result is exact."""
    qm = _mech(2)
    n = qm.N + 1; m = 64
    rng = np.random.default_rng(17)
    jac = np.zeros((qm.N, n, m)); erow = np.zeros((n, m)); b = np.zeros((n, m)); xs = np.zeros((n, m))
    for c in range(m):
        perm = np.roll(np.arange(n), rng.integers(1, n)) if c % 2 else rng.permutation(n)
        dsc = 2.0 ** rng.integers(-8, 9, size=n)
        A = np.zeros((n, n)); A[np.arange(n), perm] = dsc
        J = (np.eye(n) - A) / 0.5
        jac[:, :, c] = J[:qm.N]; erow[:, c] = J[qm.N]
        b[:, c] = rng.integers(-9, 10, size=n)
        xs[perm, c] = b[:, c] / dsc
    x = _solve(qm, dict(jac=jac, erow=erow, gamma=np.full(m, 0.5), b=b), m)
    assert np.array_equal(x, xs)


def test_gamma_zero_returns_b():
    qm = _mech(2)
    d = newton_inputs(qm.N, 40, seed=9)
    d["gamma"] = np.zeros_like(d["gamma"])
    assert np.array_equal(_solve(qm, d, 40), d["b"])


@pytest.mark.parametrize("cfg", [1, 2])
def test_on_jacobians_of_the_synthetic_mechanisms(cfg):
    """Matrices of the path itself: the ORACLE's Jacobian and energy row on config states (no input comes from the CUDA path),
    b = (wdot, Tdot), gamma * max|J| in [1e-2, 1e3]."""
    qm = _mech(cfg)
    m = qss_synth.config_mechanism(cfg); n = 96 + 3
    om = oracle.OracleMech(m)
    C, T = qss_synth.config_states(cfg, n)
    ev = oracle.evaluate(om, C, T, n); en = oracle.evaluate_energy(om, C, T, n)
    jac = np.ascontiguousarray(ev["jac"]); erow = np.ascontiguousarray(en["erow"])
    b = np.ascontiguousarray(np.vstack([ev["wdot"], en["tdot"][None]]))
    Jmax = np.maximum(np.abs(jac).max((0, 1)), np.abs(erow).max(0))
    gamma = 10.0 ** np.random.default_rng(cfg).uniform(-2.0, 3.0, size=jac.shape[2]) / np.where(Jmax > 0, Jmax, 1.0)
    d = dict(jac=jac, erow=erow, gamma=gamma, b=b)
    x = _solve(qm, d, n)
    ref = oracle.newton_solve(jac, erow, gamma, b, n, quad=True)
    cells = np.arange(n)
    g = gates.newton_gates(gates.newton_matrix(jac, erow, gamma, cells), b[:, :n].T, x[:, :n].T, ref["x"][:, :n].T)
    print("cfg%d path Jacobians: eta %.2e, well-conditioned %.2f, forward error there %.2e, error / bound %.2e"
          % (cfg, g["eta_worst"], g["wellcond_frac"], g["fwd_worst_wellcond"], g["fwd_worst_over_bound"]))
    gates.assert_newton(g, floor=0.0)


def test_full_size_residual_on_every_cell_and_sampled_cells_against_oracle():
    """BASELINE configs[1] size (2^20 cells, 36 x 36), the launch configuration bench.py times: inputs drawn on the device by
    torch's seeded generator; the backward error of EVERY cell with torch fp64 (a property that holds at any size), 256 sampled
    cells against the oracle."""
    import torch
    qm = _mech(2)
    n = 1 << 20
    d = newton_inputs_torch(qm.N, n, seed=2, device="cuda")
    x = qm.newton_solve(d["jac"], d["erow"], d["gamma"], d["b"], n)
    torch.cuda.synchronize()
    assert torch.isfinite(x).all()
    N = qm.N
    eta_max = 0.0
    for lo in range(0, n, 1 << 17):                                  # chunks: the residual needs a copy of the matrix
        sl = slice(lo, lo + (1 << 17))
        J = torch.cat([d["jac"][:, :, sl], d["erow"][None, :, sl]], 0)                    # [n, n, cells]
        A = -d["gamma"][sl][None, None] * J
        A[torch.arange(N + 1), torch.arange(N + 1)] += 1.0
        r = torch.einsum("ijc,jc->ic", A, x[:, sl]) - d["b"][:, sl]
        eta = r.abs().amax(0) / (A.abs().sum(1).amax(0) * x[:, sl].abs().amax(0) + d["b"][:, sl].abs().amax(0))
        eta_max = max(eta_max, float(eta.max()))
    print("full size: worst backward error (fp64 residual) %.2e" % eta_max)
    assert eta_max <= 1e-12                                          # the fp64 residual itself rounds at ~n eps; the sampled cells use extended precision
    cells = np.random.default_rng(1).choice(n, 256, replace=False)
    ct = torch.from_numpy(cells).cuda()
    sub = dict(jac=np.ascontiguousarray(d["jac"][:, :, ct].cpu().numpy()), erow=np.ascontiguousarray(d["erow"][:, ct].cpu().numpy()),
               gamma=np.ascontiguousarray(d["gamma"][ct].cpu().numpy()), b=np.ascontiguousarray(d["b"][:, ct].cpu().numpy()))
    ref = oracle.newton_solve(sub["jac"], sub["erow"], sub["gamma"], sub["b"])
    g = gates.newton_gates(gates.newton_matrix(sub["jac"], sub["erow"], sub["gamma"], np.arange(256)), sub["b"].T,
                           x[:, ct].cpu().numpy().T, ref["x"].T)
    gates.assert_newton(g)


def test_unsupported_matrix_order_fails_loudly():
    import torch
    import paper_2405_05974_b200 as qss
    qm = _mech(3)                                                    # 100 transported species
    t = torch.zeros((qm.N, qm.N + 1, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(qss.QssError) as e:
        qm.newton_solve(t, None, torch.ones(4, dtype=torch.float64, device="cuda"), torch.zeros((qm.N, 4), dtype=torch.float64, device="cuda"))
    assert e.value.code == -5
