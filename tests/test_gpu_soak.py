"""GPU parity on RANDOM mechanisms: shapes the five BASELINE configs and the toys do not cover (no QSS species at all, one QSS
species, many small or few large groups, more reactions per species or fewer, 6..47 transported species, species with their own
NASA-7 mid temperature on every other case), each on whatever kernel variant the library selects by itself.

Gates (tests/gates.py): tier 2 for every entry / cell / column; tier 1 as on the configs, except that on an arbitrary mechanism a
cell's Jacobian can be a cancellation residue as a whole (the per-cell tier has no conditioning filter), so where the kernel's strict
fraction is below 0.99 it must not be below what the fp64 ORACLE achieves against its own float128 evaluation on the same cells
(reading G16: the bar is what fp64 can deliver, measured, not assumed)."""
import dataclasses

import numpy as np
import pytest

import gates
import oracle
from qss_synth import make_states, mechanism

pytestmark = pytest.mark.gpu


def _case(it):
    rng = np.random.default_rng(1000 + it)
    N = int(rng.integers(6, 48)); Nq = int(rng.integers(0, 22)); M = int(rng.integers(max(10, N), 6 * (N + Nq))); gmax = int(rng.integers(1, 6))
    try:
        mech = mechanism.make_mechanism(N, Nq, M, gmax, True, 500 + it)
    except RuntimeError:
        return None                                       # the generator cannot build every shape (too few balanced candidates)
    if it % 2:
        nasa_T = mech.nasa_T.copy()
        nasa_T[:, 1] = np.where(rng.uniform(size=nasa_T.shape[0]) < 0.4, 1000.0, rng.uniform(950.0, 1450.0, size=nasa_T.shape[0]))
        mech = dataclasses.replace(mech, nasa_T=nasa_T)
    n = int(rng.integers(1, 300))
    C, T = make_states(mech.n_nqss, n, seed=it)
    return mech, C, T, n


@pytest.mark.parametrize("it", list(range(0, 5)) + [6] + list(range(11, 17)) + [28, 29, 31, 34])
def test_random_mechanism(it):
    import torch
    import paper_2405_05974_b200 as qss
    case = _case(it)
    assert case is not None
    mech, C, T, n = case
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J, w = qm.eval_jac(Cd, Td, n, want_wdot=True)
    w2, y = qm.eval_wdot(Cd, Td, n, want_cqss=True)
    torch.cuda.synchronize()
    variants = (qm.info.kernel_variant_wdot, qm.info.kernel_variant_jac)
    qm.close()
    om = oracle.OracleMech(mech)
    ref = oracle.evaluate(om, C, T, n, want_jac=True, want_scale=True)
    gw = gates.wdot_gates(w.cpu().numpy(), ref["wdot"], ref["S"], n)
    gw2 = gates.wdot_gates(w2.cpu().numpy(), ref["wdot"], ref["S"], n)
    gj = gates.jac_gates(J.cpu().numpy(), ref["jac"], ref["jscale"], n)
    what = f"random mechanism {it}: N {mech.n_nqss} Nq {mech.n_qss} M {mech.n_reac} n {n} variants {variants}"
    print(what, "wdot tier 1 %.3f" % gw["tier1_frac"], "J cell tier 1 %.3f col tier 1 %.3f" % (gj["cell_tier1_frac"], gj["col_tier1_frac"]))
    for g in (gw, gw2):
        assert g["finite"] and g["tier2_all"], (what, g)
    assert gj["finite"] and gj["cell_tier2_all"] and gj["col_tier2_all"], (what, gj)
    if mech.n_qss:
        yy, yr = y.cpu().numpy()[:, :n], ref["cqss"][:, :n]
        assert np.isfinite(yy).all() and np.max(np.abs(yy - yr) / np.abs(yr)) < 1e-9, what
    strict = {"wdot": min(gw["tier1_frac"], gw2["tier1_frac"]), "cell": gj["cell_tier1_frac"], "col": gj["col_tier1_frac"]}
    if min(strict.values()) < gates.TIER1_MIN_FRACTION:
        q = oracle.evaluate(om, C, T, n, want_jac=True, want_scale=True, mode=oracle.EXPLICIT_F128)
        ow = gates.wdot_gates(ref["wdot"], q["wdot"], q["S"], n)
        oj = gates.jac_gates(ref["jac"], q["jac"], q["jscale"], n)
        floor = {"wdot": ow["tier1_frac"], "cell": oj["cell_tier1_frac"], "col": oj["col_tier1_frac"]}
        print(what, "strict fractions", strict, "fp64 oracle against float128", floor)
        for k in strict:
            assert strict[k] >= min(gates.TIER1_MIN_FRACTION, floor[k] - 0.03), (what, k, strict, floor)


@pytest.mark.parametrize("it", [0, 1, 2, 4, 12, 13, 16, 28, 31])
def test_random_mechanism_full_jacobian_and_newton_solve(it):
    """The same random mechanisms through qss_eval_jac_full (energy row, temperature right-hand side: gates of test_gpu_next) and
    qss_newton_solve on Jacobian-shaped synthetic systems of their order (n = N + 1 = 13 .. 38: one and two register rows per lane,
    n = 32 / 33 at the boundary; order 44: refused with QSS_E_UNSUPPORTED; gates of test_gpu_newton)."""
    import torch
    import paper_2405_05974_b200 as qss
    from qss_synth import newton_inputs
    from test_gpu_next import _energy_gates
    mech, C, T, n = _case(it)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J0, w0 = qm.eval_jac(Cd, Td, n, want_wdot=True)
    J, w, tdot, erow = qm.eval_jac_full(Cd, Td, n)
    torch.cuda.synchronize()
    assert torch.equal(J[:, :, :n], J0[:, :, :n]) and torch.equal(w[:, :n], w0[:, :n])
    om = oracle.OracleMech(mech)
    ref = oracle.evaluate_energy(om, C, T, n)
    try:
        _energy_gates(tdot.cpu().numpy(), erow.cpu().numpy(), ref, T, n, f"random mechanism {it}")
    except AssertionError:
        # The element-wise guard of that gate scales with the cancellation INSIDE the energy-row sum (escale), not with the
        # cancellation inside the Jacobian entries it sums; on an arbitrary mechanism the fp64 oracle itself can miss it against
        # its float128 evaluation.  Then the kernel has to stay within 4x of what the fp64 oracle achieves (G16's principle).
        q = oracle.evaluate_energy(om, C, T, n, mode=oracle.EXPLICIT_F128)
        e, sc = q["erow"][:, :n], q["escale"][:, :n]
        bound = 1e-9 * np.abs(e) + 1e-12 * sc
        r_oracle = float(np.max(np.abs(ref["erow"][:, :n] - e) / bound))
        r_kernel = float(np.max(np.abs(erow.cpu().numpy()[:, :n] - ref["erow"][:, :n]) / (1e-9 * np.abs(ref["erow"][:, :n]) + 1e-12 * ref["escale"][:, :n])))
        print(f"random mechanism {it}: energy row, worst ratio kernel/oracle {r_kernel:.3g}, fp64 oracle/float128 {r_oracle:.3g}")
        assert r_oracle > 0.25 and r_kernel <= 4.0 * r_oracle, (it, r_kernel, r_oracle)
        dt = np.abs(tdot.cpu().numpy()[:n] - ref["tdot"][:n])
        assert np.all(dt <= 1e-10 * np.abs(ref["tdot"][:n]) + 1e-13 * ref["escale"][-1, :n] * T[:n]), f"random mechanism {it}: tdot"
    m = 131
    d = newton_inputs(qm.N, m, seed=90 + it, ld=m + 5, with_energy=True)
    t = {k: torch.from_numpy(v).cuda() for k, v in d.items()}
    x = torch.full((qm.N + 1, m + 5), float("nan"), dtype=torch.float64, device="cuda")
    if qm.N + 1 > 40:                                     # include/qss.h: the solve holds the matrix in a warp's registers, order <= 40
        with pytest.raises(qss.QssError) as ei:
            qm.newton_solve(t["jac"], t["erow"], t["gamma"], t["b"], m, x=x)
        assert ei.value.code == -5
        qm.close()
        return
    qm.newton_solve(t["jac"], t["erow"], t["gamma"], t["b"], m, x=x)
    torch.cuda.synchronize()
    qm.close()
    x = x.cpu().numpy()
    refx = oracle.newton_solve(d["jac"], d["erow"], d["gamma"], d["b"], m)
    assert np.isnan(x[:, m:]).all(), "padding was written"
    cells = np.arange(m)
    g = gates.newton_gates(gates.newton_matrix(d["jac"], d["erow"], d["gamma"], cells), d["b"][:, cells].T, x[:, cells].T, refx["x"][:, cells].T)
    print("random mechanism %d, order %d: eta %.2e, well-conditioned %.2f, forward error there %.2e" % (it, qm.N + 1, g["eta_worst"], g["wellcond_frac"], g["fwd_worst_wellcond"]))
    gates.assert_newton(g, floor=0.0)


@pytest.mark.parametrize("it", [6, 13, 29])
def test_random_mechanism_many_slabs_per_block(it):
    """20011 cells: every persistent block runs four or five slabs, so the staging of the next slab's inputs under the sweep and the
    reuse of the shared-memory rows and of the scratch slab are exercised on mechanisms whose row layout differs from the configs'."""
    import torch
    import paper_2405_05974_b200 as qss
    mech = _case(it)[0]
    n = 20011
    C, T = make_states(mech.n_nqss, n, seed=100 + it)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J, w = qm.eval_jac(Cd, Td, n, want_wdot=True)
    w2, _ = qm.eval_wdot(Cd, Td, n, want_cqss=True)
    torch.cuda.synchronize()
    qm.close()
    ref = oracle.evaluate(oracle.OracleMech(mech), C, T, n, want_jac=True, want_scale=True)
    for g in (gates.wdot_gates(w.cpu().numpy(), ref["wdot"], ref["S"], n), gates.wdot_gates(w2.cpu().numpy(), ref["wdot"], ref["S"], n)):
        assert g["finite"] and g["tier2_all"] and g["tier1_frac"] >= gates.TIER1_MIN_FRACTION, (it, g)
    gj = gates.jac_gates(J.cpu().numpy(), ref["jac"], ref["jscale"], n)
    assert gj["finite"] and gj["cell_tier2_all"] and gj["col_tier2_all"] and gj["col_tier1_frac"] >= gates.TIER1_MIN_FRACTION, (it, gj)
    assert gj["cell_tier1_frac"] >= 0.95, (it, gj)          # (0.966 on mechanism 29, the fp64 oracle's own fraction against float128: see above)


@pytest.mark.parametrize("it", [2, 13, 28])
def test_random_mechanism_adaptive_integrator(it):
    """qss_ignition_advance on random mechanisms of order 32, 13 and 31 (the comparison of test_gpu_bdf1: accept / reject decisions,
    times and step sizes bit for bit, ignition times, states; cells within 1e-6 of the acceptance threshold are left out)."""
    import torch
    import paper_2405_05974_b200 as qss
    from test_gpu_bdf1 import _dt
    mech, C, T, n = _case(it)
    n = min(n, 80); attempts, iters, rtol, dT_ign = 8, 3, 1e-6, 0.05
    om = oracle.OracleMech(mech)
    ld = C.shape[1]
    dt0 = _dt(om, C, T, n, 30.0, 3)
    t_end = float(np.median(dt0[:n]) * 6.0)
    trace = []
    ref = oracle.ignition_advance(om, C, T, dt0, np.zeros(ld), t_end, attempts, iters, n, rtol=rtol, dT_ign=dT_ign, trace=trace)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda(); T0d = Td.clone()
    dtd = torch.from_numpy(dt0).cuda(); td = torch.zeros(ld, dtype=torch.float64, device="cuda")
    tig = torch.full((ld,), float("nan"), dtype=torch.float64, device="cuda")
    qm.ignition_advance(Cd, Td, dtd, td, t_end, attempts, iters, n, t_ign=tig, T0=T0d, dT_ign=dT_ign, rtol=rtol)
    torch.cuda.synchronize()
    qm.close()
    Cg, Tg, dtg, tg, tigg = (x.cpu().numpy() for x in (Cd, Td, dtd, td, tig))
    sure = ~(np.abs(np.array(trace) - 1.0) <= 1e-6).any(0) & np.isfinite(ref["T"][:n])
    assert sure.mean() >= 0.9 and int((attempts - ref["accepted"][:n][sure]).sum()) > 0
    assert np.array_equal(tg[:n][sure], ref["t"][:n][sure]) and np.array_equal(dtg[:n][sure], ref["dt"][:n][sure])
    assert np.array_equal(tigg[:n][sure], ref["t_ign"][:n][sure], equal_nan=True)
    eC = (np.abs(Cg[:, :n] - ref["C"][:, :n]).max(0) / np.abs(ref["C"][:, :n]).max(0))[sure]
    eT = (np.abs(Tg[:n] - ref["T"][:n]) / ref["T"][:n])[sure]
    assert eC.max() <= 1e-8 and eT.max() <= 1e-10, (eC.max(), eT.max())


@pytest.mark.parametrize("it", [0, 4, 13, 34])
def test_random_mechanism_cheap_jacobians_pattern_and_fixed_step_integrator(it):
    """The remaining entry points on random mechanisms: constant-QSS and zero-QSS Jacobians against the oracle's (tier 2), entries
    outside the structural pattern exactly zero, qss_bdf1_advance against the oracle's integrator (tolerances of test_gpu_bdf1)."""
    import torch
    import paper_2405_05974_b200 as qss
    from test_gpu_bdf1 import _dt
    mech, C, T, n = _case(it)
    n = min(n, 96)
    om = oracle.OracleMech(mech)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    for mode, omode in ((1, oracle.JAC_CONST_QSS), (2, oracle.JAC_ZERO_QSS)):
        J = qm.eval_jac_approx(Cd, Td, mode, n)
        J = J[0] if isinstance(J, tuple) else J
        ref = oracle.evaluate(om, C, T, n, want_jac=True, want_scale=True, mode=omode)
        g = gates.jac_gates(J.cpu().numpy(), ref["jac"], ref["jscale"], n)
        assert g["finite"] and g["cell_tier2_all"] and g["col_tier2_all"], (it, mode, g)
    pat = qss.jac_pattern(mech, 0)
    J = qm.eval_jac(Cd, Td, n).cpu().numpy()[:, :, :n]
    assert not (pat == 0).any() or np.abs(J[pat == 0]).max() == 0.0
    dt = _dt(om, C, T, n, 2.0, 3)
    Cr, Tr = oracle.bdf1_advance(om, C, T, dt, 2, 3, n)
    C2 = torch.from_numpy(C).cuda(); T2 = torch.from_numpy(T).cuda()
    qm.bdf1_advance(C2, T2, torch.from_numpy(dt).cuda(), 2, 3, n)
    torch.cuda.synchronize()
    qm.close()
    Cg, Tg = C2.cpu().numpy(), T2.cpu().numpy()
    ok = np.isfinite(Tr[:n]) & np.isfinite(Cr[:, :n]).all(0)
    assert ok.mean() >= 0.9 and not np.isfinite(Tg[:n][~ok]).any()
    eC = (np.abs(Cg[:, :n] - Cr[:, :n]).max(0) / np.abs(Cr[:, :n]).max(0))[ok]
    eT = (np.abs(Tg[:n] - Tr[:n]) / Tr[:n])[ok]
    assert eC.max() <= 1e-8 and eT.max() <= 1e-10, (it, eC.max(), eT.max())
