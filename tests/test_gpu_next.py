"""GPU parity of the NEXT rows built so far: NEXT-1, the temperature right-hand side and the energy row of the
(N+1) x (N+1) Jacobian (qss_eval_energy; Eq. 7), and NEXT-3, the paper's simplified Jacobians
(qss_eval_jac_approx; constant-QSS AJ and zero-QSS AJ, L232), against the CPU oracle on the same seeded inputs."""
import numpy as np
import pytest

import gates
import oracle
import qss_synth
from qss_synth import make_states

pytestmark = pytest.mark.gpu


def _energy_gates(tdot, erow, ref, T, n, what):
    e, s = ref["erow"][:, :n], ref["escale"][:, :n]
    d = np.abs(erow[:, :n] - e)
    assert np.isfinite(erow[:, :n]).all() and np.isfinite(tdot[:n]).all(), what
    bound = 1e-9 * np.abs(e) + 1e-12 * s
    assert np.all(d <= bound), f"{what}: energy row, worst ratio {float(np.max(d / bound)):.3g}"
    # strict tier over the entries that are not cancellation residues, as for the species block (reading G16)
    well = s <= 1e3 * np.abs(e)
    assert well.mean() > 0.5 and (d[well] <= 1e-9 * np.abs(e[well])).mean() >= 0.99, what
    dt = np.abs(tdot[:n] - ref["tdot"][:n])
    assert np.all(dt <= 1e-10 * np.abs(ref["tdot"][:n]) + 1e-13 * s[-1] * T[:n]), f"{what}: tdot"


@pytest.mark.parametrize("name,n", [("cfg1", 4096), ("cfg2", 2048 + 19), ("cfg3", 192 + 5), ("toy_dag", 77), ("toy_nonqss", 33)])
def test_energy_row_and_temperature_rhs(name, n):
    import torch
    import paper_2405_05974_b200 as qss
    if name.startswith("cfg"):
        mech = qss_synth.config_mechanism(int(name[3])); C, T = qss_synth.config_states(int(name[3]), n)
    else:
        mech = getattr(qss_synth, name)(); C, T = make_states(mech.n_nqss, n, seed=5)
    ld = C.shape[1]
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J, w = qm.eval_jac(Cd, Td, n, want_wdot=True)
    tdot = torch.full((ld,), float("nan"), dtype=torch.float64, device="cuda")
    erow = torch.full((qm.N + 1, ld), float("nan"), dtype=torch.float64, device="cuda")
    qm.eval_energy(Cd, Td, w, J, n, tdot=tdot, erow=erow)
    torch.cuda.synchronize()
    ref = oracle.evaluate_energy(oracle.OracleMech(mech), C, T, n)
    _energy_gates(tdot.cpu().numpy(), erow.cpu().numpy(), ref, T, n, name)
    if ld > n:
        assert torch.isnan(tdot[n:]).all() and torch.isnan(erow[:, n:]).all(), "padding was written"
    qm.close()


@pytest.mark.parametrize("name,n", [("cfg1", 1024 + 3), ("cfg2", 512 + 7), ("toy_dag", 77), ("toy3", 40)])
@pytest.mark.parametrize("mode", [1, 2])
def test_simplified_jacobians(name, n, mode):
    """Constant-QSS AJ (mode 1) and zero-QSS AJ (mode 2) against the oracle's modes of the same definition; mode 0 through the same
    entry point is the exact Jacobian bit for bit."""
    import torch
    import paper_2405_05974_b200 as qss
    if name.startswith("cfg"):
        mech = qss_synth.config_mechanism(int(name[3])); C, T = qss_synth.config_states(int(name[3]), n)
    else:
        mech = getattr(qss_synth, name)(); C, T = make_states(mech.n_nqss, n, seed=5)
    qm = qss.QssMech(mech, 0)
    assert qm.info.kernel_variant_jac == 3
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    Ja = qm.eval_jac_approx(Cd, Td, mode, n).cpu().numpy()
    J0 = qm.eval_jac_approx(Cd, Td, 0, n)
    assert torch.equal(J0[:, :, :n], qm.eval_jac(Cd, Td, n)[:, :, :n])
    om = oracle.OracleMech(mech)
    ref = oracle.evaluate(om, C, T, n, mode=oracle.JAC_CONST_QSS if mode == 1 else oracle.JAC_ZERO_QSS, want_scale=True)
    gates.assert_jac(Ja, ref["jac"], ref["jscale"], n, f"{name} simplified Jacobian mode {mode}")
    qm.close()


def test_simplified_jacobians_need_variant_3():
    import torch
    import paper_2405_05974_b200 as qss
    mech = qss_synth.config_mechanism(3)
    qm = qss.QssMech(mech, 0)
    C, T = qss_synth.config_states(3, 64)
    with pytest.raises(qss.QssError) as e:
        qm.eval_jac_approx(torch.from_numpy(C).cuda(), torch.from_numpy(T).cuda(), 1, 64)
    assert e.value.code == -5
    qm.close()


@pytest.mark.parametrize("name,n", [("cfg1", 1024 + 2), ("cfg2", 512 + 6), ("cfg3", 96)])
def test_finite_difference_temperature_column(name, n):
    """NEXT-3 (reading G22): qss_eval_jac_fdt against oracle.evaluate_fdT.  The species columns are the exact
    kernel's (bit for bit); the T column is a difference of two wdot evaluations, so its gate is the wdot gate of both, divided
    by the step: |d col| <= (tol(w+) + tol(w-)) / (T+ - T-), tol(w) = 1e-10 |w| + 1e-13 S."""
    import torch
    import paper_2405_05974_b200 as qss
    cfg = int(name[3])
    mech = qss_synth.config_mechanism(cfg); C, T = qss_synth.config_states(cfg, n)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J, w = qm.eval_jac_fdT(Cd, Td, n, want_wdot=True)
    Jex = qm.eval_jac(Cd, Td, n)
    torch.cuda.synchronize()
    J = J.cpu().numpy(); Jex = Jex.cpu().numpy()
    N = qm.N
    assert np.array_equal(J[:, :N, :n], Jex[:, :N, :n])
    ref = oracle.evaluate_fdT(oracle.OracleMech(mech), C, T, n)
    h = (ref["Tp"] - ref["Tm"])[:n]
    S = ref["S"][:, :n]
    bound = (1e-10 * (np.abs(ref["wdot_p"][:, :n]) + np.abs(ref["wdot_m"][:, :n])) + 2.02e-13 * S) / h
    d = np.abs(J[:, N, :n] - ref["jac"][:, N, :n])
    assert np.isfinite(J[:, N, :n]).all()
    print("%s FD-in-T column: worst |d| / bound %.3g" % (name, float((d / bound).max())))
    assert (d <= bound).all()
    g = gates.wdot_gates(w.cpu().numpy(), ref["wdot"], ref["S"], n)
    assert g["finite"] and g["tier2_all"]
    qm.close()


@pytest.mark.parametrize("name,n", [("cfg1", 512 + 3), ("toy3", 70), ("cfg2", 256)])
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_sparsity_pattern_and_packed_output(name, n, mode):
    """NEXT-3 (Table 4): outside the structural pattern the kernel's Jacobian is exactly 0.0; qss_jac_pack gathers the
    pattern's rows bit for bit (the dense output stays the reference, which is gated against the oracle elsewhere)."""
    import torch
    import paper_2405_05974_b200 as qss
    mech = qss_synth.config_mechanism(int(name[3])) if name.startswith("cfg") else getattr(qss_synth, name)()
    if name.startswith("cfg"):
        C, T = qss_synth.config_states(int(name[3]), n)
    else:
        C, T = make_states(mech.n_nqss, n, seed=5)
    qm = qss.QssMech(mech, 0)
    if mode and qm.info.kernel_variant_jac != 3:
        pytest.skip("simplified Jacobians need kernel variant 3")
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J = qm.eval_jac_approx(Cd, Td, mode, n)
    pat = qss.jac_pattern(mech, mode).astype(bool)
    Jh = J.cpu().numpy()
    assert (Jh[:, :, :n][~pat] == 0.0).all()
    idx = torch.from_numpy(np.flatnonzero(pat.ravel()).astype(np.int32)).cuda()
    ld = C.shape[1]
    packed = torch.full((idx.numel(), ld), float("nan"), dtype=torch.float64, device="cuda")
    qm.jac_pack(J, idx, n, packed=packed)
    torch.cuda.synchronize()
    ph = packed.cpu().numpy()
    assert np.array_equal(ph[:, :n], Jh.reshape(-1, ld)[np.flatnonzero(pat.ravel())][:, :n])
    assert np.isnan(ph[:, n + (n & 1):]).all()                           # (16-byte stores: at most one padding cell behind an odd count is written)
    qm.close()


def test_parsed_mechanism_runs_on_the_kernels():
    """NEXT-4, second half: CHEMKIN-format text -> frontend.parse_chemkin -> linearisation -> qss_mech_create -> the Jacobian kernel,
    against the oracle on the same description (third-body, fall-off with a three-parameter Troe line, an irreversible reaction,
    duplicates)."""
    import torch
    import paper_2405_05974_b200 as qss
    from paper_2405_05974_b200 import frontend as fe
    from test_frontend import TEXT
    d = fe.linearise(fe.parse_chemkin(TEXT, qss=["A", "B", "AB2"]), "reaction")
    n = 200
    rng = np.random.default_rng(2)
    C = np.ascontiguousarray(10.0 ** rng.uniform(-4.0, 1.0, size=(d.n_nqss, n))); T = rng.uniform(700.0, 2400.0, size=n)
    qm = qss.QssMech(d, 0, strict_balance=True)
    J, w = qm.eval_jac(torch.from_numpy(C).cuda(), torch.from_numpy(T).cuda(), n, want_wdot=True)
    torch.cuda.synchronize()
    ref = oracle.evaluate(oracle.OracleMech(d), C, T, n, want_scale=True)
    gw = gates.wdot_gates(w.cpu().numpy(), ref["wdot"], ref["S"], n)
    gj = gates.jac_gates(J.cpu().numpy(), ref["jac"], ref["jscale"], n)
    print("parsed mechanism: kernel variant %d; wdot tier 1 %.3f, tier 2 worst %.3g; Jacobian tier 2 %s" % (qm.info.kernel_variant_jac, gw["tier1_frac"], gw["tier2_worst"], gj.get("cell_tier2_all")))
    assert gw["finite"] and gw["tier2_all"] and gw["tier1_frac"] >= 0.99
    assert gj["finite"] and all(v for k, v in gj.items() if k.endswith("tier2_all"))
    qm.close()


def test_parsed_mechanism_with_per_species_mid_temperatures():
    """The syntax and the thermodynamic data of real mechanism files (test_frontend.TEXT2: every species its own Tmid, three-parameter
    Troe line, duplicates, irreversible steps) through the generated kernel: the range-interval sets of -ln Kc (qss_gen3.cpp)."""
    import torch
    import paper_2405_05974_b200 as qss
    from paper_2405_05974_b200 import frontend as fe
    from test_frontend import TEXT2
    d = fe.linearise(fe.parse_chemkin(TEXT2, qss=["CH2(S)", "O"]), "reaction")
    n = 300
    rng = np.random.default_rng(4)
    C = np.ascontiguousarray(10.0 ** rng.uniform(-4.0, 1.0, size=(d.n_nqss, n)))
    T = rng.uniform(900.0, 1500.0, size=n)                  # mostly BETWEEN the species' breakpoints (1000 .. 1392 K)
    T[:8] = sorted(set(d.nasa_T[:, 1]))[:8]                 # and exactly on some of them
    qm = qss.QssMech(d, 0)
    assert qm.info.kernel_variant_jac == 3
    J, w = qm.eval_jac(torch.from_numpy(C).cuda(), torch.from_numpy(T).cuda(), n, want_wdot=True)
    torch.cuda.synchronize()
    ref = oracle.evaluate(oracle.OracleMech(d), C, T, n, want_scale=True)
    gw = gates.wdot_gates(w.cpu().numpy(), ref["wdot"], ref["S"], n)
    gj = gates.jac_gates(J.cpu().numpy(), ref["jac"], ref["jscale"], n)
    print("parsed mechanism, per-species Tmid: wdot tier 1 %.3f, tier 2 worst %.3g; Jacobian cell tier 1 %.3f" % (gw["tier1_frac"], gw["tier2_worst"], gj["cell_tier1_frac"]))
    assert gw["finite"] and gw["tier2_all"] and gw["tier1_frac"] >= 0.99
    assert gj["finite"] and gj["cell_tier2_all"] and gj["col_tier2_all"] and gj["cell_tier1_frac"] >= 0.99
    qm.close()


@pytest.mark.parametrize("name,n", [("cfg1", 4096), ("cfg2", 2048 + 19), ("toy_dag", 77), ("cfg3", 96 + 5)])
def test_full_jacobian_in_one_call(name, n):
    """qss_eval_jac_full: jac and wdot bit for bit those of qss_eval_jac; tdot and the energy row against the oracle with the gates
    of qss_eval_energy."""
    import torch
    import paper_2405_05974_b200 as qss
    if name.startswith("cfg"):
        mech = qss_synth.config_mechanism(int(name[3])); C, T = qss_synth.config_states(int(name[3]), n)
    else:
        mech = getattr(qss_synth, name)(); C, T = make_states(mech.n_nqss, n, seed=5)
    ld = C.shape[1]
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J0, w0 = qm.eval_jac(Cd, Td, n, want_wdot=True)
    tdot = torch.full((ld,), float("nan"), dtype=torch.float64, device="cuda")
    erow = torch.full((qm.N + 1, ld), float("nan"), dtype=torch.float64, device="cuda")
    J, w, _, _ = qm.eval_jac_full(Cd, Td, n, tdot=tdot, erow=erow)
    torch.cuda.synchronize()
    assert torch.equal(J[:, :, :n], J0[:, :, :n]) and torch.equal(w[:, :n], w0[:, :n])
    ref = oracle.evaluate_energy(oracle.OracleMech(mech), C, T, n)
    _energy_gates(tdot.cpu().numpy(), erow.cpu().numpy(), ref, T, n, name + " (one call)")
    if ld > n:
        assert torch.isnan(tdot[n:]).all() and torch.isnan(erow[:, n:]).all(), "padding was written"
    qm.close()


@pytest.mark.parametrize("cfg,n", [(2, 1000 + 7), (1, 4096), (2, 1), (3, 37)])
def test_aos_export_for_external_batched_solvers(cfg, n):
    """qss_jac_to_aos is an index permutation: bit for bit the numpy transpose of the SoA arrays, row-major and column-major, with
    and without the energy row; padding cells are not read into the output; the row-major matrices solve like qss_newton_solve's
    (torch.linalg.solve on I - gamma J of a few cells, a LIBRARY routine standing in for the external solver)."""
    import torch
    import paper_2405_05974_b200 as qss
    mech = qss_synth.config_mechanism(cfg)
    N = mech.n_nqss
    rng = np.random.default_rng(cfg + n)
    ld = n + 9
    jac = np.full((N, N + 1, ld), np.nan); erow = np.full((N + 1, ld), np.nan)
    jac[:, :, :n] = rng.normal(size=(N, N + 1, n)); erow[:, :n] = rng.normal(size=(N + 1, n))
    qm = qss.QssMech(mech, 0)
    Jd = torch.from_numpy(jac).cuda(); Ed = torch.from_numpy(erow).cuda()
    full = np.concatenate([jac, erow[None]], 0)                                    # [N+1, N+1, ld]
    for with_e in (True, False):
        src = full if with_e else jac
        for cm in (False, True):
            out = qm.jac_to_aos(Jd, Ed if with_e else None, n, col_major=cm).cpu().numpy()
            want = np.transpose(src[:, :, :n], (2, 1, 0) if cm else (2, 0, 1))
            assert out.shape == want.shape and np.array_equal(out, want), (with_e, cm)
    if N + 1 <= 40 and n >= 4:
        gamma = np.full(ld, 1e-2); b = rng.normal(size=(N + 1, ld))
        x = qm.newton_solve(Jd, Ed, torch.from_numpy(gamma).cuda(), torch.from_numpy(b).cuda(), n).cpu().numpy()
        A = torch.eye(N + 1, dtype=torch.float64, device="cuda")[None] - 1e-2 * qm.jac_to_aos(Jd, Ed, n)[:4]
        xs = torch.linalg.solve(A, torch.from_numpy(np.ascontiguousarray(b[:, :4].T)).cuda()).cpu().numpy()
        assert np.allclose(xs, x[:, :4].T, rtol=1e-9, atol=1e-12)
    qm.close()


@pytest.mark.parametrize("cfg,n", [(2, 2048 + 19), (1, 4096), (2, 31)])
def test_mapping_microbenchmark_species_sums(cfg, n):
    """qss_bench_species_sums (north_star subsystem 3): both mappings give wdot = S Q; reference: the dense net stoichiometric
    matrix assembled in numpy from the mechanism description."""
    import torch
    import paper_2405_05974_b200 as qss
    mech = qss_synth.config_mechanism(cfg)
    N, M = mech.n_nqss, mech.n_reac
    S = np.zeros((N, M))
    for j in range(M):
        for t in range(mech.reac_ptr[j], mech.reac_ptr[j + 1]):
            if mech.reac_sp[t] < N:
                S[mech.reac_sp[t], j] -= mech.reac_nu[t]
        for t in range(mech.prod_ptr[j], mech.prod_ptr[j + 1]):
            if mech.prod_sp[t] < N:
                S[mech.prod_sp[t], j] += mech.prod_nu[t]
    rng = np.random.default_rng(cfg)
    ld = n + 5
    Q = np.full((M, ld), np.nan); Q[:, :n] = rng.normal(size=(M, n)) * 10.0 ** rng.uniform(-3, 3, size=(M, n))
    ref = S @ Q[:, :n]
    scale = np.abs(S) @ np.abs(Q[:, :n])
    qm = qss.QssMech(mech, 0)
    Qd = torch.from_numpy(Q).cuda()
    out = []
    for mode in (0, 1):
        w = torch.full((N, ld), float("nan"), dtype=torch.float64, device="cuda")
        qm.bench_species_sums(mode, Qd, n, wdot=w)
        torch.cuda.synchronize()
        wh = w.cpu().numpy()
        assert np.isnan(wh[:, n:]).all(), "padding was written"
        assert np.all(np.abs(wh[:, :n] - ref) <= 1e-13 * scale + 1e-300), (mode, float(np.max(np.abs(wh[:, :n] - ref) / (scale + 1e-300))))
        out.append(wh[:, :n])
    assert np.allclose(out[0], out[1], rtol=0.0, atol=1e-13 * scale.max())
    qm.close()


def test_full_size_cfg2_padded_leading_dimension_full_jacobian_sampled():
    """BASELINE.json configs[1] at full size in the layout bench.py times (leading dimension = 2^20 + 64): qss_eval_jac_full; 128
    sampled cells against the oracle (species block, wdot, energy row, Tdot); the 64 padding cells of every row stay untouched."""
    import torch
    import paper_2405_05974_b200 as qss
    mech = qss_synth.config_mechanism(2)
    C0, T0 = qss_synth.config_states(2)
    n = qss_synth.CONFIGS[2]["n_cells"]; ld = n + 64
    C = np.empty((C0.shape[0], ld)); T = np.empty(ld)
    C[:, :n] = C0[:, :n]; T[:n] = T0[:n]; C[:, n:] = C0[:, :1]; T[n:] = T0[0]
    qm = qss.QssMech(mech, 0)
    N = qm.N
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    f64 = dict(dtype=torch.float64, device="cuda")
    J = torch.empty((N, N + 1, ld), **f64); w = torch.empty((N, ld), **f64); td = torch.empty((ld,), **f64); er = torch.empty((N + 1, ld), **f64)
    for a in (J, w, td, er):
        a[..., n:] = float("nan")
    qm.eval_jac_full(Cd, Td, n, jac=J, wdot=w, tdot=td, erow=er)
    torch.cuda.synchronize()
    assert torch.isfinite(J[:, :, :n]).all() and torch.isfinite(w[:, :n]).all() and torch.isfinite(er[:, :n]).all() and torch.isfinite(td[:n]).all()
    assert torch.isnan(J[:, :, n:]).all() and torch.isnan(w[:, n:]).all() and torch.isnan(er[:, n:]).all() and torch.isnan(td[n:]).all()
    idx = np.sort(np.random.default_rng(7).choice(n, size=128, replace=False)); idx[0], idx[-1] = 0, n - 1
    it = torch.from_numpy(idx).cuda()
    Cs = np.ascontiguousarray(C[:, idx]); Ts = np.ascontiguousarray(T[idx])
    om = oracle.OracleMech(mech)
    ref = oracle.evaluate(om, Cs, Ts, want_jac=True, want_scale=True)
    gates.assert_wdot(w[:, it].cpu().numpy(), ref["wdot"], ref["S"], what="cfg2 full (padded ld) wdot", cfg=2)
    gates.assert_jac(J[:, :, it].cpu().numpy(), ref["jac"], ref["jscale"], what="cfg2 full (padded ld) jac", cfg=2)
    _energy_gates(td[it].cpu().numpy(), er[:, it].cpu().numpy(), oracle.evaluate_energy(om, Cs, Ts), Ts, 128, "cfg2 full (padded ld)")
    qm.close()
