"""GPU parity: libqss (CUDA, through the C-ABI binding) against the CPU oracle, element by element on the
same seeded inputs.  Gates: tests/gates.py (wdot relative 1e-10, Jacobian normwise
relative 1e-9 per cell and per column, two tiers)."""
import numpy as np
import pytest

import gates
import oracle
import qss_synth
from qss_synth import make_states

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


def _gpu_eval(mech, C, T, n_cells, want_jac=True):
    import paper_2405_05974_b200 as qss
    torch = _torch()
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    ld = C.shape[1]
    out = {}
    # poison outputs so that untouched entries are detected
    wdot = torch.full((qm.N, ld), float("nan"), dtype=torch.float64, device="cuda")
    cq = torch.full((max(qm.Nq, 1), ld), float("nan"), dtype=torch.float64, device="cuda")
    w, y = qm.eval_wdot(Cd, Td, n_cells, wdot=wdot, cqss=cq, want_cqss=True)
    out["wdot"] = w.cpu().numpy(); out["cqss"] = y.cpu().numpy()
    if want_jac:
        jac = torch.full((qm.N, qm.N + 1, ld), float("nan"), dtype=torch.float64, device="cuda")
        wd2 = torch.full((qm.N, ld), float("nan"), dtype=torch.float64, device="cuda")
        J, w2 = qm.eval_jac(Cd, Td, n_cells, jac=jac, wdot=wd2, want_wdot=True)
        out["jac"] = J.cpu().numpy(); out["wdot_from_jac"] = w2.cpu().numpy()
        jac.fill_(float("nan"))
        out["jac_only"] = qm.eval_jac(Cd, Td, n_cells, jac=jac).cpu().numpy()
    torch.cuda.synchronize()
    qm.close()
    return out


def _check(mech, C, T, n_cells, what, want_jac=True, cfg=None):
    om = oracle.OracleMech(mech)
    ref = oracle.evaluate(om, C, T, n_cells, want_jac=want_jac, want_scale=want_jac)
    got = _gpu_eval(mech, C, T, n_cells, want_jac)
    n = n_cells
    g = gates.assert_wdot(got["wdot"], ref["wdot"], ref["S"], n, what + " wdot", cfg=cfg)
    if mech.n_qss:
        y, yr = got["cqss"][:, :n], ref["cqss"][:, :n]
        assert np.isfinite(y).all() and (y >= 0).all()
        assert np.max(np.abs(y - yr) / np.abs(yr)) < 1e-9, what + " cqss"
    # padding cells (c >= n_cells) must not be written
    if C.shape[1] > n:
        assert np.isnan(got["wdot"][:, n:]).all(), what + ": wdot padding was written"
    if want_jac:
        gates.assert_wdot(got["wdot_from_jac"], ref["wdot"], ref["S"], n, what + " wdot (jac pass)")
        gj = gates.assert_jac(got["jac"], ref["jac"], ref["jscale"], n, what + " jac", cfg=cfg)
        assert np.array_equal(got["jac"][:, :, :n], got["jac_only"][:, :, :n]), what + ": jac differs with/without wdot output"
        if C.shape[1] > n:
            assert np.isnan(got["jac"][:, :, n:]).all(), what + ": jac padding was written"
        g.update(gj)
    if cfg is not None:      # G16 stays evidence: the unfiltered strict-tier fractions next to the filtered ones
        print(f"[gates] {what}: wdot tier-1 {g['tier1_frac']:.4f} (unfiltered {g['tier1_frac_unfiltered']:.4f}, well-conditioned {g['wellcond_frac']:.4f})"
              + (f"; columns tier-1 {g['col_tier1_frac']:.4f} (unfiltered {g['col_tier1_frac_unfiltered']:.4f}, well-conditioned {g['col_wellcond_frac']:.4f})" if want_jac else ""))
    return g


@pytest.mark.parametrize("name", ["toy1", "toy2", "toy3", "toy_dag", "toy_nonqss"])
def test_toys(name):
    mech = getattr(qss_synth, name)()
    n = 77                                     # ragged: 2 full warps of cells + a tail, ld padded to 96
    C, T = make_states(mech.n_nqss, n, seed=5)
    _check(mech, C, T, n, name)


def test_cfg1_full():
    mech = qss_synth.config_mechanism(1)
    C, T = qss_synth.config_states(1)
    _check(mech, C, T, 4096, "cfg1", cfg=1)


@pytest.mark.parametrize("cfg,n", [(2, 4096 + 37), (3, 1024 + 5), (5, 160 + 3)])
def test_configs_small(cfg, n):
    mech = qss_synth.config_mechanism(cfg)
    C, T = qss_synth.config_states(cfg, n)
    g = _check(mech, C, T, n, f"cfg{cfg}", cfg=cfg)
    print(f"cfg{cfg}", g)


def test_kernel_variants_selected_and_general_kernel_on_cfg2(monkeypatch):
    """cfg1/cfg2: the Jacobian and wdot alone run on kernel variant 3 (generated per mechanism, reaction-per-lane rate phases);
    cfg3 on the general variant 0.  QSS_VARIANT=2 selects the round-1 specialised kernel,
    QSS_VARIANT=0 the general kernel: both must meet the same gates on cfg2.  A silent fall-back would show up here."""
    import paper_2405_05974_b200 as qss
    for cfg, want_jac, want_wdot in ((1, 3, 3), (2, 3, 3), (3, 0, 0)):
        qm = qss.QssMech(qss_synth.config_mechanism(cfg), 0)
        assert qm.info.kernel_variant_jac == want_jac and qm.info.kernel_variant_wdot == want_wdot
        qm.close()
    mech = qss_synth.config_mechanism(2)
    n = 256 + 9
    C, T = qss_synth.config_states(2, n)
    for force, want in (("2", 2), ("0", 0)):
        monkeypatch.setenv("QSS_VARIANT", force)
        qm = qss.QssMech(mech, 0)
        assert qm.info.kernel_variant_jac == want
        qm.close()
        _check(mech, C, T, n, f"cfg2 (variant {want})")


@pytest.mark.parametrize("name", ["toy1", "toy2", "toy3", "toy_dag"])
@pytest.mark.parametrize("variant", ["2", "3"])
def test_many_slabs_per_block_on_small_mechanisms(name, variant, monkeypatch):
    """More than 2 * 32 * n_SM cells, so that every persistent block takes a 2nd and later slab: their inputs come through the
    cp.async staging rows (in variant 2 those rows could coincide with the zero rows of the thermo tables and a
    staged T was overwritten with 0 -> NaN; no earlier test reached it, the toys ran one slab per block)."""
    monkeypatch.setenv("QSS_VARIANT", variant)
    mech = getattr(qss_synth, name)()
    n = 20000 + 7
    C, T = make_states(mech.n_nqss, n, seed=9)
    _check(mech, C, T, n, f"{name} variant {variant}, many slabs")


def test_table_interpreter_when_specialisation_is_off(monkeypatch):
    """QSS_JIT=0: the Jacobian sweep runs on the table interpreter of variant 1 (what a box without NVRTC gets): same
    gates."""
    import paper_2405_05974_b200 as qss
    monkeypatch.setenv("QSS_JIT", "0")
    mech = qss_synth.config_mechanism(2)
    qm = qss.QssMech(mech, 0)
    assert qm.info.kernel_variant_jac == 1
    qm.close()
    n = 1024 + 13
    C, T = qss_synth.config_states(2, n)
    _check(mech, C, T, n, "cfg2 (interpreter)")
    mech = qss_synth.toy_dag()
    C, T = make_states(mech.n_nqss, 77, seed=5)
    _check(mech, C, T, 77, "toy_dag (interpreter)")


def test_specialised_and_interpreter_kernels_agree(monkeypatch):
    """The generated kernel (variant 3) and the table interpreter (variant 1) compute the same quantities with different
    operation orders (rate constants from folded NASA-7 sums, reaction-per-lane): their Jacobians and wdot meet the parity gates
    against each other (the oracle's running-error scales decide what "equal" means where terms cancel)."""
    mech = qss_synth.config_mechanism(2)
    n = 640 + 11
    C, T = qss_synth.config_states(2, n)
    a = _gpu_eval(mech, C, T, n)
    monkeypatch.setenv("QSS_JIT", "0")
    b = _gpu_eval(mech, C, T, n)
    ref = oracle.evaluate(oracle.OracleMech(mech), C, T, n, want_jac=True, want_scale=True)
    gates.assert_wdot(a["wdot"], b["wdot"], ref["S"], n, "variant 3 against variant 1, wdot")
    gates.assert_jac(a["jac"], b["jac"], ref["jscale"], n, "variant 2 against variant 1")


def test_column_streams_in_global_memory(monkeypatch):
    """When the hot tables do not fit the kernel-parameter constant bank the column streams of the table interpreter move
    to global memory (QSS_CS_GLOBAL=1 forces it): same results."""
    monkeypatch.setenv("QSS_CS_GLOBAL", "1")
    monkeypatch.setenv("QSS_JIT", "0")
    for mech, n, what in ((qss_synth.config_mechanism(2), 512 + 21, "cfg2 (streams in global memory)"),
                          (qss_synth.toy_dag(), 77, "toy_dag (streams in global memory)")):
        C, T = (qss_synth.config_states(2, n) if mech.n_reac > 100 else make_states(mech.n_nqss, n, seed=5))
        _check(mech, C, T, n, what)


def test_cfg4_field_small():
    mech = qss_synth.config_mechanism(4)
    C, T = qss_synth.config_states(4, 16 ** 3)           # 16^3 cells of the multipulse-shaped field
    _check(mech, np.ascontiguousarray(C), np.ascontiguousarray(T), C.shape[1], "cfg4", cfg=4)


@pytest.mark.parametrize("n", [1, 31, 32, 33])
def test_tiny_and_ragged_cell_counts(n):
    mech = qss_synth.config_mechanism(1)
    C, T = make_states(mech.n_nqss, n, seed=11, ld=64)
    _check(mech, C, T, n, f"cfg1 n={n}")


def test_zero_concentrations_and_tmid_tie_break():
    """Degenerate inputs: species with C_k = 0 (the partial derivatives are products of the OTHER molecules, never
    r / C_k: reading G12) and cells exactly at T = Tmid = 1000 K (reading G9: the high NASA range applies)."""
    mech = qss_synth.config_mechanism(2)
    n = 128 + 7
    C, T = qss_synth.config_states(2, n)
    rng = np.random.default_rng(3)
    for c in range(0, n, 3):                               # zero out 1-4 random species in every third cell
        C[rng.choice(mech.n_nqss, size=rng.integers(1, 5), replace=False), c] = 0.0
    T[5:n:11] = 1000.0
    g = _check(mech, np.ascontiguousarray(C), np.ascontiguousarray(T), n, "cfg2 zeros/Tmid")
    print(g)


@pytest.mark.parametrize("env", [{}, {"QSS_VARIANT": "2"}, {"QSS_JIT": "0"}, {"QSS_VARIANT": "0"}])
def test_chemkin_placeholder_troe_parameters(env, monkeypatch):
    """CHEMKIN files write T*** ~ 1e-30 and T*, T** ~ 1e30 for an absent Troe term: the exponentials must saturate to 0 / 1 / 0 in
    every kernel variant (the branch-free exp is only valid for |x| < 2^30 and returned inf / NaN there)."""
    import dataclasses
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    mech = qss_synth.config_mechanism(2)
    troe = mech.troe.copy()
    idx = np.flatnonzero(mech.rtype == 2)
    troe[idx[0::3], 1:] = (1.0e-30, 1.0e30, 1.0e30)
    troe[idx[1::3], 3] = 1.0e30
    mech = dataclasses.replace(mech, troe=troe)
    n = 96 + 5
    C, T = qss_synth.config_states(2, n)
    _check(mech, C, T, n, f"cfg2 placeholder Troe {env}")


@pytest.mark.parametrize("env", [{}, {"QSS_JIT": "0"}, {"QSS_VARIANT": "0"}])
def test_species_with_their_own_mid_temperatures(env, monkeypatch):
    """Real NASA-7 data give every species its own Tmid (the synthetic configs use 1000 K throughout).  Then a reaction's species
    sit in different ranges for T between their breakpoints: the generated kernel folds -ln Kc below the smallest and above the
    largest Tmid of a reaction and once per interval between consecutive breakpoints in between (qss_gen3.cpp); the other variants evaluate g/RT per
    species.  Same parity gates for all of them."""
    import dataclasses
    import paper_2405_05974_b200 as qss
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    mech = qss_synth.config_mechanism(2)
    rng = np.random.default_rng(17)
    nasa_T = mech.nasa_T.copy()
    nasa_T[:, 1] = rng.uniform(900.0, 1500.0, size=nasa_T.shape[0])
    mech = dataclasses.replace(mech, nasa_T=nasa_T)
    qm = qss.QssMech(mech, 0)
    variants = (qm.info.kernel_variant_wdot, qm.info.kernel_variant_jac)
    qm.close()
    assert variants == ((3, 3) if not env else (1, 1) if "QSS_JIT" in env else (0, 0)), variants
    n = 160 + 3
    C, T = qss_synth.config_states(2, n)
    T[: n // 2] = rng.uniform(880.0, 1520.0, size=n // 2)          # half of the cells between the breakpoints
    T[3] = nasa_T[0, 1]; T[4] = nasa_T[40, 1]                        # exactly at a species' Tmid (G9: high range)
    _check(mech, C, np.ascontiguousarray(T), n, f"cfg2 per-species Tmid {env} variants {variants}")


@pytest.mark.parametrize("env", [{}, {"QSS_VARIANT": "2"}, {"QSS_VARIANT": "0"}])
def test_extreme_temperatures_and_concentration_scales(env, monkeypatch):
    """Outside the sampled ranges: T = 200 .. 6000 K (beyond both NASA ranges: the polynomials extrapolate, rate constants span
    hundreds of decades), whole cells scaled by 1e-150 .. 1e12.  Where the preconditions of include/qss.h fail (a cell scaled into
    underflow, a cell with one species only, an all-zero cell: a QSS species without consumption, M = 0) the oracle's result is
    not finite and the kernel's must not be either: no silent number."""
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    mech = qss_synth.config_mechanism(2)
    n = 64
    C, T = qss_synth.config_states(2, n)
    C = C.copy(); T = T.copy()
    T[0:6] = (250.0, 300.0, 3500.0, 5000.0, 200.0, 6000.0)
    C[:, 6] *= 1e-20; C[:, 7] *= 1e-150; C[:, 9] *= 1e6; C[:, 10] *= 1e12
    bad = [8, 11, 12, 13]
    C[:, 8] *= 1e-300
    C[:, 11] = 0.0; C[3, 11] = 1.0
    C[:, 12] = 5e-324
    C[:, 13] = 0.0
    good = np.array([c for c in range(n) if c not in bad])
    with np.errstate(all="ignore"):
        ref = oracle.evaluate(oracle.OracleMech(mech), C, T, n, want_jac=True, want_scale=True)
    got = _gpu_eval(mech, C, T, n)
    for c in bad:
        fin_ref = np.isfinite(ref["wdot"][:, c]).all() and np.isfinite(ref["jac"][:, :, c]).all()
        fin_got = np.isfinite(got["wdot"][:, c]).all() and np.isfinite(got["jac"][:, :, c]).all()
        assert fin_got == fin_ref, (c, fin_ref, fin_got)
    gw = gates.wdot_gates(got["wdot"][:, good], ref["wdot"][:, good], ref["S"][:, good], len(good))
    gj = gates.jac_gates(got["jac"][:, :, good], ref["jac"][:, :, good], ref["jscale"][:, :, good], len(good))
    print(env, "wdot tier 2 worst %.2g; Jacobian tier 2 worst %.2g / %.2g" % (gw["tier2_worst"], gj["cell_tier2_worst"], gj["col_tier2_worst"]))
    assert gw["finite"] and gw["tier2_all"] and gj["finite"] and gj["cell_tier2_all"] and gj["col_tier2_all"]
    assert gw["tier1_frac"] >= 0.99 and gj["cell_tier1_frac"] >= 0.99


@pytest.mark.parametrize("cfg,n", [(2, (1 << 18) + 77), (1, 1 << 18), (3, 1 << 14)])
def test_run_to_run_bit_identity(cfg, n):
    """No kernel uses atomics or depends on the order in which warps or blocks run: repeated calls on the same inputs, with dozens
    of slabs per persistent block, return the same bits (a race between the warps of a block or between a block's consecutive slabs
    would show here; compute-sanitizer is not available on this pool)."""
    import paper_2405_05974_b200 as qss
    torch = _torch()
    mech = qss_synth.config_mechanism(cfg)
    C, T = qss_synth.config_states(cfg, n)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J0, w0 = qm.eval_jac(Cd, Td, n, want_wdot=True)
    ww0, y0 = qm.eval_wdot(Cd, Td, n, want_cqss=True)
    assert torch.equal(w0[:, :n], ww0[:, :n])              # the two kernels compute wdot by the same operations
    for _ in range(4):
        J, w = qm.eval_jac(Cd, Td, n, want_wdot=True)
        ww, y = qm.eval_wdot(Cd, Td, n, want_cqss=True)
        torch.cuda.synchronize()
        assert torch.equal(J[:, :, :n], J0[:, :, :n]) and torch.equal(w[:, :n], w0[:, :n])
        assert torch.equal(ww[:, :n], ww0[:, :n]) and torch.equal(y[:, :n], y0[:, :n])
    qm.close()


def test_paper_style_sampling():
    """States drawn the way the paper validates its Jacobian: C ~ U[1e-4, 1] mol/m^3 for every
    species, T ~ U[300, 1300] K (both NASA ranges, very small rate constants at the cold end)."""
    mech = qss_synth.config_mechanism(2)
    n = 512 + 3
    rng = np.random.default_rng(42)
    ld = (n + 31) // 32 * 32
    C = np.empty((mech.n_nqss, ld)); T = np.empty(ld)
    C[:, :n] = rng.uniform(1e-4, 1.0, size=(mech.n_nqss, n)); T[:n] = rng.uniform(300.0, 1300.0, size=n)
    C[:, n:] = C[:, :1]; T[n:] = T[0]
    g = _check(mech, C, T, n, "cfg2 paper-style states")
    print(g)


def test_non_default_stream_graph_capture_and_padding():
    """qss_eval_* only enqueue on the caller's stream: a captured CUDA graph replays to the same result; ld > ncells
    with a large pad leaves the padding untouched."""
    import paper_2405_05974_b200 as qss
    torch = _torch()
    mech = qss_synth.config_mechanism(2)
    n, ld = 500, 1024
    C, T = make_states(mech.n_nqss, n, seed=21, ld=ld)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J0, w0 = qm.eval_jac(Cd, Td, n, want_wdot=True)
    torch.cuda.synchronize()
    J = torch.full_like(J0, float("nan")); w = torch.full_like(w0, float("nan"))
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        qm.eval_jac(Cd, Td, n, jac=J, wdot=w, want_wdot=True)          # warm-up on the side stream
        s.synchronize()
        J.fill_(float("nan")); w.fill_(float("nan"))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            qm.eval_jac(Cd, Td, n, jac=J, wdot=w, want_wdot=True)
        g.replay()
        s.synchronize()
    assert torch.equal(J[:, :, :n], J0[:, :, :n]) and torch.equal(w[:, :n], w0[:, :n])
    assert torch.isnan(J[:, :, n:]).all() and torch.isnan(w[:, n:]).all()
    ref = oracle.evaluate(oracle.OracleMech(mech), C, T, n, want_jac=True, want_scale=True)
    gates.assert_jac(J.cpu().numpy(), ref["jac"], ref["jscale"], n, "graph replay jac")


def test_host_buffer_call_matches_the_device_call():
    """qss_eval_jac_host (pinned host buffers, chunked copy/compute pipeline) returns exactly what qss_eval_jac does."""
    import paper_2405_05974_b200 as qss
    torch = _torch()
    mech = qss_synth.config_mechanism(1)
    n = 70000 + 13                                         # > 2^16 cells: 8 chunks with a ragged last one
    C, T = make_states(mech.n_nqss, n, seed=31)
    ld = C.shape[1]
    qm = qss.QssMech(mech, 0)
    J0, w0 = qm.eval_jac(torch.from_numpy(C).cuda(), torch.from_numpy(T).cuda(), n, want_wdot=True)
    torch.cuda.synchronize()
    Ch = torch.from_numpy(C).pin_memory(); Th = torch.from_numpy(T).pin_memory()
    Jh = torch.full((qm.N, qm.N + 1, ld), float("nan"), dtype=torch.float64).pin_memory()
    Wh = torch.full((qm.N, ld), float("nan"), dtype=torch.float64).pin_memory()
    scratch = torch.empty(qm.host_scratch_bytes(n, ld) + 256, dtype=torch.uint8, device="cuda")
    qm.eval_jac_host(Ch, Th, Jh, Wh, scratch, n)
    assert torch.equal(Jh[:, :, :n], J0[:, :, :n].cpu()) and torch.equal(Wh[:, :n], w0[:, :n].cpu())
    assert torch.isnan(Jh[:, :, n:]).all() and torch.isnan(Wh[:, n:]).all()


def test_zero_cells_is_a_noop():
    import paper_2405_05974_b200 as qss
    torch = _torch()
    mech = qss_synth.config_mechanism(1)
    qm = qss.QssMech(mech, 0)
    C = torch.ones((qm.N, 32), dtype=torch.float64, device="cuda"); T = torch.full((32,), 1000.0, dtype=torch.float64, device="cuda")
    w = torch.full((qm.N, 32), -7.0, dtype=torch.float64, device="cuda")
    qm.eval_wdot(C, T, 0, wdot=w)
    torch.cuda.synchronize()
    assert (w == -7.0).all()


def test_bad_arguments_are_rejected():
    import paper_2405_05974_b200 as qss
    torch = _torch()
    mech = qss_synth.config_mechanism(1)
    qm = qss.QssMech(mech, 0)
    C = torch.ones((qm.N, 32), dtype=torch.float64, device="cuda"); T = torch.full((32,), 1000.0, dtype=torch.float64, device="cuda")
    with pytest.raises(qss.QssError) as e:
        qm.eval_wdot(C, T, 64)                            # ncells > ld
    assert e.value.code == -1
    small = torch.empty(256, dtype=torch.uint8, device="cuda")
    qm._ws[(True, torch.cuda.current_stream().cuda_stream)] = small
    with pytest.raises(qss.QssError) as e:
        qm.eval_jac(C, T, 32)                             # workspace too small
    assert e.value.code == -1


@pytest.mark.parametrize("cfg,nsample", [(3, 128), (4, 128), (5, 48)])
def test_full_size_other_configs_sampled(cfg, nsample):
    """BASELINE.json configs[2], [3], [4] at their full sizes (2^19 cells, the 128^3 field, 2^18 cells) in the launch
    configuration bench.py uses; sampled cells (first, last, random) are recomputed one by one by the oracle and every
    output must be finite."""
    import paper_2405_05974_b200 as qss
    torch = _torch()
    mech = qss_synth.config_mechanism(cfg)
    C, T = qss_synth.config_states(cfg)
    n = qss_synth.CONFIGS[cfg]["n_cells"]
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(np.ascontiguousarray(C)).cuda(); Td = torch.from_numpy(np.ascontiguousarray(T)).cuda()
    J, w = qm.eval_jac(Cd, Td, n, want_wdot=True)
    torch.cuda.synchronize()
    assert torch.isfinite(w[:, :n]).all() and torch.isfinite(J[:, :, :n]).all()
    idx = np.sort(np.random.default_rng(100 + cfg).choice(n, size=nsample, replace=False))
    idx[0], idx[-1] = 0, n - 1
    it = torch.from_numpy(idx).cuda()
    Js = J[:, :, it].cpu().numpy(); ws = w[:, it].cpu().numpy()
    del J, w
    Cs = np.ascontiguousarray(C[:, idx]); Ts = np.ascontiguousarray(T[idx])
    ref = oracle.evaluate(oracle.OracleMech(mech), Cs, Ts, want_jac=True, want_scale=True)
    gates.assert_wdot(ws, ref["wdot"], ref["S"], what=f"cfg{cfg} full wdot", cfg=cfg)
    gates.assert_jac(Js, ref["jac"], ref["jscale"], what=f"cfg{cfg} full jac", cfg=cfg)


def test_full_size_cfg2_sampled():
    """BASELINE.json configs[1] at full size (2^20 cells) in the launch configuration bench.py times;
    256 sampled cells are recomputed one by one by the oracle."""
    import paper_2405_05974_b200 as qss
    torch = _torch()
    mech = qss_synth.config_mechanism(2)
    C, T = qss_synth.config_states(2)
    n = C.shape[1]
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    J, w = qm.eval_jac(Cd, Td, n, want_wdot=True)
    torch.cuda.synchronize()
    rng = np.random.default_rng(99)
    idx = np.sort(rng.choice(n, size=256, replace=False))
    idx[0], idx[-1] = 0, n - 1
    it = torch.from_numpy(idx).cuda()
    Js = J[:, :, it].cpu().numpy(); ws = w[:, it].cpu().numpy()
    assert torch.isfinite(w).all() and torch.isfinite(J).all()
    Cs = np.ascontiguousarray(C[:, idx]); Ts = np.ascontiguousarray(T[idx])
    ref = oracle.evaluate(oracle.OracleMech(mech), Cs, Ts, want_jac=True, want_scale=True)
    gates.assert_wdot(ws, ref["wdot"], ref["S"], what="cfg2 full wdot", cfg=2)
    gates.assert_jac(Js, ref["jac"], ref["jscale"], what="cfg2 full jac", cfg=2)
