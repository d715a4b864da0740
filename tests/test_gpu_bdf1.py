"""GPU parity of NEXT-4 (first half): the 0-D constant-volume integrator qss_bdf1_advance (DESIGN.md
reading G21) against the oracle's integrator of the same algorithm (oracle.bdf1_advance) on the same seeded states.

Tolerance: every Newton iteration solves a linear system whose conditioning enters the forward error (gates.newton_gates), and
`newton_iters` iterations of a contracting map re-absorb most of it; what is asserted is normwise agreement of the final state,
|dC| <= 1e-8 max|C| per cell and |dT| <= 1e-10 T, on cells where the oracle's own float64 result is reproducible to that level
(every cell here: the comparison prints the worst ratio)."""
import numpy as np
import pytest

import oracle
import qss_synth
from qss_synth import make_states

pytestmark = pytest.mark.gpu


def _dt(om, C, T, n, theta, seed):
    ev = oracle.evaluate(om, C, T, n); en = oracle.evaluate_energy(om, C, T, n)
    jm = np.maximum(np.abs(ev["jac"]).max((0, 1)), np.abs(en["erow"]).max(0))
    rng = np.random.default_rng(seed)
    return theta * 10.0 ** rng.uniform(-0.5, 0.5, size=C.shape[1]) / np.where(jm > 0, jm, 1.0)


@pytest.mark.parametrize("name,n,theta,nsub,iters", [("cfg1", 257, 3.0, 3, 3), ("cfg2", 96 + 5, 3.0, 2, 3), ("cfg2", 64, 100.0, 2, 4),
                                                     ("toy_dag", 40, 2.0, 4, 3), ("toy3", 33, 1.0, 2, 2)])
def test_bdf1_against_oracle(name, n, theta, nsub, iters):
    import torch
    import paper_2405_05974_b200 as qss
    if name.startswith("cfg"):
        mech = qss_synth.config_mechanism(int(name[3])); C, T = qss_synth.config_states(int(name[3]), n)
    else:
        mech = getattr(qss_synth, name)(); C, T = make_states(mech.n_nqss, n, seed=5)
    om = oracle.OracleMech(mech)
    dt = _dt(om, C, T, n, theta, 3)
    Cr, Tr = oracle.bdf1_advance(om, C, T, dt, nsub, iters, n)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda(); dtd = torch.from_numpy(dt).cuda()
    qm.bdf1_advance(Cd, Td, dtd, nsub, iters, n)
    torch.cuda.synchronize()
    Cg, Tg = Cd.cpu().numpy(), Td.cpu().numpy()
    ld = C.shape[1]
    if ld > n:                                                           # padding untouched (bit for bit, NaN included)
        assert np.array_equal(Cg[:, n:], C[:, n:], equal_nan=True) and np.array_equal(Tg[n:], T[n:], equal_nan=True)
    # a cell on which the fixed-step Newton iteration diverges (no step-size control, reading G21) ends non-finite in the oracle:
    # the kernel must end non-finite in T there too; everything else is compared
    ok = np.isfinite(Tr[:n]) & np.isfinite(Cr[:, :n]).all(0)
    assert ok.mean() >= 0.98 and not np.isfinite(Tg[:n][~ok]).any()
    assert np.isfinite(Cg[:, :n][:, ok]).all() and np.isfinite(Tg[:n][ok]).all()
    moved = np.abs(Cr[:, :n] - C[:, :n]).max(0)[ok] > 1e-6 * np.abs(C[:, :n]).max(0)[ok]
    eC = (np.abs(Cg[:, :n] - Cr[:, :n]).max(0) / np.abs(Cr[:, :n]).max(0))[ok]
    eT = (np.abs(Tg[:n] - Tr[:n]) / Tr[:n])[ok]
    print("%s: %d of %d cells moved, %d diverged in the oracle; worst normwise dC %.2e, worst dT/T %.2e"
          % (name, int(moved.sum()), n, int((~ok).sum()), eC.max(), eT.max()))
    assert moved.sum() >= n // 4
    assert eC.max() <= 1e-8 and eT.max() <= 1e-10
    qm.close()


def test_zero_substeps_and_unsupported():
    import torch
    import paper_2405_05974_b200 as qss
    mech = qss_synth.config_mechanism(1); C, T = qss_synth.config_states(1, 64)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda(); dt = torch.zeros(C.shape[1], dtype=torch.float64, device="cuda")
    qm.bdf1_advance(Cd, Td, dt, 2, 2, 64)                                # h = 0: the identity (delta = 0 exactly)
    qm.bdf1_advance(Cd, Td, dt, 0, 2, 64)
    torch.cuda.synchronize()
    assert np.array_equal(Cd.cpu().numpy(), C, equal_nan=True) and np.array_equal(Td.cpu().numpy(), T, equal_nan=True)
    qm.close()
    qm3 = qss.QssMech(qss_synth.config_mechanism(3), 0)
    C3, T3 = qss_synth.config_states(3, 32)
    with pytest.raises(qss.QssError) as e:
        qm3.bdf1_advance(torch.from_numpy(C3).cuda(), torch.from_numpy(T3).cuda(), torch.zeros(C3.shape[1], dtype=torch.float64, device="cuda"), 1, 1, 32)
    assert e.value.code == -5
    qm3.close()


@pytest.mark.parametrize("name,n,attempts,iters,rtol", [("cfg1", 257, 12, 3, 1e-6), ("cfg2", 64 + 5, 8, 3, 1e-6), ("toy_dag", 40, 20, 2, 1e-8)])
def test_adaptive_integrator_with_ignition_time_against_oracle(name, n, attempts, iters, rtol):
    """qss_ignition_advance against oracle.ignition_advance (reading G23).  Accept / reject are decisions on a floating-point number:
    both sides take them in fp64 from the same definition; cells where the oracle's criterion comes within 1e-6 of the threshold in any
    attempt are excluded (printed), the others must agree in EVERYTHING: number of accepted attempts, times, step sizes bit for bit,
    ignition times, and the state within the tolerance of the fixed-step test."""
    import torch
    import paper_2405_05974_b200 as qss
    if name.startswith("cfg"):
        mech = qss_synth.config_mechanism(int(name[3])); C, T = qss_synth.config_states(int(name[3]), n)
    else:
        mech = getattr(qss_synth, name)(); C, T = make_states(mech.n_nqss, n, seed=5)
    om = oracle.OracleMech(mech)
    ld = C.shape[1]
    dt0 = _dt(om, C, T, n, 30.0, 3)                                     # deliberately too large for many cells: rejections happen
    t_end = float(np.median(dt0[:n]) * 6.0)
    dT_ign = 0.05
    trace = []
    ref = oracle.ignition_advance(om, C, T, dt0, np.zeros(ld), t_end, attempts, iters, n, rtol=rtol, dT_ign=dT_ign, trace=trace)
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda(); T0d = Td.clone()
    dtd = torch.from_numpy(dt0).cuda(); td = torch.zeros(ld, dtype=torch.float64, device="cuda")
    tig = torch.full((ld,), float("nan"), dtype=torch.float64, device="cuda")
    qm.ignition_advance(Cd, Td, dtd, td, t_end, attempts, iters, n, t_ign=tig, T0=T0d, dT_ign=dT_ign, rtol=rtol)
    torch.cuda.synchronize()
    Cg, Tg, dtg, tg, tigg = (x.cpu().numpy() for x in (Cd, Td, dtd, td, tig))
    tr = np.array(trace)                                                 # [attempts, n]
    sure = ~(np.abs(tr - 1.0) <= 1e-6).any(0) & np.isfinite(ref["T"][:n])
    rejected = int((attempts - ref["accepted"][:n][sure]).sum())
    print("%s: %d of %d cells compared, %d rejected attempts among them, %d ignition times, reached t_end: %d"
          % (name, int(sure.sum()), n, rejected, int(np.isfinite(ref["t_ign"][:n][sure]).sum()), int((ref["t"][:n][sure] == t_end).sum())))
    assert sure.mean() >= 0.95 and rejected > 0
    assert np.array_equal(tg[:n][sure], ref["t"][:n][sure]) and np.array_equal(dtg[:n][sure], ref["dt"][:n][sure])
    assert np.array_equal(tigg[:n][sure], ref["t_ign"][:n][sure], equal_nan=True)
    eC = (np.abs(Cg[:, :n] - ref["C"][:, :n]).max(0) / np.abs(ref["C"][:, :n]).max(0))[sure]
    eT = (np.abs(Tg[:n] - ref["T"][:n]) / ref["T"][:n])[sure]
    assert eC.max() <= 1e-8 and eT.max() <= 1e-10, (eC.max(), eT.max())
    if ld > n:
        assert np.array_equal(Cg[:, n:], C[:, n:], equal_nan=True) and np.array_equal(tg[n:], np.zeros(ld - n))
    qm.close()


def test_integrator_sequence_and_newton_solve_replay_from_a_cuda_graph():
    """qss_bdf1_advance is a FIXED launch sequence on the caller's stream (no host decision, no allocation, no synchronisation:
    include/qss.h), and so are qss_eval_jac_full and qss_newton_solve: captured once in a CUDA graph and replayed on restored
    inputs they give bit for bit what the eager calls gave."""
    import torch
    import paper_2405_05974_b200 as qss
    mech = qss_synth.config_mechanism(2)
    n = 200
    C, T = qss_synth.config_states(2, n)
    ld = C.shape[1]
    om = oracle.OracleMech(mech)
    dt = _dt(om, C, T, n, 3.0, 3)
    qm = qss.QssMech(mech, 0)
    C0 = torch.from_numpy(C).cuda(); T0 = torch.from_numpy(T).cuda(); dtd = torch.from_numpy(dt).cuda()
    Ce, Te = C0.clone(), T0.clone()
    ws = qm.bdf1_advance(Ce, Te, dtd, 2, 3, n)                                   # eager, default stream
    J0, w0, td0, er0 = qm.eval_jac_full(Ce, Te, n)
    gamma = dtd.clone()
    b = torch.cat([w0, td0[None, :]], 0).contiguous()
    x0 = qm.newton_solve(J0, er0, gamma, b, n)
    torch.cuda.synchronize()
    Cg, Tg = C0.clone(), T0.clone()
    J = torch.empty_like(J0); w = torch.empty_like(w0); td = torch.empty_like(td0); er = torch.empty_like(er0); x = torch.empty_like(x0)
    bg = torch.empty_like(b)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        qm.bdf1_advance(Cg, Tg, dtd, 2, 3, n, workspace=ws)                      # warm-up on the side stream (run-time compilation done)
        qm.eval_jac_full(Cg, Tg, n, jac=J, wdot=w, tdot=td, erow=er)
        qm.newton_solve(J, er, gamma, b, n, x=x)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            qm.bdf1_advance(Cg, Tg, dtd, 2, 3, n, workspace=ws)
            qm.eval_jac_full(Cg, Tg, n, jac=J, wdot=w, tdot=td, erow=er)
            bg[: qm.N].copy_(w); bg[qm.N].copy_(td)
            qm.newton_solve(J, er, gamma, bg, n, x=x)
        for _ in range(2):                                                       # two replays, inputs restored before each
            Cg.copy_(C0); Tg.copy_(T0)
            for a in (J, w, td, er, x, bg):
                a.fill_(float("nan"))
            g.replay()
        s.synchronize()
    assert torch.equal(Cg[:, :n], Ce[:, :n]) and torch.equal(Tg[:n], Te[:n])
    assert torch.equal(J[:, :, :n], J0[:, :, :n]) and torch.equal(er[:, :n], er0[:, :n]) and torch.equal(x[:, :n], x0[:, :n])
    qm.close()
