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
