"""qss_eval_wdot_static (include/qss.h): the allocation-free entry point -- the general slab kernel with its workspace in a static
device array inside the library -- against the existing path (qss_eval_wdot with a caller-supplied workspace), on two calls in a
row that share the array: different mechanisms and cell counts, so that the second call meets the first one's leftovers.
Tolerance: the wdot gate of the other GPU tests (1e-10 |w| + 1e-13 S, S the oracle's running-error scale; gates.py) against the
handle's default kernel (variant 3 here: another summation order), and bit for bit against the same general kernel selected with
QSS_VARIANT=0.  (Named test_zz_*: pytest collects it last, so a failure here hides no other test under -x.)"""
import numpy as np
import pytest

import gates
import oracle
import qss_synth

pytestmark = pytest.mark.gpu


def _case(cfg, n, variant_env, monkeypatch):
    import torch
    import paper_2405_05974_b200 as qss
    if variant_env is None:
        monkeypatch.delenv("QSS_VARIANT", raising=False)
    else:
        monkeypatch.setenv("QSS_VARIANT", variant_env)
    mech = qss_synth.config_mechanism(cfg)
    C, T = qss_synth.config_states(cfg, n)
    ld = C.shape[1]
    qm = qss.QssMech(mech, 0)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    w_ref, y_ref = qm.eval_wdot(Cd, Td, n, want_cqss=True)                  # the existing path
    w = torch.full((qm.N, ld), float("nan"), dtype=torch.float64, device="cuda")
    y = torch.full((max(qm.Nq, 1), ld), float("nan"), dtype=torch.float64, device="cuda")
    before = torch.cuda.memory_allocated()
    qm.eval_wdot_static(Cd, Td, n, wdot=w, cqss=y)
    assert torch.cuda.memory_allocated() == before                           # (torch's view: the binding allocated nothing either)
    torch.cuda.synchronize()
    variant = qm.info.kernel_variant_wdot
    qm.close()
    return mech, C, T, ld, w.cpu().numpy(), y.cpu().numpy()[:mech.n_qss], w_ref.cpu().numpy(), y_ref.cpu().numpy(), variant


def _check(cfg, n, variant_env, monkeypatch):
    mech, C, T, ld, w, y, w_ref, y_ref, variant = _case(cfg, n, variant_env, monkeypatch)
    assert np.isfinite(w[:, :n]).all()
    if ld > n:
        assert np.isnan(w[:, n:]).all(), "padding was written"
    if variant_env == "0":
        assert variant == 0 and np.array_equal(w[:, :n], w_ref[:, :n]) and np.array_equal(y[:, :n], y_ref[:, :n])      # the same kernel: bit for bit
    S = oracle.evaluate(oracle.OracleMech(mech), C, T, n, want_jac=False)["S"][:, :n]
    d = np.abs(w[:, :n] - w_ref[:, :n])
    bound = gates.WDOT_RTOL * np.abs(w_ref[:, :n]) + gates.WDOT_GUARD * S
    assert (d <= bound).all(), float((d / bound).max())
    assert np.allclose(y[:, :n], y_ref[:, :n], rtol=1e-9, atol=0.0)
    return variant


def test_static_workspace_entry_point_two_calls_in_a_row(monkeypatch):
    v1 = _check(2, 2048 + 19, None, monkeypatch)          # call 1: cfg2, ragged tail, against the handle's default kernel
    v2 = _check(1, 4096, None, monkeypatch)               # call 2: another mechanism on the same array (leftovers of call 1)
    assert v1 == 3 and v2 == 3
    _check(2, 2048 + 19, "0", monkeypatch)                # calls 3, 4: against the same general kernel with a caller's workspace
    _check(3, 192 + 5, "0", monkeypatch)
    _check(5, 64 + 3, None, monkeypatch)                  # the largest mechanism: 2.3 MB of workspace per block, 3 blocks fit


def test_static_workspace_rejects_bad_arguments():
    import torch
    import paper_2405_05974_b200 as qss
    mech = qss_synth.config_mechanism(1)
    qm = qss.QssMech(mech, 0)
    C, T = qss_synth.config_states(1, 64)
    Cd = torch.from_numpy(C).cuda(); Td = torch.from_numpy(T).cuda()
    w = torch.zeros((qm.N, C.shape[1]), dtype=torch.float64, device="cuda")
    with pytest.raises(qss.QssError) as e:
        qm.eval_wdot_static(Cd, Td, C.shape[1] + 1, wdot=w)                  # ncells > ld
    assert e.value.code == -1
    qm.eval_wdot_static(Cd, Td, 0, wdot=w)                                   # zero cells: nothing launched
    qm.close()
