"""CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT): ctypes binding of oracle/liboracle.so.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
It shares no code with the CUDA path; the only common input is a `qss_synth.Mechanism` (pure data).
"""
from __future__ import annotations

import ctypes as ct

import numpy as np

from . import build as _build

EXPLICIT_F64, EXPLICIT_F128, JAC_DUAL, JAC_CSTEP, JAC_CONST_QSS, JAC_ZERO_QSS = 0, 1, 2, 3, 4, 5

_lib = None


class _Mech(ct.Structure):
    _fields_ = [("n_nqss", ct.c_int32), ("n_qss", ct.c_int32), ("n_reac", ct.c_int32),
                ("nasa_T", ct.c_void_p), ("nasa_lo", ct.c_void_p), ("nasa_hi", ct.c_void_p),
                ("rtype", ct.c_void_p), ("dir_mask", ct.c_void_p),
                ("reac_ptr", ct.c_void_p), ("reac_sp", ct.c_void_p), ("reac_nu", ct.c_void_p),
                ("prod_ptr", ct.c_void_p), ("prod_sp", ct.c_void_p), ("prod_nu", ct.c_void_p),
                ("arr", ct.c_void_p), ("arr_low", ct.c_void_p), ("troe", ct.c_void_p),
                ("eff_ptr", ct.c_void_p), ("eff_sp", ct.c_void_p), ("eff_val", ct.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        _lib = ct.CDLL(_build.build())
        _lib.oracle_eval.restype = ct.c_int
        _lib.oracle_eval.argtypes = [ct.c_void_p, ct.c_int64, ct.c_int64] + [ct.c_void_p] * 7 + [ct.c_int, ct.c_int]
        _lib.oracle_eval_energy.restype = ct.c_int
        _lib.oracle_eval_energy.argtypes = [ct.c_void_p, ct.c_int64, ct.c_int64] + [ct.c_void_p] * 5 + [ct.c_int, ct.c_int]
        _lib.oracle_rate_constants.restype = ct.c_int
        _lib.oracle_rate_constants.argtypes = [ct.c_void_p, ct.c_void_p, ct.c_double, ct.c_void_p, ct.c_void_p]
        _lib.oracle_closure_check.restype = ct.c_int
        _lib.oracle_closure_check.argtypes = [ct.c_void_p, ct.c_void_p, ct.c_double] + [ct.c_void_p] * 3
        _lib.oracle_max_threads.restype = ct.c_int
        _lib.oracle_newton_solve.restype = ct.c_int
        _lib.oracle_newton_solve.argtypes = [ct.c_int, ct.c_int64, ct.c_int64] + [ct.c_void_p] * 6 + [ct.c_int]
    return _lib


class OracleMech:
    """Holds contiguous copies of a qss_synth.Mechanism's arrays and the C struct pointing at them."""

    def __init__(self, mech):
        self.N, self.Nq, self.M = mech.n_nqss, mech.n_qss, mech.n_reac
        self._keep = {}
        s = _Mech()
        s.n_nqss, s.n_qss, s.n_reac = mech.n_nqss, mech.n_qss, mech.n_reac
        spec = dict(nasa_T=np.float64, nasa_lo=np.float64, nasa_hi=np.float64, rtype=np.int32, dir_mask=np.uint8,
                    reac_ptr=np.int32, reac_sp=np.int32, reac_nu=np.int32, prod_ptr=np.int32, prod_sp=np.int32,
                    prod_nu=np.int32, arr=np.float64, arr_low=np.float64, troe=np.float64, eff_ptr=np.int32,
                    eff_sp=np.int32, eff_val=np.float64)
        for name, dt in spec.items():
            a = np.ascontiguousarray(getattr(mech, name), dtype=dt)
            if a.size == 0:
                a = np.zeros(1, dtype=dt)
            self._keep[name] = a
            setattr(s, name, a.ctypes.data)
        self.c = s

    def _ptr(self):
        return ct.addressof(self.c)


def _p(a):
    return None if a is None else a.ctypes.data


def _threads(nthreads: int, n_cells: int) -> int:
    """nthreads = 0 means "all", but never more threads than there are groups of 8 cells: a team of many threads for a handful of cells
    costs far more than the work (the cells are independent, so the results do not depend on it)."""
    return nthreads if nthreads > 0 else max(1, min(max_threads(), (n_cells + 7) // 8))


def evaluate(om: OracleMech, C: np.ndarray, T: np.ndarray, n_cells: int | None = None, *, want_jac=True,
             want_scale=False, mode=EXPLICIT_F64, nthreads=0):
    """C [N, ld], T [ld] float64. Returns dict(wdot [N,ld], cqss [Nq,ld], S [N,ld], jac [N,N+1,ld], jscale)."""
    assert C.dtype == np.float64 and T.dtype == np.float64 and C.flags.c_contiguous and T.flags.c_contiguous
    N, Nq = om.N, om.Nq
    ld = C.shape[1]
    n_cells = ld if n_cells is None else n_cells
    assert C.shape[0] == N and T.shape[0] == ld and n_cells <= ld
    out = dict(wdot=np.zeros((N, ld)), cqss=np.zeros((max(Nq, 1), ld)), S=np.zeros((N, ld)))
    out["jac"] = np.zeros((N, N + 1, ld)) if want_jac else None
    out["jscale"] = np.zeros((N, N + 1, ld)) if (want_jac and want_scale) else None
    rc = lib().oracle_eval(om._ptr(), n_cells, ld, _p(C), _p(T), _p(out["wdot"]), _p(out["cqss"]), _p(out["S"]),
                           _p(out["jac"]), _p(out["jscale"]), mode, _threads(nthreads, n_cells))
    if rc != 0:
        raise RuntimeError(f"oracle_eval failed rc={rc}")
    out["cqss"] = out["cqss"][:Nq]
    return out


def evaluate_energy(om: OracleMech, C: np.ndarray, T: np.ndarray, n_cells: int | None = None, *, mode=EXPLICIT_F64, nthreads=0):
    """Temperature right-hand side and energy row (NEXT-1). Returns dict(tdot [ld], erow [N+1, ld], escale [N+1, ld])."""
    assert C.dtype == np.float64 and T.dtype == np.float64 and C.flags.c_contiguous and T.flags.c_contiguous
    ld = C.shape[1]
    n_cells = ld if n_cells is None else n_cells
    out = dict(tdot=np.zeros(ld), erow=np.zeros((om.N + 1, ld)), escale=np.zeros((om.N + 1, ld)))
    rc = lib().oracle_eval_energy(om._ptr(), n_cells, ld, _p(C), _p(T), _p(out["tdot"]), _p(out["erow"]), _p(out["escale"]), mode, _threads(nthreads, n_cells))
    if rc != 0:
        raise RuntimeError(f"oracle_eval_energy failed rc={rc}")
    return out


def newton_solve(jac: np.ndarray, erow, gamma: np.ndarray, b: np.ndarray, n_cells: int | None = None, *, quad=False):
    """NEXT-2: x = (I - gamma J)^-1 b per cell by Gaussian elimination with partial pivoting (qss_newton_oracle.cpp).
    jac [N, N+1, ld], erow [N+1, ld] or None (then the N x N species block), gamma [ld], b [n, ld].
    Returns dict(x [n, ld], info [ld])."""
    N, ld = jac.shape[0], jac.shape[2]
    n = N + 1 if erow is not None else N
    assert jac.shape == (N, N + 1, ld) and b.shape == (n, ld) and gamma.shape == (ld,)
    for a in (jac, gamma, b) + ((erow,) if erow is not None else ()):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    assert erow is None or erow.shape == (N + 1, ld)
    n_cells = ld if n_cells is None else n_cells
    out = dict(x=np.zeros((n, ld)), info=np.zeros(ld, dtype=np.int32))
    rc = lib().oracle_newton_solve(N, n_cells, ld, _p(jac), _p(erow) if erow is not None else None, _p(gamma), _p(b), _p(out["x"]),
                                   _p(out["info"]), 1 if quad else 0)
    if rc != 0:
        raise RuntimeError(f"oracle_newton_solve failed rc={rc}")
    return out


def evaluate_fdT(om: OracleMech, C: np.ndarray, T: np.ndarray, n_cells: int | None = None):
    """NEXT-3, the paper's own temperature column (d wdot / dT "via finite difference by computing the species'
    production rate twice at different temperatures"; L234: central differences, perturbation 1e-4; reading G22):
        dT = 1e-4 T,  T+ = T + dT,  T- = T - dT,   J[:, N] = (wdot(C, T+) - wdot(C, T-)) / (T+ - T-)
    (the perturbation is taken relative to T; the divisor is the difference of the rounded temperatures).  The species columns are the
    explicit ones.  Returns the dict of `evaluate` with that column replaced."""
    ld = C.shape[1]
    n = ld if n_cells is None else n_cells
    out = evaluate(om, C, T, n, want_jac=True, want_scale=True)
    dT = 1e-4 * T
    Tp = T + dT
    Tm = T - dT
    wp = evaluate(om, C, np.ascontiguousarray(Tp), n, want_jac=False)["wdot"]
    wm = evaluate(om, C, np.ascontiguousarray(Tm), n, want_jac=False)["wdot"]
    out["jac"][:, om.N, :n] = (wp[:, :n] - wm[:, :n]) / (Tp[:n] - Tm[:n])
    out["wdot_p"], out["wdot_m"], out["Tp"], out["Tm"] = wp, wm, Tp, Tm
    return out


def bdf1_advance(om: OracleMech, C: np.ndarray, T: np.ndarray, dt: np.ndarray, nsub: int, newton_iters: int, n_cells: int | None = None,
                 *, history=False):
    """NEXT-4 (0D constant-volume reactor, the interval "divided into substeps over which the chemical state is
    advanced"; L183-188: implicit scheme, Newton method with the chemical Jacobian; reading G21): `nsub` backward-Euler
    substeps of size dt[c] per cell, each solved by `newton_iters` full Newton iterations, step by step as written:
        phi = (C, T),  f = (wdot, Tdot);   phi_0 = phi^n
        F(phi_m) = phi_m - phi^n - h f(phi_m);   (I - h J(phi_m)) delta = -F(phi_m);   phi_{m+1} = phi_m + delta,  C := max(C, 0)
        phi^{n+1} = phi_{newton_iters}
    with J the full (N+1) x (N+1) Jacobian (species block + energy row) and the linear solve of `newton_solve`.
    Returns (C, T) after the last substep (new arrays, padding untouched); with history=True also the list of T after every substep."""
    ld = C.shape[1]
    n = ld if n_cells is None else n_cells
    N = om.N
    C = C.copy(); T = T.copy()
    h = np.ascontiguousarray(dt, dtype=np.float64)
    hist = []
    for _ in range(nsub):
        Cn, Tn = C.copy(), T.copy()
        for _m in range(newton_iters):
            ev = evaluate(om, C, T, n, want_jac=True)
            en = evaluate_energy(om, C, T, n)
            jac, erow = ev["jac"], en["erow"]
            b = np.zeros((N + 1, ld))
            b[:N, :n] = (Cn[:, :n] - C[:, :n]) + h[:n] * ev["wdot"][:, :n]
            b[N, :n] = (Tn[:n] - T[:n]) + h[:n] * en["tdot"][:n]
            x = newton_solve(np.ascontiguousarray(jac), np.ascontiguousarray(erow), h, b, n)["x"]
            C[:, :n] = np.maximum(C[:, :n] + x[:N, :n], 0.0)
            T[:n] = T[:n] + x[N, :n]
        hist.append(T.copy())
    return (C, T, hist) if history else (C, T)


def ignition_advance(om: OracleMech, C, T, dt, t, t_end, n_attempts, newton_iters, n_cells=None, *, rtol=1e-6, atol_C=1e-12, atol_T=1e-6,
                     T0=None, dT_ign=400.0, t_ign=None, grow=1.5, shrink=0.25, trace=None):
    """NEXT-4, adaptive form of `bdf1_advance` (substeps inside which the integrator "employs its own variable size
    time-stepping strategy"; ignition delay L126: "the earliest time after which the initial temperature increased by at least 400K";
    DESIGN.md reading G23).  `n_attempts` attempts per cell, each: h = min(dt, t_end - t) (0 once t_end is reached: the identity),
    `newton_iters` full Newton iterations of the backward-Euler step as in `bdf1_advance`, then with delta = the LAST Newton update
        err = max( max_i |delta_i| / (atol_C + rtol |C_i|),  |delta_T| / (atol_T + rtol |T|) )      (C, T: the iterate it was added to)
    ACCEPT when err <= 1, everything is finite and the new T > 0: t += h, dt := grow dt, and t_ign := t (new) if it is still NaN and
    T_new - T0 >= dT_ign; else REJECT: (C, T) back to the start of the attempt, dt := shrink dt.
    All arrays are per cell and updated in copies: returns dict(C, T, dt, t, t_ign, accepted [ld] (count), err_last [ld]).
    `trace`: a list that receives err of every attempt (for tests that exclude decisions within rounding of the threshold)."""
    ld = C.shape[1]
    n = ld if n_cells is None else n_cells
    N = om.N
    C = C.copy(); T = T.copy(); dt = np.array(dt, dtype=np.float64); t = np.array(t, dtype=np.float64)
    t_ign = np.full(ld, np.nan) if t_ign is None else np.array(t_ign, dtype=np.float64)
    T0 = T.copy() if T0 is None else np.asarray(T0, dtype=np.float64)
    accepted = np.zeros(ld, dtype=np.int64); err_last = np.zeros(ld)
    for _a in range(n_attempts):
        Cn, Tn = C.copy(), T.copy()
        h = np.zeros(ld); h[:n] = np.minimum(dt[:n], np.maximum(t_end - t[:n], 0.0))
        with np.errstate(all="ignore"):
            for _m in range(newton_iters):
                ev = evaluate(om, C, T, n, want_jac=True); en = evaluate_energy(om, C, T, n)
                b = np.zeros((N + 1, ld))
                b[:N, :n] = (Cn[:, :n] - C[:, :n]) + h[:n] * ev["wdot"][:, :n]
                b[N, :n] = (Tn[:n] - T[:n]) + h[:n] * en["tdot"][:n]
                x = newton_solve(np.ascontiguousarray(ev["jac"]), np.ascontiguousarray(en["erow"]), np.ascontiguousarray(h), b, n)["x"]
                if _m == newton_iters - 1:
                    eC = (np.abs(x[:N, :n]) / (atol_C + rtol * np.abs(C[:, :n]))).max(0)
                    eT = np.abs(x[N, :n]) / (atol_T + rtol * np.abs(T[:n]))
                    err = np.where(np.isnan(eC) | np.isnan(eT), np.inf, np.maximum(eC, eT))
                C[:, :n] = np.maximum(C[:, :n] + x[:N, :n], 0.0)
                T[:n] = T[:n] + x[N, :n]
            ok = (err <= 1.0) & np.isfinite(C[:, :n]).all(0) & np.isfinite(T[:n]) & (T[:n] > 0.0)
        if trace is not None:
            trace.append(err.copy())
        err_last[:n] = err
        rej = ~ok
        C[:, :n][:, rej] = Cn[:, :n][:, rej]; T[:n][rej] = Tn[:n][rej]
        t[:n] = np.where(ok, t[:n] + h[:n], t[:n])
        dt[:n] = np.where(ok, grow * dt[:n], shrink * dt[:n])
        accepted[:n] += ok
        ign = ok & np.isnan(t_ign[:n]) & (T[:n] - T0[:n] >= dT_ign)
        t_ign[:n] = np.where(ign, t[:n], t_ign[:n])
    return dict(C=C, T=T, dt=dt, t=t, t_ign=t_ign, accepted=accepted, err_last=err_last)


def rate_constants(om: OracleMech, C1: np.ndarray, T: float):
    C1 = np.ascontiguousarray(C1, dtype=np.float64)
    kf = np.zeros(om.M); kb = np.zeros(om.M)
    rc = lib().oracle_rate_constants(om._ptr(), _p(C1), float(T), _p(kf), _p(kb))
    if rc != 0:
        raise RuntimeError("oracle_rate_constants failed")
    return kf, kb


def closure_check(om: OracleMech, C1: np.ndarray, T: float):
    C1 = np.ascontiguousarray(C1, dtype=np.float64)
    n = max(om.Nq, 1)
    y = np.zeros(n); res = np.zeros(n); sc = np.zeros(n)
    rc = lib().oracle_closure_check(om._ptr(), _p(C1), float(T), _p(y), _p(res), _p(sc))
    if rc != 0:
        raise RuntimeError("oracle_closure_check failed")
    return y[:om.Nq], res[:om.Nq], sc[:om.Nq]


def max_threads() -> int:
    return int(lib().oracle_max_threads())
