"""paper_2405_05974_b200 -- thin Python binding of libqss (include/qss.h).

Argument marshalling only: every step of the hot path (rate constants, QSS closure, wdot, analytical
Jacobian; Eq. 2-4, 6, 7, 9) runs in the CUDA kernels of csrc/.  PyTorch is used for device memory
and streams.  There is no CPU fallback: importing works without a GPU (so the ABI can be checked), but
creating a mechanism or evaluating anything requires a CUDA device and the built library.
"""
from __future__ import annotations

import ctypes as ct
import os

import numpy as np

from . import build as _build

__all__ = ["lib", "QssMech", "QssError", "EXPORTS", "STATUS"]

EXPORTS = ["qss_mech_create", "qss_mech_validate", "qss_mech_specialise_check", "qss_mech_destroy", "qss_mech_info", "qss_mech_qss_order", "qss_eval_wdot",
           "qss_eval_jac", "qss_eval_jac_approx", "qss_eval_energy", "qss_newton_solve", "qss_newton_specialise_check", "qss_bdf1_workspace_bytes", "qss_bdf1_advance", "qss_ignition_advance", "qss_jac_fdt_workspace_bytes", "qss_eval_jac_fdt", "qss_mech_jac_pattern", "qss_jac_pack", "qss_jac_to_aos", "qss_eval_jac_full", "qss_eval_wdot_static", "qss_bench_species_sums", "qss_host_scratch_bytes", "qss_eval_jac_host", "qss_bench_dfma", "qss_last_error"]
STATUS = {0: "QSS_OK", -1: "QSS_E_INVALID", -2: "QSS_E_QUADRATIC", -3: "QSS_E_QSS_FANOUT", -4: "QSS_E_NO_SINK",
          -5: "QSS_E_UNSUPPORTED", -6: "QSS_E_CUDA", -7: "QSS_E_UNBALANCED"}


class QssError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class _Desc(ct.Structure):
    _fields_ = [("n_elem", ct.c_int32), ("n_nqss", ct.c_int32), ("n_qss", ct.c_int32), ("n_reac", ct.c_int32),
                ("elem_weight", ct.c_void_p), ("comp", ct.c_void_p),
                ("nasa_T", ct.c_void_p), ("nasa_lo", ct.c_void_p), ("nasa_hi", ct.c_void_p),
                ("type", ct.c_void_p), ("dir_mask", ct.c_void_p),
                ("reac_ptr", ct.c_void_p), ("reac_sp", ct.c_void_p), ("reac_nu", ct.c_void_p),
                ("prod_ptr", ct.c_void_p), ("prod_sp", ct.c_void_p), ("prod_nu", ct.c_void_p),
                ("arr", ct.c_void_p), ("arr_low", ct.c_void_p), ("troe", ct.c_void_p),
                ("eff_ptr", ct.c_void_p), ("eff_sp", ct.c_void_p), ("eff_val", ct.c_void_p),
                ("strict_balance", ct.c_int32)]


class _Info(ct.Structure):
    _fields_ = [("n_nqss", ct.c_int32), ("n_qss", ct.c_int32), ("n_reac", ct.c_int32),
                ("n_groups", ct.c_int32), ("max_group", ct.c_int32), ("n_levels", ct.c_int32),
                ("group_size", ct.c_int32 * 64),
                ("slots_wdot", ct.c_double), ("slots_jac", ct.c_double),
                ("bytes_wdot", ct.c_double), ("bytes_jac", ct.c_double),
                ("workspace_bytes_wdot", ct.c_size_t), ("workspace_bytes_jac", ct.c_size_t),
                ("kernel_variant_wdot", ct.c_int32), ("kernel_variant_jac", ct.c_int32)]


_lib = None


def lib():
    """Loads (building first if the sources are newer) libqss.so. Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ct.CDLL(path)
        vp, i64 = ct.c_void_p, ct.c_int64
        L.qss_mech_create.restype = ct.c_int; L.qss_mech_create.argtypes = [vp, ct.c_int, ct.POINTER(vp)]
        L.qss_mech_validate.restype = ct.c_int; L.qss_mech_validate.argtypes = [vp, vp, vp, vp]
        L.qss_mech_specialise_check.restype = ct.c_int; L.qss_mech_specialise_check.argtypes = [vp, ct.c_int, ct.c_int, vp]
        L.qss_mech_destroy.restype = ct.c_int; L.qss_mech_destroy.argtypes = [vp]
        L.qss_mech_info.restype = ct.c_int; L.qss_mech_info.argtypes = [vp, ct.POINTER(_Info)]
        L.qss_mech_qss_order.restype = ct.c_int; L.qss_mech_qss_order.argtypes = [vp, vp, vp]
        L.qss_eval_wdot.restype = ct.c_int; L.qss_eval_wdot.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, ct.c_size_t, vp]
        L.qss_eval_jac.restype = ct.c_int; L.qss_eval_jac.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, ct.c_size_t, vp]
        L.qss_eval_jac_approx.restype = ct.c_int; L.qss_eval_jac_approx.argtypes = [vp, i64, i64, vp, vp, vp, ct.c_int, vp, ct.c_size_t, vp]
        L.qss_eval_energy.restype = ct.c_int; L.qss_eval_energy.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp, vp]
        L.qss_newton_solve.restype = ct.c_int; L.qss_newton_solve.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp]
        L.qss_bench_species_sums.restype = ct.c_int; L.qss_bench_species_sums.argtypes = [vp, ct.c_int, i64, i64, vp, vp, vp]
        L.qss_eval_wdot_static.restype = ct.c_int; L.qss_eval_wdot_static.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
        L.qss_eval_jac_full.restype = ct.c_int; L.qss_eval_jac_full.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp, vp, ct.c_size_t, vp]
        L.qss_mech_jac_pattern.restype = ct.c_int; L.qss_mech_jac_pattern.argtypes = [vp, ct.c_int, vp]
        L.qss_jac_pack.restype = ct.c_int; L.qss_jac_pack.argtypes = [vp, i64, i64, ct.c_int32, vp, vp, vp, vp]
        L.qss_jac_to_aos.restype = ct.c_int; L.qss_jac_to_aos.argtypes = [vp, i64, i64, vp, vp, ct.c_int, vp, vp]
        L.qss_ignition_advance.restype = ct.c_int
        L.qss_ignition_advance.argtypes = [vp, i64, i64, vp, vp, vp, vp, ct.c_double, vp, vp, ct.c_double, ct.c_int, ct.c_int, ct.c_double, ct.c_double, ct.c_double, vp, ct.c_size_t, vp]
        L.qss_jac_fdt_workspace_bytes.restype = ct.c_size_t; L.qss_jac_fdt_workspace_bytes.argtypes = [vp, i64]
        L.qss_eval_jac_fdt.restype = ct.c_int; L.qss_eval_jac_fdt.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, ct.c_size_t, vp]
        L.qss_bdf1_workspace_bytes.restype = ct.c_size_t; L.qss_bdf1_workspace_bytes.argtypes = [vp, i64]
        L.qss_bdf1_advance.restype = ct.c_int; L.qss_bdf1_advance.argtypes = [vp, i64, i64, vp, vp, vp, ct.c_int, ct.c_int, vp, ct.c_size_t, vp]
        L.qss_newton_specialise_check.restype = ct.c_int; L.qss_newton_specialise_check.argtypes = [ct.c_int, ct.c_int, ct.c_int, ct.c_int, vp]
        L.qss_host_scratch_bytes.restype = ct.c_size_t; L.qss_host_scratch_bytes.argtypes = [vp, i64, i64]
        L.qss_eval_jac_host.restype = ct.c_int; L.qss_eval_jac_host.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, ct.c_size_t, vp]
        L.qss_bench_dfma.restype = ct.c_int; L.qss_bench_dfma.argtypes = [ct.c_int, ct.c_int, vp, ct.POINTER(ct.c_double), vp]
        L.qss_last_error.restype = ct.c_char_p; L.qss_last_error.argtypes = []
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise QssError(rc, lib().qss_last_error().decode())


_DESC_SPEC = dict(elem_weight=np.float64, comp=np.int32, nasa_T=np.float64, nasa_lo=np.float64, nasa_hi=np.float64,
                  type=np.int32, dir_mask=np.uint8, reac_ptr=np.int32, reac_sp=np.int32, reac_nu=np.int32,
                  prod_ptr=np.int32, prod_sp=np.int32, prod_nu=np.int32, arr=np.float64, arr_low=np.float64,
                  troe=np.float64, eff_ptr=np.int32, eff_sp=np.int32, eff_val=np.float64)


def make_desc(mech, strict_balance=False):
    """qss_mech_desc_t from any object with the fields of qss_synth.Mechanism. Returns (desc, keepalive)."""
    d = _Desc()
    d.strict_balance = 1 if strict_balance else 0
    d.n_elem, d.n_nqss, d.n_qss, d.n_reac = int(mech.n_elem), int(mech.n_nqss), int(mech.n_qss), int(mech.n_reac)
    keep = {}
    for name, dt in _DESC_SPEC.items():
        src = getattr(mech, "rtype" if name == "type" else name)
        a = np.ascontiguousarray(src, dtype=dt)
        if a.size == 0:
            a = np.zeros(1, dtype=dt)
        keep[name] = a
        setattr(d, name, a.ctypes.data)
    return d, keep


def validate(mech, strict_balance=False):
    """Host-only validation + QSS solve order (no CUDA). Returns (n_groups, order, group_of)."""
    d, keep = make_desc(mech, strict_balance)
    ng = ct.c_int32()
    nq = max(int(mech.n_qss), 1)
    order = np.zeros(nq, dtype=np.int32); grp = np.zeros(nq, dtype=np.int32)
    _check(lib().qss_mech_validate(ct.addressof(d), ct.addressof(ng), order.ctypes.data, grp.ctypes.data))
    del keep
    return ng.value, order[:mech.n_qss], grp[:mech.n_qss]


def specialise_check(mech, cc=(10, 0)) -> int:
    """Host-only: generate the mechanism-specialised Jacobian kernel source and compile it with NVRTC for compute
    capability `cc` (no device needed). Returns the size of the device image in bytes."""
    d, keep = make_desc(mech)
    nbytes = ct.c_size_t()
    _check(lib().qss_mech_specialise_check(ct.addressof(d), int(cc[0]), int(cc[1]), ct.addressof(nbytes)))
    del keep
    return nbytes.value


def jac_pattern(mech, mode: int = 0):
    """Host-only: structural non-zero pattern [N, N+1] (uint8) of the Jacobian of `mode` (qss_mech_jac_pattern)."""
    import numpy as np
    d, keep = make_desc(mech)
    pat = np.zeros((mech.n_nqss, mech.n_nqss + 1), dtype=np.uint8)
    _check(lib().qss_mech_jac_pattern(ct.addressof(d), int(mode), pat.ctypes.data))
    del keep
    return pat


def newton_specialise_check(n_species: int, with_energy: bool = True, cc=(10, 0)) -> int:
    """Host-only: compile the Newton-solve kernel for a mechanism of `n_species` transported species with NVRTC (no device
    needed). Returns the size of the device image in bytes."""
    nbytes = ct.c_size_t()
    _check(lib().qss_newton_specialise_check(int(n_species), 1 if with_energy else 0, int(cc[0]), int(cc[1]), ct.addressof(nbytes)))
    return nbytes.value


def _ptr(t):
    return None if t is None else ct.c_void_p(t.data_ptr())


class QssMech:
    """A compiled mechanism on one CUDA device (qss_mech_create / qss_mech_destroy)."""

    def __init__(self, mech, device: int = 0, strict_balance: bool = False):
        self._h = ct.c_void_p()
        d, keep = make_desc(mech, strict_balance)
        _check(lib().qss_mech_create(ct.addressof(d), int(device), ct.byref(self._h)))
        del keep
        self.device = int(device)
        info = _Info()
        _check(lib().qss_mech_info(self._h, ct.byref(info)))
        self.info = info
        self.N, self.Nq, self.M = info.n_nqss, info.n_qss, info.n_reac
        self._ws = {}

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().qss_mech_destroy(self._h)
            self._h = ct.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def qss_order(self):
        order = np.zeros(max(self.Nq, 1), dtype=np.int32); grp = np.zeros(max(self.Nq, 1), dtype=np.int32)
        _check(lib().qss_mech_qss_order(self._h, order.ctypes.data, grp.ctypes.data))
        return order[:self.Nq], grp[:self.Nq]

    def group_sizes(self):
        return [int(self.info.group_size[g]) for g in range(min(self.info.n_groups, 64))]

    def workspace(self, jac: bool):
        """Scratch slab of the kernels, one per (call kind, CUDA stream): evaluations enqueued on two streams must not share it."""
        import torch
        key = (bool(jac), torch.cuda.current_stream().cuda_stream)
        if key not in self._ws:
            nbytes = self.info.workspace_bytes_jac if jac else self.info.workspace_bytes_wdot
            self._ws[key] = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=f"cuda:{self.device}")
        return self._ws[key]

    @staticmethod
    def _stream():
        import torch
        return ct.c_void_p(torch.cuda.current_stream().cuda_stream)

    def eval_wdot(self, C, T, ncells=None, wdot=None, cqss=None, want_cqss=False):
        """C [N, ld], T [ld] float64 CUDA tensors. Returns wdot [N, ld] (and cqss [Nq, ld])."""
        import torch
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        assert C.dtype == torch.float64 and T.dtype == torch.float64 and C.is_contiguous() and T.is_contiguous()
        assert C.shape[0] == self.N and T.shape[0] == ld
        if wdot is None:
            wdot = torch.empty((self.N, ld), dtype=torch.float64, device=C.device)
        if want_cqss and cqss is None:
            cqss = torch.empty((max(self.Nq, 1), ld), dtype=torch.float64, device=C.device)
        ws = self.workspace(False)
        _check(lib().qss_eval_wdot(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(wdot), _ptr(cqss), _ptr(ws),
                                   ws.numel(), self._stream()))
        return (wdot, cqss[:self.Nq]) if want_cqss else wdot

    def eval_jac(self, C, T, ncells=None, jac=None, wdot=None, want_wdot=False):
        """Returns jac [N, N+1, ld] (and wdot [N, ld])."""
        import torch
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        assert C.dtype == torch.float64 and T.dtype == torch.float64 and C.is_contiguous() and T.is_contiguous()
        assert C.shape[0] == self.N and T.shape[0] == ld
        if jac is None:
            jac = torch.empty((self.N, self.N + 1, ld), dtype=torch.float64, device=C.device)
        if want_wdot and wdot is None:
            wdot = torch.empty((self.N, ld), dtype=torch.float64, device=C.device)
        ws = self.workspace(True)
        _check(lib().qss_eval_jac(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(jac), _ptr(wdot), _ptr(ws),
                                  ws.numel(), self._stream()))
        return (jac, wdot) if want_wdot else jac

    def eval_jac_approx(self, C, T, mode, ncells=None, jac=None):
        """The paper's simplified Jacobians: mode 0 exact, 1 constant-QSS AJ, 2 zero-QSS AJ. Returns jac [N, N+1, ld]."""
        import torch
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        assert C.dtype == torch.float64 and T.dtype == torch.float64 and C.is_contiguous() and T.is_contiguous()
        if jac is None:
            jac = torch.empty((self.N, self.N + 1, ld), dtype=torch.float64, device=C.device)
        ws = self.workspace(True)
        _check(lib().qss_eval_jac_approx(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(jac), int(mode), _ptr(ws), ws.numel(), self._stream()))
        return jac

    def bench_species_sums(self, mode, Q, ncells=None, wdot=None):
        """Mapping micro-benchmark (qss_bench_species_sums): wdot [N, ld] = S Q from Q [M, ld]; mode 0 lane = cell, mode 1 warp per cell."""
        import torch
        ld = Q.shape[1]
        ncells = ld if ncells is None else int(ncells)
        assert Q.is_contiguous() and Q.shape[0] == self.info.n_reac
        if wdot is None:
            wdot = torch.empty((self.N, ld), dtype=torch.float64, device=Q.device)
        _check(lib().qss_bench_species_sums(self._h, int(mode), ncells, ld, _ptr(Q), _ptr(wdot), self._stream()))
        return wdot

    def eval_wdot_static(self, C, T, ncells=None, wdot=None, cqss=None):
        """wdot through the allocation-free entry point (qss_eval_wdot_static): `wdot` (and `cqss`) are the caller's tensors; no
        workspace is passed and nothing is allocated by the library.  Calls that overlap on the GPU race."""
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        assert wdot is not None and wdot.is_contiguous() and wdot.shape == (self.N, ld)
        _check(lib().qss_eval_wdot_static(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(wdot), _ptr(cqss), self._stream()))
        return wdot

    def eval_jac_full(self, C, T, ncells=None, jac=None, wdot=None, tdot=None, erow=None):
        """Full (N+1) x (N+1) Jacobian and both right-hand sides in one call (qss_eval_jac_full). Returns (jac, wdot, tdot, erow)."""
        import torch
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        f64 = dict(dtype=torch.float64, device=C.device)
        jac = torch.empty((self.N, self.N + 1, ld), **f64) if jac is None else jac
        wdot = torch.empty((self.N, ld), **f64) if wdot is None else wdot
        tdot = torch.empty((ld,), **f64) if tdot is None else tdot
        erow = torch.empty((self.N + 1, ld), **f64) if erow is None else erow
        ws = self.workspace(True)
        _check(lib().qss_eval_jac_full(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(jac), _ptr(wdot), _ptr(tdot), _ptr(erow), _ptr(ws), ws.numel(), self._stream()))
        return jac, wdot, tdot, erow

    def eval_energy(self, C, T, wdot, jac, ncells=None, tdot=None, erow=None):
        """Temperature right-hand side tdot [ld] and energy row erow [N+1, ld] of the full (N+1) x (N+1) Jacobian (qss_eval_energy)."""
        import torch
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        assert wdot.is_contiguous() and jac.is_contiguous() and wdot.shape == (self.N, ld) and jac.shape == (self.N, self.N + 1, ld)
        if tdot is None:
            tdot = torch.empty((ld,), dtype=torch.float64, device=C.device)
        if erow is None:
            erow = torch.empty((self.N + 1, ld), dtype=torch.float64, device=C.device)
        _check(lib().qss_eval_energy(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(wdot), _ptr(jac), _ptr(tdot), _ptr(erow), self._stream()))
        return tdot, erow

    def newton_solve(self, jac, erow, gamma, b, ncells=None, x=None):
        """x = (I - gamma J)^-1 b per cell (qss_newton_solve); J = [jac; erow], or the N x N species block when erow is None."""
        import torch
        ld = jac.shape[2]
        ncells = ld if ncells is None else int(ncells)
        n = self.N + (1 if erow is not None else 0)
        assert jac.is_contiguous() and jac.shape == (self.N, self.N + 1, ld) and b.is_contiguous() and b.shape == (n, ld)
        assert gamma.is_contiguous() and gamma.numel() >= ncells and (erow is None or (erow.is_contiguous() and erow.shape == (self.N + 1, ld)))
        if x is None:
            x = torch.empty((n, ld), dtype=torch.float64, device=jac.device)
        _check(lib().qss_newton_solve(self._h, ncells, ld, _ptr(jac), _ptr(erow), _ptr(gamma), _ptr(b), _ptr(x), self._stream()))
        return x

    def eval_jac_fdT(self, C, T, ncells=None, jac=None, wdot=None, want_wdot=False):
        """Jacobian with the temperature column by central finite differences of wdot (qss_eval_jac_fdt)."""
        import torch
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        if jac is None:
            jac = torch.empty((self.N, self.N + 1, ld), dtype=torch.float64, device=C.device)
        if wdot is None and want_wdot:
            wdot = torch.empty((self.N, ld), dtype=torch.float64, device=C.device)
        ws = torch.empty(int(lib().qss_jac_fdt_workspace_bytes(self._h, ld)), dtype=torch.uint8, device=C.device)
        _check(lib().qss_eval_jac_fdt(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(jac), _ptr(wdot), _ptr(ws), ws.numel(), self._stream()))
        return (jac, wdot) if want_wdot else jac

    def jac_pack(self, jac, idx, ncells=None, packed=None):
        """Rows idx (int32 CUDA tensor of i*(N+1)+k) of the dense Jacobian gathered into [len(idx), ld] (qss_jac_pack)."""
        import torch
        ld = jac.shape[2]
        ncells = ld if ncells is None else int(ncells)
        assert jac.is_contiguous() and idx.dtype == torch.int32 and idx.is_contiguous()
        if packed is None:
            packed = torch.empty((idx.numel(), ld), dtype=torch.float64, device=jac.device)
        _check(lib().qss_jac_pack(self._h, ncells, ld, idx.numel(), _ptr(idx), _ptr(jac), _ptr(packed), self._stream()))
        return packed

    def jac_to_aos(self, jac, erow=None, ncells=None, col_major=False, out=None):
        """One contiguous matrix per cell for external batched solvers (qss_jac_to_aos): [ncells, rows, N+1] row-major, or
        [ncells, N+1, rows] (the column-major matrix) when col_major; rows = N + 1 with the energy row, else N."""
        import torch
        ld = jac.shape[2]
        ncells = ld if ncells is None else int(ncells)
        rows = self.N + 1 if erow is not None else self.N
        assert jac.is_contiguous() and (erow is None or erow.is_contiguous())
        if out is None:
            out = torch.empty((ncells, self.N + 1, rows) if col_major else (ncells, rows, self.N + 1), dtype=torch.float64, device=jac.device)
        _check(lib().qss_jac_to_aos(self._h, ncells, ld, _ptr(jac), _ptr(erow), int(bool(col_major)), _ptr(out), self._stream()))
        return out

    def bdf1_advance(self, C, T, dt, nsub, newton_iters, ncells=None, workspace=None):
        """Advances (C, T) IN PLACE by `nsub` backward-Euler substeps of size dt per cell (qss_bdf1_advance)."""
        import torch
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        assert C.is_contiguous() and T.is_contiguous() and dt.is_contiguous() and C.shape == (self.N, ld) and T.shape == (ld,)
        need = int(lib().qss_bdf1_workspace_bytes(self._h, ld))
        if workspace is None or workspace.numel() < need:
            workspace = torch.empty(need, dtype=torch.uint8, device=C.device)
        _check(lib().qss_bdf1_advance(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(dt), int(nsub), int(newton_iters), _ptr(workspace), workspace.numel(), self._stream()))
        return workspace

    def ignition_advance(self, C, T, dt, t, t_end, n_attempts, newton_iters, ncells=None, t_ign=None, T0=None, dT_ign=400.0, rtol=1e-6,
                         atol_C=1e-12, atol_T=1e-6, workspace=None):
        """Adaptive backward-Euler attempts with ignition time (qss_ignition_advance); C, T, dt, t, t_ign are updated IN PLACE."""
        import torch
        ld = C.shape[1]
        ncells = ld if ncells is None else int(ncells)
        for a in (C, T, dt, t):
            assert a.is_contiguous() and a.dtype == torch.float64
        need = int(lib().qss_bdf1_workspace_bytes(self._h, ld))
        if workspace is None or workspace.numel() < need:
            workspace = torch.empty(need, dtype=torch.uint8, device=C.device)
        _check(lib().qss_ignition_advance(self._h, ncells, ld, _ptr(C), _ptr(T), _ptr(dt), _ptr(t), float(t_end), _ptr(t_ign), _ptr(T0), float(dT_ign),
                                          int(n_attempts), int(newton_iters), float(rtol), float(atol_C), float(atol_T), _ptr(workspace), workspace.numel(),
                                          self._stream()))
        return workspace

    def host_scratch_bytes(self, ncells, ld):
        return int(lib().qss_host_scratch_bytes(self._h, int(ncells), int(ld)))

    def eval_jac_host(self, C_host, T_host, jac_host, wdot_host, scratch, ncells=None):
        """End-to-end call on HOST (ideally pinned) torch tensors; `scratch` is a CUDA uint8 tensor."""
        ld = C_host.shape[1]
        ncells = ld if ncells is None else int(ncells)
        _check(lib().qss_eval_jac_host(self._h, ncells, ld, _ptr(C_host), _ptr(T_host), _ptr(jac_host),
                                       _ptr(wdot_host), _ptr(scratch), scratch.numel(), self._stream()))


def bench_dfma(blocks: int, iters: int, sink):
    """Launches the fp64-FMA micro-benchmark on the current stream; returns the number of lane-FMAs issued."""
    n = ct.c_double()
    import torch
    _check(lib().qss_bench_dfma(int(blocks), int(iters), _ptr(sink), ct.byref(n),
                                ct.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return n.value
