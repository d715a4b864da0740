"""Parity gates (SURVEY.md section 8(c) "Gates").

north_star: relative 1e-10 on wdot, normwise relative 1e-9 on the Jacobian. Made precise as two tiers:
  tier 1 (strict, no guard) must hold for >= 99 % of the items of a config;
  tier 2 (guarded by the running-error scales S and J_scale of the oracle) must hold for 100 %.
The Jacobian is gated per cell (Frobenius, Eq. 10) AND per column (the whole-matrix norm cannot
see the T column).
"""
from __future__ import annotations

import numpy as np

WDOT_RTOL, WDOT_GUARD = 1e-10, 1e-13
JAC_RTOL, JAC_GUARD = 1e-9, 1e-12
TIER1_MIN_FRACTION = 0.99
COL_COND_MAX = 1e3
WDOT_COND_MAX = 1e4


def wdot_gates(w, w_ref, S, n_cells=None):
    n = w_ref.shape[1] if n_cells is None else n_cells
    w, w_ref, S = w[:, :n], w_ref[:, :n], S[:, :n]
    d = np.abs(w - w_ref)
    finite = np.isfinite(w).all()
    # an entry whose value is a cancellation residue (S > COND_MAX |w|) loses >= 4 digits in ANY fp64
    # evaluation (the oracle itself misses 1e-10 there against its float128 referee, e.g. toy3 species D at
    # |w|/S = 1e-12); strict tier 1 is taken over the well-conditioned entries, tier 2 covers every entry.
    well = S <= WDOT_COND_MAX * np.abs(w_ref)
    t1 = (d <= WDOT_RTOL * np.abs(w_ref))[well]
    bound2 = WDOT_RTOL * np.abs(w_ref) + WDOT_GUARD * S
    t2 = d <= bound2
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio2 = np.where(bound2 > 0, d / bound2, np.where(d == 0, 0.0, np.inf))
    t1_all = d <= WDOT_RTOL * np.abs(w_ref)
    return dict(finite=bool(finite), tier1_frac=float(t1.mean()) if t1.size else 1.0,
                tier1_frac_unfiltered=float(t1_all.mean()) if t1_all.size else 1.0,
                wellcond_frac=float(well.mean()) if well.size else 1.0,
                tier2_all=bool(t2.all()), tier2_worst=float(ratio2.max()) if ratio2.size else 0.0)


def jac_gates(J, J_ref, J_scale, n_cells=None):
    """J arrays [N, N+1, ld]."""
    n = J_ref.shape[2] if n_cells is None else n_cells
    J, J_ref, J_scale = J[:, :, :n], J_ref[:, :, :n], J_scale[:, :, :n]
    finite = np.isfinite(J).all()
    d2 = (J - J_ref) ** 2
    # per cell (Frobenius)
    dF = np.sqrt(d2.sum((0, 1))); rF = np.sqrt((J_ref ** 2).sum((0, 1))); sF = np.sqrt((J_scale ** 2).sum((0, 1)))
    # per (cell, column)
    dC = np.sqrt(d2.sum(0)); rC = np.sqrt((J_ref ** 2).sum(0)); sC = np.sqrt((J_scale ** 2).sum(0))
    out = dict(finite=bool(finite))
    for name, d, r, s in (("cell", dF, rF, sF), ("col", dC, rC, sC)):
        t1 = d <= JAC_RTOL * r
        if name == "col":
            # a column whose norm is a cancellation residue (||J_scale|| > COND_MAX ||J||) carries no
            # digits in ANY fp64 evaluation; strict tier 1 is taken over the well-conditioned columns,
            # the guarded tier 2 still covers every column.
            well = s <= COL_COND_MAX * r
            out["col_wellcond_frac"] = float(well.mean()) if well.size else 1.0
            out["col_tier1_frac_unfiltered"] = float(t1.mean()) if t1.size else 1.0
            t1 = t1[well]
        b2 = JAC_RTOL * r + JAC_GUARD * s
        with np.errstate(divide="ignore", invalid="ignore"):
            ratio2 = np.where(b2 > 0, d / b2, np.where(d == 0, 0.0, np.inf))
            rel = np.where(r > 0, d / r, 0.0)
        out[f"{name}_tier1_frac"] = float(t1.mean()) if t1.size else 1.0
        out[f"{name}_tier2_all"] = bool((d <= b2).all())
        out[f"{name}_tier2_worst"] = float(ratio2.max()) if ratio2.size else 0.0
        out[f"{name}_rel_median"] = float(np.median(rel)) if rel.size else 0.0
        out[f"{name}_rel_max"] = float(rel.max()) if rel.size else 0.0
    # T column on its own
    relT = np.where(rC[-1] > 0, dC[-1] / np.where(rC[-1] > 0, rC[-1], 1.0), 0.0)
    out["Tcol_rel_median"] = float(np.median(relT)) if relT.size else 0.0
    return out


# Floors under the well-conditioned filter of tier 1 (reading G16): the filter depends on the ORACLE's data only
# (S, w_ref, J_scale, J_ref), so a change that inflated the scales and hollowed out tier 1 would trip these.
# Values: the fractions measured on the oracle (cfg1/2/3/5: wdot 0.987-0.996, columns 0.83-0.99; cfg4, the cold
# 750 K background of the field where forward and reverse rates cancel: 0.96 / 0.48) minus a margin.
WELLCOND_FLOOR = {1: (0.97, 0.75), 2: (0.97, 0.75), 3: (0.97, 0.75), 4: (0.93, 0.40), 5: (0.97, 0.75)}


def assert_wdot(w, w_ref, S, n_cells=None, what="wdot", cfg=None):
    g = wdot_gates(w, w_ref, S, n_cells)
    assert g["finite"], f"{what}: non-finite values"
    if cfg in WELLCOND_FLOOR:
        assert g["wellcond_frac"] >= WELLCOND_FLOOR[cfg][0], f"{what}: well-conditioned fraction {g['wellcond_frac']:.4f} under its floor"
    assert g["tier1_frac"] >= TIER1_MIN_FRACTION, f"{what}: tier-1 pass fraction {g['tier1_frac']:.5f} < 0.99 ({g})"
    assert g["tier2_all"], f"{what}: tier-2 violated, worst ratio {g['tier2_worst']:.3g} ({g})"
    return g


def assert_jac(J, J_ref, J_scale, n_cells=None, what="jac", cfg=None):
    g = jac_gates(J, J_ref, J_scale, n_cells)
    assert g["finite"], f"{what}: non-finite values"
    if cfg in WELLCOND_FLOOR:
        assert g["col_wellcond_frac"] >= WELLCOND_FLOOR[cfg][1], f"{what}: well-conditioned column fraction {g['col_wellcond_frac']:.4f} under its floor"
    for k in ("cell", "col"):
        assert g[f"{k}_tier1_frac"] >= TIER1_MIN_FRACTION, f"{what}: {k} tier-1 fraction {g[f'{k}_tier1_frac']:.5f} ({g})"
        assert g[f"{k}_tier2_all"], f"{what}: {k} tier-2 violated, worst {g[f'{k}_tier2_worst']:.3g} ({g})"
    return g
