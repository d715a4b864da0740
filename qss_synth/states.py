"""Seeded synthetic cell states (C [mol/m^3], T [K]) in the SoA, cell-innermost layout.

Recipe: SURVEY.md section 8(d) / DESIGN.md "Input recipe". cfg1/2/3/5: T ~ U[800,2500] K, P ~ U[1,50] atm,
mole fractions log-uniform 1e-12..1 renormalised. cfg4: 128^3 multipulse-ignition-shaped field
(PAPER.md L381 describes the real case, which is not available).
"""
from __future__ import annotations

import numpy as np

from .mechanism import CONFIGS, Mechanism, config_mechanism

R_GAS = 8.31446261815324   # J/(mol K)
ATM = 101325.0             # Pa


def _pad(n_cells: int, align: int = 32) -> int:
    return (n_cells + align - 1) // align * align


def make_states(n_nqss: int, n_cells: int, seed: int, ld: int | None = None,
                T_range=(800.0, 2500.0), P_range_atm=(1.0, 50.0), logx_range=(-12.0, 0.0)):
    """Returns C [n_nqss, ld] and T [ld] (float64, C-contiguous). Padding cells (c >= n_cells) hold a
    benign state (copy of cell 0) so kernels may touch them."""
    ld = _pad(n_cells) if ld is None else ld
    rng = np.random.default_rng(seed)
    T = rng.uniform(T_range[0], T_range[1], size=n_cells)
    P = rng.uniform(P_range_atm[0], P_range_atm[1], size=n_cells) * ATM
    X = 10.0 ** rng.uniform(logx_range[0], logx_range[1], size=(n_nqss, n_cells))
    X /= X.sum(axis=0, keepdims=True)
    C = np.empty((n_nqss, ld)); Tp = np.empty(ld)
    C[:, :n_cells] = X * (P / (R_GAS * T))[None, :]
    Tp[:n_cells] = T
    if ld > n_cells:
        C[:, n_cells:] = C[:, :1]; Tp[n_cells:] = Tp[0]
    return C, Tp


def make_field_states(n_nqss: int, n: int, seed: int, n_kernels: int = 8):
    """cfg4-shaped field on an n^3 grid, x fastest: 750 K background + Gaussian hot kernels, 40 atm,
    premixed fuel/oxidiser/diluent base composition, products scaled by the local T excess, log-uniform
    radicals."""
    rng = np.random.default_rng(seed)
    n_cells = n ** 3
    Tk = rng.uniform(1800.0, 2600.0, size=n_kernels)
    rho = rng.uniform(4.0, 12.0, size=n_kernels) * (n / 128.0)
    ctr = rng.uniform(0.0, n, size=(n_kernels, 3))
    ax = np.arange(n, dtype=np.float64) + 0.5
    T = np.full((n, n, n), 750.0)            # index order [z][y][x]
    for k in range(n_kernels):
        gx = np.exp(-(ax - ctr[k, 0]) ** 2 / (2 * rho[k] ** 2))
        gy = np.exp(-(ax - ctr[k, 1]) ** 2 / (2 * rho[k] ** 2))
        gz = np.exp(-(ax - ctr[k, 2]) ** 2 / (2 * rho[k] ** 2))
        T += (Tk[k] - 750.0) * gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
    T = np.minimum(T, 3000.0).reshape(-1)
    theta = np.clip((T - 750.0) / 1850.0, 0.0, 1.0)
    X = np.empty((n_nqss, n_cells))
    X[0] = 0.02 * (1.0 - theta)                          # fuel
    X[1] = 0.20 * (1.0 - theta) + 0.01                   # oxidiser
    X[2] = 0.75                                          # diluent
    X[3] = 0.10 * theta + 1e-12                          # products
    X[4] = 0.10 * theta + 1e-12
    X[0] += 1e-12
    for k in range(5, n_nqss):                           # radicals
        X[k] = 10.0 ** rng.uniform(-12.0, -3.0, size=n_cells)
    X /= X.sum(axis=0, keepdims=True)
    P = 40.0 * ATM
    C = X * (P / (R_GAS * T))[None, :]
    return np.ascontiguousarray(C), np.ascontiguousarray(T)


def config_states(cfg: int, n_cells: int | None = None):
    """States of BASELINE.json config `cfg` (state seed = 1000 + cfg). `n_cells` truncates/overrides the
    config's cell count (cfg4: grid edge n = round(n_cells^(1/3)))."""
    mech: Mechanism = config_mechanism(cfg)
    full = CONFIGS[cfg]["n_cells"]
    n_cells = full if n_cells is None else n_cells
    if cfg == 4:
        n = int(round(n_cells ** (1.0 / 3.0)))
        return make_field_states(mech.n_nqss, n, 1000 + cfg)
    return make_states(mech.n_nqss, n_cells, 1000 + cfg)
