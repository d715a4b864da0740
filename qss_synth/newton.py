"""Seeded synthetic inputs of the Newton solve (NEXT-2): per-cell Jacobian-shaped matrices, step factors and right-hand sides.

No arithmetic of the method: random arrays with the SHAPE of a chemical Jacobian (Table 4: 36-49 % fill of
the species block; dense temperature column and energy row; negative diagonal; entries spread over many decades) in the SoA
layout of the library, `gamma` such that `gamma * max|J|` spans [1e-2, 1e3] (from "explicit would do" to strongly stiff), and a
right-hand side of mixed signs.  Stand-in for Jacobians of the paper's mechanisms, which are not available; the tests also
feed the solve with Jacobians the oracle evaluates on the synthetic mechanisms.
"""
from __future__ import annotations

import numpy as np

FILL = 0.45
DECADES = 8.0


def newton_inputs(N: int, ncells: int, seed: int, ld: int | None = None, with_energy: bool = True):
    """Returns dict(jac [N, N+1, ld], erow [N+1, ld] or None, gamma [ld], b [n, ld]) as numpy float64; paddings are NaN."""
    ld = ncells if ld is None else ld
    rng = np.random.default_rng(seed)
    n = N + 1 if with_energy else N

    def block(rows):
        mag = 10.0 ** rng.uniform(0.0, DECADES, size=(rows, N + 1, ncells))
        sgn = np.where(rng.random((rows, N + 1, ncells)) < 0.5, -1.0, 1.0)
        keep = rng.random((rows, N + 1, ncells)) < FILL
        return mag * sgn * keep

    jac = np.full((N, N + 1, ld), np.nan)
    J = block(N)
    J[:, N, :] = 10.0 ** rng.uniform(0.0, DECADES - 2.0, size=(N, ncells)) * np.where(rng.random((N, ncells)) < 0.5, -1.0, 1.0)
    i = np.arange(N)
    J[i, i, :] = -(10.0 ** rng.uniform(DECADES - 3.0, DECADES, size=(N, ncells)))
    jac[:, :, :ncells] = J
    erow = None
    if with_energy:
        erow = np.full((N + 1, ld), np.nan)
        erow[:, :ncells] = 10.0 ** rng.uniform(0.0, DECADES, size=(N + 1, ncells)) * np.where(rng.random((N + 1, ncells)) < 0.5, -1.0, 1.0)
    amax = np.abs(J).max((0, 1)) if ncells else np.zeros(0)
    gamma = np.full(ld, np.nan)
    gamma[:ncells] = 10.0 ** rng.uniform(-2.0, 3.0, size=ncells) / amax
    b = np.full((n, ld), np.nan)
    b[:, :ncells] = rng.normal(size=(n, ncells)) * 10.0 ** rng.uniform(-3.0, 3.0, size=(n, ncells))
    return dict(jac=jac, erow=erow, gamma=gamma, b=b)


def newton_inputs_torch(N: int, ncells: int, seed: int, device, with_energy: bool = True):
    """The same recipe drawn with torch's generator on `device` (for the full-size cases: 10 GB of Jacobians are not drawn on the
    host).  Not bit-identical to `newton_inputs`; ld = ncells."""
    import torch
    g = torch.Generator(device=device); g.manual_seed(seed)
    f64 = dict(dtype=torch.float64, device=device, generator=g)
    n = N + 1 if with_energy else N

    def signed(shape, lo, hi):
        out = torch.rand(shape, **f64).mul_(hi - lo).add_(lo).mul_(np.log(10.0)).exp_()
        out.mul_(torch.rand(shape, **f64).lt_(0.5).mul_(2.0).sub_(1.0))
        return out

    jac = signed((N, N + 1, ncells), 0.0, DECADES)
    jac.mul_(torch.rand((N, N + 1, ncells), **f64).lt_(FILL))
    jac[:, N, :] = signed((N, ncells), 0.0, DECADES - 2.0)
    i = torch.arange(N, device=device)
    jac[i, i, :] = -signed((N, ncells), DECADES - 3.0, DECADES).abs_()
    erow = signed((N + 1, ncells), 0.0, DECADES) if with_energy else None
    amax = jac.abs().amax((0, 1))
    gamma = torch.rand(ncells, **f64).mul_(5.0).sub_(2.0).mul_(np.log(10.0)).exp_() / amax
    b = torch.randn((n, ncells), **f64) * torch.rand((n, ncells), **f64).mul_(6.0).sub_(3.0).mul_(np.log(10.0)).exp_()
    return dict(jac=jac, erow=erow, gamma=gamma, b=b)
