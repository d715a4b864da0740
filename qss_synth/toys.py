"""Small hand-built mechanisms for closed-form pins and edge cases (SURVEY.md section 8(c) "Pins").

Thermo of the toys: every species shares a1..a6 and differs only in a7, so for a reaction with
sum(nu) = 0 the equilibrium constant is exactly Kc = exp(sum_s nu_s a7_s) (the polynomial parts of
h/RT and s/R cancel) -- a closed form the tests can state without evaluating any NASA polynomial.
"""
from __future__ import annotations

import numpy as np

from .mechanism import Mechanism, assemble, make_mechanism, T_LOW, T_MID, T_HIGH

_COMMON = np.array([4.0, 1.0e-3, -2.0e-7, 0.0, 0.0, -1.0e3])


def _toy_thermo(a7):
    n = len(a7)
    lo = np.zeros((n, 7)); lo[:, :6] = _COMMON; lo[:, 6] = a7
    hi = lo.copy()
    nasa_T = np.tile(np.array([T_LOW, T_MID, T_HIGH]), (n, 1))
    return nasa_T, lo, hi


def _arr(k, beta=0.0, Ea=0.0):
    return (float(k), float(beta), float(Ea))


def toy1(k1f=3.0e3, k2f=7.0e2, a7=(1.0, 0.4, 2.2), beta=(0.0, 0.0), Ea=(0.0, 0.0)) -> Mechanism:
    """A <=> Q (k1f), Q <=> B (k2f); A, B transported, Q QSS. north_star's 3-species 2-reaction toy."""
    comp = [[1], [1], [1]]                               # A, B, Q  (isomers)
    T, lo, hi = _toy_thermo(np.array(a7))
    rx = [dict(reac=[(0, 1)], prod=[(2, 1)], arr=_arr(k1f, beta[0], Ea[0])),
          dict(reac=[(2, 1)], prod=[(1, 1)], arr=_arr(k2f, beta[1], Ea[1]))]
    return assemble(2, 1, comp, T, lo, hi, rx, elem_weight=[12.011])


def toy2(k1f=3.0e3, k2f=5.0e4, k3f=7.0e2, a7=(1.0, 0.4, 2.2, 1.7)) -> Mechanism:
    """A <=> Q1, Q1 <=> Q2, Q2 <=> B: one coupled QSS group of size 2."""
    comp = [[1]] * 4                                     # A, B, Q1, Q2
    T, lo, hi = _toy_thermo(np.array(a7))
    rx = [dict(reac=[(0, 1)], prod=[(2, 1)], arr=_arr(k1f)),
          dict(reac=[(2, 1)], prod=[(3, 1)], arr=_arr(k2f)),
          dict(reac=[(3, 1)], prod=[(1, 1)], arr=_arr(k3f))]
    return assemble(2, 2, comp, T, lo, hi, rx, elem_weight=[12.011])


def toy3(k1f=4.0e2, k2f=9.0e3, a7=(1.0, 0.4, 0.9, 1.3, 2.0)) -> Mechanism:
    """A + B <=> Q + D, Q <=> E (bimolecular); transported A, B, D, E; QSS Q."""
    comp = [[1, 0], [0, 1], [0, 1], [1, 0], [1, 0]]      # A, B, D, E, Q
    T, lo, hi = _toy_thermo(np.array(a7))
    rx = [dict(reac=[(0, 1), (1, 1)], prod=[(4, 1), (2, 1)], arr=_arr(k1f)),
          dict(reac=[(4, 1)], prod=[(3, 1)], arr=_arr(k2f))]
    return assemble(4, 1, comp, T, lo, hi, rx, elem_weight=[12.011, 1.008])


def toy_dag(seed: int = 7) -> Mechanism:
    """Exercises: one-sided (dir_mask) reactions giving a DAG of QSS groups whose natural index order is
    NOT topological, one genuine SCC of size 2, a QSS species on both sides of a reaction, a
    stoichiometric coefficient 2, third-body and Troe reactions touching QSS species."""
    rng = np.random.default_rng(seed)
    # transported A B C D (0..3); QSS stored in the order Q3 Q5 Q1 Q4 Q2 -> indices 4..8
    A, B, C, D = 0, 1, 2, 3
    Q3, Q5, Q1, Q4, Q2 = 4, 5, 6, 7, 8
    comp = [[1]] * 4 + [[1]] * 5
    comp[C] = [2]                                        # C is a dimer: C <=> 2A style reactions balance
    a7 = rng.uniform(0.0, 2.0, size=9)
    T, lo, hi = _toy_thermo(a7)
    lo[:, 0] += rng.uniform(-0.5, 0.5, size=9)           # break the common-polynomial degeneracy a little
    hi[:, 0] = lo[:, 0]
    def k():
        return 10.0 ** rng.uniform(2.0, 5.0)
    def ar():
        return (k(), rng.uniform(-1.0, 1.0), rng.uniform(0.0, 2.0e4))
    rx = [
        dict(reac=[(A, 1)], prod=[(Q1, 1)], arr=ar()),
        dict(reac=[(Q1, 1)], prod=[(Q2, 1)], arr=ar(), dir_mask=1),                 # Q1 -> Q2 only
        dict(reac=[(Q2, 1)], prod=[(B, 1)], arr=ar()),
        dict(reac=[(Q2, 1), (A, 1)], prod=[(Q3, 1), (D, 1)], arr=ar(), dir_mask=1),  # Q2 -> Q3 only
        dict(reac=[(Q3, 1)], prod=[(D, 1)], arr=ar()),
        dict(reac=[(A, 1), (Q3, 1)], prod=[(B, 1), (Q3, 1)], arr=ar()),              # same QSS both sides
        dict(reac=[(C, 1)], prod=[(A, 2)], arr=ar()),                                # nu = 2, sum nu = +1
        dict(reac=[(C, 1)], prod=[(Q1, 1), (B, 1)], arr=ar(), type=1,
             eff=[(A, 2.5), (D, 0.7)]),
        dict(reac=[(B, 1)], prod=[(Q3, 1)], arr=ar(), type=2,
             arr_low=(k() * 1e-2, rng.uniform(-1.0, 1.0), rng.uniform(0.0, 2.0e4)),
             troe=(0.6, 120.0, 1500.0, 5000.0), eff=[(C, 3.0)]),
        dict(reac=[(Q3, 1)], prod=[(Q4, 1)], arr=ar(), dir_mask=1),                 # Q3 -> Q4 only
        dict(reac=[(Q4, 1)], prod=[(Q5, 1)], arr=ar()),                             # SCC {Q4, Q5}
        dict(reac=[(Q5, 1)], prod=[(A, 1)], arr=ar()),
        dict(reac=[(Q4, 1), (B, 1)], prod=[(A, 2)], arr=ar(), dir_mask=2),           # reverse only: 2A -> Q4 + B
        dict(reac=[(D, 1)], prod=[(B, 1)], arr=ar(), type=1, eff=[(B, 1.8)]),        # no QSS species
    ]
    return assemble(4, 5, comp, T, lo, hi, rx, elem_weight=[12.011])


def toy_nonqss(seed: int = 11) -> Mechanism:
    """A mechanism with no QSS species at all (textbook non-QSS analytic Jacobian)."""
    return make_mechanism(8, 0, 24, 1, True, seed)
