"""Seeded synthetic QSS mechanisms shaped like BASELINE.json's configs.

Recipe: SURVEY.md section 8(d) / DESIGN.md "Input recipe". Stands in for the paper's reduced mechanisms
(13-4-CH4, 35-18 n-dodecane, 55-33 n-heptane), which are not in this container.

Only data is produced here: element compositions, balanced reactions, Arrhenius / third-body / Troe
parameters, NASA-7 fits. No rate, closure or Jacobian arithmetic lives in this module.
"""
from __future__ import annotations

import dataclasses
import hashlib
import math
from typing import Dict, List, Tuple

import numpy as np

ELEM_WEIGHT = np.array([12.011, 1.008, 15.999, 14.007])  # C, H, O, N  (g/mol)
KCAL = 4184.0                                            # J per kcal
T_LOW, T_MID, T_HIGH = 300.0, 1000.0, 3500.0
T_REF = 298.15

# (n_nqss, n_qss, n_reac, g_max, typed, n_cells)  -- BASELINE.json configs[0..4] are cfg1..cfg5
CONFIGS: Dict[int, dict] = {
    1: dict(n_nqss=9, n_qss=3, n_reac=30, g_max=3, typed=False, n_cells=4096),
    2: dict(n_nqss=35, n_qss=18, n_reac=270, g_max=4, typed=True, n_cells=1 << 20),
    3: dict(n_nqss=60, n_qss=40, n_reac=600, g_max=6, typed=True, n_cells=1 << 19),
    4: dict(n_nqss=35, n_qss=18, n_reac=270, g_max=4, typed=True, n_cells=128 ** 3),  # cfg2's mechanism
    5: dict(n_nqss=150, n_qss=80, n_reac=1500, g_max=8, typed=True, n_cells=1 << 18),
}


@dataclasses.dataclass
class Mechanism:
    """Flat mechanism description (host numpy arrays), one field per array of the C-ABI description."""
    n_elem: int
    n_nqss: int
    n_qss: int
    n_reac: int
    elem_weight: np.ndarray   # [n_elem] f64
    comp: np.ndarray          # [n_sp, n_elem] i32, transported species first
    nasa_T: np.ndarray        # [n_sp, 3] f64  Tlow, Tmid, Thigh
    nasa_lo: np.ndarray       # [n_sp, 7] f64
    nasa_hi: np.ndarray       # [n_sp, 7] f64
    rtype: np.ndarray         # [n_reac] i32  0 Arrhenius, 1 third-body, 2 Troe falloff
    dir_mask: np.ndarray      # [n_reac] u8   bit0 forward, bit1 reverse
    reac_ptr: np.ndarray      # CSR reactants
    reac_sp: np.ndarray
    reac_nu: np.ndarray
    prod_ptr: np.ndarray      # CSR products
    prod_sp: np.ndarray
    prod_nu: np.ndarray
    arr: np.ndarray           # [n_reac, 3] A, beta, Ea[J/mol]   (high-pressure limit for type 2)
    arr_low: np.ndarray       # [n_reac, 3] low-pressure limit (type 2 only)
    troe: np.ndarray          # [n_reac, 4] alpha, T***, T*, T**  (type 2 only)
    eff_ptr: np.ndarray       # CSR non-unity third-body efficiencies (transported species only)
    eff_sp: np.ndarray
    eff_val: np.ndarray

    @property
    def n_sp(self) -> int:
        return self.n_nqss + self.n_qss

    def species_weight(self) -> np.ndarray:
        return self.comp.astype(np.float64) @ self.elem_weight

    def sha256(self) -> str:
        h = hashlib.sha256()
        for f in dataclasses.fields(self):
            v = getattr(self, f.name)
            h.update(f.name.encode())
            h.update(np.ascontiguousarray(v).tobytes() if isinstance(v, np.ndarray) else repr(v).encode())
        return h.hexdigest()

    def reaction_sides(self, j: int) -> Tuple[List[Tuple[int, int]], List[Tuple[int, int]]]:
        r = [(int(self.reac_sp[p]), int(self.reac_nu[p])) for p in range(self.reac_ptr[j], self.reac_ptr[j + 1])]
        p = [(int(self.prod_sp[q]), int(self.prod_nu[q])) for q in range(self.prod_ptr[j], self.prod_ptr[j + 1])]
        return r, p


def assemble(n_nqss: int, n_qss: int, comp, nasa_T, nasa_lo, nasa_hi, reactions, elem_weight=None) -> Mechanism:
    """Build a Mechanism from a python list of reaction dicts:
    {reac: [(sp, nu)..], prod: [(sp, nu)..], type, dir_mask, arr, arr_low, troe, eff: [(sp, val)..]}"""
    comp = np.asarray(comp, dtype=np.int32)
    n_elem = comp.shape[1]
    if elem_weight is None:
        elem_weight = ELEM_WEIGHT[:n_elem]
    M = len(reactions)
    reac_ptr, reac_sp, reac_nu = [0], [], []
    prod_ptr, prod_sp, prod_nu = [0], [], []
    eff_ptr, eff_sp, eff_val = [0], [], []
    arr = np.zeros((M, 3)); arr_low = np.zeros((M, 3)); troe = np.zeros((M, 4))
    rtype = np.zeros(M, dtype=np.int32); dmask = np.zeros(M, dtype=np.uint8)
    for j, r in enumerate(reactions):
        for s, nu in r["reac"]:
            reac_sp.append(s); reac_nu.append(nu)
        reac_ptr.append(len(reac_sp))
        for s, nu in r["prod"]:
            prod_sp.append(s); prod_nu.append(nu)
        prod_ptr.append(len(prod_sp))
        for s, v in r.get("eff", []):
            eff_sp.append(s); eff_val.append(v)
        eff_ptr.append(len(eff_sp))
        rtype[j] = r.get("type", 0)
        dmask[j] = r.get("dir_mask", 3)
        arr[j] = r["arr"]
        if "arr_low" in r:
            arr_low[j] = r["arr_low"]
        if "troe" in r:
            troe[j] = r["troe"]
    i32 = lambda a: np.asarray(a, dtype=np.int32)
    return Mechanism(
        n_elem=n_elem, n_nqss=n_nqss, n_qss=n_qss, n_reac=M,
        elem_weight=np.asarray(elem_weight, dtype=np.float64), comp=comp,
        nasa_T=np.asarray(nasa_T, dtype=np.float64), nasa_lo=np.asarray(nasa_lo, dtype=np.float64),
        nasa_hi=np.asarray(nasa_hi, dtype=np.float64), rtype=rtype, dir_mask=dmask,
        reac_ptr=i32(reac_ptr), reac_sp=i32(reac_sp), reac_nu=i32(reac_nu),
        prod_ptr=i32(prod_ptr), prod_sp=i32(prod_sp), prod_nu=i32(prod_nu),
        arr=arr, arr_low=arr_low, troe=troe,
        eff_ptr=i32(eff_ptr), eff_sp=i32(eff_sp), eff_val=np.asarray(eff_val, dtype=np.float64))


# ------------------------------------------------------------------------------------------------
# species
# ------------------------------------------------------------------------------------------------
def _draw_compositions(rng: np.random.Generator, n_sp: int) -> np.ndarray:
    n_base = math.ceil(n_sp / 4)
    comps: List[np.ndarray] = []
    count: Dict[tuple, int] = {}

    def try_add(c) -> None:
        if c.min() < 0 or c.max() > 4 or c.sum() == 0:
            return
        t = tuple(int(x) for x in c)
        if count.get(t, 0) >= 2:          # at most two isomers per composition
            return
        count[t] = count.get(t, 0) + 1
        comps.append(np.array(t, dtype=np.int64))

    while len(comps) < n_base:
        try_add(rng.integers(0, 3, size=4))
    guard = 0
    while len(comps) < n_sp:
        i, j = rng.integers(0, len(comps), size=2)
        c = comps[i] + comps[j] if rng.random() < 0.6 else comps[i] - comps[j]
        try_add(c)
        guard += 1
        if guard > 200000:
            raise RuntimeError("composition draw did not converge")
    comps_arr = np.stack(comps)
    return comps_arr[rng.permutation(n_sp)]


def draw_nasa(rng: np.random.Generator, comp: np.ndarray):
    """NASA-7 two-range fits with cp/R in [3.5, 12] on 300-3500 K, continuous (cp, h, s) at 1000 K."""
    n_sp, n_elem = comp.shape
    eta = rng.uniform(-2e4, 2e4, size=n_elem)            # element-additive enthalpy part [K]
    nasa_T = np.tile(np.array([T_LOW, T_MID, T_HIGH]), (n_sp, 1))
    lo = np.zeros((n_sp, 7)); hi = np.zeros((n_sp, 7))
    grid_lo = np.linspace(T_LOW, T_MID, 29); grid_hi = np.linspace(T_MID, T_HIGH, 51)

    def cp_coeffs(Ta, Tb, ua, ub, e, f, g):
        c1 = (ub - ua) / (Tb - Ta); c0 = ua - c1 * Ta
        return np.array([c0 + e * Ta * Tb,
                         c1 - e * (Ta + Tb) + f * Ta * Tb,
                         e - f * (Ta + Tb) + g * Ta * Tb,
                         f - g * (Ta + Tb),
                         g])

    def cp_eval(a, T):
        return a[0] + T * (a[1] + T * (a[2] + T * (a[3] + T * a[4])))

    def h_poly(a, T):   # h/R without a6
        return T * (a[0] + T * (a[1] / 2 + T * (a[2] / 3 + T * (a[3] / 4 + T * a[4] / 5))))

    def s_poly(a, T):   # s/R without a7
        return a[0] * math.log(T) + T * (a[1] + T * (a[2] / 2 + T * (a[3] / 3 + T * a[4] / 4)))

    for s in range(n_sp):
        u0 = rng.uniform(3.5, 6.0); u1 = rng.uniform(u0, 9.0); u2 = rng.uniform(u1, 12.0)
        amp = rng.uniform(-0.3, 0.3, size=2)
        skew = rng.uniform(-0.3, 0.3, size=2)
        quart = rng.uniform(-0.1, 0.1, size=2)
        for rng_i, (Ta, Tb, ua, ub, grid, dst) in enumerate(
                ((T_LOW, T_MID, u0, u1, grid_lo, lo), (T_MID, T_HIGH, u1, u2, grid_hi, hi))):
            e = amp[rng_i] * 4.0 / (Tb - Ta) ** 2
            f = e * skew[rng_i] / Tb
            g = e * quart[rng_i] / Tb ** 2
            for _ in range(60):
                a = cp_coeffs(Ta, Tb, ua, ub, e, f, g)
                v = cp_eval(a, grid)
                if v.min() >= 3.5 and v.max() <= 12.0:
                    break
                e *= 0.5; f *= 0.5; g *= 0.5
            else:
                a = cp_coeffs(Ta, Tb, ua, ub, 0.0, 0.0, 0.0)
            dst[s, :5] = a
        n_atoms = int(comp[s].sum())
        h298 = float(comp[s] @ eta) + rng.uniform(-1e4, 1e4)
        s298 = 20.0 + 2.5 * n_atoms + rng.uniform(-2.0, 2.0)
        lo[s, 5] = h298 - h_poly(lo[s], T_REF)
        lo[s, 6] = s298 - s_poly(lo[s], T_REF)
        hi[s, 5] = (h_poly(lo[s], T_MID) + lo[s, 5]) - h_poly(hi[s], T_MID)
        hi[s, 6] = (s_poly(lo[s], T_MID) + lo[s, 6]) - s_poly(hi[s], T_MID)
    return nasa_T, lo, hi


# ------------------------------------------------------------------------------------------------
# reactions
# ------------------------------------------------------------------------------------------------
def _enumerate_candidates(comp: np.ndarray, n_nqss: int):
    """Balanced candidates A<=>B, A<=>B+C, A+B<=>C+D (incl. 2A) with at most one QSS molecule per side
    and no species on both sides. Returned as (reactants, products) lists of (sp, nu)."""
    n_sp = comp.shape[0]
    is_q = np.arange(n_sp) >= n_nqss
    key = [tuple(int(x) for x in comp[s]) for s in range(n_sp)]

    def side(pair):
        a, b = pair
        return [(a, 2)] if a == b else [(a, 1), (b, 1)]

    def nq(pair):
        return int(is_q[pair[0]]) + int(is_q[pair[1]])

    by_comp: Dict[tuple, List[int]] = {}
    for s in range(n_sp):
        by_comp.setdefault(key[s], []).append(s)
    pair_sum: Dict[tuple, List[Tuple[int, int]]] = {}
    for a in range(n_sp):
        for b in range(a, n_sp):
            if nq((a, b)) > 1:
                continue
            k = tuple(int(x) for x in comp[a] + comp[b])
            pair_sum.setdefault(k, []).append((a, b))
    cands = []
    for k, sps in by_comp.items():                       # A <=> B (isomers)
        for i in range(len(sps)):
            for j in range(i + 1, len(sps)):
                cands.append(([(sps[i], 1)], [(sps[j], 1)]))
    for s in range(n_sp):                                # A <=> B + C
        for pr in pair_sum.get(key[s], []):
            if s in pr:
                continue
            cands.append(([(s, 1)], side(pr)))
    for k, prs in pair_sum.items():                      # A + B <=> C + D
        for i in range(len(prs)):
            for j in range(i + 1, len(prs)):
                if set(prs[i]) & set(prs[j]):
                    continue
                cands.append((side(prs[i]), side(prs[j])))
    return cands


def _qss_of(side, n_nqss):
    q = [s for s, _ in side if s >= n_nqss]
    return q[0] if q else None


class _UF:
    def __init__(self, n):
        self.p = list(range(n)); self.sz = [1] * n

    def find(self, x):
        while self.p[x] != x:
            self.p[x] = self.p[self.p[x]]; x = self.p[x]
        return x

    def union(self, a, b):
        a, b = self.find(a), self.find(b)
        if a == b:
            return
        if self.sz[a] < self.sz[b]:
            a, b = b, a
        self.p[b] = a; self.sz[a] += self.sz[b]

    def size(self, x):
        return self.sz[self.find(x)]


def make_mechanism(n_nqss: int, n_qss: int, n_reac: int, g_max: int, typed: bool, seed: int) -> Mechanism:
    for attempt in range(64):
        rng = np.random.default_rng([seed, attempt])
        m = _try_make(rng, n_nqss, n_qss, n_reac, g_max, typed)
        if m is not None:
            return m
    raise RuntimeError("mechanism generation failed")


def _try_make(rng, n_nqss, n_qss, n_reac, g_max, typed):
    n_sp = n_nqss + n_qss
    comp = _draw_compositions(rng, n_sp)
    cands = _enumerate_candidates(comp, n_nqss)
    if len(cands) < n_reac:
        return None
    order = rng.permutation(len(cands))
    used = np.zeros(len(cands), dtype=bool)
    chosen: List[int] = []
    uf = _UF(n_qss)

    qr = [_qss_of(c[0], n_nqss) for c in cands]
    qp = [_qss_of(c[1], n_nqss) for c in cands]

    # 1. every QSS species gets one reaction whose other side is QSS-free (a sink and a source)
    for q in range(n_nqss, n_sp):
        pick = None
        for ci in order:
            if used[ci]:
                continue
            if (qr[ci] == q and qp[ci] is None) or (qp[ci] == q and qr[ci] is None):
                pick = ci; break
        if pick is None:
            return None
        used[pick] = True; chosen.append(int(pick))
    # 2. grow one coupling component to exactly g_max
    if g_max > 1 and n_qss > 0:
        progress = True
        while max(uf.size(i) for i in range(n_qss)) < g_max and progress:
            progress = False
            big = max(range(n_qss), key=lambda i: uf.size(i))
            for ci in order:
                if used[ci] or qr[ci] is None or qp[ci] is None:
                    continue
                a, b = qr[ci] - n_nqss, qp[ci] - n_nqss
                ra, rb, rbig = uf.find(a), uf.find(b), uf.find(big)
                if ra == rb or (ra != rbig and rb != rbig):
                    continue
                if uf.size(a) + uf.size(b) > g_max:
                    continue
                uf.union(a, b); used[ci] = True; chosen.append(int(ci)); progress = True
                break
        if max(uf.size(i) for i in range(n_qss)) != g_max:
            return None
    # 3. random fill
    for ci in order:
        if len(chosen) >= n_reac:
            break
        if used[ci]:
            continue
        if qr[ci] is not None and qp[ci] is not None:
            a, b = qr[ci] - n_nqss, qp[ci] - n_nqss
            if uf.find(a) != uf.find(b) and uf.size(a) + uf.size(b) > g_max:
                continue
            uf.union(a, b)
        used[ci] = True; chosen.append(int(ci))
    if len(chosen) < n_reac:
        return None
    chosen = [chosen[i] for i in rng.permutation(len(chosen))]

    # kinetics
    reactions = []
    for ci in chosen:
        reac, prod = cands[ci]
        if rng.random() < 0.5:
            reac, prod = prod, reac
        r = dict(reac=list(reac), prod=list(prod), dir_mask=3)
        u = rng.random()
        r["type"] = 0 if (not typed or u < 0.7) else (1 if u < 0.9 else 2)
        r["arr"] = (10.0 ** rng.uniform(6.0, 14.0), rng.uniform(-2.0, 2.0), rng.uniform(0.0, 50.0) * KCAL)
        if r["type"] >= 1:
            k = int(rng.integers(3, 7))
            sps = rng.choice(n_nqss, size=min(k, n_nqss), replace=False)
            r["eff"] = [(int(s), float(rng.uniform(0.5, 5.0))) for s in sorted(sps)]
        if r["type"] == 2:
            r["arr_low"] = (r["arr"][0] * 10.0 ** rng.uniform(-4.0, 0.0), rng.uniform(-2.0, 2.0),
                            rng.uniform(0.0, 50.0) * KCAL)
            r["troe"] = (rng.uniform(0.2, 0.9), rng.uniform(50.0, 500.0), rng.uniform(500.0, 3000.0),
                         rng.uniform(2000.0, 8000.0))
        reactions.append(r)
    nasa_T, lo, hi = draw_nasa(rng, comp)
    return assemble(n_nqss, n_qss, comp, nasa_T, lo, hi, reactions)


_CACHE: Dict[int, Mechanism] = {}


def config_mechanism(cfg: int) -> Mechanism:
    """Mechanism of BASELINE.json config `cfg` (1-based). Seed = config index; cfg1 uses seed 0 as
    BASELINE.json states; cfg4 reuses cfg2's mechanism."""
    if cfg == 4:
        cfg = 2
    if cfg not in _CACHE:
        c = CONFIGS[cfg]
        seed = 0 if cfg == 1 else cfg
        _CACHE[cfg] = make_mechanism(c["n_nqss"], c["n_qss"], c["n_reac"], c["g_max"], c["typed"], seed)
    return _CACHE[cfg]
