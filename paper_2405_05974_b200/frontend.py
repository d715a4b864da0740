"""Mechanism front-end (second half): CHEMKIN-format or Cantera-YAML-format text -> the flat description `qss_mech_create` takes, and
the three linearisation methods of PAPER.md section 2.2 (L77-122, Algorithm 1) that make a QSS choice admissible for the
algebraic closure.  Host logic only (numpy); nothing here runs on the path.

Subset of the format that is read (everything else raises `MechanismError`, nothing is skipped silently):
  ELEMENTS / SPECIES / THERMO [ALL] (NASA-7, the fixed-column four-line records) / REACTIONS [units] ... END
  reactions  `2A + B <=> C + D   A  beta  Ea`   with `<=>` or `=` (reversible) and `=>` (forward only);
  `+ M` (third body) and `(+M)` (fall-off) with the auxiliary lines `LOW / A0 beta0 E0 /`, `TROE / alpha T*** T* [T**] /` and
  efficiencies `NAME / value /`; `DUPLICATE` is accepted (duplicates are separate reactions here anyway).
  Units: A in cm^3-mol-s, Ea in cal/mol unless the REACTIONS line says KCAL/MOLE, JOULES/MOLE, KJOULES/MOLE or KELVINS; converted
  to the library's SI-molar units (reading G4): A x (1e-6)^(order - 1), Ea in J/mol.
  Not read: REV, PLOG, CHEB, SRI, explicit collision partners `(+SPECIES)`, fractional or real stoichiometric coefficients, MOLECULES.
A fall-off reaction given with three Troe parameters gets T** = 1e30 (the term exp(-T**/T) then vanishes; the library's
exponential saturates for such placeholders).  Efficiencies of QSS species are dropped (M sums the transported species, G7) and
reported in `warnings`.
"""
from __future__ import annotations

import dataclasses
import itertools
import re
from typing import Dict, List, Sequence, Tuple

import numpy as np

CAL = 4.184
R_GAS = 8.31446261815324
ATOMIC_WEIGHT = {"H": 1.008, "C": 12.011, "O": 15.999, "N": 14.007, "AR": 39.948, "HE": 4.002602}


class MechanismError(ValueError):
    pass


@dataclasses.dataclass
class MechanismDescription:
    """The arrays of `qss_mech_desc_t` (include/qss.h) plus names.  Species 0..n_nqss-1 are transported, the rest QSS."""
    n_elem: int
    n_nqss: int
    n_qss: int
    n_reac: int
    elem_weight: np.ndarray
    comp: np.ndarray
    nasa_T: np.ndarray
    nasa_lo: np.ndarray
    nasa_hi: np.ndarray
    rtype: np.ndarray
    dir_mask: np.ndarray
    reac_ptr: np.ndarray
    reac_sp: np.ndarray
    reac_nu: np.ndarray
    prod_ptr: np.ndarray
    prod_sp: np.ndarray
    prod_nu: np.ndarray
    arr: np.ndarray
    arr_low: np.ndarray
    troe: np.ndarray
    eff_ptr: np.ndarray
    eff_sp: np.ndarray
    eff_val: np.ndarray
    species: List[str] = dataclasses.field(default_factory=list)
    elements: List[str] = dataclasses.field(default_factory=list)
    equations: List[str] = dataclasses.field(default_factory=list)
    warnings: List[str] = dataclasses.field(default_factory=list)

    @property
    def n_sp(self) -> int:
        return self.n_nqss + self.n_qss

    def side(self, j: int, which: int) -> List[Tuple[int, int]]:
        """[(species, nu)] of the reactants (which = 0) or products (which = 1) of reaction j."""
        ptr, sp, nu = (self.reac_ptr, self.reac_sp, self.reac_nu) if which == 0 else (self.prod_ptr, self.prod_sp, self.prod_nu)
        return [(int(sp[t]), int(nu[t])) for t in range(int(ptr[j]), int(ptr[j + 1]))]


# ---------------------------------------------------------------------------------------------------------------------------
# CHEMKIN-format text
# ---------------------------------------------------------------------------------------------------------------------------
_SECTION = re.compile(r"^(ELEMENTS|ELEM|SPECIES|SPEC|THERMO|THERM|REACTIONS|REAC|END)\b", re.I)
_AUX = re.compile(r"([^\s/]+)\s*/([^/]*)/")
_UNSUPPORTED_AUX = {"REV", "PLOG", "CHEB", "SRI", "LT", "RLT", "HIGH", "FORD", "RORD", "TCHEB", "PCHEB", "XSMI", "UNITS", "EXCI", "JAN", "FIT1", "MOME", "COLLEFF", "STICK"}


def _strip(line: str) -> str:
    return line.split("!", 1)[0].rstrip()


def _num(tok: str) -> float:
    return float(tok.replace("D", "E").replace("d", "e"))


def _split_sections(text: str) -> Dict[str, List[str]]:
    sec: Dict[str, List[str]] = {}
    cur = None
    for raw in text.splitlines():
        line = _strip(raw)
        if not line.strip():
            continue
        m = _SECTION.match(line.strip())
        if m:
            key = m.group(1).upper()[:4]
            if key == "END":
                cur = None
                continue
            cur = {"ELEM": "ELEMENTS", "SPEC": "SPECIES", "THER": "THERMO", "REAC": "REACTIONS"}[key]
            rest = line.strip()[m.end():]
            closes = cur != "THERMO" and rest.split()[-1:] == ["END"] or rest.upper().split()[-1:] == ["END"] and cur != "THERMO"
            if closes:
                rest = rest[:rest.upper().rindex("END")]
            sec.setdefault(cur, [])
            sec[cur].append("\0HEADER " + rest)        # the remainder of the keyword line (units, THERMO ALL, names on the same line)
            if closes:
                cur = None
            continue
        if cur is None:
            raise MechanismError(f"text outside a section: {line!r}")
        if cur in ("ELEMENTS", "SPECIES") and line.upper().split()[-1:] == ["END"]:      # `... names END` on one line
            sec[cur].append(line.strip()[:line.strip().upper().rindex("END")])
            cur = None
            continue
        sec[cur].append(line if cur == "THERMO" else line.strip())
    for need in ("ELEMENTS", "SPECIES", "THERMO", "REACTIONS"):
        if need not in sec:
            raise MechanismError(f"section {need} is missing")
    return sec


def _names(lines: Sequence[str]) -> List[str]:
    out: List[str] = []
    for ln in lines:
        ln = ln.replace("\0HEADER", " ")
        for tok in ln.split():
            if "/" in tok:
                raise MechanismError(f"isotope / weight overrides are not read: {tok!r}")
            up = tok.upper()
            if up in out:
                raise MechanismError(f"{tok} is listed twice")
            out.append(up)
    return out


def _thermo(lines: Sequence[str], species: Sequence[str], elements: Sequence[str]):
    """NASA-7 records: line 1 name, composition (4 x [symbol(2) count(3)] from column 25, a fifth from column 74), Tlow, Thigh, Tmid
    (columns 46-55, 56-65, 66-73); lines 2-4 fifteen-character fields: a1..a5 HIGH | a6 a7 HIGH, a1 a2 a3 LOW | a4..a7 LOW."""
    body = [ln for ln in lines if not ln.startswith("\0HEADER")]
    if not body:
        raise MechanismError("THERMO section is empty")
    defaults = None
    first = body[0].split()
    if len(first) == 3 and all(re.fullmatch(r"[0-9.+\-EeDd]+", t) for t in first):
        defaults = [_num(t) for t in first]
        body = body[1:]
    found = {}
    i = 0
    while i < len(body):
        l1 = body[i].ljust(80)
        if i + 3 >= len(body):
            raise MechanismError(f"truncated thermo record at {l1[:18].strip()!r}")
        name = l1[:18].split()[0].upper() if l1[:18].split() else ""
        comp = {}
        for col in (24, 29, 34, 39, 73):
            sym, cnt = l1[col:col + 2].strip().upper(), l1[col + 2:col + 5].strip()
            if sym and sym != "0" and cnt:
                c = _num(cnt)
                if c != int(c):
                    raise MechanismError(f"{name}: non-integer composition")
                if int(c):
                    comp[sym] = comp.get(sym, 0) + int(c)
        try:
            tlow, thigh = _num(l1[45:55]), _num(l1[55:65])
            tmid = _num(l1[65:73]) if l1[65:73].strip() else (defaults[1] if defaults else None)
        except ValueError as e:
            raise MechanismError(f"{name}: temperature fields: {e}")
        if tmid is None:
            raise MechanismError(f"{name}: no common temperature")
        co = []
        for ln in body[i + 1:i + 4]:
            ln = ln.ljust(80)
            co += [ln[k:k + 15] for k in range(0, 75, 15)]
        try:
            vals = [_num(x) for x in co[:14]]
        except ValueError as e:
            raise MechanismError(f"{name}: coefficient fields: {e}")
        if name in species and name not in found:
            for sym in comp:
                if sym not in elements:
                    raise MechanismError(f"{name}: element {sym} is not declared")
            found[name] = (comp, (tlow, tmid, thigh), vals[7:14], vals[0:7])
        i += 4
    missing = [s for s in species if s not in found]
    if missing:
        raise MechanismError(f"no thermo record for {missing}")
    return found


def _side(text: str, species: Sequence[str], eq: str):
    """`2A+B+M` -> ([(index, nu)], has_M)."""
    out: List[Tuple[int, int]] = []
    has_m = False
    for tok in text.split("+"):
        tok = tok.strip().upper()
        if not tok:
            raise MechanismError(f"{eq}: empty term (species names containing '+' are not read)")
        if tok == "M":
            has_m = True
            continue
        nu, name = 1, tok
        if name not in species:
            m = re.match(r"^(\d+)(.+)$", tok)
            if m and m.group(2) in species:
                nu, name = int(m.group(1)), m.group(2)
            else:
                raise MechanismError(f"{eq}: unknown species {tok!r} (real coefficients are not read)")
        if nu < 1:
            raise MechanismError(f"{eq}: coefficient {nu}")
        for k, (s0, n0) in enumerate(out):
            if s0 == species.index(name):
                out[k] = (s0, n0 + nu)
                break
        else:
            out.append((species.index(name), nu))
    return out, has_m


def _equation(eq: str, species: Sequence[str]):
    """`A+B(+M)<=>C(+M)` -> (reactants, products, reversible, third body `+ M`, fall-off `(+M)`)."""
    body = eq.replace(" ", "").upper()
    falloff = "(+M)" in body
    if re.search(r"\(\+[^M)]", body) or re.search(r"\(\+M[^)]", body):
        raise MechanismError(f"{eq}: explicit collision partners are not read")
    body = body.replace("(+M)", "")
    if "<=>" in body: lhs, rhs, rev = *body.split("<=>", 1), True
    elif "=>" in body: lhs, rhs, rev = *body.split("=>", 1), False
    elif "=" in body: lhs, rhs, rev = *body.split("=", 1), True
    else: raise MechanismError(f"{eq}: no '=' in the reaction")
    re_, m1 = _side(lhs, species, eq)
    pr_, m2 = _side(rhs, species, eq)
    if m1 != m2:
        raise MechanismError(f"{eq}: M on one side only")
    if falloff and m1:
        raise MechanismError(f"{eq}: both +M and (+M)")
    return re_, pr_, rev, m1, falloff


def _reactions(lines: Sequence[str], species: Sequence[str]):
    e_unit, header = CAL, " ".join(ln.replace("\0HEADER", "") for ln in lines if ln.startswith("\0HEADER")).upper().split()
    for tok in header:
        if tok in ("CAL/MOLE", "CAL/MOL"): e_unit = CAL
        elif tok in ("KCAL/MOLE", "KCAL/MOL"): e_unit = 1e3 * CAL
        elif tok in ("JOULES/MOLE", "JOULES/MOL"): e_unit = 1.0
        elif tok in ("KJOULES/MOLE", "KJOULES/MOL", "KJOU/MOLE"): e_unit = 1e3
        elif tok in ("KELVINS", "KELVIN"): e_unit = R_GAS
        elif tok in ("MOLES", "MOLE"): pass
        else: raise MechanismError(f"REACTIONS: unit keyword {tok!r} is not read")
    recs: List[dict] = []
    for ln in lines:
        if ln.startswith("\0HEADER"):
            continue
        up = ln.upper()
        if up.startswith("DUP"):
            continue
        if "/" in ln:                                             # auxiliary line of the last reaction
            if not recs:
                raise MechanismError(f"auxiliary line before any reaction: {ln!r}")
            pairs = _AUX.findall(ln)
            if not pairs or _AUX.sub("", ln).strip():
                raise MechanismError(f"cannot read the auxiliary line {ln!r}")
            for key, val in pairs:
                key = key.upper()
                nums = val.split()
                if key == "LOW":
                    recs[-1]["low"] = [_num(x) for x in nums]
                elif key == "TROE":
                    recs[-1]["troe"] = [_num(x) for x in nums]
                elif key in _UNSUPPORTED_AUX:
                    raise MechanismError(f"{recs[-1]['eq']}: {key} is not read")
                elif key in species:
                    recs[-1]["eff"].append((species.index(key), _num(nums[0])))
                else:
                    raise MechanismError(f"{recs[-1]['eq']}: unknown auxiliary keyword or species {key!r}")
            continue
        f = ln.split()
        if len(f) < 4:
            raise MechanismError(f"cannot read the reaction line {ln!r}")
        try:
            A, beta, Ea = (_num(x) for x in f[-3:])
        except ValueError:
            raise MechanismError(f"cannot read the rate parameters of {ln!r}")
        eq = "".join(f[:-3])
        re_, pr_, rev, m1, falloff = _equation(eq, species)
        recs.append(dict(eq=eq, reac=re_, prod=pr_, rev=rev, type=2 if falloff else (1 if m1 else 0), A=A, beta=beta, Ea=Ea * e_unit,
                         low=None, troe=None, eff=[], e_unit=e_unit, vol_unit=1e-6))
    for r in recs:
        if r["type"] == 2 and (r["low"] is None or r["troe"] is None):
            raise MechanismError(f"{r['eq']}: a fall-off reaction needs LOW and TROE (Lindemann form is not read)")
        if r["type"] != 2 and (r["low"] is not None or r["troe"] is not None):
            raise MechanismError(f"{r['eq']}: LOW / TROE without (+M)")
        if r["type"] == 0 and r["eff"]:
            raise MechanismError(f"{r['eq']}: efficiencies without a third body")
        if r["low"] is not None and len(r["low"]) != 3:
            raise MechanismError(f"{r['eq']}: LOW takes three numbers")
        if r["troe"] is not None and len(r["troe"]) not in (3, 4):
            raise MechanismError(f"{r['eq']}: TROE takes three or four numbers")
    return recs


def parse_chemkin(text: str, qss: Sequence[str] = ()) -> MechanismDescription:
    """CHEMKIN-format mechanism text (+ the names of the QSS species) -> flat description, transported species first."""
    sec = _split_sections(text)
    elements = _names(sec["ELEMENTS"])
    names = _names(sec["SPECIES"])
    for e in elements:
        if e not in ATOMIC_WEIGHT:
            raise MechanismError(f"element {e}: atomic weight not known to the front-end")
    qset = [q.upper() for q in qss]
    for q in qset:
        if q not in names:
            raise MechanismError(f"QSS species {q} is not in SPECIES")
    thermo = _thermo(sec["THERMO"], names, elements)
    recs = _reactions(sec["REACTIONS"], names)
    return _assemble(elements, names, qset, thermo, recs)


def _assemble(elements, names, qset, thermo, recs) -> MechanismDescription:
    """Flat description from parsed parts.  thermo[name] = (composition dict, (Tlow, Tmid, Thigh), a_low[7], a_high[7]); a reaction record
    carries A in (vol_unit m^3 per quantity)^(order - 1) / s and activation energies already multiplied into J/mol where noted."""
    order = [s for s in names if s not in qset] + [s for s in names if s in qset]       # file order inside each class
    new_of = {names.index(s): i for i, s in enumerate(order)}
    N, Nq, M = len(names) - len(qset), len(qset), len(recs)
    comp = np.zeros((len(order), len(elements)), dtype=np.int32)
    nT = np.zeros((len(order), 3)); lo = np.zeros((len(order), 7)); hi = np.zeros((len(order), 7))
    for i, s in enumerate(order):
        c, tt, l7, h7 = thermo[s]
        for sym, cnt in c.items():
            comp[i, elements.index(sym)] = cnt
        nT[i], lo[i], hi[i] = tt, l7, h7
    warnings: List[str] = []
    rp, rs, rn, pp, ps, pn, ep, es, ev = [0], [], [], [0], [], [], [0], [], []
    rtype = np.zeros(M, dtype=np.int32); mask = np.zeros(M, dtype=np.uint8)
    arr = np.zeros((M, 3)); low = np.zeros((M, 3)); troe = np.zeros((M, 4))
    for j, r in enumerate(recs):
        for sp_, nu in r["reac"]: rs.append(new_of[sp_]); rn.append(nu)
        for sp_, nu in r["prod"]: ps.append(new_of[sp_]); pn.append(nu)
        rp.append(len(rs)); pp.append(len(ps))
        order_f = sum(nu for _, nu in r["reac"])
        rtype[j] = r["type"]; mask[j] = 3 if r["rev"] else 1
        # cm^3-mol-s -> m^3-mol-s: a rate constant of order n carries (cm^3/mol)^(n-1); a third body adds one order; the
        # fall-off limits: k_inf order n, k_0 order n + 1
        arr[j] = (r["A"] * r["vol_unit"] ** (order_f - 1 + (1 if r["type"] == 1 else 0)), r["beta"], r["Ea"])
        if r["type"] == 2:
            low[j] = (r["low"][0] * r["vol_unit"] ** order_f, r["low"][1], r["low"][2] * r["e_unit"])
            t4 = list(r["troe"]) + ([1e30] if len(r["troe"]) == 3 else [])
            troe[j] = t4
        for sp_, val in r["eff"]:
            if new_of[sp_] >= N:
                warnings.append(f"{r['eq']}: efficiency of the QSS species {names[sp_]} dropped (M sums the transported species)")
                continue
            es.append(new_of[sp_]); ev.append(val)
        ep.append(len(es))
    i32 = lambda a: np.asarray(a, dtype=np.int32)
    return MechanismDescription(
        n_elem=len(elements), n_nqss=N, n_qss=Nq, n_reac=M, elem_weight=np.array([ATOMIC_WEIGHT[e] for e in elements]), comp=comp,
        nasa_T=nT, nasa_lo=lo, nasa_hi=hi, rtype=rtype, dir_mask=mask, reac_ptr=i32(rp), reac_sp=i32(rs), reac_nu=i32(rn),
        prod_ptr=i32(pp), prod_sp=i32(ps), prod_nu=i32(pn), arr=arr, arr_low=low, troe=troe, eff_ptr=i32(ep), eff_sp=i32(es),
        eff_val=np.asarray(ev, dtype=np.float64), species=order, elements=list(elements), equations=[r["eq"] for r in recs], warnings=warnings)


# ---------------------------------------------------------------------------------------------------------------------------
# Cantera-YAML-format text (the subset that matches the CHEMKIN subset above)
# ---------------------------------------------------------------------------------------------------------------------------
_YAML_EA = {"cal/mol": CAL, "kcal/mol": 1e3 * CAL, "J/mol": 1.0, "kJ/mol": 1e3, "J/kmol": 1e-3, "K": R_GAS}
_YAML_LEN = {"m": 1.0, "cm": 1e-2}
_YAML_QTY = {"mol": 1.0, "kmol": 1e3}


def parse_yaml(text: str, qss: Sequence[str] = ()) -> MechanismDescription:
    """Cantera-YAML-format mechanism text -> flat description.  Read: a top-level `units` mapping (length m | cm, quantity mol | kmol,
    activation-energy cal/mol | kcal/mol | J/mol | kJ/mol | J/kmol | K; defaults m, kmol, J/kmol as in that format), the element and
    species lists of the FIRST phase, `species` entries with `composition` and `thermo: {model: NASA7, temperature-ranges: [lo, mid, hi],
    data: [[a1..a7 low], [a1..a7 high]]}`, `reactions` entries with `equation`, `rate-constant: {A, b, Ea}`, `type: three-body` (or `+ M`
    in the equation) with `efficiencies`, `type: falloff` with `low-P-rate-constant`, `high-P-rate-constant`, `Troe: {A, T3, T1[, T2]}`;
    `duplicate`.  Numbers only: quantities written as strings with units, other reaction types or rate forms raise MechanismError."""
    import yaml
    try:
        doc = yaml.safe_load(text)
    except yaml.YAMLError as e:
        raise MechanismError(f"not YAML: {e}")
    if not isinstance(doc, dict) or "phases" not in doc or "species" not in doc or "reactions" not in doc:
        raise MechanismError("the document needs `phases`, `species` and `reactions`")
    un = doc.get("units", {}) or {}
    try:
        length, qty, e_unit = _YAML_LEN[un.get("length", "m")], _YAML_QTY[un.get("quantity", "kmol")], _YAML_EA[un.get("activation-energy", "J/kmol")]
    except KeyError as e:
        raise MechanismError(f"units: {e} is not read")
    for k in un:
        if k not in ("length", "quantity", "activation-energy", "time", "mass", "pressure", "temperature", "energy"):
            raise MechanismError(f"units: {k} is not read")
    if un.get("time", "s") != "s":
        raise MechanismError("units: time other than s is not read")
    vol_unit = length ** 3 / qty
    phase = doc["phases"][0]
    elements = [str(e).upper() for e in phase.get("elements", [])]
    names = [str(x).upper() for x in phase.get("species", [])]
    if not elements or not names or any(isinstance(x, dict) for x in phase.get("species", [])):
        raise MechanismError("the first phase needs plain `elements` and `species` lists")
    for e in elements:
        if e not in ATOMIC_WEIGHT:
            raise MechanismError(f"element {e}: atomic weight not known to the front-end")
    qset = [q.upper() for q in qss]
    for q in qset:
        if q not in names:
            raise MechanismError(f"QSS species {q} is not in the phase")

    def num(v, what):
        if isinstance(v, bool) or not isinstance(v, (int, float)):
            raise MechanismError(f"{what}: {v!r} is not a plain number (quantities with units are not read)")
        return float(v)

    thermo = {}
    for sp in doc["species"]:
        name = str(sp.get("name", "")).upper()
        th = sp.get("thermo", {})
        if th.get("model") != "NASA7":
            raise MechanismError(f"{name}: thermo model {th.get('model')!r} is not read")
        tr, data = th.get("temperature-ranges", []), th.get("data", [])
        if len(tr) != 3 or len(data) != 2 or any(len(d) != 7 for d in data):
            raise MechanismError(f"{name}: NASA7 needs three temperatures and two sets of seven coefficients")
        comp = {}
        for sym, cnt in (sp.get("composition", {}) or {}).items():
            c = num(cnt, f"{name}: composition")
            if c != int(c) or str(sym).upper() not in elements:
                raise MechanismError(f"{name}: composition {sym}: {cnt}")
            if int(c):
                comp[str(sym).upper()] = int(c)
        if name in names and name not in thermo:
            thermo[name] = (comp, tuple(num(x, f"{name}: temperature") for x in tr), [num(x, name) for x in data[0]], [num(x, name) for x in data[1]])
    missing = [x for x in names if x not in thermo]
    if missing:
        raise MechanismError(f"no species entry for {missing}")

    def rate(d, eq):
        if not isinstance(d, dict) or set(d) != {"A", "b", "Ea"}:
            raise MechanismError(f"{eq}: a rate constant needs exactly A, b, Ea")
        return num(d["A"], eq), num(d["b"], eq), num(d["Ea"], eq) * e_unit

    recs = []
    for r in doc["reactions"]:
        eq = str(r.get("equation", ""))
        for k in r:
            if k not in ("equation", "rate-constant", "type", "efficiencies", "low-P-rate-constant", "high-P-rate-constant", "Troe", "duplicate", "note"):
                raise MechanismError(f"{eq}: {k} is not read")
        re_, pr_, rev, m1, falloff = _equation(eq, names)
        typ = r.get("type", "falloff" if falloff else ("three-body" if m1 else "elementary"))
        if typ == "elementary" and (m1 or falloff) or typ == "three-body" and not m1 or typ == "falloff" and not falloff or typ not in ("elementary", "three-body", "falloff"):
            raise MechanismError(f"{eq}: type {typ!r} does not match the equation or is not read")
        rec = dict(eq=eq.replace(" ", ""), reac=re_, prod=pr_, rev=rev, type={"elementary": 0, "three-body": 1, "falloff": 2}[typ], low=None, troe=None,
                   eff=[], e_unit=1.0, vol_unit=vol_unit)
        if typ == "falloff":
            if "Troe" not in r or "low-P-rate-constant" not in r or "high-P-rate-constant" not in r or "rate-constant" in r:
                raise MechanismError(f"{eq}: a fall-off reaction needs low-P-rate-constant, high-P-rate-constant and Troe (Lindemann form is not read)")
            rec["A"], rec["beta"], rec["Ea"] = rate(r["high-P-rate-constant"], eq)
            rec["low"] = list(rate(r["low-P-rate-constant"], eq))
            tro = r["Troe"]
            if not isinstance(tro, dict) or not {"A", "T3", "T1"} <= set(tro) or not set(tro) <= {"A", "T3", "T1", "T2"}:
                raise MechanismError(f"{eq}: Troe needs A, T3, T1 and optionally T2")
            rec["troe"] = [num(tro["A"], eq), num(tro["T3"], eq), num(tro["T1"], eq)] + ([num(tro["T2"], eq)] if "T2" in tro else [])
        else:
            if "rate-constant" not in r or "Troe" in r or "low-P-rate-constant" in r:
                raise MechanismError(f"{eq}: needs rate-constant only")
            rec["A"], rec["beta"], rec["Ea"] = rate(r["rate-constant"], eq)
        eff = r.get("efficiencies", {}) or {}
        if eff and typ == "elementary":
            raise MechanismError(f"{eq}: efficiencies without a third body")
        for sp_, val in eff.items():
            if str(sp_).upper() not in names:
                raise MechanismError(f"{eq}: efficiency of unknown species {sp_}")
            rec["eff"].append((names.index(str(sp_).upper()), num(val, eq)))
        recs.append(rec)
    return _assemble(elements, names, qset, thermo, recs)


# ---------------------------------------------------------------------------------------------------------------------------
# Linearisation of the QSS closure (section 2.2)
# ---------------------------------------------------------------------------------------------------------------------------
def quadratic_couplings(d: MechanismDescription) -> List[Tuple[int, int]]:
    """[(reaction j, side)] with "two or more QSS species on the same side of an elementary reaction" (L73: a quadratic coupling;
    side 0 reactants, 1 products), counted in molecules (2 Q on a side is one), enabled directions or not."""
    out = []
    for j in range(d.n_reac):
        for side in (0, 1):
            if sum(nu for sp, nu in d.side(j, side) if sp >= d.n_nqss) >= 2:
                out.append((j, side))
    return out


def _offending(d: MechanismDescription) -> List[Tuple[int, int]]:
    """The couplings that still bind: a side with >= 2 QSS molecules that an ENABLED direction consumes (side s is consumed by
    direction s).  A side that is only produced is the fan-out case, which the library's closure also refuses (QSS_E_QSS_FANOUT)."""
    return [(j, s) for j, s in quadratic_couplings(d) if (int(d.dir_mask[j]) >> s) & 1]


def reclassify(d: MechanismDescription, to_transported: Sequence[int]) -> MechanismDescription:
    """The QSS species `to_transported` (indices into d.species) become transported species (appended behind the transported ones,
    order kept); every index array is renumbered."""
    move = sorted(set(int(x) for x in to_transported))
    for x in move:
        if not (d.n_nqss <= x < d.n_sp):
            raise MechanismError(f"species {x} is not a QSS species")
    order = list(range(d.n_nqss)) + move + [x for x in range(d.n_nqss, d.n_sp) if x not in move]
    new_of = np.empty(d.n_sp, dtype=np.int32)
    new_of[order] = np.arange(d.n_sp, dtype=np.int32)
    return dataclasses.replace(
        d, n_nqss=d.n_nqss + len(move), n_qss=d.n_qss - len(move), comp=d.comp[order], nasa_T=d.nasa_T[order], nasa_lo=d.nasa_lo[order],
        nasa_hi=d.nasa_hi[order], reac_sp=new_of[d.reac_sp] if len(d.reac_sp) else d.reac_sp, prod_sp=new_of[d.prod_sp] if len(d.prod_sp) else d.prod_sp,
        eff_sp=new_of[d.eff_sp] if len(d.eff_sp) else d.eff_sp, species=[d.species[x] for x in order] if d.species else [])


def species_linearisation_sets(d: MechanismDescription, max_size: int | None = None) -> List[Tuple[int, ...]]:
    """Algorithm 1 (L97-113): A = the QSS species involved in at least one quadratic coupling ("a reactant in the elementary reaction
    where a quadratic coupling ... is found", L77: the QSS species of a coupled side); subsets of A of growing size i; the first size
    at which turning a subset into non-QSS species leaves no quadratic coupling returns ALL such subsets of that size (the list B)."""
    qc = quadratic_couplings(d)
    if not qc:
        return [()]
    A = sorted({sp for j, s in qc for sp, _ in d.side(j, s) if sp >= d.n_nqss})
    top = len(A) if max_size is None else min(max_size, len(A))
    for i in range(1, top + 1):
        B = []
        for sub in itertools.combinations(A, i):
            gone = set(sub)
            if all(sum(nu for sp, nu in d.side(j, s) if sp >= d.n_nqss and sp not in gone) < 2 for j, s in qc):
                B.append(sub)
        if B:
            return B
    return []


def linearise(d: MechanismDescription, method: str, species_set: Sequence[int] | None = None) -> MechanismDescription:
    """The three methods of section 2.2:
      "species"   turn a smallest set of coupled QSS species into transported species (Algorithm 1; `species_set` picks one of
                  `species_linearisation_sets`, default the first);
      "reaction"  "ignore the complete reaction to conserve chemical balance" (L77): both directions of every reaction with a
                  quadratic coupling are switched off;
      "one_sided" only the direction that CONSUMES the coupled side is switched off ("removes only the reaction direction that induces the quadratic coupling", L77).  The other direction then produces two
                  QSS molecules, which the library's subtraction-free closure does not take (QSS_E_QSS_FANOUT)."""
    if method == "species":
        if species_set is None:
            sets = species_linearisation_sets(d)
            if not sets:
                raise MechanismError("no subset of the coupled QSS species removes every quadratic coupling")
            species_set = sets[0]
        return reclassify(d, species_set)
    mask = d.dir_mask.copy()
    for j, s in quadratic_couplings(d):
        if method == "reaction":
            mask[j] = 0
        elif method == "one_sided":
            mask[j] &= np.uint8(~(1 << s) & 3)
        else:
            raise MechanismError(f"unknown linearisation method {method!r}")
    return dataclasses.replace(d, dir_mask=mask)
