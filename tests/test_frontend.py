"""Mechanism front-end (NEXT-4, second half; paper_2405_05974_b200/frontend.py): CHEMKIN-format ingestion and the three
linearisation methods of PAPER.md section 2.2 (L73-122, Algorithm 1).  Host logic; the mechanism text below is made up for the
test (species A2, B2, AB ..., invented rate parameters): no published mechanism is reproduced."""
from __future__ import annotations

import itertools

import numpy as np
import pytest

import oracle
import paper_2405_05974_b200 as qss
from paper_2405_05974_b200 import frontend as fe


def nasa_record(name, comp, a1, a6, a7, tlow=300.0, thigh=3500.0, tmid=1000.0):
    """Four fixed-column lines; the same constant-cp fit in both ranges (cp/R = a1, h/RT = a1 + a6/T, s/R = a1 ln T + a7)."""
    c = "".join("%-2s%3d" % (e, n) for e, n in comp) + " " * (5 * (4 - len(comp)))
    l1 = "%-18s%-6s%s%s%10.2f%10.2f%8.2f" % (name, "test", c, "G", tlow, thigh, tmid)
    l1 = l1.ljust(79) + "1"
    co = [a1, 0.0, 0.0, 0.0, 0.0, a6, a7] * 2
    f = ["%15.8E" % v for v in co]
    return "\n".join([l1, ("".join(f[0:5])).ljust(79) + "2", ("".join(f[5:10])).ljust(79) + "3", ("".join(f[10:14])).ljust(79) + "4"])


SPECIES = [("A2", [("H", 2)], 3.5, -1000.0, 1.0), ("B2", [("O", 2)], 3.6, -1100.0, 2.0), ("AB", [("H", 1), ("O", 1)], 3.7, 4000.0, 3.0),
           ("A2B", [("H", 2), ("O", 1)], 4.2, -29000.0, 1.5), ("A", [("H", 1)], 2.5, 25000.0, -0.5), ("B", [("O", 1)], 2.6, 29000.0, 0.5),
           ("AB2", [("H", 1), ("O", 2)], 4.5, 1000.0, 2.5), ("A2B2", [("H", 2), ("O", 2)], 5.0, -17000.0, 2.2)]

TEXT = """! a made-up H/O-shaped test mechanism
ELEMENTS H O END
SPECIES A2 B2 AB
        A2B A B AB2 A2B2 END
THERMO ALL
   300.000  1000.000  3500.000
%s
END
REACTIONS
A + B2 <=> B + AB            3.5E+15  -0.40   16600.0   ! bimolecular, cal/mol
B + A2 = A + AB              5.0E+04   2.67    6290.0
AB + A2 <=> A + A2B          2.2E+08   1.51    3430.0
2AB <=> B + A2B              3.6E+04   2.40   -2110.0
A + B2 + M <=> AB2 + M       2.8E+18  -0.86       0.0
   A2B/11.0/ B2/0.78/ A/2.0/
A + AB2 => 2AB               7.1E+13   0.00     295.0
AB + AB (+M) <=> A2B2 (+M)   7.4E+13  -0.37       0.0
   LOW / 2.3E+18 -0.90 -1700.0 /
   TROE / 0.735 94.0 1756.0 5182.0 /
   A2/2.0/ A2B/6.0/
AB2 + AB2 <=> A2B2 + B2      1.3E+11   0.00   -1630.0
  DUPLICATE
AB2 + AB2 <=> A2B2 + B2      4.2E+14   0.00   12000.0
  DUPLICATE
A2B2 + A (+M) <=> A2B + AB (+M)  2.4E+13  0.00  3970.0
   LOW / 1.0E+17 0.0 1000.0 /   TROE / 0.5 100.0 2000.0 /
END
""" % "\n".join(nasa_record(n, c, a1, a6, a7) for n, c, a1, a6, a7 in SPECIES)


def test_parse_layout_units_and_thermo():
    d = fe.parse_chemkin(TEXT, qss=["A", "B"])
    assert d.species == ["A2", "B2", "AB", "A2B", "AB2", "A2B2", "A", "B"] and (d.n_nqss, d.n_qss, d.n_reac) == (6, 2, 10)
    sp = d.species.index
    assert d.side(0, 0) == [(sp("A"), 1), (sp("B2"), 1)] and d.side(0, 1) == [(sp("B"), 1), (sp("AB"), 1)]
    assert d.side(3, 0) == [(sp("AB"), 2)] and d.side(5, 1) == [(sp("AB"), 2)] and d.side(6, 0) == [(sp("AB"), 2)]
    assert list(d.rtype) == [0, 0, 0, 0, 1, 0, 2, 0, 0, 2] and list(d.dir_mask) == [3, 3, 3, 3, 3, 1, 3, 3, 3, 3]
    # cm^3-mol-s -> m^3-mol-s, cal -> J: bimolecular 1e-6, two reactants + M 1e-12, fall-off k_inf (2 reactants) 1e-6, k_0 1e-12
    assert np.isclose(d.arr[0, 0], 3.5e15 * 1e-6) and np.isclose(d.arr[0, 2], 16600.0 * 4.184) and d.arr[0, 1] == -0.40
    assert np.isclose(d.arr[4, 0], 2.8e18 * 1e-12) and np.isclose(d.arr[6, 0], 7.4e13 * 1e-6) and np.isclose(d.arr_low[6, 0], 2.3e18 * 1e-12)
    assert np.isclose(d.arr_low[6, 2], -1700.0 * 4.184) and list(d.troe[6]) == [0.735, 94.0, 1756.0, 5182.0] and list(d.troe[9]) == [0.5, 100.0, 2000.0, 1e30]
    # efficiencies: CSR on transported species; the QSS species' one is dropped with a warning
    e4 = {d.species[s]: v for s, v in zip(d.eff_sp[d.eff_ptr[4]:d.eff_ptr[5]], d.eff_val[d.eff_ptr[4]:d.eff_ptr[5]])}
    assert e4 == {"A2B": 11.0, "B2": 0.78} and any("efficiency of the QSS species A" in w for w in d.warnings)
    # thermo: composition, ranges, HIGH range first in the file, LOW second
    assert list(d.comp[sp("A2B")]) == [2, 1] and list(d.nasa_T[sp("A2B")]) == [300.0, 1000.0, 3500.0]
    assert np.allclose(d.nasa_hi[sp("A2B")], [4.2, 0, 0, 0, 0, -29000.0, 1.5]) and np.allclose(d.nasa_lo[sp("A")], [2.5, 0, 0, 0, 0, 25000.0, -0.5])
    assert np.allclose(d.elem_weight, [1.008, 15.999])
    # the description is one the library takes (strict element balance included) and the oracle evaluates
    ng, order, grp = qss.validate(d, strict_balance=True)
    assert ng >= 1 and sorted(order) == [0, 1]
    C = np.ascontiguousarray(np.random.default_rng(0).uniform(0.01, 1.0, size=(6, 4))); T = np.array([900.0, 1200.0, 1500.0, 2000.0])
    out = oracle.evaluate(oracle.OracleMech(d), C, T)
    assert np.isfinite(out["jac"]).all() and np.abs(out["wdot"]).max() > 0
    a = d.comp[:6].astype(float)
    assert np.abs(a.T @ out["wdot"]).max() <= 1e-9 * (np.abs(a).T @ out["S"]).max()       # elements conserved: stoichiometry and order intact


@pytest.mark.parametrize("bad,msg", [("A + XX <=> B + AB 1.0 0 0", "unknown species"), ("A + B2 <=> B + AB 1.0 0 0\n REV / 1 0 0 /", "REV"),
                                     ("A + B2 (+A2B) <=> AB2 (+A2B) 1.0 0 0", "collision partners"), ("A + B2 + M <=> AB2 1.0 0 0", "one side"),
                                     ("AB + AB (+M) <=> A2B2 (+M) 1.0 0 0", "LOW and TROE"), ("A + B2 <=> B + AB 1.0 0", "cannot read")])
def test_what_is_not_read_is_an_error(bad, msg):
    text = TEXT[:TEXT.index("REACTIONS")] + "REACTIONS\n" + bad + "\nEND\n"
    with pytest.raises(fe.MechanismError) as e:
        fe.parse_chemkin(text)
    assert msg in str(e.value)
    with pytest.raises(fe.MechanismError):
        fe.parse_chemkin(TEXT.replace("SPECIES A2 B2 AB", "SPECIES A2 B2 AB ZZ"))                  # no thermo record
    with pytest.raises(fe.MechanismError):
        fe.parse_chemkin(TEXT, qss=["NOPE"])


def test_linearisation_methods():
    """QSS = {A, B, AB2}: quadratic couplings in `A + AB2 => 2AB` (reactants A + AB2) and in both `AB2 + AB2 <=> A2B2 + B2`."""
    d = fe.parse_chemkin(TEXT, qss=["A", "B", "AB2"])
    qc = fe.quadratic_couplings(d)
    by_eq = {(d.equations[j], s) for j, s in qc}
    assert by_eq == {("A+AB2=>2AB", 0), ("AB2+AB2<=>A2B2+B2", 0)} and len(qc) == 3
    with pytest.raises(qss.QssError) as e:
        qss.validate(d)
    assert e.value.code == -2                                           # QSS_E_QUADRATIC
    # species method: Algorithm 1 against brute force over ALL subsets of ALL QSS species by growing size
    sets = fe.species_linearisation_sets(d)
    def clean(gone):
        return all(sum(nu for sp, nu in d.side(j, s) if sp >= d.n_nqss and sp not in gone) < 2 for j in range(d.n_reac) for s in (0, 1))
    brute = []
    for i in range(1, d.n_qss + 1):
        brute = [c for c in itertools.combinations(range(d.n_nqss, d.n_sp), i) if clean(set(c))]
        if brute:
            break
    assert sorted(sets) == sorted(brute) and len(sets[0]) == len(brute[0])
    ds = fe.linearise(d, "species")
    assert ds.n_qss == d.n_qss - len(sets[0]) and not fe.quadratic_couplings(ds)
    qss.validate(ds, strict_balance=True)
    assert sorted(ds.species) == sorted(d.species) and ds.species[:d.n_nqss] == d.species[:d.n_nqss]
    # a chosen set
    d2 = fe.linearise(d, "species", sets[-1])
    assert [d.species[x] for x in sets[-1]] == d2.species[d.n_nqss:d.n_nqss + len(sets[-1])]
    # reaction method: every coupled reaction loses both directions; the rest is untouched; the library takes the result
    dr = fe.linearise(d, "reaction")
    coupled = {j for j, _ in qc}
    assert all(dr.dir_mask[j] == 0 for j in coupled) and all(dr.dir_mask[j] == d.dir_mask[j] for j in range(d.n_reac) if j not in coupled)
    qss.validate(dr, strict_balance=True)
    # one-sided method: only the consuming direction goes; what stays produces two QSS molecules -> the closure refuses it
    do = fe.linearise(d, "one_sided")
    j = d.equations.index("AB2+AB2<=>A2B2+B2")
    assert do.dir_mask[j] == 2 and do.dir_mask[d.equations.index("A+AB2=>2AB")] == 0
    with pytest.raises(qss.QssError) as e:
        qss.validate(do)
    assert e.value.code == -3                                           # QSS_E_QSS_FANOUT
    with pytest.raises(fe.MechanismError):
        fe.linearise(d, "nonsense")


YAML = """
units: {length: cm, quantity: mol, activation-energy: cal/mol}
phases:
- name: gas
  thermo: ideal-gas
  elements: [H, O]
  species: [A2, B2, AB, A2B, A, B, AB2, A2B2]
species:
%s
reactions:
- equation: A + B2 <=> B + AB
  rate-constant: {A: 3.5e+15, b: -0.40, Ea: 16600.0}
- equation: B + A2 = A + AB
  rate-constant: {A: 5.0e+04, b: 2.67, Ea: 6290.0}
- equation: AB + A2 <=> A + A2B
  rate-constant: {A: 2.2e+08, b: 1.51, Ea: 3430.0}
- equation: 2 AB <=> B + A2B
  rate-constant: {A: 3.6e+04, b: 2.40, Ea: -2110.0}
- equation: A + B2 + M <=> AB2 + M
  type: three-body
  rate-constant: {A: 2.8e+18, b: -0.86, Ea: 0.0}
  efficiencies: {A2B: 11.0, B2: 0.78, A: 2.0}
- equation: A + AB2 => 2 AB
  rate-constant: {A: 7.1e+13, b: 0.0, Ea: 295.0}
- equation: AB + AB (+M) <=> A2B2 (+M)
  type: falloff
  low-P-rate-constant: {A: 2.3e+18, b: -0.90, Ea: -1700.0}
  high-P-rate-constant: {A: 7.4e+13, b: -0.37, Ea: 0.0}
  Troe: {A: 0.735, T3: 94.0, T1: 1756.0, T2: 5182.0}
  efficiencies: {A2: 2.0, A2B: 6.0}
- equation: AB2 + AB2 <=> A2B2 + B2
  duplicate: true
  rate-constant: {A: 1.3e+11, b: 0.0, Ea: -1630.0}
- equation: AB2 + AB2 <=> A2B2 + B2
  duplicate: true
  rate-constant: {A: 4.2e+14, b: 0.0, Ea: 12000.0}
- equation: A2B2 + A (+M) <=> A2B + AB (+M)
  type: falloff
  low-P-rate-constant: {A: 1.0e+17, b: 0.0, Ea: 1000.0}
  high-P-rate-constant: {A: 2.4e+13, b: 0.0, Ea: 3970.0}
  Troe: {A: 0.5, T3: 100.0, T1: 2000.0}
""" % "\n".join("- name: %s\n  composition: {%s}\n  thermo:\n    model: NASA7\n    temperature-ranges: [300.0, 1000.0, 3500.0]\n    data:\n    - [%r, 0.0, 0.0, 0.0, 0.0, %r, %r]\n    - [%r, 0.0, 0.0, 0.0, 0.0, %r, %r]"
                % (n, ", ".join("%s: %d" % (e, k) for e, k in c), a1, a6, a7, a1, a6, a7) for n, c, a1, a6, a7 in SPECIES)


def test_yaml_ingestion_gives_the_same_description_as_chemkin():
    """The same made-up mechanism in the Cantera-YAML format: every array of the flat description equals the CHEMKIN one's (the thermo
    coefficients up to the 9 digits the fixed-column records carry); other units convert (kmol, m, J/kmol defaults)."""
    a = fe.parse_chemkin(TEXT, qss=["A", "B"]); b = fe.parse_yaml(YAML, qss=["A", "B"])
    assert a.species == b.species and a.elements == b.elements and a.equations == b.equations
    for f in ("rtype", "dir_mask", "reac_ptr", "reac_sp", "reac_nu", "prod_ptr", "prod_sp", "prod_nu", "eff_ptr", "eff_sp", "comp"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f
    for f in ("arr", "arr_low", "troe", "eff_val", "nasa_T", "elem_weight"):
        assert np.allclose(getattr(a, f), getattr(b, f), rtol=1e-14, atol=0.0), f
    assert np.allclose(a.nasa_lo, b.nasa_lo, rtol=1e-8) and np.allclose(a.nasa_hi, b.nasa_hi, rtol=1e-8)
    qss.validate(b, strict_balance=True)
    # the format's default units: m, kmol, J/kmol -> a bimolecular A is per (m^3/kmol), Ea per kmol
    si = YAML.replace("units: {length: cm, quantity: mol, activation-energy: cal/mol}\n", "")
    c = fe.parse_yaml(si, qss=["A", "B"])
    assert np.isclose(c.arr[0, 0], 3.5e15 * 1e-3) and np.isclose(c.arr[0, 2], 16600.0 * 1e-3) and np.isclose(c.arr[4, 0], 2.8e18 * 1e-6)
    # what is not read is an error
    for bad, msg in ((YAML.replace("Ea: 295.0", "Ea: 295.0 cal/mol"), "not a plain number"), (YAML.replace("type: three-body", "type: pressure-dependent-Arrhenius"), "type"),
                     (YAML.replace("model: NASA7", "model: NASA9", 1), "NASA9"), (YAML.replace("length: cm", "length: mm"), "units")):
        with pytest.raises(fe.MechanismError) as e:
            fe.parse_yaml(bad)
        assert msg in str(e.value), (msg, str(e.value))


# ---- the same ingestion on the syntax real mechanism files use -----------------------------------------------------------------
_NAMES2 = {"A2": "H2", "B2": "O2", "AB": "OH", "A2B": "H2O", "A": "H", "B": "O", "AB2": "HO2", "A2B2": "H2O2"}
TEXT2 = """! lower-case keywords, D exponents, tabs, species names with brackets and dashes, a THERMO block without ALL,
! every species with its own mid temperature, LOW / TROE with blanks, a three-parameter TROE line, DUPLICATE / DUP
elements
h  o
end
species
H2 O2 OH H2O
H O HO2 H2O2 CH2(S) C2H4OOH1-2
end
thermo
   300.000  1000.000  5000.000
%s
end
reactions   cal/mole  moles
H+O2<=>O+OH                 3.547D+15 -0.406 1.6599E+4   ! D exponent, no blanks in the equation
O+H2=H+OH\t\t0.508E+05   2.67   0.629E+04
2OH(+M)<=>H2O2(+M)          1.11e14 -0.37 0.0
     low  /  2.01E+17   -0.584  -2293.00/
     troe/  0.7346   94.00  1756.00  5182.00 /
     H2/2.00/ H2O/6.00/
H+O2(+M)=HO2(+M)  1.475E+12 0.60 0.00
   LOW/6.366E+20 -1.72 524.8/
   TROE/0.8 1E-30 1E+30/
   H2/2.0/ H2O/11./ O2/0.78/
H+OH+M=H2O+M     3.800E+22 -2.00 0.0
   H2/2.5/ H2O/12/
HO2+H=>2OH        7.079E+13 0.00 295.0
HO2+HO2=H2O2+O2   4.200E+14 0.00 1.1982E+04
 DUPLICATE
HO2+HO2=H2O2+O2   1.300E+11 0.00 -1.6293E+3
 DUP
CH2(S)+H2=>H2+H+H   1.0E+13 0.0 0.0
C2H4OOH1-2=>H2O2+CH2(S)  2.0E+10 0.5 1000.0
O+H2O2=>O+2OH   3.0E+12 0.0 500.0                 ! a QSS species as the collision partner, written out on both sides
CH2(S)+H2O<=>CH2(S)+H+OH  1.0E+11 0.0 9000.0
O+H2O2(+M)=>O+2OH(+M)   3.0E+12 0.0 500.0
 LOW/1.0E+16 0.0 100.0/
 TROE/0.6 100.0 1800.0/
end
""" % "\n".join([nasa_record(_NAMES2[n], c, a1, a6, a7, tmid=1000.0 + 37.0 * i) for i, (n, c, a1, a6, a7) in enumerate(SPECIES)]
                + [nasa_record("CH2(S)", [("H", 2)], 3.4, 500.0, 1.0, tmid=1392.0),
                   nasa_record("C2H4OOH1-2", [("H", 2), ("O", 2)], 5.1, -15000.0, 2.0, tmid=1388.0)])


def test_parse_the_syntax_of_real_mechanism_files():
    d = fe.parse_chemkin(TEXT2, qss=["CH2(S)", "O"])
    assert d.n_reac == 13 and d.n_qss == 2 and d.n_nqss == 8
    assert list(d.rtype) == [0, 0, 2, 2, 1, 0, 0, 0, 0, 0, 0, 0, 2]
    assert sorted(d.nasa_T[:, 1]) == sorted([1000.0 + 37.0 * i for i in range(8)] + [1392.0, 1388.0])
    assert list(d.troe[2]) == [0.7346, 94.0, 1756.0, 5182.0] and list(d.troe[3]) == [0.8, 1e-30, 1e30, 1e30]
    assert np.isclose(d.arr[0, 0], 3.547e15 * 1e-6) and np.isclose(d.arr[0, 2], 1.6599e4 * 4.184)      # cm^3/mol/s -> m^3/mol/s, cal -> J
    dl = fe.linearise(d, "reaction")
    assert dl.n_reac == 13                                   # no quadratic coupling among {CH2(S), O} in this set
    qss.validate(dl)


def test_species_on_both_sides_of_a_reaction_gets_no_term():
    """PAPER.md Eq. 3 (L62-64): wdot_i = sum_j nu_ij Q_j with the NET coefficient.  A collision partner written out on both sides
    (A + B => B + C) has nu = 0: its production rate is exactly zero, however fast the reaction is, and the other species see
    k [A][B] (closed form).  In TEXT2 (CH2(S) + H2 => H2 + 2 H next to slow H2 reactions) the float64 oracle then agrees with its
    float128 evaluation within the wdot gates; accumulated side by side, -Q + Q would leave rounding noise of Q ~ 1e11 in a rate of 1e-2."""
    import gates
    text = """ELEMENTS H O END
SPECIES A2 B2 AB END
THERMO ALL
   300.000  1000.000  3500.000
%s
END
REACTIONS MOLES KELVINS
A2 + B2 => B2 + 2AB     1.0E+20  0.0  0.0
END
""" % "\n".join([nasa_record("A2", [("H", 2)], 3.5, -1000.0, 1.0), nasa_record("B2", [("O", 2)], 3.6, -1100.0, 2.0), nasa_record("AB", [("H", 1)], 2.5, 25000.0, -0.5)])
    d = fe.parse_chemkin(text, qss=[])
    C = np.array([[0.3], [7.0], [0.01]]); T = np.array([1234.0])
    w = oracle.evaluate(oracle.OracleMech(d), C, T, 1, want_jac=False)["wdot"][:, 0]
    q = 1.0e20 * 1e-6 * 0.3 * 7.0                                   # cm^3/mol/s -> m^3/mol/s
    assert w[1] == 0.0 and np.isclose(w[0], -q, rtol=1e-14) and np.isclose(w[2], 2.0 * q, rtol=1e-14)
    d2 = fe.linearise(fe.parse_chemkin(TEXT2, qss=["CH2(S)", "O"]), "reaction")
    n = 64
    rng = np.random.default_rng(4)
    C = np.ascontiguousarray(10.0 ** rng.uniform(-4.0, 1.0, size=(d2.n_nqss, n))); T = rng.uniform(900.0, 1500.0, size=n)
    om = oracle.OracleMech(d2)
    r64 = oracle.evaluate(om, C, T, n, want_jac=False)
    r128 = oracle.evaluate(om, C, T, n, want_jac=False, mode=oracle.EXPLICIT_F128)
    g = gates.wdot_gates(r64["wdot"], r128["wdot"], r128["S"], n)
    assert g["tier2_all"] and g["tier1_frac"] >= 0.99, g
