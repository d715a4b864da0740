"""Writes tests/golden/oracle_toys.txt: wdot, C_QSS and the Jacobian of the CPU oracle (explicit fp64 mode) on the toy mechanisms and cfg1
at a few seeded states, one number per line with 17 significant digits.  Calls only `oracle/` and the seeded input generators
(`qss_synth/`); nothing here comes from the CUDA path.  The paper prints no value that applies to a synthetic mechanism (all its
tables are for its own mechanisms), so this fixture is a REGRESSION pin: it freezes the oracle's arithmetic as of the
commit that wrote it, so that a later change of the oracle cannot pass unnoticed (tests/test_oracle_pins.py::test_golden_regression).
Usage: python tests/golden/make_golden.py   (from the repository root)"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import qss_synth  # noqa: E402

CASES = [("toy1", 3), ("toy2", 3), ("toy3", 3), ("toy_dag", 3), ("toy_nonqss", 3), ("cfg1", 2)]


def values(name, n):
    if name.startswith("cfg"):
        mech = qss_synth.config_mechanism(int(name[3])); C, T = qss_synth.config_states(int(name[3]), n)
    else:
        mech = getattr(qss_synth, name)(); C, T = qss_synth.make_states(mech.n_nqss, n, seed=12)
    o = oracle.evaluate(oracle.OracleMech(mech), C, T, n)
    e = oracle.evaluate_energy(oracle.OracleMech(mech), C, T, n)
    return np.concatenate([o["wdot"][:, :n].ravel(), o["cqss"][:, :n].ravel(), o["jac"][:, :, :n].ravel(), e["tdot"][:n], e["erow"][:, :n].ravel()])


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_toys.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ (explicit fp64 mode); regression pin, not a value of the paper\n")
        for name, n in CASES:
            v = values(name, n)
            f.write("# %s %d cells %d values: wdot, cqss, jac, tdot, erow (C order, cells innermost)\n" % (name, n, v.size))
            for x in v:
                f.write("%.17e\n" % x)
    print(path)


if __name__ == "__main__":
    main()
