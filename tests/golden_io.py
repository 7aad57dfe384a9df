"""Readers for the small text fixtures under tests/golden/ (values printed in the paper)."""
import os

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def table1():
    rows = {}
    with open(os.path.join(HERE, "paper_table1.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            L, b, be, m2, m2e, xi, xie, k = line.split()
            rows[int(L)] = dict(beta=float(b), beta_err=float(be), m2=float(m2), m2_err=float(m2e),
                                xi=float(xi), xi_err=float(xie), kmcs=int(k))
    return rows


def constants():
    out = {}
    with open(os.path.join(HERE, "paper_constants.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, val = line.split()[:2]
            out[name] = float(val)
    return out
