"""Readers for the small text fixtures under tests/golden/ (each file carries its own citation)."""
import os
from fractions import Fraction

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_sections(name):
    """'[section]' headed blocks of whitespace-separated rationals -> {section: list of rows of Fraction}."""
    sec, cur = {}, None
    with open(os.path.join(GOLDEN, name)) as fh:
        for ln in fh:
            ln = ln.strip()
            if not ln or ln.startswith("#"):
                continue
            if ln.startswith("["):
                cur = ln[1:-1]
                sec[cur] = []
                continue
            sec[cur].append([Fraction(t) for t in ln.split()])
    return sec


def as_array(rows, dtype=np.float64):
    return np.array([[float(v) for v in r] for r in rows], dtype=dtype)


def read_philox_kat():
    out = []
    with open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) as fh:
        for ln in fh:
            ln = ln.strip()
            if not ln or ln.startswith("#"):
                continue
            w = [int(t, 16) for t in ln.split()]
            out.append((w[0:4], w[4:6], tuple(w[6:10])))
    return out
