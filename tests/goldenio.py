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


def read_philox_field_values():
    """tests/golden/philox_field_values.txt -> (values, blocks): values = [(seed, site, word or None, phi)],
    blocks = [(seed, q, (w0, w1, w2, w3))]."""
    values, blocks = [], []
    with open(os.path.join(GOLDEN, "philox_field_values.txt")) as fh:
        for ln in fh:
            t = ln.split()
            if not t or t[0].startswith("#"):
                continue
            if t[0] == "value":
                values.append((int(t[1]), int(t[2]), None if t[3] == "-" else int(t[3], 16), float(t[4])))
            elif t[0] == "block":
                blocks.append((int(t[1]), int(t[2]), tuple(int(w, 16) for w in t[3:7])))
    return values, blocks
