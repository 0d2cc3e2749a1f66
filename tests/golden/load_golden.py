"""Parser for the text fixtures in this directory (no arithmetic)."""
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


def load(name: str) -> dict:
    out = {}
    with open(os.path.join(_HERE, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, _, val = line.partition(":")
            rows = [[float(x) for x in part.split()] for part in val.split("|")]
            out[key.strip()] = rows
    return out


def fig5_tables():
    """E_t[r] = [100*(t+1) + 10*r + 1, 100*(t+1) + 10*r + 2], as typed in the fixture's header."""
    return [np.array([[100 * (t + 1) + 10 * r + 1, 100 * (t + 1) + 10 * r + 2] for r in range(3)],
                     dtype=np.float32) for t in range(4)]
