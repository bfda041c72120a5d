"""Shared test helpers (no physics): golden-file reader."""
import os

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden(name):
    """Parse tests/golden/<name>: 'key = value' lines ('#' comments); values are floats or float lists."""
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = line.split("=", 1)
            vals = [float(x) for x in v.replace(",", " ").split()]
            out[k.strip()] = vals[0] if len(vals) == 1 else vals
    return out
