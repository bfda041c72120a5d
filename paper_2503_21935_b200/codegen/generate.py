"""Build step: generate the per-process CUDA headers under csrc/gen/."""
from __future__ import annotations

import os

from . import diagrams, emit

PROCESSES = {"gg_tt": 2, "gg_ttg": 3, "gg_ttgg": 4, "gg_ttggg": 5}
_CSRC = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "csrc")


def generate_all(outdir=None, only=None):
    outdir = outdir or os.path.join(_CSRC, "gen")
    os.makedirs(outdir, exist_ok=True)
    written = []
    for name, ngl in PROCESSES.items():
        if only and name not in only:
            continue
        st = diagrams.build(ngl)
        text = emit.Emitter(name, st).emit()
        cm, fl = emit.tables(st)
        text += f"// constant tables of {name}\n"
        text += f"#define ME_CMAT_{name.upper()} {{{cm}}}\n#define ME_FLOWS_{name.upper()} {{{fl}}}\n"
        path = os.path.join(outdir, f"proc_{name}.cuh")
        old = open(path).read() if os.path.exists(path) else None
        if old != text:
            with open(path, "w") as f:
                f.write(text)
        written.append(path)
    return written
