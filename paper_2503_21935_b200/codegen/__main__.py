"""python -m paper_2503_21935_b200.codegen [outdir]  -- write csrc/gen/proc_*.cuh (build step)."""
import sys

from .generate import generate_all

if __name__ == "__main__":
    generate_all(sys.argv[1] if len(sys.argv) > 1 else None)
