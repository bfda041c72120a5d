"""CPU tests of the product's host side: the build-time generator (colour algebra, diagram structure),
the C-ABI library's exported symbols, and the binding's refusal to run without a GPU.
No oracle code is used to produce expected values here: pins are the SU(3) facts of
tests/golden/color_matrix.txt and the diagram counts of BASELINE.json configs.
"""
import ctypes
import os
import re
from fractions import Fraction

import numpy as np
import pytest

from helpers import read_golden
from paper_2503_21935_b200.codegen import colour, diagrams

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = read_golden("color_matrix.txt")


@pytest.fixture(scope="module")
def structures():
    return {n: diagrams.build(n) for n in (2, 3, 4, 5)}


def test_diagram_counts(structures):
    # BASELINE.json configs: 3 / 16 / 123 / 1240 diagrams, 2 / 6 / 24 / 120 colours
    assert [structures[n].ndiag for n in (2, 3, 4, 5)] == [3, 16, 123, 1240]
    assert [len(structures[n].flows) for n in (2, 3, 4, 5)] == [2, 6, 24, 120]
    assert [structures[n].denom for n in (2, 3, 4, 5)] == [256, 256, 512, 1536]


def test_colour_matrix_pins(structures):
    for n in (2, 3, 4, 5):
        st = structures[n]
        c = np.array(st.cmat_num, dtype=np.float64) / st.cmat_den
        assert st.cmat_den == int(GOLD[f"den_{n}"])
        assert np.array_equal(c, c.T)
        ev = np.linalg.eigvalsh(c)
        lo, hi = GOLD[f"eig_{n}"]
        assert ev[0] > 0 and abs(ev[0] - lo) < 2e-3 * max(1, lo) and abs(ev[-1] - hi) < 1e-2
        # diagonal = N_c C_F^n = 3 (4/3)^n
        assert all(Fraction(st.cmat_num[i][i], st.cmat_den) == 3 * Fraction(4, 3) ** n for i in range(len(c)))
    assert structures[2].cmat_num[0] == [int(x) for x in GOLD["row0_2"]]
    assert structures[3].cmat_num[0] == [int(x) for x in GOLD["row0_3"]]
    assert structures[4].cmat_num[0][:8] == [int(x) for x in GOLD["row0_4_head"]]
    assert sorted(set(v for r in structures[4].cmat_num for v in r)) == sorted(int(x) for x in GOLD["distinct_4"])
    offdiag = [structures[5].cmat_num[i][j] for i in range(120) for j in range(120) if i != j]
    assert max(offdiag) == int(GOLD["max_offdiag_5"])
    assert len(set(v for r in structures[5].cmat_num for v in r)) == int(GOLD["ndistinct_5"])


def test_colour_matrix_group_structure(structures):
    # C_{sigma tau} depends only on sigma^-1 tau
    st = structures[4]
    fl = st.flows
    seen = {}
    for i, s in enumerate(fl):
        for j, t in enumerate(fl):
            rel = tuple(s.index(x) for x in t)
            assert seen.setdefault(rel, st.cmat_num[i][j]) == st.cmat_num[i][j]


def test_fierz_against_explicit_generators():
    # Tr(T^a T^b T^a T^b) summed = -2/3 and Tr(T^a T^a T^b T^b) = 16/3 for SU(3), from explicit matrices
    lam = np.zeros((8, 3, 3), dtype=complex)
    lam[0][0, 1] = lam[0][1, 0] = 1
    lam[1][0, 1] = -1j; lam[1][1, 0] = 1j
    lam[2][0, 0] = 1; lam[2][1, 1] = -1
    lam[3][0, 2] = lam[3][2, 0] = 1
    lam[4][0, 2] = -1j; lam[4][2, 0] = 1j
    lam[5][1, 2] = lam[5][2, 1] = 1
    lam[6][1, 2] = -1j; lam[6][2, 1] = 1j
    lam[7] = np.diag([1, 1, -2]) / np.sqrt(3)
    T = lam / 2
    abab = sum(np.trace(T[a] @ T[b] @ T[a] @ T[b]) for a in range(8) for b in range(8)).real
    aabb = sum(np.trace(T[a] @ T[a] @ T[b] @ T[b]) for a in range(8) for b in range(8)).real
    c = colour.colour_matrix([(0, 1), (1, 0)])
    assert abs(float(c[0][0]) - aabb) < 1e-12 and abs(float(c[0][1]) - abab) < 1e-12


def test_commutator_signs_and_reflection(structures):
    # [[a,b],c] = abc - bac - cab + cba
    s = colour.commutator(colour.commutator(colour.leaf(0), colour.leaf(1)), colour.leaf(4))
    assert dict(s) == {(0, 1, 4): 1, (1, 0, 4): -1, (4, 0, 1): -1, (4, 1, 0): 1}
    # every tree's strings have unit coefficients; ordered currents exist for every canonical sequence
    st = structures[4]
    assert all(abs(c) == 1 for t in st.trees for c in t.strings.values())
    assert len(st.ordered) == 6 + 12 + 12
    # photon decoupling: the sum over all orderings of a tree's strings vanishes (commutators are traceless sums)
    assert all(sum(t.strings.values()) == 0 for t in st.trees if t.kind != "leaf")


def test_generated_sources_are_deterministic(tmp_path):
    from paper_2503_21935_b200.codegen.generate import generate_all
    a = generate_all(str(tmp_path / "a"), only=["gg_ttg"])
    b = generate_all(str(tmp_path / "b"), only=["gg_ttg"])
    assert [os.path.basename(x) for x in a] == [os.path.basename(x) for x in b]
    for x, y in zip(a, b):
        assert open(x).read() == open(y).read()
    txt = open([x for x in a if os.path.basename(x) == "proc_gg_ttg.cuh"][0]).read()
    assert "vvv_current" in txt and "vvvv_currents" in txt and "row_prop" in txt and txt.count("J[") == 6


def _declared_symbols():
    hdr = open(os.path.join(ROOT, "include", "me_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(me_[a-z_]+)\s*\(", hdr)))


def test_library_exports_every_declared_symbol():
    """The C-ABI library loads on a machine without a GPU and exports everything include/me_b200.h declares."""
    from paper_2503_21935_b200 import me
    if not os.path.exists(me.LIB_PATH):
        from paper_2503_21935_b200 import build
        build.build()
    lib = ctypes.CDLL(me.LIB_PATH)
    names = _declared_symbols()
    assert set(names) == set(me.EXPORTS)
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/me_b200.h but not exported"


def test_no_cpu_fallback_without_gpu():
    """Without a CUDA device the product must fail loudly (no CPU path)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2503_21935_b200 import me
    if not os.path.exists(me.LIB_PATH):
        pytest.skip("library not built")
    with pytest.raises(me.MEError):
        me.MatrixElement("gg_tt", "fp64")


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2503_21935_b200")
    for root, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(root, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "me_oracle" not in txt, f


def test_group_layout_tables_are_consistent():
    """Lane-group layout (codegen/emit_group.py): slots, level tables and per-role word streams."""
    import itertools
    from paper_2503_21935_b200.codegen import emit_group as EG
    for n, nslot, ntwin in ((4, 22, 6), (5, 105, 0)):
        g = EG.Group("t", n)
        # n = 4: the even-length currents are stored twice (+J and -J), the tables point at the copy with the sign
        assert len(g.slot) == nslot == sum(len(g.level_seqs[L]) for L in range(1, n)) and len(g.twin) == ntwin
        assert g.nslot == nslot + ntwin and sorted(g.twin.values()) == list(range(nslot, nslot + ntwin))
        assert all(len(s) % 2 == 0 for s in g.twin)
        # canonical sequences: one of each {seq, reversed seq}; the reflection sign is (-1)^(len+1)
        for L in range(1, n + 1):
            allseq = [s for c in itertools.combinations(range(n), L) for s in itertools.permutations(c)]
            assert len(g.level_seqs[L]) * (1 if L == 1 else 2) == len(allseq)
            for s in allseq:
                can, sgn = EG.canonical(s)
                assert can in g.level_seqs[L] and sgn == (1 if can == s else (-1) ** (L + 1))
        # level tables: every operand slot was produced by a lower level; masks partition the task's set
        for L in range(2, n + 1):
            tab, nv3, nv4 = g.level_table(L), L - 1, (L - 1) * (L - 2) // 2
            W = 2 + nv3 + nv4
            assert len(tab) == W * len(g.level_seqs[L])
            lower = {g.slot[s] for k in range(1, L) for s in g.level_seqs[k]} | {v for s, v in g.twin.items() if len(s) < L}
            for t, seq in enumerate(g.level_seqs[L]):
                w = tab[t * W:(t + 1) * W]
                assert (w[0] >> 8) & 31 == EG.mask_of(seq)
                for x in w[2:]:
                    assert ntwin == 0 or (x >> 31) == 0          # with twins no word carries a sign bit
                for x in w[2:2 + nv3]:
                    assert (x & 255) in lower and ((x >> 8) & 255) in lower
                    assert ((x >> 16) & 31) | ((x >> 21) & 31) == EG.mask_of(seq) and ((x >> 16) & 31) & ((x >> 21) & 31) == 0
                for x in w[2 + nv3:]:
                    assert {x & 255, (x >> 8) & 255, (x >> 16) & 255} <= lower
        # race freedom of the warp-synchronous tree: the leaves occupy slots 0..n-1 (lane i writes slot i), every other
        # slot (and twin) has exactly ONE writing task, and (checked above) every reader sits at a higher level, i.e.
        # behind the __syncwarp() that closes the writer's level
        assert [g.slot[(i,)] for i in range(n)] == list(range(n))
        writers = list(range(n))
        for L in range(2, n):
            tab, W = g.level_table(L), 2 + (L - 1) + (L - 1) * (L - 2) // 2
            for t in range(len(g.level_seqs[L])):
                writers.append(tab[t * W] & 255)
                if (tab[t * W] >> 16) & 255:
                    writers.append((tab[t * W] >> 16) & 255)
        assert sorted(writers) == list(range(g.nslot))
        # top level: every flow is initialised exactly once (as a canonical sequence or as its reverse)
        W = 2 + (n - 1) + (n - 1) * (n - 2) // 2
        top = g.level_table(n)
        flows = [f for t in range(len(g.level_seqs[n])) for f in (top[t * W + 1] & 127, (top[t * W + 1] >> 8) & 127)]
        assert sorted(flows) == list(range(len(g.flows)))
        # role streams: same length for every first gluon, every flow is a leaf of exactly one role
        leaves = []
        for s1 in range(n):
            st = g.role_stream(s1)
            assert len(st) == len(g.role_stream(0))
            leaves += [(w >> 16) & 127 for w in st if (w >> 8) & 31 == (1 << n) - 1]
            assert ntwin == 0 or all((w >> 31) == 0 for w in st if (w >> 8) & 31 != (1 << n) - 1)
        assert sorted(leaves) == list(range(len(g.flows)))
        fl = g.flops()
        assert fl["per_gluon_combination"] == fl["tree"] + fl["walk"] + fl["colour"]


def test_diagram_tables_cover_every_channel_and_flow():
    """codegen/emit_diag.py (multichannel tables): one channel per Feynman diagram, every closure has a channel, every
    colour flow is reached by some diagram, and the sizes are those of the diagram counts 3 / 16 / 123 / 1240."""
    from paper_2503_21935_b200.codegen import diagrams, emit_diag
    for name, ngl, ndiag in (("gg_tt", 2, 3), ("gg_ttg", 3, 16), ("gg_ttgg", 4, 123)):
        st = diagrams.build(ngl)
        dg = emit_diag.Diagrams(name, st)
        assert len(dg.keys) == ndiag == st.ndiag and dg.keys == sorted(set(dg.keys))
        assert {dg.chan[c[2]] for c in dg.closures} == set(range(ndiag))
        reached = [any(row[c] for row in dg.allowed) for c in range(len(st.flows))]
        assert all(reached)
        # a diagram made of single gluons on the quark line feeds exactly one flow (the order of attachment)
        for k, row in zip(dg.keys, dg.allowed):
            if "(" not in k and "[" not in k:
                assert sum(row) == 1 and st.flows[row.index(1)] == tuple(int(x) for x in k.split("|"))
