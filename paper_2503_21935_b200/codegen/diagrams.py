"""Feynman-diagram structure of g g -> t tbar + (n-2) g for the build-time generator.

PAPER.md:11/21: in the paper the diagram code is produced by MG5aMC's code generator, which is not
available here; this module is the small generator that replaces it for the configs of BASELINE.json.

Every tree diagram is the quark line t -> tbar with gluon trees ("blocks") attached in some order; a
gluon tree over a set S of external gluons is a leaf, a three-gluon vertex joining two sub-trees or a
four-gluon vertex joining three (three colour/Lorentz terms).  With the phase-stripped rules of
csrc/me_ops.cuh the colour coefficient of every (diagram, flow) pair is the +-1 of the nested
commutator expansion, so that

    J_sigma = sum_{j=0}^{n-1}  Psi(s_1..s_j) . Jord-slash(s_{j+1}..s_n) . v
    Psi(s_1..s_k) = [ sum_{j<k} Psi(s_1..s_j) Jord-slash(s_{j+1}..s_k) ] (qslash+m)/(q^2-m^2+i m G)
    Jord(seq)     = sum_{trees T on set(seq)} sign_T(seq) J_T           (sign of seq in T's commutator)

i.e. the jamp of flow sigma is accumulated flow by flow ("jamp accumulation per colour flow",
BASELINE.json north_star (c)) from the same Feynman diagrams the oracle enumerates one by one.
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

from . import colour


@dataclass
class Tree:
    tid: int
    legs: tuple            # sorted gluon particle indices
    kind: str              # "leaf" | "v3" | "v4"
    children: tuple = ()   # child tree ids
    term: int = 0          # v4: 0,1,2
    group: int = -1        # v4: id shared by the three terms of one vertex (one op computes all three)
    strings: colour.Strings = field(default_factory=colour.Strings)
    ndiag: int = 1         # number of Feynman topologies this tree stands for (always 1; v4 terms share)


@dataclass
class Structure:
    ngl: int
    gluons: tuple                 # gluon particle indices (0, 1, 4, ...)
    npar: int
    trees: list                   # all Tree objects; ids are indices
    trees_on: dict                # sorted leg tuple -> [tree ids]
    flows: list                   # tuples, lexicographic permutations of gluons
    ordered: dict                 # canonical ordered seq -> [(sign, tree id)]
    ndiag: int
    cmat_num: list                # integer numerators of the colour matrix
    cmat_den: int
    denom: int                    # spin/colour average x identical-particle factor


def _partitions2(legs):
    """Unordered 2-partitions {A,B} of the tuple legs, lowest leg in A."""
    first, rest = legs[0], legs[1:]
    for r in range(0, len(rest)):
        for extra in itertools.combinations(rest, r):
            a = (first,) + extra
            b = tuple(x for x in rest if x not in extra)
            if b:
                yield a, b


def _partitions3(legs):
    """Unordered 3-partitions {A,B,C}: lowest leg in A, lowest of the remainder in B."""
    for a, rest in _partitions2(legs):
        for b, c in _partitions2(rest):
            yield a, b, c


def canonical(seq):
    """Representative of {seq, reversed(seq)} and the reflection sign: Jord(rev) = (-1)^(len+1) Jord(seq)."""
    seq = tuple(seq)
    if len(seq) == 1 or seq[0] < seq[-1]:
        return seq, 1
    return tuple(reversed(seq)), (-1) ** (len(seq) + 1)


def build(ngl: int, gluons=None, npar=None, denom=None, ndiag_factor=None) -> Structure:
    """gg -> t tbar + (ngl-2) g by default.  Other quark-line processes with the same colour structure pass their own
    gluon particle indices, particle count, averaging factor and a function ndiag(count over ordered block
    partitions) -> number of Feynman diagrams (see build_dy)."""
    gluons = (0, 1) + tuple(range(4, ngl + 2)) if gluons is None else tuple(gluons)
    npar = ngl + 2 if npar is None else npar
    trees, trees_on = [], {}

    def new_tree(**kw):
        t = Tree(tid=len(trees), **kw)
        trees.append(t)
        trees_on.setdefault(t.legs, []).append(t.tid)
        return t

    for g in gluons:
        new_tree(legs=(g,), kind="leaf", strings=colour.leaf(g))
    ngroup = 0
    for size in range(2, ngl + 1):
        for legs in itertools.combinations(gluons, size):
            for a_legs, b_legs in _partitions2(legs):
                for a in trees_on[a_legs]:
                    for b in trees_on[b_legs]:
                        new_tree(legs=legs, kind="v3", children=(a, b),
                                 strings=colour.commutator(trees[a].strings, trees[b].strings))
            for a_legs, b_legs, c_legs in _partitions3(legs):
                for a in trees_on[a_legs]:
                    for b in trees_on[b_legs]:
                        for c in trees_on[c_legs]:
                            sa, sb, sc = trees[a].strings, trees[b].strings, trees[c].strings
                            cols = (colour.commutator(colour.commutator(sa, sb), sc),
                                    colour.commutator(colour.commutator(sa, sc), sb),
                                    colour.commutator(colour.commutator(sb, sc), sa))
                            for term in range(3):
                                new_tree(legs=legs, kind="v4", children=(a, b, c), term=term, group=ngroup,
                                         strings=cols[term])
                            ngroup += 1

    # ordered currents: Jord(seq) = sum_T sign_T(seq) J_T; keep canonical sequences only
    allord = {}
    for size in range(2, ngl + 1):
        for seq in itertools.permutations(gluons, size):
            terms = []
            for tid in trees_on[tuple(sorted(seq))]:
                c = trees[tid].strings.get(tuple(seq), 0)
                assert c in (-1, 0, 1)
                if c:
                    terms.append((c, tid))
            allord[tuple(seq)] = terms
    ordered = {}
    for seq, terms in allord.items():
        can, sgn = canonical(seq)
        if can == seq:
            ordered[seq] = terms
        else:
            # reflection identity of colour-ordered currents (checked, not assumed)
            assert {tid: c for c, tid in allord[can]} == {tid: c * sgn for c, tid in terms}

    # diagram count: ordered set partitions of the gluons into blocks x tree topologies per block
    # (the three terms of a four-gluon vertex are one topology: count trees whose v4 nodes all have term 0)
    primary = {}
    for t in trees:
        primary[t.tid] = all(primary[c] for c in t.children) and (t.kind != "v4" or t.term == 0)
    ntop = {legs: sum(1 for t in tids if primary[t]) for legs, tids in trees_on.items()}

    def count(rem):
        if not rem:
            return 1
        total = 0
        for r in range(1, len(rem) + 1):
            for blk in itertools.combinations(rem, r):
                rest = tuple(x for x in rem if x not in blk)
                total += ntop[blk] * count(rest)
        return total

    ndiag = count(gluons)
    if ndiag_factor is not None:
        # an extra colourless attachment on the quark line (one of nb bosons): a diagram with k blocks has k + 1 places
        def count_k(rem, k):
            if not rem:
                return k + 1
            total = 0
            for r in range(1, len(rem) + 1):
                for blk in itertools.combinations(rem, r):
                    rest = tuple(x for x in rem if x not in blk)
                    total += ntop[blk] * count_k(rest, k + 1)
            return total
        ndiag = ndiag_factor * count_k(gluons, 0)
    flows = colour.flows_of(gluons)
    cm = colour.colour_matrix(flows)
    den = 1
    for row in cm:
        for x in row:
            if den % x.denominator:
                den = den * x.denominator // _gcd(den, x.denominator)
    num = [[int(x * den) for x in row] for row in cm]
    fact = 1
    for k in range(2, ngl - 1):
        fact *= k
    return Structure(ngl=ngl, gluons=gluons, npar=npar, trees=trees, trees_on=trees_on, flows=flows,
                     ordered=ordered, ndiag=ndiag, cmat_num=num, cmat_den=den,
                     denom=(4 * 64 * fact) if denom is None else denom)


def build_dy(ngl: int = 3) -> Structure:
    """g ubar -> tau+ tau- + (ngl-1) g + ubar (Table 4 for ngl = 3):
    particles 0 = g, 1 = ubar (in), 2 = tau+, 3 = tau-, 4.. = g, last = ubar (out); one quark line with ngl gluons and one
    photon / Z -> tau pair attached: the colour structure is that of a quark line with ngl gluons."""
    gluons = (0,) + tuple(range(4, ngl + 3))
    fact = 1
    for k in range(2, ngl):
        fact *= k
    return build(ngl, gluons=gluons, npar=ngl + 4, denom=4 * 24 * fact, ndiag_factor=2)


def _gcd(a, b):
    while b:
        a, b = b, a % b
    return a
