"""Colour algebra for the build-time generator (exact integer / rational arithmetic, no floats).

g g -> t tbar + (n-2) g in the trace basis T_sigma = (T^{a_s1} ... T^{a_sn})_{ij}:

* ``commutator`` / ``Strings``: a gluon tree's colour tensor, contracted with T^x on its parent
  line, is a nested commutator of its leaves (f^{abx} T^x = -i [T^a, T^b]); we keep only the REAL
  sign of every string because the powers of -i are common to a whole diagram class and drop out
  (DESIGN.md "phase stripping").
* ``colour_matrix``: C_{sigma tau} = sum_{a_1..a_n} Tr(T^{a_s1}..T^{a_sn} T^{a_tn}..T^{a_t1}) reduced
  with the SU(N) Fierz identity  T^a_{ij} T^a_{kl} = 1/2 (d_il d_jk - 1/N d_ij d_kl).

Nothing here is shared with oracle/ (which sums explicit Gell-Mann matrices by brute force).
"""
from __future__ import annotations

import itertools
from fractions import Fraction
from functools import lru_cache

NC = 3


class Strings(dict):
    """Formal integer combination of words (tuples of gluon leg labels)."""

    def add(self, word, coef):
        v = self.get(word, 0) + coef
        if v:
            self[word] = v
        else:
            self.pop(word, None)


def leaf(leg) -> Strings:
    s = Strings()
    s[(leg,)] = 1
    return s


def concat(a: Strings, b: Strings) -> Strings:
    r = Strings()
    for wa, ca in a.items():
        for wb, cb in b.items():
            r.add(wa + wb, ca * cb)
    return r


def commutator(a: Strings, b: Strings) -> Strings:
    """[a, b] = a b - b a."""
    r = concat(a, b)
    for w, c in concat(b, a).items():
        r.add(w, -c)
    return r


# ---------------------------------------------------------------------------------------------
# traces:  a product of traces is a tuple of words; every index appears exactly twice overall.
# ---------------------------------------------------------------------------------------------
def _canon(word):
    """Cyclic canonical form of a trace word."""
    if not word:
        return word
    k = min(range(len(word)), key=lambda i: word[i:] + word[:i])
    return word[k:] + word[:k]


@lru_cache(maxsize=None)
def _eval(traces) -> Fraction:
    """Value of prod_k Tr(word_k) summed over all repeated adjoint indices."""
    traces = tuple(sorted(_canon(w) for w in traces))
    for ti, w in enumerate(traces):
        if not w:
            continue
        a = w[0]
        rest = traces[:ti] + traces[ti + 1:]
        if a in w[1:]:
            # Tr(T^a B T^a C) = 1/2 [ Tr(B) Tr(C) - 1/N Tr(B C) ]
            j = w.index(a, 1)
            b, c = w[1:j], w[j + 1:]
            return Fraction(1, 2) * (_eval(rest + (b, c)) - Fraction(1, NC) * _eval(rest + (b + c,)))
        # the partner sits in another trace: Tr(T^a B) Tr(T^a C) = 1/2 [ Tr(B C) - 1/N Tr(B) Tr(C) ]
        for tj, w2 in enumerate(rest):
            if a in w2:
                k = w2.index(a)
                c = w2[k + 1:] + w2[:k]
                b = w[1:]
                rest2 = rest[:tj] + rest[tj + 1:]
                return Fraction(1, 2) * (_eval(rest2 + (b + c,)) - Fraction(1, NC) * _eval(rest2 + (b, c)))
        raise ValueError("unpaired index")
    # only empty traces left: Tr(1) = N each
    return Fraction(NC) ** len(traces)


def colour_matrix(flows):
    """C[s][t] as Fractions for the list of flows (tuples of leg labels, all permutations of one set).

    (T_s)_{ij} conj((T_t)_{ij}) summed over i, j and all adjoint indices = Tr(T_s T_t^dagger), and
    T_t^dagger is the reversed word (the generators are hermitian).
    """
    n = len(flows)
    out = [[None] * n for _ in range(n)]
    for s in range(n):
        for t in range(n):
            word = tuple(flows[s]) + tuple(reversed(flows[t]))
            out[s][t] = _eval((word,))
    return out


def flows_of(gluons):
    """Colour flows in the exported order: lexicographic permutations of the gluon particle indices."""
    return [tuple(p) for p in itertools.permutations(sorted(gluons))]
