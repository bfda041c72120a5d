"""Pins for the oracle's building blocks: Dirac algebra, external wavefunctions, colour matrix, counts.

Everything is checked against what the mathematics fixes (Clifford algebra, Dirac equation, helicity
eigenvalue equation, completeness relations, SU(3) identities), never against the oracle itself.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import oracle as O
from helpers import read_golden

S0 = np.eye(2, dtype=complex)
SIG = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]], dtype=complex),
       np.array([[1, 0], [0, -1]], dtype=complex)]
Z2 = np.zeros((2, 2), dtype=complex)
# Dirac representation built here from Pauli matrices (independent of the C++ formula)
G = [np.block([[S0, Z2], [Z2, -S0]])] + [np.block([[Z2, s], [-s, Z2]]) for s in SIG]
METRIC = np.diag([1.0, -1.0, -1.0, -1.0])

MOMS = [
    (np.array([0.3, -0.4, 0.5]), 173.0),
    (np.array([120.0, 35.0, -610.0]), 173.0),
    (np.array([0.0, 0.0, 750.0]), 0.0),
    (np.array([0.0, 0.0, -750.0]), 0.0),
    (np.array([-200.0, 310.0, 4.0]), 0.0),
    (np.array([0.0, 0.0, -55.0]), 173.0),
]


def fourvec(p3, m):
    return np.array([math.sqrt(m * m + p3 @ p3), *p3])


def test_gamma_matrices_here_satisfy_clifford():
    for mu in range(4):
        for nu in range(4):
            acom = G[mu] @ G[nu] + G[nu] @ G[mu]
            assert np.allclose(acom, 2 * METRIC[mu, nu] * np.eye(4))


def test_slash_is_gamma_contraction():
    rng = np.random.default_rng(5)
    for _ in range(5):
        a = rng.normal(size=4) + 1j * rng.normal(size=4)
        want = sum(G[m] * (METRIC[m, m] * a[m]) for m in range(4))
        assert np.allclose(O.slash(a), want, atol=1e-15)


@pytest.mark.parametrize("p3,m", MOMS)
@pytest.mark.parametrize("lam", [1, -1])
def test_spinors(p3, m, lam):
    p = fourvec(p3, m)
    ps = sum(G[mu] * (METRIC[mu, mu] * p[mu]) for mu in range(4))
    u = O.wavefunction("u", p, m, lam)
    v = O.wavefunction("v", p, m, lam)
    scale = p[0]
    # Dirac equation
    assert np.abs((ps - m * np.eye(4)) @ u).max() < 1e-13 * scale**1.5
    assert np.abs((ps + m * np.eye(4)) @ v).max() < 1e-13 * scale**1.5
    # normalisation u^dagger u = 2E
    assert abs(u.conj() @ u - 2 * p[0]) < 1e-12 * scale
    assert abs(v.conj() @ v - 2 * p[0]) < 1e-12 * scale
    # helicity: Sigma.phat u = lam u ; for v the physical helicity is opposite to the Sigma.phat eigenvalue
    phat = p3 / np.linalg.norm(p3)
    sp = sum(phat[i] * np.block([[SIG[i], Z2], [Z2, SIG[i]]]) for i in range(3))
    assert np.abs(sp @ u - lam * u).max() < 1e-12 * math.sqrt(scale)
    assert np.abs(sp @ v + lam * v).max() < 1e-12 * math.sqrt(scale)
    # bar = dagger gamma0
    assert np.allclose(O.wavefunction("ubar", p, m, lam), u.conj() @ G[0])
    assert np.allclose(O.wavefunction("vbar", p, m, lam), v.conj() @ G[0])


@pytest.mark.parametrize("p3,m", MOMS)
def test_spin_sums(p3, m):
    p = fourvec(p3, m)
    ps = sum(G[mu] * (METRIC[mu, mu] * p[mu]) for mu in range(4))
    su = sum(np.outer(O.wavefunction("u", p, m, l), O.wavefunction("ubar", p, m, l)) for l in (1, -1))
    sv = sum(np.outer(O.wavefunction("v", p, m, l), O.wavefunction("vbar", p, m, l)) for l in (1, -1))
    assert np.allclose(su, ps + m * np.eye(4), atol=1e-11 * p[0])
    assert np.allclose(sv, ps - m * np.eye(4), atol=1e-11 * p[0])


@pytest.mark.parametrize("p3", [m[0] for m in MOMS])
def test_polarisation_vectors(p3):
    p = fourvec(p3, 0.0)
    e = {l: O.wavefunction("eps", p, 0.0, l) for l in (1, -1)}
    for l in (1, -1):
        dot = lambda a, b: a[0] * b[0] - a[1:] @ b[1:]
        assert abs(dot(e[l], p)) < 1e-13 * p[0]             # transverse
        assert abs(dot(e[l], e[l].conj()) + 1) < 1e-14      # normalised
        assert abs(dot(e[l], e[-l].conj())) < 1e-14         # orthogonal
        phat = p3 / np.linalg.norm(p3)
        assert np.abs(1j * np.cross(phat, e[l][1:]) - l * e[l][1:]).max() < 1e-14   # helicity eigenstate
    # completeness with the light-cone reference n = (1, -phat)
    n = np.array([1.0, *(-p3 / np.linalg.norm(p3))])
    pol = sum(np.outer(e[l], e[l].conj()) for l in (1, -1))
    want = -METRIC + (np.outer(p, n) + np.outer(n, p)) / (p[0] * n[0] + p3 @ p3 / np.linalg.norm(p3))
    assert np.allclose(pol, want, atol=1e-13)


def test_counts_and_tables():
    # P8: diagram counts named by BASELINE.json configs; helicity / colour table conventions R7, R8
    want = {"ee_mumu": (4, 16, 1, 2, 4), "gg_tt": (4, 16, 2, 3, 256), "gg_ttg": (5, 32, 6, 16, 256),
            "gg_ttgg": (6, 64, 24, 123, 512), "gg_ttggg": (7, 128, 120, 1240, 1536)}
    for p, (npar, ncomb, ncol, ndiag, denom) in want.items():
        i = O.info(p)
        assert (i["npar"], i["ncomb"], i["ncol"], i["ndiag"], i["denom"]) == (npar, ncomb, ncol, ndiag, denom)
        ht = O.helicity_table(p)
        rows = list(itertools.product([-1, 1], repeat=npar))
        assert [tuple(r) for r in ht.tolist()] == rows
        if p != "ee_mumu":
            gl = [0, 1] + list(range(4, npar))
            assert [tuple(r) for r in O.color_table(p).tolist()] == list(itertools.permutations(gl))


@pytest.mark.parametrize("n,proc", [(2, "gg_tt"), (3, "gg_ttg"), (4, "gg_ttgg"), (5, "gg_ttggg")])
def test_colour_matrix(n, proc):
    g = read_golden("color_matrix.txt")
    C = O.color_matrix(proc)
    den = g["den_%d" % n]
    Ci = C * den
    assert np.abs(Ci - np.round(Ci)).max() < 1e-9          # integers over den
    assert np.abs(C - C.T).max() == 0 or np.abs(C - C.T).max() < 1e-12
    ev = np.linalg.eigvalsh(C)
    assert ev[0] > 0                                        # positive definite
    lo, hi = g["eig_%d" % n]
    assert abs(ev[0] - lo) < 2e-3 * lo and abs(ev[-1] - hi) < 2e-3 * hi
    # diagonal = 3 (4/3)^n
    assert np.allclose(np.diag(C), 3 * (4 / 3) ** n, rtol=1e-13)
    if n in (2, 3):
        assert np.allclose(Ci[0], g["row0_%d" % n], atol=1e-9)
    if n == 4:
        assert np.allclose(Ci[0, :8], g["row0_4_head"], atol=1e-9)
        assert sorted(set(np.round(Ci).astype(int).ravel().tolist())) == sorted(int(x) for x in g["distinct_4"])
    if n == 5:
        vals = set(np.round(Ci).astype(int).ravel().tolist())
        assert len(vals) == int(g["ndistinct_5"])
        off = Ci - np.diag(np.diag(Ci))
        assert round(off.max()) == int(g["max_offdiag_5"])
    # group structure: C_{sigma tau} depends only on sigma^-1 tau
    flows = [tuple(r) for r in O.color_table(proc).tolist()]
    gl = sorted(flows[0])
    pos = {x: i for i, x in enumerate(gl)}
    seen = {}
    for a, fa in enumerate(flows):
        inv = {x: i for i, x in enumerate(fa)}
        for b, fb in enumerate(flows):
            key = tuple(inv[x] for x in fb)        # sigma^-1 tau as a permutation of positions
            v = round(Ci[a, b])
            assert seen.setdefault(key, v) == v
    # Fierz closed form for the diagonal and for one transposition of adjacent gluons:
    #   Tr(T^a1..T^an T^an..T^a1) = 3 CF^n ;  swapping two adjacent generators: CF -> (CF - CA/2) once
    cf, ca = 4 / 3, 3.0
    a = 0
    fb = list(flows[0])
    fb[0], fb[1] = fb[1], fb[0]
    b = flows.index(tuple(fb))
    assert abs(C[a, b] - 3 * cf ** (n - 1) * (cf - ca / 2)) < 1e-12
