"""ORACLE Route B (test infrastructure, NOT the product): colour-ordered Berends-Giele recursion.

BASELINE.json north_star asks for "a Berends-Giele recursion cross-check on the tiny processes".
This file computes the colour-ordered partial amplitudes A(t; g_s1 ... g_sn; tbar) of
g g -> t tbar + (n-2) g by the off-shell recursion over ordered gluon strings -- no diagram list,
no colour decomposition -- in numpy, in the CHIRAL representation with its own wavefunction
formulas, so that it shares neither the algorithm, the language nor the Dirac representation with
Route A (oracle/me_oracle.cpp).  It is compared with Route A's J_sigma in tests/test_oracle_routeb.py.

Ordered rules (same literal Feynman rules as Route A, projected on one colour ordering using
f^{abx} T^x = -i (T^a T^b - T^b T^a)):
  G(s_a..s_b) = (-i/K^2) [ g (-i) sum_c W3(G(a..c), G(c+1..b)) + (-i g^2) sum_{c<d} W4(G(a..c), G(c+1..d), G(d+1..b)) ]
  W3(A,B)^r = (A.B)(kA-kB)^r + B^r ((kB-k3).A) + A^r ((k3-kA).B),   k3 = -(kA+kB)
  W4(A,B,C) = (A.B) C + (B.C) A - 2 (A.C) B
  L(s_1..s_k) = sum_a L(s_1..s_{a-1}) [i g Gslash(s_a..s_k)] [i (qslash + m)/(q^2 - m^2 + i m Gamma)],  L() = ubar(t)
  A(sigma)    = sum_a L(s_1..s_{a-1}) [i g Gslash(s_a..s_n)] v(tbar)
"""
from __future__ import annotations

import itertools
import math

import numpy as np

_s0 = np.eye(2, dtype=complex)
_sig = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]], dtype=complex),
        np.array([[1, 0], [0, -1]], dtype=complex)]
_Z = np.zeros((2, 2), dtype=complex)
GAMMA = [np.block([[_Z, _s0], [_s0, _Z]])] + [np.block([[_Z, s], [-s, _Z]]) for s in _sig]
METRIC = np.array([1.0, -1.0, -1.0, -1.0])


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def slash(a):
    return sum(GAMMA[m] * (METRIC[m] * a[m]) for m in range(4))


def _chi(p, lam):
    px, py, pz = p[1], p[2], p[3]
    pp = math.sqrt(px * px + py * py + pz * pz)
    if px == 0.0 and py == 0.0 and pz < 0.0:
        return np.array([0, 1], dtype=complex) if lam > 0 else np.array([-1, 0], dtype=complex)
    n = 1.0 / math.sqrt(2.0 * pp * (pp + pz))
    if lam > 0:
        return n * np.array([pp + pz, px + 1j * py])
    return n * np.array([-px + 1j * py, pp + pz])


def spinor_u(p, m, lam):
    pp = math.sqrt(p[1] ** 2 + p[2] ** 2 + p[3] ** 2)
    wp, wm = math.sqrt(p[0] + pp), math.sqrt(max(p[0] - pp, 0.0))
    if m > 0:
        wm = m / wp
    w = {1: wp, -1: wm}
    x = _chi(p, lam)
    return np.concatenate([w[-lam] * x, w[lam] * x])


def spinor_v(p, m, lam):
    pp = math.sqrt(p[1] ** 2 + p[2] ** 2 + p[3] ** 2)
    wp, wm = math.sqrt(p[0] + pp), math.sqrt(max(p[0] - pp, 0.0))
    if m > 0:
        wm = m / wp
    w = {1: wp, -1: wm}
    x = _chi(p, -lam)
    return np.concatenate([-lam * w[lam] * x, lam * w[-lam] * x])


def bar(u):
    return u.conj() @ GAMMA[0]


def polvec(p, lam):
    px, py, pz = p[1], p[2], p[3]
    pt = math.hypot(px, py)
    pp = math.sqrt(pt * pt + pz * pz)
    if pt == 0.0:
        e1 = np.array([0.0, 1.0, 0.0, 0.0])
        e2 = np.array([0.0, 0.0, math.copysign(1.0, pz), 0.0])
    else:
        e1 = np.array([0.0, px * pz, py * pz, -pt * pt]) / (pp * pt)
        e2 = np.array([0.0, -py, px, 0.0]) / pt
    return (-lam * e1 - 1j * e2) / math.sqrt(2.0)


def ordered_amplitudes(momenta, gs, hel, mt=173.0, wt=0.0):
    """All n! colour-ordered amplitudes of one event for one helicity assignment.

    momenta [npar][4]; particles 0,1 incoming g, 2 = t, 3 = tbar, 4.. outgoing g; hel: +-1 per particle.
    Returns (list of orderings as tuples of gluon particle indices in lexicographic order, complex array).
    """
    p = np.asarray(momenta, dtype=float)
    npar = p.shape[0]
    gl = [0, 1] + list(range(4, npar))
    k = {i: (p[i] if i < 2 else -p[i]) for i in range(npar)}  # incoming convention
    eps = {}
    for i in gl:
        e = polvec(p[i], hel[i])
        eps[i] = e if i < 2 else e.conj()
    ub = bar(spinor_u(p[2], mt, hel[2]))
    v = spinor_v(p[3], mt, hel[3])

    gcache = {}

    def G(s):  # ordered gluon current over the string s (tuple of particle indices)
        if s in gcache:
            return gcache[s]
        if len(s) == 1:
            r = (eps[s[0]].astype(complex), k[s[0]].astype(complex))
        else:
            K = sum(k[i] for i in s).astype(complex)
            k3 = -K
            acc = np.zeros(4, dtype=complex)
            for c in range(1, len(s)):
                A, kA = G(s[:c])
                B, kB = G(s[c:])
                W3 = mdot(A, B) * (kA - kB) + B * mdot(kB - k3, A) + A * mdot(k3 - kA, B)
                acc += gs * (-1j) * W3
            for c in range(1, len(s) - 1):
                for d in range(c + 1, len(s)):
                    A, _ = G(s[:c])
                    B, _ = G(s[c:d])
                    C, _ = G(s[d:])
                    W4 = mdot(A, B) * C + mdot(B, C) * A - 2.0 * mdot(A, C) * B
                    acc += (-1j * gs * gs) * W4
            r = ((-1j / mdot(K, K)) * acc, K)
        gcache[s] = r
        return r

    lcache = {}

    def L(s):  # ordered quark-line current with trailing propagator
        if s in lcache:
            return lcache[s]
        if len(s) == 0:
            r = ub
        else:
            q = p[2] - sum(k[i] for i in s)
            den = mdot(q, q) - mt * mt + 1j * mt * wt
            prop = 1j * (slash(q) + mt * np.eye(4)) / den
            acc = np.zeros(4, dtype=complex)
            for a in range(len(s)):
                acc += L(s[:a]) @ (1j * gs * slash(G(s[a:])[0]))
            r = acc @ prop
        lcache[s] = r
        return r

    orders = list(itertools.permutations(sorted(gl)))
    out = np.zeros(len(orders), dtype=complex)
    for n, s in enumerate(orders):
        amp = 0.0
        for a in range(len(s)):
            amp += L(s[:a]) @ (1j * gs * slash(G(s[a:])[0])) @ v
        out[n] = amp
    return orders, out


# ----------------------------------------------------------------------------------------------------------------
# Route B': ONE Feynman diagram from its structural key (multichannel pins, reading R17).
# Key grammar (me_oracle.cpp build_channels): leaf = particle index; "(A,B)" three-gluon vertex; "[A,B,C]" four-gluon
# vertex; blocks attached to the quark line from t to tbar separated by "|".  Literal Feynman rules as in the header,
# colour stripped; a four-gluon vertex has three colour-structure terms, so a diagram with v of them has 3^v term
# amplitudes.  Chiral representation, numpy: shares nothing with Route A except the statement of the rules.
# ----------------------------------------------------------------------------------------------------------------
def _parse_tree(s, pos):
    if s[pos] in "([":
        close = ")" if s[pos] == "(" else "]"
        kids = []
        pos += 1
        while True:
            kid, pos = _parse_tree(s, pos)
            kids.append(kid)
            if s[pos] == ",":
                pos += 1
            else:
                assert s[pos] == close
                return tuple(kids), pos + 1
    end = pos
    while end < len(s) and s[end].isdigit():
        end += 1
    return int(s[pos:end]), end


def diagram_term_amplitudes(key, momenta, gs, hel, mt=173.0, wt=0.0):
    """Amplitudes of the colour-structure terms of the diagram `key` for one event and helicity assignment."""
    p = np.asarray(momenta, dtype=float)
    k = {i: (p[i] if i < 2 else -p[i]) for i in range(p.shape[0])}

    def tree(t):
        """list of (current, momentum) over the term choices of the four-gluon vertices below t"""
        if isinstance(t, int):
            e = polvec(p[t], hel[t])
            return [((e if t < 2 else e.conj()).astype(complex), k[t].astype(complex))]
        subs = [tree(c) for c in t]
        out = []
        for combo in itertools.product(*subs):
            K = sum(c[1] for c in combo)
            prop = -1j / mdot(K, K)
            if len(t) == 2:
                (A, kA), (B, kB) = combo
                k3 = -K
                W = mdot(A, B) * (kA - kB) + B * mdot(kB - k3, A) + A * mdot(k3 - kA, B)
                out.append((prop * gs * W, K))
            else:
                A, B, C = (c[0] for c in combo)
                for W in (mdot(A, C) * B - mdot(B, C) * A, mdot(A, B) * C - mdot(B, C) * A, mdot(A, B) * C - mdot(A, C) * B):
                    out.append((prop * (-1j * gs * gs) * W, K))
        return out

    blocks = []
    for b in key.split("|"):
        t, end = _parse_tree(b, 0)
        assert end == len(b)
        blocks.append(tree(t))
    ub = bar(spinor_u(p[2], mt, hel[2]))
    v = spinor_v(p[3], mt, hel[3])
    amps = []
    for combo in itertools.product(*blocks):
        row = ub
        q = p[2].astype(complex)
        for j, (cur, K) in enumerate(combo):
            row = row @ (1j * gs * slash(cur))
            if j + 1 < len(combo):
                q = q - K
                den = mdot(q, q) - mt * mt + 1j * mt * wt
                row = row @ (1j * (slash(q) + mt * np.eye(4)) / den)
        amps.append(row @ v)
    return np.array(amps)
