"""Pins of the oracle's mixed EW+QCD class (Table 4: g u~ -> tau+ tau- g g u~):
g ubar -> tau+ tau- + (n-1) g + ubar through a photon or a Z, n = 1, 2, 3 gluons.

None of these re-types the oracle: an absolute closed form (the classic q qbar g photon-exchange result, crossed),
the exact factorisation of the electroweak part helicity by helicity, gauge invariance on every gluon, conservation
of the quark current, Lorentz invariance, coupling scaling, Bose symmetry, diagram and helicity counts.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from oracle import rambo as I

DY = ["gux_taptamux", "gux_taptamgux", "gux_taptamggux"]
NGL = {"gux_taptamux": 1, "gux_taptamgux": 2, "gux_taptamggux": 3}
NO_Z = dict(wz=1e20)   # Z exchange suppressed by s / (MZ GZ) ~ 1e-16 (a huge mass would destroy sw^2 by cancellation)


def mdot(a, b):
    return a[..., 0] * b[..., 0] - (a[..., 1:] * b[..., 1:]).sum(-1)


def ew_constants(mz=91.188, aewm1=132.507, gf=1.16639e-5):
    """(alpha, G_F, M_Z) scheme of DESIGN.md reading R5, written from its definition."""
    alpha = 1.0 / aewm1
    mw2 = 0.5 * mz**2 + math.sqrt(0.25 * mz**4 - math.pi * alpha * mz**2 / (math.sqrt(2.0) * gf))
    sw2 = 1.0 - mw2 / mz**2
    e = math.sqrt(4.0 * math.pi * alpha)
    g = e / math.sqrt(sw2 * (1.0 - sw2))
    coup = {}
    for name, q, t3 in (("u", 2.0 / 3.0, 0.5), ("tau", -1.0, -0.5)):
        coup[name] = dict(Q=q, L=g * (t3 - q * sw2), R=g * (-q * sw2))
    return e, coup


def test_diagram_flow_and_helicity_counts():
    # q qbar + n g has 1 / 3 / 16 diagrams; a diagram whose quark line carries k gluon trees has k + 1 places for the
    # boson, and there are two bosons.  n = 1: 2 x 2; n = 2: 2 x (2 x 3 + 1 x 2); n = 3: 2 x (6 x 4 + 6 x 3 + 4 x 2)
    for proc, nd, ncol, denom in zip(DY, (4, 16, 100), (1, 2, 6), (96, 96, 192)):
        i = O.info(proc)
        n = NGL[proc]
        assert (i["npar"], i["ncomb"], i["ncol"], i["ndiag"], i["denom"]) == (n + 4, 1 << (n + 4), ncol, nd, denom)
        # massless fermion lines conserve helicity: incoming and outgoing ubar alike, tau+ tau- opposite
        mom = I.make_momenta(proc, 4, seed=5)
        good = O.good_helicities(proc, mom, 1.2)
        ht = O.helicity_table(proc)
        want = (ht[:, 1] == ht[:, -1]) & (ht[:, 2] == -ht[:, 3])
        assert np.array_equal(good.astype(bool), want) and good.sum() == 1 << (n + 2)
        assert np.array_equal(O.color_table(proc)[0], [0] + list(range(4, n + 3)))


def test_closed_form_one_gluon_photon_exchange():
    """Sum over spins and colours of |M|^2 for q qbar g l+ l- through a photon (the e+ e- -> q qbar g result, all
    momenta incoming): 8 e^4 Qq^2 g_s^2 C_F N_c [(q.l+)^2 + (q.l-)^2 + (q'.l+)^2 + (q'.l-)^2] / |(l+.l-)(q.g)(q'.g)|."""
    proc = "gux_taptamux"
    mom = I.make_momenta(proc, 64, seed=9)
    gs = I.make_gs(64, seed=9)
    e, coup = ew_constants()
    g, q, lp, lm, q2 = (mom[:, k] for k in range(5))
    num = mdot(q, lp)**2 + mdot(q, lm)**2 + mdot(q2, lp)**2 + mdot(q2, lm)**2
    closed = 8.0 * e**4 * coup["u"]["Q"]**2 * gs**2 * 4.0 * num / np.abs(mdot(lp, lm) * mdot(q, g) * mdot(q2, g))
    got = O.me(proc, mom, gs, params=NO_Z)
    assert np.allclose(got, closed / 96.0, rtol=1e-11, atol=0)


@pytest.mark.parametrize("proc", DY)
def test_electroweak_factorisation_helicity_by_helicity(proc):
    """One boson between two massless lines: |M_h|^2(photon + Z) / |M_h|^2(photon) = |1 + g_X^u g_Y^tau s /
    (e^2 Qu Qtau (s - MZ^2 + i MZ GZ))|^2, X (Y) the chirality of the quark (lepton) line: an incoming antiquark of
    helicity +1 is the antiparticle of the LEFT-handed quark; an outgoing tau- of helicity -1 is left-handed."""
    mom = I.make_momenta(proc, 2, seed=4)
    gs = 1.2
    e, coup = ew_constants()
    full = O.me_helicities(proc, mom, gs)
    phot = O.me_helicities(proc, mom, gs, params=NO_Z)
    ht = O.helicity_table(proc)
    mz, wz = 91.188, 2.441
    seen = set()
    for ev in range(2):
        s = mdot(mom[ev, 2] + mom[ev, 3], mom[ev, 2] + mom[ev, 3])
        for h in range(len(ht)):
            if not (ht[h, 1] == ht[h, -1] and ht[h, 2] == -ht[h, 3]):   # helicity-violating rows: rounding noise only
                assert full[ev, h] < 1e-20 * full[ev].max() and phot[ev, h] < 1e-20 * phot[ev].max()
                continue
            x = "L" if ht[h, 1] > 0 else "R"
            y = "L" if ht[h, 3] < 0 else "R"
            seen.add(x + y)
            r = abs(1.0 + coup["u"][x] * coup["tau"][y] * s / (e * e * coup["u"]["Q"] * coup["tau"]["Q"] * (s - mz * mz + 1j * mz * wz)))**2
            assert full[ev, h] / phot[ev, h] == pytest.approx(r, rel=1e-10)
    assert seen == {"LL", "LR", "RL", "RR"}


@pytest.mark.parametrize("proc", DY)
def test_ward_identity_on_every_gluon_and_quark_current_conservation(proc):
    i = O.info(proc)
    mom = I.make_momenta(proc, 2, seed=11)
    ht = O.helicity_table(proc)
    hels = [h for h in range(i["ncomb"]) if ht[h, 1] == ht[h, -1] and ht[h, 2] == -ht[h, 3]][::5]
    gluons = [0] + list(range(4, i["npar"] - 1))
    for e in range(2):
        for h in hels:
            j0 = O.jamps(proc, mom[e], 1.2, h)
            assert np.abs(j0).max() > 0
            for leg in gluons:
                jw = O.jamps(proc, mom[e], 1.2, h, ward_leg=leg)
                assert np.abs(jw).max() < 1e-10 * mom[e, leg, 0] * np.abs(j0).max()
            # lepton current -> boson momentum: the amplitude vanishes (vector and axial currents of a massless line)
            jq = O.jamps(proc, mom[e], 1.2, h, ward_leg=-2)
            assert np.abs(jq).max() < 1e-10 * 1500.0 * np.abs(j0).max() / 1e-2


@pytest.mark.parametrize("proc", DY)
def test_lorentz_invariance_and_coupling_scaling(proc):
    nev = 3
    mom = I.make_momenta(proc, nev, seed=21)
    a = O.me(proc, mom, 1.2)
    b = O.me(proc, I.lorentz_transform(mom, seed=8), 1.2)
    assert np.allclose(a, b, rtol=1e-9, atol=0)
    assert np.allclose(O.me(proc, mom, 1.2) / O.me(proc, mom, 1.1), (1.2 / 1.1)**(2 * NGL[proc]), rtol=1e-12)
    # alpha_EM^2: both exchanges scale with e^4 in this scheme only through e and sw; photon-only is exactly e^4
    r = O.me(proc, mom, 1.2, params=dict(NO_Z, aewm1=100.0)) / O.me(proc, mom, 1.2, params=NO_Z)
    assert np.allclose(r, (132.507 / 100.0)**2, rtol=1e-10)


def test_bose_symmetry_of_the_final_gluons():
    for proc, a, b in (("gux_taptamgux", None, None), ("gux_taptamggux", 4, 5)):
        mom = I.make_momenta(proc, 2, seed=2)
        if a is None:
            continue
        sw = mom.copy()
        sw[:, [a, b]] = mom[:, [b, a]]
        assert np.allclose(O.me(proc, mom, 1.2), O.me(proc, sw, 1.2), rtol=1e-11, atol=0)


def _boost_to(p, Q):
    """Boost momenta p (given in the rest frame of their sum) to the frame where the sum is Q."""
    m = math.sqrt(mdot(Q, Q))
    b, g = Q[1:] / Q[0], Q[0] / m
    bp, b2 = (p[:, 1:] * b).sum(1), (b * b).sum()
    out = np.empty_like(p)
    out[:, 0] = g * (p[:, 0] + bp)
    out[:, 1:] = p[:, 1:] + ((g - 1.0) * bp / b2)[:, None] * b + (g * p[:, 0])[:, None] * b
    return out


def test_soft_gluon_limit_two_gluons_to_one():
    """A soft final gluon k factorises (eikonal approximation, colour conservation T_q + T_q' + T_g = 0):
    ME(2 gluons) -> g_s^2 [C_A (w_qg + w_q'g) - (C_A - 2 C_F) w_qq'] ME(1 gluon), w_ij = p_i.p_j / ((p_i.k)(p_j.k)),
    with corrections linear in the gluon energy.  Ties the normalisation and the colour factors of the two-gluon process
    to the one-gluon process, whose value is fixed by the closed form above."""
    base = I.make_momenta("gux_taptamux", 1, seed=3)[0]          # 0 g, 1 ubar -> 2 tau+, 3 tau-, 4 ubar
    P = base[0] + base[1]
    d = np.array([1.0, 0.3, -0.5, math.sqrt(0.66)])
    gs = 1.2
    me1 = O.me("gux_taptamux", base[None], gs)[0]
    dev = []
    for eps in (1e-3, 1e-4, 1e-5):
        k = eps * 750.0 * d
        Q = P - k
        fin = _boost_to(base[2:] * (math.sqrt(mdot(Q, Q)) / 1500.0), Q)   # the hard final state takes the exact recoil
        mom = np.stack([base[0], base[1], fin[0], fin[1], k, fin[2]])[None]
        assert np.allclose(mom[0, :2].sum(0), mom[0, 2:].sum(0), atol=1e-9) and np.allclose(mdot(fin, fin), 0, atol=1e-6)
        w = lambda a, b: mdot(a, b) / (mdot(a, k) * mdot(b, k))
        g, q, q2 = base[0], base[1], base[4]
        eik = 3.0 * (w(q, g) + w(q2, g)) - (3.0 - 8.0 / 3.0) * w(q, q2)
        dev.append(O.me("gux_taptamgux", mom, gs)[0] / (gs * gs * eik * me1) - 1.0)
    assert abs(dev[2]) < 5e-5 and dev[1] == pytest.approx(10 * dev[2], rel=0.05) and dev[0] == pytest.approx(100 * dev[2], rel=0.1)
