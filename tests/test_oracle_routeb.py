"""P14: Route A (Feynman diagrams + colour decomposition, C++) == Route B (colour-ordered Berends-Giele
recursion, numpy, chiral representation) on the tiny processes (BASELINE.json north_star)."""
import numpy as np
import pytest

from oracle import bg_numpy as B
from oracle import oracle as O
from oracle import rambo as I


@pytest.mark.parametrize("proc,nev", [("gg_tt", 3), ("gg_ttg", 3), ("gg_ttgg", 1), ("gg_ttggg", 1)])
@pytest.mark.parametrize("wt", [0.0, 1.4915])
def test_route_a_equals_route_b(proc, nev, wt):
    i = O.info(proc)
    mom = I.make_momenta(proc, nev, seed=17)
    ht = O.helicity_table(proc)
    flows = [tuple(r) for r in O.color_table(proc).tolist()]
    gs = 1.17
    hels = {"gg_ttgg": [0, 7, 21, 38, 63], "gg_ttggg": [5, 42, 77, 100, 126]}.get(proc, range(i["ncomb"]))
    for e in range(nev):
        for h in hels:
            ja = O.jamps(proc, mom[e], gs, h, params=dict(wt=wt))
            orders, jb = B.ordered_amplitudes(mom[e], gs, ht[h], mt=173.0, wt=wt)
            assert [tuple(o) for o in orders] == flows
            scale = np.abs(ja).max()
            if scale < 1e-14:
                assert np.abs(jb).max() < 1e-12
                continue
            # the two routes use different Dirac representations and spinor phase conventions: J_sigma may
            # differ by ONE phase common to all sigma of this helicity; moduli and relative phases must agree
            k = np.argmax(np.abs(ja))
            phase = ja[k] / jb[k]
            assert abs(abs(phase) - 1) < 1e-10
            assert np.abs(ja - phase * jb).max() < 1e-10 * scale


def test_route_b_colour_summed_me_matches():
    proc = "gg_ttg"
    mom = I.make_momenta(proc, 2, seed=3)
    ht = O.helicity_table(proc)
    C = O.color_matrix(proc)
    for e in range(2):
        tot = 0.0
        for h in range(32):
            _, jb = B.ordered_amplitudes(mom[e], 1.2, ht[h], wt=1.4915)
            tot += (jb.conj() @ C @ jb).real
        assert tot / 256 == pytest.approx(O.me(proc, mom[e:e + 1], 1.2)[0], rel=1e-11)
