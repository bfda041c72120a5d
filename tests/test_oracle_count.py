"""Counted mode of the oracle (north_star "FLOPs per ME counted by the instrumented oracle").

The counting build is the SAME source compiled with a scalar that counts its operations, so the checks are:
it computes the same ME as the plain build, the count is a deterministic, value-independent function of the
process and of the number of helicities evaluated, it is linear in that number, and its pieces agree with
operation counts worked out by hand from the formulas the oracle's header states."""
import numpy as np
import pytest

from oracle import oracle as O
from oracle import rambo as I

GG = ["gg_tt", "gg_ttg", "gg_ttgg", "gg_ttggg"]


@pytest.mark.parametrize("proc", ["ee_mumu"] + GG)
def test_counted_build_computes_the_same_me(proc):
    mom = I.make_momenta(proc, 2, seed=6)
    for e in range(2):
        c = O.count_ops(proc, mom[e], 1.19)
        assert c["me"] == pytest.approx(O.me(proc, mom[e:e + 1], 1.19)[0], rel=1e-13)
        assert c["flops"] > 0


@pytest.mark.parametrize("proc", GG)
def test_count_is_value_independent_and_linear_in_helicities(proc):
    i = O.info(proc)
    mom = I.make_momenta(proc, 2, seed=6)
    masks = []
    for k in (1, 2, 3):
        m = np.zeros(i["ncomb"], dtype=np.uint8)
        m[[5, 9, 14][:k]] = 1
        masks.append(m)
    f = [O.count_ops(proc, mom[0], 1.19, mask=m)["flops"] for m in masks]
    assert f[1] - f[0] == f[2] - f[1] > 0                 # one more helicity costs the same every time
    assert O.count_ops(proc, mom[1], 1.3, mask=masks[2])["flops"] == f[2]   # no data-dependent branches


def test_count_pieces_match_hand_counts():
    """gg_tt, one helicity.  From the oracle's formulas (complex multiply = 4 mul + 2 add, complex add = 2 add):
    the colour sum over 2 flows is 4 terms of conj(J)*C*J (2 + 6) plus 4 complex accumulations (2) plus nothing
    else = 40; the three closures are each a row*4x4 product (16 cmul + 16 cadd = 128), a row.col product
    (4 cmul + 4 cadd = 32) and i*g_s*(..) (complex*real 2, complex*complex 6)."""
    proc = "gg_tt"
    i = O.info(proc)
    mom = I.make_momenta(proc, 1, seed=6)[0]
    one = np.zeros(i["ncomb"], dtype=np.uint8); one[3] = 1
    two = one.copy(); two[7] = 1
    per_hel = O.count_ops(proc, mom, 1.2, mask=two)["flops"] - O.count_ops(proc, mom, 1.2, mask=one)["flops"]
    cen = O.census(proc)
    colour = 4 * (2 + 6 + 2)
    closures = cen["closure"] * (128 + 32 + 2 + 6)
    jamp = cen["jamp_terms"] * (6 + 2)
    assert per_hel > colour + closures + jamp
    # the remainder is wavefunctions, the one three-gluon current and the two quark-line steps: bounded by hand
    # (each chain step = vertex 128 + i g_s 8 + slash/mass/propagator 128 + ~60; the current ~ 200; externals ~ 300)
    rest = per_hel - colour - closures - jamp
    assert 500 < rest < 1500, rest


def test_counted_flops_order_of_magnitude():
    """The oracle's count (4x4 matrices, every diagram) must exceed the generated kernel's algorithmic count
    (~0.96 MFLOP for gg_ttgg with helicity sharing) and stay within ~10x of
    SURVEY.md 8(d)'s estimate of 1.6 MFLOP per ME for the one-current-once-per-helicity accounting."""
    proc = "gg_ttgg"
    mom = I.make_momenta(proc, 1, seed=1)[0]
    f = O.count_ops(proc, mom, 1.2)["flops"]
    assert 1.0e6 < f < 2.0e7, f
