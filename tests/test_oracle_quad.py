"""Pins of the quadruple-precision build of the oracle (O.me_quad, -DORC_QUAD): the arbiter of the accuracy-tail test.

It is the same source as the fp64 oracle with a 113-bit scalar, so it inherits that oracle's pins provided it really is
the same computation (pin 1) and really carries more digits (pins 2, 3)."""
import numpy as np
import pytest

from oracle import oracle as O
from oracle import rambo as I


def mdot(a, b):
    return a[..., 0] * b[..., 0] - a[..., 1] * b[..., 1] - a[..., 2] * b[..., 2] - a[..., 3] * b[..., 3]


@pytest.mark.parametrize("process,n", [("ee_mumu", 64), ("gg_tt", 64), ("gg_ttg", 32), ("gg_ttgg", 12), ("gg_ttggg", 1),
                                       ("gux_taptamux", 32), ("gux_taptamggux", 12)])
def test_quad_equals_fp64_oracle_on_ordinary_events(process, n):
    """Pin 1: same computation.  On well-conditioned events the two builds agree to fp64 rounding."""
    mom = I.make_momenta(process, n, seed=21)
    gs = I.make_gs(n, seed=21, alphas=None)
    a, b = O.me(process, mom, gs), O.me_quad(process, mom, gs)
    assert np.abs(a / b - 1).max() < 1e-12


def test_quad_against_the_gg_tt_closed_form():
    """Pin 2: the textbook gg -> t tbar result (tests/test_oracle_pins.py P3), here evaluated in numpy's extended
    precision; the quad build must sit at the rounding of its double inputs and output, not further off than the fp64 oracle."""
    n = 512
    mom = I.make_momenta("gg_tt", n, seed=1).astype(np.longdouble)
    gs = I.make_gs(n, seed=1).astype(np.longdouble)
    mt = np.longdouble(173.0)
    s = mdot(mom[:, 0] + mom[:, 1], mom[:, 0] + mom[:, 1])
    t1, t2 = 2 * mdot(mom[:, 0], mom[:, 2]) / s, 2 * mdot(mom[:, 1], mom[:, 2]) / s
    rho = 4 * mt * mt / s
    closed = gs**4 * (1 / (6 * t1 * t2) - np.longdouble(3) / 8) * (t1**2 + t2**2 + rho - rho**2 / (4 * t1 * t2))
    m64, g64 = mom.astype(np.float64), gs.astype(np.float64)
    q = np.abs(O.me_quad("gg_tt", m64, g64, params=dict(wt=0.0)) / closed - 1).astype(np.float64)
    d = np.abs(O.me("gg_tt", m64, g64, params=dict(wt=0.0)) / closed - 1).astype(np.float64)
    # the inputs are on shell to 1e-16 only, which the closed form and the diagrams see differently near t1 t2 -> rho/4
    print("median / max: quad", np.median(q), q.max(), " fp64", np.median(d), d.max())
    # (forward / backward points: the closed form itself loses digits there, as in P3, for both builds alike)
    assert np.median(q) < 2e-15 and q.max() < 1e-10
    assert np.median(q) <= np.median(d)


def test_quad_is_frame_independent_where_fp64_is_not():
    """Pin 3: more digits where it matters.  The most collinear gluon pair of the tail-test batch (s_45 / s ~ 1e-6) makes
    the fp64 oracle frame dependent at the 1e-10 level; with exactly transformed inputs the quad build must not be.
    Exact transforms: rotations by multiples of 90 degrees and reflections (signed permutations of the axes)."""
    process, nevt = "gux_taptamggux", 16384
    mom = I.make_momenta(process, nevt, seed=1)
    gs = I.make_gs(nevt, seed=1, alphas=None)
    s = 2 * mdot(mom[:, 0], mom[:, 1])
    s45 = 2 * mdot(mom[:, 4], mom[:, 5])
    e = int(np.argmin(s45 / s))
    assert s45[e] / s[e] < 1e-5
    p0 = mom[e:e + 1]
    frames = [p0]
    for perm, sign in (((0, 2, 3, 1), (1, 1, 1, 1)), ((0, 3, 1, 2), (1, 1, 1, 1)), ((0, 2, 1, 3), (1, 1, -1, 1)), ((0, 1, 3, 2), (1, -1, 1, 1))):
        frames.append(p0[:, :, list(perm)] * np.array(sign, dtype=np.float64))   # proper rotations (det +1), exact in fp64
    d = np.array([O.me(process, f, gs[e:e + 1])[0] for f in frames])
    q = np.array([O.me_quad(process, f, gs[e:e + 1])[0] for f in frames])
    spread = lambda v: np.abs(v / v[0] - 1).max()
    print("frame spread: quad", spread(q), " fp64", spread(d), " s45/s", s45[e] / s[e], "event", e)
    assert spread(q) < 1e-14, spread(q)
    assert spread(q) < spread(d) or spread(d) < 1e-14
