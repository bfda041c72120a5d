"""Pins of oracle.select (reading R11).

The paper is silent on the selection rule, so nothing here can pin the READING against the paper ("parity
unpinned" stays in DESIGN.md).  What the mathematics fixes once R11 is adopted is tested instead, each fact
chosen so that a plausible slip in the scan (<= for <, cumulating masked rows, a wrong fallback index, colour
weights taken from the wrong axis) fails one of them:
  * limits of the random number: r -> 0+ picks the first good row, r -> 1- the last good row;
  * the total of the running sums is the filtered ME of O.me (a different code path: no scan);
  * the probability of picking h is |M_h|^2 / S and of picking c is w_c / sum w: chi-square over 1e5 seeded
    uniforms on one fixed event, with the expected probabilities from O.me_helicities / O.jamps;
  * a masked-out row is never selected;
  * the colour weights are sum over good h of |J_c(h)|^2 with J from the single-helicity entry point O.jamps.
"""
import numpy as np
import pytest

from oracle import oracle as O
from oracle import rambo as I


def _one_event(proc, seed=5):
    mom = I.make_momenta(proc, 1, seed=seed)
    return mom, 1.21


def test_select_limits_of_the_random_number():
    proc = "gg_ttg"
    mom, gs = _one_event(proc)
    i = O.info(proc)
    mask = np.zeros(i["ncomb"], dtype=np.uint8)
    good_rows = [3, 6, 7, 12, 21, 29]          # hand-made mask: first good row 3, last good row 29
    mask[good_rows] = 1
    tiny, almost1 = np.array([5e-324]), np.array([1.0 - 2.0 ** -53])
    lo = O.select(proc, mom, gs, tiny, tiny, mask=mask)
    hi = O.select(proc, mom, gs, almost1, almost1, mask=mask)
    assert lo["selhel"][0] == 3 and hi["selhel"][0] == 29
    assert lo["selcol"][0] == 0 and hi["selcol"][0] == i["ncol"] - 1
    # r = 0 exactly: 0 < cum of the first good row (its |M_h|^2 is positive) -> still the first good row
    z = O.select(proc, mom, gs, np.zeros(1), np.zeros(1), mask=mask)
    assert z["selhel"][0] == 3 and z["selcol"][0] == 0


@pytest.mark.parametrize("proc", ["gg_tt", "gg_ttg", "gg_ttgg"])
def test_select_total_is_the_filtered_me(proc):
    n = 5
    mom = I.make_momenta(proc, n, seed=9)
    gs = I.make_gs(n, seed=9)
    rh, rc = I.make_rnd(n, seed=9)
    i = O.info(proc)
    rng = np.random.default_rng(3)
    mask = (rng.random(i["ncomb"]) < 0.6).astype(np.uint8)
    mask[1] = 1
    sel = O.select(proc, mom, gs, rh, rc, mask=mask)
    assert np.allclose(sel["me"], O.me(proc, mom, gs, mask=mask), rtol=1e-14, atol=0)
    assert np.allclose(sel["cumhel"][:, -1] / i["denom"], O.me(proc, mom, gs, mask=mask), rtol=1e-14, atol=0)
    # the running sums never move on a masked-out row and never decrease
    d = np.diff(np.concatenate([np.zeros((n, 1)), sel["cumhel"]], axis=1), axis=1)
    assert np.all(d[:, mask == 0] == 0) and np.all(d >= 0)
    assert np.all(mask[sel["selhel"]] == 1)


def _chi2(obs, p):
    n = obs.sum()
    keep = p > 0
    assert np.all(obs[~keep] == 0), "an outcome of probability zero was selected"
    exp = n * p[keep]
    return float(((obs[keep] - exp) ** 2 / exp).sum()), int(keep.sum()) - 1


@pytest.mark.parametrize("proc", ["gg_tt", "gg_ttg"])
def test_select_frequencies_follow_the_weights(proc):
    nsamp = 100_000
    mom1, gs = _one_event(proc, seed=12)
    i = O.info(proc)
    mask = np.ones(i["ncomb"], dtype=np.uint8)
    mask[[2, 5, i["ncomb"] - 1]] = 0                     # some rows masked out, including the last one
    mom = np.repeat(mom1, nsamp, axis=0)
    rh, rc = I.make_rnd(nsamp, seed=77)
    sel = O.select(proc, mom, gs, rh, rc, mask=mask)
    # expected probabilities from entry points that do no scanning
    mh = O.me_helicities(proc, mom1, gs)[0] * mask
    ph = mh / mh.sum()
    w = np.zeros(i["ncol"])
    for h in np.nonzero(mask)[0]:
        w += np.abs(O.jamps(proc, mom1[0], gs, int(h))) ** 2
    pc = w / w.sum()
    for got, p in ((sel["selhel"], ph), (sel["selcol"], pc)):
        obs = np.bincount(got, minlength=len(p)).astype(float)
        chi2, dof = _chi2(obs, p)
        assert chi2 < dof + 6.0 * np.sqrt(2.0 * dof) + 10.0, f"chi2 {chi2:.1f} for {dof} dof"
        # every outcome with a sizeable probability does occur (a scan that stops early would miss the tail)
        assert np.all(obs[p * nsamp > 50] > 0)
    assert np.all(mask[sel["selhel"]] == 1)
    # colour weights are the helicity-summed |J_c|^2 of the good rows
    assert np.allclose(sel["cumcol"][0], np.cumsum(w), rtol=1e-12)


def test_select_agrees_with_a_sorted_search():
    """np.searchsorted restates 'first index with r*S < cum': a library routine instead of the scan."""
    proc, n = "gg_ttg", 400
    mom = I.make_momenta(proc, n, seed=2)
    gs = I.make_gs(n, seed=2)
    rh, rc = I.make_rnd(n, seed=2)
    mask = O.good_helicities(proc, mom, gs)
    sel = O.select(proc, mom, gs, rh, rc, mask=mask)
    good = np.nonzero(mask)[0]
    for e in range(n):
        cum = sel["cumhel"][e, good]
        k = np.searchsorted(cum, rh[e] * cum[-1], side="right")
        assert sel["selhel"][e] == good[min(k, len(good) - 1)]
        cc = sel["cumcol"][e]
        k = np.searchsorted(cc, rc[e] * cc[-1], side="right")
        assert sel["selcol"][e] == min(k, len(cc) - 1)
