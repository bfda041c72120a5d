"""Harness inputs: counter-based PRNG and RAMBO."""
import math

import numpy as np
import pytest

from oracle import rambo as I


def test_uniforms_are_counter_based_and_open_interval():
    a = I.uniforms(1, 0, 0, 1000)
    b = I.uniforms(1, 0, 500, 500)
    assert np.array_equal(a[500:], b)                 # pure function of the index
    assert not np.array_equal(a, I.uniforms(2, 0, 0, 1000))
    assert not np.array_equal(a, I.uniforms(1, 1, 0, 1000))
    u = I.uniforms(1, 3, 0, 200000)
    assert u.min() > 0 and u.max() < 1
    assert abs(u.mean() - 0.5) < 4 / math.sqrt(12 * len(u))
    assert abs(u.var() - 1 / 12) < 1e-3


@pytest.mark.parametrize("proc", list(I.PROCESSES))
def test_rambo_momenta_are_physical(proc):
    p = I.make_momenta(proc, 512, seed=1)
    npar = I.PROCESSES[proc]["npar"]
    assert p.shape == (512, npar, 4)
    tot = p[:, :2].sum(1) - p[:, 2:].sum(1)
    assert np.abs(tot).max() < 1e-9                   # momentum conservation
    m2 = p[..., 0] ** 2 - (p[..., 1:] ** 2).sum(-1)
    masses = [0, 0] + [173.0 * t for t in I.PROCESSES[proc]["final_top"]]
    assert np.abs(m2 - np.array(masses) ** 2).max() < 1e-6
    assert (p[..., 0] > 0).all()
    # chunked generation gives the same events
    q = I.make_momenta(proc, 100, seed=1, start=412)
    assert np.array_equal(q, p[412:])


def test_rambo_weights():
    # N=2: the flat weight is the two-body phase space beta/(8 pi)
    _, w = I.make_momenta("gg_tt", 8, return_weight=True)
    beta = math.sqrt(1 - 4 * 173.0**2 / 1500.0**2)
    assert np.allclose(w, beta / (8 * math.pi), rtol=1e-12)
    _, w = I.make_momenta("ee_mumu", 8, return_weight=True)
    assert np.allclose(w, 1 / (8 * math.pi), rtol=1e-12)
    # N=3 massless: Phi_3 = s / (2 (4 pi)^3 ) * 1/2 ... closed form (pi/2)^2 s (2pi)^-5 / 2
    r = I.uniforms(5, 0, 0, 12 * 16).reshape(16, 3, 4)
    _, w = I.rambo(r, [0, 0, 0], 1500.0)
    assert np.allclose(w, 1500.0**2 / (256 * math.pi**3), rtol=1e-12)
    # N=3 massive (t tbar g): <W> must equal the Dalitz-plot integral (219.272)
    _, w = I.make_momenta("gg_ttg", 200000, seed=2, return_weight=True)
    assert abs(w.mean() - 219.272) < 4 * w.std() / math.sqrt(len(w))


def test_lorentz_transform_preserves_invariants():
    p = I.make_momenta("gg_ttgg", 64, seed=1)
    q = I.lorentz_transform(p, seed=3)
    md = lambda a, b: a[..., 0] * b[..., 0] - (a[..., 1:] * b[..., 1:]).sum(-1)
    for i in range(6):
        for j in range(6):
            assert np.allclose(md(p[:, i], p[:, j]), md(q[:, i], q[:, j]), rtol=1e-9, atol=1e-6)
    assert np.abs(q[:, :, 1:3]).min() > 0             # general frame: incoming no longer along z
