"""me_generate (device-side seeded inputs) against its numpy oracle oracle/rambo.py: same
counter-based uniforms (bit-exact), same RAMBO algorithm (fp64; equal up to the rounding of the device math
library), physical momenta, and an ME computed from device-made inputs equal to the ME from oracle-made inputs."""
import numpy as np
import pytest

from oracle import rambo as I

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("process", ["ee_mumu", "gg_tt", "gg_ttg", "gg_ttgg", "gg_ttggg", "gux_taptamux", "gux_taptamggux"])
def test_generate_matches_harness(process):
    import torch
    from paper_2503_21935_b200.me import MatrixElement
    assert torch.cuda.is_available()
    n, start, seed = 5000 + 77, 12345, 3
    m = MatrixElement(process, "fp64")
    mom, gs, rh, rc, wt = m.generate(n, seed=seed, start=start, want_weight=True)
    torch.cuda.synchronize()
    mom, gs, rh, rc, wt = (x.cpu().numpy() for x in (mom, gs, rh, rc, wt))
    ref_mom, ref_wt = I.make_momenta(process, n, seed=seed, start=start, return_weight=True)
    ref_rh, ref_rc = I.make_rnd(n, seed=seed, start=start)
    # the uniforms are integer arithmetic + one exact scaling: bit-exact
    assert np.array_equal(rh, ref_rh) and np.array_equal(rc, ref_rc)
    assert np.allclose(gs, I.make_gs(n, seed=seed, alphas=None, start=start), rtol=1e-15, atol=0)
    # momenta: log/sin/cos/sqrt differ by an ulp between libm and the device library
    scale = 1500.0
    assert np.max(np.abs(mom - ref_mom)) <= 1e-10 * scale
    assert np.allclose(wt, ref_wt, rtol=1e-10, atol=0)
    # physical: momentum conservation and on-shell masses
    tot = mom[:, 0] + mom[:, 1] - mom[:, 2:].sum(axis=1)
    assert np.max(np.abs(tot)) <= 1e-9 * scale
    m2 = mom[:, :, 0] ** 2 - (mom[:, :, 1:] ** 2).sum(axis=2)
    masses = np.array([0.0, 0.0] + [173.0 * t for t in I.PROCESSES[process]["final_top"]])
    assert np.max(np.abs(m2 - masses[None, :] ** 2)) <= 1e-9 * scale ** 2
    # fixed alpha_s
    _, gs2, _, _ = m.generate(16, seed=seed, alphas=0.118)
    assert np.allclose(gs2.cpu().numpy(), np.sqrt(4 * np.pi * 0.118), rtol=1e-15)
    m.close()


def test_me_from_device_inputs_equals_me_from_host_inputs():
    import torch
    from paper_2503_21935_b200.me import MatrixElement
    n = 4096 + 5
    m = MatrixElement("gg_ttgg", "fp64")
    mom, gs, rh, rc = m.generate(n, seed=1)
    m.filter_helicities(mom, gs)
    me_d, sh_d, sc_d = m.compute(mom, gs, rh, rc)
    hm = torch.from_numpy(I.make_momenta("gg_ttgg", n, seed=1)).cuda()
    hg = torch.from_numpy(I.make_gs(n, seed=1)).cuda()
    hrh, hrc = (torch.from_numpy(x).cuda() for x in I.make_rnd(n, seed=1))
    me_h, sh_h, sc_h = m.compute(hm, hg, hrh, hrc)
    torch.cuda.synchronize()
    a, b = me_d.cpu().numpy(), me_h.cpu().numpy()
    assert np.max(np.abs(a - b) / b) <= 1e-9
    assert np.mean(sh_d.cpu().numpy() == sh_h.cpu().numpy()) > 0.999
    assert np.mean(sc_d.cpu().numpy() == sc_h.cpu().numpy()) > 0.999
    m.close()
