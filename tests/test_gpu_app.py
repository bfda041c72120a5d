"""The self-contained path (me_generate -> me_compute, the standalone application of PAPER.md:41) against closed-form
cross sections: sigma = <ME x phase-space weight> / (2 s) over flat RAMBO points must reproduce SURVEY.md 8(c) P2
(e+ e- -> mu+ mu-, 0.04722784 pb) and P4 (g g -> t tbar at Gamma_t = 0, 6.860453 pb) within the Monte Carlo error.
Also the measured-peak entry points used by bench.py's roofline."""
import math

import pytest

pytestmark = pytest.mark.gpu
GEV2_TO_PB = 0.3893793721e9


@pytest.mark.parametrize("process,params,sigma_pb", [("ee_mumu", None, 0.04722784), ("gg_tt", dict(wt=0.0), 6.860453)])
def test_cross_section_from_device_made_events(process, params, sigma_pb):
    import torch
    from paper_2503_21935_b200.me import MatrixElement
    m = MatrixElement(process, "fp64", params=params)
    n, s1, s2 = 1 << 20, 0.0, 0.0
    for it in range(4):
        mom, gs, rh, rc, wt = m.generate(n, seed=5, start=it * n, alphas=0.118, want_weight=True)
        if it == 0:
            m.filter_helicities(mom, gs)
        me = m.compute(mom, gs)[0]
        x = me * wt
        s1 += float(x.sum()); s2 += float((x * x).sum())
    torch.cuda.synchronize()
    ntot = 4 * n
    mean = s1 / ntot
    err = math.sqrt(max(s2 / ntot - mean * mean, 0.0) / ntot)
    flux = 2.0 * 1500.0**2
    sigma, dsigma = mean / flux * GEV2_TO_PB, err / flux * GEV2_TO_PB
    assert abs(sigma - sigma_pb) < 4.0 * dsigma and dsigma < 2e-3 * sigma_pb, (sigma, dsigma)
    m.close()


def test_measured_peaks_are_sane():
    from paper_2503_21935_b200.me import fma_peak, mma_peak
    f64, f32, dmma, tf32 = fma_peak("fp64"), fma_peak("fp32"), mma_peak("dmma"), mma_peak("tf32")
    assert 20.0 < f64 < 45.0 and 50.0 < f32 < 90.0      # B200: 37 / 74 TFLOP/s nominal
    assert 0.8 * f64 < dmma < 1.25 * f64                 # DMMA runs on the FP64 units
    assert tf32 > 2.0 * f32                              # the TF32 tensor pipe is a pipe of its own


def test_one_gluon_drell_yan_against_the_closed_form_on_the_gpu():
    """g ubar -> tau+ tau- ubar through the photon alone (Z switched off by a huge width): the crossed q qbar g result
    8 e^4 Qu^2 g_s^2 C_F N_c [(q.l+)^2 + (q.l-)^2 + (q'.l+)^2 + (q'.l-)^2] / |(l+.l-)(q.g)(q'.g)| / 96, evaluated in numpy
    from the momenta the device made -- an absolute value for the CUDA path that does not pass through the CPU checker."""
    import numpy as np
    import torch
    from paper_2503_21935_b200.me import MatrixElement
    m = MatrixElement("gux_taptamux", "fp64", params=dict(wz=1e20))
    mom, gs, rh, rc = m.generate(1 << 16, seed=4)
    m.filter_helicities(mom, gs)
    me = m.compute(mom, gs)[0].cpu().numpy()
    p, g = mom.cpu().numpy(), gs.cpu().numpy()
    dot = lambda a, b: a[:, 0] * b[:, 0] - (a[:, 1:] * b[:, 1:]).sum(1)
    gl, q, lp, lm, q2 = (p[:, k] for k in range(5))
    e2 = 4.0 * math.pi / 132.507
    num = dot(q, lp)**2 + dot(q, lm)**2 + dot(q2, lp)**2 + dot(q2, lm)**2
    closed = 8.0 * e2 * e2 * (4.0 / 9.0) * g * g * 4.0 * num / np.abs(dot(lp, lm) * dot(q, gl) * dot(q2, gl)) / 96.0
    rel = np.abs(me - closed) / closed
    # flat RAMBO without cuts: nearly collinear points lose digits in the closed form's own invariants
    assert np.median(rel) < 1e-13 and np.quantile(rel, 0.999) < 1e-9 and rel.max() < 1e-6
    m.close()


def test_two_to_two_closed_forms_event_by_event_on_the_gpu():
    """SURVEY.md 8(c) P1 and P3 evaluated in numpy from the device-made momenta, against the CUDA path directly:
    gg -> t tbar at Gamma_t = 0:  ME = g_s^4 [1/(6 t1 t2) - 3/8] [t1^2 + t2^2 + rho - rho^2/(4 t1 t2)], t_i = 2 k_i.p_t / s;
    e+ e- -> mu+ mu-:  ME = u^2 (|A_LL|^2 + |A_RR|^2) + t^2 (|A_LR|^2 + |A_RL|^2), A_XY = e^2/s + g_X g_Y/(s - MZ^2 + i MZ GZ)."""
    import numpy as np
    from paper_2503_21935_b200.me import MatrixElement
    dot = lambda a, b: a[:, 0] * b[:, 0] - (a[:, 1:] * b[:, 1:]).sum(1)
    n = 1 << 16
    m = MatrixElement("gg_tt", "fp64", params=dict(wt=0.0))
    mom, gs, rh, rc = m.generate(n, seed=6)
    m.filter_helicities(mom, gs)
    me = m.compute(mom, gs)[0].cpu().numpy()
    p, g = mom.cpu().numpy(), gs.cpu().numpy()
    s = 1500.0**2
    t1, t2, rho = 2.0 * dot(p[:, 0], p[:, 2]) / s, 2.0 * dot(p[:, 1], p[:, 2]) / s, 4.0 * 173.0**2 / s
    closed = g**4 * (1.0 / (6.0 * t1 * t2) - 0.375) * (t1**2 + t2**2 + rho - rho**2 / (4.0 * t1 * t2))
    assert np.max(np.abs(me - closed) / closed) < 1e-10
    m.close()

    m = MatrixElement("ee_mumu", "fp64")
    mom, gs, rh, rc = m.generate(n, seed=6)
    m.filter_helicities(mom, None)
    me = m.compute(mom, None)[0].cpu().numpy()
    p = mom.cpu().numpy()
    mz, wz, alpha, gf = 91.188, 2.441, 1.0 / 132.507, 1.16639e-5
    mw2 = 0.5 * mz**2 + math.sqrt(0.25 * mz**4 - math.pi * alpha * mz**2 / (math.sqrt(2.0) * gf))
    sw2 = 1.0 - mw2 / mz**2
    e2 = 4.0 * math.pi * alpha
    gz = math.sqrt(e2 / (sw2 * (1.0 - sw2)))
    gl, gr = gz * (sw2 - 0.5), gz * sw2
    prop = 1.0 / (s - mz * mz + 1j * mz * wz)
    a = {x + y: e2 / s + cx * cy * prop for x, cx in (("L", gl), ("R", gr)) for y, cy in (("L", gl), ("R", gr))}
    t = -2.0 * dot(p[:, 1], p[:, 3])    # (p_e- - p_mu-)^2
    u = -2.0 * dot(p[:, 1], p[:, 2])    # (p_e- - p_mu+)^2
    closed = u**2 * (abs(a["LL"])**2 + abs(a["RR"])**2) + t**2 * (abs(a["LR"])**2 + abs(a["RL"])**2)
    assert np.max(np.abs(me - closed) / closed) < 1e-10
    m.close()
