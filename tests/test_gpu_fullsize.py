"""Full-size GPU checks at BASELINE.json's sizes, in the launch configuration bench.py times (me_compute with
selection on, default grid): sampled outputs against the oracle one by one, plus properties that hold at any
size (finite, positive, selections inside the good set / colour range, independence from the batch split)."""
import numpy as np
import pytest

from oracle import rambo as I

pytestmark = pytest.mark.gpu

ALPHAS = {"ee_mumu": 0.118, "gg_tt": 0.118, "gg_ttg": 0.118, "gg_ttgg": None, "gg_ttggg": 0.118, "gux_taptamggux": None}
# (process, precision, events = BASELINE config size (gg_ttgg: bench.py's default step), oracle samples, tolerance)
CASES = [("ee_mumu", "fp64", 16384, 256, 1e-10), ("gg_tt", "fp64", 524288, 256, 1e-10), ("gg_tt", "fp32", 524288, 256, 1e-3),
         ("gg_ttg", "fp64", 524288, 256, 1e-10), ("gg_ttg", "mixed", 524288, 256, 1e-5),
         ("gg_ttgg", "fp64", 1 << 20, 192, 1e-10), ("gg_ttgg", "fp32", 1 << 20, 192, 1e-3), ("gg_ttgg", "mixed", 1 << 20, 192, 1e-5),
         ("gg_ttggg", "fp64", 262144, 24, 1e-10), ("gg_ttggg", "fp32", 262144, 24, 1e-3),
         ("gux_taptamggux", "fp64", 524288, 256, 1e-10), ("gux_taptamggux", "fp32", 524288, 256, 1e-3)]


@pytest.mark.parametrize("process,precision,nevt,nsample,tol", CASES)
def test_fullsize_sampled_against_oracle(process, precision, nevt, nsample, tol):
    import torch
    from oracle import oracle as O
    from paper_2503_21935_b200.me import MatrixElement
    assert torch.cuda.is_available()
    mom = I.make_momenta(process, nevt, seed=1)
    gs = I.make_gs(nevt, seed=1, alphas=ALPHAS[process])
    rh, rc = I.make_rnd(nevt, seed=1)
    m = MatrixElement(process, precision)
    d_mom, d_gs = torch.from_numpy(mom).cuda(), torch.from_numpy(gs).cuda()
    mask = m.filter_helicities(d_mom, d_gs)
    me, sh, sc = m.compute(d_mom, d_gs, torch.from_numpy(rh).cuda(), torch.from_numpy(rc).cuda())
    torch.cuda.synchronize()
    me, sh, sc = me.cpu().numpy(), sh.cpu().numpy(), sc.cpu().numpy()
    # properties at any size
    assert np.all(np.isfinite(me)) and np.all(me > 0)
    assert np.all(mask[sh] == 1)
    assert sc.min() >= 0 and sc.max() < m.ncol
    # the last, ragged part of the batch computed alone gives the same numbers (no dependence on the grid)
    tail = nevt - 1000 - 37
    me2, _, _ = m.compute(d_mom[tail:].contiguous(), d_gs[tail:].contiguous())
    torch.cuda.synchronize()
    assert np.array_equal(me2.cpu().numpy(), me[tail:])
    # sampled outputs, one by one, against the oracle (stride chosen to hit first / middle / last tiles)
    idx = np.unique(np.concatenate([np.linspace(0, nevt - 1, nsample).astype(np.int64), [0, nevt - 1]]))
    ref_mask = O.good_helicities(process, mom[:min(nevt, 256)], gs[:min(nevt, 256)])
    assert np.array_equal(mask, ref_mask)
    ref = O.me(process, mom[idx], gs[idx], mask=ref_mask)
    rel = np.abs(me[idx] - ref) / ref
    assert rel.max() <= tol, f"max rel diff {rel.max():.3e} at event {idx[rel.argmax()]}"
    if precision == "fp32":
        assert np.median(rel) <= 1e-5
    m.close()


@pytest.mark.parametrize("process,nevt", [("gg_ttg", 65536), ("gg_ttgg", 65536), ("gg_ttggg", 2048), ("gux_taptamggux", 16384)])
def test_accuracy_tail_every_event(process, nevt):
    """Every event of a larger batch against the oracle (flat RAMBO has a soft/collinear tail, no cuts): the
    BASELINE tolerances hold for the worst event, not only for sampled ones (accuracy)."""
    import torch
    from oracle import oracle as O
    from paper_2503_21935_b200.me import MatrixElement
    mom = I.make_momenta(process, nevt, seed=1)
    gs = I.make_gs(nevt, seed=1, alphas=ALPHAS[process])
    ref = O.me(process, mom, gs)
    d_mom, d_gs = torch.from_numpy(mom).cuda(), torch.from_numpy(gs).cuda()
    for precision, tol in (("fp64", 1e-10), ("mixed", 1e-5), ("fp32", 1e-3)):
        m = MatrixElement(process, precision)
        m.filter_helicities(d_mom, d_gs)
        me = m.compute(d_mom, d_gs)[0].cpu().numpy()
        rel = np.abs(me - ref) / ref
        bad = np.nonzero(rel > tol)[0]
        # Where the fp64 oracle and the CUDA path disagree beyond the tolerance, the quadruple-precision build of the
        # oracle (O.me_quad, same source with a 113-bit scalar; pinned in tests/test_oracle_quad.py) decides: the CUDA
        # value must agree with IT within the stated tolerance.  No allowance beyond that (DESIGN.md section 8,
        # "accuracy tail"): seen for one nearly collinear gluon pair (s_45 / s = 1e-6) of the all-massless process,
        # where the fp64 oracle itself is frame dependent at 2e-11.
        assert len(bad) <= 64, f"{precision}: {len(bad)} events above {tol} against the fp64 oracle"
        if len(bad):
            refq = O.me_quad(process, mom[bad], gs[bad])
            relq = np.abs(me[bad] - refq) / refq
            worst = int(np.argmax(relq))
            assert relq.max() <= tol, (f"{precision}: event {bad[worst]}: rel diff {relq[worst]:.3e} against the quad oracle "
                                       f"({rel[bad[worst]]:.3e} against the fp64 oracle, which is off the quad one by "
                                       f"{abs(ref[bad[worst]] / refq[worst] - 1):.3e})")
        if precision == "fp32":
            assert np.median(rel) <= 1e-5
        m.close()
