"""Multichannel on the GPU (me_compute_multichannel, reading R17) against the oracle:
channel numbering, single-diagram-enhancement numerator / denominator (fp64 in every build, tolerance 1e-10), the
channel-restricted colour selection, and the ME itself unchanged."""
import numpy as np
import pytest

from oracle import rambo as I

pytestmark = pytest.mark.gpu

NEVT = {"gg_tt": 2048 + 77, "gg_ttg": 1024 + 77, "gg_ttgg": 256 + 13, "gg_ttggg": 24}
ALPHAS = {"gg_tt": 0.118, "gg_ttg": 0.118, "gg_ttgg": None, "gg_ttggg": 0.118}
TOL = {"fp64": 1e-10, "mixed": 1e-5, "fp32": 1e-3}


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.mark.parametrize("process", list(NEVT))
def test_channel_table_matches_oracle(torch_cuda, process):
    from oracle import oracle as O
    from paper_2503_21935_b200.me import MatrixElement
    m = MatrixElement(process, "fp64")
    assert m.channel_table() == O.channel_keys(process) and len(m.channel_table()) == m.ndiag
    m.close()


@pytest.mark.parametrize("process,precision", [("gg_tt", "fp64"), ("gg_ttg", "fp64"), ("gg_ttg", "fp32"), ("gg_ttgg", "fp64"),
                                               ("gg_ttgg", "mixed"), ("gg_ttggg", "fp64")])
def test_multichannel_matches_oracle(torch_cuda, process, precision):
    from oracle import oracle as O
    from paper_2503_21935_b200.me import MatrixElement
    torch = torch_cuda
    dev = torch.device("cuda:0")
    n = NEVT[process]
    mom = I.make_momenta(process, n, seed=3)
    gs = I.make_gs(n, seed=3, alphas=ALPHAS[process])
    rh, rc = I.make_rnd(n, seed=3)
    ndiag = O.info(process)["ndiag"]
    # a mix of channels in one launch, including the first and the last one
    chan = (I.uniforms(3, 7, 0, n) * ndiag).astype(np.int32)
    chan[0], chan[-1] = 0, ndiag - 1
    m = MatrixElement(process, precision)
    d = lambda x: torch.from_numpy(x).to(dev)
    mask = m.filter_helicities(d(mom), d(gs))
    me, sh, sc, num, den = m.compute_multichannel(d(mom), d(gs), d(chan), d(rh), d(rc))
    torch.cuda.synchronize()
    ref_mask = O.good_helicities(process, mom, gs)
    assert np.array_equal(mask, ref_mask)
    allnum = O.multichannel(process, mom, gs, mask=ref_mask)
    ref_num, ref_den = allnum[np.arange(n), chan], allnum.sum(axis=1)
    assert np.abs(num.cpu().numpy() / ref_num - 1).max() <= 1e-10
    assert np.abs(den.cpu().numpy() / ref_den - 1).max() <= 1e-10
    sel = O.select(process, mom, gs, rh, rc, mask=ref_mask, channel=chan)
    assert np.abs(me.cpu().numpy() / sel["me"] - 1).max() <= TOL[precision]
    # colour selection: always an allowed flow; equal to the oracle's except within tolerance of a boundary
    allowed = O.channel_flows(process)
    got = sc.cpu().numpy()
    assert np.all(allowed[chan, got])
    bad = np.nonzero(got != sel["selcol"])[0]
    for e in bad:
        cum, tot = sel["cumcol"][e], sel["cumcol"][e, -1]
        lo, hi = sorted((int(got[e]), int(sel["selcol"][e])))
        assert np.min(np.abs(rc[e] * tot - cum[lo:hi])) <= TOL[precision] * tot
    assert len(bad) <= max(2, 4 * TOL[precision] * allowed.shape[1] * n)
    assert np.mean(sh.cpu().numpy() == sel["selhel"]) > 0.99
    m.close()


@pytest.mark.parametrize("process,n", [("gg_ttgg", 2 * 4736 + 1234), ("gg_ttggg", 900)])
def test_multichannel_colour_selection_over_several_chunks(torch_cuda, process, n):
    """The lane-group pipeline cuts a batch into chunks; every chunk must read ITS events' channels.  One call over several
    chunks against two calls of unequal size (bit-identical), and every selected flow allowed for the event's own channel."""
    from oracle import oracle as O
    from paper_2503_21935_b200.me import MatrixElement
    torch = torch_cuda
    dev = torch.device("cuda:0")
    d = lambda x: torch.from_numpy(x).to(dev)
    mom, gs = d(I.make_momenta(process, n, seed=9)), d(I.make_gs(n, seed=9, alphas=ALPHAS[process]))
    rh, rc = (d(x) for x in I.make_rnd(n, seed=9))
    ndiag = O.info(process)["ndiag"]
    chan_np = (I.uniforms(9, 7, 0, n) * ndiag).astype(np.int32)
    chan = d(chan_np)
    m = MatrixElement(process, "fp64")
    m.filter_helicities(mom, gs)
    one = m.compute_multichannel(mom, gs, chan, rh, rc)
    torch.cuda.synchronize()
    assert m.launch_info()["chunk_events"] < n, "the case must span several chunks"
    k = n // 3 + 1
    a = m.compute_multichannel(mom[:k].contiguous(), gs[:k].contiguous(), chan[:k].contiguous(), rh[:k].contiguous(), rc[:k].contiguous())
    b = m.compute_multichannel(mom[k:].contiguous(), gs[k:].contiguous(), chan[k:].contiguous(), rh[k:].contiguous(), rc[k:].contiguous())
    torch.cuda.synchronize()
    for i in range(5):
        assert torch.equal(torch.cat([a[i], b[i]]), one[i]), f"output {i} depends on the split"
    allowed = O.channel_flows(process)
    assert np.all(allowed[chan_np, one[2].cpu().numpy()])
    m.close()


def test_multichannel_errors(torch_cuda):
    from paper_2503_21935_b200.me import MatrixElement, MEError
    torch = torch_cuda
    m = MatrixElement("ee_mumu", "fp64")
    mom = torch.from_numpy(I.make_momenta("ee_mumu", 8, seed=1)).cuda()
    m.filter_helicities(mom, None)
    with pytest.raises(MEError):
        m.compute_multichannel(mom, None, torch.zeros(8, dtype=torch.int32, device="cuda"))
    assert m.channel_table() == []
    m.close()
    # the mixed EW+QCD process has no channel kernel either
    m = MatrixElement("gux_taptamggux", "fp64")
    mom = torch.from_numpy(I.make_momenta("gux_taptamggux", 8, seed=1)).cuda()
    gs = torch.from_numpy(I.make_gs(8, seed=1)).cuda()
    m.filter_helicities(mom, gs)
    with pytest.raises(MEError):
        m.compute_multichannel(mom, gs, torch.zeros(8, dtype=torch.int32, device="cuda"))
    assert m.channel_table() == [] and m.ndiag == 100 and m.ncol == 6 and m.denom == 192
    assert np.array_equal(m.color_table()[0], [0, 4, 5])
    m.close()
