"""GPU parity: the CUDA path (through the C ABI) against the scalar CPU oracle, element by element, on
the same seeded RAMBO inputs.  Tolerances are BASELINE.json north_star's: max relative difference
1e-10 (fp64), 1e-5 (mixed), 1e-3 with median 1e-5 (fp32); helicity / colour choices bit-exact except
where the oracle's cumulative weight lies within tolerance of the random number.
"""
import numpy as np
import pytest

from oracle import rambo as I

pytestmark = pytest.mark.gpu

TOL = {"fp64": 1e-10, "mixed": 1e-5, "fp32": 1e-3}
# events per parity case: several 128-thread tiles plus a ragged tail; the oracle finishes in seconds
NEVT = {"ee_mumu": 16384, "gg_tt": 8192 + 77, "gg_ttg": 4096 + 77, "gg_ttgg": 1024 + 77, "gg_ttggg": 128 + 13,
        "gux_taptamggux": 2048 + 77, "gux_taptamux": 8192 + 77, "gux_taptamgux": 4096 + 77}
ALPHAS = {"ee_mumu": 0.118, "gg_tt": 0.118, "gg_ttg": 0.118, "gg_ttgg": None, "gg_ttggg": 0.118, "gux_taptamggux": None, "gux_taptamux": None, "gux_taptamgux": None}
BUILDS = [("ee_mumu", "fp64"), ("gg_tt", "fp64"), ("gg_tt", "fp32"), ("gg_ttg", "fp64"), ("gg_ttg", "fp32"),
          ("gg_ttg", "mixed"), ("gg_ttgg", "fp64"), ("gg_ttgg", "fp32"), ("gg_ttgg", "mixed"),
          ("gg_ttggg", "fp64"), ("gg_ttggg", "fp32"), ("gg_ttggg", "mixed"),
          # mixed EW+QCD class (Table 4)
          ("gux_taptamggux", "fp64"), ("gux_taptamggux", "fp32"), ("gux_taptamggux", "mixed"),
          ("gux_taptamux", "fp64"), ("gux_taptamux", "fp32"), ("gux_taptamgux", "fp64"), ("gux_taptamgux", "fp32")]


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


_cache = {}


def oracle_case(process):
    """Seeded inputs and the oracle's answers (ME, good mask, selections), computed once per process."""
    if process not in _cache:
        from oracle import oracle as O
        n = NEVT[process]
        mom = I.make_momenta(process, n, seed=1)
        gs = I.make_gs(n, seed=1, alphas=ALPHAS[process])
        rh, rc = I.make_rnd(n, seed=1)
        mask = O.good_helicities(process, mom, gs)
        sel = O.select(process, mom, gs, rh, rc, mask=mask)
        _cache[process] = dict(mom=mom, gs=gs, rh=rh, rc=rc, mask=mask, sel=sel)
    return _cache[process]


def run_gpu(torch, process, precision, case, select=True):
    from paper_2503_21935_b200.me import MatrixElement
    dev = torch.device("cuda:0")
    m = MatrixElement(process, precision)
    mom = torch.from_numpy(case["mom"]).to(dev)
    gs = torch.from_numpy(case["gs"]).to(dev)
    rh = torch.from_numpy(case["rh"]).to(dev) if select else None
    rc = torch.from_numpy(case["rc"]).to(dev) if select else None
    mask = m.filter_helicities(mom, gs)
    me, sh, sc = m.compute(mom, gs, rh, rc)
    torch.cuda.synchronize()
    res = dict(me=me.cpu().numpy(), mask=mask, info=m.launch_info())
    if select:
        res["selhel"], res["selcol"] = sh.cpu().numpy(), sc.cpu().numpy()
    m.close()
    return res


@pytest.mark.parametrize("process,precision", BUILDS)
def test_me_matches_oracle(torch_cuda, process, precision):
    case = oracle_case(process)
    got = run_gpu(torch_cuda, process, precision, case)
    ref = case["sel"]["me"]
    assert np.all(np.isfinite(got["me"]))
    rel = np.abs(got["me"] - ref) / ref
    assert rel.max() <= TOL[precision], f"max rel diff {rel.max():.3e} at event {rel.argmax()}"
    if precision == "fp32":
        assert np.median(rel) <= 1e-5
    # the good-helicity mask comes from the fp64 filter in every build: it must equal the oracle's
    assert np.array_equal(got["mask"], case["mask"])


def _check_selection(sel_gpu, sel_ref, cum, rnd, tol):
    """Exact match, except where r*S is within tol*S of the cumulative boundary separating the two answers."""
    bad = np.nonzero(sel_gpu != sel_ref)[0]
    for e in bad:
        tot = cum[e, -1]
        lo, hi = sorted((int(sel_gpu[e]), int(sel_ref[e])))
        # boundaries crossed between the two answers: cum[lo] .. cum[hi-1]
        d = np.min(np.abs(rnd[e] * tot - cum[e, lo:hi]))
        assert d <= tol * tot, f"event {e}: gpu {sel_gpu[e]} oracle {sel_ref[e]}, distance {d / tot:.3e} of total"
    return len(bad)


@pytest.mark.parametrize("process,precision", BUILDS)
def test_selection_matches_oracle(torch_cuda, process, precision):
    case = oracle_case(process)
    got = run_gpu(torch_cuda, process, precision, case)
    tol = TOL[precision]        # north_star: mismatches only where the cumulative weight is within tolerance of r
    sel = case["sel"]
    nbad_h = _check_selection(got["selhel"], sel["selhel"], sel["cumhel"], case["rh"], tol)
    nbad_c = _check_selection(got["selcol"], sel["selcol"], sel["cumcol"], case["rc"], tol)
    n = len(case["rh"])
    # boundary cases must be rare: r falls within tol of one of the ngood (ncol) boundaries with probability
    # ~2 tol ngood; twice that is allowed.  A wrong rule would disagree on a finite fraction of events.
    ngood, ncol = int(case["mask"].sum()), sel["cumcol"].shape[1]
    assert nbad_h <= max(2, 4 * tol * ngood * n) and nbad_c <= max(2, 4 * tol * ncol * n)
    # selected helicities are good ones, colours are in range
    assert np.all(case["mask"][got["selhel"]] == 1)
    assert got["selcol"].min() >= 0 and got["selcol"].max() < sel["cumcol"].shape[1]


def test_selection_off_gives_same_me(torch_cuda):
    case = oracle_case("gg_ttg")
    a = run_gpu(torch_cuda, "gg_ttg", "fp64", case, select=True)
    b = run_gpu(torch_cuda, "gg_ttg", "fp64", case, select=False)
    assert np.array_equal(a["me"], b["me"])


def test_tables_match_oracle(torch_cuda):
    from oracle import oracle as O
    from paper_2503_21935_b200.me import MatrixElement, PROCESSES
    for p in PROCESSES:
        m = MatrixElement(p, "fp64")
        i = O.info(p)
        assert (m.npar, m.ncomb, m.ncol, m.ndiag, m.denom) == (i["npar"], i["ncomb"], i["ncol"], i["ndiag"], i["denom"])
        assert np.array_equal(m.helicity_table(), O.helicity_table(p))
        assert np.array_equal(m.color_table(), O.color_table(p))
        assert np.allclose(m.color_matrix(), O.color_matrix(p), rtol=0, atol=1e-12)
        m.close()


def test_host_path_and_edge_cases(torch_cuda):
    torch = torch_cuda
    from paper_2503_21935_b200.me import MatrixElement, MEError
    case = oracle_case("gg_tt")
    m = MatrixElement("gg_tt", "fp64")
    mom = torch.from_numpy(case["mom"]).cuda()
    gs = torch.from_numpy(case["gs"]).cuda()
    with pytest.raises(MEError):  # compute before a helicity mask exists
        m.compute(mom, gs)
    m.filter_helicities(mom, gs)
    # empty batch
    me, _, _ = m.compute(mom[:0], gs[:0])
    assert me.shape == (0,)
    # single event and a ragged count
    for n in (1, 129):
        me, _, _ = m.compute(mom[:n].contiguous(), gs[:n].contiguous())
        torch.cuda.synchronize()
        assert np.allclose(me.cpu().numpy(), case["sel"]["me"][:n], rtol=1e-10, atol=0)
    # host buffers (the e2e path of bench.py)
    me_h, sh, sc = m.compute_host(case["mom"], case["gs"], case["rh"], case["rc"])
    assert np.allclose(me_h, case["sel"]["me"], rtol=1e-10, atol=0)
    assert np.mean(sh == case["sel"]["selhel"]) > 0.999 and np.mean(sc == case["sel"]["selcol"]) > 0.999
    # exported / imported mask round trip
    mask = m.get_good_helicities()
    m2 = MatrixElement("gg_tt", "fp64")
    m2.set_good_helicities(mask)
    me2, _, _ = m2.compute(mom, gs)
    torch.cuda.synchronize()
    assert np.allclose(me2.cpu().numpy(), case["sel"]["me"], rtol=1e-10, atol=0)
    with pytest.raises(MEError):
        MatrixElement("gg_nothing", "fp64")
    m.close(); m2.close()


def test_physics_invariants_on_gpu(torch_cuda):
    """Properties that hold at any size (used again at full size in test_gpu_fullsize.py)."""
    torch = torch_cuda
    from paper_2503_21935_b200.me import MatrixElement
    for p, ngl in (("gg_ttg", 3), ("gg_ttgg", 4)):
        n = 2048
        mom = I.make_momenta(p, n, seed=3)
        m = MatrixElement(p, "fp64")
        d = torch.from_numpy(mom).cuda()
        g1 = torch.full((n,), 1.2, dtype=torch.float64, device="cuda")
        g2 = torch.full((n,), 1.1, dtype=torch.float64, device="cuda")
        m.filter_helicities(d, g1)
        a = m.compute(d, g1)[0].cpu().numpy()
        b = m.compute(d, g2)[0].cpu().numpy()
        assert np.allclose(a / b, (1.2 / 1.1) ** (2 * ngl), rtol=1e-12)  # ME ~ alpha_s^n
        # Lorentz invariance (all helicities kept: a boost mixes them).  Holds at Gamma_t = 0 only: the fixed
        # width breaks gauge invariance, hence frame independence, at O(1e-7) (reading R4)
        m.close()
        m = MatrixElement(p, "fp64", params=dict(wt=0.0))
        m.set_good_helicities(np.ones(m.ncomb, dtype=np.uint8))
        a = m.compute(d, g1)[0].cpu().numpy()
        lt = torch.from_numpy(I.lorentz_transform(mom, seed=5)).cuda()
        c = m.compute(lt, g1)[0].cpu().numpy()
        assert np.max(np.abs(c - a) / a) < 1e-8
        # Bose symmetry: exchanging the two last final-state gluons' momenta
        if ngl == 4:
            sw = mom.copy(); sw[:, [4, 5]] = sw[:, [5, 4]]
            c = m.compute(torch.from_numpy(sw).cuda(), g1)[0].cpu().numpy()
            assert np.max(np.abs(c - a) / a) < 1e-10
        m.close()


@pytest.mark.parametrize("process", ["gg_ttg", "gg_ttgg", "gg_ttggg"])
def test_partial_helicity_mask_matches_oracle(torch_cuda, process):
    """An imported good-helicity mask that drops helicities (me_set_good_helicities): ME, helicity and colour
    selections are those of the oracle with the same mask (both kernel layouts)."""
    torch = torch_cuda
    from oracle import oracle as O
    from paper_2503_21935_b200.me import MatrixElement
    case = oracle_case(process)
    n = {"gg_ttg": 1000, "gg_ttgg": 333, "gg_ttggg": 45}[process]
    mom, gs, rh, rc = case["mom"][:n], case["gs"][:n], case["rh"][:n], case["rc"][:n]
    ncomb = len(case["mask"])
    mask = (np.arange(ncomb) % 3 != 1).astype(np.uint8)  # drops a third of the rows, keeps the last one or not
    mask[-1] = 0
    ref = O.select(process, mom, gs, rh, rc, mask=mask)
    m = MatrixElement(process, "fp64")
    m.set_good_helicities(mask)
    me, sh, sc = m.compute(torch.from_numpy(mom).cuda(), torch.from_numpy(gs).cuda(), torch.from_numpy(rh).cuda(),
                           torch.from_numpy(rc).cuda())
    torch.cuda.synchronize()
    me, sh, sc = me.cpu().numpy(), sh.cpu().numpy(), sc.cpu().numpy()
    assert np.max(np.abs(me - ref["me"]) / ref["me"]) <= 1e-10
    assert np.all(mask[sh] == 1)
    _check_selection(sh, ref["selhel"], ref["cumhel"], rh, 1e-9)
    _check_selection(sc, ref["selcol"], ref["cumcol"], rc, 1e-9)
    m.close()


def test_group_kernel_edge_batches(torch_cuda):
    """gg_ttgg (lane-group kernel): empty, single-event and ragged batches, host-buffer path."""
    torch = torch_cuda
    from paper_2503_21935_b200.me import MatrixElement
    case = oracle_case("gg_ttgg")
    m = MatrixElement("gg_ttgg", "fp64")
    mom = torch.from_numpy(case["mom"]).cuda()
    gs = torch.from_numpy(case["gs"]).cuda()
    m.filter_helicities(mom, gs)
    me, _, _ = m.compute(mom[:0], gs[:0])
    assert me.shape == (0,)
    for n in (1, 2, 65):
        me, _, _ = m.compute(mom[:n].contiguous(), gs[:n].contiguous())
        torch.cuda.synchronize()
        assert np.allclose(me.cpu().numpy(), case["sel"]["me"][:n], rtol=1e-10, atol=0)
    me_h, sh, sc = m.compute_host(case["mom"], case["gs"], case["rh"], case["rc"])
    assert np.allclose(me_h, case["sel"]["me"], rtol=1e-10, atol=0)
    assert np.mean(sh == case["sel"]["selhel"]) > 0.999 and np.mean(sc == case["sel"]["selcol"]) > 0.999
    m.close()


@pytest.mark.parametrize("process,precision,n", [("gg_ttgg", "fp64", 2 * 4736 + 1234), ("gg_ttgg", "fp32", 2 * 4736 + 1234),
                                                 ("gg_ttggg", "fp64", 900), ("gg_ttggg", "mixed", 900)])
def test_lane_group_pipeline_is_deterministic_and_chunk_independent(torch_cuda, process, precision, n):
    """The lane-group pipeline is warp-synchronous shared-memory code whose scratch is reused from chunk to chunk
    (compute-sanitizer is closed on this pool): a race or a wrong chunk offset would show as
    run-to-run or split-dependent differences.  Two runs of the same batch are bit-identical, and so are the results
    of the batch done in one call (several internal chunks on two streams) and in two calls of unequal size."""
    from paper_2503_21935_b200.me import MatrixElement
    dev = torch_cuda.device("cuda:0")
    mom = torch_cuda.from_numpy(I.make_momenta(process, n, seed=5)).to(dev)
    gs = torch_cuda.from_numpy(I.make_gs(n, seed=5, alphas=ALPHAS[process])).to(dev)
    rh, rc = (torch_cuda.from_numpy(x).to(dev) for x in I.make_rnd(n, seed=5))
    m = MatrixElement(process, precision)
    m.filter_helicities(mom, gs)
    runs = []
    for _ in range(3):
        me, sh, sc = m.compute(mom, gs, rh, rc)
        torch_cuda.cuda.synchronize()
        runs.append((me.clone(), sh.clone(), sc.clone()))
    for r in runs[1:]:
        assert all(torch_cuda.equal(x, y) for x, y in zip(r, runs[0]))
    k = n // 3 + 1
    a = m.compute(mom[:k].contiguous(), gs[:k].contiguous(), rh[:k].contiguous(), rc[:k].contiguous())
    b = m.compute(mom[k:].contiguous(), gs[k:].contiguous(), rh[k:].contiguous(), rc[k:].contiguous())
    torch_cuda.cuda.synchronize()
    for i in range(3):
        assert torch_cuda.equal(torch_cuda.cat([a[i], b[i]]), runs[0][i])
    m.close()


def test_pipeline_scratch_follows_the_batch_size(torch_cuda):
    """gg_ttgg: a fresh handle owns no pipeline scratch; small batches take little; me_reserve sizes it up front; a call no
    larger than an earlier one does not change it; results do not depend on the scratch size."""
    from paper_2503_21935_b200.me import MatrixElement
    torch = torch_cuda
    case = oracle_case("gg_ttgg")
    mom, gs = torch.from_numpy(case["mom"]).cuda(), torch.from_numpy(case["gs"]).cuda()
    m = MatrixElement("gg_ttgg", "fp64")
    assert m.launch_info()["scratch_bytes"] == 0
    m.filter_helicities(mom[:64].contiguous(), gs[:64].contiguous())
    small, _, _ = m.compute(mom[:300].contiguous(), gs[:300].contiguous())
    torch.cuda.synchronize()
    s0 = m.launch_info()["scratch_bytes"]
    assert 0 < s0 < (64 << 20)
    m.compute(mom[:200].contiguous(), gs[:200].contiguous())
    assert m.launch_info()["scratch_bytes"] == s0
    m.reserve(1 << 20)
    s1 = m.launch_info()["scratch_bytes"]
    assert s1 == (2 << 30)   # the cap of a gg_ttgg handle
    big, _, _ = m.compute(mom, gs)
    torch.cuda.synchronize()
    assert m.launch_info()["scratch_bytes"] == s1
    assert torch.equal(big[:300], small)
    assert np.abs(big.cpu().numpy() / case["sel"]["me"] - 1).max() <= 1e-10
    m.close()
