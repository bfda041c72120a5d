"""me_compute_noalloc (include/me_b200.h) against the existing me_compute path.

me_compute_noalloc serves callers that cannot let this library call cudaMalloc: applications that have handed the
whole GPU to their own memory pool or run under a fixed device-memory budget, and loops that cannot afford the
device-wide stall an allocation may cause.  It therefore keeps its kernel's scratch (the running helicity sums used
to draw the helicity) in a fixed 4 MiB array inside the library, shared by every call on the GPU and never cleared.
What is checked here:

  * two calls in a row, the first filling the array to its limit (16384 events), the second smaller and on other
    events, so that it runs over the first call's leftovers: each must reproduce me_compute (handle path, gg_ttg,
    fp64) within the fp64 tolerance of the parity tests (1e-10 relative on ME), with the same helicity and colour choices;
  * a batch beyond the limit is refused with a message that says why, and nothing is written.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the
parity tests.  The test does not depend on what ran before it (fresh process or after the whole suite).
"""
import numpy as np
import pytest

from oracle import rambo as I

pytestmark = pytest.mark.gpu

TOL = 1e-10   # fp64 tolerance of tests/test_gpu_parity.py


def _inputs(torch, n, seed):
    dev = torch.device("cuda:0")
    mom = torch.from_numpy(I.make_momenta("gg_ttg", n, seed=seed)).to(dev)
    gs = torch.from_numpy(I.make_gs(n, seed=seed, alphas=None)).to(dev)
    rh, rc = (torch.from_numpy(x).to(dev) for x in I.make_rnd(n, seed=seed))
    return mom, gs, rh, rc


def test_noalloc_matches_handle_path_on_two_calls_in_a_row():
    import torch
    from paper_2503_21935_b200 import me as M

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    handle = M.MatrixElement("gg_ttg", "fp64")
    first = True
    for n, seed in ((M.NOALLOC_MAX_EVENTS, 5), (4096 + 77, 6)):
        mom, gs, rh, rc = _inputs(torch, n, seed)
        if first:
            mask = handle.filter_helicities(mom, gs)
            first = False
        ref_me, ref_sh, ref_sc = handle.compute(mom, gs, rh, rc)
        # outputs preset to a sentinel: every entry must be overwritten
        out = torch.full((n,), -1.0, dtype=torch.float64, device=mom.device)
        sh = torch.full((n,), -7, dtype=torch.int32, device=mom.device)
        sc = torch.full((n,), -7, dtype=torch.int32, device=mom.device)
        M.compute_noalloc(mom, gs, rh, rc, good_mask=mask, out=out, selhel=sh, selcol=sc)
        torch.cuda.synchronize()
        a, b = out.cpu().numpy(), ref_me.cpu().numpy()
        assert np.all(np.isfinite(a)) and np.all(a > 0)
        rel = np.abs(a - b) / b
        assert rel.max() <= TOL, f"{n} events: max rel diff {rel.max():.3e} at event {rel.argmax()}"
        # same code, same inputs: the choices are the same wherever the MEs are bit-identical (everywhere, in practice)
        same = a == b
        assert np.array_equal(sh.cpu().numpy()[same], ref_sh.cpu().numpy()[same])
        assert np.array_equal(sc.cpu().numpy()[same], ref_sc.cpu().numpy()[same])
        assert same.mean() > 0.99
        assert np.all(mask[sh.cpu().numpy()] == 1)
    # no mask = all 32 helicity combinations; for a massive top the filter keeps them all, so the result is the same
    if mask.all():
        out2, _, _ = M.compute_noalloc(mom, gs)
        torch.cuda.synchronize()
        assert np.array_equal(out2.cpu().numpy(), a)
    handle.close()


def test_noalloc_refuses_a_batch_beyond_its_scratch():
    import torch
    from paper_2503_21935_b200 import me as M

    n = M.NOALLOC_MAX_EVENTS + 1
    dev = torch.device("cuda:0")
    mom = torch.zeros((n, 5, 4), dtype=torch.float64, device=dev)
    gs = torch.ones(n, dtype=torch.float64, device=dev)
    out = torch.full((n,), -1.0, dtype=torch.float64, device=dev)
    with pytest.raises(M.MEError, match="batch too large.*16385.*16384"):
        M.compute_noalloc(mom, gs, out=out)
    torch.cuda.synchronize()
    assert bool((out == -1.0).all())
