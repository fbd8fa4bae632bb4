"""ipa_nll_eval_static: the one entry point that needs no caller workspace (scratch in a static __device__ array of the
library).  Its output against the existing path (ipa_nll_eval with an own workspace) on the same inputs, two calls in a
row, so that the second call runs on the scratch the first one left behind.  In a file of its own that pytest collects
last: the suite runs with pytest -x."""
import ctypes as C
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import ipa_inputs as inp  # noqa: E402

LO, HI = inp.LO, inp.HI


def test_static_scratch_holds_the_stated_maximum():
    """host logic: the workspace of IPA_STATIC_MAX_K sets fits the array the header states; the symbol is exported"""
    import paper_1706_01420_b200 as ipa
    hdr = open(os.path.join(ROOT, "include", "ipanll.h")).read()
    assert "#define IPA_STATIC_MAX_K 16" in hdr and "#define IPA_STATIC_SCRATCH_BYTES (288 * 1024)" in hdr
    assert ipa.IPA_STATIC_MAX_K == 16
    assert ipa.ipa_workspace_bytes(10 ** 8, ipa.IPA_STATIC_MAX_K) <= 288 * 1024
    assert hasattr(ipa.lib(), "ipa_nll_eval_static")
    assert "IPA_STATIC_MAX_K" in ipa.lib().ipa_strerror(-5).decode()


@pytest.mark.gpu
def test_static_entry_point_matches_the_workspace_path_twice():
    import torch
    import paper_1706_01420_b200 as ipa
    assert torch.cuda.is_available()
    n = 300_001                                           # 73 full tiles and a ragged tail
    x, _, _ = ipa.ipa_toy_generate([21], inp.GEN, -1.0, -1.0, LO, HI, n)
    batch9, _ = inp.fd_batch(inp.GEN)                     # central-difference batch: 9 sets, 5 shapes (grouped kernel)
    rng = np.random.Generator(np.random.Philox(16))
    sets16 = [dict(inp.P2, mu=5280 + rng.uniform(-5, 5), sigma=rng.uniform(12, 18), f=rng.uniform(0.1, 0.6),
                   k=rng.uniform(-0.003, -0.001)) for _ in range(16)]
    sets16[3] = dict(sets16[3], sigma=-1.0)               # a domain error inside the batch: status 1, NLL +inf
    calls = [(batch9, 1, False), (sets16, 0, False), (inp.GEN, 1, True), (batch9, 1, False)]
    out = torch.empty(16, dtype=torch.float64, device="cuda")
    st = torch.empty(16, dtype=torch.int32, device="cuda")
    first = None
    for params, pol, want_lp in calls:                    # calls in a row on one stream: each runs on the scratch of the last
        K = ipa.pack_params(params).shape[0]
        ref, ref_lp, ref_st = ipa.ipa_nll_eval(x, params, LO, HI, want_logpdf=want_lp, policy=pol)
        got, got_lp, got_st = ipa.ipa_nll_eval_static(x, params, LO, HI, want_logpdf=want_lp, out=out[:K], status=st[:K],
                                                      policy=pol)
        torch.cuda.synchronize()
        a, b = got.cpu().numpy(), ref.cpu().numpy()
        assert (got_st.cpu().numpy() == ref_st.cpu().numpy()).all()
        fin = np.isfinite(b)
        assert (np.isfinite(a) == fin).all() and np.all(a[~fin] == b[~fin])
        assert np.all(np.abs(a[fin] - b[fin]) <= 1e-10 * np.abs(b[fin]))      # the tolerance of the parity tests
        assert np.array_equal(a[fin], b[fin])                                   # same kernels, same geometry: same bits
        if want_lp:
            assert torch.equal(got_lp, ref_lp)
        if first is None:
            first = a.copy()
    assert np.array_equal(first, a)                       # the same batch again, after other calls used the scratch

    # beyond the maximum: a clear error, nothing enqueued, the outputs untouched
    out.fill_(-7.0)
    with pytest.raises(ipa.IpaError, match="IPA_STATIC_MAX_K"):
        ipa.ipa_nll_eval_static(x, sets16 + [inp.GEN], LO, HI, out=torch.empty(17, dtype=torch.float64, device="cuda"))
    one = C.c_void_p(out.data_ptr())
    p17 = ipa.pack_params(sets16 + [inp.GEN])
    rc = ipa.lib().ipa_nll_eval_static(C.c_void_p(x.data_ptr()), n, p17.ctypes.data_as(C.c_void_p), 17,
                                       ipa.binding._Range(LO, HI), one, None, None, None, None)
    assert rc == -5
    rc = ipa.lib().ipa_nll_eval_static(C.c_void_p(x.data_ptr()), n, p17.ctypes.data_as(C.c_void_p), 0,
                                       ipa.binding._Range(LO, HI), one, None, None, None, None)
    assert rc == -1
    torch.cuda.synchronize()
    assert bool((out == -7.0).all())
    # and the entry point still works after the rejected calls
    got = ipa.ipa_nll_eval_static(x, inp.GEN, LO, HI, out=out[:1], status=st[:1], policy=1)[0]
    ref = ipa.ipa_nll_eval(x, inp.GEN, LO, HI, policy=1)[0]
    torch.cuda.synchronize()
    assert got.item() == ref.item()
