"""Small invocations of every kernel of the library, written to run under compute-sanitizer
(SURVEY.md section 4 T-d, section 5 "Race detection"):

    compute-sanitizer --tool racecheck|memcheck|initcheck python tests/sanitizer_cases.py [case ...]

(compute-sanitizer is closed on the GPU pool of this build -- profiles/r02_sanitizer.md records the refusal; the
script also runs on its own, and tests/test_gpu_parity.py::test_repeatability_stress is the race evidence that
can be produced without the tool.)

Cases are tiny (the tools slow kernels down 10-1000x) but span several tiles, a ragged tail, grouped and
ungrouped batches, empty segments, the generator's warp-shared lists and the ticketed reductions.  The
script only checks that the calls complete and the results are finite; parity is tests/test_gpu_parity.py.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import ipa_inputs as inp  # noqa: E402

LO, HI = inp.LO, inp.HI


def main(argv):
    import torch
    import paper_1706_01420_b200 as ipa
    want = set(argv) or {"nll", "grad", "seg", "gen", "binned", "prep"}
    x = torch.from_numpy(inp.standin_masses(1, 9000)).cuda()
    batch, _ = inp.fd_batch(inp.GEN)
    done = []
    if "nll" in want:
        # K = 9 grouped batch with per-event output, ragged size; K = 2 ungrouped; misaligned start
        for xs in (x[:4099], x[1:8200]):
            nll, lp, st = ipa.ipa_nll_eval(xs, batch, LO, HI, want_logpdf=True)
            nll2, _, _ = ipa.ipa_nll_eval(xs, [inp.GEN, inp.P2], LO, HI)
            torch.cuda.synchronize()
            assert torch.isfinite(nll).all() and torch.isfinite(nll2).all() and torch.isfinite(lp).all()
        ns, nb, _ = ipa.ipa_norm([inp.GEN, inp.P2], LO, HI)
        torch.cuda.synchronize()
        assert torch.isfinite(ns).all() and torch.isfinite(nb).all()
        done.append("nll")
    if "grad" in want:
        nll, g, st = ipa.ipa_nll_grad_eval(x[:4099], [inp.GEN, inp.P2], LO, HI)
        torch.cuda.synchronize()
        assert torch.isfinite(nll).all() and torch.isfinite(g).all()
        done.append("grad")
    if "seg" in want:
        T = 70
        rng = np.random.Generator(np.random.Philox(5))
        off = np.concatenate([[0], np.sort(rng.integers(0, x.numel(), size=T - 1)), [x.numel()]]).astype(np.int64)
        off[10] = off[9]
        off = np.maximum.accumulate(off)
        nll, st = ipa.ipa_nll_eval_segmented(x, torch.from_numpy(off).cuda(), inp.toy_param_sets(T, seed=11), LO, HI)
        torch.cuda.synchronize()
        assert torch.isfinite(nll).all()
        done.append("seg")
    if "gen" in want:
        xm, off, ovf = ipa.ipa_toy_generate([1], inp.GEN, -1.0, -1.0, LO, HI, 5000)
        xt, offt, ovft = ipa.ipa_toy_generate(inp.toy_seeds(6), inp.P2, 300.0, 700.0, LO, HI, 8000)
        torch.cuda.synchronize()
        assert torch.isfinite(xm).all() and ovf.item() == 0 and ovft.item() == 0
        assert torch.isfinite(xt[: int(offt[-1].item())]).all()
        done.append("gen")
    if "binned" in want:
        nbins = 1000
        counts = ipa.ipa_hist_fill(x, LO, HI, nbins)
        ns, nb, kk = inp.scan_grid(5, 4, n_obs=float(x.numel()))
        scan = ipa.ipa_binned_nll_scan(counts, LO, HI, inp.GEN, ns, nb, kk)
        nu = ipa.ipa_expected_hist(nbins, LO, HI, inp.GEN, 250.0, 8750.0, -0.002)
        nu0 = ipa.ipa_expected_hist(nbins, LO, HI, inp.GEN, 0.0, 9000.0, -0.002)
        toys = ipa.ipa_poisson_hist_toys(nu, np.arange(1, 13, dtype=np.uint64))
        q = ipa.ipa_cls_teststat(toys, nu, nu0)
        qo = ipa.ipa_cls_teststat(counts, nu, nu0)
        c = ipa.ipa_cls_count_ge(q, qo)
        cl = ipa.ipa_cls_from_counts(c, 12, c, 12)
        sm = ipa.ipa_gauss_smear(ipa.ipa_signal_shape(nbins, LO, HI, inp.GEN), LO, HI, 10.0)
        scan2 = ipa.ipa_binned_nll_scan_shape(counts, LO, HI, sm, ns, nb, kk)
        torch.cuda.synchronize()
        assert torch.isfinite(scan).all() and torch.isfinite(scan2).all() and torch.isfinite(q).all()
        done.append("binned")
    if "prep" in want:
        xs = ipa.ipa_events_prepare(x, LO, HI)
        off = torch.tensor([0, 0, 17, 4000, 4000, 9000], dtype=torch.int64, device="cuda")
        xs2 = ipa.ipa_events_prepare(x, LO, HI, off)
        torch.cuda.synchronize()
        assert abs(xs.sum().item() - x.sum().item()) < 1e-6 * abs(x.sum().item()) and xs2.numel() == x.numel()
        done.append("prep")
    print("sanitizer cases completed:", " ".join(done))


if __name__ == "__main__":
    main(sys.argv[1:])
