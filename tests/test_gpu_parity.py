"""GPU parity: the CUDA path (through the C ABI of include/ipanll.h) against the CPU oracle on the
same seeded inputs.  Tolerances are BASELINE.json's: per-event log-pdf 1e-10 absolute, total NLL
1e-10 relative, finite-difference gradient 1e-7 relative (reading D18), integer work bit-exact.
"""
import numpy as np
import pytest

import ipa_inputs as inp

pytestmark = pytest.mark.gpu

LO, HI = inp.LO, inp.HI


@pytest.fixture(scope="module")
def ipa():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1706_01420_b200 as m
    m.lib()
    return m


@pytest.fixture(scope="module")
def torch_():
    import torch
    return torch


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def grad_ok(g_gpu, g_orc):
    """reading D18; 4 components (finite differences over (mu, sigma, f, k)) or 5 (analytic: + beta)"""
    s = np.array([inp.GRAD_SCALE[name] for name in inp.GRAD_NAMES])[:len(g_orc)]
    return np.all(np.abs(g_gpu - g_orc) <= 1e-7 * np.maximum(np.abs(g_orc), 1.0 / s))


def mismatches(got, ref, what, tol=1e-9):
    """Generator parity: number of events further than `tol` from the oracle generator's;
    at most floor(1e-6 n) accept-reject flips are allowed, i.e. NONE for n <= 1e6 (a flip needs a uniform within
    ~1e-15 of the acceptance ratio).  The count is printed."""
    assert got.shape == ref.shape
    bad = int((~(np.abs(got - ref) <= tol)).sum())
    print(f"[generator parity] {what}: {bad} of {got.size} events differ from the oracle's by more than {tol:g}")
    assert bad <= got.size // 1_000_000, (what, bad, got.size)
    return bad


@pytest.fixture(scope="module")
def x1(orc):
    """config 1: 10,000 events, seed 1, from the oracle's generator"""
    return orc.generate_mixture(1, 10000, inp.GEN, LO, HI)


@pytest.mark.parametrize("shape", ["P1", "P2", "T1", "T2"])     # T1, T2: zeta = 0 Student-t core (row f4, reading D3)
@pytest.mark.parametrize("policy", [0, 1])
def test_config1_logpdf_nll_gradient(ipa, torch_, orc, x1, shape, policy):
    theta = {"P1": inp.GEN, "P2": inp.P2, "T1": inp.T1, "T2": inp.T2}[shape]
    batch, _ = inp.fd_batch(theta)
    idx, h = inp.fd_spec()
    xd = dev(torch_, x1)
    nll, lp, st = ipa.ipa_nll_eval(xd, batch, LO, HI, want_logpdf=True, policy=policy)
    nll_g, grad, st_g = ipa.ipa_nll_fd_gradient(xd, theta, idx, h, LO, HI, policy=policy)   # row G: its own 2P+1 batch
    torch_.cuda.synchronize()
    nll, lp, st = nll.cpu().numpy(), lp.cpu().numpy(), st.cpu().numpy()
    assert (st == 0).all() and (st_g.cpu().numpy() == 0).all()
    assert np.array_equal(nll_g.cpu().numpy(), nll)          # same batch (theta +/- h built inside the library), same sums
    ref, ref_g = orc.fd_gradient(x1, theta, idx, h, LO, HI)  # the oracle's own batch and differences
    for k in range(batch.shape[0]):
        ref_lp = orc.logpdf(x1, batch[k], LO, HI)
        assert np.abs(lp[k] - ref_lp).max() <= 1e-10
    assert np.all(np.abs(nll - ref) <= 1e-10 * np.abs(ref))
    assert grad_ok(grad.cpu().numpy(), ref_g)


def test_batch_independence_and_determinism(ipa, torch_, x1):
    batch, _ = inp.fd_batch(inp.GEN)
    xd = dev(torch_, x1)
    a, _, _ = ipa.ipa_nll_eval(xd, batch, LO, HI)
    b, _, _ = ipa.ipa_nll_eval(xd, batch, LO, HI)
    singles = [ipa.ipa_nll_eval(xd, batch[k], LO, HI)[0] for k in range(batch.shape[0])]
    perm = np.arange(batch.shape[0])[::-1].copy()
    c, _, _ = ipa.ipa_nll_eval(xd, batch[perm], LO, HI)
    torch_.cuda.synchronize()
    a, b, c = a.cpu().numpy(), b.cpu().numpy(), c.cpu().numpy()
    assert np.array_equal(a, b)  # run-to-run bitwise
    assert np.array_equal(a, np.array([s.item() for s in singles]))  # set k does not depend on its batch
    assert np.array_equal(a[perm], c)
    # sets sharing a signal shape are evaluated as a group: the first set of a group may be invalid (f out of
    # range), members may be pure signal / pure background; every valid member equals its stand-alone value
    grp = [dict(inp.GEN, f=1.5), dict(inp.GEN), dict(inp.GEN, f=0.2, k=-0.001), dict(inp.P2), dict(inp.GEN, f=1.0),
           dict(inp.GEN, f=0.0), dict(inp.P2, k=0.0)]
    g, _, st = ipa.ipa_nll_eval(xd, grp, LO, HI)
    alone = [ipa.ipa_nll_eval(xd, q, LO, HI)[0] for q in grp]
    torch_.cuda.synchronize()
    g = g.cpu().numpy()
    assert list(st.cpu().numpy()) == [1, 0, 0, 0, 0, 0, 0] and np.isposinf(g[0])
    assert np.array_equal(g[1:], np.array([s.item() for s in alone[1:]]))


@pytest.mark.parametrize("n", [0, 1, 2, 31, 1023, 1024, 1025, 4099])
def test_ragged_sizes_and_misalignment(ipa, torch_, orc, x1, n):
    big = dev(torch_, x1)
    for off in (0, 1):  # off=1: 8-byte but not 16-byte aligned -> scalar-load path
        xd = big[off:off + n]
        nll, lp, _ = ipa.ipa_nll_eval(xd, [inp.GEN, inp.P2], LO, HI, want_logpdf=True)
        torch_.cuda.synchronize()
        ref = orc.nll(x1[off:off + n], [inp.GEN, inp.P2], LO, HI)
        got = nll.cpu().numpy()
        if n == 0:
            assert np.array_equal(got, [0.0, 0.0]) and not np.signbit(got).any()
        else:
            assert np.all(np.abs(got - ref) <= 1e-10 * np.abs(ref))
            assert np.abs(lp[0].cpu().numpy() - orc.logpdf(x1[off:off + n], inp.GEN, LO, HI)).max() <= 1e-10


def test_norm(ipa, torch_, orc):
    sets = [dict(inp.GEN), dict(inp.P2)]
    sets.append(dict(inp.GEN, k=0.0))
    sets.append(dict(inp.GEN, n=1.0, n2=1.0))
    sets.append(dict(inp.GEN, mu=4900.0))           # range entirely inside the right tail
    sets.append(dict(inp.GEN, mu=5590.0, a2=0.5))   # right join inside, range cuts the core
    sets.append(dict(inp.P2, zeta=8.0, **{"lambda": 2.2}))
    sets.append(dict(inp.GEN, zeta=40.0))
    ns, nb, st = ipa.ipa_norm(sets, LO, HI)
    torch_.cuda.synchronize()
    ns, nb, st = ns.cpu().numpy(), nb.cpu().numpy(), st.cpu().numpy()
    for i, p in enumerate(sets):
        ost, o = orc.norm(p, LO, HI)
        assert st[i] == ost == 0
        assert abs(ns[i] / o["NS"] - 1) <= 2e-13, (i, ns[i], o["NS"])
        assert abs(nb[i] / o["NB"] - 1) <= 1e-14


def test_domain_status_does_not_poison_batch(ipa, torch_, orc, x1):
    bad = [dict(inp.GEN, sigma=-1.0), dict(inp.GEN, f=1.5), dict(inp.GEN, zeta=0.0), dict(inp.GEN, mu=float("nan")),
           dict(inp.GEN, beta=5.0)]  # beta=5: slope at the right join is positive -> status 2
    batch = [inp.GEN] + bad + [inp.P2]
    nll, _, st = ipa.ipa_nll_eval(dev(torch_, x1), batch, LO, HI)
    torch_.cuda.synchronize()
    nll, st = nll.cpu().numpy(), st.cpu().numpy()
    assert list(st) == [0, 1, 1, 1, 1, 2, 0]
    assert np.isposinf(nll[1:6]).all()
    ref = orc.nll(x1, [inp.GEN, inp.P2], LO, HI)
    assert np.all(np.abs(nll[[0, 6]] - ref) <= 1e-10 * np.abs(ref))
    assert orc.shape_consts(bad[4])[0] == 2


def test_limits_f0_f1_k0_outside_and_nan(ipa, torch_, orc, x1):
    x = x1[:3000].copy()
    x[:4] = [4990.0, 5610.0, LO, HI]  # events outside the range: same formulae, no clipping
    sets = [dict(inp.GEN, f=0.0), dict(inp.GEN, f=1.0), dict(inp.GEN, k=0.0), dict(inp.P2, f=1.0)]
    nll, lp, st = ipa.ipa_nll_eval(dev(torch_, x), sets, LO, HI, want_logpdf=True)
    torch_.cuda.synchronize()
    assert (st.cpu().numpy() == 0).all()
    for i, p in enumerate(sets):
        assert np.abs(lp[i].cpu().numpy() - orc.logpdf(x, p, LO, HI)).max() <= 1e-10
    ref = orc.nll(x, sets, LO, HI)
    assert np.all(np.abs(nll.cpu().numpy() - ref) <= 1e-10 * np.abs(ref))
    x[7] = float("nan")
    nll, _, _ = ipa.ipa_nll_eval(dev(torch_, x), inp.GEN, LO, HI)
    assert np.isnan(nll.cpu().numpy()[0])


def test_direct_mode_shapes(ipa, torch_, orc, x1):
    """Shapes whose core interval is too wide for one polynomial run the per-event Bessel path."""
    x = x1[:2000]
    sets = [dict(inp.GEN, zeta=0.2), dict(inp.GEN, zeta=0.05, **{"lambda": -2.0}), dict(inp.GEN, a=6.0, a2=7.0)]
    nll, lp, st = ipa.ipa_nll_eval(dev(torch_, x), sets, LO, HI, want_logpdf=True)
    torch_.cuda.synchronize()
    assert (st.cpu().numpy() == 0).all()
    for i, p in enumerate(sets):
        assert np.abs(lp[i].cpu().numpy() - orc.logpdf(x, p, LO, HI)).max() <= 1e-10, i
    ref = orc.nll(x, sets, LO, HI)
    assert np.all(np.abs(nll.cpu().numpy() - ref) <= 1e-10 * np.abs(ref))


def test_hypothesis_like_sweep(ipa, torch_, orc, x1):
    """Random valid shapes over the domain (seeded): per-event parity and normalisation."""
    rng = np.random.Generator(np.random.Philox(77))
    x = x1[:1500]
    sets = []
    for _ in range(24):
        sets.append(dict(mu=5280 + rng.uniform(-60, 60), sigma=rng.uniform(5, 40), **{"lambda": rng.uniform(-3, 3)},
                         zeta=10 ** rng.uniform(-0.3, 1.5), beta=rng.uniform(-0.01, 0.01), a=rng.uniform(0.8, 3.5),
                         n=rng.uniform(1.0, 6.0), a2=rng.uniform(0.8, 3.5), n2=rng.uniform(1.0, 6.0),
                         f=rng.uniform(0.05, 0.95), k=rng.uniform(-0.004, 0.001)))
    nll, lp, st = ipa.ipa_nll_eval(dev(torch_, x), sets, LO, HI, want_logpdf=True)
    torch_.cuda.synchronize()
    st = st.cpu().numpy()
    for i, p in enumerate(sets):
        ost, _ = orc.shape_consts(p)
        assert st[i] == ost
        if ost == 0:
            assert np.abs(lp[i].cpu().numpy() - orc.logpdf(x, p, LO, HI)).max() <= 1e-10, (i, p)


def test_cuda_graph_capture_and_side_stream(ipa, torch_, orc, x1):
    """The call enqueues on the caller's stream, never synchronises, and can be captured in a CUDA graph."""
    xd = dev(torch_, x1)
    batch, _ = inp.fd_batch(inp.GEN)
    ws = ipa.workspace(x1.size, 32)
    out = torch_.empty(9, dtype=torch_.float64, device="cuda")
    st = torch_.empty(9, dtype=torch_.int32, device="cuda")
    ref, _, _ = ipa.ipa_nll_eval(xd, batch, LO, HI)
    side = torch_.cuda.Stream()
    side.wait_stream(torch_.cuda.current_stream())
    with torch_.cuda.stream(side):
        ipa.ipa_nll_eval(xd, batch, LO, HI, ws=ws, stream=side, out=out, status=st)      # warm-up on the side stream
        side.synchronize()
        assert torch_.equal(out, ref)
        g = torch_.cuda.CUDAGraph()
        out.zero_()
        with torch_.cuda.graph(g, stream=side):
            ipa.ipa_nll_eval(xd, batch, LO, HI, ws=ws, stream=torch_.cuda.current_stream(), out=out, status=st)
        assert float(out.abs().sum()) == 0.0          # capture enqueues nothing
        g.replay()
        side.synchronize()
        assert torch_.equal(out, ref)
        out.zero_()
        g.replay()
        g.replay()
        torch_.cuda.synchronize()
        assert torch_.equal(out, ref)


# ---------------------------------------------------------------------------------------------
# generators (T0, T1), segmented NLL (T2)
# ---------------------------------------------------------------------------------------------
def test_mixture_generator_matches_oracle(ipa, torch_, orc):
    n = 20000
    for theta, seed in ((inp.GEN, 1), (inp.P2, 9)):
        x, off, ovf = ipa.ipa_toy_generate([seed], theta, -1.0, -1.0, LO, HI, n)
        torch_.cuda.synchronize()
        ref = orc.generate_mixture(seed, n, theta, LO, HI)
        got = x.cpu().numpy()
        assert list(off.cpu().numpy()) == [0, n] and ovf.item() == 0
        mismatches(got, ref, f"mixture seed {seed}")
        assert ((got >= LO) & (got <= HI)).all()
        # a shard of the same dataset (ipa_options.first_slot): slots 7001 .. 7001 + 5000 - 1, bitwise the same events
        part, _, _ = ipa.ipa_toy_generate([seed], theta, -1.0, -1.0, LO, HI, 5000, first_slot=7001)
        torch_.cuda.synchronize()
        assert torch_.equal(part, x[7001:12001])


@pytest.mark.parametrize("case", ["beta_large", "mode_left_of_range", "mode_left_of_range_b", "range_inside_left_tail",
                                  "range_inside_right_tail", "n_equal_one", "student_t_beta"])
def test_signal_envelope_cases(ipa, torch_, orc, case):
    """Reading D13 (revised): exact tails + boxes on the core.  Signal-only draws (f = 1) in the cases the old flat
    envelope got wrong or slow (advisor finding, round 1): beta != 0, the maximum at a range end, the range inside
    one tail, n = 1, the Student-t core.  No event differs from the oracle generator's, and the flag that records
    a core value above its box (code 2) stays clear."""
    theta = dict({"beta_large": dict(inp.P2, beta=0.05), "mode_left_of_range": dict(inp.GEN, mu=4998.0, sigma=3.0),
                  "mode_left_of_range_b": dict(inp.GEN, mu=4995.0, sigma=5.0, beta=-0.02),
                  "range_inside_left_tail": dict(inp.GEN, mu=5700.0, n=1.0), "range_inside_right_tail": dict(inp.P2, mu=4900.0),
                  "n_equal_one": dict(inp.GEN, n=1.0, n2=1.0), "student_t_beta": inp.T2}[case], f=1.0)
    n = 30000
    x, _, ovf = ipa.ipa_toy_generate([77], theta, -1.0, -1.0, LO, HI, n)
    torch_.cuda.synchronize()
    assert ovf.item() == 0
    got = x.cpu().numpy()
    assert ((got >= LO) & (got <= HI)).all()
    mismatches(got, orc.generate_mixture(77, n, theta, LO, HI), f"signal envelope, {case}")


def test_range_inside_one_tail_with_a_large_exponent(ipa, torch_, orc):
    """Advisor finding (round 1): F(ul) - F(ur) of the tail normalisation cancels when the whole range lies inside one
    tail and n is large; the difference is now formed directly (ipa_powint_diff)."""
    x = np.linspace(LO, HI, 2001)
    for mu in (5610.0, 5627.0, 5700.0):
        th = dict(inp.GEN, mu=mu, sigma=0.89, a=2.34, n=66.0)
        nll, lp, st = ipa.ipa_nll_eval(dev(torch_, x), th, LO, HI, want_logpdf=True)
        ns, _, _ = ipa.ipa_norm(th, LO, HI)
        torch_.cuda.synchronize()
        ost, o = orc.norm(th, LO, HI)
        assert st.item() == ost == 0
        assert abs(ns.item() / o["NS"] - 1) <= 1e-12
        assert np.abs(lp[0].cpu().numpy() - orc.logpdf(x, th, LO, HI)).max() <= 1e-10


def test_toy_generator_and_segmented_nll(ipa, torch_, orc):
    T = 24
    seeds = inp.toy_seeds(T)
    ms, mb = 300.0, 700.0
    _, off_ref = orc.toy_generate(seeds, inp.GEN, ms, mb, LO, HI, offsets_only=True)
    cap = int(off_ref[-1])
    x, off, ovf = ipa.ipa_toy_generate(seeds, inp.GEN, ms, mb, LO, HI, cap)
    torch_.cuda.synchronize()
    assert np.array_equal(off.cpu().numpy(), off_ref) and ovf.item() == 0   # Poisson yields: bit-exact
    x_ref, _ = orc.toy_generate(seeds, inp.GEN, ms, mb, LO, HI)
    got = x.cpu().numpy()
    mismatches(got, x_ref, "24 toys")
    # per-toy parameter sets (reading D17), NLL of every toy in one launch, on the GPU-generated events
    sets = inp.toy_param_sets(T)
    nll, st = ipa.ipa_nll_eval_segmented(x, off, sets, LO, HI)
    torch_.cuda.synchronize()
    ref = orc.nll_segmented(got, off_ref, sets, LO, HI)
    assert (st.cpu().numpy() == 0).all()
    assert np.all(np.abs(nll.cpu().numpy() - ref) <= 1e-10 * np.abs(ref))
    # capacity too small: offsets still written, overflow flagged, nothing written past capacity
    x2, off2, ovf2 = ipa.ipa_toy_generate(seeds, inp.GEN, ms, mb, LO, HI, cap - 100)
    torch_.cuda.synchronize()
    assert ovf2.item() == 1 and np.array_equal(off2.cpu().numpy(), off_ref)


def test_segmented_many_sets_and_empty_segments(ipa, torch_, orc, x1):
    """T > IPA_MAX_K (parameter sets travel through the workspace) with empty and tiny segments."""
    T = 70
    rng = np.random.Generator(np.random.Philox(5))
    cuts = np.sort(rng.integers(0, x1.size, size=T - 1))
    off = np.concatenate([[0], cuts, [x1.size]]).astype(np.int64)
    off[10] = off[9]  # force an empty segment
    off = np.maximum.accumulate(off)
    sets = inp.toy_param_sets(T, seed=11)
    nll, st = ipa.ipa_nll_eval_segmented(dev(torch_, x1), dev(torch_, off), sets, LO, HI)
    torch_.cuda.synchronize()
    ref = orc.nll_segmented(x1, off, sets, LO, HI)
    got = nll.cpu().numpy()
    assert np.all(np.abs(got - ref) <= 1e-10 * np.abs(ref) + 0.0)
    assert got[9] == 0.0 or off[10] != off[9]


# ---------------------------------------------------------------------------------------------
# binned path (B1-B3)
# ---------------------------------------------------------------------------------------------
def test_hist_fill_exact(ipa, torch_, orc, x1):
    x = np.concatenate([x1, [LO, HI, LO - 1e-9, HI + 1e-9, np.nextafter(HI, 0)]])
    for nbins in (1, 7, 1000, 10000):
        c = ipa.ipa_hist_fill(dev(torch_, x), LO, HI, nbins)
        torch_.cuda.synchronize()
        assert np.array_equal(c.cpu().numpy().astype(np.uint64), orc.hist_fill(x, LO, HI, nbins))


def test_binned_scan_expected_hist_and_poisson_toys(ipa, torch_, orc):
    nbins = 1000
    x = inp.standin_masses(5, 200000, f=0.02)
    counts = orc.hist_fill(x, LO, HI, nbins)
    ns, nb, kk = inp.scan_grid(12, 9, n_obs=float(x.size))
    cd = dev(torch_, counts.astype(np.int64))
    got = ipa.ipa_binned_nll_scan(cd, LO, HI, inp.GEN, ns, nb, kk)
    torch_.cuda.synchronize()
    ref = orc.binned_nll_scan(counts, LO, HI, inp.GEN, ns, nb, kk)
    assert np.all(np.abs(got.cpu().numpy() - ref) <= 1e-10 * np.abs(ref))
    nu = ipa.ipa_expected_hist(nbins, LO, HI, inp.GEN, 2500.0, 1e5, -0.002)
    torch_.cuda.synchronize()
    nu_ref = orc.expected_hist(nbins, LO, HI, inp.GEN, 2500.0, 1e5, -0.002)
    assert np.all(np.abs(nu.cpu().numpy() - nu_ref) <= 1e-12 * nu_ref)
    seeds = np.arange(1, 41, dtype=np.uint64)
    mean = np.concatenate([nu_ref[:500], [0.0, 0.3, 3.0, 9.99, 10.0, 55.5]])
    toys = ipa.ipa_poisson_hist_toys(dev(torch_, mean), seeds)
    torch_.cuda.synchronize()
    ref_t = orc.poisson_hist_toys(mean, seeds)
    got_t = toys.cpu().numpy().astype(np.uint32)
    mismatches(got_t.astype(np.float64), ref_t.astype(np.float64), "per-bin Poisson toys", tol=0.0)   # integer draws: equal
    # few bins, many toys (a block then covers several toys at a time), one bin, one toy
    for m2, T2 in ((np.array([0.0, 4.5, 12.0, 3e4, 7e4]), 301), (np.array([37.5]), 77), (mean[:300], 1), (mean[:257], 3)):
        sd = np.arange(100, 100 + T2, dtype=np.uint64)
        g2 = ipa.ipa_poisson_hist_toys(dev(torch_, m2), sd)
        torch_.cuda.synchronize()
        assert np.array_equal(g2.cpu().numpy().astype(np.uint32).reshape(T2, m2.size), orc.poisson_hist_toys(m2, sd).reshape(T2, m2.size))


# ---------------------------------------------------------------------------------------------
# optional preparation: events grouped by a coarse bin index (stable counting sort); reading E4
# ---------------------------------------------------------------------------------------------
def coarse_bins(x, nb=256):
    """bin index of the header: clamp(floor((x - lo) nb / (hi - lo)), 0, nb - 1), NaN -> last bin (host restatement)."""
    t = (x - LO) * (nb / (HI - LO))
    b = np.where(t < nb, np.floor(np.where(np.isnan(t), 0.0, t)), nb - 1)
    b = np.where(np.isnan(t), nb - 1, b)
    return np.clip(b, 0, nb - 1).astype(np.int64)


def stable_by_bin(x):
    return x[np.argsort(coarse_bins(x), kind="stable")]


@pytest.mark.parametrize("n", [0, 1, 31, 8191, 8192, 8193, 100_003, 2_500_000])
def test_events_prepare_is_the_stable_counting_sort(ipa, torch_, orc, n):
    """Integer / index work: bit-exact against numpy's stable argsort on the bin index, for sizes below, at and above
    one tile, several tiles per block and several blocks, ragged tails; events outside the range, at the edges, NaN."""
    x = inp.standin_masses(21, max(n, 1))[:n].copy()
    if n >= 31:
        x[:9] = [LO, HI, LO - 3.0, HI + 2.0, np.nextafter(HI, 0), 5279.99999, 5280.0, float("nan"), 5000.29296875]
    xd = dev(torch_, x)
    a = ipa.ipa_events_prepare(xd, LO, HI)
    b = ipa.ipa_events_prepare(xd, LO, HI)
    torch_.cuda.synchronize()
    got = a.cpu().numpy()
    assert np.array_equal(got, stable_by_bin(x), equal_nan=True)
    assert np.array_equal(got, b.cpu().numpy(), equal_nan=True)         # run to run
    assert np.array_equal(xd.cpu().numpy(), x, equal_nan=True)          # input untouched
    if n >= 8193:                                                        # misaligned input (8-byte aligned only), sorted input
        assert np.array_equal(ipa.ipa_events_prepare(xd[1:], LO, HI).cpu().numpy(), stable_by_bin(x[1:]), equal_nan=True)
        assert np.array_equal(ipa.ipa_events_prepare(a, LO, HI).cpu().numpy(), got, equal_nan=True)     # idempotent


def test_prepared_nll(ipa, torch_, orc, x1):
    x = np.concatenate([x1, [LO, HI, 5250.0, 5250.0, 5310.0]])
    xd = dev(torch_, x)
    xs = ipa.ipa_events_prepare(xd, LO, HI)
    idx, h = inp.fd_spec()
    a, ga, _ = ipa.ipa_nll_fd_gradient(xd, inp.P2, idx, h, LO, HI)
    b, gb, _ = ipa.ipa_nll_fd_gradient(xs, inp.P2, idx, h, LO, HI)
    _, lp, _ = ipa.ipa_nll_eval(xs, inp.P2, LO, HI, want_logpdf=True)
    torch_.cuda.synchronize()
    a, b = a.cpu().numpy(), b.cpu().numpy()
    assert np.all(np.abs(a - b) <= 1e-12 * np.abs(a))            # order changes rounding only
    ref, ref_g = orc.fd_gradient(x, inp.P2, idx, h, LO, HI)      # oracle: original order, pairwise
    assert np.all(np.abs(b - ref) <= 1e-10 * np.abs(ref))
    assert grad_ok(gb.cpu().numpy(), ref_g) and grad_ok(ga.cpu().numpy(), ref_g)
    assert np.abs(lp[0].cpu().numpy() - orc.logpdf(xs.cpu().numpy(), inp.P2, LO, HI)).max() <= 1e-10


def test_segmented_prepare(ipa, torch_, orc, x1):
    off = np.array([0, 0, 17, 4000, 4000, 10000], dtype=np.int64)
    xd, od = dev(torch_, x1), dev(torch_, off)
    xs = ipa.ipa_events_prepare(xd, LO, HI, od)
    torch_.cuda.synchronize()
    got = xs.cpu().numpy()
    for t in range(off.size - 1):
        assert np.array_equal(got[off[t]:off[t + 1]], stable_by_bin(x1[off[t]:off[t + 1]]))
    sets = inp.toy_param_sets(off.size - 1, seed=3)
    a, _ = ipa.ipa_nll_eval_segmented(xs, od, sets, LO, HI)
    torch_.cuda.synchronize()
    ref = orc.nll_segmented(x1, off, sets, LO, HI)
    assert np.all(np.abs(a.cpu().numpy() - ref) <= 1e-10 * np.abs(ref))


# ---------------------------------------------------------------------------------------------
# full size, in the launch configuration bench.py times (config 3: 1e8 events, K = 1 and K = 9)
# ---------------------------------------------------------------------------------------------
def test_full_size_sampled(ipa, torch_, orc):
    """Config 3 at full size on the events bench.py times: 1e8 events of the model, seed 3, from the device generator
    (checked against the oracle's generator on a prefix); K = 1 and K = 9, degree policy 1, as generated and prepared.
    The 1e8-event total is compared with the SINGLE-THREAD oracle (pairwise sum, original order)."""
    n = 100_000_000
    xd, _, ovf = ipa.ipa_toy_generate([3], inp.GEN, -1.0, -1.0, LO, HI, n)
    torch_.cuda.synchronize()
    assert ovf.item() == 0
    x = xd.cpu().numpy()
    mismatches(x[:300_000], orc.generate_mixture(3, 300_000, inp.GEN, LO, HI), "config 3 prefix")
    batch, _ = inp.fd_batch(inp.GEN)
    nll1, lp, _ = ipa.ipa_nll_eval(xd, inp.GEN, LO, HI, want_logpdf=True, policy=1)
    nll9, _, _ = ipa.ipa_nll_eval(xd, batch, LO, HI, policy=1)
    torch_.cuda.synchronize()
    # property: the reduction equals the fp64 sum of the per-event outputs
    s = -lp[0].sum().item()
    assert abs(nll1.item() - s) <= 1e-11 * abs(s)
    assert nll9[0].item() == nll1.item()
    # sampled outputs against the oracle, one by one (includes the ragged last tile)
    rng = np.random.Generator(np.random.Philox(123))
    idx = np.concatenate([rng.integers(0, n, size=40000), np.arange(n - 3000, n), np.arange(0, 3000)])
    got = lp[0][torch_.from_numpy(idx).cuda()].cpu().numpy()
    assert np.abs(got - orc.logpdf(x[idx], inp.GEN, LO, HI)).max() <= 1e-10
    del lp
    # total at 1e8 events against the single-thread oracle
    ref1 = orc.nll(x, inp.GEN, LO, HI)[0]
    rel = abs(nll1.item() - ref1) / abs(ref1)
    print(f"[config 3] NLL gpu {nll1.item():.17g} oracle (1 thread) {ref1:.17g} rel diff {rel:.3g}")
    assert rel <= 1e-10
    # the whole K = 9 batch against the single-thread oracle on the first 1e7 events
    m = 10_000_000
    ref9 = orc.nll(x[:m], batch, LO, HI)
    part, _, _ = ipa.ipa_nll_eval(xd[:m], batch, LO, HI, policy=1)
    assert np.all(np.abs(part.cpu().numpy() - ref9) <= 1e-10 * np.abs(ref9))
    # the prepared layout bench.py times: same total up to rounding, sampled outputs against the oracle
    xs = ipa.ipa_events_prepare(xd, LO, HI)
    nlls, lps, _ = ipa.ipa_nll_eval(xs, inp.GEN, LO, HI, want_logpdf=True, policy=1)
    nlls9, _, _ = ipa.ipa_nll_eval(xs, batch, LO, HI, policy=1)
    torch_.cuda.synchronize()
    assert abs(nlls.item() - nll1.item()) <= 1e-12 * abs(nll1.item())
    assert abs(nlls.item() - ref1) <= 1e-10 * abs(ref1) and nlls9[0].item() == nlls.item()
    assert np.all(np.abs(nlls9.cpu().numpy() - nll9.cpu().numpy()) <= 1e-12 * np.abs(nll9.cpu().numpy()))
    # the prepared array is the stable counting sort of the input: grouped by non-decreasing bin, a permutation
    bins = ((xs - LO) * (256.0 / (HI - LO))).floor().clamp_(0, 255)
    assert bool((bins[1:] >= bins[:-1]).all().item())
    assert np.array_equal(xs[:1_000_000].cpu().numpy(), stable_by_bin(x)[:1_000_000])
    del bins
    sel = torch_.from_numpy(idx).cuda()
    assert np.abs(lps[0][sel].cpu().numpy() - orc.logpdf(xs[sel].cpu().numpy(), inp.GEN, LO, HI)).max() <= 1e-10
    parts, _, _ = ipa.ipa_nll_eval(ipa.ipa_events_prepare(xd[:m], LO, HI), batch, LO, HI, policy=1)
    assert np.all(np.abs(parts.cpu().numpy() - ref9) <= 1e-10 * np.abs(ref9))


# ---------------------------------------------------------------------------------------------
# full size, config 4 (1000 toys x ~1e5 events generated on the device, one segmented launch) and
# config 5 (1e8 events -> 1000 bins, 100 x 100 scan, 10 000 Poisson toy histograms)
# ---------------------------------------------------------------------------------------------
def test_config4_full_size_sampled(ipa, torch_, orc):
    T = 1000
    seeds = inp.toy_seeds(T)
    ms, mb = 30000.0, 70000.0
    _, off_ref = orc.toy_generate(seeds, inp.GEN, ms, mb, LO, HI, offsets_only=True)
    cap = int(off_ref[-1])
    x, off, ovf = ipa.ipa_toy_generate(seeds, inp.GEN, ms, mb, LO, HI, cap)
    sets = inp.toy_param_sets(T)
    nll, st = ipa.ipa_nll_eval_segmented(x, off, sets, LO, HI)
    xs = ipa.ipa_events_prepare(x, LO, HI, off)
    nll_s, _ = ipa.ipa_nll_eval_segmented(xs, off, sets, LO, HI)
    torch_.cuda.synchronize()
    assert ovf.item() == 0 and np.array_equal(off.cpu().numpy(), off_ref)      # all 1000 Poisson yields: bit-exact
    assert abs(cap - 1e8) < 5e5
    nll, nll_s = nll.cpu().numpy(), nll_s.cpu().numpy()
    assert (st.cpu().numpy() == 0).all()
    assert np.all(np.abs(nll - nll_s) <= 1e-12 * np.abs(nll))                  # per-toy sort: rounding only
    pick = [0, 1, 137, 499, 998, 999]
    # events of the sampled toys against the oracle's generator (same seeds -> same counters)
    x_ref, o_ref = orc.toy_generate(seeds[pick], inp.GEN, ms, mb, LO, HI)
    for j, t in enumerate(pick):
        got = x[off_ref[t]:off_ref[t + 1]].cpu().numpy()
        ref = x_ref[o_ref[j]:o_ref[j + 1]]
        assert got.size == ref.size
        mismatches(got, ref, f"config 4 toy {t}")
        # NLL of the toy with its own parameter set, oracle on the GPU-generated events
        r = orc.nll(got, sets[t], LO, HI)[0]
        assert abs(nll[t] - r) <= 1e-10 * abs(r), t
        single, _, _ = ipa.ipa_nll_eval(x[off_ref[t]:off_ref[t + 1]], sets[t], LO, HI)
        assert abs(single.item() - nll[t]) <= 1e-12 * abs(nll[t])
    # property at full size: every toy's NLL per event sits at the population value 6.09 +- 5 sigma
    per_event = nll / np.diff(off_ref)
    assert np.all(np.abs(per_event - 6.0901) < 0.02)


def test_config5_full_size(ipa, torch_, orc):
    n, nbins = 100_000_000, 1000
    x = inp.standin_masses(5, n, f=2.5e-5)
    xd = dev(torch_, x)
    counts = ipa.ipa_hist_fill(xd, LO, HI, nbins)
    torch_.cuda.synchronize()
    c_ref = orc.hist_fill(x, LO, HI, nbins)
    got = counts.cpu().numpy().astype(np.uint64)
    assert np.array_equal(got, c_ref) and int(got.sum()) == n                  # integer work: exact
    cm = ipa.ipa_hist_fill(xd[1:], LO, HI, nbins)                              # 8-byte-aligned start: scalar head
    assert np.array_equal(cm.cpu().numpy().astype(np.uint64), orc.hist_fill(x[1:], LO, HI, nbins))
    del xd
    ns, nb, kk = inp.scan_grid(100, 100, n_obs=float(n))
    scan = ipa.ipa_binned_nll_scan(counts, LO, HI, inp.GEN, ns, nb, kk)
    torch_.cuda.synchronize()
    scan = scan.cpu().numpy()
    ref = orc.binned_nll_scan(c_ref, LO, HI, inp.GEN, ns, nb, kk)
    assert np.all(np.abs(scan - ref) <= 1e-10 * np.abs(ref))
    # 10 000 toy histograms: 5 000 background-only at the best k, 5 000 with ns = 2500 (reading D16)
    kbest = kk[int(np.argmin(ref))]
    seeds = np.arange(1, 10001, dtype=np.uint64)
    for ns_gen, sd in ((0.0, seeds[:5000]), (2500.0, seeds[5000:])):
        nu = ipa.ipa_expected_hist(nbins, LO, HI, inp.GEN, ns_gen, n - ns_gen, kbest)
        toys = ipa.ipa_poisson_hist_toys(nu, sd)
        torch_.cuda.synchronize()
        nu_ref = orc.expected_hist(nbins, LO, HI, inp.GEN, ns_gen, n - ns_gen, kbest)
        assert np.all(np.abs(nu.cpu().numpy() - nu_ref) <= 1e-12 * nu_ref)
        t = toys.cpu().numpy().astype(np.uint32)
        sample = np.array([0, 1, 2499, 4999])
        ref_t = orc.poisson_hist_toys(nu_ref, sd[sample])
        mismatches(t[sample].astype(np.float64), ref_t.astype(np.float64), f"config 5 Poisson toys ns={ns_gen}", tol=0.0)
        # property over all toys: pulls of the counts are standard normal
        pull = (t.astype(np.float64) - nu_ref[None, :]) / np.sqrt(nu_ref[None, :])
        assert abs(pull.mean()) < 3e-3 and abs(pull.std() - 1.0) < 3e-3


# ---------------------------------------------------------------------------------------------
# CLs on binned toys (reading F2)
# ---------------------------------------------------------------------------------------------
def test_cls_teststat_counts_and_levels(ipa, torch_, orc):
    n, nbins, T = 10_000_000, 1000, 5000
    x = inp.standin_masses(5, n, f=2.5e-4)                       # "data": 2 500 signal-like events in 1e7
    data = ipa.ipa_hist_fill(dev(torch_, x), LO, HI, nbins)       # uint64 payload
    c_ref = orc.hist_fill(x, LO, HI, nbins)
    ns, k = 2500.0, -0.002
    nu_b = ipa.ipa_expected_hist(nbins, LO, HI, inp.GEN, 0.0, float(n), k)
    nu_sb = ipa.ipa_expected_hist(nbins, LO, HI, inp.GEN, ns, float(n) - ns, k)
    nu_b_ref = orc.expected_hist(nbins, LO, HI, inp.GEN, 0.0, float(n), k)
    nu_sb_ref = orc.expected_hist(nbins, LO, HI, inp.GEN, ns, float(n) - ns, k)
    toys_b = ipa.ipa_poisson_hist_toys(nu_b, np.arange(1, T + 1, dtype=np.uint64))
    toys_sb = ipa.ipa_poisson_hist_toys(nu_sb, np.arange(T + 1, 2 * T + 1, dtype=np.uint64))
    q_obs = ipa.ipa_cls_teststat(data, nu_sb, nu_b)
    q_b = ipa.ipa_cls_teststat(toys_b, nu_sb, nu_b)
    q_sb = ipa.ipa_cls_teststat(toys_sb, nu_sb, nu_b)
    c_b = ipa.ipa_cls_count_ge(q_b, q_obs)
    c_sb = ipa.ipa_cls_count_ge(q_sb, q_obs)
    cl = ipa.ipa_cls_from_counts(c_sb, T, c_b, T)
    torch_.cuda.synchronize()
    # statistic: the oracle on the GPU's own toy histograms and expected histograms' oracle twins
    scale = 2.0 * ns                                              # size of the two terms that cancel in q
    for q_gpu, toys in ((q_b, toys_b), (q_sb, toys_sb)):
        ref = orc.cls_teststat(toys.cpu().numpy().astype(np.uint32), nu_sb_ref, nu_b_ref)
        assert np.all(np.abs(q_gpu.cpu().numpy() - ref) <= 1e-10 * (np.abs(ref) + scale))
    ref_obs = orc.cls_teststat(c_ref.reshape(1, -1), nu_sb_ref, nu_b_ref)[0]
    assert abs(q_obs.item() - ref_obs) <= 1e-10 * (abs(ref_obs) + scale)
    # counting is integer work: exact against the oracle on the GPU's q values
    qb, qsb = q_b.cpu().numpy(), q_sb.cpu().numpy()
    assert c_b.item() == orc.cls_count_ge(qb, q_obs.item()) and c_sb.item() == orc.cls_count_ge(qsb, q_obs.item())
    assert np.array_equal(cl.cpu().numpy(), orc.cls_from_counts(c_sb.item(), T, c_b.item(), T), equal_nan=True)
    # ragged shapes: rows that are not 16-byte aligned take the scalar loads (both count widths)
    rng = np.random.Generator(np.random.Philox(8))
    for nb_, T_ in ((7, 9), (1, 3), (1001, 17)):
        vb = rng.uniform(0.5, 300.0, nb_)
        vsb = vb * rng.uniform(1.0, 1.5, nb_)
        cnt = rng.poisson(vb, size=(T_, nb_))
        for dt_np, dt_t in ((np.uint32, torch_.int32), (np.uint64, torch_.int64)):
            qg = ipa.ipa_cls_teststat(dev(torch_, cnt.astype(np.int64)).to(dt_t), dev(torch_, vsb), dev(torch_, vb))
            ref = orc.cls_teststat(cnt.astype(dt_np), vsb, vb)
            assert np.all(np.abs(qg.cpu().numpy() - ref) <= 1e-10 * (np.abs(ref) + 2 * (vsb - vb).sum()))
    # properties at this size: q is larger (more background-like) on background-only toys, so CL_b >= CL_sb for any
    # observed value, and the two ensembles are separated by about the expected significance (2.5 sigma here)
    v = cl.cpu().numpy()
    assert 0.0 <= v[0] <= v[1] <= 1.0
    assert (qb.mean() - qsb.mean()) > 1.5 * max(qb.std(), qsb.std())


# ---------------------------------------------------------------------------------------------
# maximum sizes: more than 2^31 events (64-bit indexing end to end)
# ---------------------------------------------------------------------------------------------
def test_more_than_2_pow_31_events(ipa, torch_, orc):
    n = 2 ** 31 + 4099                                         # 17.2 GB of events; ragged last tile
    x = torch_.empty(n, dtype=torch_.float64, device="cuda")
    half = n // 2
    x[:half] = 5250.0                                          # core region
    x[half:] = 5400.0                                          # right tail
    sets = [inp.GEN, inp.P2]
    nll, _, st = ipa.ipa_nll_eval(x, sets, LO, HI)
    counts = ipa.ipa_hist_fill(x, LO, HI, 1000)
    torch_.cuda.synchronize()
    assert (st.cpu().numpy() == 0).all()
    got = nll.cpu().numpy()
    for i, p in enumerate(sets):
        l = orc.logpdf(np.array([5250.0, 5400.0]), p, LO, HI)
        ref = -(half * l[0] + (n - half) * l[1])
        assert abs(got[i] - ref) <= 1e-10 * abs(ref)
    c = counts.cpu().numpy()
    assert int(c.sum()) == n and int(c[416]) == half and int(c[666]) == n - half   # bins of 5250 and 5400
    # the layout preparation at the same size (64-bit output positions, 32-bit per-block counts): interleave the two
    # values, prepare, and the result is the two runs again
    del counts
    x[0::2] = 5400.0
    x[1::2] = 5250.0
    n5400 = (n + 1) // 2
    y = ipa.ipa_events_prepare(x, LO, HI)
    torch_.cuda.synchronize()
    assert bool((y[:n - n5400] == 5250.0).all().item()) and bool((y[n - n5400:] == 5400.0).all().item())
    nll2, _, _ = ipa.ipa_nll_eval(y, sets, LO, HI)
    l = orc.logpdf(np.array([5250.0, 5400.0]), sets[0], LO, HI)
    ref = -((n - n5400) * l[0] + n5400 * l[1])
    assert abs(nll2[0].item() - ref) <= 1e-10 * abs(ref)


# ---------------------------------------------------------------------------------------------
# analytic gradient in one pass
# ---------------------------------------------------------------------------------------------
def test_analytic_gradient_vs_oracle(ipa, torch_, orc, x1):
    for x in (x1, np.sort(x1), x1[:4099], x1[1:2050]):                 # unsorted / sorted / ragged / misaligned
        xd = dev(torch_, x1)[1:2050] if x.size == 2049 else dev(torch_, x)
        sets = [inp.GEN, inp.P2, dict(inp.GEN, zeta=0.2), dict(inp.GEN, f=0.0), dict(inp.GEN, f=1.0),
                dict(inp.GEN, sigma=-1.0), dict(inp.P2, k=0.0)]
        nll, grad, st = ipa.ipa_nll_grad_eval(xd, sets, LO, HI)
        plain, _, _ = ipa.ipa_nll_eval(xd, sets, LO, HI)
        torch_.cuda.synchronize()
        nll, grad, st, plain = nll.cpu().numpy(), grad.cpu().numpy(), st.cpu().numpy(), plain.cpu().numpy()
        assert list(st) == [0, 0, 0, 4, 4, 1, 0]
        assert np.isposinf(nll[3:6]).all() and np.isnan(grad[3:6]).all()
        for i in (0, 1, 2, 6):
            ref_nll, ref_g = orc.nll_gradient(x, sets[i], LO, HI)
            assert abs(nll[i] - ref_nll) <= 1e-10 * abs(ref_nll)
            assert abs(nll[i] - plain[i]) <= 1e-12 * abs(plain[i])     # same value as ipa_nll_eval up to rounding
            assert grad_ok(grad[i], ref_g), (i, grad[i], ref_g)


def test_student_t_core_all_entry_points(ipa, torch_, orc, x1):
    """Row f4, reading D3: the zeta = 0 Student-t core through every unbinned entry point -- sorted (region-uniform
    warps) and as-generated layouts, a batch mixing Bessel and Student-t sets, the analytic gradient, the segmented
    call, ipa_norm, the domain rule (zeta = 0 needs lambda < 0) and the generator."""
    sets = [inp.T1, inp.GEN, inp.T2, dict(inp.T1, **{"lambda": 0.5}), dict(inp.T2, f=0.2, k=-0.001)]
    for x in (x1, np.sort(x1)):
        xd = dev(torch_, x)
        nll, lp, st = ipa.ipa_nll_eval(xd, sets, LO, HI, want_logpdf=True)
        gn, grad, gst = ipa.ipa_nll_grad_eval(xd, [inp.T1, inp.T2], LO, HI)
        torch_.cuda.synchronize()
        nll, lp, st = nll.cpu().numpy(), lp.cpu().numpy(), st.cpu().numpy()
        assert list(st) == [0, 0, 0, 1, 0] and np.isposinf(nll[3]) and np.isnan(lp[3]).all()
        for i in (0, 1, 2, 4):
            assert np.abs(lp[i] - orc.logpdf(x, sets[i], LO, HI)).max() <= 1e-10
            ref = orc.nll(x, sets[i], LO, HI)[0]
            assert abs(nll[i] - ref) <= 1e-10 * abs(ref)
        for i, th in enumerate((inp.T1, inp.T2)):
            ref_nll, ref_g = orc.nll_gradient(x, th, LO, HI)
            assert gst[i].item() == 0 and abs(gn[i].item() - ref_nll) <= 1e-10 * abs(ref_nll)
            assert grad_ok(grad[i].cpu().numpy(), ref_g), (i, grad[i], ref_g)
    ns, nb, st = ipa.ipa_norm([inp.T1, inp.T2, dict(inp.T1, mu=5700.0, n=1.0)], LO, HI)
    torch_.cuda.synchronize()
    for i, th in enumerate((inp.T1, inp.T2, dict(inp.T1, mu=5700.0, n=1.0))):
        _, nrm = orc.norm(th, LO, HI)
        assert st[i].item() == 0 and abs(ns[i].item() / nrm["NS"] - 1) <= 2e-13 and abs(nb[i].item() / nrm["NB"] - 1) <= 1e-14
    off = np.array([0, 3000, 3000, 10000], dtype=np.int64)
    seg, sst = ipa.ipa_nll_eval_segmented(dev(torch_, x1), dev(torch_, off), [inp.T1, inp.GEN, inp.T2], LO, HI)
    torch_.cuda.synchronize()
    ref = orc.nll_segmented(x1, off, [inp.T1, inp.GEN, inp.T2], LO, HI)
    assert np.all(np.abs(seg.cpu().numpy() - ref) <= 1e-10 * np.abs(ref))
    for th, seed in ((inp.T1, 41), (inp.T2, 42)):
        xg, _, ovf = ipa.ipa_toy_generate([seed], th, -1.0, -1.0, LO, HI, 20000)
        torch_.cuda.synchronize()
        assert ovf.item() == 0
        mismatches(xg.cpu().numpy(), orc.generate_mixture(seed, 20000, th, LO, HI), f"Student-t mixture seed {seed}")


def test_analytic_gradient_many_sets_one_pass_per_group(ipa, torch_, orc, x1):
    """Gradient kernel v2: up to 4 sets per event read, more sets in groups (one ticket counter per group); every set
    equals its stand-alone evaluation bitwise and the oracle within tolerance, for K = 1 .. 9 and ragged sizes."""
    xd = dev(torch_, x1[:8191])
    sets = [dict(inp.GEN, mu=5280.0 + 0.3 * i, f=0.25 + 0.01 * i) for i in range(9)]
    sets[5] = inp.P2
    sets[7] = inp.T2
    alone = [ipa.ipa_nll_grad_eval(xd, q, LO, HI) for q in sets]
    for K in (1, 4, 5, 9):
        nll, grad, st = ipa.ipa_nll_grad_eval(xd, sets[:K], LO, HI)
        torch_.cuda.synchronize()
        assert (st.cpu().numpy() == 0).all()
        for i in range(K):
            assert nll[i].item() == alone[i][0].item() and torch_.equal(grad[i], alone[i][1][0])
    for i in (0, 5, 7, 8):
        ref_nll, ref_g = orc.nll_gradient(x1[:8191], sets[i], LO, HI)
        assert abs(alone[i][0].item() - ref_nll) <= 1e-10 * abs(ref_nll)
        assert grad_ok(alone[i][1][0].cpu().numpy(), ref_g)


def test_analytic_gradient_1e6_and_fit_minimum(ipa, torch_, orc):
    n = 1_000_000
    x = orc.generate_mixture(2, n, inp.GEN, LO, HI)
    xd = ipa.ipa_events_prepare(dev(torch_, x), LO, HI)
    for theta in (inp.GEN, dict(inp.GEN, mu=5281.0, sigma=16.0, f=0.32, k=-0.0019)):
        nll, grad, st = ipa.ipa_nll_grad_eval(xd, theta, LO, HI)
        torch_.cuda.synchronize()
        ref_nll, ref_g = orc.nll_gradient(x, theta, LO, HI)
        assert st.item() == 0 and abs(nll.item() - ref_nll) <= 1e-10 * abs(ref_nll)
        assert grad_ok(grad[0].cpu().numpy(), ref_g)
    # consistency with the finite-difference batch of the same library (truncation error of the differences)
    idx, h = inp.fd_spec()
    fd = ipa.ipa_nll_fd_gradient(xd, inp.GEN, idx, h, LO, HI)[1].cpu().numpy()
    an = ipa.ipa_nll_grad_eval(xd, inp.GEN, LO, HI)[1][0].cpu().numpy()[:4]
    s = np.array([inp.GRAD_SCALE[k] for k in inp.FLOATED])
    assert np.all(np.abs(fd - an) <= 1e-3 * np.maximum(np.abs(an), 1.0 / s))


def test_maximum_batch_of_32_sets(ipa, torch_, orc, x1):
    """K = IPA_MAX_K: the largest shared-memory footprint of the streaming kernel (grouped and ungrouped)."""
    xd = dev(torch_, np.sort(x1))
    rng = np.random.Generator(np.random.Philox(32))
    distinct = [dict(inp.GEN, mu=5280 + rng.uniform(-5, 5), sigma=rng.uniform(12, 18), f=rng.uniform(0.1, 0.6),
                     k=rng.uniform(-0.003, -0.001)) for _ in range(32)]
    shared = [dict(inp.P2, f=rng.uniform(0.1, 0.6), k=rng.uniform(-0.003, -0.001)) for _ in range(32)]   # one shape
    for sets in (distinct, shared):
        nll, _, st = ipa.ipa_nll_eval(xd, sets, LO, HI)
        torch_.cuda.synchronize()
        assert (st.cpu().numpy() == 0).all()
        got = nll.cpu().numpy()
        ref = orc.nll(np.sort(x1), sets, LO, HI)
        assert np.all(np.abs(got - ref) <= 1e-10 * np.abs(ref))
        for i in (0, 13, 31):
            assert got[i] == ipa.ipa_nll_eval(xd, sets[i], LO, HI)[0].item()
    # above 28 sets the batch runs as two launches (shared memory): rows of the per-event output, odd split
    nll29, lp29, _ = ipa.ipa_nll_eval(xd, distinct[:29], LO, HI, want_logpdf=True)
    torch_.cuda.synchronize()
    for i in (0, 14, 15, 28):
        one, lp1, _ = ipa.ipa_nll_eval(xd, distinct[i], LO, HI, want_logpdf=True)
        assert nll29[i].item() == one.item() and bool((lp29[i] == lp1[0]).all())
    with pytest.raises(ipa.IpaError):
        ipa.ipa_nll_eval(xd, distinct + [inp.GEN], LO, HI)          # 33 sets: invalid argument


def test_nll_evaluator_matches_the_plain_calls(ipa, torch_, orc, x1):
    """NllEvaluator (the fit loop's evaluator: buffers allocated once, results read back through pinned memory) against
    ipa_nll_eval / ipa_nll_grad_eval on the same inputs: same library calls, same bits; calls in a row, a side stream."""
    xd = dev(torch_, x1)
    side = torch_.cuda.Stream()
    side.wait_stream(torch_.cuda.current_stream())
    b9, _ = inp.fd_batch(inp.GEN)
    bad = np.array(b9[:3]); bad[1, 1] = -1.0                 # a domain error: +inf, status 1
    for ev in (ipa.NllEvaluator(xd, LO, HI, policy=1), ipa.NllEvaluator(xd, LO, HI, policy=1, stream=side)):
        for th in (b9, inp.GEN, bad, b9):
            K = ipa.pack_params(th).shape[0]
            got = ev(th)
            ref, _, st = ipa.ipa_nll_eval(xd, th, LO, HI, policy=1)
            torch_.cuda.synchronize()
            assert got.shape == (K,) and np.array_equal(got, ref.cpu().numpy())
            assert np.array_equal(ev.status(K), st.cpu().numpy())
        n5, g5 = ev.gradient(b9[:5])
        rn, rg, _ = ipa.ipa_nll_grad_eval(xd, b9[:5], LO, HI, policy=1)
        torch_.cuda.synchronize()
        assert np.array_equal(n5, rn.cpu().numpy()) and np.array_equal(g5, rg.cpu().numpy())
    assert abs(got[0] - orc.nll(x1, inp.GEN, LO, HI)) <= 1e-10 * abs(got[0])


def test_core_cells(ipa, torch_, orc):
    """Cells of the core (A1e): a warp of a sorted or prepared array runs the low-degree polynomial of its cell, a warp of
    the same events in random order the full polynomial; both against the oracle, per event."""
    full = ipa.ipa_core_degree(inp.GEN, LO, HI, policy=1)
    info = ipa.ipa_core_cells(inp.GEN, LO, HI, policy=1)
    assert info[0] == 4 and all(3 <= d < 16 for d in info[1:5]) and max(info[1:5]) < full
    hb = [int(v) for v in info[5:11]]
    assert hb == sorted(hb) and info[11] == info[12] == 2 ** 31 - 1
    # boundaries sit on the edges of the coarse bins of ipa_events_prepare (bin width (HI - LO) / 256)
    edges = np.array(hb, dtype=np.int64) << 32
    xb = edges.view(np.float64)
    assert np.all(np.abs((xb - LO) * 256 / (HI - LO) - np.rint((xb - LO) * 256 / (HI - LO))) < 1e-3)
    assert ipa.ipa_core_cells(inp.GEN, LO, HI, policy=0)[0] == 0          # degree 1 (K_{1/2}): nothing to gain
    assert ipa.ipa_core_cells(dict(inp.GEN, sigma=0.02), LO, HI, policy=1)[0] == 0   # core narrower than the high-word resolution allows
    x = orc.generate_mixture(11, 300_000, inp.GEN, LO, HI)           # the oracle's own generator: no input from the CUDA path
    # the boundary doubles themselves and their neighbours
    x[:18] = np.concatenate([xb, np.nextafter(xb, 0.0), np.nextafter(xb, 1e9)])
    xs = np.sort(x)
    perm = np.random.Generator(np.random.Philox(5)).permutation(x.size)
    ref = orc.logpdf(xs, inp.GEN, LO, HI)
    for P, pol in ((inp.GEN, 1), (inp.P2, 0), (dict(inp.GEN, a=0.8, a2=3.0, beta=0.02), 1)):
        if P is not inp.GEN:
            ref = orc.logpdf(xs, P, LO, HI)
            assert ipa.ipa_core_cells(P, LO, HI, policy=pol)[0] == 4
        n1, lp_s, _ = ipa.ipa_nll_eval(dev(torch_, xs), P, LO, HI, want_logpdf=True, policy=pol)
        n2, lp_r, _ = ipa.ipa_nll_eval(dev(torch_, xs[perm]), P, LO, HI, want_logpdf=True, policy=pol)
        n3 = ipa.ipa_nll_eval(ipa.ipa_events_prepare(dev(torch_, xs[perm]), LO, HI), P, LO, HI, policy=pol)[0]
        torch_.cuda.synchronize()
        a, b = lp_s[0].cpu().numpy(), lp_r[0].cpu().numpy()
        assert np.abs(a - ref).max() <= 1e-10 and np.abs(b - ref[perm]).max() <= 1e-10
        assert np.abs(a[perm] - b).max() <= 2e-13 and (a[perm] != b).any()      # two polynomials for the same function
        tot = orc.nll(xs, P, LO, HI)
        for v in (n1, n2, n3):
            assert abs(v.item() - tot) <= 1e-10 * abs(tot)
        # analytic gradient (f1): value and derivative chains of the cell polynomials (sorted) / of the full one (shuffled)
        ref_n, ref_g = orc.nll_gradient(xs, P, LO, HI)
        for arr in (xs, xs[perm]):
            gn, gg, _ = ipa.ipa_nll_grad_eval(dev(torch_, arr), P, LO, HI, policy=pol)
            assert abs(gn.item() - ref_n) <= 1e-10 * abs(ref_n) and grad_ok(gg.cpu().numpy().reshape(-1), ref_g)


# ---------------------------------------------------------------------------------------------
# Gaussian-smeared signal shape feeding the binned path (reading F3)
# ---------------------------------------------------------------------------------------------
def test_gauss_smear_and_given_shape_binned_path(ipa, torch_, orc):
    for nbins, s0, theta in ((1000, 10.0, inp.GEN), (333, 3.3, inp.P2), (1000, 0.0, inp.GEN), (64, 40.0, inp.GEN)):
        sig = ipa.ipa_signal_shape(nbins, LO, HI, theta)
        sm = ipa.ipa_gauss_smear(sig, LO, HI, s0)
        torch_.cuda.synchronize()
        sig_ref = orc.signal_shape(nbins, LO, HI, theta)
        sm_ref = orc.gauss_smear(sig_ref, LO, HI, s0)
        assert np.abs(sig.cpu().numpy() - sig_ref).max() <= 1e-13 * sig_ref.max()
        assert np.abs(sm.cpu().numpy() - sm_ref).max() <= 1e-13 * sm_ref.max()
        # the oracle on the GPU's own input: the convolution alone
        assert np.abs(sm.cpu().numpy() - orc.gauss_smear(sig.cpu().numpy(), LO, HI, s0)).max() <= 1e-14 * sm_ref.max()
        n_obs = 1.0e6
        nu = ipa.ipa_expected_hist_shape(sm, LO, HI, 2500.0, n_obs - 2500.0, -0.002)
        nu_ref = orc.expected_hist_shape(LO, HI, sm_ref, 2500.0, n_obs - 2500.0, -0.002)
        assert np.all(np.abs(nu.cpu().numpy() - nu_ref) <= 1e-12 * nu_ref)
        counts = np.random.Generator(np.random.Philox(nbins)).poisson(nu_ref).astype(np.uint64)
        ns, nb, kk = inp.scan_grid(7, 5, n_obs=n_obs)
        got = ipa.ipa_binned_nll_scan_shape(dev(torch_, counts.astype(np.int64)), LO, HI, sm, ns, nb, kk)
        torch_.cuda.synchronize()
        ref = orc.binned_nll_scan_shape(counts, LO, HI, sm_ref, ns, nb, kk)
        assert np.all(np.abs(got.cpu().numpy() - ref) <= 1e-10 * np.abs(ref))
    # a shape with no content: flagged, not a crash
    zero = torch_.zeros(100, dtype=torch_.float64, device="cuda")
    bad = ipa.ipa_binned_nll_scan_shape(dev(torch_, np.ones(100, dtype=np.int64)), LO, HI, zero, [1.0], [10.0], [-0.002])
    assert np.isposinf(bad.cpu().numpy()).all()


# ---------------------------------------------------------------------------------------------
# extended likelihood (reading D4)
# ---------------------------------------------------------------------------------------------
def test_extended_likelihood(ipa, torch_, orc, x1):
    xd = dev(torch_, x1)
    sets = [inp.GEN, inp.P2, inp.GEN, inp.P2, inp.GEN]
    ns = np.array([3000.0, 120.5, 0.0, 9000.0, -1.0])
    nb = np.array([7000.0, 9900.0, 10000.0, 0.0, 5.0])
    nll, st = ipa.ipa_nll_eval_extended(xd, sets, ns, nb, LO, HI)
    torch_.cuda.synchronize()
    nll, st = nll.cpu().numpy(), st.cpu().numpy()
    assert list(st) == [0, 0, 0, 0, 1] and np.isposinf(nll[4])
    for i in range(4):
        ref = orc.nll_extended(x1, sets[i], ns[i], nb[i], LO, HI)
        assert abs(nll[i] - ref) <= 1e-10 * abs(ref), (i, nll[i], ref)


def test_edge_cases_of_the_next_rows(ipa, torch_, orc, x1):
    """Empty and one-element inputs of the rows added after the hot path (f1-f4)."""
    xd = dev(torch_, x1)
    nll, grad, st = ipa.ipa_nll_grad_eval(xd[:0], inp.GEN, LO, HI)                       # n = 0
    assert nll.item() == 0.0 and not np.signbit(nll.item()) and np.all(grad.cpu().numpy() == 0.0) and st.item() == 0
    nll, grad, _ = ipa.ipa_nll_grad_eval(xd[:1], inp.P2, LO, HI)                          # n = 1
    r_nll, r_g = orc.nll_gradient(x1[:1], inp.P2, LO, HI)
    assert abs(nll.item() - r_nll) <= 1e-12 * abs(r_nll) and grad_ok(grad[0].cpu().numpy(), r_g)
    e, st = ipa.ipa_nll_eval_extended(xd[:0], inp.GEN, 3.0, 4.0, LO, HI)                  # no events: -log L = ns + nb
    assert e.item() == 7.0 and st.item() == 0
    one = dev(torch_, np.array([2.0]))
    assert ipa.ipa_gauss_smear(one, LO, HI, 50.0).item() == pytest.approx(orc.gauss_smear(np.array([2.0]), LO, HI, 50.0)[0], rel=1e-14)
    q = ipa.ipa_cls_teststat(dev(torch_, np.array([5], dtype=np.int64)).to(torch_.int32), dev(torch_, np.array([6.5])),
                             dev(torch_, np.array([4.0])))
    assert abs(q.item() - orc.cls_teststat(np.array([[5]], dtype=np.uint32), [6.5], [4.0])[0]) <= 1e-12


def test_categories_with_shared_parameter_sets(ipa, torch_, orc, x1):
    """Row f4: segments (categories) mapped onto a smaller list of parameter sets."""
    off = np.array([0, 1500, 1500, 4000, 7777, 10000], dtype=np.int64)
    sets = [dict(inp.GEN), dict(inp.P2), dict(inp.GEN, f=1.5)]            # the last one is invalid
    m = np.array([1, 0, 0, 1, 2], dtype=np.int32)
    nll, st = ipa.ipa_nll_eval_categories(dev(torch_, x1), dev(torch_, off), sets, m, LO, HI)
    torch_.cuda.synchronize()
    nll, st = nll.cpu().numpy(), st.cpu().numpy()
    assert list(st) == [0, 0, 0, 0, 1] and np.isposinf(nll[4])
    ref = orc.nll_segmented(x1, off[:5], [sets[i] for i in m[:4]], LO, HI)
    assert np.all(np.abs(nll[:4] - ref) <= 1e-10 * np.abs(ref) + 0.0) and nll[1] == 0.0
    with pytest.raises(ipa.IpaError):
        ipa.ipa_nll_eval_categories(dev(torch_, x1), dev(torch_, off), sets, [0, 1, 2, 3, 0], LO, HI)   # index out of range


def test_null_stream_and_error_codes(ipa, torch_, x1):
    """cuda_stream = NULL (legacy default stream) through the raw C ABI; argument errors on a live device."""
    import ctypes as C
    L = ipa.lib()
    xd = dev(torch_, x1)
    P = ipa.pack_params(inp.GEN)
    ws = ipa.workspace(x1.size, 1)
    out = torch_.empty(1, dtype=torch_.float64, device="cuda")
    rng = ipa.binding._Range(LO, HI)
    rc = L.ipa_nll_eval(C.c_void_p(xd.data_ptr()), x1.size, P.ctypes.data_as(C.c_void_p), 1, rng, C.c_void_p(out.data_ptr()),
                        None, None, None, C.c_void_p(ws.data_ptr()), ws.numel(), None)
    assert rc == 0
    torch_.cuda.synchronize()
    ref, _, _ = ipa.ipa_nll_eval(xd, inp.GEN, LO, HI)
    assert out.item() == ref.item()
    # workspace too small / misaligned, inverted range, K = 0
    assert L.ipa_nll_eval(C.c_void_p(xd.data_ptr()), x1.size, P.ctypes.data_as(C.c_void_p), 1, rng, C.c_void_p(out.data_ptr()),
                          None, None, None, C.c_void_p(ws.data_ptr()), 16, None) == -2
    assert L.ipa_nll_eval(C.c_void_p(xd.data_ptr()), x1.size, P.ctypes.data_as(C.c_void_p), 1, rng, C.c_void_p(out.data_ptr()),
                          None, None, None, C.c_void_p(ws.data_ptr() + 8), ws.numel() - 8, None) == -2
    assert L.ipa_nll_eval(C.c_void_p(xd.data_ptr()), x1.size, P.ctypes.data_as(C.c_void_p), 1, ipa.binding._Range(HI, LO),
                          C.c_void_p(out.data_ptr()), None, None, None, C.c_void_p(ws.data_ptr()), ws.numel(), None) == -1
    assert L.ipa_nll_eval(C.c_void_p(xd.data_ptr()), x1.size, P.ctypes.data_as(C.c_void_p), 0, rng, C.c_void_p(out.data_ptr()),
                          None, None, None, C.c_void_p(ws.data_ptr()), ws.numel(), None) == -1
    assert L.ipa_strerror(-2).decode().startswith("workspace")


# ---------------------------------------------------------------------------------------------
# race evidence without a sanitizer (compute-sanitizer is closed on this GPU pool: profiles/r02_sanitizer.md):
# every kernel that stages through shared memory, takes a ticket or shares lists inside a warp is launched many
# times on the same inputs; any data race on the result path shows up as a run-to-run difference
# ---------------------------------------------------------------------------------------------
def test_repeatability_stress(ipa, torch_, x1):
    xd = dev(torch_, np.concatenate([x1] * 7)[:65_537 + 4096 * 3 + 5])          # several tiles per block, ragged tail
    batch, _ = inp.fd_batch(inp.P2)
    T = 70
    rng = np.random.Generator(np.random.Philox(5))
    off = np.concatenate([[0], np.sort(rng.integers(0, xd.numel(), size=T - 1)), [xd.numel()]]).astype(np.int64)
    od = dev(torch_, off)
    sets = inp.toy_param_sets(T, seed=11)
    seeds = inp.toy_seeds(6)

    def run():
        nll, lp, _ = ipa.ipa_nll_eval(xd, batch, LO, HI, want_logpdf=True)
        _, g, _ = ipa.ipa_nll_grad_eval(xd, [inp.GEN, inp.P2], LO, HI)
        seg, _ = ipa.ipa_nll_eval_segmented(xd, od, sets, LO, HI)
        xt, offt, _ = ipa.ipa_toy_generate(seeds, inp.P2, 3000.0, 7000.0, LO, HI, 70_000)
        xp = ipa.ipa_events_prepare(xd, LO, HI)
        xq = ipa.ipa_events_prepare(xd, LO, HI, od)
        h = ipa.ipa_hist_fill(xd, LO, HI, 1000)
        torch_.cuda.synchronize()
        return [t.clone() for t in (nll, lp, g, seg, xt[: int(offt[-1].item())], xp, xq, h)]
    first = run()
    for _ in range(30):
        for a, b in zip(first, run()):
            assert torch_.equal(a, b)


def test_no_write_outside_the_outputs(ipa, torch_, x1):
    """Bounds evidence without memcheck (profiles/r02_sanitizer.md): every output of the main calls is carved out of
    ONE arena pre-filled with a canary byte, with guard zones in between; after the calls (through the raw C ABI, exact
    sizes, ragged n) every byte outside the outputs still holds the canary and every output byte was written where the
    call promises a value."""
    import ctypes as C
    L = ipa.lib()
    CAN = 0xA5
    arena = torch_.full((1 << 22,), CAN, dtype=torch_.uint8, device="cuda")
    cursor, taken = [4096], []

    def carve(nbytes, align=256):
        start = (cursor[0] + align - 1) // align * align
        cursor[0] = start + nbytes + 512                       # 512-byte guard zone after every output
        taken.append((start, start + nbytes))
        return arena[start:start + nbytes]

    def ptr(t):
        return C.c_void_p(t.data_ptr())

    n, K, T = 4099, 2, 5
    xd = dev(torch_, x1[:n])
    P = ipa.pack_params([inp.GEN, inp.P2])
    rng = ipa.binding._Range(LO, HI)
    ws = ipa.workspace(n, 8)
    nll, lp, st = carve(8 * K), carve(8 * K * n), carve(4 * K)
    assert L.ipa_nll_eval(ptr(xd), n, P.ctypes.data_as(C.c_void_p), K, rng, ptr(nll), ptr(lp), ptr(st), None, ptr(ws),
                          ws.numel(), None) == 0
    gn, gg, gs = carve(8 * K), carve(8 * 5 * K), carve(4 * K)
    assert L.ipa_nll_grad_eval(ptr(xd), n, P.ctypes.data_as(C.c_void_p), K, rng, ptr(gn), ptr(gg), ptr(gs), None, ptr(ws),
                               ws.numel(), None) == 0
    off = dev(torch_, np.array([0, 7, 7, 1030, 4000, n], dtype=np.int64))
    PT = ipa.pack_params(inp.toy_param_sets(T, seed=3))
    sn, ss = carve(8 * T), carve(4 * T)
    assert L.ipa_nll_eval_segmented(ptr(xd), ptr(off), T, PT.ctypes.data_as(C.c_void_p), rng, ptr(sn), ptr(ss), None, ptr(ws),
                                    ws.numel(), None) == 0
    xp = carve(8 * n)
    wsp = torch_.empty(ipa.ipa_prepare_workspace_bytes(n, 0), dtype=torch_.uint8, device="cuda")
    assert L.ipa_events_prepare(ptr(xd), n, None, 0, rng, ptr(xp), ptr(wsp), wsp.numel(), None) == 0
    xq = carve(8 * n)
    assert L.ipa_events_prepare(ptr(xd), n, ptr(off), T, rng, ptr(xq), ptr(wsp), wsp.numel(), None) == 0
    hist = carve(8 * 1000)
    assert L.ipa_hist_fill(ptr(xd), n, rng, 1000, ptr(hist), None) == 0
    cap = 3001
    xg, og, ov, sg = carve(8 * cap), carve(8 * 2), carve(4), carve(4)
    seeds = np.array([9], dtype=np.uint64)
    PG = ipa.pack_params(inp.GEN)
    assert L.ipa_toy_generate(seeds.ctypes.data_as(C.c_void_p), 1, PG.ctypes.data_as(C.c_void_p), 1, C.c_double(-1.0),
                              C.c_double(-1.0), rng, cap, ptr(xg), ptr(og), ptr(ov), ptr(sg), None, ptr(ws), ws.numel(), None) == 0
    torch_.cuda.synchronize()
    host = arena.cpu().numpy()
    mask = np.ones(host.size, dtype=bool)
    for a, b in taken:
        mask[a:b] = False
    assert (host[mask] == CAN).all(), "a kernel wrote outside its output"
    # the promised outputs were all written (a double made of canary bytes is a fixed finite pattern)
    can8 = np.frombuffer(bytes([CAN] * 8), dtype=np.float64)[0]
    for t in (nll, lp, gn, gg, sn, xp, xq, xg):
        v = t.cpu().numpy().view(np.float64)
        assert not (v == can8).any()
    assert np.array_equal(np.sort(xp.cpu().numpy().view(np.float64)), np.sort(x1[:n]))
    assert int(hist.cpu().numpy().view(np.uint64).sum()) == n


def test_host_buffer_path_in_pieces(ipa, torch_, orc):
    """nll_host (the e2e leg of bench.py): the events travel in pieces on a copy stream while the pieces already on the device
    are evaluated; the sum of the pieces equals the single call up to rounding and the oracle within tolerance."""
    n = 5_000_001
    x = inp.standin_masses(23, n)
    xh = torch_.from_numpy(x).pin_memory()
    batch = [inp.GEN, inp.P2]
    got = ipa.nll_host(xh, batch, LO, HI).numpy()
    one = ipa.nll_host(xh, batch, LO, HI, chunks=1).numpy()
    assert np.all(np.abs(got - one) <= 1e-12 * np.abs(one))
    ref = orc.nll(x, batch, LO, HI, nthreads=8)
    assert np.all(np.abs(got - ref) <= 1e-10 * np.abs(ref))
    assert np.array_equal(got, ipa.nll_host(xh, batch, LO, HI).numpy())          # run to run
