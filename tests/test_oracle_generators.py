"""Pins of the oracle's generators and binned path (rows T0, T1, B1-B3; readings D13-D16).

Philox is pinned against the CUDA toolkit's own header implementation compiled for the host
(library routine, different code); the samplers are pinned by exact distributional facts.
"""
import math
import os
import shutil
import subprocess

import numpy as np
import pytest

import ipa_inputs as inp

LO, HI = inp.LO, inp.HI
P1, P2 = inp.GEN, inp.P2
HERE = os.path.dirname(os.path.abspath(__file__))


def test_philox_vs_cuda_toolkit_header(orc, tmp_path):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("no nvcc")
    exe = str(tmp_path / "philox_host")
    subprocess.check_call([nvcc, "-Wno-deprecated-gpu-targets", "-o", exe, os.path.join(HERE, "philox_curand_host.cu")])
    rng = np.random.default_rng(77)
    cases = rng.integers(0, 2 ** 32, size=(256, 6), dtype=np.uint64)
    cases[0] = 0
    cases[1] = 2 ** 32 - 1
    cases[2] = [1, 0, 0, 0, 0, 0]
    cases[3] = [0, 0, 1, 0, 0, 0]
    out = subprocess.run([exe], input="\n".join(" ".join(str(int(v)) for v in c) for c in cases), text=True,
                         capture_output=True, check=True).stdout.split("\n")
    for c, line in zip(cases, out):
        ref = np.array([int(v) for v in line.split()], dtype=np.uint32)
        got = orc.philox4x32_10(c[:2], c[2:])
        assert (got == ref).all(), (c, got, ref)


def test_uniform_mapping(orc):
    """u = ((w0>>5) 2^26 + (w1>>6) + 0.5) 2^-53 in (0,1) (reading D13), checked from the raw words."""
    for seed, slot, att, stream in [(1, 0, 0, 0), (2 ** 40 + 5, 2 ** 33 + 1, 7, 2), (99, 12345, 3, 1)]:
        w = orc.philox4x32_10([seed & 0xFFFFFFFF, seed >> 32], [slot & 0xFFFFFFFF, slot >> 32, att, stream]).astype(np.uint64)
        u = orc.uniforms2(seed, slot, att, stream)
        for j in (0, 1):
            ref = ((int(w[2 * j]) >> 5) * 2 ** 26 + (int(w[2 * j + 1]) >> 6) + 0.5) / 2 ** 53
            assert u[j] == ref and 0.0 < u[j] < 1.0
    us = np.array([orc.uniforms2(5, i, 0, 0) for i in range(20000)]).ravel()
    assert abs(us.mean() - 0.5) < 4 / math.sqrt(12 * us.size) and abs(us.var() - 1 / 12) < 2e-3


def test_poisson_moments(orc):
    """mean / variance / skewness at means {0.5, 5, 50, 3e4, 1e5} (C8.12)."""
    for mean, n in ((0.5, 40000), (5.0, 40000), (50.0, 40000), (3e4, 40000), (1e5, 40000)):
        k = np.array([orc.poisson(1234, i, 3, mean) for i in range(n)], dtype=np.float64)
        se = math.sqrt(mean / n)
        assert abs(k.mean() - mean) < 4.5 * se, (mean, k.mean())
        assert abs(k.var() - mean) < 5 * mean * math.sqrt(2.0 / n + 1.0 / (mean * n)), (mean, k.var())
        skew = ((k - k.mean()) ** 3).mean() / k.std() ** 3
        assert abs(skew - 1 / math.sqrt(mean)) < 5 * math.sqrt(6.0 / n) + 0.02, (mean, skew)
    assert orc.poisson(1, 0, 3, 0.0) == 0


def test_poisson_small_mean_exact_pmf(orc):
    n = 60000
    k = np.array([orc.poisson(42, i, 4, 3.2) for i in range(n)])
    for j in range(9):
        p = math.exp(-3.2) * 3.2 ** j / math.factorial(j)
        assert abs((k == j).mean() - p) < 5 * math.sqrt(p * (1 - p) / n)


def _chi2_vs_pdf(orc, x, p, nb=200):
    edges = np.linspace(LO, HI, nb + 1)
    obs, _ = np.histogram(x, edges)
    # expected from the oracle's own normalised mixture pdf, Simpson within each bin
    def pdf(t):
        return np.exp(orc.logpdf(t, p, LO, HI))
    a, b = edges[:-1], edges[1:]
    m = 0.5 * (a + b)
    exp = x.size * (b - a) / 6 * (pdf(a) + 4 * pdf(m) + pdf(b))
    return float(((obs - exp) ** 2 / exp).sum()), nb


def test_mixture_generator_chi2(orc):
    """chi^2 of generated events against f S + (1-f) B in 200 bins (C8.12)."""
    for seed, p in ((1, P1), (7, P2)):
        x = orc.generate_mixture(seed, 60000, p, LO, HI)
        assert x.min() >= LO and x.max() <= HI
        chi2, nb = _chi2_vs_pdf(orc, x, p)
        assert chi2 < nb + 5 * math.sqrt(2 * nb), chi2
        # deterministic and prefix-stable: slot i does not depend on n
        assert (orc.generate_mixture(seed, 100, p, LO, HI) == x[:100]).all()
    assert abs((np.abs(orc.generate_mixture(1, 60000, P1, LO, HI) - 5280) <= 30).mean() - 0.34443) < 0.01


def test_toy_generator_structure(orc):
    seeds = inp.toy_seeds(6)
    x, off = orc.toy_generate(seeds, P1, 300.0, 700.0, LO, HI)
    assert off[0] == 0 and (np.diff(off) > 0).all() and off[-1] == x.size
    for t, s in enumerate(seeds):
        ns, nb = orc.poisson(int(s), 0, 3, 300.0), orc.poisson(int(s), 1, 3, 700.0)
        assert off[t + 1] - off[t] == ns + nb
        seg = x[off[t]:off[t + 1]]
        # signal block first: concentrated around mu; background block: spread over the range
        assert (np.abs(seg[:ns] - 5280) < 30).mean() > 0.8
        assert (np.abs(seg[ns:] - 5280) < 30).mean() < 0.2
    _, off2 = orc.toy_generate(seeds, P1, 300.0, 700.0, LO, HI, offsets_only=True)
    assert (off2 == off).all()
    # a per-toy parameter array gives the same events as the single set when all rows are equal
    x3, off3 = orc.toy_generate(seeds, [P1] * 6, 300.0, 700.0, LO, HI)
    assert (off3 == off).all() and (x3 == x).all()


def test_background_inverse_cdf_ks(orc):
    sp = pytest.importorskip("scipy.stats")
    x = orc.generate_mixture(11, 20000, dict(P1, f=0.0), LO, HI)
    k = P1["k"]
    cdf = lambda t: np.expm1(k * (t - LO)) / math.expm1(k * (HI - LO))
    assert sp.kstest(x, cdf).pvalue > 1e-3


def test_hist_fill_exact(orc):
    rng = np.random.default_rng(2)
    x = np.concatenate([rng.uniform(LO, HI, 50000), [LO, HI, LO - 1, HI + 1, 5000.6, 5599.4]])
    c = orc.hist_fill(x, LO, HI, 1000)
    ref, _ = np.histogram(x[(x >= LO) & (x <= HI)], bins=1000, range=(LO, HI))
    assert c.sum() == 50004 and c.dtype == np.uint64
    # numpy's binning differs only in how it treats edges that are not representable; compare exactly
    # against the stated rule instead: bin = floor((x-lo)*nbins/(hi-lo)), x==hi -> last bin
    b = np.floor((x - LO) * (1000 / (HI - LO))).astype(np.int64)
    keep = (x >= LO) & (x <= HI)
    b = np.minimum(b[keep], 999)
    assert (np.bincount(b, minlength=1000) == c.astype(np.int64)).all()
    assert np.abs(ref - c.astype(np.int64)).sum() <= 4


def test_binned_nll_definition(orc):
    """B2 (reading D15) against a direct numpy evaluation built from orc.log_I only."""
    nb_ = 50
    rng = np.random.default_rng(4)
    counts = rng.poisson(200, nb_).astype(np.uint64)
    counts[3] = 0
    ns, nb, kk = np.array([0.0, 120.0, 500.0]), np.array([10000.0, 9880.0, 9500.0]), np.array([-0.002, -0.0021, 0.0])
    got = orc.binned_nll_scan(counts, LO, HI, P1, ns, nb, kk)
    c = LO + (np.arange(nb_) + 0.5) * (HI - LO) / nb_
    s = np.exp([orc.log_I(P1, float(t) - P1["mu"]) for t in c]); s /= s.sum()
    for q in range(3):
        b = np.exp(kk[q] * c); b /= b.sum()
        nu = ns[q] * s + nb[q] * b
        n = counts.astype(np.float64)
        ref = float(math.fsum(nu - np.where(n > 0, n * np.log(nu), 0.0)))
        assert abs(got[q] - ref) <= 1e-12 * abs(ref)
        e = orc.expected_hist(nb_, LO, HI, P1, ns[q], nb[q], kk[q])
        assert np.allclose(e, nu, rtol=1e-13, atol=0) and abs(e.sum() - (ns[q] + nb[q])) <= 1e-9


def test_binned_scan_minimum_near_truth(orc):
    """Scan minimum near the generating (ns, k) (C8.12), small version of config 5."""
    nbins, N, nsig = 200, 200000, 2500
    x = np.concatenate([orc.generate_mixture(5, nsig, dict(P1, f=1.0), LO, HI),
                        orc.generate_mixture(6, N - nsig, dict(P1, f=0.0), LO, HI)])
    counts = orc.hist_fill(x, LO, HI, nbins)
    NS, NB, KK = inp.scan_grid(21, 21, n_obs=float(N))
    nll = orc.binned_nll_scan(counts, LO, HI, P1, NS, NB, KK)
    q = int(np.argmin(nll))
    assert abs(NS[q] - nsig) <= 750 and abs(KK[q] + 0.002) <= 1.01e-4


def test_poisson_hist_toys(orc):
    mean = np.array([0.0, 0.7, 8.0, 120.0, 1e5])
    t = orc.poisson_hist_toys(mean, np.arange(1, 3001, dtype=np.uint64))
    assert t.shape == (3000, 5) and t.dtype == np.uint32 and (t[:, 0] == 0).all()
    for b in range(1, 5):
        col = t[:, b].astype(np.float64)
        assert abs(col.mean() - mean[b]) < 4.5 * math.sqrt(mean[b] / 3000)
        assert abs(col.var() / mean[b] - 1) < 0.15
    # element (t, b) depends only on (seed_t, b, mean_b)
    assert orc.poisson(7, 3, 4, 120.0) == t[6, 3]


# ---------------------------------------------------------------------------------------------
# PTRS branch of the Poisson sampler (mean >= 10: the branch configs 4 and 5 use).  Pins:
#  (i)   exact probability function: chi^2 of 2e6 draws against scipy.stats.poisson.pmf (bins pooled to
#        an expectation >= 20);
#  (ii)  a theorem of rejection sampling: with k = floor(G(U)), G'(U) = a/us^2 + b and the acceptance test
#        V <= p(k) G'(U) / inv_alpha, the acceptance probability per attempt is EXACTLY 1/inv_alpha as long as
#        the hat dominates p everywhere AND the two squeeze steps never change the decision of the full test.
#        So the mean number of attempts must equal inv_alpha; a squeeze constant that accepts (or rejects)
#        what the full comparison would not shows up here long before it distorts the distribution;
#  (iii) the quick acceptance (us >= 0.07 and V <= v_r) is taken with probability (1 - 2*0.07) v_r per attempt
#        (U and V independent uniforms).
# test_ptrs_pins_detect_wrong_constants shows that each single mistyped constant fails (i) or (ii).
# ---------------------------------------------------------------------------------------------
def _pooled_chi2(k, mean, n):
    sp = pytest.importorskip("scipy.stats")
    lo_k = int(max(0, math.floor(mean - 12 * math.sqrt(mean)) - 5))
    hi_k = int(math.ceil(mean + 12 * math.sqrt(mean)) + 5)
    ks = np.arange(lo_k, hi_k + 1)
    exp = n * sp.poisson.pmf(ks, mean)
    obs = np.bincount(np.clip(k, lo_k, hi_k) - lo_k, minlength=ks.size).astype(np.float64)
    assert k.min() >= 0 and (k < lo_k).sum() + (k > hi_k).sum() == 0      # 12 sigma: nothing outside
    # pool from both ends towards the mode until every bin expects >= 20
    o, e, acc_o, acc_e = [], [], 0.0, 0.0
    for oi, ei in zip(obs, exp):
        acc_o += oi
        acc_e += ei
        if acc_e >= 20.0:
            o.append(acc_o); e.append(acc_e); acc_o = acc_e = 0.0
    o[-1] += acc_o
    e[-1] += acc_e
    o, e = np.array(o), np.array(e)
    return float(((o - e) ** 2 / e).sum()), o.size - 1


def _ptrs_constants(mean):
    b = 0.931 + 2.53 * math.sqrt(mean)
    return b, 1.1239 + 1.1328 / (b - 3.4), 0.9277 - 3.6224 / (b - 2.0)


@pytest.mark.parametrize("mean", [10.0, 37.5, 1.0e3, 3.0e4, 7.0e4, 1.0e5])
def test_poisson_ptrs_exact_pmf_and_acceptance(orc, mean):
    n = 2_000_000
    k, attempts, exit_ = orc.poisson_array(4242, 0, n, 3, mean, diagnostics=True)
    assert np.array_equal(k[:200], [orc.poisson(4242, i, 3, mean) for i in range(200)])       # same draws as the scalar call
    chi2, dof = _pooled_chi2(k, mean, n)
    assert chi2 < dof + 4.5 * math.sqrt(2 * dof), (mean, chi2, dof)
    b, inv_alpha, vr = _ptrs_constants(mean)
    p = 1.0 / inv_alpha
    se = math.sqrt((1 - p) / p ** 2 / n)                       # geometric number of attempts
    assert abs(attempts.mean() - inv_alpha) < 4.5 * se, (mean, attempts.mean(), inv_alpha)
    pf = 0.86 * vr
    quick_first = ((attempts == 1) & (exit_ == 1)).mean()
    assert abs(quick_first - pf) < 4.5 * math.sqrt(pf * (1 - pf) / n), (mean, quick_first, pf)


def _ptrs_numpy(mean, n, rng, c):
    """Hoermann's transformed rejection with squeeze, vectorised, with every constant taken from `c` -- only used to
    show that the pins above have the power to see a single wrong constant (it is not the oracle)."""
    sp = pytest.importorskip("scipy.special")
    smu = math.sqrt(mean)
    b = c["b0"] + c["b1"] * smu
    a = c["a0"] + c["a1"] * b
    inv_alpha = c["ia0"] + c["ia1"] / (b - c["ia2"])
    vr = c["vr0"] - c["vr1"] / (b - c["vr2"])
    out = np.full(n, -1, dtype=np.int64)
    attempts = np.zeros(n, dtype=np.int64)
    todo = np.arange(n)
    while todo.size:
        U = rng.random(todo.size) - 0.5
        V = rng.random(todo.size)
        attempts[todo] += 1
        us = 0.5 - np.abs(U)
        kf = np.floor((2.0 * a / us + b) * U + mean + c["shift"])
        quick = (us >= c["s0"]) & (V <= vr)
        rej = ~quick & ((kf < 0) | ((us < c["s1"]) & (V > us)))
        full = ~quick & ~rej
        ok = np.zeros(todo.size, dtype=bool)
        kk = np.where(full, kf, 1.0)
        ok[full] = (np.log(V[full]) + math.log(inv_alpha) - np.log(a / (us[full] ** 2) + b)
                    <= -mean + kk[full] * math.log(mean) - sp.gammaln(kk[full] + 1.0))
        acc = quick | ok
        out[todo[acc]] = kf[acc].astype(np.int64)
        todo = todo[~acc]
    return out, attempts, inv_alpha


PTRS_PUBLISHED = dict(b0=0.931, b1=2.53, a0=-0.059, a1=0.02483, ia0=1.1239, ia1=1.1328, ia2=3.4, vr0=0.9277, vr1=3.6224,
                      vr2=2.0, shift=0.43, s0=0.07, s1=0.013)


def test_ptrs_pins_detect_wrong_constants():
    """Power of pins (i) and (ii): the published constants pass; a single mistyped constant that breaks the sampler
    (a squeeze step that overrides the full comparison, or a hat that no longer dominates) fails one of them at
    mean 1e3 or 3e4.  The full comparison V <= p(k) G'(U) / inv_alpha is exact for whatever k is proposed, so
    constants that only move the hat inside its slack (e.g. the 0.43 shift, the 3.4 and 2.0 offsets) change the
    efficiency, not the distribution: the pins rightly stay green for those, and they are not listed."""
    n = 2_000_000

    def verdict(c, mean, seed):
        k, att, inv_alpha = _ptrs_numpy(mean, n, np.random.Generator(np.random.Philox(seed)), c)
        chi2, dof = _pooled_chi2(k, mean, n) if (k.min() >= 0 and abs(k.mean() - mean) < 5) else (1e30, 1)
        p = 1.0 / inv_alpha
        se = math.sqrt((1 - p) / p ** 2 / n)
        return chi2 < dof + 4.5 * math.sqrt(2 * dof) and abs(att.mean() - inv_alpha) < 4.5 * se
    for mean in (1.0e3, 3.0e4):
        assert verdict(PTRS_PUBLISHED, mean, 1)
    mutations = dict(vr0=0.9727, s0=0.04, s1=0.031, b1=2.35, a1=0.02843, ia0=1.0239, b0=9.31, vr1=0.36224)
    for j, (name, wrong) in enumerate(mutations.items()):
        c = dict(PTRS_PUBLISHED, **{name: wrong})
        assert not (verdict(c, 1.0e3, 100 + j) and verdict(c, 3.0e4, 200 + j)), (name, wrong)


# ---- signal draws under the piecewise envelope (reading D13 as revised in round 2) ---------------------------------
ENV_CASES = {
    "config": P1,
    "beta_nonzero": P2,
    "beta_large": dict(P2, beta=0.05),
    "mode_left_of_range": dict(P1, mu=4998.0, sigma=3.0),          # the advisor's case: maximum at the range end
    "mode_left_of_range_b": dict(P1, mu=4995.0, sigma=5.0, beta=-0.02),
    "range_inside_left_tail": dict(P1, mu=5700.0, n=1.0),
    "range_inside_right_tail": dict(P2, mu=4900.0),
    "student_t": inp.T1,
    "student_t_beta": inp.T2,
    "n_equal_one": dict(P1, n=1.0, n2=1.0),
}


def _signal_cdf(orc, p, grid):
    """CDF of S on `grid` by composite Simpson (16 sub-intervals per cell) of the oracle's normalised signal density
    (exp of logpdf at f = 1); the joins and the mode are grid points, so every cell is smooth."""
    a, b = grid[:-1], grid[1:]
    t = a[:, None] + (b - a)[:, None] * np.linspace(0.0, 1.0, 17)[None, :]
    f = np.exp(orc.logpdf(t.ravel(), dict(p, f=1.0), LO, HI)).reshape(t.shape)
    cell = (b - a) / 48 * (f[:, 0] + f[:, -1] + 4 * f[:, 1:-1:2].sum(axis=1) + 2 * f[:, 2:-1:2].sum(axis=1))
    return np.concatenate([[0.0], np.cumsum(cell)])


@pytest.mark.parametrize("case", sorted(ENV_CASES))
def test_signal_draws_follow_the_density(orc, case):
    """chi^2 (100 equal-probability bins) and KS of the signal draws against the integral of the oracle's S, which is
    pinned on its own (test_oracle_ipatia / test_oracle_studentt): independent of how the draws are made.  Covers
    beta != 0, the mode outside the range, ranges inside one tail, n = 1 and the Student-t core."""
    sp = pytest.importorskip("scipy.stats")
    p = ENV_CASES[case]
    n = 40000
    x, attempts, violated, inv_acc, worst = orc.generate_signal_diag(123, n, p, LO, HI)
    assert x.min() >= LO and x.max() <= HI and not violated
    assert worst <= 0.0                                   # the envelope bounds the core everywhere on a dense grid
    special = [p["mu"] + d for d in (-p["a"] * p["sigma"], 0.0, p["a2"] * p["sigma"]) if LO < p["mu"] + d < HI]
    grid = np.unique(np.concatenate([np.linspace(LO, HI, 24001), special]))   # 0.025 steps: the CDF is interpolated linearly
    cdf = _signal_cdf(orc, p, grid)
    assert abs(cdf[-1] - 1.0) <= 1e-9
    u = np.interp(x, grid, cdf)                           # probability integral transform: uniform if x ~ S
    assert sp.kstest(u, "uniform").pvalue > 1e-3
    obs, _ = np.histogram(u, bins=100, range=(0.0, 1.0))
    chi2 = float(((obs - n / 100) ** 2 / (n / 100)).sum())
    assert chi2 < 99 + 5 * math.sqrt(2 * 99), chi2
    # acceptance theorem: attempts per event = envelope weight / N_S (mean of a geometric law), here 1 .. 1.4
    assert 1.0 <= inv_acc <= 1.4
    assert abs(attempts - inv_acc) <= 5 * math.sqrt(inv_acc * (inv_acc - 1) / n) + 1e-3, (attempts, inv_acc)


def test_signal_draws_are_slot_addressed(orc):
    """A draw depends on (seed, slot) only: prefix-stable and equal inside the mixture and the toy generators."""
    a = orc.generate_signal_diag(9, 500, P1, LO, HI)[0]
    b = orc.generate_signal_diag(9, 2000, P1, LO, HI)[0]
    assert (a == b[:500]).all()
    m = orc.generate_mixture(9, 2000, dict(P1, f=1.0), LO, HI)
    assert (m == b).all()
