"""Pins of the oracle's CLs functions (reading F2).  The paper prints no
CLs number and no formula for its statistic, so the pins are the definition evaluated in
mpmath, the linearity of q in the counts, its Poisson expectation, and the one-bin case where CL_sb is a
Poisson cumulative probability (scipy)."""
import mpmath as mp
import numpy as np
import scipy.stats

import ipa_inputs as inp

LO, HI = inp.LO, inp.HI


def test_teststat_definition_mpmath(orc):
    mp.mp.dps = 40
    nu_b = np.array([3.5, 120.25, 0.7, 45.0, 9e4])
    nu_sb = nu_b + np.array([0.2, 30.0, 1.9, 0.0, 210.0])
    counts = np.array([[3, 130, 0, 44, 90211], [0, 0, 0, 0, 0], [9, 99, 4, 61, 89000]], dtype=np.uint32)
    got = orc.cls_teststat(counts, nu_sb, nu_b)
    for t in range(counts.shape[0]):
        ref = 2 * sum((mp.mpf(float(a)) - mp.mpf(float(b))) - int(n) * mp.log(mp.mpf(float(a)) / mp.mpf(float(b)))
                      for a, b, n in zip(nu_sb, nu_b, counts[t]))
        assert abs(got[t] - float(ref)) <= 1e-13 * max(1.0, abs(float(ref)))
    assert np.array_equal(got, orc.cls_teststat(counts.astype(np.uint64), nu_sb, nu_b))   # both count widths
    # zero counts: q = 2 (sum nu_sb - sum nu_b); equal hypotheses: q = 0
    assert abs(got[1] - 2 * (nu_sb.sum() - nu_b.sum())) < 1e-10
    assert np.all(orc.cls_teststat(counts, nu_b, nu_b) == 0.0)


def test_teststat_is_affine_in_the_counts(orc):
    rng = np.random.Generator(np.random.Philox(3))
    nu_b = rng.uniform(5, 500, 40)
    nu_sb = nu_b * rng.uniform(1.0, 1.3, 40)
    n1 = rng.poisson(nu_b).astype(np.uint32)
    n2 = rng.poisson(nu_sb).astype(np.uint32)
    q0, q1, q2, q12 = orc.cls_teststat(np.array([0 * n1, n1, n2, n1 + n2]), nu_sb, nu_b)
    assert abs((q12 - q0) - ((q1 - q0) + (q2 - q0))) <= 1e-11 * abs(q0)


def test_expectation_and_one_bin_poisson_cdf(orc):
    # expected histograms of the config-5 model (1000 bins), toys from the oracle's own Poisson sampler
    nb_tot, ns = 1.0e6, 400.0
    nu_b = orc.expected_hist(1000, LO, HI, inp.GEN, 0.0, nb_tot, -0.002)
    nu_sb = orc.expected_hist(1000, LO, HI, inp.GEN, ns, nb_tot, -0.002)
    seeds = np.arange(1, 2001, dtype=np.uint64)
    for truth in (nu_b, nu_sb):
        q = orc.cls_teststat(orc.poisson_hist_toys(truth, seeds), nu_sb, nu_b)
        lr = np.log(nu_sb / nu_b)
        mean = 2 * ((nu_sb - nu_b).sum() - (truth * lr).sum())
        sd = 2 * np.sqrt((truth * lr * lr).sum())
        assert abs(q.mean() - mean) < 5 * sd / np.sqrt(q.size)
        assert abs(q.std() / sd - 1) < 0.1
    # one bin: q decreases with n, so {q >= q_obs} = {n <= n_obs} and CL_sb is the Poisson CDF at n_obs
    vb, vsb, n_obs = np.array([50.0]), np.array([62.0]), np.uint32(55)
    seeds = np.arange(1, 40001, dtype=np.uint64)
    q_obs = orc.cls_teststat(np.array([[n_obs]], dtype=np.uint32), vsb, vb)[0]
    out = []
    for truth in (vsb, vb):
        toys = orc.poisson_hist_toys(truth, seeds)
        q = orc.cls_teststat(toys, vsb, vb)
        c = orc.cls_count_ge(q, q_obs)
        assert c == int((toys[:, 0] <= n_obs).sum())                      # exact: same event
        p = scipy.stats.poisson.cdf(int(n_obs), truth[0])
        assert abs(c / seeds.size - p) < 5 * np.sqrt(p * (1 - p) / seeds.size)
        out.append(c)
    cl = orc.cls_from_counts(out[0], seeds.size, out[1], seeds.size)
    assert cl[0] == out[0] / seeds.size and cl[1] == out[1] / seeds.size and cl[2] == cl[0] / cl[1]
    assert np.isnan(orc.cls_from_counts(0, 10, 0, 10)[2])
