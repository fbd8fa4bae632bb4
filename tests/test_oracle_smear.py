"""Pins of the oracle's Gaussian smearing and given-shape binned path (reading F3).
The paper shows only the call, so the pins are: numpy's convolution on the same kernel
(a library routine for the special case of a full-support linear convolution), the delta response, the
closed form Gaussian * Gaussian = Gaussian of the summed variances, conservation of the content, and the
reduction of the given-shape functions to the built-in-shape ones."""
import numpy as np

import ipa_inputs as inp

LO, HI = inp.LO, inp.HI


def kernel(nbins, sigma0):
    w = (HI - LO) / nbins
    M = int(np.ceil(8 * sigma0 / w))
    m = np.arange(-M, M + 1)
    g = np.exp(-(m * w) ** 2 / (2 * sigma0 ** 2))
    return g / g.sum(), M


def test_smear_equals_numpy_convolution_and_delta_response(orc):
    rng = np.random.Generator(np.random.Philox(4))
    nbins, s0 = 300, 7.5
    sig = rng.uniform(0, 1, nbins)
    g, M = kernel(nbins, s0)
    ref = np.convolve(sig, g, mode="full")[M:M + nbins]
    got = orc.gauss_smear(sig, LO, HI, s0)
    assert np.abs(got - ref).max() <= 1e-14
    delta = np.zeros(nbins)
    delta[140] = 2.5
    out = orc.gauss_smear(delta, LO, HI, s0)
    assert np.abs(out[140 - M:140 + M + 1] - 2.5 * g).max() <= 1e-16 and out[:140 - M].sum() == 0.0
    assert abs(out.sum() - 2.5) <= 1e-14                              # content conserved away from the edges
    assert np.array_equal(orc.gauss_smear(sig, LO, HI, 0.0), sig)     # sigma0 = 0: identity


def test_gaussian_smeared_by_gaussian_is_the_gaussian_of_summed_variances(orc):
    nbins, s1, s0 = 1200, 9.0, 12.0
    w = (HI - LO) / nbins
    c = LO + (np.arange(nbins) + 0.5) * w
    g1 = np.exp(-(c - 5300.0) ** 2 / (2 * s1 ** 2))
    out = orc.gauss_smear(g1, LO, HI, s0)
    st = np.hypot(s1, s0)
    ref = (s1 / st) * np.exp(-(c - 5300.0) ** 2 / (2 * st ** 2))      # continuous result; the grid error is ~exp(-2 pi^2 s^2/w^2)
    assert np.abs(out - ref).max() <= 1e-12


def test_given_shape_functions_reduce_to_the_builtin_shape(orc):
    nbins = 1000
    sig = orc.signal_shape(nbins, LO, HI, inp.GEN)
    nu = orc.expected_hist_shape(LO, HI, sig, 2500.0, 1e6, -0.002)
    assert np.abs(nu / orc.expected_hist(nbins, LO, HI, inp.GEN, 2500.0, 1e6, -0.002) - 1).max() <= 1e-15
    counts = np.random.Generator(np.random.Philox(6)).poisson(nu).astype(np.uint64)
    ns, nb, kk = inp.scan_grid(5, 4, n_obs=1e6 + 2500)
    a = orc.binned_nll_scan_shape(counts, LO, HI, sig, ns, nb, kk)
    b = orc.binned_nll_scan(counts, LO, HI, inp.GEN, ns, nb, kk)
    assert np.all(np.abs(a - b) <= 1e-14 * np.abs(b))
    # the smeared Ipatia is wider: variance grows by sigma0^2 (tails truncated by the range: loose bound)
    sm = orc.gauss_smear(sig, LO, HI, 10.0)
    c = LO + (np.arange(nbins) + 0.5) * (HI - LO) / nbins
    var = lambda s: (s * (c - 5280.0) ** 2).sum() / s.sum()
    assert abs((var(sm) - var(sig)) / 100.0 - 1.0) < 0.05
