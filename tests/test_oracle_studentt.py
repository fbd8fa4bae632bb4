"""Pins of the oracle's zeta = 0 Student-t core (reading D3; PAPER.md:226-236
`Free('lb', -2.0, ...)` without zeta, ref. [10] at PAPER.md:450):

    G(d) = (d^2 + delta^2)^{lambda - 1/2} e^{beta d},  lambda < 0,
    delta = sigma sqrt(-2 lambda - 2) for lambda < -1, delta = sigma for -1 <= lambda < 0.

Everything the oracle is compared with here is built from mpmath / scipy primitives only: the zeta -> 0 limit of the
Bessel core of reading C1 (mpmath besselk), mpmath quadrature, the Gamma-function closed form of the integral,
scipy's Student-t density.
"""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import stats

import ipa_inputs as inp

mp.mp.dps = 30
LO, HI = inp.LO, inp.HI
T1 = inp.T1          # lambda = -2 (the Upsilon example's value), beta = 0
T2 = inp.T2          # lambda = -0.7 (delta = sigma branch), beta != 0, asymmetric tails


class MPStudent:
    """mpmath restatement of the definition with the Student-t core."""

    def __init__(self, p, lo=LO, hi=HI):
        g = lambda name: mp.mpf(p[name])
        self.mu, self.sigma, self.lam, self.beta = g("mu"), g("sigma"), g("lambda"), g("beta")
        self.a, self.n, self.a2, self.n2, self.f, self.k = g("a"), g("n"), g("a2"), g("n2"), g("f"), g("k")
        self.lo, self.hi = mp.mpf(lo), mp.mpf(hi)
        self.delta = self.sigma * mp.sqrt(-2 * self.lam - 2) if self.lam < -1 else self.sigma
        self.d0, self.d1 = -self.a * self.sigma, self.a2 * self.sigma
        self.G0, self.G1 = self.G(self.d0), self.G(self.d1)
        self.L0 = mp.diff(lambda d: mp.log(self.G(d)), self.d0)
        self.L1 = mp.diff(lambda d: mp.log(self.G(d)), self.d1)
        pts = sorted({self.lo, self.hi, *[self.mu + d for d in (self.d0, 0, self.d1) if self.lo < self.mu + d < self.hi]})
        self.NS = mp.quad(lambda x: self.I(x - self.mu), pts)
        self.NB = (mp.exp(self.k * (self.hi - self.lo)) - 1) / self.k

    def G(self, d):
        return (d * d + self.delta ** 2) ** (self.lam - mp.mpf(1) / 2) * mp.exp(self.beta * d)

    def I(self, d):
        if d < self.d0:
            return self.G0 * (1 - (d - self.d0) * self.L0 / self.n) ** (-self.n)
        if d > self.d1:
            return self.G1 * (1 - (d - self.d1) * self.L1 / self.n2) ** (-self.n2)
        return self.G(d)

    def l(self, x):
        x = mp.mpf(x)
        return mp.log(self.f * self.I(x - self.mu) / self.NS + (1 - self.f) * mp.exp(self.k * (x - self.lo)) / self.NB)


def test_limit_of_the_bessel_core(orc):
    """(i) zeta -> 0 of reading C1's core, computed with mpmath's besselk (not the oracle's): delta(zeta) ->
    sigma sqrt(-2 lambda - 2) and log G(d) - log G(0) -> the Student-t form, with an error that shrinks with zeta."""
    lam, sigma, beta = mp.mpf(-2), mp.mpf(15), mp.mpf("0.004")
    p = dict(T1, beta=float(beta))
    nu = lam - mp.mpf(1) / 2
    prev = None
    for zeta in (mp.mpf("1e-3"), mp.mpf("1e-4"), mp.mpf("1e-5"), mp.mpf("1e-6")):
        Kl, Kl1 = mp.besselk(lam, zeta), mp.besselk(lam + 1, zeta)
        delta = sigma * mp.sqrt(zeta * Kl / Kl1)
        alpha = mp.sqrt(zeta * Kl1 / Kl) / sigma
        G = lambda d: mp.sqrt(d * d + delta ** 2) ** nu * mp.exp(beta * d) * mp.besselk(nu, alpha * mp.sqrt(d * d + delta ** 2))
        st, c = orc.shape_consts(p)
        assert st == 0
        err = abs(delta - mp.mpf(c["delta"])) / delta
        for d in (-40.0, -7.5, 3.0, 22.0, 60.0):
            ref = mp.log(G(mp.mpf(d))) - mp.log(G(mp.mpf(0)))
            got = mp.mpf(orc.core_logG(p, d)) - mp.mpf(orc.core_logG(p, 0.0))
            err = max(err, abs(got - ref))
        assert err <= 20 * zeta ** 2 + 1e-14, (zeta, err)        # the correction is O(zeta^2)
        if prev is not None and prev > 1e-12:
            assert err < prev / 50
        prev = err
    # the same limit through the oracle's OWN Bessel core at a small zeta
    small = dict(p, zeta=1e-4)
    for d in (-30.0, 12.0, 45.0):
        a = orc.core_logG(small, d) - orc.core_logG(small, 0.0)
        b = orc.core_logG(p, d) - orc.core_logG(p, 0.0)
        assert abs(a - b) <= 1e-6
        assert abs(orc.core_logderiv(small, d) - orc.core_logderiv(p, d)) <= 1e-7


def test_scipy_student_t_density(orc):
    """beta = 0, joins far outside the range: S(x) is the truncated Student-t density with -2 lambda degrees of
    freedom and scale delta / sqrt(-2 lambda) (a library routine)."""
    for lam in (-2.0, -0.7, -1.0, -5.5):
        p = dict(T1, **{"lambda": lam}, a=60.0, a2=60.0)
        df = -2.0 * lam
        delta = p["sigma"] * math.sqrt(-2 * lam - 2) if lam < -1 else p["sigma"]
        s = delta / math.sqrt(df)
        dist = stats.t(df, loc=p["mu"], scale=s)
        mass = dist.cdf(HI) - dist.cdf(LO)
        for x in (5003.0, 5200.0, 5271.25, 5280.0, 5333.0, 5590.0):
            ref = dist.pdf(x) / mass
            assert abs(orc.signal_pdf(p, LO, HI, x) - ref) <= 2e-12 * ref, (lam, x)


def test_gamma_closed_form_and_variance(orc):
    """int_{-inf}^{inf} (d^2+delta^2)^{lambda-1/2} dd = delta^{2 lambda} sqrt(pi) Gamma(-lambda)/Gamma(1/2-lambda), and for
    lambda < -1 the variance of the symmetric core is sigma^2 (the Student-t variance relation behind delta)."""
    for lam in (-2.0, -1.4, -3.3):
        p = dict(T1, **{"lambda": lam})
        _, c = orc.shape_consts(p)
        G = lambda d: mp.exp(mp.mpf(orc.core_logG(p, float(d))))
        with mp.workdps(20):
            m0 = 2 * mp.quad(G, [0, 10, 40, 150, 600, 3000, 1e5, mp.inf])
            m2 = 2 * mp.quad(lambda d: d * d * G(d), [0, 10, 40, 150, 600, 3000, 1e5, mp.inf])
            ref = mp.mpf(c["delta"]) ** (2 * lam) * mp.sqrt(mp.pi) * mp.gamma(-lam) / mp.gamma(mp.mpf(1) / 2 - lam)
        assert abs(m0 - ref) <= 1e-12 * ref
        assert abs(m2 / m0 - p["sigma"] ** 2) <= 1e-9 * p["sigma"] ** 2, lam
    assert orc.shape_consts(dict(T1, **{"lambda": -0.7}))[1]["delta"] == T1["sigma"]


def test_constants_normalisation_and_logpdf_vs_mpmath(orc):
    """(ii) join constants, N_S by mpmath quadrature, per-event l and a tiny NLL for both Student-t shape points."""
    rng = np.random.default_rng(12)
    xs = np.concatenate([rng.uniform(LO, HI, 20), rng.normal(5280, 20, 20).clip(LO, HI), [LO, HI]])
    for p in (T1, T2, dict(T2, mu=5030.0), dict(T1, mu=5700.0, n=1.0)):
        m = MPStudent(p)
        st, c = orc.shape_consts(p)
        assert st == 0
        assert abs(mp.mpf(c["delta"]) - m.delta) <= 1e-15 * m.delta and c["alpha"] == 0.0
        assert abs(mp.mpf(c["L0"]) - m.L0) <= 1e-14 * abs(m.L0) and abs(mp.mpf(c["L1"]) - m.L1) <= 1e-14 * abs(m.L1)
        assert abs(mp.mpf(c["logG0"]) - mp.log(m.G0)) <= 1e-14 and abs(mp.mpf(c["logG1"]) - mp.log(m.G1)) <= 1e-14
        st2, nrm = orc.norm(p, LO, HI)
        assert st2 == 0 and abs(mp.mpf(nrm["NS"]) - m.NS) <= 1e-13 * m.NS
        got = orc.logpdf(xs, p, LO, HI)
        for x, g in zip(xs, got):
            assert abs(mp.mpf(float(g)) - m.l(float(x))) <= 3e-14, (p, x)
        ref = -sum(m.l(float(x)) for x in xs[:16])
        assert abs(mp.mpf(float(orc.nll(xs[:16], p, LO, HI)[0])) - ref) <= 1e-14 * abs(ref)
        S = lambda x: mp.mpf(orc.signal_pdf(p, LO, HI, float(x)))
        with mp.workdps(20):
            pts = sorted({mp.mpf(LO), mp.mpf(HI), *[mp.mpf(p["mu"] + d) for d in (-p["a"] * p["sigma"], 0, p["a2"] * p["sigma"])
                                                    if LO < p["mu"] + d < HI]})
            assert abs(mp.quad(S, pts, maxdegree=8) - 1) <= 1e-13


def test_join_continuity(orc):
    """(iii) value and slope of I continuous at both joins; L equals the numerical log-derivative of the core."""
    for p in (T1, T2):
        _, c = orc.shape_consts(p)
        for dj, Lj in ((c["d0"], c["L0"]), (c["d1"], c["L1"])):
            eps = 1e-4
            inside = dj + eps if dj < 0 else dj - eps
            outside = dj - eps if dj < 0 else dj + eps
            at = orc.log_I(p, dj)
            s_in = (orc.log_I(p, inside) - at) / (inside - dj)
            s_out = (orc.log_I(p, outside) - at) / (outside - dj)
            assert abs(s_in - Lj) <= 1e-4 * abs(Lj) and abs(s_out - Lj) <= 1e-4 * abs(Lj)
            h = 1e-3
            num = (orc.core_logG(p, dj + h) - orc.core_logG(p, dj - h)) / (2 * h)
            assert abs(num - Lj) <= 1e-7 * abs(Lj)


def test_analytic_gradient_and_domain(orc):
    """The analytic gradient (row f1) with the Student-t core against central differences of the oracle's NLL with
    O(h^2) convergence (the sigma-homogeneity power of G is 2 nu here, not nu); domain rules of zeta = 0."""
    x = inp.standin_masses(21, 4000)
    for p in (T1, T2):
        nll, g5 = orc.nll_gradient(x, p, LO, HI)
        g = g5[:4]
        assert abs(nll - orc.nll(x, p, LO, HI)[0]) <= 1e-12 * abs(nll)
        hb = 1e-4                                             # beta (fifth component) by central differences
        fdb = (orc.nll(x, dict(p, beta=p["beta"] + hb), LO, HI)[0] - orc.nll(x, dict(p, beta=p["beta"] - hb), LO, HI)[0]) / (2 * hb)
        assert abs(fdb - g5[4]) <= 1e-5 * max(abs(g5[4]), 1.0 / inp.GRAD_SCALE["beta"])
        idx, h = inp.fd_spec()
        _, g1 = orc.fd_gradient(x, p, idx, h, LO, HI)
        _, g2 = orc.fd_gradient(x, p, idx, h / 2, LO, HI)
        s = np.array([inp.GRAD_SCALE[k] for k in inp.FLOATED])
        e1, e2 = np.abs(g1 - g), np.abs(g2 - g)
        assert np.all(e2 <= 1e-5 * np.maximum(np.abs(g), 1.0 / s)), (g, g2)
        assert np.all((e2 <= 0.35 * e1) | (e1 <= 1e-7 * np.maximum(np.abs(g), 1.0 / s)))
    assert orc.shape_consts(dict(T1, **{"lambda": 0.5}))[0] == 1       # zeta = 0 needs lambda < 0
    assert orc.shape_consts(dict(T1, **{"lambda": 0.0}))[0] == 1
    assert orc.shape_consts(dict(T1, zeta=-0.0))[0] == 0               # -0.0 == 0
    assert orc.shape_consts(dict(T1, beta=5.0))[0] == 2                # join slope sign (reading D9)
