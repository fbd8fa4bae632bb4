"""Pins of the oracle's Ipatia density, normalisation, per-event log-likelihood and NLL
(oracle/ipa_oracle.cpp; readings C1-C3, C5 in DESIGN.md / SURVEY.md 8(c)).

The reference implementation used for comparison here is built ONLY from mpmath primitives
(besselk, quad, log) at 30+ digits, i.e. different arithmetic, different Bessel algorithm and
different quadrature from the oracle's.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import ipa_inputs as inp

mp.mp.dps = 30
GOLD = os.path.join(os.path.dirname(__file__), "golden")
LO, HI = inp.LO, inp.HI
P1, P2 = inp.GEN, inp.P2


# ---- mpmath restatement of the DEFINITION (C1-C3), used as an independent reference -------------
class MPModel:
    def __init__(self, p, lo=LO, hi=HI):
        g = lambda name: mp.mpf(p[name])
        self.p = p
        self.mu, self.sigma, self.lam, self.zeta, self.beta = g("mu"), g("sigma"), g("lambda"), g("zeta"), g("beta")
        self.a, self.n, self.a2, self.n2, self.f, self.k = g("a"), g("n"), g("a2"), g("n2"), g("f"), g("k")
        self.lo, self.hi = mp.mpf(lo), mp.mpf(hi)
        Kl, Kl1 = mp.besselk(self.lam, self.zeta), mp.besselk(self.lam + 1, self.zeta)
        self.delta = self.sigma * mp.sqrt(self.zeta * Kl / Kl1)
        self.alpha = mp.sqrt(self.zeta * Kl1 / Kl) / self.sigma
        self.nu = self.lam - mp.mpf(1) / 2
        self.d0, self.d1 = -self.a * self.sigma, self.a2 * self.sigma
        self.G0, self.G1 = self.G(self.d0), self.G(self.d1)
        self.L0, self.L1 = mp.diff(lambda d: mp.log(self.G(d)), self.d0), mp.diff(lambda d: mp.log(self.G(d)), self.d1)
        pts = sorted({self.lo, self.hi, *[self.mu + d for d in (self.d0, 0, self.d1) if self.lo < self.mu + d < self.hi]})
        self.NS = mp.quad(lambda x: self.I(x - self.mu), pts)
        self.NB = (mp.exp(self.k * (self.hi - self.lo)) - 1) / self.k if self.k != 0 else self.hi - self.lo

    def G(self, d):
        r = mp.sqrt(d * d + self.delta ** 2)
        return r ** self.nu * mp.exp(self.beta * d) * mp.besselk(self.nu, self.alpha * r)

    def I(self, d):
        if d < self.d0:
            return self.G0 * (1 - (d - self.d0) * self.L0 / self.n) ** (-self.n)
        if d > self.d1:
            return self.G1 * (1 - (d - self.d1) * self.L1 / self.n2) ** (-self.n2)
        return self.G(d)

    def l(self, x):
        x = mp.mpf(x)
        S = self.I(x - self.mu) / self.NS
        B = mp.exp(self.k * (x - self.lo)) / self.NB
        return mp.log(self.f * S + (1 - self.f) * B)


@pytest.fixture(scope="module")
def mp1():
    return MPModel(P1)


@pytest.fixture(scope="module")
def mp2():
    return MPModel(P2)


def _golden():
    rows = []
    for line in open(os.path.join(GOLD, "worked_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        s, q, arg, val = line.split()
        rows.append((s, q, arg, float(val)))
    return rows


def test_golden_values_agree_with_independent_mpmath(mp1, mp2):
    """The golden file itself is re-derived here from the definition with mpmath."""
    for s, q, arg, val in _golden():
        m = mp1 if s == "P1" else mp2
        if q == "l":
            ref = m.l(arg)
        elif q == "S":
            ref = m.I(mp.mpf(arg) - m.mu) / m.NS
        elif q in ("core", "left", "right"):
            continue
        else:
            ref = getattr(m, q)
        assert abs(ref - mp.mpf(val)) <= 5e-16 * abs(ref), (s, q, arg)


def test_worked_example_golden(orc):
    """Oracle vs tests/golden/worked_example.txt."""
    for s, q, arg, val in _golden():
        p = P1 if s == "P1" else P2
        st, c = orc.shape_consts(p)
        st2, nrm = orc.norm(p, LO, HI)
        assert st == 0 and st2 == 0
        if q in ("delta", "alpha", "L0", "L1"):
            got = c[q]
        elif q in ("G0", "G1"):
            got = math.exp(c["log" + q])
        elif q in ("NS", "core", "left", "right", "NB"):
            got = nrm[q]
        elif q == "S":
            got = orc.signal_pdf(p, LO, HI, float(arg))
        else:
            got = float(orc.logpdf(np.array([float(arg)]), p, LO, HI)[0])
        assert abs(got - val) <= 2e-15 * max(1.0, abs(val)) if q == "l" else abs(got - val) <= 4e-15 * abs(val), (s, q, arg, got, val)


def test_logpdf_vs_mpmath_random_points(orc, mp1, mp2):
    rng = np.random.default_rng(3)
    xs = np.concatenate([rng.uniform(LO, HI, 25), rng.normal(5280, 20, 25).clip(LO, HI)])
    for p, m in ((P1, mp1), (P2, mp2)):
        got = orc.logpdf(xs, p, LO, HI)
        for x, g in zip(xs, got):
            assert abs(mp.mpf(float(g)) - m.l(float(x))) <= 2e-15 * 8, (x, g)


def test_pdf_integrates_to_one(orc):
    """int_lo^hi S dx = 1 by independent adaptive quadrature of the oracle's S (C8.4)."""
    for p in (P1, P2, dict(P1, mu=5020.0), dict(P2, mu=5590.0, zeta=0.3)):
        S = lambda x: mp.mpf(orc.signal_pdf(p, LO, HI, float(x)))
        with mp.workdps(20):
            pts = sorted({mp.mpf(LO), mp.mpf(HI), *[mp.mpf(p["mu"] + d) for d in (-p["a"] * p["sigma"], 0, p["a2"] * p["sigma"])
                                                    if LO < p["mu"] + d < HI]})
            tot = mp.quad(S, pts, maxdegree=8)
        assert abs(tot - 1) <= 1e-13, (p, tot)


def test_midpoint_sum_converges_quadratically(orc):
    """The paper normalises by summing the kernel output on a bin grid; that
    midpoint sum converges O(h^2) to the oracle's exact N_S (reading D6)."""
    _, nrm = orc.norm(P1, LO, HI)
    errs = []
    for nb in (2000, 4000, 8000):
        c = LO + (np.arange(nb) + 0.5) * (HI - LO) / nb
        tot = sum(math.exp(orc.log_I(P1, float(x) - P1["mu"])) for x in c) * (HI - LO) / nb
        errs.append(abs(tot - nrm["NS"]))
    assert errs[0] < 1e-3 * nrm["NS"]
    assert 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0


def test_background_normalisation_matches_paper_formula(orc):
    """integral_exp = (exp(k Mmax)-exp(k Mmin))/k, Mmax-Mmin at k=0; the oracle's
    shifted form is that divided by exp(k lo)."""
    for k in (-0.002, 0.0, 0.0013, -1e-12, 3e-11):
        _, nrm = orc.norm(dict(P1, k=k), LO, HI)
        if k != 0 and abs(k) > 1e-9:
            ref = (mp.exp(mp.mpf(k) * HI) - mp.exp(mp.mpf(k) * LO)) / mp.mpf(k) / mp.exp(mp.mpf(k) * LO)
        else:
            ref = mp.mpf(HI - LO) * (1 + mp.mpf(k) * (HI - LO) / 2)
        assert abs(mp.mpf(nrm["NB"]) - ref) <= 1e-15 * ref


def test_hyperbolic_special_case(orc):
    """lambda=1: log G(d) = (1/2) log(pi/(2 alpha)) + beta d - alpha sqrt(d^2+delta^2)  (C8.5)."""
    for p in (P1, dict(P1, beta=0.02, zeta=3.0)):
        _, c = orc.shape_consts(p)
        for d in (-29.0, -3.3, 0.0, 11.0, 30.0):
            ref = 0.5 * math.log(math.pi / (2 * c["alpha"])) + p["beta"] * d - c["alpha"] * math.hypot(d, c["delta"])
            assert abs(orc.core_logG(p, d) - ref) <= 1e-14


def test_gaussian_limit(orc):
    """zeta -> infinity, beta = 0: alpha/delta -> 1/sigma^2 with relative correction ~1.5/zeta and
    log G(d) - log G(0) -> -d^2/(2 sigma^2) (C8.6)."""
    for zeta, tol in ((1e2, 2e-3), (1e3, 2e-4), (1e4, 2e-5)):
        p = dict(P1, zeta=zeta)
        _, c = orc.shape_consts(p)
        corr = c["alpha"] / c["delta"] * p["sigma"] ** 2 - 1
        assert abs(corr - 1.5 / zeta) <= tol * 1.5 / zeta * 10
        for d in (5.0, 15.0, 25.0):
            got = orc.core_logG(p, d) - orc.core_logG(p, 0.0)
            assert abs(got + d * d / (2 * p["sigma"] ** 2)) <= 3.0 / zeta * (d * d / (2 * p["sigma"] ** 2)) + 1e-12


def test_core_variance_is_sigma_squared(orc):
    """The (delta, alpha) parametrisation makes sigma^2 the variance of the untruncated symmetric
    core (C8.7)."""
    for lam, zeta in ((1.0, 1.0), (-1.3, 2.0), (0.4, 5.0)):
        p = dict(P1, **{"lambda": lam}, zeta=zeta, beta=0.0)
        G = lambda d: mp.exp(mp.mpf(orc.core_logG(p, float(d))))
        with mp.workdps(15):
            m0 = 2 * mp.quad(G, [0, 10, 40, 150, 600, 3000])
            m2 = 2 * mp.quad(lambda d: d * d * G(d), [0, 10, 40, 150, 600, 3000])
        assert abs(m2 / m0 - 225.0) <= 1e-6 * 225.0


def test_join_continuity_value_and_slope(orc):
    """I and dI/dd are continuous at d0 and d1 (C8.8); L(d) equals the numerical log-derivative."""
    for p in (P1, P2):
        _, c = orc.shape_consts(p)
        for dj, Lj in ((c["d0"], c["L0"]), (c["d1"], c["L1"])):
            eps = 1e-4
            inside = dj + eps if dj < 0 else dj - eps
            outside = dj - eps if dj < 0 else dj + eps
            at = orc.log_I(p, dj)
            # value: both one-sided limits approach log I(dj) linearly with the same slope
            s_in = (orc.log_I(p, inside) - at) / (inside - dj)
            s_out = (orc.log_I(p, outside) - at) / (outside - dj)
            assert abs(s_in - Lj) <= 1e-4 * abs(Lj) and abs(s_out - Lj) <= 1e-4 * abs(Lj)
            assert abs(s_in - s_out) <= 2e-4 * abs(Lj)
            h = 1e-3
            num = (orc.core_logG(p, dj + h) - orc.core_logG(p, dj - h)) / (2 * h)
            assert abs(num - orc.core_logderiv(p, dj)) <= 1e-9 * max(1, abs(num)) + 1e-7 * abs(num)
            assert abs(orc.core_logderiv(p, dj) - Lj) <= 1e-15 * abs(Lj)


def test_logderiv_formula_vs_mpmath(orc, mp2):
    for d in (-20.0, -1.0, 0.5, 17.0, 33.0):
        ref = mp.diff(lambda t: mp.log(mp2.G(t)), mp.mpf(d))
        assert abs(mp.mpf(orc.core_logderiv(P2, d)) - ref) <= 1e-14 * max(1, abs(ref))


def test_brute_force_tiny_nll(orc, mp1, mp2):
    """N<=16: NLL against a naive high-precision loop (C8.10); batch == singles; permutation."""
    rng = np.random.default_rng(8)
    xs = rng.uniform(LO, HI, 16)
    xs[:6] = rng.normal(5280, 15, 6)
    for p, m in ((P1, mp1), (P2, mp2)):
        ref = -sum(m.l(float(x)) for x in xs)
        got = orc.nll(xs, p, LO, HI)[0]
        assert abs(mp.mpf(float(got)) - ref) <= 1e-14 * abs(ref)
    both = orc.nll(xs, [P1, P2], LO, HI)
    assert both[0] == orc.nll(xs, P1, LO, HI)[0] and both[1] == orc.nll(xs, P2, LO, HI)[0]
    big = rng.uniform(LO, HI, 5000)
    a, b = orc.nll(big, P1, LO, HI)[0], orc.nll(rng.permutation(big), P1, LO, HI)[0]
    assert abs(a - b) <= 1e-13 * abs(a)
    assert orc.nll(np.empty(0), P1, LO, HI)[0] == 0.0


def test_pairwise_sum_equals_sum_of_logpdf(orc):
    rng = np.random.default_rng(9)
    xs = rng.uniform(LO, HI, 3001)
    l = orc.logpdf(xs, P1, LO, HI)
    assert abs(orc.nll(xs, P1, LO, HI)[0] + math.fsum(l)) <= 1e-14 * abs(math.fsum(l))
    thr = orc.nll(np.tile(xs, 3), P1, LO, HI, nthreads=4)[0]
    assert abs(thr - orc.nll(np.tile(xs, 3), P1, LO, HI)[0]) <= 1e-14 * abs(thr)


def test_limits_f0_f1_and_k0(orc):
    xs = np.array([5010.0, 5280.0, 5555.0])
    l0 = orc.logpdf(xs, dict(P1, f=0.0), LO, HI)
    _, nrm = orc.norm(P1, LO, HI)
    assert np.allclose(l0, P1["k"] * (xs - LO) - math.log(nrm["NB"]), rtol=0, atol=1e-14)
    l1 = orc.logpdf(xs, dict(P1, f=1.0), LO, HI)
    assert np.allclose(l1, [math.log(orc.signal_pdf(P1, LO, HI, x)) for x in xs], rtol=0, atol=1e-14)
    lk = orc.logpdf(xs, dict(P1, f=0.0, k=0.0), LO, HI)
    assert np.allclose(lk, -math.log(HI - LO), rtol=0, atol=1e-15)


def test_domain_status(orc):
    bad = [dict(P1, sigma=0.0), dict(P1, zeta=-1.0), dict(P1, a=0.0), dict(P1, n2=-2.0), dict(P1, f=1.5),
           dict(P1, mu=float("nan"))]
    for p in bad:
        assert orc.shape_consts(p)[0] == 1
        assert orc.nll(np.array([5100.0]), p, LO, HI)[0] == float("inf")
    # a huge |beta| flips the slope at a join: status 2 (reading D9)
    assert orc.shape_consts(dict(P1, beta=5.0))[0] == 2
    assert orc.nll(np.array([5100.0]), dict(P1, beta=5.0), LO, HI)[0] == float("inf")


def test_range_inside_one_tail_and_n_equal_one(orc):
    """Clipping of C5: a fit range that lies entirely inside the left tail, and n=1 (log form)."""
    p = dict(P1, mu=5700.0, n=1.0)
    m = MPModel(p)
    _, nrm = orc.norm(p, LO, HI)
    assert abs(mp.mpf(nrm["NS"]) - m.NS) <= 1e-14 * m.NS
    assert nrm["core"] == 0.0 and nrm["right"] == 0.0
    p = dict(P2, n=1.0, n2=1.0)
    m = MPModel(p)
    _, nrm = orc.norm(p, LO, HI)
    assert abs(mp.mpf(nrm["NS"]) - m.NS) <= 1e-14 * m.NS


def test_range_deep_inside_one_tail_with_a_large_exponent(orc):
    """C5 between two points of the same tail: with n = 66 and the range far from the peak, F(ul) and F(ur) agree to
    all digits and must not be subtracted; N_S and the per-event values against the closed form in mpmath at 50 digits
    (mpmath's own quadrature needs that many digits here: the integrand spans 50 decades)."""
    for mu in (5610.0, 5627.0, 5700.0):
        p = dict(P1, mu=mu, sigma=0.89, a=2.34, n=66.0)
        with mp.workdps(50):
            m = MPModel(p)
            ul = 1 - (m.lo - m.mu - m.d0) * m.L0 / m.n
            ur = 1 - (m.hi - m.mu - m.d0) * m.L0 / m.n
            F = lambda u: (u ** (1 - m.n) - 1) / (1 - m.n)
            closed = m.G0 * (m.n / m.L0) * (F(ul) - F(ur))
            assert abs(closed - m.NS) <= mp.mpf("1e-13") * closed          # closed form = mpmath quadrature (its own accuracy)
            st, nrm = orc.norm(p, LO, HI)
            assert st == 0 and abs(mp.mpf(nrm["NS"]) - closed) <= 2e-14 * closed, (mu, nrm["NS"], closed)
            xs = np.array([LO, 5123.4, 5400.0, 5599.0, HI])
            got = orc.logpdf(xs, p, LO, HI)
            for x, g in zip(xs, got):
                assert abs(mp.mpf(float(g)) - m.l(float(x))) <= 1e-13, (mu, x)


def test_population_facts(orc):
    """E[-l] = 6.0901249 per event and P(core) = 0.34443 for the config model (C8.9)."""
    l = lambda x: orc.logpdf(np.array([float(x)]), P1, LO, HI)[0]
    with mp.workdps(15):
        pts = [LO, 5250, 5280, 5310, HI]
        ent = -mp.quad(lambda x: mp.exp(l(x)) * l(x), pts)
        core = mp.quad(lambda x: mp.exp(l(x)), [5250, 5280, 5310])
    assert abs(ent - 6.0901249) <= 2e-7
    assert abs(core - 0.34443) <= 1e-5
