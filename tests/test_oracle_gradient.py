"""Pins of the oracle's analytic NLL gradient (oracle/ipa_oracle.cpp orc_nll_gradient).
The paper gives no derivative formulae (PAPER.md:36, 383 only mention analytic gradients), so the pins are:
the derivative of the DEFINITION taken by mpmath (numerical differentiation at 40 digits of an mpmath-only
restatement of C1-C3, including its quad-based normalisation), the second-order convergence of the oracle's
own central differences towards the analytic value, and the exact limits f = 0, f = 1, k = 0."""
import mpmath as mp
import numpy as np
import pytest

import ipa_inputs as inp
from test_oracle_ipatia import MPModel

LO, HI = inp.LO, inp.HI
NAMES = inp.GRAD_NAMES          # (mu, sigma, f, k, beta)


def mp_nll(p, xs):
    m = MPModel(p)
    return -sum(m.l(x) for x in xs)


@pytest.mark.parametrize("shape", ["P1", "P2"])
def test_gradient_vs_mpmath_derivative_of_the_definition(orc, shape):
    mp.mp.dps = 40
    theta = dict(inp.GEN if shape == "P1" else inp.P2)
    xs = [5003.5, 5249.0, 5262.25, 5281.0, 5299.75, 5330.5, 5588.0]      # both tails, both sides of the core
    nll, g = orc.nll_gradient(np.array(xs), theta, LO, HI)
    assert abs(nll - float(mp_nll(theta, xs))) <= 1e-12 * abs(nll)
    for j, name in enumerate(NAMES):
        def f(v, name=name):
            q = dict(theta)
            q[name] = v
            return mp_nll(q, xs)
        h = mp.mpf(10) ** -12 * max(1, abs(theta[name]))
        ref = (f(mp.mpf(theta[name]) + h) - f(mp.mpf(theta[name]) - h)) / (2 * h)   # 40 digits: error ~ h^2
        assert abs(g[j] - float(ref)) <= 2e-9 * max(abs(float(ref)), 1.0 / inp.GRAD_SCALE[name] * 1e-3), (name, g[j], ref)


def test_fd_gradient_batch_layout_and_quadratic_convergence(orc):
    """Row G (reading C6), orc.fd_gradient: the batch is theta, theta +/- h_j e_j in the order (mu, sigma, f, k); the
    differences converge to the analytic gradient (pinned above by mpmath) like h^2 -- a wrong sign, index, step or
    denominator fails one of the two checks."""
    # few events, none within the largest step of a join (the density is only C^1 there)
    x = np.array([5010.0, 5120.0, 5236.0, 5266.0, 5279.0, 5291.5, 5322.0, 5470.0])
    theta = inp.as_array(inp.P2)
    _, g = orc.nll_gradient(x, theta, LO, HI)
    g = g[:4]
    idx, h0 = inp.fd_spec()
    errs = []
    for scale in (1.0, 0.5):
        h = scale * 20 * h0
        nll, fd = orc.fd_gradient(x, theta, idx, h, LO, HI)
        for j in range(4):                                       # layout: plain NLLs at the displaced points
            tp, tm = theta.copy(), theta.copy()
            tp[idx[j]] += h[j]
            tm[idx[j]] -= h[j]
            assert nll[2 * j + 1] == orc.nll(x, tp, LO, HI)[0] and nll[2 * j + 2] == orc.nll(x, tm, LO, HI)[0]
        assert nll[0] == orc.nll(x, theta, LO, HI)[0]
        errs.append(fd - g)
    assert np.all(np.abs(errs[0]) < 1e-3 * np.maximum(1.0, np.abs(g)))
    ratio = errs[0] / errs[1]
    assert np.all((3.0 < ratio) & (ratio < 5.0)), ratio          # O(h^2): halving h divides the error by 4
    # a subset of the parameters in another order
    nll2, fd2 = orc.fd_gradient(x, theta, idx[[3, 0]], (20 * h0)[[3, 0]], LO, HI)
    _, fd1 = orc.fd_gradient(x, theta, idx, 20 * h0, LO, HI)
    assert np.array_equal(fd2, fd1[[3, 0]]) and nll2.size == 5


def test_gradient_limits(orc):
    x = orc.generate_mixture(7, 500, inp.GEN, LO, HI)
    # f = 0: no dependence on the signal shape; f = 1: none on k; k = 0 uses the series of d ln N_B / d k
    _, g0 = orc.nll_gradient(x, dict(inp.GEN, f=0.0), LO, HI)
    assert g0[0] == 0.0 and g0[1] == 0.0 and g0[4] == 0.0
    _, g1 = orc.nll_gradient(x, dict(inp.GEN, f=1.0), LO, HI)
    assert g1[3] == 0.0
    _, gk = orc.nll_gradient(x, dict(inp.GEN, k=0.0), LO, HI)
    _, gk2 = orc.nll_gradient(x, dict(inp.GEN, k=1e-9), LO, HI)
    assert np.all(np.abs(gk - gk2) <= 1e-6 * np.maximum(1.0, np.abs(gk)))
    # beta by central differences of the oracle's own NLL (O(h^2)), at a shape with beta != 0 and asymmetric tails
    xb = inp.standin_masses(31, 3000)
    _, gb = orc.nll_gradient(xb, inp.P2, LO, HI)
    errs = []
    for h in (2e-4, 1e-4):
        fd = (orc.nll(xb, dict(inp.P2, beta=inp.P2["beta"] + h), LO, HI)[0] - orc.nll(xb, dict(inp.P2, beta=inp.P2["beta"] - h), LO, HI)[0]) / (2 * h)
        errs.append(fd - gb[4])
    assert abs(errs[1]) <= 1e-5 * max(abs(gb[4]), 1.0 / inp.GRAD_SCALE["beta"]) and 3.0 < errs[0] / errs[1] < 5.0
    # at the generating parameters of a large sample every component is small in units of its error
    xl = orc.generate_mixture(2, 100000, inp.GEN, LO, HI)
    _, g = orc.nll_gradient(xl, inp.GEN, LO, HI)
    s = np.array([inp.GRAD_SCALE[k] for k in NAMES]) / np.sqrt(10.0)
    assert np.all(np.abs(g * s) < 5.0)
