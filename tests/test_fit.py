"""Config 2 (BASELINE.json): the host minimiser loop.  CPU part: the minimiser driving the ORACLE NLL
recovers the generating parameters of a seeded toy (a pin of the oracle's NLL and FD
gradient that does not come from the oracle itself: the truth is the generator's input).  GPU part:
the same minimiser driving ipa_nll_eval lands on the same parameters to 1e-6 relative.
"""
import os

import numpy as np
import pytest

import ipa_inputs as inp
from paper_1706_01420_b200 import minimiser

LO, HI = inp.LO, inp.HI


def start_point():
    th = inp.as_array(inp.GEN)
    for name, d in inp.FIT_START_SHIFT.items():
        th[inp.IDX[name]] += d
    return th


def fit(nll_batch, grad_batch=None):
    return minimiser.minimise(nll_batch, start_point(), inp.FLOATED, inp.FD_STEPS, inp.GRAD_SCALE, grad_batch=grad_batch)


def test_oracle_fit_recovers_generating_parameters(orc):
    n = 100_000
    x = orc.generate_mixture(2, n, inp.GEN, LO, HI)
    nthreads = max(1, os.cpu_count() or 1)
    res = fit(lambda th: orc.nll(x, th, LO, HI, nthreads=nthreads))
    assert res.edm < 1e-6
    assert 100 <= res.n_evals <= 600
    for name in inp.FLOATED:
        pull = (res.par[name] - inp.GEN[name]) / res.errors[name]
        assert abs(pull) < 4.0, (name, res.par[name], res.errors[name])
    # errors scale like 1/sqrt(N) from the 1e4-event scale of reading D18
    for name in inp.FLOATED:
        assert 0.1 < res.errors[name] / (inp.GRAD_SCALE[name] / np.sqrt(n / 1e4)) < 3.0
    # the FD gradient at the minimum vanishes (in 1/sigma units)
    idx, h = inp.fd_spec()
    _, g = orc.fd_gradient(x, res.theta, idx, h, LO, HI, nthreads=nthreads)
    assert np.all(np.abs(g) * np.array([res.errors[k] for k in inp.FLOATED]) < 1e-3)


def test_minimiser_on_a_quadratic():
    """The minimiser itself (no likelihood): exact minimum and covariance of a correlated quadratic."""
    A = np.array([[4.0, 1.0, 0.0, 0.0], [1.0, 3.0, 0.5, 0.0], [0.0, 0.5, 2.0, 0.2], [0.0, 0.0, 0.2, 1.0]])
    sc = np.array([inp.GRAD_SCALE[k] for k in inp.FLOATED])
    H = A / np.outer(sc, sc)
    x0 = np.array([inp.GEN[k] for k in inp.FLOATED])
    idx = [inp.IDX[k] for k in inp.FLOATED]

    def f(th):
        d = th[:, idx] - x0
        return 0.5 * np.einsum("ki,ij,kj->k", d, H, d) + 7.0
    res = fit(f)
    assert np.allclose([res.par[k] for k in inp.FLOATED], x0, rtol=0, atol=1e-6 * sc.max())
    assert np.allclose(res.cov, np.linalg.inv(H), rtol=1e-5)
    assert abs(res.nll - 7.0) < 1e-9


def test_oracle_fit_with_analytic_gradient_lands_on_the_same_minimum(orc):
    """Row f1 in the fit loop: the analytic gradient drives the same minimiser to the minimum the
    finite-difference fit finds (the two differ by the truncation error of the differences)."""
    n = 20_000
    x = orc.generate_mixture(2, n, inp.GEN, LO, HI)

    def nll_batch(th):
        return orc.nll(x, th, LO, HI)

    def grad_batch(th):
        out = [orc.nll_gradient(x, t, LO, HI) for t in th]
        return np.array([o[0] for o in out]), np.array([o[1][:4] for o in out])      # (mu, sigma, f, k) of the five components
    a = fit(nll_batch)
    b = fit(nll_batch, grad_batch)
    assert b.edm < 1e-9
    for name in inp.FLOATED:
        assert abs(a.par[name] - b.par[name]) <= 1e-4 * a.errors[name], (name, a.par[name], b.par[name])
        assert abs(a.errors[name] / b.errors[name] - 1) < 1e-3
    assert b.n_calls < a.n_calls + 20


@pytest.mark.gpu
def test_config2_fit_parity_gpu_vs_oracle(orc):
    import torch
    import paper_1706_01420_b200 as ipa
    n = 1_000_000
    x = orc.generate_mixture(2, n, inp.GEN, LO, HI)
    xd = torch.from_numpy(x).cuda()
    ws = ipa.workspace(n, 32)

    def gpu_nll(th):
        nll, _, _ = ipa.ipa_nll_eval(xd, th, LO, HI, ws=ws)
        return nll.cpu().numpy()
    res_g = fit(gpu_nll)
    nthreads = max(1, os.cpu_count() or 1)
    res_o = fit(lambda th: orc.nll(x, th, LO, HI, nthreads=nthreads))
    assert 150 <= res_g.n_evals <= 600
    for name in inp.FLOATED:
        a, b = res_g.par[name], res_o.par[name]
        assert abs(a - b) <= 1e-6 * abs(b), (name, a, b)
        assert abs((b - inp.GEN[name]) / res_o.errors[name]) < 4.5
    assert abs(res_g.nll - res_o.nll) <= 1e-10 * abs(res_o.nll)
    # prepared layout: same minimum
    xs = ipa.ipa_events_prepare(xd, LO, HI)

    def gpu_nll_sorted(th):
        nll, _, _ = ipa.ipa_nll_eval(xs, th, LO, HI, ws=ws)
        return nll.cpu().numpy()
    res_s = fit(gpu_nll_sorted)
    for name in inp.FLOATED:
        assert abs(res_s.par[name] - res_o.par[name]) <= 1e-6 * abs(res_o.par[name])

    # the same fit driven by the analytic gradient (row f1): same minimum
    def gpu_grad(th):
        nll, g, _ = ipa.ipa_nll_grad_eval(xs, th, LO, HI, ws=ws)
        return nll.cpu().numpy(), g.cpu().numpy()[:, :4]
    res_a = fit(gpu_nll_sorted, gpu_grad)
    assert res_a.edm < 1e-9
    for name in inp.FLOATED:
        assert abs(res_a.par[name] - res_o.par[name]) <= 1e-6 * abs(res_o.par[name]), (name, res_a.par[name])
