"""ctypes binding of oracle/libipa_oracle.so (numpy in, numpy out).  TEST INFRASTRUCTURE.

Every function is a thin marshalling wrapper; the arithmetic is in ipa_oracle.cpp, whose
comments cite the passage each routine follows.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

PARAM_FIELDS = ("mu", "sigma", "lambda", "zeta", "beta", "a", "n", "a2", "n2", "f", "k")
NPAR = len(PARAM_FIELDS)

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        d, i64, i32, u64, u32, vp = C.c_double, C.c_int64, C.c_int, C.c_uint64, C.c_uint32, C.c_void_p
        L.orc_besselk_scaled.restype = d; L.orc_besselk_scaled.argtypes = [d, d]
        L.orc_log_besselk.restype = d; L.orc_log_besselk.argtypes = [d, d]
        L.orc_zeta_int.restype = d; L.orc_zeta_int.argtypes = [i32]
        L.orc_shape_consts.restype = i32; L.orc_shape_consts.argtypes = [vp, vp]
        for name in ("orc_log_I", "orc_core_logG", "orc_core_logderiv"):
            getattr(L, name).restype = d; getattr(L, name).argtypes = [vp, d]
        L.orc_norm.restype = i32; L.orc_norm.argtypes = [vp, d, d, vp]
        L.orc_logpdf.restype = i32; L.orc_logpdf.argtypes = [vp, i64, vp, d, d, vp]
        L.orc_signal_pdf.restype = d; L.orc_signal_pdf.argtypes = [vp, d, d, d]
        L.orc_nll.restype = i32; L.orc_nll.argtypes = [vp, i64, vp, i32, d, d, vp, i32]
        L.orc_fd_gradient.restype = i32; L.orc_fd_gradient.argtypes = [vp, i64, vp, i32, vp, vp, d, d, i32, vp, vp]
        L.orc_nll_segmented.restype = i32; L.orc_nll_segmented.argtypes = [vp, vp, i64, vp, d, d, vp]
        L.orc_philox4x32_10.restype = None; L.orc_philox4x32_10.argtypes = [vp, vp, vp]
        L.orc_uniforms2.restype = None; L.orc_uniforms2.argtypes = [u64, u64, u32, u32, vp]
        L.orc_poisson.restype = i64; L.orc_poisson.argtypes = [u64, u64, u32, d]
        L.orc_poisson_array.restype = None; L.orc_poisson_array.argtypes = [u64, u64, i64, u32, d, vp, vp]
        L.orc_generate_mixture.restype = i32; L.orc_generate_mixture.argtypes = [u64, i64, vp, d, d, vp]
        L.orc_generate_signal_diag.restype = i32; L.orc_generate_signal_diag.argtypes = [u64, i64, vp, d, d, vp, vp, vp]
        L.orc_toy_generate.restype = i32
        L.orc_toy_generate.argtypes = [vp, i64, vp, i32, d, d, d, d, i64, vp, vp]
        L.orc_hist_fill.restype = None; L.orc_hist_fill.argtypes = [vp, i64, d, d, i32, vp]
        L.orc_binned_nll_scan.restype = i32
        L.orc_binned_nll_scan.argtypes = [vp, i32, d, d, vp, vp, vp, vp, i64, vp]
        L.orc_expected_hist.restype = i32; L.orc_expected_hist.argtypes = [i32, d, d, vp, d, d, d, vp]
        L.orc_poisson_hist_toys.restype = None; L.orc_poisson_hist_toys.argtypes = [vp, i32, vp, i64, vp]
        L.orc_norm_derivs.restype = i32; L.orc_norm_derivs.argtypes = [vp, d, d, vp]
        L.orc_nll_gradient.restype = i32; L.orc_nll_gradient.argtypes = [vp, i64, vp, d, d, vp, vp]
        L.orc_gauss_smear.restype = None; L.orc_gauss_smear.argtypes = [vp, i32, d, d, d, vp]
        L.orc_expected_hist_shape.restype = i32; L.orc_expected_hist_shape.argtypes = [i32, d, d, vp, d, d, d, vp]
        L.orc_binned_nll_scan_shape.restype = i32
        L.orc_binned_nll_scan_shape.argtypes = [vp, i32, d, d, vp, vp, vp, vp, i64, vp]
        L.orc_signal_shape.restype = i32; L.orc_signal_shape.argtypes = [i32, d, d, vp, vp]
        L.orc_nll_extended.restype = i32; L.orc_nll_extended.argtypes = [vp, i64, vp, d, d, d, d, vp]
        L.orc_cls_teststat.restype = None; L.orc_cls_teststat.argtypes = [vp, i32, i64, i32, vp, vp, vp]
        L.orc_cls_count_ge.restype = i64; L.orc_cls_count_ge.argtypes = [vp, i64, d]
        L.orc_cls_from_counts.restype = None; L.orc_cls_from_counts.argtypes = [i64, i64, i64, i64, vp]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def pack_params(p):
    """dict / sequence of dicts / (K,11) array -> contiguous (K,11) float64 array."""
    if isinstance(p, dict):
        p = [p]
    if isinstance(p, (list, tuple)) and len(p) and isinstance(p[0], dict):
        arr = np.array([[q[name] for name in PARAM_FIELDS] for q in p], dtype=np.float64)
    else:
        arr = np.array(p, dtype=np.float64)
        if arr.ndim == 1:
            arr = arr[None, :]
    assert arr.ndim == 2 and arr.shape[1] == NPAR
    return np.ascontiguousarray(arr)


def besselk_scaled(nu, x):
    return lib().orc_besselk_scaled(float(nu), float(x))


def log_besselk(nu, x):
    return lib().orc_log_besselk(float(nu), float(x))


def zeta_int(k):
    return lib().orc_zeta_int(int(k))


def shape_consts(p):
    """-> (status, dict(delta, alpha, d0, d1, logG0, logG1, L0, L1))"""
    P = pack_params(p)
    out = np.full(8, np.nan)
    st = lib().orc_shape_consts(_p(P), _p(out))
    return st, dict(zip(("delta", "alpha", "d0", "d1", "logG0", "logG1", "L0", "L1"), out.tolist()))


def log_I(p, d):
    P = pack_params(p)
    return lib().orc_log_I(_p(P), float(d))


def core_logG(p, d):
    P = pack_params(p)
    return lib().orc_core_logG(_p(P), float(d))


def core_logderiv(p, d):
    P = pack_params(p)
    return lib().orc_core_logderiv(_p(P), float(d))


def norm(p, lo, hi):
    """-> (status, dict(NS, core, left, right, NB))"""
    P = pack_params(p)
    out = np.full(5, np.nan)
    st = lib().orc_norm(_p(P), float(lo), float(hi), _p(out))
    return st, dict(zip(("NS", "core", "left", "right", "NB"), out.tolist()))


def signal_pdf(p, lo, hi, x):
    P = pack_params(p)
    return lib().orc_signal_pdf(_p(P), float(lo), float(hi), float(x))


def logpdf(x, p, lo, hi):
    x = np.ascontiguousarray(x, dtype=np.float64)
    P = pack_params(p)
    out = np.empty_like(x)
    lib().orc_logpdf(_p(x), x.size, _p(P), float(lo), float(hi), _p(out))
    return out


def nll(x, p, lo, hi, nthreads=1):
    """NLL for K parameter sets -> (K,) float64.  nthreads=1 is the oracle proper."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    P = pack_params(p)
    out = np.empty(P.shape[0])
    lib().orc_nll(_p(x), x.size, _p(P), P.shape[0], float(lo), float(hi), _p(out), int(nthreads))
    return out


def fd_gradient(x, theta, idx, h, lo, hi, nthreads=1):
    """Central-difference gradient (row G, reading C6) over the parameter fields idx[P] with steps h[P].
    -> (nll[2P+1] of the batch theta, theta +/- h_j e_j, grad[P])."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    P = pack_params(theta)
    assert P.shape[0] == 1
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    h = np.ascontiguousarray(h, dtype=np.float64)
    nll = np.empty(2 * idx.size + 1)
    g = np.empty(idx.size)
    st = lib().orc_fd_gradient(_p(x), x.size, _p(P), idx.size, _p(idx), _p(h), float(lo), float(hi), int(nthreads),
                               _p(nll), _p(g))
    assert st == 0, st
    return nll, g


def nll_segmented(x, offsets, p, lo, hi):
    x = np.ascontiguousarray(x, dtype=np.float64)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    P = pack_params(p)
    T = offsets.size - 1
    assert P.shape[0] == T
    out = np.empty(T)
    lib().orc_nll_segmented(_p(x), _p(offsets), T, _p(P), float(lo), float(hi), _p(out))
    return out


def philox4x32_10(key, ctr):
    key = np.ascontiguousarray(key, dtype=np.uint32)
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(key), _p(ctr), _p(out))
    return out


def uniforms2(seed, slot, attempt, stream):
    out = np.empty(2)
    lib().orc_uniforms2(int(seed), int(slot), int(attempt), int(stream), _p(out))
    return out


def poisson(seed, slot, stream, mean):
    return lib().orc_poisson(int(seed), int(slot), int(stream), float(mean))


def poisson_array(seed, slot0, n, stream, mean, diagnostics=False):
    """n draws at consecutive slots (same values as n calls of poisson); with diagnostics also (attempts[n], exit[n])."""
    out = np.empty(int(n), dtype=np.int64)
    diag = np.empty((int(n), 2), dtype=np.int32) if diagnostics else None
    lib().orc_poisson_array(int(seed), int(slot0), int(n), int(stream), float(mean), _p(out), _p(diag) if diagnostics else None)
    return (out, diag[:, 0], diag[:, 1]) if diagnostics else out


def generate_mixture(seed, n, p, lo, hi):
    P = pack_params(p)
    x = np.empty(int(n))
    st = lib().orc_generate_mixture(int(seed), int(n), _p(P), float(lo), float(hi), _p(x))
    assert st == 0, st
    return x


def generate_signal_diag(seed, n, p, lo, hi):
    """n signal draws (f ignored) -> (x[n], attempts per event, envelope violated?, envelope weight / N_S,
    max over a dense grid of log G - log(box height))."""
    P = pack_params(p)
    x = np.empty(int(n))
    diag = np.zeros(2, dtype=np.int64)
    env = np.zeros(2)
    st = lib().orc_generate_signal_diag(int(seed), int(n), _p(P), float(lo), float(hi), _p(x), _p(diag), _p(env))
    assert st == 0, st
    return x, diag[0] / max(int(n), 1), bool(diag[1]), float(env[0]), float(env[1])


def toy_generate(seeds, gen, mean_sig, mean_bkg, lo, hi, offsets_only=False):
    seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
    P = pack_params(gen)
    T = seeds.size
    stride = 1 if P.shape[0] == T and T > 1 else 0
    offsets = np.empty(T + 1, dtype=np.int64)
    lib().orc_toy_generate(_p(seeds), T, _p(P), stride, float(mean_sig), float(mean_bkg), float(lo), float(hi), 0,
                           None, _p(offsets))
    if offsets_only:
        return None, offsets
    x = np.empty(int(offsets[-1]))
    st = lib().orc_toy_generate(_p(seeds), T, _p(P), stride, float(mean_sig), float(mean_bkg), float(lo), float(hi),
                                x.size, _p(x), _p(offsets))
    assert st == 0, st
    return x, offsets


def hist_fill(x, lo, hi, nbins):
    x = np.ascontiguousarray(x, dtype=np.float64)
    counts = np.zeros(int(nbins), dtype=np.uint64)
    lib().orc_hist_fill(_p(x), x.size, float(lo), float(hi), int(nbins), _p(counts))
    return counts


def binned_nll_scan(counts, lo, hi, shape, ns, nb, k):
    counts = np.ascontiguousarray(counts, dtype=np.uint64)
    P = pack_params(shape)
    ns = np.ascontiguousarray(ns, dtype=np.float64)
    nb = np.ascontiguousarray(nb, dtype=np.float64)
    k = np.ascontiguousarray(k, dtype=np.float64)
    out = np.empty(ns.size)
    st = lib().orc_binned_nll_scan(_p(counts), counts.size, float(lo), float(hi), _p(P), _p(ns), _p(nb), _p(k),
                                   ns.size, _p(out))
    assert st == 0, st
    return out


def expected_hist(nbins, lo, hi, shape, ns, nb, k):
    P = pack_params(shape)
    out = np.empty(int(nbins))
    st = lib().orc_expected_hist(int(nbins), float(lo), float(hi), _p(P), float(ns), float(nb), float(k), _p(out))
    assert st == 0, st
    return out


def poisson_hist_toys(mean, seeds):
    mean = np.ascontiguousarray(mean, dtype=np.float64)
    seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
    out = np.empty((seeds.size, mean.size), dtype=np.uint32)
    lib().orc_poisson_hist_toys(_p(mean), mean.size, _p(seeds), seeds.size, _p(out))
    return out


def cls_teststat(counts, nu_sb, nu_b):
    """q_t for T toy histograms counts[T, nbins] (uint32 or uint64); reading F2."""
    counts = np.ascontiguousarray(counts)
    assert counts.dtype in (np.uint32, np.uint64)
    counts2 = counts.reshape(-1, np.asarray(nu_b).size)
    nu_sb = np.ascontiguousarray(nu_sb, dtype=np.float64)
    nu_b = np.ascontiguousarray(nu_b, dtype=np.float64)
    out = np.empty(counts2.shape[0])
    lib().orc_cls_teststat(_p(counts2), counts.dtype.itemsize, counts2.shape[0], nu_b.size, _p(nu_sb), _p(nu_b), _p(out))
    return out


def cls_count_ge(q, q_obs):
    q = np.ascontiguousarray(q, dtype=np.float64)
    return int(lib().orc_cls_count_ge(_p(q), q.size, float(q_obs)))


def cls_from_counts(count_sb, T_sb, count_b, T_b):
    out = np.empty(3)
    lib().orc_cls_from_counts(int(count_sb), int(T_sb), int(count_b), int(T_b), _p(out))
    return out


def nll_gradient(x, p, lo, hi):
    """Analytic (nll, d nll / d (mu, sigma, f, k, beta)) of one parameter set; SURVEY.md 8(f) row f1."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    P = pack_params(p)
    assert P.shape[0] == 1
    nll = np.empty(1)
    g = np.empty(5)
    st = lib().orc_nll_gradient(_p(x), x.size, _p(P), float(lo), float(hi), _p(nll), _p(g))
    assert st == 0, st
    return float(nll[0]), g


def norm_derivs(p, lo, hi):
    """(d ln N_S / d mu, d ln N_S / d sigma, d ln N_B / d k, d ln N_S / d beta) of one parameter set."""
    P = pack_params(p)
    out = np.empty(4)
    st = lib().orc_norm_derivs(_p(P), float(lo), float(hi), _p(out))
    assert st == 0, st
    return out


def gauss_smear(sig, lo, hi, sigma0):
    """Gaussian smearing of a histogram-like array on the bin grid (reading F3)."""
    sig = np.ascontiguousarray(sig, dtype=np.float64)
    out = np.empty_like(sig)
    lib().orc_gauss_smear(_p(sig), sig.size, float(lo), float(hi), float(sigma0), _p(out))
    return out


def signal_shape(nbins, lo, hi, shape):
    out = np.empty(int(nbins))
    st = lib().orc_signal_shape(int(nbins), float(lo), float(hi), _p(pack_params(shape)), _p(out))
    assert st == 0, st
    return out


def expected_hist_shape(lo, hi, sig, ns, nb, k):
    sig = np.ascontiguousarray(sig, dtype=np.float64)
    out = np.empty_like(sig)
    st = lib().orc_expected_hist_shape(sig.size, float(lo), float(hi), _p(sig), float(ns), float(nb), float(k), _p(out))
    assert st == 0, st
    return out


def binned_nll_scan_shape(counts, lo, hi, sig, ns, nb, k):
    counts = np.ascontiguousarray(counts, dtype=np.uint64)
    sig = np.ascontiguousarray(sig, dtype=np.float64)
    ns = np.ascontiguousarray(ns, dtype=np.float64)
    nb = np.ascontiguousarray(nb, dtype=np.float64)
    k = np.ascontiguousarray(k, dtype=np.float64)
    out = np.empty(ns.size)
    st = lib().orc_binned_nll_scan_shape(_p(counts), counts.size, float(lo), float(hi), _p(sig), _p(ns), _p(nb), _p(k),
                                         ns.size, _p(out))
    assert st == 0, st
    return out


def nll_extended(x, p, ns, nb, lo, hi):
    """Extended -log L = (ns + nb) - sum log(ns S + nb B) of one shape (its f is ignored); reading D4."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    P = pack_params(p)
    out = np.empty(1)
    st = lib().orc_nll_extended(_p(x), x.size, _p(P), float(ns), float(nb), float(lo), float(hi), _p(out))
    assert st == 0, st
    return float(out[0])
