"""CPU-side checks of the CUDA library: it builds, loads and exports every symbol include/ipanll.h
declares; argument validation works without a GPU; compute calls fail loudly without one; and the
kernels' __host__ __device__ arithmetic, compiled for the CPU by tests/devmath_host.cu, agrees with
the oracle (the same source runs on the GPU in the `-m gpu` tests)."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

import ipa_inputs as inp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
LO, HI = inp.LO, inp.HI


@pytest.fixture(scope="module")
def ipa():
    import paper_1706_01420_b200 as m
    m.lib()
    return m


def test_library_exports_every_declared_symbol(ipa):
    hdr = open(os.path.join(ROOT, "include", "ipanll.h")).read()
    declared = set(re.findall(r"\b(ipa_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(ipa.EXPORTS), declared ^ set(ipa.EXPORTS)
    L = ipa.lib()
    for name in declared:
        assert hasattr(L, name), name
    out = subprocess.check_output(["nm", "-D", "--defined-only", ipa.library_path()], text=True)
    for name in declared:
        assert re.search(r"\bT %s\b" % name, out), name
    # the product library must not link the oracle nor contain its symbols
    assert "orc_" not in out
    assert ipa.ipa_version().startswith("ipanll")


def test_sm100a_image_present(ipa):
    out = subprocess.check_output(["cuobjdump", "-lelf", ipa.library_path()], text=True)
    assert "sm_100a" in out


def test_argument_validation_without_gpu(ipa):
    L = ipa.lib()
    P = ipa.pack_params(inp.GEN)
    rng = ipa.binding._Range(LO, HI)
    bad = ipa.binding._Range(HI, LO)
    one = C.c_void_p(256)  # non-null dummy; never dereferenced because validation fails first
    p = P.ctypes.data_as(C.c_void_p)
    assert L.ipa_nll_eval(one, -1, p, 1, rng, one, None, None, None, one, 1 << 30, None) == -1
    assert L.ipa_nll_eval(one, 10, p, 0, rng, one, None, None, None, one, 1 << 30, None) == -1
    assert L.ipa_nll_eval(one, 10, p, 33, rng, one, None, None, None, one, 1 << 30, None) == -1
    assert L.ipa_nll_eval(one, 10, p, 1, bad, one, None, None, None, one, 1 << 30, None) == -1
    assert L.ipa_nll_eval(None, 10, p, 1, rng, one, None, None, None, one, 1 << 30, None) == -1
    assert L.ipa_nll_eval(C.c_void_p(260), 10, p, 1, rng, one, None, None, None, one, 1 << 30, None) == -1
    assert L.ipa_nll_eval(one, 10, p, 1, rng, one, None, None, None, one, 16, None) == -2
    assert L.ipa_nll_eval(one, 10, p, 1, rng, one, None, None, None, C.c_void_p(264), 1 << 30, None) == -2
    # options: an unknown degree policy or a non-zero reserved field is an argument error
    for pol, res, slot in ((2, 0, 0), (-1, 0, 0), (0, 7, 0), (0, 0, -1)):
        o = ipa.binding._Options()
        o.degree_policy = pol
        o.reserved = res
        o.first_slot = slot
        assert L.ipa_nll_eval(one, 10, p, 1, rng, one, None, None, C.byref(o), one, 1 << 30, None) == -1
    assert L.ipa_norm(None, 1, rng, one, one, None, None, one, 1 << 30, None) == -1
    idx = np.array([0, 11], dtype=np.int32)
    hh = np.array([0.01, 0.01])
    assert L.ipa_nll_fd_gradient(one, 10, p, 2, idx.ctypes.data_as(C.c_void_p), hh.ctypes.data_as(C.c_void_p), rng, one, one,
                                 None, None, one, 1 << 30, None) == -1           # field index out of range
    assert L.ipa_nll_fd_gradient(one, 10, p, 12, idx.ctypes.data_as(C.c_void_p), hh.ctypes.data_as(C.c_void_p), rng, one, one,
                                 None, None, one, 1 << 30, None) == -1           # P > 11
    assert L.ipa_events_prepare(one, 10, None, 0, rng, one, one, 1 << 30, None) == -1      # output aliases the input
    assert L.ipa_events_prepare(one, 2 ** 32, None, 0, rng, C.c_void_p(512), one, 1 << 30, None) == -1
    assert L.ipa_events_prepare(one, 10, None, 0, rng, C.c_void_p(512), one, 16, None) == -2
    assert ipa.ipa_prepare_workspace_bytes(10 ** 8) >= 256 * 296 * 4 and ipa.ipa_prepare_workspace_bytes(10 ** 5, 7) == 256
    assert L.ipa_hist_fill(one, 5, rng, 0, one, None) == -1
    assert L.ipa_strerror(-2).decode().startswith("workspace")
    assert ipa.ipa_workspace_bytes(10 ** 8, 9) >= 9 * 600
    assert ipa.ipa_workspace_bytes(10 ** 8, 1000) > ipa.ipa_workspace_bytes(10 ** 8, 9)


def test_compute_fails_loudly_without_gpu(ipa):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(ipa.IpaError):
        ipa.ipa_norm(inp.GEN, LO, HI)
    with pytest.raises(ipa.IpaError):
        ipa.ipa_nll_eval(torch.zeros(4, dtype=torch.float64), inp.GEN, LO, HI)


# ---- the kernels' arithmetic, compiled for the host ------------------------------------------------
@pytest.fixture(scope="module")
def emu(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("emu") / "libdevmath_host.so")
    subprocess.check_call(["nvcc", "-arch=sm_100a", "-O2", "-std=c++17", "-Xcompiler", "-fPIC", "-shared",
                           "-I", os.path.join(ROOT, "include"), "-o", out, os.path.join(ROOT, "tests", "devmath_host.cu")])
    L = C.CDLL(out)
    d, vp, ll = C.c_double, C.c_void_p, C.c_longlong
    L.emu_besselk_scaled.restype = d; L.emu_besselk_scaled.argtypes = [d, d]
    L.emu_consts.argtypes = [vp, d, d, C.c_int, vp]
    L.emu_logpdf.argtypes = [vp, d, d, C.c_int, vp, ll, vp]
    L.emu_logI.argtypes = [vp, d, d, vp, ll, vp]
    L.emu_cells.argtypes = [vp, d, d, C.c_int, vp]
    L.emu_grad.argtypes = [vp, d, d, C.c_int, vp, ll, vp]
    L.emu_uniforms2.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, vp]
    L.emu_poisson.restype = ll; L.emu_poisson.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, d]
    return L


def test_device_bessel_vs_mpmath(emu):
    import mpmath as mp
    mp.mp.dps = 30
    worst = 0.0
    for nu in (0.0, 0.3, 0.5, 1.0, 1.8, 2.5, -1.3, 5.0):
        for x in (1e-3, 0.01, 0.1, 0.5, 1.0, 2.0, 3.43, 10.0, 50.0, 300.0, 700.0):
            ref = mp.besselk(nu, x) * mp.exp(x)
            worst = max(worst, float(abs((mp.mpf(emu.emu_besselk_scaled(nu, x)) - ref) / ref)))
    assert worst <= 3e-15


@pytest.mark.parametrize("policy", [0, 1])
@pytest.mark.parametrize("shape", ["P1", "P2", "direct", "T1", "T2"])
def test_device_math_vs_oracle(emu, orc, shape, policy):
    P = {"P1": inp.GEN, "P2": inp.P2, "direct": dict(inp.GEN, zeta=0.2), "T1": inp.T1, "T2": inp.T2}[shape]
    p = inp.as_array(P)
    out = np.zeros(15)
    emu.emu_consts(p.ctypes.data, LO, HI, policy, out.ctypes.data)
    st, sc = orc.shape_consts(P)
    _, nm = orc.norm(P, LO, HI)
    assert out[0] == 0 and st == 0
    assert out[2] == {"direct": 1, "T1": 2, "T2": 2}.get(shape, 0)      # mode 2: zeta = 0 Student-t core (row f4)
    if shape == "P1":
        assert out[1] == (1 if policy == 0 else 27)   # K_{1/2}: H(z) is linear in z; 27 = a-priori degree of a general order
    assert abs(out[3] / nm["NS"] - 1) <= 5e-14 and abs(out[4] / nm["NB"] - 1) <= 1e-15
    assert abs(np.sqrt(out[5]) / sc["delta"] - 1) <= 1e-14
    assert abs(out[6] / sc["alpha"] - 1) <= 1e-14 if sc["alpha"] else out[6] == 0.0
    assert abs(out[7] - sc["logG0"]) <= 1e-13 and abs(out[9] / sc["L0"] - 1) <= 1e-13 and abs(out[10] / sc["L1"] - 1) <= 1e-13
    # row f1: derivatives of the normalisations (d ln N_S / d mu, d ln N_S / d sigma, d ln N_B / d k)
    nd = orc.norm_derivs(P, LO, HI)
    assert abs(out[11] - nd[0]) <= 1e-12 * max(abs(nd[0]), 1e-3)
    assert abs(out[12] - nd[1]) <= 1e-11 * abs(nd[1]) and abs(out[13] - nd[2]) <= 1e-13 * abs(nd[2])
    assert abs(out[14] - nd[3]) <= 1e-11 * max(abs(nd[3]), 1e-2)          # d ln N_S / d beta (fifth gradient component)
    n = 4000 if shape != "direct" else 400
    x = inp.standin_masses(1, n)
    x[:5] = [LO, HI, 5280.0, 5250.0, 5310.0]
    got = np.empty_like(x)
    emu.emu_logpdf(p.ctypes.data, LO, HI, policy, x.ctypes.data, x.size, got.ctypes.data)
    assert np.abs(got - orc.logpdf(x, P, LO, HI)).max() <= 2e-14
    d = np.linspace(-300.0, 330.0, 501)
    gi = np.empty_like(d)
    emu.emu_logI(p.ctypes.data, LO, HI, d.ctypes.data, d.size, gi.ctypes.data)
    assert np.abs(gi - np.array([orc.log_I(P, v) for v in d])).max() <= 5e-14


@pytest.mark.parametrize("shape", ["GEN", "P2", "asym", "offgrid"])
def test_device_core_cells_vs_oracle(emu, orc, shape):
    """Cells of the core (prologue A1e, host build): each cell polynomial against the oracle on a dense sorted grid (the
    host 'warp' is 8 consecutive events, so nearly every group lies in one cell), the full one on the same events shuffled."""
    P, pol = {"GEN": (inp.GEN, 1), "P2": (inp.P2, 0), "asym": (dict(inp.GEN, a=0.8, a2=3.0, beta=0.02), 1),
              "offgrid": (dict(inp.GEN, mu=5281.37, sigma=13.1), 1)}[shape]
    p = inp.as_array(P)
    info = np.zeros(13, dtype=np.int32)
    emu.emu_cells(p.ctypes.data, LO, HI, pol, info.ctypes.data)
    assert info[0] == 4 and all(0 <= g <= 3 for g in info[1:5])          # Horner groups of 4: degree 4 g + 3 at most
    hb = [int(v) for v in info[5:11]]
    assert hb == sorted(hb)
    real = [v for v in hb if 0 < v < 2 ** 31 - 1]
    xb = (np.array(real, dtype=np.int64) << 32).view(np.float64)
    xl, xr = P["mu"] - P["a"] * P["sigma"], P["mu"] + P["a2"] * P["sigma"]
    assert np.all((xb > xl) & (xb < xr))
    x = np.sort(np.concatenate([np.linspace(xl - 5.0, xr + 5.0, 60000), xb, np.nextafter(xb, 0.0), np.nextafter(xb, 1e9)]))
    ref = orc.logpdf(x, P, LO, HI)
    got = np.empty_like(x)
    emu.emu_logpdf(p.ctypes.data, LO, HI, pol, x.ctypes.data, x.size, got.ctypes.data)
    assert np.abs(got - ref).max() <= 2e-14
    perm = np.random.Generator(np.random.Philox(9)).permutation(x.size)
    xp = x[perm].copy()
    got2 = np.empty_like(x)
    emu.emu_logpdf(p.ctypes.data, LO, HI, pol, xp.ctypes.data, xp.size, got2.ctypes.data)
    assert np.abs(got2 - ref[perm]).max() <= 2e-14
    assert (got[perm] != got2).any()                                       # the sorted pass did run the cell polynomials
    # analytic gradient (row f1) through the cell polynomials: value and derivative chains, four consecutive events per group
    g1, g2 = np.zeros(6), np.zeros(6)
    emu.emu_grad(p.ctypes.data, LO, HI, pol, x.ctypes.data, x.size, g1.ctypes.data)
    emu.emu_grad(p.ctypes.data, LO, HI, pol, xp.ctypes.data, xp.size, g2.ctypes.data)
    ref_n, ref_g = orc.nll_gradient(x, P, LO, HI)
    assert abs(g1[0] - ref_n) <= 1e-12 * abs(ref_n) and abs(g2[0] - ref_n) <= 1e-12 * abs(ref_n)
    tol = 1e-7 * np.maximum(np.abs(ref_g), 1.0 / np.array([inp.GRAD_SCALE[k] for k in inp.GRAD_NAMES]))   # reading D18
    assert np.all(np.abs(g1[1:] - ref_g) <= tol) and np.all(np.abs(g2[1:] - ref_g) <= tol)
    assert (g1 != g2).any()
    # no cells: degree below 16 (K_{1/2} under the adaptive policy), a core too narrow for the high-word resolution
    for Q, qpol in ((inp.GEN, 0), (dict(inp.GEN, sigma=0.02), 1), (inp.T1, 1), (dict(inp.GEN, zeta=0.2), 1)):
        emu.emu_cells(inp.as_array(Q).ctypes.data, LO, HI, qpol, info.ctypes.data)
        assert info[0] == 0


def test_device_core_cells_random_shapes(emu, orc):
    """Random shapes and ranges, among them cores that straddle a power of two (the unit of the high word of x doubles
    there): every cell polynomial against the oracle on a sorted grid that holds the boundary doubles and their neighbours."""
    rng = np.random.Generator(np.random.Philox(77))
    with_cells = 0
    for it in range(60):
        if it % 2:
            base = 2.0 ** rng.integers(-3, 14)
            sigma = base * rng.uniform(0.002, 0.02)
            mu = base + rng.uniform(-2, 2) * sigma
        else:
            base = 5280.0 * rng.choice([1.0, 1e-3, 37.0])
            mu, sigma = base * (1 + rng.uniform(-0.01, 0.01)), base / 5280.0 * rng.uniform(3, 30)
        sc = base / 5280.0
        lo, hi = mu - rng.uniform(8, 20) * sigma, mu + rng.uniform(8, 20) * sigma
        lo = lo if lo > 0 else 0.2 * mu
        P = dict(mu=mu, sigma=sigma, zeta=10 ** rng.uniform(-0.3, 1.2), beta=rng.uniform(-0.02, 0.02) / sc,
                 a=rng.uniform(0.7, 3.5), n=rng.uniform(1.1, 6), a2=rng.uniform(0.7, 3.5), n2=rng.uniform(1.1, 6),
                 f=rng.uniform(0.05, 0.95), k=rng.uniform(-0.004, 0.001) / sc)
        P["lambda"] = rng.uniform(-3, 2)
        p = inp.as_array(P)
        c, info = np.zeros(15), np.zeros(13, dtype=np.int32)
        emu.emu_consts(p.ctypes.data, lo, hi, 1, c.ctypes.data)
        emu.emu_cells(p.ctypes.data, lo, hi, 1, info.ctypes.data)
        if c[0] != 0 or info[0] == 0:
            continue
        with_cells += 1
        xl, xr = mu - P["a"] * sigma, mu + P["a2"] * sigma
        xb = (np.array([int(v) for v in info[5:11] if 0 < v < 2 ** 31 - 1], dtype=np.int64) << 32).view(np.float64)
        assert np.all((xb > xl) & (xb < xr))
        x = np.sort(np.concatenate([np.linspace(max(lo, xl - 3 * sigma), min(hi, xr + 3 * sigma), 8000), xb,
                                    np.nextafter(xb, 0.0), np.nextafter(xb, 1e300)]))
        got = np.empty_like(x)
        emu.emu_logpdf(p.ctypes.data, lo, hi, 1, x.ctypes.data, x.size, got.ctypes.data)
        assert np.abs(got - orc.logpdf(x, P, lo, hi)).max() <= 5e-14, P
    assert with_cells >= 15


def test_device_generators_vs_oracle(emu, orc):
    rng = np.random.Generator(np.random.Philox(3))
    for _ in range(200):
        seed, slot = int(rng.integers(0, 2 ** 63)), int(rng.integers(0, 2 ** 40))
        att, stream = int(rng.integers(0, 1000)), int(rng.integers(0, 5))
        u = np.empty(2)
        emu.emu_uniforms2(seed, slot, att, stream, u.ctypes.data)
        assert np.array_equal(u, orc.uniforms2(seed, slot, att, stream))
    for mean in (0.5, 5.0, 9.99, 10.0, 50.0, 3.0e4, 7.0e4, 1.0e5):
        for slot in range(300):
            assert emu.emu_poisson(1234, slot, 3, mean) == orc.poisson(1234, slot, 3, mean)


def test_gauss_legendre_table(emu):
    """The prologue's generated 16-point rule: equals Newton on P_16 and numpy's leggauss, integrates
    polynomials of degree <= 31 exactly."""
    import ctypes as C
    arr = [np.zeros(16) for _ in range(4)]
    emu.emu_gl16.restype = None
    emu.emu_gl16.argtypes = [C.c_void_p] * 4
    emu.emu_gl16(*[a.ctypes.data_as(C.c_void_p) for a in arr])
    tx, tw, nx, nw = arr
    assert np.abs(tx - nx).max() < 5e-16 and np.abs(tw - nw).max() < 5e-16
    gx, gw = np.polynomial.legendre.leggauss(16)
    assert np.abs(np.sort(tx) - gx).max() < 5e-16 and np.abs(tw[np.argsort(tx)] - gw).max() < 5e-16
    for deg in (0, 2, 30):
        assert abs((tw * tx ** deg).sum() - 2.0 / (deg + 1)) < 1e-15


def test_chebyshev_integer_table(emu):
    """The prologue's generated table of integer Chebyshev coefficients equals the three-term recurrence
    T_{j+1} = 2 t T_j - T_{j-1} evaluated in int64 (48 x 48 entries)."""
    emu.emu_cheb_table_mismatches.restype = C.c_int
    assert emu.emu_cheb_table_mismatches() == 0


@pytest.mark.parametrize("shape", ["P1", "P2", "direct", "T1", "T2"])
def test_device_gradient_math_vs_oracle(emu, orc, shape):
    """Row f1: the CUDA path's per-event gradient arithmetic (host build) against the oracle's analytic gradient."""
    P = {"P1": inp.GEN, "P2": inp.P2, "direct": dict(inp.GEN, zeta=0.2), "T1": inp.T1, "T2": inp.T2}[shape]
    p = inp.as_array(P)
    n = 3000 if shape != "direct" else 300
    for x in (inp.standin_masses(11, n), np.sort(inp.standin_masses(12, n))):      # mixed and region-uniform groups
        out = np.zeros(6)
        emu.emu_grad(p.ctypes.data, LO, HI, 1, x.ctypes.data, x.size, out.ctypes.data)
        nll, g = orc.nll_gradient(x, P, LO, HI)
        assert abs(out[0] - nll) <= 1e-12 * abs(nll)
        s = np.array([inp.GRAD_SCALE[k] for k in inp.GRAD_NAMES])
        assert np.all(np.abs(out[1:] - g) <= 1e-9 * np.maximum(np.abs(g), 1.0 / s)), (out[1:], g)


def test_device_fastmath_vs_mpmath(emu):
    """The streaming kernels' own sqrt / exp / log (csrc/ipa_fastmath.cuh, host build of the same source) against
    mpmath at 30 digits: sqrt <= 2e-16 relative, e^{-|D|} <= 3e-16 relative, log <= 2.5e-16 + 1.5e-16 |log u| absolute,
    log on [1,2] <= 2.5e-16 absolute, the fused softplus eb + log(1 + e^D) <= 2.5e-16 (1 + |eb| + |D|)."""
    import mpmath as mp
    mp.mp.dps = 30
    rng = np.random.Generator(np.random.Philox(17))
    vp = C.c_void_p

    def run(fn, *arrs):
        out = np.empty_like(arrs[0])
        getattr(emu, fn)(*[a.ctypes.data_as(vp) for a in arrs], C.c_longlong(arrs[0].size), out.ctypes.data_as(vp))
        return out
    for name in ("emu_fsqrt", "emu_fexp_negabs_t", "emu_flog_t", "emu_flog12_t", "emu_fsoftplus_add_t", "emu_flog", "emu_fexp_neg"):
        getattr(emu, name).restype = None
    q = np.concatenate([10.0 ** rng.uniform(-3, 8, 4000), [1.0, 2.0, 4.0, 83.349, 983.0, 1e-300, 1e300]])
    got = run("emu_fsqrt", q)
    assert max(abs(mp.mpf(float(g)) / mp.sqrt(mp.mpf(float(v))) - 1) for g, v in zip(got, q)) <= 2e-16
    # gradient kernel: 1/u by one third-order step, sqrt and 1/sqrt from one step (<= 2.5e-16 relative each)
    emu.emu_frcp3.restype = None
    emu.emu_fsqrt_rsqrt.restype = None
    got = run("emu_frcp3", q)
    assert max(abs(mp.mpf(float(g)) * mp.mpf(float(v)) - 1) for g, v in zip(got, q)) <= 2.5e-16
    r, ri = np.empty_like(q), np.empty_like(q)
    emu.emu_fsqrt_rsqrt(q.ctypes.data_as(vp), C.c_longlong(q.size), r.ctypes.data_as(vp), ri.ctypes.data_as(vp))
    assert max(abs(mp.mpf(float(g)) / mp.sqrt(mp.mpf(float(v))) - 1) for g, v in zip(r, q)) <= 2e-16
    assert max(abs(mp.mpf(float(g)) * mp.sqrt(mp.mpf(float(v))) - 1) for g, v in zip(ri, q)) <= 2.5e-16
    D = np.concatenate([rng.uniform(-60, 60, 6000), rng.uniform(-1, 1, 2000) * 1e-3, [0.0, -0.0, 1e-300, 700.0, -745.0, 1.0e4, -1.0e4,
                                                                                     4.9e6, np.log(2) / 512, -np.log(2) / 512]])
    got = run("emu_fexp_negabs_t", D)
    for g, v in zip(got, D):
        ref = mp.exp(-abs(mp.mpf(float(v))))
        assert abs(mp.mpf(float(g)) - ref) <= 3e-16 * ref + 1e-300, (v, g)
    u = np.concatenate([10.0 ** rng.uniform(-8, 8, 6000), 1.0 + rng.uniform(0, 1, 2000) * 2.0 ** -rng.integers(1, 40, 2000),
                        [1.0, 2.0, 0.5, 9.75, 1.0 + 2.0 ** -52, 2.0 - 2.0 ** -52, 1e-300, 1e300]])
    for fn in ("emu_flog_t", "emu_flog"):
        got = run(fn, u)
        for g, v in zip(got, u):
            ref = mp.log(mp.mpf(float(v)))
            assert abs(mp.mpf(float(g)) - ref) <= 2.5e-16 + 1.5e-16 * abs(ref), (fn, v, g)
    s = np.concatenate([1.0 + rng.uniform(0, 1, 6000), 1.0 + 10.0 ** rng.uniform(-20, 0, 2000), [1.0, 2.0, 1.5, 1.0 + 2.0 ** -52,
                                                                                             2.0 - 2.0 ** -52, 1.0 + 2.0 ** -9]])
    s = np.minimum(s, 2.0)
    got = run("emu_flog12_t", s)
    assert max(abs(mp.mpf(float(g)) - mp.log(mp.mpf(float(v)))) for g, v in zip(got, s)) <= 2.5e-16
    eb = rng.uniform(-12, -4, D.size)
    Ds = np.where(np.abs(D) > 1.3e6, np.sign(D) * 1.3e6, D)        # the softplus' own exponential: |D| < 1.4e6
    got = run("emu_fsoftplus_add_t", eb, Ds)
    for g, b, v in zip(got, eb, Ds):
        ref = mp.mpf(float(b)) + mp.log(1 + mp.exp(mp.mpf(float(v))))
        assert abs(mp.mpf(float(g)) - ref) <= 2.5e-16 * (1 + abs(b) + abs(v)), (b, v, g)      # three roundings of O(|eb| + |D|) terms
    # NaN in, NaN out; the table index of a NaN stays inside the table
    nan = np.array([np.nan])
    assert np.isnan(run("emu_flog12_t", nan)[0])           # (the general log rebuilds the mantissa: a NaN event is
    assert np.isnan(run("emu_fsoftplus_add_t", nan, nan)[0])   #  carried by E_B = k d + const, tested on the GPU)
