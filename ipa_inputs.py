"""Seeded synthetic inputs shared by the tests, bench.py and __graft_entry__.smoke().

This module holds NONE of the method's arithmetic (no Ipatia density, no Bessel function, no
likelihood): it only fixes the configuration constants of BASELINE.json / SURVEY.md 8(d) and
builds parameter batches and stand-in event arrays with numpy.  Both the oracle (oracle/) and the
CUDA path (paper_1706_01420_b200/) consume what it returns; neither is imported here.

Config-faithful datasets ("drawn by accept-reject from the Ipatia + exponential model") are
produced by the method's own toy generator (row T1): oracle.generate_mixture on the CPU side,
ipa_toy_generate on the GPU side -- two independent implementations of the same counter-based
(Philox-4x32-10) recipe, DESIGN.md "Input recipe".
"""
import numpy as np

PARAM_FIELDS = ("mu", "sigma", "lambda", "zeta", "beta", "a", "n", "a2", "n2", "f", "k")
NPAR = len(PARAM_FIELDS)
IDX = {name: i for i, name in enumerate(PARAM_FIELDS)}

LO, HI = 5000.0, 5600.0  # fit range of every config (BASELINE.json)

# generating model of every config (BASELINE.json configs[0]; lambda = zeta = 1: reading D2)
GEN = dict(mu=5280.0, sigma=15.0, **{"lambda": 1.0}, zeta=1.0, beta=0.0, a=2.0, n=3.0, a2=2.0, n2=3.0,
           f=0.3, k=-0.002)
# second, general shape point (reading D2): non-half-integer order, beta != 0, asymmetric tails
P2 = dict(mu=5280.0, sigma=15.0, **{"lambda": -1.3}, zeta=2.0, beta=0.01, a=1.5, n=2.5, a2=2.2, n2=4.0,
          f=0.3, k=-0.002)
# zeta = 0 Student-t core (row f4, reading D3): T1 has the Upsilon example's lambda = -2, T2 the
# delta = sigma branch (-1 <= lambda < 0) with beta != 0 and asymmetric tails
T1 = dict(mu=5280.0, sigma=15.0, **{"lambda": -2.0}, zeta=0.0, beta=0.0, a=2.0, n=3.0, a2=2.0, n2=3.0, f=0.3, k=-0.002)
T2 = dict(mu=5280.0, sigma=15.0, **{"lambda": -0.7}, zeta=0.0, beta=0.004, a=1.2, n=2.5, a2=1.8, n2=4.0, f=0.3, k=-0.002)

FLOATED = ("mu", "sigma", "f", "k")                   # reading C6: order of the floated parameters
FD_STEPS = dict(mu=0.01, sigma=0.01, f=1e-4, k=1e-6)  # reading C6: central-difference steps
GRAD_SCALE = dict(mu=0.3, sigma=0.3, f=0.007, k=7e-5,  # reading D18: ~1 sigma fit errors at N=1e4
                  beta=1.2e-3)                         # analytic gradient only (fifth component): 1 / (sqrt(N_sig) sigma)
GRAD_NAMES = ("mu", "sigma", "f", "k", "beta")         # components of the analytic gradient (row f1)
FIT_START_SHIFT = dict(mu=1.0, sigma=1.0, f=0.02, k=1e-4)


def as_array(p):
    """dict -> (11,) float64 in PARAM_FIELDS order."""
    return np.array([p[name] for name in PARAM_FIELDS], dtype=np.float64)


def as_dict(v):
    return {name: float(v[i]) for i, name in enumerate(PARAM_FIELDS)}


def fd_batch(theta, floated=FLOATED, steps=FD_STEPS):
    """Central-difference batch (reading C6): row 0 = theta, rows 2j+1 / 2j+2 = theta +/- h_j e_j.

    Returns (batch[(2P+1), 11], h[P]).  theta +/- h is computed ONCE here, in fp64, and the same
    array is handed to the oracle and to the CUDA path.
    """
    base = as_array(theta) if isinstance(theta, dict) else np.array(theta, dtype=np.float64)
    P = len(floated)
    batch = np.tile(base, (2 * P + 1, 1))
    h = np.array([steps[name] for name in floated], dtype=np.float64)
    for j, name in enumerate(floated):
        batch[2 * j + 1, IDX[name]] = base[IDX[name]] + h[j]
        batch[2 * j + 2, IDX[name]] = base[IDX[name]] - h[j]
    return batch, h


def fd_spec(floated=FLOATED, steps=FD_STEPS):
    """(idx[P] int32 field indices, h[P] steps) of the central-difference gradient (reading C6): the arguments of
    oracle.fd_gradient and ipa_nll_fd_gradient, which both build the batch of fd_batch() and take the differences
    themselves (row G is method code: it lives on each side, not here)."""
    return (np.array([IDX[name] for name in floated], dtype=np.int32),
            np.array([steps[name] for name in floated], dtype=np.float64))


def standin_masses(seed, n, f=0.3, mu=5280.0, sigma=15.0, k=-0.002, lo=LO, hi=HI):
    """Stand-in event array with the structure of the paper's toy data:
    a narrow heavy-tailed peak of relative weight f on a falling exponential, all inside [lo, hi].
    Peak = mu + 0.8 sigma * Student-t(4) (out-of-range draws are replaced by background draws);
    background = inverse CDF of the truncated exponential.  About 34 % of the events fall inside
    [mu-2 sigma, mu+2 sigma], as for the generating model.  Used where an input must not come from
    either implementation of the method (full-size parity at 1e8 events).
    """
    rng = np.random.Generator(np.random.Philox(int(seed)))
    n = int(n)
    u = rng.random(n)
    w = hi - lo
    x = lo + np.log1p(u * np.expm1(k * w)) / k if k != 0.0 else lo + u * w
    is_sig = rng.random(n) < f
    peak = mu + 0.8 * sigma * rng.standard_t(4, size=n)
    ok = is_sig & (peak >= lo) & (peak <= hi)
    x[ok] = peak[ok]
    return np.ascontiguousarray(x, dtype=np.float64)


def toy_seeds(T, first=1001):
    """seeds 1001 .. 1000+T."""
    return np.arange(first, first + int(T), dtype=np.uint64)


def toy_param_sets(T, seed=4, theta=GEN):
    """Config 4, 'each toy with its own parameter set' (reading D17): the generating theta with
    (mu, sigma, f, k) displaced by (0.1, 0.1, 0.002, 2e-5) x standard normals (numpy Philox stream)."""
    rng = np.random.Generator(np.random.Philox(int(seed)))
    base = as_array(theta)
    out = np.tile(base, (int(T), 1))
    z = rng.standard_normal((int(T), 4))
    for j, (name, s) in enumerate((("mu", 0.1), ("sigma", 0.1), ("f", 0.002), ("k", 2e-5))):
        out[:, IDX[name]] += s * z[:, j]
    return out


def scan_grid(n_ns=100, n_k=100, n_obs=1.0e8):
    """Config 5 grid (reading D16): ns uniform on [0, 5000] x k uniform on [-0.0025, -0.0015],
    nb = N_obs - ns.  Returns flat arrays (ns, nb, k) of n_ns*n_k points, ns-major."""
    ns = np.linspace(0.0, 5000.0, int(n_ns))
    kk = np.linspace(-0.0025, -0.0015, int(n_k))
    NS, KK = np.meshgrid(ns, kk, indexing="ij")
    NS = NS.ravel().copy()
    KK = KK.ravel().copy()
    return NS, float(n_obs) - NS, KK
