"""Host-side minimiser loop of the fit (harness, BASELINE.json config 2).

The paper hands its FCN to iminuit's MIGRAD; iminuit is not in this image, so
this is a small variable-metric minimiser in the same spirit: finite-difference gradients, a BFGS
update of the inverse Hessian, and EDM = g^T V g / 2 as the convergence measure, finished by Newton
steps on a finite-difference Hessian.  It holds NO arithmetic of the likelihood: it only calls

    nll_batch(thetas[K, 11]) -> nll[K]

which is `ipa_nll_eval` on the GPU (one K-batch per call: the 2P+1 central-difference points, or all
trial points of a line search, cost one pass over the events) or the oracle in the tests.  The same
code, start point, steps and tolerances drive both, so the two fits can be compared parameter by
parameter.
"""
import numpy as np

PARAM_FIELDS = ("mu", "sigma", "lambda", "zeta", "beta", "a", "n", "a2", "n2", "f", "k")
IDX = {name: i for i, name in enumerate(PARAM_FIELDS)}


class FitResult(dict):
    __getattr__ = dict.get


def _batched(nll_batch, thetas, max_k):
    thetas = np.ascontiguousarray(thetas, dtype=np.float64)
    out = np.empty(thetas.shape[0])
    for s in range(0, thetas.shape[0], max_k):
        out[s:s + max_k] = np.asarray(nll_batch(thetas[s:s + max_k]), dtype=np.float64)
    return out


def minimise(nll_batch, theta0, floated, steps, scale, max_k=32, edm_tol=1e-9, max_iter=60, newton_iter=4,
             grad_batch=None):
    """Minimise NLL over the `floated` parameters.

    grad_batch(thetas[K, 11]) -> (nll[K], grad[K, P]) (optional): analytic gradient with respect to the floated
    parameters in their order (`ipa_nll_grad_eval` for (mu, sigma, f, k)).  When given, gradients come from it
    (one call per point instead of a 2P+1 batch) and the Newton finish differences the analytic gradient.

    theta0   (11,) start values (fixed parameters stay at these values)
    steps    {name: h}: central-difference step per floated parameter (reading C6)
    scale    {name: s}: expected size of a 1-sigma error; internal coordinates are theta / s
    Returns FitResult(theta, par{name}, errors{name}, cov, nll, edm, n_calls, n_evals, iterations).
    """
    theta0 = np.array(theta0, dtype=np.float64)
    P = len(floated)
    idx = np.array([IDX[n] for n in floated])
    h = np.array([steps[n] for n in floated], dtype=np.float64)
    s = np.array([scale[n] for n in floated], dtype=np.float64)
    counters = {"calls": 0, "evals": 0}

    def evaluate(points):  # points: (m, P) values of the floated parameters
        th = np.tile(theta0, (points.shape[0], 1))
        th[:, idx] = points
        counters["calls"] += (points.shape[0] + max_k - 1) // max_k
        counters["evals"] += points.shape[0]
        v = _batched(nll_batch, th, max_k)
        return np.where(np.isfinite(v), v, np.inf)

    def fd_batch(p):  # row 0 = p, rows 2j+1 / 2j+2 = p +/- h_j e_j  (same layout as ipa_inputs.fd_batch)
        pts = np.tile(p, (2 * P + 1, 1))
        for j in range(P):
            pts[2 * j + 1, j] = p[j] + h[j]
            pts[2 * j + 2, j] = p[j] - h[j]
        return pts

    def gradients(points):  # analytic: (m, P) points -> nll[m], grad[m, P]
        th = np.tile(theta0, (points.shape[0], 1))
        th[:, idx] = points
        counters["calls"] += 1
        counters["evals"] += points.shape[0]
        v, g = grad_batch(th)
        return np.asarray(v, dtype=np.float64), np.asarray(g, dtype=np.float64)

    def value_gradient(p):
        if grad_batch is not None:
            v, g = gradients(p[None, :])
            return v[0], g[0], np.zeros(P)          # no second derivatives: the metric starts from `scale`
        v = evaluate(fd_batch(p))
        g = (v[1::2] - v[2::2]) / (2.0 * h)
        d2 = (v[1::2] + v[2::2] - 2.0 * v[0]) / (h * h)
        return v[0], g, d2

    p = theta0[idx].copy()
    f0, g, d2 = value_gradient(p)
    # internal coordinates u = p / s: gradient gu = g s, inverse Hessian Vu
    Vu = np.diag(np.where(d2 > 0, 1.0 / np.maximum(d2 * s * s, 1e-300), 1.0))
    edm = np.inf
    it = 0
    trial = np.array([1.0, 0.5, 2.0, 0.25, 0.1, 4.0, 0.03])
    for it in range(1, max_iter + 1):
        gu = g * s
        edm = 0.5 * gu @ Vu @ gu
        if edm < 1e-5:           # close enough for the Newton finish
            break
        du = -Vu @ gu
        if gu @ du >= 0:         # not a descent direction: reset the metric
            Vu = np.diag(np.where(d2 > 0, 1.0 / np.maximum(d2 * s * s, 1e-300), 1.0))
            du = -Vu @ gu
        # line search: all trial step lengths in one batch
        pts = p[None, :] + trial[:, None] * (du * s)[None, :]
        vals = evaluate(pts)
        best = int(np.argmin(vals))
        if not vals[best] < f0:
            trial_small = np.array([0.01, 0.003, 0.001, 3e-4, 1e-4])
            pts = p[None, :] + trial_small[:, None] * (du * s)[None, :]
            vals = evaluate(pts)
            best = int(np.argmin(vals))
            if not vals[best] < f0:
                break
        p_new = pts[best]
        f_new, g_new, d2 = value_gradient(p_new)
        # BFGS update of the inverse Hessian in internal coordinates
        su = (p_new - p) / s
        yu = (g_new - g) * s
        sy = su @ yu
        if sy > 1e-12 * np.linalg.norm(su) * np.linalg.norm(yu):
            I = np.eye(P)
            A = I - np.outer(su, yu) / sy
            Vu = A @ Vu @ A.T + np.outer(su, su) / sy
        p, f0, g = p_new, f_new, g_new

    # Newton finish on a finite-difference Hessian (central second differences, one batch per iteration)
    H = None
    for _ in range(newton_iter if grad_batch is None else 0):
        pts = [fd_batch(p)]
        pairs = [(i, j) for i in range(P) for j in range(i + 1, P)]
        for (i, j) in pairs:
            for si, sj in ((1, 1), (1, -1), (-1, 1), (-1, -1)):
                q = p.copy()
                q[i] += si * h[i]
                q[j] += sj * h[j]
                pts.append(q[None, :])
        v = evaluate(np.vstack(pts))
        f0 = v[0]
        g = (v[1:2 * P + 1:2] - v[2:2 * P + 1:2]) / (2.0 * h)
        H = np.diag((v[1:2 * P + 1:2] + v[2:2 * P + 1:2] - 2.0 * v[0]) / (h * h))
        off = 2 * P + 1
        for n_, (i, j) in enumerate(pairs):
            pp, pm, mp, mm = v[off + 4 * n_: off + 4 * n_ + 4]
            H[i, j] = H[j, i] = (pp - pm - mp + mm) / (4.0 * h[i] * h[j])
        try:
            step = -np.linalg.solve(H, g)
        except np.linalg.LinAlgError:
            break
        gu = g * s
        Hu_inv = np.linalg.inv(H * np.outer(s, s))
        edm = 0.5 * gu @ Hu_inv @ gu
        if not np.all(np.isfinite(step)):
            break
        p = p + step
        if edm < edm_tol and np.all(np.abs(step) < 1e-6 * s):
            break
    for _ in range(newton_iter if grad_batch is not None else 0):
        # Hessian column j = central difference of the analytic gradient along parameter j: 2P + 1 points, one call
        pts = fd_batch(p)
        v, gg = gradients(pts)
        f0, g = v[0], gg[0]
        H = np.empty((P, P))
        for j in range(P):
            H[:, j] = (gg[2 * j + 1] - gg[2 * j + 2]) / (2.0 * h[j])
        H = 0.5 * (H + H.T)
        try:
            step = -np.linalg.solve(H, g)
        except np.linalg.LinAlgError:
            break
        gu = g * s
        edm = 0.5 * gu @ np.linalg.inv(H * np.outer(s, s)) @ gu
        if not np.all(np.isfinite(step)):
            break
        p = p + step
        if edm < edm_tol and np.all(np.abs(step) < 1e-6 * s):
            break
    f_final = evaluate(p[None, :])[0]
    theta = theta0.copy()
    theta[idx] = p
    cov = np.linalg.inv(H) if H is not None else Vu * np.outer(s, s)
    return FitResult(theta=theta, par={n: float(p[j]) for j, n in enumerate(floated)},
                     errors={n: float(np.sqrt(abs(cov[j, j]))) for j, n in enumerate(floated)}, cov=cov,
                     nll=float(f_final), edm=float(edm), n_calls=counters["calls"], n_evals=counters["evals"],
                     iterations=it)
