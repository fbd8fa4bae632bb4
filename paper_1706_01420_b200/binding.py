"""ctypes binding of libipanll.so: same names as include/ipanll.h, torch tensors for device memory
and streams (plumbing only).  Each wrapper marshals arguments, sizes the workspace and checks the
return code; no arithmetic of the method happens here.
"""
import ctypes as C
import functools
import os

import numpy as np
import torch

from . import build as _build

__all__ = [
    "PARAM_FIELDS", "NPAR", "IPA_MAX_K", "IpaError", "lib", "library_path", "pack_params", "workspace",
    "ipa_version", "ipa_workspace_bytes", "ipa_norm", "ipa_core_degree", "ipa_core_cells", "ipa_nll_grad_eval", "ipa_nll_fd_gradient",
    "ipa_nll_eval_extended", "ipa_nll_eval_categories", "ipa_nll_eval", "ipa_nll_eval_static", "IPA_STATIC_MAX_K", "NllEvaluator",
    "ipa_nll_eval_segmented", "ipa_toy_generate", "ipa_hist_fill", "ipa_binned_nll_scan", "ipa_expected_hist",
    "ipa_poisson_hist_toys", "ipa_signal_shape", "ipa_gauss_smear", "ipa_expected_hist_shape", "ipa_binned_nll_scan_shape",
    "ipa_cls_teststat", "ipa_cls_count_ge", "ipa_cls_from_counts", "ipa_events_prepare",
    "ipa_prepare_workspace_bytes", "ipa_fp64_peak_probe", "nll_host", "EXPORTS",
]

PARAM_FIELDS = ("mu", "sigma", "lambda", "zeta", "beta", "a", "n", "a2", "n2", "f", "k")
NPAR = len(PARAM_FIELDS)
IPA_MAX_K = 32
IPA_STATIC_MAX_K = 16        # ipa_nll_eval_static: sets per call that the built-in scratch holds

# every symbol include/ipanll.h declares
EXPORTS = (
    "ipa_strerror", "ipa_last_cuda_error", "ipa_version", "ipa_workspace_bytes",
    "ipa_norm", "ipa_core_degree", "ipa_core_cells", "ipa_nll_eval", "ipa_nll_fd_gradient", "ipa_nll_eval_extended", "ipa_nll_grad_eval", "ipa_nll_eval_segmented", "ipa_nll_eval_categories", "ipa_toy_generate", "ipa_hist_fill",
    "ipa_binned_nll_scan", "ipa_expected_hist", "ipa_poisson_hist_toys", "ipa_signal_shape", "ipa_gauss_smear",
    "ipa_expected_hist_shape", "ipa_binned_nll_scan_shape", "ipa_cls_teststat", "ipa_cls_count_ge",
    "ipa_cls_from_counts", "ipa_prepare_workspace_bytes", "ipa_events_prepare",
    "ipa_fp64_peak_probe", "ipa_nll_eval_static",
)


class IpaError(RuntimeError):
    pass


class _Range(C.Structure):
    _fields_ = [("lo", C.c_double), ("hi", C.c_double)]


class _Options(C.Structure):
    _fields_ = [("degree_policy", C.c_int32), ("reserved", C.c_int32), ("first_slot", C.c_int64)]


def _opt(policy, first_slot=0):
    """policy None -> NULL options (library defaults), else an ipa_options with that degree policy."""
    if policy is None and not first_slot:
        return None
    o = _Options()
    o.degree_policy = int(policy or 0)
    o.first_slot = int(first_slot)
    return C.byref(o)


_lib = None


def library_path():
    return _build.LIB


def lib():
    """Load (building if needed) libipanll.so.  Fails loudly if it cannot be built or loaded."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, i64, i32, d, sz = C.c_void_p, C.c_int64, C.c_int, C.c_double, C.c_size_t
    L.ipa_strerror.restype = C.c_char_p; L.ipa_strerror.argtypes = [i32]
    L.ipa_last_cuda_error.restype = C.c_char_p; L.ipa_last_cuda_error.argtypes = []
    L.ipa_version.restype = C.c_char_p; L.ipa_version.argtypes = []
    L.ipa_workspace_bytes.restype = sz; L.ipa_workspace_bytes.argtypes = [i64, i64, i64]
    op = vp  # const ipa_options* (NULL or byref(_Options))
    L.ipa_norm.restype = i32; L.ipa_norm.argtypes = [vp, i32, _Range, vp, vp, vp, op, vp, sz, vp]
    L.ipa_core_degree.restype = i32; L.ipa_core_degree.argtypes = [vp, i32, _Range, vp, op, vp, sz, vp]
    L.ipa_core_cells.restype = i32; L.ipa_core_cells.argtypes = [vp, i32, _Range, vp, op, vp, sz, vp]
    L.ipa_nll_eval.restype = i32; L.ipa_nll_eval.argtypes = [vp, i64, vp, i32, _Range, vp, vp, vp, op, vp, sz, vp]
    L.ipa_nll_eval_static.restype = i32; L.ipa_nll_eval_static.argtypes = [vp, i64, vp, i32, _Range, vp, vp, vp, op, vp]
    L.ipa_nll_fd_gradient.restype = i32
    L.ipa_nll_fd_gradient.argtypes = [vp, i64, vp, i32, vp, vp, _Range, vp, vp, vp, op, vp, sz, vp]
    L.ipa_nll_eval_extended.restype = i32
    L.ipa_nll_eval_extended.argtypes = [vp, i64, vp, vp, vp, i32, _Range, vp, vp, op, vp, sz, vp]
    L.ipa_nll_grad_eval.restype = i32; L.ipa_nll_grad_eval.argtypes = [vp, i64, vp, i32, _Range, vp, vp, vp, op, vp, sz, vp]
    L.ipa_nll_eval_segmented.restype = i32
    L.ipa_nll_eval_segmented.argtypes = [vp, vp, i64, vp, _Range, vp, vp, op, vp, sz, vp]
    L.ipa_nll_eval_categories.restype = i32
    L.ipa_nll_eval_categories.argtypes = [vp, vp, i64, vp, i64, vp, _Range, vp, vp, op, vp, sz, vp]
    L.ipa_toy_generate.restype = i32
    L.ipa_toy_generate.argtypes = [vp, i64, vp, i64, d, d, _Range, i64, vp, vp, vp, vp, op, vp, sz, vp]
    L.ipa_hist_fill.restype = i32; L.ipa_hist_fill.argtypes = [vp, i64, _Range, i32, vp, vp]
    L.ipa_binned_nll_scan.restype = i32
    L.ipa_binned_nll_scan.argtypes = [vp, i32, _Range, vp, vp, vp, vp, i64, vp, op, vp, sz, vp]
    L.ipa_expected_hist.restype = i32; L.ipa_expected_hist.argtypes = [i32, _Range, vp, d, d, d, vp, op, vp, sz, vp]
    L.ipa_poisson_hist_toys.restype = i32; L.ipa_poisson_hist_toys.argtypes = [vp, i32, vp, i64, vp, vp, sz, vp]
    L.ipa_signal_shape.restype = i32; L.ipa_signal_shape.argtypes = [i32, _Range, vp, vp, op, vp, sz, vp]
    L.ipa_gauss_smear.restype = i32; L.ipa_gauss_smear.argtypes = [vp, i32, _Range, d, vp, vp]
    L.ipa_expected_hist_shape.restype = i32; L.ipa_expected_hist_shape.argtypes = [i32, _Range, vp, d, d, d, vp, vp, sz, vp]
    L.ipa_binned_nll_scan_shape.restype = i32
    L.ipa_binned_nll_scan_shape.argtypes = [vp, i32, _Range, vp, vp, vp, vp, i64, vp, vp, sz, vp]
    L.ipa_cls_teststat.restype = i32; L.ipa_cls_teststat.argtypes = [vp, i32, i64, i32, vp, vp, vp, vp, sz, vp]
    L.ipa_cls_count_ge.restype = i32; L.ipa_cls_count_ge.argtypes = [vp, i64, vp, vp, vp]
    L.ipa_cls_from_counts.restype = i32; L.ipa_cls_from_counts.argtypes = [vp, i64, vp, i64, vp, vp]
    L.ipa_prepare_workspace_bytes.restype = sz; L.ipa_prepare_workspace_bytes.argtypes = [i64, i64]
    L.ipa_events_prepare.restype = i32; L.ipa_events_prepare.argtypes = [vp, i64, vp, i64, _Range, vp, vp, sz, vp]
    L.ipa_fp64_peak_probe.restype = i32; L.ipa_fp64_peak_probe.argtypes = [i64, vp, vp]
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        L = lib()
        msg = L.ipa_strerror(rc).decode()
        extra = L.ipa_last_cuda_error().decode()
        raise IpaError(f"libipanll: {msg} ({rc})" + (f": {extra}" if extra else ""))


def _need_cuda():
    if not torch.cuda.is_available():
        raise IpaError("libipanll needs a CUDA device (sm_100a); there is no CPU fallback")


def _alloc_on_stream(fn):
    """Run a wrapper under `with torch.cuda.stream(stream)` when a stream is given, so that the tensors it allocates
    (workspace, outputs) belong to the stream the kernels are enqueued on: the caching allocator then cannot hand
    their memory to another stream while that work is pending."""
    @functools.wraps(fn)
    def wrapped(*args, **kwargs):
        st = kwargs.get("stream")
        if st is None or not torch.cuda.is_available():
            return fn(*args, **kwargs)
        with torch.cuda.stream(st):
            return fn(*args, **kwargs)
    return wrapped


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _dptr(t, dtype=None):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device tensors must be contiguous CUDA tensors"
    if dtype is not None:
        assert t.dtype == dtype, (t.dtype, dtype)
    return C.c_void_p(t.data_ptr())


def _hptr(a):
    return a.ctypes.data_as(C.c_void_p)


def pack_params(p):
    """dict / list of dicts / (K,11) array -> contiguous (K,11) float64 numpy array."""
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


def ipa_version():
    return lib().ipa_version().decode()


def ipa_workspace_bytes(n, K, nbins=0):
    return int(lib().ipa_workspace_bytes(int(n), int(K), int(nbins)))


def workspace(n, K, nbins=0, device="cuda"):
    """Allocate a workspace tensor (uint8) large enough for the given sizes."""
    _need_cuda()
    return torch.empty(ipa_workspace_bytes(n, K, nbins), dtype=torch.uint8, device=device)


def _ws(ws, n, K, nbins=0):
    if ws is None:
        ws = workspace(n, K, nbins)
    return ws


@_alloc_on_stream
def ipa_norm(params, lo, hi, ws=None, stream=None, out=None, policy=None):
    """-> (norm_sig[K], norm_bkg[K], status[K]) device tensors (out = the same triple, preallocated)."""
    _need_cuda()
    P = pack_params(params)
    K = P.shape[0]
    ws = _ws(ws, 0, K)
    if out is not None:
        ns, nb, st = out
    else:
        ns = torch.empty(K, dtype=torch.float64, device="cuda")
        nb = torch.empty(K, dtype=torch.float64, device="cuda")
        st = torch.empty(K, dtype=torch.int32, device="cuda")
    _check(lib().ipa_norm(_hptr(P), K, _Range(lo, hi), _dptr(ns), _dptr(nb), _dptr(st), _opt(policy), _dptr(ws), ws.numel(),
                          _stream(stream)))
    return ns, nb, st


@_alloc_on_stream
def ipa_core_degree(params, lo, hi, ws=None, stream=None, policy=None):
    """Degree of the core approximant per set (-1 direct mode, -2 domain error); int for a single set."""
    _need_cuda()
    P = pack_params(params)
    K = P.shape[0]
    ws = _ws(ws, 0, K)
    out = torch.empty(K, dtype=torch.int32, device="cuda")
    _check(lib().ipa_core_degree(_hptr(P), K, _Range(lo, hi), _dptr(out), _opt(policy), _dptr(ws), ws.numel(), _stream(stream)))
    r = out.cpu().numpy()
    return int(r[0]) if K == 1 else r


def ipa_core_cells(params, lo, hi, ws=None, stream=None, policy=None):
    """Cells of the core per set: int32 array [K, 13] = (ncell, 4 degrees, 6 boundary high words, 2 pads); [13] for one set."""
    _need_cuda()
    P = pack_params(params)
    K = P.shape[0]
    ws = _ws(ws, 0, K)
    out = torch.empty((K, 13), dtype=torch.int32, device="cuda")
    _check(lib().ipa_core_cells(_hptr(P), K, _Range(lo, hi), _dptr(out), _opt(policy), _dptr(ws), ws.numel(), _stream(stream)))
    r = out.cpu().numpy()
    return r[0] if K == 1 else r


@_alloc_on_stream
def ipa_nll_eval(x, params, lo, hi, want_logpdf=False, ws=None, stream=None, out=None, status=None, policy=None):
    """NLL of the events in device tensor x (fp64) for K parameter sets.

    -> (nll[K], logpdf[K,n] or None, status[K]) device tensors; nothing is synchronised.
    """
    _need_cuda()
    P = pack_params(params)
    K = P.shape[0]
    n = x.numel()
    ws = _ws(ws, n, K)
    nll = out if out is not None else torch.empty(K, dtype=torch.float64, device="cuda")
    st = status if status is not None else torch.empty(K, dtype=torch.int32, device="cuda")
    lp = torch.empty((K, n), dtype=torch.float64, device="cuda") if want_logpdf else None
    _check(lib().ipa_nll_eval(_dptr(x, torch.float64) if n else None, n, _hptr(P), K, _Range(lo, hi), _dptr(nll),
                              _dptr(lp), _dptr(st), _opt(policy), _dptr(ws), ws.numel(), _stream(stream)))
    return nll, lp, st


@_alloc_on_stream
def ipa_nll_eval_static(x, params, lo, hi, want_logpdf=False, stream=None, out=None, status=None, policy=None):
    """ipa_nll_eval on the library's built-in scratch (no workspace): K <= IPA_STATIC_MAX_K sets.  The C entry point
    allocates nothing; pass `out` [K] float64 and `status` [K] int32 device tensors to keep this wrapper from allocating too.
    Calls share the scratch: calls that overlap on the GPU race.  -> (nll[K], logpdf[K,n] or None, status[K])."""
    _need_cuda()
    P = pack_params(params)
    K = P.shape[0]
    n = x.numel()
    nll = out if out is not None else torch.empty(K, dtype=torch.float64, device="cuda")
    st = status if status is not None else torch.empty(K, dtype=torch.int32, device="cuda")
    lp = torch.empty((K, n), dtype=torch.float64, device="cuda") if (want_logpdf and K <= IPA_STATIC_MAX_K) else None
    _check(lib().ipa_nll_eval_static(_dptr(x, torch.float64) if n else None, n, _hptr(P), K, _Range(lo, hi), _dptr(nll),
                                     _dptr(lp), _dptr(st), _opt(policy), _stream(stream)))
    return nll, lp, st


_cudart = None


def _runtime():
    """The CUDA runtime libipanll.so itself is linked against (already loaded: looked up by its soname)."""
    global _cudart
    if _cudart is None:
        lib()
        R = C.CDLL("libcudart.so.12")
        R.cudaMemcpyAsync.restype = C.c_int
        R.cudaMemcpyAsync.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_int, C.c_void_p]
        R.cudaStreamSynchronize.restype = C.c_int
        R.cudaStreamSynchronize.argtypes = [C.c_void_p]
        _cudart = R
    return _cudart


class NllEvaluator:
    """The inner loop of a fit: many ipa_nll_eval / ipa_nll_grad_eval calls on ONE event array, each followed by a read of
    the K results on the host.  Workspace, device outputs and a pinned host buffer are allocated once; a call packs the
    parameter sets, enqueues the library call and one device-to-host copy of the results on the stream, and waits for
    that stream.  Argument marshalling only: the arithmetic is the library's.

        ev = NllEvaluator(x, lo, hi)            # x: device tensor (fp64), stays alive and unchanged
        nll = ev(thetas)                        # numpy [K]; +inf for a set with a domain error
        nll, grad = ev.gradient(thetas)         # numpy [K], [K, 5]  (mu, sigma, f, k, beta)
    """

    def __init__(self, x, lo, hi, policy=None, stream=None):
        _need_cuda()
        assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
        self.x, self.n = x, x.numel()
        self.range = _Range(lo, hi)
        self.opt = _opt(policy)
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self._st = C.c_void_p(self.stream.cuda_stream)
        with torch.cuda.stream(self.stream):
            self.ws = workspace(self.n, IPA_MAX_K)
            self.dev = torch.empty(IPA_MAX_K * 7, dtype=torch.float64, device="cuda")   # nll [K] | grad [K, 5] | status
        self.host = torch.empty(IPA_MAX_K * 7, dtype=torch.float64).pin_memory()
        self._hnp = self.host.numpy()
        self._hst = self._hnp[IPA_MAX_K * 6:].view(np.int32)
        base = self.dev.data_ptr()
        self._xp = C.c_void_p(x.data_ptr()) if self.n else None
        self._nll = C.c_void_p(base)
        self._grad = C.c_void_p(base + 8 * IPA_MAX_K)
        self._status = C.c_void_p(base + 48 * IPA_MAX_K)
        self._wsp, self._wsn = C.c_void_p(self.ws.data_ptr()), self.ws.numel()
        self._devp, self._hostp = C.c_void_p(base), C.c_void_p(self.host.data_ptr())
        self._lib, self._rt = lib(), _runtime()

    def _read(self):
        rc = self._rt.cudaMemcpyAsync(self._hostp, self._devp, IPA_MAX_K * 56, 2, self._st)       # 2 = device to host
        rc = rc or self._rt.cudaStreamSynchronize(self._st)
        if rc:
            raise IpaError(f"CUDA runtime error {rc} while reading the results")

    def __call__(self, params):
        P = pack_params(params)
        K = P.shape[0]
        _check(self._lib.ipa_nll_eval(self._xp, self.n, _hptr(P), K, self.range, self._nll, None, self._status, self.opt,
                                      self._wsp, self._wsn, self._st))
        self._read()
        return self._hnp[:K].copy()

    def gradient(self, params):
        P = pack_params(params)
        K = P.shape[0]
        _check(self._lib.ipa_nll_grad_eval(self._xp, self.n, _hptr(P), K, self.range, self._nll, self._grad, self._status,
                                           self.opt, self._wsp, self._wsn, self._st))
        self._read()
        return self._hnp[:K].copy(), self._hnp[IPA_MAX_K:IPA_MAX_K + 5 * K].reshape(K, 5).copy()

    def status(self, K):
        """status codes of the K sets of the last call"""
        return self._hst[:K].copy()


@_alloc_on_stream
def ipa_nll_fd_gradient(x, theta, idx, h, lo, hi, ws=None, stream=None, policy=None):
    """Central-difference gradient from ONE K = 2P+1 pass (row G, reading C6): idx[P] parameter-field indices, h[P] steps.
    -> (nll[2P+1], grad[P], status[2P+1]) device tensors."""
    _need_cuda()
    P = pack_params(theta)
    assert P.shape[0] == 1
    idx = np.ascontiguousarray(idx, dtype=np.int32).ravel()
    h = np.ascontiguousarray(h, dtype=np.float64).ravel()
    assert idx.size == h.size
    n = x.numel()
    K = 2 * idx.size + 1
    ws = _ws(ws, n, K)
    nll = torch.empty(K, dtype=torch.float64, device="cuda")
    grad = torch.empty(idx.size, dtype=torch.float64, device="cuda")
    st = torch.empty(K, dtype=torch.int32, device="cuda")
    _check(lib().ipa_nll_fd_gradient(_dptr(x, torch.float64) if n else None, n, _hptr(P), idx.size, _hptr(idx), _hptr(h),
                                     _Range(lo, hi), _dptr(nll), _dptr(grad), _dptr(st), _opt(policy), _dptr(ws), ws.numel(),
                                     _stream(stream)))
    return nll, grad, st


@_alloc_on_stream
def ipa_nll_eval_extended(x, params, ns, nb, lo, hi, ws=None, stream=None, policy=None):
    """Extended -log L = (ns+nb) - sum log(ns S + nb B) for K (shape, ns, nb) triples -> (nll[K], status[K])."""
    _need_cuda()
    P = pack_params(params)
    K = P.shape[0]
    ns = np.ascontiguousarray(np.broadcast_to(np.asarray(ns, dtype=np.float64), (K,)))
    nb = np.ascontiguousarray(np.broadcast_to(np.asarray(nb, dtype=np.float64), (K,)))
    n = x.numel()
    ws = _ws(ws, n, K)
    nll = torch.empty(K, dtype=torch.float64, device="cuda")
    st = torch.empty(K, dtype=torch.int32, device="cuda")
    _check(lib().ipa_nll_eval_extended(_dptr(x, torch.float64) if n else None, n, _hptr(P), _hptr(ns), _hptr(nb), K,
                                       _Range(lo, hi), _dptr(nll), _dptr(st), _opt(policy), _dptr(ws), ws.numel(), _stream(stream)))
    return nll, st


@_alloc_on_stream
def ipa_nll_grad_eval(x, params, lo, hi, ws=None, stream=None, policy=None):
    """NLL and analytic gradient w.r.t. (mu, sigma, f, k, beta): -> (nll[K], grad[K, 5], status[K]) device tensors."""
    _need_cuda()
    P = pack_params(params)
    K = P.shape[0]
    n = x.numel()
    ws = _ws(ws, n, K)
    nll = torch.empty(K, dtype=torch.float64, device="cuda")
    grad = torch.empty((K, 5), dtype=torch.float64, device="cuda")
    st = torch.empty(K, dtype=torch.int32, device="cuda")
    _check(lib().ipa_nll_grad_eval(_dptr(x, torch.float64) if n else None, n, _hptr(P), K, _Range(lo, hi), _dptr(nll),
                                   _dptr(grad), _dptr(st), _opt(policy), _dptr(ws), ws.numel(), _stream(stream)))
    return nll, grad, st


@_alloc_on_stream
def ipa_nll_eval_segmented(x, offsets, params, lo, hi, ws=None, stream=None, policy=None):
    """-> (nll[T], status[T]); offsets is an int64 device tensor [T+1]."""
    _need_cuda()
    P = pack_params(params)
    T = offsets.numel() - 1
    assert P.shape[0] == T
    ws = _ws(ws, x.numel(), T)
    nll = torch.empty(T, dtype=torch.float64, device="cuda")
    st = torch.empty(T, dtype=torch.int32, device="cuda")
    _check(lib().ipa_nll_eval_segmented(_dptr(x, torch.float64), _dptr(offsets, torch.int64), T, _hptr(P),
                                        _Range(lo, hi), _dptr(nll), _dptr(st), _opt(policy), _dptr(ws), ws.numel(), _stream(stream)))
    return nll, st


@_alloc_on_stream
def ipa_nll_eval_categories(x, offsets, params, set_of_segment, lo, hi, ws=None, stream=None, policy=None):
    """Segments (categories) sharing parameter sets: segment t uses params[set_of_segment[t]] -> (nll[T], status[T])."""
    _need_cuda()
    P = pack_params(params)
    T = offsets.numel() - 1
    m = np.ascontiguousarray(set_of_segment, dtype=np.int32).ravel()
    assert m.size == T
    ws = _ws(ws, x.numel(), max(T, P.shape[0]))
    nll = torch.empty(T, dtype=torch.float64, device="cuda")
    st = torch.empty(T, dtype=torch.int32, device="cuda")
    _check(lib().ipa_nll_eval_categories(_dptr(x, torch.float64), _dptr(offsets, torch.int64), T, _hptr(P), P.shape[0],
                                         _hptr(m), _Range(lo, hi), _dptr(nll), _dptr(st), _opt(policy), _dptr(ws), ws.numel(),
                                         _stream(stream)))
    return nll, st


@_alloc_on_stream
def ipa_toy_generate(seeds, gen, mean_sig, mean_bkg, lo, hi, capacity, ws=None, stream=None, x=None, policy=None,
                     status=None, first_slot=0):
    """Toy generation.  mean_sig < 0 selects mixture mode (one toy of exactly `capacity` events: the slots
    first_slot .. first_slot + capacity - 1 of the seeded dataset).

    -> (x[capacity], offsets[T+1] int64, overflow[1] int32) device tensors; `status` (int32 [gen_count], optional)
    receives the domain status of the generating sets."""
    _need_cuda()
    seeds = np.ascontiguousarray(seeds, dtype=np.uint64).ravel()
    T = seeds.size
    P = pack_params(gen)
    ws = _ws(ws, capacity, T)
    if x is None:
        x = torch.empty(int(capacity), dtype=torch.float64, device="cuda")
    off = torch.empty(T + 1, dtype=torch.int64, device="cuda")
    ovf = torch.zeros(1, dtype=torch.int32, device="cuda")
    _check(lib().ipa_toy_generate(_hptr(seeds), T, _hptr(P), P.shape[0], float(mean_sig), float(mean_bkg),
                                  _Range(lo, hi), int(capacity), _dptr(x) if capacity else None, _dptr(off), _dptr(ovf),
                                  _dptr(status, torch.int32), _opt(policy, first_slot), _dptr(ws), ws.numel(), _stream(stream)))
    return x, off, ovf


@_alloc_on_stream
def ipa_hist_fill(x, lo, hi, nbins, stream=None):
    _need_cuda()
    counts = torch.empty(int(nbins), dtype=torch.int64, device="cuda")  # uint64 payload
    n = x.numel()
    _check(lib().ipa_hist_fill(_dptr(x, torch.float64) if n else None, n, _Range(lo, hi), int(nbins), _dptr(counts),
                               _stream(stream)))
    return counts


@_alloc_on_stream
def _pack_points(ns, nb, k):
    """The three scan-point arrays back to back in one host buffer: the library then uploads them with one copy."""
    ns = np.asarray(ns, dtype=np.float64).ravel()
    buf = np.empty((3, ns.size), dtype=np.float64)
    buf[0], buf[1], buf[2] = ns, np.asarray(nb, dtype=np.float64).ravel(), np.asarray(k, dtype=np.float64).ravel()
    return buf[0], buf[1], buf[2]


def ipa_binned_nll_scan(counts, lo, hi, shape, ns, nb, k, ws=None, stream=None, policy=None):
    _need_cuda()
    P = pack_params(shape)
    ns, nb, k = _pack_points(ns, nb, k)
    npts, nbins = ns.size, counts.numel()
    ws = _ws(ws, 0, npts, nbins)
    out = torch.empty(npts, dtype=torch.float64, device="cuda")
    _check(lib().ipa_binned_nll_scan(_dptr(counts, torch.int64), nbins, _Range(lo, hi), _hptr(P), _hptr(ns), _hptr(nb),
                                     _hptr(k), npts, _dptr(out), _opt(policy), _dptr(ws), ws.numel(), _stream(stream)))
    return out


@_alloc_on_stream
def ipa_expected_hist(nbins, lo, hi, shape, ns, nb, k, ws=None, stream=None, policy=None):
    _need_cuda()
    P = pack_params(shape)
    ws = _ws(ws, 0, 1, nbins)
    out = torch.empty(int(nbins), dtype=torch.float64, device="cuda")
    _check(lib().ipa_expected_hist(int(nbins), _Range(lo, hi), _hptr(P), float(ns), float(nb), float(k), _dptr(out),
                                   _opt(policy), _dptr(ws), ws.numel(), _stream(stream)))
    return out


@_alloc_on_stream
def ipa_poisson_hist_toys(mean, seeds, ws=None, stream=None):
    _need_cuda()
    seeds = np.ascontiguousarray(seeds, dtype=np.uint64).ravel()
    T, nbins = seeds.size, mean.numel()
    ws = _ws(ws, 0, T)
    out = torch.empty((T, nbins), dtype=torch.int32, device="cuda")  # uint32 payload
    _check(lib().ipa_poisson_hist_toys(_dptr(mean, torch.float64), nbins, _hptr(seeds), T, _dptr(out), _dptr(ws),
                                       ws.numel(), _stream(stream)))
    return out


@_alloc_on_stream
def ipa_signal_shape(nbins, lo, hi, shape, ws=None, stream=None, policy=None):
    """Un-normalised signal shape at the bin centres (device tensor [nbins])."""
    _need_cuda()
    P = pack_params(shape)
    ws = _ws(ws, 0, 1, nbins)
    out = torch.empty(int(nbins), dtype=torch.float64, device="cuda")
    _check(lib().ipa_signal_shape(int(nbins), _Range(lo, hi), _hptr(P), _dptr(out), _opt(policy), _dptr(ws), ws.numel(),
                                  _stream(stream)))
    return out


@_alloc_on_stream
def ipa_gauss_smear(sig, lo, hi, sigma0, stream=None):
    """Gaussian smearing of a shape on the bin grid (reading F3) -> new device tensor."""
    _need_cuda()
    out = torch.empty_like(sig)
    _check(lib().ipa_gauss_smear(_dptr(sig, torch.float64), sig.numel(), _Range(lo, hi), float(sigma0), _dptr(out),
                                 _stream(stream)))
    return out


@_alloc_on_stream
def ipa_expected_hist_shape(sig, lo, hi, ns, nb, k, ws=None, stream=None):
    _need_cuda()
    nbins = sig.numel()
    ws = _ws(ws, 0, 1, nbins)
    out = torch.empty(nbins, dtype=torch.float64, device="cuda")
    _check(lib().ipa_expected_hist_shape(nbins, _Range(lo, hi), _dptr(sig, torch.float64), float(ns), float(nb), float(k),
                                         _dptr(out), _dptr(ws), ws.numel(), _stream(stream)))
    return out


@_alloc_on_stream
def ipa_binned_nll_scan_shape(counts, lo, hi, sig, ns, nb, k, ws=None, stream=None):
    _need_cuda()
    ns, nb, k = _pack_points(ns, nb, k)
    npts, nbins = ns.size, counts.numel()
    ws = _ws(ws, 0, npts, nbins)
    out = torch.empty(npts, dtype=torch.float64, device="cuda")
    _check(lib().ipa_binned_nll_scan_shape(_dptr(counts, torch.int64), nbins, _Range(lo, hi), _dptr(sig, torch.float64),
                                           _hptr(ns), _hptr(nb), _hptr(k), npts, _dptr(out), _dptr(ws), ws.numel(),
                                           _stream(stream)))
    return out


@_alloc_on_stream
def ipa_cls_teststat(counts, nu_sb, nu_b, ws=None, stream=None):
    """q[T] of T histograms counts[T, nbins] (int32 payload = uint32 toys, int64 payload = uint64 data)."""
    _need_cuda()
    nbins = nu_b.numel()
    assert counts.dtype in (torch.int32, torch.int64) and counts.numel() % nbins == 0
    T = counts.numel() // nbins
    ws = _ws(ws, 0, 1, nbins)
    q = torch.empty(T, dtype=torch.float64, device="cuda")
    _check(lib().ipa_cls_teststat(_dptr(counts), counts.element_size(), T, nbins, _dptr(nu_sb, torch.float64),
                                  _dptr(nu_b, torch.float64), _dptr(q), _dptr(ws), ws.numel(), _stream(stream)))
    return q


@_alloc_on_stream
def ipa_cls_count_ge(q, q_obs, stream=None):
    """-> int64 device tensor [1]: number of q >= q_obs[0] (q_obs a device tensor)."""
    _need_cuda()
    out = torch.empty(1, dtype=torch.int64, device="cuda")
    _check(lib().ipa_cls_count_ge(_dptr(q, torch.float64), q.numel(), _dptr(q_obs, torch.float64), _dptr(out), _stream(stream)))
    return out


@_alloc_on_stream
def ipa_cls_from_counts(count_sb, T_sb, count_b, T_b, stream=None):
    """-> device tensor [CL_sb, CL_b, CL_s]."""
    _need_cuda()
    out = torch.empty(3, dtype=torch.float64, device="cuda")
    _check(lib().ipa_cls_from_counts(_dptr(count_sb, torch.int64), int(T_sb), _dptr(count_b, torch.int64), int(T_b),
                                     _dptr(out), _stream(stream)))
    return out


def ipa_prepare_workspace_bytes(n, T=0):
    return int(lib().ipa_prepare_workspace_bytes(int(n), int(T)))


@_alloc_on_stream
def ipa_events_prepare(x, lo, hi, offsets=None, stream=None, out=None, ws=None):
    """One-off preparation: stable counting sort of the events on the coarse bin index (inside each segment if
    offsets is given).  -> new device tensor (or `out`); x is left untouched."""
    _need_cuda()
    n = x.numel()
    T = offsets.numel() - 1 if offsets is not None else 0
    if out is None:
        out = torch.empty_like(x)
    if ws is None:
        ws = torch.empty(max(256, ipa_prepare_workspace_bytes(n, T)), dtype=torch.uint8, device="cuda")
    _check(lib().ipa_events_prepare(_dptr(x, torch.float64) if n else None, n, _dptr(offsets, torch.int64), T, _Range(lo, hi),
                                    _dptr(out) if n else None, _dptr(ws), ws.numel(), _stream(stream)))
    return out


@_alloc_on_stream
def ipa_fp64_peak_probe(iters, stream=None):
    _need_cuda()
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    _check(lib().ipa_fp64_peak_probe(int(iters), _dptr(out), _stream(stream)))
    return out


_copy_stream = None


def nll_host(x_host, params, lo, hi, x_dev=None, ws=None, policy=None, chunks=8):
    """End-to-end convenience used by bench.py's e2e leg: host (pinned) events in, host NLL out.
    The events travel host -> device in `chunks` pieces on a copy stream while ipa_nll_eval runs on the pieces already
    there (the copy, not the arithmetic, bounds this path: 800 MB at PCIe speed against 0.6 ms of kernel); the K partial
    sums of the pieces are added in order (plumbing, as in sharding.combine_nll), copied back, and the call synchronises."""
    global _copy_stream
    _need_cuda()
    n = x_host.numel()
    if x_dev is None:
        x_dev = torch.empty(n, dtype=torch.float64, device="cuda")
    if chunks <= 1 or n < (1 << 22):
        x_dev.copy_(x_host, non_blocking=True)
        nll, _, _ = ipa_nll_eval(x_dev, params, lo, hi, ws=ws, policy=policy)
        return nll.cpu()
    if _copy_stream is None:
        _copy_stream = torch.cuda.Stream()
    cur = torch.cuda.current_stream()
    K = pack_params(params).shape[0]
    ws = _ws(ws, n, K)
    parts = torch.empty((chunks, K), dtype=torch.float64, device="cuda")
    edges = [((n * c // chunks) // 2) * 2 for c in range(chunks)] + [n]      # even starts keep the pieces 16-byte aligned
    _copy_stream.wait_stream(cur)
    for c in range(chunks):
        a, b = edges[c], edges[c + 1]
        with torch.cuda.stream(_copy_stream):
            x_dev[a:b].copy_(x_host[a:b], non_blocking=True)
            ev = torch.cuda.Event()
            ev.record(_copy_stream)
        cur.wait_event(ev)
        ipa_nll_eval(x_dev[a:b], params, lo, hi, ws=ws, out=parts[c], policy=policy)
    total = parts[0].clone()
    for c in range(1, chunks):
        total += parts[c]
    return total.cpu()
