/*
 * ipanll.h -- C ABI of libipanll.so: the B200 (sm_100a) hot path of the unbinned maximum-likelihood
 * fit of arXiv:1706.01420 ("Ipanema-beta"), Example 1: the negative log-likelihood
 *
 *      NLL(theta) = - sum_i log( f S(x_i; theta) + (1-f) B(x_i; theta) )
 *
 * of an Ipatia signal S (generalised-hyperbolic Bessel-K core with two power-law tails; the paper only
 * names it -- `__device__ double log_apIpatia`, PAPER.md:54 -- and cites its ref. [10], PAPER.md:450;
 * the definition used here is DESIGN.md reading C1) plus an exponential background B,
 * each normalised over the fit range, evaluated for a batch of K parameter sets per
 * pass over the events; plus the toy-MC generators and the binned Poisson
 * variant that feed the same likelihood.
 *
 * Conventions common to every entry point
 *   - `*_dev` pointers are CUDA device pointers, `*_host` pointers are host pointers.  The caller owns
 *     every buffer.  The library never allocates or frees device memory and never synchronises: all
 *     work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *     stream) and results are valid once the caller has synchronised that stream.  `*_host` parameter
 *     sets of up to IPA_MAX_K entries travel in the kernel-parameter space and may be reused as soon as
 *     the call returns.  Larger host arrays (more than IPA_MAX_K sets, toy seeds, scan points) are
 *     uploaded with cudaMemcpyAsync: a pageable array is staged before the call returns and may be reused
 *     immediately, a PINNED array must stay unchanged until the stream has passed the copy.  ipa_norm, ipa_core_degree and ipa_nll_eval (K <= IPA_MAX_K: the parameter sets
 *     travel in the kernel-parameter space) can be captured in a CUDA graph; a replay re-evaluates the
 *     parameter values given at capture time.  Calls that upload a host array with a copy (more than
 *     IPA_MAX_K sets, toy seeds, scan points) capture only if that array is in pinned host memory.
 *   - `ws_dev` is a scratch workspace of at least ipa_workspace_bytes(...) bytes, 256-byte aligned,
 *     private to one stream at a time.
 *   - Return value: IPA_OK (0) or a negative ipa_status.  Argument errors are detected before any
 *     work is enqueued.  CUDA launch errors are returned as IPA_ERR_CUDA (text: ipa_last_cuda_error).
 *   - Per-parameter-set DOMAIN errors do not fail the call: the set gets status != 0 in `status_dev`
 *     and NLL = +inf, so that a minimiser stepping outside the domain can recover.  Status values:
 *     0 ok; 1 basic domain (non-finite field, sigma<=0, zeta<0, zeta==0 with lambda>=0, a<=0, a2<=0, n<=0, n2<=0, f outside
 *     [0,1]); 2 join slope sign (L(d0)<=0 or L(d1)>=0: the power-law tail does not exist);
 *     3 internal numerical failure (normalisation not finite or not positive); 4 (ipa_nll_grad_eval only)
 *     f == 0 or f == 1.
 *   - Events outside [lo,hi] are evaluated by the same formulae (no clipping); NaN events give NaN.  The per-event
 *     arithmetic is valid while |log(f S) - log((1-f) B)| < 1e6 (the range of the kernels' exponential); parameter
 *     sets or events beyond that (e.g. |k (x - lo)| > 1e6) give undefined values, not an error.
 *   - ipa_norm returns the ABSOLUTE N_S, which underflows to 0 (status 0) when log N_S < -745 (e.g. zeta >~ 1000 with
 *     the unscaled Bessel core); the likelihood calls work with log N_S and are not affected.
 *     Any n >= 0 is accepted (n == 0 gives NLL = +0.0).
 *   - Determinism: for fixed device, build, n and launch geometry the results are bitwise
 *     reproducible, and the result of set k does not depend on which other sets share the batch.
 *     The per-event value may differ in the last bits (< 2e-13) between two ORDERS of the same events: a warp whose
 *     events lie in one cell of the core evaluates that cell's polynomial, any other warp the full one (ipa_core_cells).
 */
#ifndef IPANLL_H
#define IPANLL_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* One parameter set: 11 doubles.  Order follows the positional argument list of the paper's signal
 * kernel (mu, sigma, <unnamed 1>, beta, a, n, a2, n2) with the unnamed shape argument
 * expanded to (lambda, zeta) (reading D2), followed by the mixture parameters of
 * PAPER.md:77-85. */
typedef struct {
  double mu;     /* peak position */
  double sigma;  /* core width: the untruncated symmetric core has variance sigma^2 */
  double lambda; /* generalised-hyperbolic index; Bessel order nu = lambda - 1/2 */
  double zeta;   /* > 0: shape of the Bessel core (zeta -> inf: Gaussian); == 0 with lambda < 0: the zeta -> 0 limit, a
                    Student-t core (d^2+delta^2)^(lambda-1/2) e^(beta d), delta = sigma sqrt(-2 lambda-2) for lambda < -1,
                    else sigma (PAPER.md:226-236 `lb = -2.0` without zeta, ref. [10] at PAPER.md:450; reading D3) */
  double beta;   /* asymmetry, exp(beta d) factor */
  double a;      /* left join at d0 = -a sigma, a > 0 */
  double n;      /* left tail power, > 0 */
  double a2;     /* right join at d1 = +a2 sigma, a2 > 0 */
  double n2;     /* right tail power, > 0 */
  double f;      /* signal fraction in [0,1] */
  double k;      /* background slope: B(x) ~ exp(k x); k == 0 allowed */
} ipa_params;

typedef struct { double lo, hi; } ipa_range; /* fit range, finite, hi > lo */

typedef enum {
  IPA_OK = 0,
  IPA_ERR_INVALID_ARG = -1, /* null pointer, negative size, K < 1, hi <= lo, misaligned pointer */
  IPA_ERR_WORKSPACE = -2,   /* ws_bytes < ipa_workspace_bytes(...) or ws_dev misaligned */
  IPA_ERR_CUDA = -3,        /* a CUDA runtime call or launch failed */
  IPA_ERR_NO_DEVICE = -4,   /* no usable sm_100 device / kernel image */
  IPA_ERR_TOO_LARGE = -5    /* ipa_nll_eval_static: K > IPA_STATIC_MAX_K (the built-in scratch holds no more) */
} ipa_status;

const char* ipa_strerror(int code);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char* ipa_last_cuda_error(void);
/* Library build tag, e.g. "ipanll 0.1 sm_100a". */
const char* ipa_version(void);

/* Per-call options.  Every entry point that computes per-parameter-set constants takes `const ipa_options* opt_host`
 * (NULL = all defaults); the struct is read before the call returns.
 *   degree_policy  core-approximant degree (prologue): 0 = adaptive (default: the Chebyshev
 *                  series of log(z^nu K_nu(z)) is cut where its coefficients fall under the fp64 noise floor, so a
 *                  half-integer order collapses to a very short polynomial); 1 = geometric (at least the a-priori
 *                  degree a general order needs on the same z-interval -- the degree at which the Chebyshev coefficients
 *                  2 rho^-k / k of its log z term reach the noise threshold: no half-integer shortcut; reading D2).
 *   first_slot     ipa_toy_generate in mixture mode only (ignored elsewhere, must be >= 0): the call draws the events
 *                  of slots first_slot .. first_slot + capacity - 1 of the seeded dataset (an event depends on
 *                  (seed, slot) only), so G ranks can each generate their contiguous shard of ONE dataset
 *                  (DESIGN.md section 7).  Default 0.
 * Results are bitwise reproducible for fixed options; they differ between the two policies at the 1e-15 level. */
typedef struct {
  int32_t degree_policy;
  int32_t reserved;    /* must be 0 */
  int64_t first_slot;
} ipa_options;

/* Bytes of workspace needed by any call below for n events, K parameter sets (or T segments / toys:
 * pass the larger of K and T) and nbins histogram bins (0 if unused). */
size_t ipa_workspace_bytes(int64_t n, int64_t K, int64_t nbins);

/* Normalisation integrals of K parameter sets (readings C2, C5):
 *   norm_sig_dev[k] = N_S = int_lo^hi I(x - mu) dx   (closed-form tails + Gauss-Legendre core)
 *   norm_bkg_dev[k] = N_B = int_lo^hi exp(k (x - lo)) dx = expm1(k (hi-lo)) / k   (hi-lo at k=0)
 * status_dev[k] as described above (may be NULL).  Invalid sets give NaN. */
int ipa_norm(const ipa_params* p_host, int K, ipa_range r, double* norm_sig_dev, double* norm_bkg_dev,
             int32_t* status_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* Introspection of the prologue (step A1e): degree_dev[k] = degree of the core
 * approximant chosen for set k under the current degree policy, -1 for a set evaluated in direct mode
 * (per-event Bessel function), -2 for a set with a domain error.  Used by bench.py to state the
 * algorithmic work of the timed workload. */
int ipa_core_degree(const ipa_params* p_host, int K, ipa_range r, int32_t* degree_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes,
                    void* cuda_stream);

/* Introspection of the prologue, cells of the core (step A1e).  Where the full core polynomial has
 * degree 16 or more, the core interval of r = sqrt((x-mu)^2 + delta^2) is cut into 4 cells of equal ratio and each cell gets
 * its own polynomial of lower degree, refitted from the full one; a warp whose events all lie in one cell (a warp of an
 * array laid out by ipa_events_prepare, or of a sorted array, nearly always does) evaluates the cell polynomial, any other
 * warp the full one.  Both approximate the same function to the same tolerance: the value of an event can differ in the
 * last bits between two layouts of the same events, never between two runs on the same array.
 *   cells_dev [K][IPA_CELL_INFO] int32: { number of cells (4, or 0: no cells for this set),
 *                                         degree of cell 0..3 (cell 0 holds the peak),
 *                                         high 32 bits of the 6 cell boundaries in x, ascending (0 / INT32_MAX: a boundary
 *                                         outside the core on the left / on the right), INT32_MAX, INT32_MAX }
 * An event x lies in cell |#{i : hb[i] <= high word of x} - 3|.  Used by bench.py to state the algorithmic work. */
#define IPA_CELL_INFO 13
int ipa_core_cells(const ipa_params* p_host, int K, ipa_range r, int32_t* cells_dev, const ipa_options* opt_host,
                   void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* The hot path (fused into one pass): NLL of n events for K parameter sets.
 *   x_dev      [n]    event masses, fp64, 8-byte aligned
 *   p_host     [K]    parameter sets
 *   nll_dev    [K]    out: -sum_i log(f S + (1-f) B); +inf for a set with status != 0
 *   logpdf_dev [K*n]  out, optional (NULL to skip): per-event log(f S + (1-f) B), set-major; the row of a set with
 *                     status != 0 is filled with NaN
 *   status_dev [K]    out, optional
 * K <= IPA_MAX_K per call; up to 26 sets share one pass over the events, a larger batch takes two (shared memory). */
#define IPA_MAX_K 32
int ipa_nll_eval(const double* x_dev, int64_t n, const ipa_params* p_host, int K, ipa_range r,
                 double* nll_dev, double* logpdf_dev, int32_t* status_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes,
                 void* cuda_stream);

/* Finite-difference gradient of the NLL (reading C6; the paper leaves the differences to
 * Minuit): ONE pass over the events for the K = 2P+1 sets
 *   set 0 = theta,  sets 2j+1 / 2j+2 = theta with field idx_host[j] replaced by theta[idx] +/- h_host[j]
 * (each sum computed once, in fp64, on the host), then on the device
 *   grad_dev[j] = (nll[2j+1] - nll[2j+2]) / (2 h_j).
 *   theta_host [1]; idx_host [P] field indices 0..10 in the order of ipa_params; h_host [P] > 0; 1 <= P <= 11
 *   nll_dev [2P+1] out: the NLLs of the batch in that order;  grad_dev [P] out;  status_dev [2P+1] out, optional
 * A displaced set outside the domain gives +inf / NaN in its entries, as in ipa_nll_eval. */
int ipa_nll_fd_gradient(const double* x_dev, int64_t n, const ipa_params* theta_host, int P, const int32_t* idx_host,
                        const double* h_host, ipa_range r, double* nll_dev, double* grad_dev, int32_t* status_dev,
                        const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* Extended likelihood (reading D4: the paper's FCN works with yields):
 *   nll_dev[k] = (ns_k + nb_k) - sum_i log( ns_k S(x_i) + nb_k B(x_i) )
 * for K sets; the f field of p_host is ignored (the library evaluates the fraction form with
 * f = ns/(ns+nb), computed in fp64 on the host, and adds (ns+nb) - n log(ns+nb) on the device).
 * ns_k, nb_k >= 0, ns_k + nb_k > 0, else status 1.  Everything else as ipa_nll_eval. */
int ipa_nll_eval_extended(const double* x_dev, int64_t n, const ipa_params* p_host, const double* ns_host,
                          const double* nb_host, int K, ipa_range r, double* nll_dev, int32_t* status_dev,
                          const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* NLL and its ANALYTIC gradient with respect to (mu, sigma, f, k, beta) in one pass (the
 * paper mentions analytic gradients through iminuit and generated derivative code, PAPER.md:36, 383,
 * without formulae; the derivatives are those of the definition above):
 *   nll_dev  [K]              as ipa_nll_eval (same value up to rounding: the core term is evaluated with one
 *                             Horner pass for the polynomial and its derivative)
 *   grad_dev [IPA_NGRAD * K]  d NLL / d (mu, sigma, f, k, beta) of set k at grad_dev[IPA_NGRAD k .. IPA_NGRAD k + 4]
 * Needs 0 < f < 1: a set with f == 0 or f == 1 gets status 4, NLL = +inf and NaN derivatives.  The events are
 * read once for up to 4 sets (more sets: one pass per group of 4).  K <= IPA_MAX_K. */
#define IPA_NGRAD 5
int ipa_nll_grad_eval(const double* x_dev, int64_t n, const ipa_params* p_host, int K, ipa_range r,
                      double* nll_dev, double* grad_dev, int32_t* status_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes,
                      void* cuda_stream);

/* Same likelihood over T segments (toys, categories) of one event array, one parameter set per
 * segment, all in one launch (BASELINE.json config 4; PAPER.md:139-149 loops categories on the host).
 *   offsets_dev [T+1]  segment t = x_dev[offsets[t] .. offsets[t+1]), non-decreasing, on the device
 *   p_host      [T]    parameter sets (copied through the workspace by a kernel argument path)
 *   nll_dev     [T]    out */
int ipa_nll_eval_segmented(const double* x_dev, const int64_t* offsets_dev, int64_t T, const ipa_params* p_host,
                           ipa_range r, double* nll_dev, int32_t* status_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes,
                           void* cuda_stream);

/* Simultaneous categories with SHARED parameter sets (one model, several categories,
 * parameters in common): as ipa_nll_eval_segmented, but segment t is evaluated with parameter set
 * set_of_segment_host[t] in [0, K) of p_host [K]; the prologue runs once per set, not once per segment.
 * The fit's NLL is the sum of nll_dev [T] (added by the caller or by one more reduction).  Workspace:
 * ipa_workspace_bytes(n, max(K, T), 0). */
int ipa_nll_eval_categories(const double* x_dev, const int64_t* offsets_dev, int64_t T, const ipa_params* p_host, int64_t K,
                            const int32_t* set_of_segment_host, ipa_range r, double* nll_dev, int32_t* status_dev,
                            const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* Toy-MC generation on the device (readings D13, D14).
 * Toy t draws Ns ~ Poisson(mean_sig), Nb ~ Poisson(mean_bkg) from seeds_host[t] (Philox-4x32-10
 * counter-based streams), then Ns signal events by accept-reject under a flat envelope followed by
 * Nb background events by the inverse CDF of the truncated exponential.
 *   gen_host   [T] or [1] (gen_count = T or 1): generating parameter sets
 *   mean_sig/mean_bkg < 0 selects MIXTURE mode for configs 1-3: T must be 1, exactly `capacity`
 *     events are generated and the component of each event is chosen by u < f.
 *   capacity   size of x_dev in events; if the drawn total exceeds it, offsets are still written,
 *              no event beyond capacity is written and overflow_dev[0] is set to 1.
 *   x_dev      [capacity] out;  offsets_dev [T+1] out;  overflow_dev [1] out (int32; bit 0: capacity exceeded,
 *              bit 1: an accept-reject attempt cap was hit -- cannot happen for a valid shape)
 *   status_dev [gen_count] out, optional: domain status of every generating set; the events of a toy whose
 *              generating set is invalid are NaN (offsets are still written) */
int ipa_toy_generate(const uint64_t* seeds_host, int64_t T, const ipa_params* gen_host, int64_t gen_count,
                     double mean_sig, double mean_bkg, ipa_range r, int64_t capacity, double* x_dev,
                     int64_t* offsets_dev, int32_t* overflow_dev, int32_t* status_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* Histogram of n events in nbins uniform bins on [lo,hi]:
 * bin = floor((x-lo) nbins/(hi-lo)), x == hi goes to the last bin, events outside are dropped.
 * counts_dev [nbins] is overwritten. */
int ipa_hist_fill(const double* x_dev, int64_t n, ipa_range r, int nbins, uint64_t* counts_dev, void* cuda_stream);

/* Binned Poisson likelihood over a list of parameter points (reading D15):
 *   s_b = I(c_b - mu) / sum_b' I(c_b' - mu),  b_b = e^{k c_b} / sum_b' e^{k c_b'}  at bin centres c_b,
 *   nu_b = ns s_b + nb b_b,   NLL = sum_b [ nu_b - n_b log nu_b ]   (n_b = 0: nu_b).
 *   counts_dev [nbins]; shape_host: one parameter set (its f and k are ignored);
 *   ns_host, nb_host, k_host [npoints] (three uploads; ONE if the arrays lie back to back in host memory, ns then nb then k,
 *   as the Python binding packs them); nll_dev [npoints] out. */
int ipa_binned_nll_scan(const uint64_t* counts_dev, int nbins, ipa_range r, const ipa_params* shape_host,
                        const double* ns_host, const double* nb_host, const double* k_host, int64_t npoints,
                        double* nll_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* Expected histogram nu_b = ns s_b + nb b_b for one point (input of ipa_poisson_hist_toys). */
int ipa_expected_hist(int nbins, ipa_range r, const ipa_params* shape_host, double ns, double nb, double k,
                      double* nu_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* Gaussian-smeared signal shape on the bin grid ("SM = GaussSmear1(bins_cx, sigma0);
 * sigf_gpu = SM.Smear(sigf_i_gpu)"; kernel, normalisation and edges are not stated -- DESIGN.md reading F3):
 *   ipa_signal_shape   sig_dev[b] = I(c_b - mu) / I(reference point) at the bin centres c_b (not normalised):
 *                      what the paper's Ipatia kernel writes before the smearing
 *   ipa_gauss_smear    out_b = sum_j in_j g_{b-j},  g_m = exp(-(m w)^2 / (2 sigma0^2)) / sum_{|m'|<=M} g_m',
 *                      |m| <= M = ceil(8 sigma0 / w), w = bin width, in_j = 0 outside the grid; sigma0 <= 0
 *                      copies; out_dev must not alias in_dev; M <= 2800
 *   ipa_expected_hist_shape / ipa_binned_nll_scan_shape
 *                      ipa_expected_hist / ipa_binned_nll_scan with a GIVEN signal shape sig_dev [nbins] >= 0
 *                      (normalised to unit sum inside, as PAPER.md:311-312 does) instead of a parameter set;
 *                      a shape whose sum is not positive gives NaN / +inf results */
int ipa_signal_shape(int nbins, ipa_range r, const ipa_params* shape_host, double* sig_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes,
                     void* cuda_stream);
int ipa_gauss_smear(const double* in_dev, int nbins, ipa_range r, double sigma0, double* out_dev, void* cuda_stream);
int ipa_expected_hist_shape(int nbins, ipa_range r, const double* sig_dev, double ns, double nb, double k, double* nu_dev,
                            void* ws_dev, size_t ws_bytes, void* cuda_stream);
int ipa_binned_nll_scan_shape(const uint64_t* counts_dev, int nbins, ipa_range r, const double* sig_dev,
                              const double* ns_host, const double* nb_host, const double* k_host, int64_t npoints,
                              double* nll_dev, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* Per-bin Poisson toys, a separate mean per generated value:
 * counts_dev[t*nbins + b] ~ Poisson(mean_dev[b]) from key seeds_host[t], counter slot b. */
int ipa_poisson_hist_toys(const double* mean_dev, int nbins, const uint64_t* seeds_host, int64_t T,
                          uint32_t* counts_dev, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* CLs on binned toys (CL.setData, CL.setExpected(HistoPdf), CL.CLs(ns, toys); the paper
 * does not print its statistic -- DESIGN.md reading F2): likelihood ratio of two fixed expected histograms,
 *   q_t = -2 ln[ L(n_t | nu_sb) / L(n_t | nu_b) ] = 2 sum_b [ (nu_sb_b - nu_b_b) - n_tb ln(nu_sb_b / nu_b_b) ].
 *   counts_dev [T*nbins] toy (or data, T = 1) histograms, count_bytes = 4 (ipa_poisson_hist_toys) or 8
 *   (ipa_hist_fill);  nu_sb_dev, nu_b_dev [nbins] > 0 (ipa_expected_hist);  q_dev [T] out. */
int ipa_cls_teststat(const void* counts_dev, int count_bytes, int64_t T, int nbins, const double* nu_sb_dev,
                     const double* nu_b_dev, double* q_dev, void* ws_dev, size_t ws_bytes, void* cuda_stream);
/* count_dev[0] = #{ t : q_dev[t] >= q_obs_dev[0] }  (q_obs stays on the device: it is the statistic of the data). */
int ipa_cls_count_ge(const double* q_dev, int64_t T, const double* q_obs_dev, int64_t* count_dev, void* cuda_stream);
/* cl_dev = { CL_sb = count_sb/T_sb, CL_b = count_b/T_b, CL_s = CL_sb/CL_b (NaN if count_b == 0) }. */
int ipa_cls_from_counts(const int64_t* count_sb_dev, int64_t T_sb, const int64_t* count_b_dev, int64_t T_b,
                        double* cl_dev, void* cuda_stream);

/* Optional one-off preparation of the data layout: a STABLE counting sort of the events on a coarse bin index,
 *   bin(x) = clamp(floor((x - lo) IPA_PREPARE_BINS / (hi - lo)), 0, IPA_PREPARE_BINS - 1),  NaN -> last bin
 * (whole array, or inside each of T segments when offsets_dev != NULL).  The likelihood does not depend on the
 * order of the events, the data of a fit are constant over the minimiser's calls, and the
 * streaming kernels skip the core polynomial / the tail logarithm for a warp whose 32 x E events all lie in one
 * region: on events grouped by bin nearly every warp is region-uniform, for every parameter set of the fit (the
 * bins do not depend on the joins).  Unprepared input is always correct.  The output is a permutation of the
 * input and a pure function of it (original order inside a bin), so results computed from it are bitwise
 * reproducible; the sum over the prepared array differs from the sum over the original order by rounding only
 * (reading E4).  Own kernels (histogram, two scans, scatter): csrc/ipa_prepare.cuh.
 *   x_out_dev [n] must not alias x_in_dev;  n < 2^32;  ws_dev of ipa_prepare_workspace_bytes(n, T) bytes (T = 0
 *   for an unsegmented array);  r = the fit range the bins span. */
#define IPA_PREPARE_BINS 256
size_t ipa_prepare_workspace_bytes(int64_t n, int64_t T);
int ipa_events_prepare(const double* x_in_dev, int64_t n, const int64_t* offsets_dev, int64_t T, ipa_range r,
                       double* x_out_dev, void* ws_dev, size_t ws_bytes, void* cuda_stream);

/* ipa_nll_eval for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same prologue and streaming kernels, same arguments, same results bit for bit,
 * but the scratch (per-set constants, partial sums, ticket counters) lives in a file-scope `static __device__` array
 * of IPA_STATIC_SCRATCH_BYTES inside the library instead of a caller-owned workspace.  The entry point allocates and
 * frees nothing (no cudaMalloc / cudaFree / allocating library routine); inputs and outputs are still the caller's.
 *   - Limit: K <= IPA_STATIC_MAX_K parameter sets per call; a larger K returns IPA_ERR_TOO_LARGE before any work is
 *     enqueued (any n is accepted: the scratch does not grow with n).  Use ipa_nll_eval with an own workspace beyond.
 *   - Every GPU that loads the library holds the array (288 KiB) until the process exits.
 *   - The array is shared by EVERY call on a device and keeps the previous call's contents.  Each call rewrites all it
 *     reads (the prologue kernel rewrites the records and zeroes the ticket counters before the streaming kernel
 *     counts on them), so calls that follow one another on one stream, or are ordered by events, are independent.
 *     Calls that OVERLAP on the GPU (two streams, two host threads, concurrent graph launches) race on it: their
 *     results are undefined.  Such callers need ipa_nll_eval with one workspace per stream.
 *   - The array's device address is looked up once per device (cudaGetSymbolAddress, with that device current). */
#define IPA_STATIC_MAX_K 16
#define IPA_STATIC_SCRATCH_BYTES (288 * 1024)
int ipa_nll_eval_static(const double* x_dev, int64_t n, const ipa_params* p_host, int K, ipa_range r, double* nll_dev,
                        double* logpdf_dev, int32_t* status_dev, const ipa_options* opt_host, void* cuda_stream);

/* Measurement aid (not on the hot path): runs `iters` dependent DFMA per thread in 8 independent
 * chains on a full grid, for the FP64 roofline denominator.  out_dev [1]. */
int ipa_fp64_peak_probe(int64_t iters, double* out_dev, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* IPANLL_H */
