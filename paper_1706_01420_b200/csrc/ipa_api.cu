// ipa_api.cu -- the C ABI of include/ipanll.h: argument validation, workspace layout and launch
// sequencing on the caller's stream.  No allocation, no synchronisation, no CPU arithmetic of the
// method: every step of the path runs in the kernels of ipa_kernels.cuh.
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include "ipa_kernels.cuh"
#include "ipa_prepare.cuh"

static_assert(IPA_PREP_BINS == IPA_PREPARE_BINS, "bin count of ipa_events_prepare");

namespace {

thread_local std::string g_last_cuda_error;

#define IPA_CK(call)                                                                       \
  do {                                                                                     \
    cudaError_t e_ = (call);                                                               \
    if (e_ != cudaSuccess) {                                                               \
      g_last_cuda_error = std::string(#call) + ": " + cudaGetErrorString(e_);              \
      return IPA_ERR_CUDA;                                                                 \
    }                                                                                      \
  } while (0)

// degree policy of the call (NULL options = defaults); -1 = invalid options
int policy_of(const ipa_options* o) {
  if (!o) return 0;
  if ((o->degree_policy != 0 && o->degree_policy != 1) || o->reserved || o->first_slot < 0) return -1;
  return o->degree_policy;
}

constexpr int64_t kGridMax = 2048;  // upper bound of the streaming grid (partials sizing)
constexpr size_t kGradSmem = 2 * IPA_GTILE * 8 + IPA_GKB * (sizeof(IpaSetConsts) + IPA_GQ * IPA_GB * 8);

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Workspace layout (offsets in bytes, every block 256-byte aligned).
struct Layout {
  size_t consts, counter, partials, params, seeds, nsig, ntot, pts, sbin, flag, total;
};
Layout make_layout(int64_t K, int64_t nbins) {
  if (K < 1) K = 1;
  if (nbins < 0) nbins = 0;
  Layout L;
  size_t o = 0;
  L.consts = o;   o += align_up((size_t)K * sizeof(IpaSetConsts), 256);
  L.counter = o;  o += 256;
  const int64_t kk = K < IPA_MAX_K ? K : IPA_MAX_K;
  size_t pb = (size_t)kk * kGridMax * 8;
  if ((size_t)K * IPA_SEGC * 8 > pb) pb = (size_t)K * IPA_SEGC * 8;   // segmented call: T * C partials, T * C <= max(8 T, 592 + T)
  L.partials = o; o += align_up(pb, 256);
  L.params = o;   o += align_up((size_t)K * sizeof(ipa_params), 256);
  L.seeds = o;    o += align_up((size_t)K * 8, 256);
  L.nsig = o;     o += align_up((size_t)K * 8, 256);
  L.ntot = o;     o += align_up((size_t)K * 8, 256);
  L.pts = o;      o += align_up((size_t)K * 3 * 8, 256);
  L.sbin = o;     o += align_up((size_t)nbins * 8, 256);
  L.flag = o;     o += 256;
  L.total = o;
  return L;
}

// Sets per launch of the streaming kernel: each set takes its record and IPA_NB accumulators in shared memory beside the
// two staged tiles and the 17 KB of static tables.  A larger batch (up to IPA_MAX_K) runs as two launches over the events.
constexpr int kStreamKMax = 26;
static_assert(kStreamKMax * (sizeof(IpaSetConsts) + IPA_NB * 8) + 2 * IPA_NTILE * 8 + IPA_MATHTAB_DOUBLES * 8 + 1200 <= 227 * 1024,
              "streaming kernel: shared memory of a full batch");
struct DevInfo { int dev = -1; int sms = 0; bool attr_set = false; };
thread_local DevInfo g_dev;

int device_info(int* sms) {
  int dev = 0;
  IPA_CK(cudaGetDevice(&dev));
  if (g_dev.dev != dev || !g_dev.attr_set) {
    int n = 0;
    IPA_CK(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev));
    const int smem = kStreamKMax * (int)(sizeof(IpaSetConsts) + IPA_NB * 8) + 2 * IPA_NTILE * 8;
    IPA_CK(cudaFuncSetAttribute(ipa_nll_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    IPA_CK(cudaFuncSetAttribute(ipa_nll_kernel<false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    IPA_CK(cudaFuncSetAttribute(ipa_nll_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    IPA_CK(cudaFuncSetAttribute(ipa_nll_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    IPA_CK(cudaFuncSetAttribute(ipa_nll_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    IPA_CK(cudaFuncSetAttribute(ipa_nll_grad_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGradSmem));
    IPA_CK(cudaFuncSetAttribute(ipa_nll_grad_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kGradSmem));
    IPA_CK(cudaFuncSetAttribute(ipa_prep_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, IPA_PREP_SMEM));
    IPA_CK(cudaFuncSetAttribute(ipa_prep_segment_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, IPA_PREP_SMEM));
    // four resident blocks per SM need 4 x 43 KB of shared memory: ask for the largest carve-out
    IPA_CK(cudaFuncSetAttribute(ipa_prep_scatter_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    IPA_CK(cudaFuncSetAttribute(ipa_prep_segment_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    g_dev.dev = dev;
    g_dev.sms = n;
    g_dev.attr_set = true;
  }
  *sms = g_dev.sms;
  return IPA_OK;
}

bool range_ok(ipa_range r) {
  return ipa_finite(r.lo) && ipa_finite(r.hi) && r.hi > r.lo;
}
bool ws_ok(const void* ws, size_t bytes, size_t need) {
  return ws != nullptr && ((uintptr_t)ws % 256) == 0 && bytes >= need;
}

// Runs the prologue for K sets.  K <= IPA_MAX_K: the sets travel in the kernel-parameter space;
// larger batches go through the workspace with one host-to-device copy.
int run_prologue(const ipa_params* p_host, int64_t K, ipa_range r, int policy, char* ws, const Layout& L, double* norm_sig,
                 double* norm_bkg, int32_t* status_out, cudaStream_t st, bool want_grad = false) {
  IpaSetConsts* consts = reinterpret_cast<IpaSetConsts*>(ws + L.consts);
  unsigned int* counter = reinterpret_cast<unsigned int*>(ws + L.counter);
  static thread_local IpaParamBatch batch;
  const ipa_params* p_dev = nullptr;
  if (K <= IPA_MAX_K) {
    std::memcpy(batch.p, p_host, (size_t)K * sizeof(ipa_params));
  } else {
    IPA_CK(cudaMemcpyAsync(ws + L.params, p_host, (size_t)K * sizeof(ipa_params), cudaMemcpyHostToDevice, st));
    p_dev = reinterpret_cast<const ipa_params*>(ws + L.params);
  }
  ipa_prologue_kernel<<<(unsigned)K, IPA_PRO_THREADS, 0, st>>>(batch, p_dev, r.lo, r.hi,
                                                               policy | (want_grad ? 2 : 0), consts,
                                                               counter, norm_sig, norm_bkg, status_out);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

}  // namespace

// ---- built-in scratch of ipa_nll_eval_static (the one entry point that needs no caller workspace) --------------------
// A file-scope device array: every device that loads the library holds it until the process exits.  In HOST code the
// name `ipa_static_scratch` is only a stand-in for the symbol, not a device address; the address a kernel may use comes
// from cudaGetSymbolAddress, looked up once per device with that device current.
static __device__ __align__(256) unsigned char ipa_static_scratch[IPA_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_scratch_mutex;
void* g_scratch_ptr[kMaxDevices] = {};

int static_scratch(void** out) {
  if (make_layout(IPA_STATIC_MAX_K, 0).total > (size_t)IPA_STATIC_SCRATCH_BYTES) {
    g_last_cuda_error = "ipa_nll_eval_static: IPA_STATIC_SCRATCH_BYTES is smaller than the workspace of IPA_STATIC_MAX_K sets";
    return IPA_ERR_WORKSPACE;
  }
  int dev = 0;
  IPA_CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return IPA_ERR_NO_DEVICE;
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_ptr[dev]) {
    void* ptr = nullptr;
    IPA_CK(cudaGetSymbolAddress(&ptr, ipa_static_scratch));      // device `dev` is current
    if (!ptr || ((uintptr_t)ptr % 256) != 0) return IPA_ERR_WORKSPACE;
    g_scratch_ptr[dev] = ptr;
  }
  *out = g_scratch_ptr[dev];
  return IPA_OK;
}

}  // namespace

extern "C" {

const char* ipa_strerror(int code) {
  switch (code) {
    case IPA_OK: return "ok";
    case IPA_ERR_INVALID_ARG: return "invalid argument";
    case IPA_ERR_WORKSPACE: return "workspace too small or misaligned";
    case IPA_ERR_CUDA: return "CUDA error (see ipa_last_cuda_error)";
    case IPA_ERR_NO_DEVICE: return "no usable CUDA device";
    case IPA_ERR_TOO_LARGE: return "more parameter sets than the built-in scratch of ipa_nll_eval_static holds (IPA_STATIC_MAX_K)";
    default: return "unknown error code";
  }
}

const char* ipa_last_cuda_error(void) { return g_last_cuda_error.c_str(); }
const char* ipa_version(void) { return "ipanll 0.1 sm_100a"; }

size_t ipa_workspace_bytes(int64_t n, int64_t K, int64_t nbins) {
  (void)n;
  return make_layout(K, nbins).total;
}

int ipa_norm(const ipa_params* p_host, int K, ipa_range r, double* norm_sig_dev, double* norm_bkg_dev,
             int32_t* status_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  const int policy = policy_of(opt_host);
  if (!p_host || K < 1 || !range_ok(r) || !norm_sig_dev || !norm_bkg_dev || policy < 0) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(K, 0);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  return run_prologue(p_host, K, r, policy, static_cast<char*>(ws_dev), L, norm_sig_dev, norm_bkg_dev, status_dev,
                      static_cast<cudaStream_t>(cuda_stream));
}

int ipa_core_degree(const ipa_params* p_host, int K, ipa_range r, int32_t* degree_dev, const ipa_options* opt_host,
                    void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  const int policy = policy_of(opt_host);
  if (!p_host || K < 1 || !range_ok(r) || !degree_dev || policy < 0) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(K, 0);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  int rc = run_prologue(p_host, K, r, policy, ws, L, nullptr, nullptr, nullptr, st);
  if (rc) return rc;
  ipa_degree_kernel<<<(K + 127) / 128, 128, 0, st>>>(reinterpret_cast<const IpaSetConsts*>(ws + L.consts), K, degree_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_core_cells(const ipa_params* p_host, int K, ipa_range r, int32_t* cells_dev, const ipa_options* opt_host,
                   void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  static_assert(IPA_CELL_INFO == 1 + IPA_NCELL + 8, "ipanll.h: IPA_CELL_INFO");
  const int policy = policy_of(opt_host);
  if (!p_host || K < 1 || !range_ok(r) || !cells_dev || policy < 0) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(K, 0);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  int rc = run_prologue(p_host, K, r, policy, ws, L, nullptr, nullptr, nullptr, st);
  if (rc) return rc;
  ipa_cells_kernel<<<(K + 127) / 128, 128, 0, st>>>(reinterpret_cast<const IpaSetConsts*>(ws + L.consts), K, cells_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_nll_eval(const double* x_dev, int64_t n, const ipa_params* p_host, int K, ipa_range r, double* nll_dev,
                 double* logpdf_dev, int32_t* status_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes,
                 void* cuda_stream) {
  const int policy = policy_of(opt_host);
  if (n < 0 || (n > 0 && !x_dev) || !p_host || K < 1 || K > IPA_MAX_K || !range_ok(r) || !nll_dev || policy < 0)
    return IPA_ERR_INVALID_ARG;
  if (((uintptr_t)x_dev % 8) != 0) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(K, 0);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  int sms = 0;
  int rc = device_info(&sms);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  rc = run_prologue(p_host, K, r, policy, ws, L, nullptr, nullptr, nullptr, st);
  if (rc) return rc;
  const int64_t ntiles = (n + IPA_NTILE - 1) / IPA_NTILE;
  int64_t G = (int64_t)sms * IPA_NB_PER_SM;
  if (G > kGridMax) G = kGridMax;
  if (G > ntiles) G = ntiles;
  if (G < 1) G = 1;
  const int vec_ok = ((uintptr_t)x_dev % 16) == 0;
  const IpaSetConsts* consts = reinterpret_cast<const IpaSetConsts*>(ws + L.consts);
  double* partials = reinterpret_cast<double*>(ws + L.partials);
  unsigned int* counter = reinterpret_cast<unsigned int*>(ws + L.counter);
  // K <= kStreamKMax: one launch; above: two launches of half the batch each (own counter, own rows of the outputs)
  const int nlaunch = (K + kStreamKMax - 1) / kStreamKMax;
  const int kper = (K + nlaunch - 1) / nlaunch;
  for (int b = 0; b < nlaunch; ++b) {
    const int k0 = b * kper, kb = (K - k0 < kper) ? K - k0 : kper;
    const ipa_params* ph = p_host + k0;
    // sets with bitwise equal signal-shape parameters (the first 9 doubles) share the shape stage
    IpaGroups grp;
    for (int k = 0; k < IPA_MAX_K; ++k) grp.leader[k] = (signed char)k;
    for (int k = 1; k < kb; ++k)
      for (int j = 0; j < k; ++j)
        if (grp.leader[j] == j && std::memcmp(&ph[k], &ph[j], 9 * sizeof(double)) == 0) {
          grp.leader[k] = (signed char)j;
          break;
        }
    bool grouped = false;
    for (int k = 0; k < kb; ++k) grouped = grouped || grp.leader[k] != k;
    int ng = 0, nm = 0;
    for (int g = 0; g < kb; ++g) {
      if (grp.leader[g] != g) continue;
      grp.first[ng++] = (unsigned char)nm;
      for (int k = g; k < kb; ++k)
        if (grp.leader[k] == g) grp.member[nm++] = (unsigned char)k;
    }
    grp.first[ng] = (unsigned char)nm;
    grp.ngroups = (unsigned char)ng;
    for (int i = ng + 1; i <= IPA_MAX_K; ++i) grp.first[i] = (unsigned char)nm;
    for (int i = nm; i < IPA_MAX_K; ++i) grp.member[i] = 0;
    auto kern = logpdf_dev ? (grouped ? ipa_nll_kernel<true, true> : ipa_nll_kernel<true, false>)
                           : (grouped ? ipa_nll_kernel<false, true> : ipa_nll_kernel<false, false>);
    if (kb == 1 && !logpdf_dev) kern = ipa_nll_kernel<false, false, true>;
    const size_t smem = (size_t)kb * (sizeof(IpaSetConsts) + IPA_NB * 8) + 2 * IPA_NTILE * 8;
    // the first launch is a programmatic dependent of the prologue kernel enqueued just before it: its blocks load the
    // math table and their first tile while the prologue runs, and wait for its end before they read the records
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)G);
    cfg.blockDim = dim3(IPA_NB);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = (b == 0) ? 1 : 0;
    IPA_CK(cudaLaunchKernelEx(&cfg, kern, x_dev, (long long)n, vec_ok, consts + k0, kb, grp, partials + (size_t)k0 * G,
                              logpdf_dev ? logpdf_dev + (size_t)k0 * n : (double*)nullptr, counter + b, nll_dev + k0,
                              status_dev ? status_dev + k0 : (int32_t*)nullptr));
  }
  return IPA_OK;
}

int ipa_nll_fd_gradient(const double* x_dev, int64_t n, const ipa_params* theta_host, int P, const int32_t* idx_host,
                        const double* h_host, ipa_range r, double* nll_dev, double* grad_dev, int32_t* status_dev,
                        const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (!theta_host || P < 1 || P > 11 || !idx_host || !h_host || !grad_dev) return IPA_ERR_INVALID_ARG;
  ipa_params batch[2 * 11 + 1];
  IpaFdSteps hs;
  for (int j = 0; j < 2 * P + 1; ++j) batch[j] = *theta_host;
  for (int j = 0; j < 11; ++j) hs.h[j] = 1.0;
  for (int j = 0; j < P; ++j) {
    if (idx_host[j] < 0 || idx_host[j] > 10 || !(h_host[j] > 0.0) || !ipa_finite(h_host[j])) return IPA_ERR_INVALID_ARG;
    const double base = (&theta_host->mu)[idx_host[j]];
    (&batch[2 * j + 1].mu)[idx_host[j]] = base + h_host[j];
    (&batch[2 * j + 2].mu)[idx_host[j]] = base - h_host[j];
    hs.h[j] = h_host[j];
  }
  int rc = ipa_nll_eval(x_dev, n, batch, 2 * P + 1, r, nll_dev, nullptr, status_dev, opt_host, ws_dev, ws_bytes, cuda_stream);
  if (rc) return rc;
  ipa_fd_difference_kernel<<<1, 32, 0, static_cast<cudaStream_t>(cuda_stream)>>>(nll_dev, P, hs, grad_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_nll_eval_extended(const double* x_dev, int64_t n, const ipa_params* p_host, const double* ns_host,
                          const double* nb_host, int K, ipa_range r, double* nll_dev, int32_t* status_dev,
                          const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (!p_host || !ns_host || !nb_host || K < 1 || K > IPA_MAX_K) return IPA_ERR_INVALID_ARG;
  ipa_params q[IPA_MAX_K];
  double nu[IPA_MAX_K];
  for (int k = 0; k < K; ++k) {
    q[k] = p_host[k];
    nu[k] = ns_host[k] + nb_host[k];
    const bool ok = ns_host[k] >= 0.0 && nb_host[k] >= 0.0 && nu[k] > 0.0 && ipa_finite(nu[k]);
    q[k].f = ok ? ns_host[k] / nu[k] : -1.0;          // an invalid yield pair becomes a domain error of the set
    if (!ok) nu[k] = 1.0;
  }
  int rc = ipa_nll_eval(x_dev, n, q, K, r, nll_dev, nullptr, status_dev, opt_host, ws_dev, ws_bytes, cuda_stream);
  if (rc) return rc;
  IpaYields y;
  for (int k = 0; k < IPA_MAX_K; ++k) y.nu[k] = k < K ? nu[k] : 1.0;
  ipa_extended_term_kernel<<<1, IPA_MAX_K, 0, static_cast<cudaStream_t>(cuda_stream)>>>(nll_dev, K, (long long)n, y);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_nll_grad_eval(const double* x_dev, int64_t n, const ipa_params* p_host, int K, ipa_range r,
                      double* nll_dev, double* grad_dev, int32_t* status_dev, const ipa_options* opt_host, void* ws_dev,
                      size_t ws_bytes, void* cuda_stream) {
  const int policy = policy_of(opt_host);
  if (n < 0 || (n > 0 && !x_dev) || !p_host || K < 1 || K > IPA_MAX_K || !range_ok(r) || !nll_dev || !grad_dev || policy < 0)
    return IPA_ERR_INVALID_ARG;
  if (((uintptr_t)x_dev % 8) != 0) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(K, 0);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  int sms = 0;
  int rc = device_info(&sms);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  IPA_CK(cudaMemsetAsync(ws + L.counter, 0, 256, st));          // one ticket counter per group of IPA_GKB sets
  rc = run_prologue(p_host, K, r, policy, ws, L, nullptr, nullptr, nullptr, st, true);   // (zeroes the first two again)
  if (rc) return rc;
  const int64_t ntiles = (n + IPA_GTILE - 1) / IPA_GTILE;
  int64_t G = (int64_t)sms;
  if (G > ntiles) G = ntiles;
  if (G < 1) G = 1;
  if (G * IPA_GQ > kGridMax) G = kGridMax / IPA_GQ;              // partials: K x IPA_GQ x G doubles fit the K x kGridMax area
  const int vec_ok = ((uintptr_t)x_dev % 16) == 0;
  const int groups = (K + IPA_GKB - 1) / IPA_GKB;
  auto kern = (K == 1) ? ipa_nll_grad_kernel<true> : ipa_nll_grad_kernel<false>;
  // programmatic dependent of the prologue kernel just before it (as the streaming kernel of ipa_nll_eval)
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)G, (unsigned)groups);
  cfg.blockDim = dim3(IPA_GB);
  cfg.dynamicSmemBytes = kGradSmem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  IPA_CK(cudaLaunchKernelEx(&cfg, kern, x_dev, (long long)n, vec_ok, reinterpret_cast<const IpaSetConsts*>(ws + L.consts), K,
                            reinterpret_cast<double*>(ws + L.partials), reinterpret_cast<unsigned int*>(ws + L.counter),
                            nll_dev, grad_dev, status_dev));
  return IPA_OK;
}

static int segmented_common(const double* x_dev, const int64_t* offsets_dev, int64_t T, const ipa_params* p_host,
                            int64_t K, const int32_t* set_of_segment_host, ipa_range r, double* nll_dev,
                            int32_t* status_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  const int policy = policy_of(opt_host);
  if (policy < 0) return IPA_ERR_INVALID_ARG;
  if (!x_dev || !offsets_dev || T < 1 || T > 0x7fffffffLL || K < 1 || K > 0x7fffffffLL || !p_host || !range_ok(r) ||
      !nll_dev)
    return IPA_ERR_INVALID_ARG;
  if (set_of_segment_host)
    for (int64_t t = 0; t < T; ++t)
      if (set_of_segment_host[t] < 0 || set_of_segment_host[t] >= K) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(T > K ? T : K, 0);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  const IpaSetConsts* consts = reinterpret_cast<const IpaSetConsts*>(ws + L.consts);
  double* partials = reinterpret_cast<double*>(ws + L.partials);
  const int* map = nullptr;
  if (set_of_segment_host) {   // the map travels through the (otherwise unused) yields area of the workspace
    IPA_CK(cudaMemcpyAsync(ws + L.nsig, set_of_segment_host, (size_t)T * 4, cudaMemcpyHostToDevice, st));
    map = reinterpret_cast<const int*>(ws + L.nsig);
  }
  // (the copy above comes first so that the segmented kernel directly follows the prologue: programmatic dependent launch)
  int rc = run_prologue(p_host, K, r, policy, ws, L, nullptr, nullptr, nullptr, st);
  if (rc) return rc;
  // chunks per segment: IPA_SEGC, more when few segments would leave SMs idle (T * C >= resident blocks of the device)
  int sms = 0;
  rc = device_info(&sms);
  if (rc) return rc;
  int64_t C = IPA_SEGC;
  const int64_t resident = (int64_t)sms * IPA_BLOCKS_PER_SM;
  if (T * C < resident) C = (resident + T - 1) / T;
  if (C > 64) C = 64;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)T, (unsigned)C);
  cfg.blockDim = dim3(IPA_BLOCK);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  IPA_CK(cudaLaunchKernelEx(&cfg, ipa_nll_seg_kernel, x_dev, reinterpret_cast<const long long*>(offsets_dev), consts, map,
                            partials));
  ipa_seg_finalize_kernel<<<(unsigned)((T + 127) / 128), 128, 0, st>>>(partials, consts, map, T, (int)C, nll_dev, status_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_nll_eval_segmented(const double* x_dev, const int64_t* offsets_dev, int64_t T, const ipa_params* p_host,
                           ipa_range r, double* nll_dev, int32_t* status_dev, const ipa_options* opt_host, void* ws_dev,
                           size_t ws_bytes, void* cuda_stream) {
  return segmented_common(x_dev, offsets_dev, T, p_host, T, nullptr, r, nll_dev, status_dev, opt_host, ws_dev, ws_bytes,
                          cuda_stream);
}

int ipa_nll_eval_categories(const double* x_dev, const int64_t* offsets_dev, int64_t T, const ipa_params* p_host, int64_t K,
                            const int32_t* set_of_segment_host, ipa_range r, double* nll_dev, int32_t* status_dev,
                            const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (!set_of_segment_host) return IPA_ERR_INVALID_ARG;
  return segmented_common(x_dev, offsets_dev, T, p_host, K, set_of_segment_host, r, nll_dev, status_dev, opt_host, ws_dev,
                          ws_bytes, cuda_stream);
}

int ipa_toy_generate(const uint64_t* seeds_host, int64_t T, const ipa_params* gen_host, int64_t gen_count,
                     double mean_sig, double mean_bkg, ipa_range r, int64_t capacity, double* x_dev,
                     int64_t* offsets_dev, int32_t* overflow_dev, int32_t* status_dev, const ipa_options* opt_host,
                     void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  const int policy = policy_of(opt_host);
  if (policy < 0) return IPA_ERR_INVALID_ARG;
  const bool mixture = (mean_sig < 0.0) || (mean_bkg < 0.0);
  if (!seeds_host || T < 1 || T > 0x7fffffffLL || !gen_host || (gen_count != 1 && gen_count != T) || !range_ok(r) ||
      capacity < 0 || (capacity > 0 && !x_dev) || !offsets_dev)
    return IPA_ERR_INVALID_ARG;
  if (mixture && T != 1) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(T, 0);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  int sms = 0;
  int rc = device_info(&sms);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  rc = run_prologue(gen_host, gen_count, r, policy, ws, L, nullptr, nullptr, status_dev, st);
  if (rc) return rc;
  IPA_CK(cudaMemcpyAsync(ws + L.seeds, seeds_host, (size_t)T * 8, cudaMemcpyHostToDevice, st));
  const unsigned long long* seeds = reinterpret_cast<const unsigned long long*>(ws + L.seeds);
  const IpaSetConsts* consts = reinterpret_cast<const IpaSetConsts*>(ws + L.consts);
  long long* nsig = reinterpret_cast<long long*>(ws + L.nsig);
  long long* ntot = reinterpret_cast<long long*>(ws + L.ntot);
  long long* offsets = reinterpret_cast<long long*>(offsets_dev);
  int64_t chunks;
  if (mixture) {
    // offsets = {0, capacity}
    const long long two[2] = {0, (long long)capacity};
    IPA_CK(cudaMemcpyAsync(offsets, two, sizeof(two), cudaMemcpyHostToDevice, st));
    if (overflow_dev) IPA_CK(cudaMemsetAsync(overflow_dev, 0, sizeof(int32_t), st));
    chunks = (capacity + IPA_BLOCK - 1) / IPA_BLOCK;
    if (chunks > (int64_t)sms * 16) chunks = (int64_t)sms * 16;
  } else {
    ipa_toy_yields_kernel<<<(unsigned)((T + 127) / 128), 128, 0, st>>>(seeds, T, mean_sig, mean_bkg, nsig, ntot);
    IPA_CK(cudaGetLastError());
    ipa_scan_kernel<<<1, 1024, 0, st>>>(ntot, T, offsets, capacity, overflow_dev);
    IPA_CK(cudaGetLastError());
    chunks = ((int64_t)sms * 16 + T - 1) / T;
    if (chunks > 1024) chunks = 1024;
  }
  if (chunks < 1) chunks = 1;
  if (capacity > 0) {
    ipa_toy_events_kernel<<<dim3((unsigned)T, (unsigned)chunks), IPA_BLOCK, 0, st>>>(
        seeds, consts, gen_count == T && T > 1 ? 1 : 0, nsig, offsets, r.lo, r.hi, capacity, mixture ? 1 : 0,
        (mixture && opt_host) ? (long long)opt_host->first_slot : 0LL, x_dev, overflow_dev);
    IPA_CK(cudaGetLastError());
  }
  return IPA_OK;
}

int ipa_hist_fill(const double* x_dev, int64_t n, ipa_range r, int nbins, uint64_t* counts_dev, void* cuda_stream) {
  if (n < 0 || (n > 0 && !x_dev) || !range_ok(r) || nbins < 1 || !counts_dev) return IPA_ERR_INVALID_ARG;
  int sms = 0;
  int rc = device_info(&sms);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  IPA_CK(cudaMemsetAsync(counts_dev, 0, (size_t)nbins * 8, st));
  if (n == 0) return IPA_OK;
  int64_t G = (n + 255) / 256;
  if (G > (int64_t)sms * 8) G = (int64_t)sms * 8;
  const size_t hsmem = nbins <= IPA_HIST_SMEM_BINS ? (size_t)nbins * 4 : 0;
  ipa_hist_kernel<<<(unsigned)G, 256, hsmem, st>>>(x_dev, n, r.lo, r.hi, nbins,
                                               reinterpret_cast<unsigned long long*>(counts_dev));
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

static int binned_common(const uint64_t* counts_dev, int nbins, ipa_range r, const ipa_params* shape_host,
                         const double* sig_dev, const double* ns_host, const double* nb_host, const double* k_host, int64_t npoints,
                         double* nll_dev, double* nu_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes,
                         void* cuda_stream) {
  const int policy = policy_of(opt_host);
  if (policy < 0) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(npoints, nbins);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  double* sbin = reinterpret_cast<double*>(ws + L.sbin);
  int32_t* flag = reinterpret_cast<int32_t*>(ws + L.flag);
  double* pts = reinterpret_cast<double*>(ws + L.pts);
  if (sig_dev) {   // a given signal shape (row f3)
    ipa_shape_normalise_kernel<<<1, 256, 0, st>>>(sig_dev, nbins, sbin, flag);
  } else {
    ipa_params shape = *shape_host;
    shape.f = 0.5;  // f and k of the shape set are not used by the binned path
    shape.k = 0.0;
    int rc = run_prologue(&shape, 1, r, policy, ws, L, nullptr, nullptr, nullptr, st);
    if (rc) return rc;
    ipa_binned_shape_kernel<<<1, 256, 0, st>>>(reinterpret_cast<const IpaSetConsts*>(ws + L.consts), r.lo, r.hi, nbins, sbin,
                                               flag, 1);
  }
  IPA_CK(cudaGetLastError());
  if (nb_host == ns_host + npoints && k_host == nb_host + npoints) {
    // the three arrays lie back to back in host memory (the Python binding packs them so): one upload instead of three
    IPA_CK(cudaMemcpyAsync(pts, ns_host, (size_t)npoints * 24, cudaMemcpyHostToDevice, st));
  } else {
    IPA_CK(cudaMemcpyAsync(pts, ns_host, (size_t)npoints * 8, cudaMemcpyHostToDevice, st));
    IPA_CK(cudaMemcpyAsync(pts + npoints, nb_host, (size_t)npoints * 8, cudaMemcpyHostToDevice, st));
    IPA_CK(cudaMemcpyAsync(pts + 2 * npoints, k_host, (size_t)npoints * 8, cudaMemcpyHostToDevice, st));
  }
  ipa_binned_scan_kernel<<<(unsigned)npoints, IPA_SCAN_THREADS, 0, st>>>(reinterpret_cast<const unsigned long long*>(counts_dev), sbin,
                                                            nbins, r.lo, r.hi, pts, pts + npoints, pts + 2 * npoints, flag,
                                                            nll_dev, nu_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_binned_nll_scan(const uint64_t* counts_dev, int nbins, ipa_range r, const ipa_params* shape_host,
                        const double* ns_host, const double* nb_host, const double* k_host, int64_t npoints,
                        double* nll_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (!counts_dev || nbins < 1 || !range_ok(r) || !shape_host || !ns_host || !nb_host || !k_host || npoints < 1 ||
      npoints > 0x7fffffffLL || !nll_dev)
    return IPA_ERR_INVALID_ARG;
  return binned_common(counts_dev, nbins, r, shape_host, nullptr, ns_host, nb_host, k_host, npoints, nll_dev, nullptr, opt_host,
                       ws_dev, ws_bytes, cuda_stream);
}

int ipa_expected_hist(int nbins, ipa_range r, const ipa_params* shape_host, double ns, double nb, double k,
                      double* nu_dev, const ipa_options* opt_host, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (nbins < 1 || !range_ok(r) || !shape_host || !nu_dev) return IPA_ERR_INVALID_ARG;
  return binned_common(nullptr, nbins, r, shape_host, nullptr, &ns, &nb, &k, 1, nullptr, nu_dev, opt_host, ws_dev, ws_bytes,
                       cuda_stream);
}

int ipa_signal_shape(int nbins, ipa_range r, const ipa_params* shape_host, double* sig_dev, const ipa_options* opt_host,
                     void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  const int policy = policy_of(opt_host);
  if (nbins < 1 || !range_ok(r) || !shape_host || !sig_dev || policy < 0) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(1, nbins);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  ipa_params shape = *shape_host;
  shape.f = 0.5;
  shape.k = 0.0;
  int rc = run_prologue(&shape, 1, r, policy, ws, L, nullptr, nullptr, nullptr, st);
  if (rc) return rc;
  ipa_binned_shape_kernel<<<1, 256, 0, st>>>(reinterpret_cast<const IpaSetConsts*>(ws + L.consts), r.lo, r.hi, nbins, sig_dev,
                                             reinterpret_cast<int32_t*>(ws + L.flag), 0);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_gauss_smear(const double* in_dev, int nbins, ipa_range r, double sigma0, double* out_dev, void* cuda_stream) {
  if (!in_dev || !out_dev || in_dev == out_dev || nbins < 1 || !range_ok(r) || !ipa_finite(sigma0)) return IPA_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (!(sigma0 > 0.0)) {
    IPA_CK(cudaMemcpyAsync(out_dev, in_dev, (size_t)nbins * 8, cudaMemcpyDeviceToDevice, st));
    return IPA_OK;
  }
  const double w = (r.hi - r.lo) / (double)nbins;
  const double Md = ceil(8.0 * sigma0 / w);
  if (!(Md <= 2800.0)) return IPA_ERR_INVALID_ARG;               // 2M+1 taps must fit 48 KB of shared memory
  const int M = (int)Md;
  ipa_gauss_smear_kernel<<<(nbins + 255) / 256, 256, (size_t)(2 * M + 1) * 8, st>>>(in_dev, nbins, w, sigma0, M, out_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_expected_hist_shape(int nbins, ipa_range r, const double* sig_dev, double ns, double nb, double k, double* nu_dev,
                            void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (nbins < 1 || !range_ok(r) || !sig_dev || !nu_dev) return IPA_ERR_INVALID_ARG;
  return binned_common(nullptr, nbins, r, nullptr, sig_dev, &ns, &nb, &k, 1, nullptr, nu_dev, nullptr, ws_dev, ws_bytes, cuda_stream);
}

int ipa_binned_nll_scan_shape(const uint64_t* counts_dev, int nbins, ipa_range r, const double* sig_dev,
                              const double* ns_host, const double* nb_host, const double* k_host, int64_t npoints,
                              double* nll_dev, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (!counts_dev || nbins < 1 || !range_ok(r) || !sig_dev || !ns_host || !nb_host || !k_host || npoints < 1 ||
      npoints > 0x7fffffffLL || !nll_dev)
    return IPA_ERR_INVALID_ARG;
  return binned_common(counts_dev, nbins, r, nullptr, sig_dev, ns_host, nb_host, k_host, npoints, nll_dev, nullptr, nullptr,
                       ws_dev, ws_bytes, cuda_stream);
}

int ipa_poisson_hist_toys(const double* mean_dev, int nbins, const uint64_t* seeds_host, int64_t T,
                          uint32_t* counts_dev, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (!mean_dev || nbins < 1 || !seeds_host || T < 1 || !counts_dev) return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(T, 0);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  int sms = 0;
  int rc = device_info(&sms);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  IPA_CK(cudaMemcpyAsync(ws + L.seeds, seeds_host, (size_t)T * 8, cudaMemcpyHostToDevice, st));
  int bw = 256;                                                      // bins per block: a power of two
  while (bw > 1 && bw / 2 >= nbins) bw /= 2;
  const int64_t gx = ((int64_t)nbins + bw - 1) / bw;                 // bins across the threads, toys in chunks over grid y
  int64_t gy = ((int64_t)sms * 8 + gx - 1) / gx;
  const int64_t tgroups = (T + 256 / bw - 1) / (256 / bw);
  if (gy > tgroups) gy = tgroups;
  if (gy > 65535) gy = 65535;
  if (gy < 1) gy = 1;
  ipa_poisson_hist_kernel<<<dim3((unsigned)gx, (unsigned)gy), 256, 0, st>>>(mean_dev, nbins, bw,
                                                       reinterpret_cast<const unsigned long long*>(ws + L.seeds), T,
                                                       counts_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_cls_teststat(const void* counts_dev, int count_bytes, int64_t T, int nbins, const double* nu_sb_dev,
                     const double* nu_b_dev, double* q_dev, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (!counts_dev || (count_bytes != 4 && count_bytes != 8) || T < 1 || T > 0x7fffffffLL || nbins < 1 || !nu_sb_dev ||
      !nu_b_dev || !q_dev)
    return IPA_ERR_INVALID_ARG;
  const Layout L = make_layout(1, nbins);
  if (!ws_ok(ws_dev, ws_bytes, L.total)) return IPA_ERR_WORKSPACE;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(ws_dev);
  double* lr = reinterpret_cast<double*>(ws + L.sbin);
  double* csum = reinterpret_cast<double*>(ws + L.pts);
  ipa_cls_weights_kernel<<<1, 256, 0, st>>>(nu_sb_dev, nu_b_dev, nbins, lr, csum);
  IPA_CK(cudaGetLastError());
  // 128-bit loads need 16-byte aligned rows (and the weights are read in pairs)
  const int vec_ok = (((uintptr_t)counts_dev % 16) == 0 && ((size_t)nbins * (size_t)count_bytes) % 16 == 0) ? 1 : 0;
  const unsigned G = (unsigned)((T + 7) / 8);
  if (count_bytes == 4)
    ipa_cls_q_kernel<unsigned int><<<G, 256, 0, st>>>(static_cast<const unsigned int*>(counts_dev), T, nbins, vec_ok, lr,
                                                      csum, q_dev);
  else
    ipa_cls_q_kernel<unsigned long long><<<G, 256, 0, st>>>(static_cast<const unsigned long long*>(counts_dev), T, nbins,
                                                            vec_ok, lr, csum, q_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_cls_count_ge(const double* q_dev, int64_t T, const double* q_obs_dev, int64_t* count_dev, void* cuda_stream) {
  if (!q_dev || T < 1 || !q_obs_dev || !count_dev) return IPA_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  IPA_CK(cudaMemsetAsync(count_dev, 0, 8, st));
  int64_t G = (T + 255) / 256;
  if (G > 1184) G = 1184;
  ipa_cls_count_kernel<<<(unsigned)G, 256, 0, st>>>(q_dev, T, q_obs_dev, reinterpret_cast<unsigned long long*>(count_dev));
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_cls_from_counts(const int64_t* count_sb_dev, int64_t T_sb, const int64_t* count_b_dev, int64_t T_b,
                        double* cl_dev, void* cuda_stream) {
  if (!count_sb_dev || !count_b_dev || T_sb < 1 || T_b < 1 || !cl_dev) return IPA_ERR_INVALID_ARG;
  ipa_cls_from_counts_kernel<<<1, 1, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
      reinterpret_cast<const long long*>(count_sb_dev), T_sb, reinterpret_cast<const long long*>(count_b_dev), T_b, cl_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

// grid of the unsegmented preparation: two resident blocks per SM, never more blocks than tiles
static int64_t prep_grid(int64_t n, int sms) {
  const int64_t tiles = (n + IPA_PREP_TILE - 1) / IPA_PREP_TILE;
  int64_t G = IPA_PREP_BLOCKS_PER_SM * (int64_t)(sms > 0 ? sms : 148);
  if (G > tiles) G = tiles;
  return G < 1 ? 1 : G;
}

size_t ipa_prepare_workspace_bytes(int64_t n, int64_t T) {
  if (n < 0 || T < 0) return 0;
  if (T > 0) return 256;                                       // segmented: everything lives in shared memory
  const int64_t Gmax = prep_grid(n, 1024);                     // upper bound over any device (<= 2048 blocks)
  return align_up((size_t)IPA_PREP_BINS * (size_t)Gmax * 4, 256) + 2 * align_up((size_t)IPA_PREP_BINS * 8, 256);
}

int ipa_events_prepare(const double* x_in_dev, int64_t n, const int64_t* offsets_dev, int64_t T, ipa_range r,
                       double* x_out_dev, void* ws_dev, size_t ws_bytes, void* cuda_stream) {
  if (n < 0 || T < 0 || n > 0xffffffffLL || (n > 0 && (!x_in_dev || !x_out_dev || x_in_dev == x_out_dev)) || !range_ok(r))
    return IPA_ERR_INVALID_ARG;
  if (offsets_dev && (T < 1 || T > 0x7fffffffLL)) return IPA_ERR_INVALID_ARG;
  if (!offsets_dev) T = 0;
  if (n == 0) return IPA_OK;
  if (!ws_ok(ws_dev, ws_bytes, ipa_prepare_workspace_bytes(n, T))) return IPA_ERR_WORKSPACE;
  int sms = 0;
  int rc = device_info(&sms);
  if (rc) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const double scale = (double)IPA_PREP_BINS / (r.hi - r.lo);
  if (T > 0) {
    ipa_prep_segment_kernel<<<(unsigned)T, IPA_PREP_THREADS, IPA_PREP_SMEM, st>>>(
        x_in_dev, reinterpret_cast<const long long*>(offsets_dev), r.lo, scale, x_out_dev);
    IPA_CK(cudaGetLastError());
    return IPA_OK;
  }
  const int64_t G = prep_grid(n, sms);
  char* ws = static_cast<char*>(ws_dev);
  unsigned int* hist = reinterpret_cast<unsigned int*>(ws);
  size_t o = align_up((size_t)IPA_PREP_BINS * (size_t)G * 4, 256);
  unsigned long long* bintot = reinterpret_cast<unsigned long long*>(ws + o);
  unsigned long long* binbase = reinterpret_cast<unsigned long long*>(ws + o + align_up((size_t)IPA_PREP_BINS * 8, 256));
  ipa_prep_hist_kernel<<<(unsigned)G, IPA_PREP_THREADS, 0, st>>>(x_in_dev, n, r.lo, scale, hist);
  IPA_CK(cudaGetLastError());
  ipa_prep_scan_kernel<<<IPA_PREP_BINS / 8, 256, 0, st>>>(hist, (int)G, bintot);
  IPA_CK(cudaGetLastError());
  ipa_prep_binscan_kernel<<<1, IPA_PREP_BINS, 0, st>>>(bintot, binbase);
  IPA_CK(cudaGetLastError());
  ipa_prep_scatter_kernel<<<(unsigned)G, IPA_PREP_THREADS, IPA_PREP_SMEM, st>>>(x_in_dev, n, r.lo, scale, hist, binbase, x_out_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

int ipa_nll_eval_static(const double* x_dev, int64_t n, const ipa_params* p_host, int K, ipa_range r, double* nll_dev,
                        double* logpdf_dev, int32_t* status_dev, const ipa_options* opt_host, void* cuda_stream) {
  if (K > IPA_STATIC_MAX_K) {
    g_last_cuda_error = "ipa_nll_eval_static: K = " + std::to_string(K) + " parameter sets exceed IPA_STATIC_MAX_K = " +
                        std::to_string(IPA_STATIC_MAX_K) + " (use ipa_nll_eval with a workspace of your own)";
    return IPA_ERR_TOO_LARGE;
  }
  void* ws = nullptr;
  const int rc = static_scratch(&ws);
  if (rc) return rc;
  // the existing path, on the built-in scratch: the prologue rewrites every record of the K sets and zeroes the ticket
  // counters, the streaming kernel writes all the partial sums it later reads -- nothing of an earlier call is read
  return ipa_nll_eval(x_dev, n, p_host, K, r, nll_dev, logpdf_dev, status_dev, opt_host, ws, IPA_STATIC_SCRATCH_BYTES,
                      cuda_stream);
}

int ipa_fp64_peak_probe(int64_t iters, double* out_dev, void* cuda_stream) {
  if (iters < 1 || !out_dev) return IPA_ERR_INVALID_ARG;
  int sms = 0;
  int rc = device_info(&sms);
  if (rc) return rc;
  ipa_fp64_probe_kernel<<<(unsigned)(sms * 8), 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(iters, out_dev);
  IPA_CK(cudaGetLastError());
  return IPA_OK;
}

}  // extern "C"
