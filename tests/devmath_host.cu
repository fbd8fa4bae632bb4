// Test helper (tests/test_devmath_host.py): compiles the CUDA path's __host__ __device__ arithmetic
// (paper_1706_01420_b200/csrc/*.cuh) for the CPU and runs the prologue phases serially, so that the
// kernel math can be checked against the oracle on the GPU-less build box.  TEST ONLY: the product
// library never executes these functions on the host and nothing in the package links this file.
#include <cstring>
#include <vector>
#include "../paper_1706_01420_b200/csrc/ipa_kernels.cuh"

static void run_prologue_host(const ipa_params& p, double lo, double hi, int policy, IpaSetConsts* out) {
  static IpaProWork w;
  std::memset(&w, 0, sizeof(w));
  std::memset(out, 0, sizeof(*out));
  w.p = p; w.lo = lo; w.hi = hi; w.policy = policy; w.want_grad = 1;
  const int NT = IPA_PRO_THREADS;
#define ALL(stmt) for (int tid = 0; tid < NT; ++tid) { stmt; }
  ALL(ipa_pro_load_table(w, tid, NT))
  ALL(ipa_pro_phase0(w, tid))
  ALL(ipa_pro_phase1(w, tid))
  ALL(ipa_pro_phase2(w, tid))
  ALL(ipa_pro_phase3(w, tid, NT))
  ALL(ipa_pro_phase4(w, tid))
  ALL(ipa_pro_phase5(w, tid))
  ALL(ipa_pro_phase6(w, tid))
  ALL(ipa_pro_phase7(w, tid))
  ALL(ipa_pro_phase7b(w, tid))
  ALL(ipa_pro_phase8_finish(w, tid); ipa_pro_cells_nodes(w, tid))
  ALL(ipa_pro_phase9(w, tid); ipa_pro_cells_dct(w, tid))
  ALL(ipa_pro_phase10(w, tid, NT))
  ALL(ipa_pro_phase11(w, tid); ipa_pro_cells_monomial(w, ipa_pro_cells_slot(tid)))
  ALL(ipa_pro_phase12(w, *out, tid); ipa_pro_cells_record(w, *out, tid))
  ALL(ipa_pro_phase13(w, *out, tid))
#undef ALL
}

extern "C" {
int emu_sizeof_consts() { return (int)sizeof(IpaSetConsts); }
double emu_besselk_scaled(double nu, double x) { return ipa_besselk_scaled(nu, x); }
// out: status, degree, mode, normS, normB, delta2, alpha, logG0, logG1, L0 (= -uA0 n0), L1, d ln N_S/d mu,
// d ln N_S/d sigma, d ln N_B/d k, d ln N_S/d beta
void emu_consts(const ipa_params* p, double lo, double hi, int policy, double* out) {
  IpaSetConsts c;
  run_prologue_host(*p, lo, hi, policy, &c);
  out[0] = c.status; out[1] = c.degree; out[2] = c.mode; out[3] = c.normS; out[4] = c.normB;
  out[5] = c.delta2; out[6] = c.alpha; out[7] = c.logG0; out[8] = c.logG1; out[9] = -c.uA0 * c.n0; out[10] = -c.uA1 * c.n1;
  out[11] = c.dlnNS_dmu; out[12] = c.dlnNS_dsig; out[13] = c.dlnNB_dk; out[14] = c.dlnNS_dbeta;
}
// cells of the core: out = ncell, 4 sng[], 8 hb[]
void emu_cells(const ipa_params* p, double lo, double hi, int policy, int* out) {
  IpaSetConsts c;
  run_prologue_host(*p, lo, hi, policy, &c);
  out[0] = c.ncell;
  for (int s = 0; s < IPA_NCELL; ++s) out[1 + s] = c.sng[s];
  for (int i = 0; i < 8; ++i) out[1 + IPA_NCELL + i] = c.hb[i];
}
void emu_logpdf(const ipa_params* p, double lo, double hi, int policy, const double* x, long long n, double* out) {
  IpaSetConsts c;
  run_prologue_host(*p, lo, hi, policy, &c);
  for (long long i = 0; i < n; i += 8) {
    double xv[8], l[8];
    for (int e = 0; e < 8; ++e) xv[e] = (i + e < n) ? x[i + e] : x[n - 1];
    if (c.status) { for (int e = 0; e < 8; ++e) l[e] = -INFINITY; }
    else ipa_eval_set<8>(c, xv, l, ipa_h_mathtab);
    for (int e = 0; e < 8 && i + e < n; ++e) out[i + e] = l[e];
  }
}
// row f1: sums of l and of the five derivative contributions over n events (plain left-to-right sums)
void emu_grad(const ipa_params* p, double lo, double hi, int policy, const double* x, long long n, double* out) {
  IpaSetConsts c;
  run_prologue_host(*p, lo, hi, policy, &c);
  for (int q = 0; q < 6; ++q) out[q] = 0.0;
  for (long long i = 0; i < n; i += 4) {
    double xv[4], l[4], gm[4], gs[4], gf[4], gk[4], gb[4];
    for (int e = 0; e < 4; ++e) xv[e] = (i + e < n) ? x[i + e] : x[n - 1];
    ipa_eval_grad<4>(c, xv, l, gm, gs, gf, gk, gb, ipa_h_mathtab);
    for (int e = 0; e < 4 && i + e < n; ++e) {
      out[0] -= l[e]; out[1] -= gm[e]; out[2] -= gs[e]; out[3] -= gf[e]; out[4] -= gk[e]; out[5] -= gb[e];
    }
  }
}
void emu_logI(const ipa_params* p, double lo, double hi, const double* d, long long n, double* out) {
  IpaSetConsts c;
  run_prologue_host(*p, lo, hi, 0, &c);
  for (long long i = 0; i < n; ++i) out[i] = ipa_logI_rec(c, d[i]);
}
void emu_uniforms2(unsigned long long seed, unsigned long long slot, unsigned attempt, unsigned stream, double* u) {
  ipa_uniforms2(seed, slot, attempt, stream, u, u + 1);
}
// generated 16-point Gauss-Legendre table against the in-source Newton iteration on P_16
void emu_gl16(double* tab_x, double* tab_w, double* newton_x, double* newton_w) {
  for (int i = 0; i < 16; ++i) {
    tab_x[i] = IPA_GL16X(i); tab_w[i] = IPA_GL16W(i);
    ipa_gauss_legendre(16, i, &newton_x[i], &newton_w[i]);
  }
}
// generated integer Chebyshev table against the three-term recurrence; returns the number of mismatches
int emu_cheb_table_mismatches() {
  static long long T[IPA_CHEB_NC][IPA_CHEB_NC];
  int bad = 0;
  for (int j = 0; j < IPA_CHEB_NC; ++j)
    for (int k = 0; k < IPA_CHEB_NC; ++k) {
      long long v;
      if (j == 0) v = (k == 0);
      else if (j == 1) v = (k == 1);
      else v = (k > 0 ? 2 * T[j - 1][k - 1] : 0) - T[j - 2][k];
      T[j][k] = v;
      bad += (IPA_CHEBT(j, k) != v);
    }
  return bad;
}
long long emu_poisson(unsigned long long seed, unsigned long long slot, unsigned stream, double mean) {
  return ipa_poisson(seed, slot, stream, mean);
}
}

// ---- the streaming kernels' own sqrt / exp / log (csrc/ipa_fastmath.cuh) ---------------------------
extern "C" {
void emu_frcp3(const double* u, long long n, double* out) { for (long long i = 0; i < n; ++i) out[i] = ipa_frcp3(u[i]); }
void emu_fsqrt_rsqrt(const double* q, long long n, double* r, double* rinv) {
  for (long long i = 0; i < n; ++i) r[i] = ipa_fsqrt_rsqrt(q[i], &rinv[i]);
}
void emu_fsqrt(const double* q, long long n, double* out) { for (long long i = 0; i < n; ++i) out[i] = ipa_fsqrt(q[i]); }
void emu_fexp_neg(const double* a, long long n, double* out) {
  for (long long i = 0; i < n; ++i) out[i] = ipa_fexp_neg(ipa_neg_abs_clamped(a[i]));
}
void emu_flog(const double* u, long long n, double* out) { for (long long i = 0; i < n; ++i) out[i] = ipa_flog(u[i], ipa_h_logtab); }
void emu_fsoftplus(const double* D, long long n, double* out) {
  for (long long i = 0; i < n; ++i) out[i] = ipa_fsoftplus(D[i], ipa_h_logtab);
}
// table-driven versions of the streaming kernels (round 2)
void emu_fexp_negabs_t(const double* a, long long n, double* out) { for (long long i = 0; i < n; ++i) out[i] = ipa_fexp_negabs_t(a[i], ipa_h_mathtab); }
void emu_flog_t(const double* u, long long n, double* out) { for (long long i = 0; i < n; ++i) out[i] = ipa_flog_t(u[i], ipa_h_mathtab); }
void emu_flog12_t(const double* u, long long n, double* out) { for (long long i = 0; i < n; ++i) out[i] = ipa_flog12_t(u[i], ipa_h_mathtab); }
void emu_fsoftplus_add_t(const double* eb, const double* D, long long n, double* out) {
  for (long long i = 0; i < n; ++i) out[i] = ipa_fsoftplus_add_t(eb[i], D[i], ipa_h_mathtab);
}
}
