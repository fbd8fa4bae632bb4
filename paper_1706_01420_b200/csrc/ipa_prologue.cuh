// ipa_prologue.cuh -- per-parameter-set constants ("precomputed once per launch", north star):
// steps A1a-A1e of DESIGN.md.  One thread block per parameter set runs the phases below with a
// __syncthreads() between them; tests/devmath_host.cu runs the same phases serially on the CPU.
//
//   A1a  delta, alpha from K_lambda(zeta), K_{lambda+1}(zeta)                      (reading C1)
//   A1b  joins d0, d1: log G and log-derivative L = beta - alpha (d/r) K_{nu-1}/K_nu (reading C1)
//   A1e  core approximant: Chebyshev interpolation of  H(z) = log( z^nu K_nu(z) )  on
//        z in [zeta, zmax] (the core region maps onto exactly this interval, whatever mu and sigma
//        are), truncated at the fp64 noise floor and converted exactly (integer Chebyshev
//        coefficients, double-double accumulation) to a monomial in t = tA r + tB for Horner.
//   A1c  N_S: closed-form tails + 16-point Gauss-Legendre on panels [b, max(delta, 3b)] of the core
//        (each panel keeps the branch points d = +-i delta outside a Bernstein ellipse of
//        parameter >= 3.7, so 16 nodes give < 1e-18)                               (reading C5)
//   A1d  N_B = expm1(k (hi-lo)) / k
//   A1e  folded constants so that the per-event work is  Delta = E_S - E_B  and
//        l = E_B + log(1 + e^Delta).
#pragma once
#include "ipa_math.cuh"
#include "../../include/ipanll.h"

#define IPA_NCOEF 48            // max polynomial degree 47
#define IPA_MCHEB 64            // Chebyshev nodes of the core approximant
#define IPA_JMAX 256            // trapezoid table length
#define IPA_GL 16               // Gauss-Legendre nodes per panel
#define IPA_MAXPANEL 24         // 12 per side
#define IPA_PRO_THREADS 256
#define IPA_SUB 2               // threads sharing one table-based Bessel evaluation
#define IPA_NBTASK (IPA_MCHEB + 4)  // Chebyshev nodes + K_nu(z0), K_nu(z1), K_{nu-1}(z0), K_{nu-1}(z1)
#define IPA_NCELL 4              // cells of the core in r = sqrt(d^2 + delta^2), each with its own low-degree polynomial
#define IPA_CELLN 16             // coefficients per cell polynomial (degree <= 15)
#define IPA_CELLM 32             // Chebyshev nodes per cell
#define IPA_CELL_MIN_DEGREE 16   // cells only where the full polynomial is longer than a cell polynomial can be

// What the streaming kernels read, per parameter set (all fp64 except the flags).
struct alignas(16) IpaSetConsts {
  double a[IPA_NCOEF];          // Delta_core = sum_j a[j] t^j + bmk d   (a[0] carries the constants; zero above
                                // the degree, so Horner may start at any index >= degree).  16-byte aligned:
                                // the streaming kernel reads coefficient pairs with 128-bit shared loads.
  double mu, delta2;            // d = x - mu, r = sqrt(d^2 + delta2)
  double tA, tB;                // t = tA r + tB in [-1,1] on the core
  double d0, d1;                // joins
  double bmk, kd;               // beta - kd;  E_B = kd d + eB0   (kd = k; both 0 for f == 1)
  double eB0, araw0;            // araw0 = a[0] before folding: H(z) itself = sum araw t^j
  double uA0, uB0, n0, cT0;     // left tail:  u = uA0 d + uB0,  Delta = cT0 - n0 log u - kd d
  double uA1, uB1, n1, cT1;     // right tail
  double alpha, nu, cDir;       // direct mode: Delta = H(alpha r) + bmk d + cDir, H(z) = log(z^nu K_nu(z))
  double fsig, kraw;            // f and k as given (generators)
  double beta, logG0, logG1, logNS, logref;  // for the generators / binned path: log I(d)
  double normS, normB;          // N_S, N_B (absolute)
  // gradient kernel (row f1): derivatives of the normalisations and the constants of d log I / d (d, sigma)
  double dlnNS_dmu, dlnNS_dsig, dlnNB_dk, nuosig;   // nuosig = nu / sigma
  double invsig, mulo, L0, L1;                      // 1 / sigma, mu - lo, join slopes
  double A0, A1, aL0, a2L1;                         // nu/sigma - a beta, nu/sigma + a2 beta, a L0, a2 L1
  double c0s, c1s, invf, inv1mf;                    // (L0 - beta)/sigma, (L1 - beta)/sigma, 1/f, 1/(1-f)
  double dlnNS_dbeta, pad2;                         // d ln N_S / d beta (fifth gradient component)
  int32_t status, degree, mode, pure;
  int32_t hxl, hxr, pad0, pad1; // high words of the joins in x, mu+d0 and mu+d1 (0 / -1 if not positive): region
                                // classification of a whole warp by integer min/max of the events' high words
  // Cells of the core (streaming and segmented kernels).  The core interval of r = sqrt(d^2 + delta^2) is cut into
  // IPA_NCELL cells of equal ratio; cell s has its own polynomial in t_s = stA[s] r + stB[s], refitted from the
  // full one: H(alpha r) - araw0 = sa[s][0] + sum_{j>=1} sa[s][j] t_s^j, of degree 4 sng[s] + 3 at most (14 where the full
  // interval needs 27).  A warp whose events all lie in one cell (a warp of a prepared array nearly always does)
  // runs the cell polynomial; any other warp runs the full one.  The cell of an event is decided on the high word
  // of x alone: hb[] holds the high words of the 2 (IPA_NCELL - 1) cell boundaries in x, ascending (0 / INT_MAX for a
  // boundary outside the core), each boundary a double with a zero low word, so that x >= boundary is exactly
  // hi(x) >= hb; cell = | #{i : hb[i] <= hi(x)} - (IPA_NCELL - 1) |.  ncell = 0: no cells (modes 1 and 2, a cell
  // degree above 15, a core too narrow for the 2^-20 relative resolution of the high word).
  double sa[IPA_NCELL][IPA_CELLN];
  double stA[IPA_NCELL], stB[IPA_NCELL];
  int32_t hb[8];
  int32_t sng[IPA_NCELL];
  int32_t ncell, cpad[3];
  int32_t sdeg[IPA_NCELL];      // degrees of the cell polynomials (ipa_core_cells reports them; the kernels run 4 sng + 3)
};

struct IpaProWork {
  ipa_params p;
  double lo, hi;
  int policy;
  int want_grad;                // compute the normalisation derivatives of the gradient call (row f1)
  int status;
  double nu, delta, alpha, d0, d1, r0, r1, z0, z1, zc, zh;
  double part[2][32];
  double Kl, Kl1;
  double glx[IPA_GL], glw[IPA_GL];
  // trapezoid table, orders |nu| (index 0) and |nu-1| (index 1)
  double h;
  int J;
  double tc[IPA_JMAX], te[2][IPA_JMAX], tw[2][IPA_JMAX];
  double bpart[IPA_NBTASK][IPA_SUB];
  double Ks[IPA_NBTASK];        // scaled Bessel values e^z K(z) of the tasks
  double H[IPA_MCHEB], c[IPA_MCHEB];
  double ctab[4 * IPA_MCHEB];   // cos(pi m / (2 M)), m = 0 .. 4M-1 (Chebyshev nodes and the cosine transform)
  double tl_left, tl_right, NB, logNB, logf, log1mf, nulogalpha, expref;
  double tl_left2, tl_right2, dlnNB_dk, Iedge_l, Iedge_h;   // sigma-derivative tail integrals, d ln N_B / d k, I at the range ends
  double tl_left3, tl_right3;                               // beta-derivative tail integrals
  double pval3[IPA_MAXPANEL * IPA_GL], psum3[IPA_MAXPANEL]; // core part of d N_S / d beta: G d
  double pval2[IPA_MAXPANEL * IPA_GL], psum2[IPA_MAXPANEL];   // pieces of phase 12 computed by other warps in phase 11
  int degree, mode;
  alignas(16) long long T[IPA_NCOEF * IPA_NCOEF];  // copy of the integer Chebyshev table (cp.async at kernel start, used in phase 8)
  double cDir;                          // per-set constant of the core term (phase 12 -> 13)
  double normS_abs;                     // N_S (absolute) for the norm outputs (NaN for an invalid set)
  double inv_sigma, inv_f, inv_1mf, inv_n0, inv_n1, inv_zh;   // reciprocals for phase 12, formed by idle threads in phase 11
  double hK[2];                         // trapezoid steps of K_lambda(zeta), K_{lambda+1}(zeta) (phase 1 -> phase 2)
  double hmax4[4];                      // max |H| over the four quarters of the Chebyshev nodes (phase 6 -> 7)
  int dq4[4];                           // highest coefficient index above the noise threshold, per quarter (phase 7 -> 7b)
  double araw[IPA_NCOEF];
  double logG0, logG1, L0, L1;
  int npanel;
  double pa[IPA_MAXPANEL], pb[IPA_MAXPANEL], pval[IPA_MAXPANEL * IPA_GL], psum[IPA_MAXPANEL];
  double logref, dl, dh;
  // cells of the core (phase 7 geometry, 8 values at the nodes, 9 Chebyshev coefficients, 11 monomials)
  int ncell;
  int chb[8];
  double crc[IPA_NCELL], crh[IPA_NCELL];
  double cH[IPA_NCELL][IPA_CELLM], cc[IPA_NCELL][IPA_CELLM];
  double csa[IPA_NCELL][IPA_CELLN];
  int cdeg[IPA_NCELL];
};

IPA_HD bool ipa_finite(double v) { return fabs(v) <= 1.7976931348623157e308; }

// ---- evaluation helpers shared by the prologue, the generators and the binned path ---------------
IPA_HD double ipa_horner(const double* a, int D, double t) {
  double acc = a[D];
  for (int j = D - 1; j >= 0; --j) acc = fma(acc, t, a[j]);
  return acc;
}

// table-based partial sum of e^z K(z): terms j = 1+sub, 1+sub+IPA_SUB, ... < J
IPA_HD double ipa_table_partial(const IpaProWork& w, int ord, double z, int sub) {
  double s = 0.0;
  for (int j = 1 + sub; j < w.J; j += IPA_SUB) s += w.tw[ord][j] * exp(w.te[ord][j] - z * w.tc[j]);
  return s;
}

// mode 2 (zeta == 0, lambda < 0: row f4, reading D3) is the Student-t core G = (d^2 + delta^2)^nu e^{beta d}, the zeta -> 0
// limit of the Bessel core: no Bessel function, no polynomial; G is homogeneous of degree 2 nu in sigma (nu otherwise)
IPA_HD double ipa_sigpow(const IpaProWork& w) { return w.mode == 2 ? 2.0 * w.nu : w.nu; }
// H(z) = log(z^nu K_nu(z)) from the raw polynomial, r given
IPA_HD double ipa_core_H(const IpaProWork& w, double r) {
  const double z = w.alpha * r;
  if (w.mode == 0) return ipa_horner(w.araw, w.degree, (z - w.zc) / w.zh);
  return w.nu * log(z) + log(ipa_besselk_scaled(w.nu, z)) - z;
}
// log G(d) = nu log r + beta d + log K_nu(alpha r) = H - nu log alpha + beta d
IPA_HD double ipa_core_logG(const IpaProWork& w, double d) {
  if (w.mode == 2) return fma(w.nu, log(fma(d, d, w.delta * w.delta)), w.p.beta * d);
  const double r = sqrt(fma(d, d, w.delta * w.delta));
  return ipa_core_H(w, r) - w.nu * log(w.alpha) + w.p.beta * d;
}
// L(d) - beta = -alpha (d/r) K_{nu-1}/K_nu = alpha (d/r) H'(z)  (H' = -K_{nu-1}/K_nu): derivative of the fitted
// polynomial, dH/dz = (1/zh) sum_j j a_j t^{j-1}; direct mode evaluates the Bessel ratio
IPA_HD double ipa_core_Lmb(const IpaProWork& w, double d) {
  if (w.mode == 2) return 2.0 * w.nu * d / fma(d, d, w.delta * w.delta);
  const double r = sqrt(fma(d, d, w.delta * w.delta));
  const double z = w.alpha * r;
  double Hp;
  if (w.mode == 0) {
    const double t = (z - w.zc) / w.zh;
    double acc = 0.0;
    for (int j = w.degree; j >= 1; --j) acc = fma(acc, t, (double)j * w.araw[j]);
    Hp = acc / w.zh;
  } else {
    Hp = -ipa_besselk_scaled(w.nu - 1.0, z) / ipa_besselk_scaled(w.nu, z);
  }
  return w.alpha * (d / r) * Hp;
}
IPA_HD double ipa_logI(const IpaProWork& w, double d) {
  if (d < w.d0) return w.logG0 - w.p.n * log(1.0 - (d - w.d0) * w.L0 / w.p.n);
  if (d > w.d1) return w.logG1 - w.p.n2 * log(1.0 - (d - w.d1) * w.L1 / w.p.n2);
  return ipa_core_logG(w, d);
}

// ================================ phases =========================================================
// before phase 0: every thread copies its share of the integer Chebyshev table into the work area (the
// loads are in flight during the first phases; per-lane reads from global memory in phase 8 cost as
// much as building the table)
IPA_HD void ipa_pro_load_table(IpaProWork& w, int tid, int nthr) {
#ifdef __CUDA_ARCH__
  // 16-byte asynchronous copies: nobody waits for the table before phase 8 (ipa_pro_table_ready)
  for (int i = tid; i < IPA_NCOEF * IPA_NCOEF / 2; i += nthr) {
    const unsigned dst = (unsigned)__cvta_generic_to_shared(&w.T[2 * i]);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(&ipa_d_chebT[2 * i]) : "memory");
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
#else
  for (int i = tid; i < IPA_NCOEF * IPA_NCOEF; i += nthr) w.T[i] = IPA_CHEBT(0, i);
#endif
}
// before the barrier that precedes phase 8
IPA_HD void ipa_pro_table_ready() {
#ifdef __CUDA_ARCH__
  asm volatile("cp.async.wait_group 0;" ::: "memory");
#endif
}

// phase 0: validation (one thread)
IPA_HD void ipa_pro_phase0(IpaProWork& w, int tid) {
  if (tid != 0) return;
  const ipa_params& p = w.p;
  const double* v = &p.mu;
  bool ok = true;
  for (int i = 0; i < 11; ++i) ok = ok && ipa_finite(v[i]);
  ok = ok && (p.sigma > 0.0) && (p.zeta > 0.0 || (p.zeta == 0.0 && p.lambda < 0.0)) && (p.a > 0.0) && (p.a2 > 0.0) && (p.n > 0.0) && (p.n2 > 0.0) &&
       (p.f >= 0.0) && (p.f <= 1.0);
  w.status = ok ? 0 : 1;
  w.nu = p.lambda - 0.5;
  w.mode = (p.zeta == 0.0) ? 2 : 0;
  w.degree = 0;
  w.npanel = 0;
}

// phase 1: partial trapezoid sums of K_lambda(zeta) (warp 0) and K_{lambda+1}(zeta) (warp 1);
// threads 64..79 copy the 16-point Gauss-Legendre rule from the generated table.
IPA_HD void ipa_pro_phase1(IpaProWork& w, int tid) {
  if (w.status) return;
  if (tid < 64) {
    if (w.mode == 2) return;
    const int which = tid >> 5, lane = tid & 31;
    const double ord = fabs(w.p.lambda + (double)which);
    const double x = w.p.zeta;
    const double h = ipa_trap_step(ord, x);
    double s = 0.0, prev = 1.7976931348623157e308;
    for (int j = 1 + lane; j < 8192; j += 32) {
      const double term = ipa_trap_term(ord, x, h, j);
      s += term;
      if (term <= prev && term < 1e-19 * (s + 0.5)) break;
      prev = term;
    }
    w.part[which][lane] = s;
    if (lane == 0) w.hK[which] = h;
  } else if (tid < 64 + IPA_GL) {
    w.glx[tid - 64] = IPA_GL16X(tid - 64);   // generated table (gen_fastmath_tables.py); IPA_GL == 16
    w.glw[tid - 64] = IPA_GL16W(tid - 64);
  }
}

// phase 2: delta, alpha, joins, z-interval, trapezoid step and length (one thread)
IPA_HD void ipa_pro_phase2(IpaProWork& w, int tid) {
  if (w.status || tid != 0) return;
  const ipa_params& p = w.p;
  if (w.mode == 2) {
    // Student-t core: delta = lim sigma sqrt(zeta K_l/K_{l+1}) = sigma sqrt(-2 lambda - 2) for lambda < -1, else sigma
    w.delta = (p.lambda < -1.0) ? p.sigma * sqrt(-2.0 * p.lambda - 2.0) : p.sigma;
    w.alpha = 0.0;
    w.d0 = -p.a * p.sigma;
    w.d1 = p.a2 * p.sigma;
    w.r0 = sqrt(fma(w.d0, w.d0, w.delta * w.delta));
    w.r1 = sqrt(fma(w.d1, w.d1, w.delta * w.delta));
    w.z0 = w.z1 = 0.0;
    w.zc = 0.0; w.zh = 1.0;
    w.h = 1.0; w.J = 0;
    if (!ipa_finite(w.delta) || !(w.delta > 0.0)) w.status = 3;
    return;
  }
  double s0 = 0.5, s1 = 0.5;
  for (int l = 0; l < 32; ++l) { s0 += w.part[0][l]; s1 += w.part[1][l]; }
  w.Kl = s0 * w.hK[0];
  w.Kl1 = s1 * w.hK[1];
  const double q = p.zeta * w.Kl / w.Kl1;       // (delta/sigma)^2
  w.delta = p.sigma * sqrt(q);
  w.alpha = p.zeta / w.delta;                   // = sqrt(zeta K_{l+1}/K_l)/sigma, alpha delta = zeta
  w.d0 = -p.a * p.sigma;
  w.d1 = p.a2 * p.sigma;
  w.r0 = sqrt(fma(w.d0, w.d0, w.delta * w.delta));
  w.r1 = sqrt(fma(w.d1, w.d1, w.delta * w.delta));
  w.z0 = w.alpha * w.r0;
  w.z1 = w.alpha * w.r1;
  const double zmin = p.zeta;
  double zmax = fmax(w.z0, w.z1);
  zmax = fmax(zmax, zmin * 1.001);
  w.zc = 0.5 * (zmax + zmin);
  w.zh = 0.5 * (zmax - zmin);
  const double o0 = fabs(w.nu), o1 = fabs(w.nu - 1.0), om = fmax(o0, o1);
  w.h = ipa_trap_step(om, zmax);
  // table length: smallest t with zmin (cosh t - 1) - om t > 46, by fixed-point iteration
  // (cosh t - 1 >= e^t / 2 - 1, so the root of  zmin (e^t/2 - 1) - om t = 46  is an upper bound)
  double t = 4.0;
  const double izmin = 1.0 / zmin;
  for (int it = 0; it < 3; ++it) t = log(2.0 * fma(fma(om, t, 46.0), izmin, 1.0));   // increasing, < 0.01 from the root after 3
  int J = (int)(t / w.h) + 2;
  if (J > IPA_JMAX) J = IPA_JMAX;
  w.J = J;
  if (!ipa_finite(w.delta) || !(w.delta > 0.0) || !ipa_finite(w.alpha)) w.status = 3;
}

// phase 3: trapezoid table (all threads)
IPA_HD void ipa_pro_phase3(IpaProWork& w, int tid, int nthr) {
  if (w.status || w.mode == 2) return;
  for (int m = tid; m < 4 * IPA_MCHEB; m += nthr) w.ctab[m] = cos(3.14159265358979323846 * (double)m / (double)(2 * IPA_MCHEB));
  for (int j = tid; j < w.J; j += nthr) {
    const double t = (double)j * w.h;
    const double s = sinh(0.5 * t);
    w.tc[j] = 2.0 * s * s;
    const double e0 = fabs(w.nu) * t, e1 = fabs(w.nu - 1.0) * t;
    w.te[0][j] = e0;
    w.te[1][j] = e1;
    w.tw[0][j] = 0.5 * (1.0 + exp(-2.0 * e0));
    w.tw[1][j] = 0.5 * (1.0 + exp(-2.0 * e1));
  }
}

IPA_HD double ipa_pro_task_z(const IpaProWork& w, int q) {
  if (q < IPA_MCHEB) return w.zc + w.zh * w.ctab[2 * q + 1];
  return ((q - IPA_MCHEB) & 1) ? w.z1 : w.z0;
}

IPA_HD void ipa_pro_cells_geometry(IpaProWork& w);
// phase 4: Bessel tasks, IPA_SUB threads each
IPA_HD void ipa_pro_phase4(IpaProWork& w, int tid) {
  if (tid == 192) { ipa_pro_cells_geometry(w); return; }   // needs phase 2 only; this thread has no Bessel task
  if (w.status || w.mode == 2) return;
  const int q = tid / IPA_SUB, sub = tid % IPA_SUB;
  if (q >= IPA_NBTASK) return;
  const int ord = (q >= IPA_MCHEB + 2) ? 1 : 0;
  w.bpart[q][sub] = ipa_table_partial(w, ord, ipa_pro_task_z(w, q), sub);
}

// phase 5: combine partial sums; H at the Chebyshev nodes
IPA_HD void ipa_pro_phase5(IpaProWork& w, int tid) {
  if (w.status || w.mode == 2 || tid >= IPA_NBTASK) return;
  double s = 0.5;
  for (int i = 0; i < IPA_SUB; ++i) s += w.bpart[tid][i];
  const double Ks = s * w.h;
  w.Ks[tid] = Ks;
  if (tid < IPA_MCHEB) {
    const double z = ipa_pro_task_z(w, tid);
    w.H[tid] = w.nu * log(z) + log(Ks) - z;
  }
}

// phase 6: Chebyshev coefficients c_j = (2/M) sum_i H_i cos(pi j (i+1/2)/M), c_0 halved
IPA_HD void ipa_pro_phase6(IpaProWork& w, int tid) {
  if (w.status || w.mode == 2) return;
  if (tid >= IPA_MCHEB) {
    // threads 64..67: max |H| over a quarter of the nodes each (the noise threshold of the degree selection)
    if (tid < IPA_MCHEB + 4) {
      const int q = tid - IPA_MCHEB;
      double m = 0.0;
      for (int i = 0; i < IPA_MCHEB / 4; ++i) m = fmax(m, fabs(w.H[q * (IPA_MCHEB / 4) + i]));
      w.hmax4[q] = m;
    }
    return;
  }
  const int M = IPA_MCHEB;
  double s = 0.0;
  for (int i = 0; i < M; ++i) {
    const int m = (tid * (2 * i + 1)) % (4 * M);  // angle = pi m / (2M)
    s += w.H[i] * w.ctab[m];
  }
  w.c[tid] = s * (tid == 0 ? 1.0 : 2.0) / (double)M;
}

// phase 7: degree selection (four threads, finished in phase 7b) and the two joins (threads 32 and 64, other warps)
IPA_HD void ipa_pro_phase7(IpaProWork& w, int tid) {
  if (w.status) return;
  const ipa_params& p = w.p;
  if (w.mode == 2) {
    if (tid == 32) {
      w.logG0 = fma(w.nu, log(w.r0 * w.r0), p.beta * w.d0);
      w.L0 = p.beta + 2.0 * w.nu * w.d0 / (w.r0 * w.r0);
    } else if (tid == 64) {
      w.logG1 = fma(w.nu, log(w.r1 * w.r1), p.beta * w.d1);
      w.L1 = p.beta + 2.0 * w.nu * w.d1 / (w.r1 * w.r1);
    }
    return;
  }
  if (tid == 0 || tid == 96 || tid == 128 || tid == 160) {
    // four threads, a quarter of the coefficients each: highest index above the noise threshold (combined in phase 7b)
    const int q = tid == 0 ? 0 : (tid - 64) / 32;
    const double thr = 2.5e-16 * fmax(fmax(1.0, w.hmax4[0]), fmax(fmax(w.hmax4[1], w.hmax4[2]), w.hmax4[3]));
    int best = -1;
    for (int j = q * (IPA_MCHEB / 4); j < (q + 1) * (IPA_MCHEB / 4); ++j)
      if (fabs(w.c[j]) > thr) best = j;
    w.dq4[q] = best;
  } else if (tid == 32) {
    const double K0 = w.Ks[IPA_MCHEB], Km0 = w.Ks[IPA_MCHEB + 2];
    w.logG0 = w.nu * log(w.r0) + p.beta * w.d0 + log(K0) - w.z0;
    w.L0 = p.beta - w.alpha * (w.d0 / w.r0) * (Km0 / K0);
  } else if (tid == 64) {
    const double K1 = w.Ks[IPA_MCHEB + 1], Km1 = w.Ks[IPA_MCHEB + 3];
    w.logG1 = w.nu * log(w.r1) + p.beta * w.d1 + log(K1) - w.z1;
    w.L1 = p.beta - w.alpha * (w.d1 / w.r1) * (Km1 / K1);
  }
}
// phase 7b: tail validity (after a barrier)
IPA_HD void ipa_pro_phase7b(IpaProWork& w, int tid) {
  if (w.status || tid != 0) return;
  if (w.mode != 2) {
    // degree: the highest coefficient above the noise threshold, at least 1
    int D = 1;
    for (int q = 0; q < 4; ++q) D = w.dq4[q] > D ? w.dq4[q] : D;
    const double thr = 2.5e-16 * fmax(fmax(1.0, w.hmax4[0]), fmax(fmax(w.hmax4[1], w.hmax4[2]), w.hmax4[3]));
    // a-priori degree for a general order on this interval: the nearest singularity of H is z = 0, where a general
    // order carries the term (nu - 1/2) log z.  The Chebyshev coefficients of log z on the interval are exactly
    // -2 rho^-k / k (rho = t0 + sqrt(t0^2 - 1), t0 = centre / half-width): Dg = the first k where that falls under the
    // noise threshold at unit weight.  (Round 1 used ceil(37 / ln rho), i.e. rho^-k <= 1e-16 without the 1/k and
    // without the scale of H: 31 instead of 27 for the config interval; orders next to 1/2 need 23 by the noise floor.)
    const double t0 = w.zc / w.zh;
    const double rho = t0 + sqrt(t0 * t0 - 1.0);
    const double rinv = 1.0 / rho;
    int Dg = 2;
    double pw = 2.0 * rinv * rinv;                            // 2 rho^-Dg
    while (Dg < IPA_MCHEB && pw > thr * (double)Dg) { ++Dg; pw *= rinv; }
    if (w.policy == 1 && D < Dg) D = Dg;
    // conditioning of the power basis: needs rho comfortably above 1+sqrt(2)
    if (D > IPA_NCOEF - 1 || rho < 2.6) { w.mode = 1; D = 0; }
    w.degree = D;
  }
  if (!(w.L0 > 0.0) || !(w.L1 < 0.0)) w.status = 2;
}

// ---- cells of the core: low-degree polynomials refitted from the full one (no further Bessel evaluation) ----------
static_assert(IPA_NCELL == 4, "ipa_pro_cells_geometry: ratio of the cell radii is a fourth root");
// phase 7, one thread: cell boundaries.  Equal ratio in r between delta and the larger join radius gives the nominal
// boundaries in |d|; in x they are moved to the nearest edge of the IPA_PREPARE_BINS coarse bins of [lo, hi] (the layout
// of ipa_events_prepare: inside a bin the events are not ordered, so a boundary inside a bin would leave every warp of
// that bin in two cells) and truncated to a zero low word (the kernels compare high words), which moves them by less
// than one unit `quant` of the high word: every cell is fitted on its own |d| interval widened by 2 quant on both sides.
IPA_HD void ipa_pro_cells_geometry(IpaProWork& w) {
  w.ncell = 0;
  for (int i = 0; i < 8; ++i) w.chb[i] = 0x7fffffff;
  if (w.status || w.mode) return;
  const ipa_params& p = w.p;
  const double xl = p.mu + w.d0, xr = p.mu + w.d1;
  if (!(xl > 0.0) || !ipa_finite(xr)) return;
  const int ex = ipa_hi(xr) & 0x7ff00000;
  if (ex < (64 << 20)) return;
  const double quant = ipa_mk(ex - (20 << 20), 0);
  const double margin = 2.0 * quant;
  const double rmax = fmax(w.r0, w.r1), dl2 = w.delta * w.delta;
  const double qr = sqrt(sqrt(rmax / w.delta));                 // ratio of consecutive cell radii (IPA_NCELL == 4)
  const double bw = (w.hi - w.lo) / (double)IPA_PREPARE_BINS, ibw = (double)IPA_PREPARE_BINS / (w.hi - w.lo);
  // boundaries in |d| on the left (L) and on the right (R) of mu; the join where a cell boundary falls outside the core
  double rhoL[IPA_NCELL + 1], rhoR[IPA_NCELL + 1];
  rhoL[0] = rhoR[0] = 0.0;
  rhoL[IPA_NCELL] = -w.d0;
  rhoR[IPA_NCELL] = w.d1;
  double wmin = 1.7976931348623157e308, prev = 0.0, rs = w.delta;
  for (int s = 1; s < IPA_NCELL; ++s) {
    rs *= qr;
    const double rho = ipa_fsqrt((rs - w.delta) * (rs + w.delta));
    rhoL[s] = rhoR[s] = rho;
    wmin = fmin(wmin, rho - prev);
    prev = rho;
  }
  const bool snap = bw < 0.5 * wmin;
  for (int s = 1; s < IPA_NCELL; ++s) {
    double XL = p.mu - rhoL[s], XR = p.mu + rhoR[s];
    if (snap) {
      XL = fma(rint((XL - w.lo) * ibw), bw, w.lo);
      XR = fma(rint((XR - w.lo) * ibw), bw, w.lo);
    }
    const bool hasL = XL > xl, hasR = XR < xr;
    w.chb[IPA_NCELL - 1 - s] = hasL ? ipa_hi(XL) : 0;
    w.chb[IPA_NCELL - 2 + s] = hasR ? ipa_hi(XR) : 0x7fffffff;
    rhoL[s] = hasL ? p.mu - XL : -w.d0;
    rhoR[s] = hasR ? XR - p.mu : w.d1;
  }
  bool ok = true;
  for (int s = 0; s < IPA_NCELL; ++s) {
    // |d| interval of the cell: its part on the left and its part on the right, whichever exist
    const bool partL = rhoL[s + 1] > rhoL[s], partR = rhoR[s + 1] > rhoR[s];
    double a = 1.7976931348623157e308, b = 0.0;
    if (partL) { a = fmin(a, rhoL[s]); b = fmax(b, rhoL[s + 1]); }
    if (partR) { a = fmin(a, rhoR[s]); b = fmax(b, rhoR[s + 1]); }
    ok = ok && (partL || partR) && (margin < 0.01 * (b - a));
    a = fmax(0.0, a - margin);
    b = b + margin;
    const double rl = ipa_fsqrt(fma(a, a, dl2)), rh = fmin(ipa_fsqrt(fma(b, b, dl2)), rmax);
    w.crc[s] = 0.5 * (rl + rh);
    w.crh[s] = 0.5 * (rh - rl);
  }
  if (!ok) {
    for (int i = 0; i < 8; ++i) w.chb[i] = 0x7fffffff;
    return;
  }
  w.ncell = IPA_NCELL;
}
// phase 8, threads 128..255: the full Chebyshev series (Clenshaw, degree from phase 7b) at the Chebyshev nodes of the cells
IPA_HD void ipa_pro_cells_nodes(IpaProWork& w, int tid) {
  if (w.status || w.mode || !w.ncell || w.degree < IPA_CELL_MIN_DEGREE || tid < 128) return;
  const int s = (tid - 128) >> 5, i = (tid - 128) & 31;
  const double r = fma(w.crh[s], w.ctab[4 * i + 2], w.crc[s]);
  const double t = (w.alpha * r - w.zc) / w.zh;
  double b1 = 0.0, b2 = 0.0;
  for (int j = w.degree; j >= 1; --j) {
    const double b0 = fma(2.0 * t, b1, w.c[j] - b2);
    b2 = b1;
    b1 = b0;
  }
  w.cH[s][i] = fma(t, b1, w.c[0] - b2);
}
// phase 9, threads 128..255: Chebyshev coefficients of the cells (ctab[m] = cos(pi m / 128))
IPA_HD void ipa_pro_cells_dct(IpaProWork& w, int tid) {
  if (w.status || w.mode || !w.ncell || w.degree < IPA_CELL_MIN_DEGREE || tid < 128) return;
  const int s = (tid - 128) >> 5, j = (tid - 128) & 31;
  // four partial sums (the loads of one step do not wait for the additions of the one before); index 2 j (2 i + 1) stepped by 4 j
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  const int m4 = 4 * IPA_MCHEB - 1;
  int m = 2 * j;
#pragma unroll
  for (int i = 0; i < IPA_CELLM; i += 4) {
    a0 = fma(w.cH[s][i], w.ctab[m & m4], a0);
    a1 = fma(w.cH[s][i + 1], w.ctab[(m + 4 * j) & m4], a1);
    a2 = fma(w.cH[s][i + 2], w.ctab[(m + 8 * j) & m4], a2);
    a3 = fma(w.cH[s][i + 3], w.ctab[(m + 12 * j) & m4], a3);
    m += 16 * j;
  }
  w.cc[s][j] = ((a0 + a1) + (a2 + a3)) * (j == 0 ? 1.0 : 2.0) * (1.0 / (double)IPA_CELLM);
}
// phase 11: 64 slots (cell, coefficient) on threads that phase 11 leaves idle: lanes 1..31 of warps 4 and 5, lanes 1, 2 of warp 7
IPA_HD int ipa_pro_cells_slot(int tid) {
  if (tid > 128 && tid < 160) return tid - 129;
  if (tid > 160 && tid < 192) return tid - 161 + 31;
  if (tid == 225 || tid == 226) return tid - 225 + 62;
  return -1;
}
// degree of the cell (the rules of phase 7b on the cell's own interval) and its monomial coefficients (as phase 8)
IPA_HD void ipa_pro_cells_monomial(IpaProWork& w, int slot) {
  if (slot < 0 || w.status || w.mode || !w.ncell || w.degree < IPA_CELL_MIN_DEGREE) return;
  const int s = slot >> 4, k = slot & 15;
  const double thr = 2.5e-16 * fmax(fmax(1.0, w.hmax4[0]), fmax(fmax(w.hmax4[1], w.hmax4[2]), w.hmax4[3]));
  int D = 1;
  for (int j = 2; j < IPA_CELLM; ++j)
    if (fabs(w.cc[s][j]) > thr) D = j;
  if (w.policy == 1) {
    const double t0 = w.crc[s] / w.crh[s];
    const double rinv = 1.0 / (t0 + sqrt(t0 * t0 - 1.0));
    int Dg = 2;
    double pw = 2.0 * rinv * rinv;
    while (Dg < IPA_CELLM && pw > thr * (double)Dg) { ++Dg; pw *= rinv; }
    if (D < Dg) D = Dg;
  }
  if (k == 0) w.cdeg[s] = D;
  double ahi = 0.0, alo = 0.0;
  if (D < IPA_CELLN) {
    for (int j = k; j <= D; j += 2) {
      const long long v = w.T[j * IPA_NCOEF + k];
      double ph, pl, sh, sl;
      ipa_two_prod(w.cc[s][j], (double)v, &ph, &pl);
      ipa_two_sum(ahi, ph, &sh, &sl);
      sl += alo + pl;
      const double hi = sh + sl;
      alo = sl - (hi - sh);
      ahi = hi;
    }
  }
  w.csa[s][k] = ahi + alo;
}
// phase 12: the cells' part of the record (threads 128..191 the coefficients, thread 96 the rest)
IPA_HD void ipa_pro_cells_record(IpaProWork& w, IpaSetConsts& o, int tid) {
  if (tid != 96 && (tid < 128 || tid >= 128 + IPA_NCELL * IPA_CELLN)) return;
  bool on = !w.status && !w.mode && w.ncell && w.degree >= IPA_CELL_MIN_DEGREE;
  if (on)
    for (int s = 0; s < IPA_NCELL; ++s) on = on && (w.cdeg[s] < IPA_CELLN);
  if (tid != 96) {
    const int s = (tid - 128) >> 4, k = (tid - 128) & 15;
    o.sa[s][k] = on ? (k ? w.csa[s][k] : w.csa[s][0] - w.araw[0]) : 0.0;   // sa[s][0]: H - araw0 at t_s = 0
    return;
  }
  o.ncell = on ? IPA_NCELL : 0;
  o.cpad[0] = o.cpad[1] = o.cpad[2] = 0;
  for (int s = 0; s < IPA_NCELL; ++s) {
    o.sdeg[s] = on ? w.cdeg[s] : 0;
    o.stA[s] = on ? 1.0 / w.crh[s] : 0.0;
    o.stB[s] = on ? -w.crc[s] / w.crh[s] : 0.0;
    o.sng[s] = on ? (w.cdeg[s] >> 2) : 0;
  }
  for (int i = 0; i < 8; ++i) o.hb[i] = on ? w.chb[i] : 0x7fffffff;
}

// phase 8: Chebyshev -> monomial, a_k = sum_j c_j T[j][k] with the integer coefficients T[j][k] of the
// Chebyshev polynomials (generated table, exact in int64 up to degree 47: |T[47][k]| < 2^59; the host test
// rebuilds it from T_{j+1} = 2 t T_j - T_{j-1}).  Thread k accumulates its coefficient over the rows of
// matching parity in double-double.
IPA_HD void ipa_pro_phase8_finish(IpaProWork& w, int k) {
  if (w.status || w.mode || k >= IPA_NCOEF) return;
  double ahi = 0.0, alo = 0.0;
  for (int j = k; j <= w.degree; j += 2) {
    const long long v = w.T[j * IPA_NCOEF + k];
    double ph, pl, sh, sl;
    ipa_two_prod(w.c[j], (double)v, &ph, &pl);
    ipa_two_sum(ahi, ph, &sh, &sl);
    sl += alo + pl;
    const double hi = sh + sl;
    alo = sl - (hi - sh);
    ahi = hi;
  }
  w.araw[k] = (k <= w.degree) ? ahi + alo : 0.0;
}

// phase 9: range, panels, reference level (one thread)
IPA_HD void ipa_pro_phase9(IpaProWork& w, int tid) {
  if (w.status) return;
  if (tid == 0) {                 // reference level of the normalisation
    w.dl = w.lo - w.p.mu;
    w.dh = w.hi - w.p.mu;
    const double dref = fmin(fmax(0.0, w.dl), w.dh);
    w.logref = ipa_logI(w, dref);
    return;
  }
  if (tid != 32) return;          // panels of the core quadrature (another warp, at the same time)
  const double dl = w.lo - w.p.mu, dh = w.hi - w.p.mu;
  const double A = fmax(dl, w.d0), B = fmin(dh, w.d1);
  int np = 0;
  if (B > A) {
    for (int side = 0; side < 2; ++side) {
      // side 0: d >= 0 part, side 1: d <= 0 part, both in |d| = [p, q]
      double pp, qq;
      if (side == 0) { if (B <= 0.0) continue; pp = fmax(A, 0.0); qq = B; }
      else { if (A >= 0.0) continue; pp = fmax(-B, 0.0); qq = -A; }
      double b = pp;
      int cnt = 0;
      while (b < qq) {
        double nb = fmin(qq, fmax(w.delta, 3.0 * b));
        if (++cnt == IPA_MAXPANEL / 2) nb = qq;
        w.pa[np] = side == 0 ? b : -nb;
        w.pb[np] = side == 0 ? nb : -b;
        ++np;
        b = nb;
      }
    }
  }
  w.npanel = np;
}

// phase 10: quadrature nodes (all threads)
IPA_HD void ipa_pro_phase10(IpaProWork& w, int tid, int nthr) {
  if (w.status) return;
  for (int q = tid; q < w.npanel * IPA_GL; q += nthr) {
    const int pnl = q / IPA_GL, i = q % IPA_GL;
    const double c = 0.5 * (w.pa[pnl] + w.pb[pnl]), hl = 0.5 * (w.pb[pnl] - w.pa[pnl]);
    const double d = c + hl * w.glx[i];
    const double g = w.glw[i] * hl * exp(ipa_core_logG(w, d) - w.logref);
    w.pval[q] = g;
    w.pval2[q] = w.want_grad ? g * (ipa_sigpow(w) / w.p.sigma - (d / w.p.sigma) * ipa_core_Lmb(w, d)) : 0.0;   // G dlogG/dsigma
    w.pval3[q] = w.want_grad ? g * d : 0.0;                                                                    // G dlogG/dbeta
  }
}
IPA_HD void ipa_pro_phase11(IpaProWork& w, int tid) {
  if (w.status) return;
  const ipa_params& p = w.p;
  if (tid < w.npanel) {
    double s = 0.0, s2 = 0.0, s3 = 0.0;
    for (int i = 0; i < IPA_GL; ++i) { s += w.pval[tid * IPA_GL + i]; s2 += w.pval2[tid * IPA_GL + i]; s3 += w.pval3[tid * IPA_GL + i]; }
    w.psum[tid] = s;
    w.psum2[tid] = s2;
    w.psum3[tid] = s3;
  } else if (tid == 32) {          // left tail: int I and int I dlogI/dsigma, in units of exp(logref)  (reading C5)
    // with u = 1 - (d-d0) L0/n:  dlogI/dsigma = A + [a L0 - c] / u + c,  A = nu/sigma - a beta,
    // c = n (L0 - beta) / (L0 sigma);  int u^-n du and int u^-(n+1) du are ipa_powint(u, n), ipa_powint(u, n+1)
    // dlogI/dbeta = d0 + (d - d0)/u = (d0 - n/L0) + (n/L0)/u
    double left = 0.0, left2 = 0.0, left3 = 0.0;
    if (w.dl < w.d0) {
      const double dr = fmin(w.d0, w.dh);
      const double ul = 1.0 - (w.dl - w.d0) * w.L0 / p.n, ur = 1.0 - (dr - w.d0) * w.L0 / p.n;
      // F(ul) - F(ur) without cancellation (ipa_powint_diff); its scale ur^(1-n) joins the log-reference
      double ls, ls1 = 0.0;
      const double Fm = ipa_powint_diff(ul, ur, p.n, &ls);
      const double F1m = w.want_grad ? ipa_powint_diff(ul, ur, p.n + 1.0, &ls1) : 0.0;
      const double pre = p.n / w.L0, lg = w.logG0 - w.logref;
      const double F = exp(lg + ls) * Fm, F1 = w.want_grad ? exp(lg + ls1) * F1m : 0.0;
      const double A = ipa_sigpow(w) / p.sigma - p.a * p.beta, c = p.n * (w.L0 - p.beta) / (w.L0 * p.sigma);
      left = pre * F;
      left2 = pre * ((A + c) * F + (p.a * w.L0 - c) * F1);
      left3 = pre * ((w.d0 - p.n / w.L0) * F + (p.n / w.L0) * F1);
    }
    w.tl_left = left;
    w.tl_left2 = left2;
    w.tl_left3 = left3;
  } else if (tid == 64) {          // right tail: dlogI/dsigma = A' + c' - (a2 L1 + c') / u,  c' = n2 (L1 - beta) / (L1 sigma)
    double right = 0.0, right2 = 0.0, right3 = 0.0;   // dlogI/dbeta = (d1 - n2/L1) + (n2/L1)/u
    if (w.dh > w.d1) {
      const double dL = fmax(w.d1, w.dl);
      const double uh = 1.0 - (w.dh - w.d1) * w.L1 / p.n2, ul = 1.0 - (dL - w.d1) * w.L1 / p.n2;
      double ls, ls1 = 0.0;
      const double Fm = ipa_powint_diff(uh, ul, p.n2, &ls);
      const double F1m = w.want_grad ? ipa_powint_diff(uh, ul, p.n2 + 1.0, &ls1) : 0.0;
      const double pre = p.n2 / (-w.L1), lg = w.logG1 - w.logref;
      const double F = exp(lg + ls) * Fm, F1 = w.want_grad ? exp(lg + ls1) * F1m : 0.0;
      const double A = ipa_sigpow(w) / p.sigma + p.a2 * p.beta, c = p.n2 * (w.L1 - p.beta) / (w.L1 * p.sigma);
      right = pre * F;
      right2 = pre * ((A + c) * F - (p.a2 * w.L1 + c) * F1);
      right3 = pre * ((w.d1 - p.n2 / w.L1) * F + (p.n2 / w.L1) * F1);
    }
    w.tl_right = right;
    w.tl_right2 = right2;
    w.tl_right3 = right3;
  } else if (tid == 96) {          // background normalisation (shifted by lo) and d ln N_B / d k
    const double wd = w.hi - w.lo, tk = p.k * wd;
    const double NB = (fabs(tk) < 1e-8) ? wd * (1.0 + 0.5 * tk + tk * tk / 6.0) : expm1(tk) / p.k;
    w.NB = NB;
    w.logNB = log(NB);
    w.dlnNB_dk = (fabs(tk) < 1e-6) ? wd * (0.5 + tk / 12.0) : wd * exp(tk) / expm1(tk) - 1.0 / p.k;
  } else if (tid == 224) {         // I at the ends of the range (d N_S / d mu = I(lo - mu) - I(hi - mu))
    w.Iedge_l = w.want_grad ? exp(ipa_logI(w, w.dl) - w.logref) : 0.0;
    w.Iedge_h = w.want_grad ? exp(ipa_logI(w, w.dh) - w.logref) : 0.0;
  } else if (tid == 200) {
    w.inv_sigma = 1.0 / p.sigma;
    w.inv_zh = 1.0 / w.zh;
  } else if (tid == 208) {
    w.inv_f = 1.0 / p.f;
    w.inv_1mf = 1.0 / (1.0 - p.f);
  } else if (tid == 216) {
    w.inv_n0 = 1.0 / p.n;
    w.inv_n1 = 1.0 / p.n2;
  } else if (tid == 128) {
    w.logf = (p.f > 0.0) ? log(p.f) : 0.0;
    w.log1mf = (p.f < 1.0) ? log1p(-p.f) : 0.0;
  } else if (tid == 160) {
    w.nulogalpha = (w.mode == 2) ? 0.0 : w.nu * log(w.alpha);
  } else if (tid == 192) {
    w.expref = exp(w.logref);
  }
}

// phase 12: normalisations and folded constants.  Three threads of three warps write disjoint parts of the record at
// the same time (one thread took 10 000 cycles, a fifth of the prologue: a chain of divisions, a logarithm and a read
// back of a value it had just stored to global memory); each forms N_S from the same sums in the same order.
struct IpaProNorm { double NSr, logNS, cS, kd, eB0; bool ok, pure; };
IPA_HD IpaProNorm ipa_pro_norm(const IpaProWork& w) {
  IpaProNorm r;
  const ipa_params& p = w.p;
  double core = 0.0;
  for (int i = 0; i < w.npanel; ++i) core += w.psum[i];
  r.NSr = w.tl_left + core + w.tl_right;  // in units of exp(logref)
  r.ok = (r.NSr > 0.0) && ipa_finite(r.NSr) && (w.NB > 0.0) && ipa_finite(w.NB);
  r.logNS = log(r.NSr) + w.logref;
  r.pure = !(p.f < 1.0);
  // f = 0: a finite, very negative signal term (softplus(-1e4) == 0 exactly) instead of -inf; it stays far inside the
  // range |Delta| < 1.4e6 of the softplus exponential (ipa_fexp_negabs_sp)
  r.cS = (p.f > 0.0) ? w.logf - r.logNS : -1.0e4;
  r.kd = r.pure ? 0.0 : p.k;
  r.eB0 = r.pure ? 0.0 : (p.k * (p.mu - w.lo) + w.log1mf - w.logNB);
  return r;
}
IPA_HD void ipa_pro_phase12(IpaProWork& w, IpaSetConsts& o, int tid) {
  if (tid != 0 && tid != 32 && tid != 64) return;
  const ipa_params& p = w.p;
  if (w.status) {
    if (tid == 0) { o.status = w.status; o.degree = w.degree; o.mode = w.mode; o.pure = 0; o.normS = o.normB = NAN; }
    return;
  }
  const IpaProNorm r = ipa_pro_norm(w);
  if (!r.ok) {
    // (threads 32 and 64 may see w.status before or after this store: they write nothing either way)
    if (tid == 0) { w.status = 3; o.status = 3; o.degree = w.degree; o.mode = w.mode; o.pure = 0; o.normS = o.normB = NAN; }
    return;
  }
  if (tid == 0) {
    o.status = 0; o.degree = w.degree; o.mode = w.mode; o.pure = r.pure ? 1 : 0;
    w.normS_abs = r.NSr * w.expref;
    o.normS = w.normS_abs;
    o.normB = w.NB;
    o.mu = p.mu; o.d0 = w.d0; o.d1 = w.d1; o.delta2 = w.delta * w.delta;
    o.tA = w.alpha * w.inv_zh; o.tB = -w.zc * w.inv_zh;
    o.bmk = p.beta - r.kd; o.kd = r.kd; o.eB0 = r.eB0;
    o.alpha = w.alpha; o.nu = w.nu;
    w.cDir = r.cS - r.eB0 - w.nulogalpha;
    o.cDir = w.cDir;
    o.fsig = p.f; o.kraw = p.k;
    o.beta = p.beta; o.logG0 = w.logG0; o.logG1 = w.logG1; o.logNS = r.logNS; o.logref = w.logref;
    o.araw0 = w.mode ? 0.0 : w.araw[0];   // modes 1, 2: no polynomial
    const double xl = p.mu + w.d0, xr = p.mu + w.d1;
    o.hxl = (xl > 0.0) ? ipa_hi(xl) : 0;
    o.hxr = (xr > 0.0) ? ipa_hi(xr) : -1;
    o.pad0 = o.pad1 = 0;
  } else if (tid == 32) {
    const double in0 = w.inv_n0, in1 = w.inv_n1;
    o.uA0 = -w.L0 * in0; o.uB0 = fma(w.d0 * w.L0, in0, 1.0); o.n0 = p.n;  o.cT0 = w.logG0 + r.cS - r.eB0;
    o.uA1 = -w.L1 * in1; o.uB1 = fma(w.d1 * w.L1, in1, 1.0); o.n1 = p.n2; o.cT1 = w.logG1 + r.cS - r.eB0;
  } else {
    double core2 = 0.0, core3 = 0.0;
    for (int i = 0; i < w.npanel; ++i) { core2 += w.psum2[i]; core3 += w.psum3[i]; }
    const double iN = 1.0 / r.NSr, isg = w.inv_sigma;
    const double nuosig = ipa_sigpow(w) * isg;
    o.dlnNS_dmu = (w.Iedge_l - w.Iedge_h) * iN;
    o.dlnNS_dsig = (w.tl_left2 + core2 + w.tl_right2) * iN;
    o.dlnNS_dbeta = (w.tl_left3 + core3 + w.tl_right3) * iN;
    o.pad2 = 0.0;
    o.dlnNB_dk = r.pure ? 0.0 : w.dlnNB_dk;
    o.nuosig = nuosig; o.invsig = isg; o.mulo = p.mu - w.lo; o.L0 = w.L0; o.L1 = w.L1;
    o.A0 = nuosig - p.a * p.beta; o.A1 = nuosig + p.a2 * p.beta;
    o.aL0 = p.a * w.L0; o.a2L1 = p.a2 * w.L1;
    o.c0s = (w.L0 - p.beta) * isg; o.c1s = (w.L1 - p.beta) * isg;
    o.invf = w.inv_f; o.inv1mf = w.inv_1mf;
  }
}
// phase 13: coefficients (threads 0..47), after phase 12
IPA_HD void ipa_pro_phase13(IpaProWork& w, IpaSetConsts& o, int k) {
  if (k >= IPA_NCOEF) return;
  double v = 0.0;
  if (!w.status) {
    if (!w.mode) v = w.araw[k];
    if (k == 0) v += w.cDir;  // cS - eB0 - nu log alpha: the per-set constant of the core term (both modes)
  }
  o.a[k] = v;
}
