/*
 * ipa_oracle.cpp -- the ORACLE: a plain, slow, obviously-correct CPU implementation of the
 * unbinned Ipatia + exponential negative log-likelihood hot path of arXiv:1706.01420
 * ("Ipanema-beta"), Example 1 and of the toy / binned variants that feed
 * it.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or constant generator with the CUDA library (paper_1706_01420_b200/csrc) and neither
 * includes the other.
 *
 * Style: single-threaded straight-line code in the order of the definitions in DESIGN.md
 * ("Readings", C1-C5); `long double` (x87 80-bit) inside the special
 * functions and sums so that the oracle is closer to the mathematical value than any fp64
 * implementation can be; results are returned as fp64 (everything is double).
 * The only threaded routine (orc_nll with nthreads>1) hands contiguous chunks to the same
 * single-threaded routine and exists for the timed CPU baseline.
 *
 * Parity pins (tests/test_oracle_*.py): mpmath 40-digit Bessel values, closed forms for
 * half-integer order, the recurrence, the hyperbolic special case lambda=1, the worked example
 * of SURVEY.md 8(c) C8.9 (tests/golden/), normalisation against independent adaptive
 * quadrature, join continuity, the Gaussian limit, brute force on tiny inputs, fit recovery,
 * Philox against the CUDA toolkit's own host-callable header, Poisson moments.
 * Parity UNPINNED: agreement with the paper's own psIpatia.cu numerics (source not in the
 * paper; PAPER.md:54 only names it).
 */
#include <cmath>
#include <cstdint>
#include <cstring>
#include <cstdlib>
#include <vector>
#include <thread>
#include <limits>
#include <algorithm>

typedef long double ld;

extern "C" {
typedef struct {
  double mu, sigma, lambda, zeta, beta, a, n, a2, n2; /* signal shape, order of PAPER.md:65-68 */
  double f;                                           /* signal fraction */
  double k;                                           /* background exp(k x) */
} orc_params;
}

static const ld PI_L = 3.14159265358979323846264338327950288L;
static const ld EULER_GAMMA_L = 0.57721566490153286060651209008240243L;

/* ------------------------------------------------------------------------------------------
 * Riemann zeta at integer k>=2 by Euler-Maclaurin (A&S 23.2.3 summed to N, 23.1.30 tail).
 * Needed only for the Taylor series of log Gamma(1+mu) below.
 * ---------------------------------------------------------------------------------------- */
static ld zeta_int(int k) {
  const int N = 32;
  ld s = 0;
  for (int n = 1; n < N; ++n) s += powl((ld)n, -(ld)k);
  const ld Nk = powl((ld)N, -(ld)k);
  s += Nk * N / (ld)(k - 1) + Nk / 2;
  /* Bernoulli terms B_{2j}/(2j)! * k(k+1)...(k+2j-2) * N^{-k-2j+1}, j=1..6 */
  static const ld B2j[6] = {1.0L / 6, -1.0L / 30, 1.0L / 42, -1.0L / 30, 5.0L / 66, -691.0L / 2730};
  ld fact = 1;      /* (2j)! */
  ld rising = 1;    /* k(k+1)...(k+2j-2) */
  ld Npow = Nk;     /* N^{-k-2j+1} */
  for (int j = 1; j <= 6; ++j) {
    fact *= (ld)(2 * j - 1) * (ld)(2 * j);
    if (j == 1) rising = k; else rising *= (ld)(k + 2 * j - 3) * (ld)(k + 2 * j - 2);
    Npow /= (j == 1 ? (ld)N : (ld)N * N);
    s += B2j[j - 1] / fact * rising * Npow;
  }
  return s;
}

struct ZetaTable {
  ld z[96];
  ZetaTable() { z[0] = z[1] = 0; for (int k = 2; k < 96; ++k) z[k] = zeta_int(k); }
};
static const ZetaTable& zeta_table() { static ZetaTable t; return t; }

/* log Gamma(1+mu) = -gamma mu + sum_{k>=2} (-1)^k zeta(k) mu^k / k   (A&S 6.1.33), |mu|<1.
 * Split into odd part A(mu) and even part E(mu): logGamma(1+-mu) = +-A + E. */
static void loggamma1p_parts(ld mu, ld* A_over_mu, ld* E) {
  const ZetaTable& Z = zeta_table();
  const ld m2 = mu * mu;
  ld a = -EULER_GAMMA_L, e = 0, p = 1; /* p = mu^{2j} */
  for (int j = 1; 2 * j + 1 < 96; ++j) {
    p *= m2;
    e += Z.z[2 * j] * p / (ld)(2 * j);
    a -= Z.z[2 * j + 1] * p / (ld)(2 * j + 1);
    if (p < 1e-30L) break;
  }
  *A_over_mu = a;
  *E = e;
}

static ld sinhc(ld t) { /* sinh(t)/t */
  if (fabsl(t) < 1e-4L) { ld t2 = t * t; return 1 + t2 / 6 * (1 + t2 / 20); }
  return sinhl(t) / t;
}

/* ------------------------------------------------------------------------------------------
 * Temme's series (N. M. Temme, J. Comput. Phys. 19 (1975) 324) for K_mu(x), K_{mu+1}(x),
 * |mu| <= 1/2, 0 < x <= 2.   Returns the UNscaled values.
 *   K_mu   = sum_k c_k f_k,   K_{mu+1} = (2/x) sum_k c_k h_k,   c_k = (x^2/4)^k / k!
 *   f_0 = (mu pi / sin mu pi) [ cosh(s) G1(mu) + (sinh(s)/s) ln(2/x) G2(mu) ],  s = mu ln(2/x)
 *   p_0 = (1/2)(2/x)^mu Gamma(1+mu),  q_0 = (1/2)(x/2)^mu Gamma(1-mu)
 *   f_k = (k f_{k-1} + p_{k-1} + q_{k-1})/(k^2-mu^2), p_k = p_{k-1}/(k-mu), q_k = q_{k-1}/(k+mu)
 *   h_k = p_k - k f_k
 *   G1 = [1/Gamma(1-mu) - 1/Gamma(1+mu)]/(2 mu) = e^{-E} sinh(A)/mu,  G2 = e^{-E} cosh(A)
 * ---------------------------------------------------------------------------------------- */
static void temme_series(ld mu, ld x, ld* Kmu, ld* Kmu1) {
  ld Aom, E;
  loggamma1p_parts(mu, &Aom, &E);
  const ld A = mu * Aom;
  const ld G1 = expl(-E) * sinhc(A) * Aom;
  const ld G2 = expl(-E) * coshl(A);
  const ld gam_p = expl(A + E);  /* Gamma(1+mu) */
  const ld gam_m = expl(-A + E); /* Gamma(1-mu) */
  const ld L = logl(2 / x);
  const ld s = mu * L;
  const ld mupi = mu * PI_L;
  const ld fact = (fabsl(mupi) < 1e-10L) ? 1.0L : mupi / sinl(mupi);
  ld f = fact * (coshl(s) * G1 + sinhc(s) * L * G2);
  ld p = 0.5L * expl(s) * gam_p;
  ld q = 0.5L * expl(-s) * gam_m;
  ld c = 1, sum = f, sum1 = p;
  const ld x2q = x * x / 4;
  for (int k = 1; k < 500; ++k) {
    f = (k * f + p + q) / ((ld)k * k - mu * mu);
    p /= (k - mu);
    q /= (k + mu);
    c *= x2q / k;
    const ld t = c * f, t1 = c * (p - k * f);
    sum += t;
    sum1 += t1;
    if (fabsl(t) < 1e-22L * fabsl(sum) && fabsl(t1) < 1e-22L * fabsl(sum1)) break;
  }
  *Kmu = sum;
  *Kmu1 = sum1 * 2 / x;
}

/* ------------------------------------------------------------------------------------------
 * x > 2: Miller's backward recurrence on z_n = U(mu+1/2+n, 2mu+1, 2x) (Temme 1975, sect. 3):
 *   K_mu(x) = sqrt(pi) (2x)^mu e^{-x} z_0                                  (DLMF 13.6.10)
 *   z_{n-1} = 2(n+x) z_n - A_{n+1} z_{n+1},  A_n = (n-1/2)^2 - mu^2        (DLMF 13.3.7)
 *   sum_{n>=0} C_n z_n = (2x)^{-mu-1/2},  C_0 = 1, C_n = C_{n-1} A_n / n
 *   K_{mu+1}/K_mu = [ 1/2 + mu + x - A_1 z_1/z_0 ] / x
 * z_n is the minimal solution, so starting from (0, tiny) at a large N and recurring down
 * gives the right ratios; N is doubled until the result is stable.
 * Returns the SCALED values e^x K.
 * ---------------------------------------------------------------------------------------- */
static void miller_once(ld mu, ld x, int N, ld* Ks, ld* K1s) {
  const ld mu2 = mu * mu;
  std::vector<ld> C(N + 2);
  C[0] = 1;
  for (int n = 1; n <= N + 1; ++n) C[n] = C[n - 1] * (((ld)n - 0.5L) * ((ld)n - 0.5L) - mu2) / n;
  ld tn1 = 0, tn = 1e-300L, S = C[N] * tn; /* t_{N+1}=0, t_N=tiny */
  ld t1_keep = 0;
  for (int n = N; n >= 1; --n) {
    const ld An1 = ((ld)n + 0.5L) * ((ld)n + 0.5L) - mu2;
    const ld tm = 2 * ((ld)n + x) * tn - An1 * tn1; /* t_{n-1} */
    tn1 = tn;
    tn = tm;
    S += C[n - 1] * tn;
    if (n == 1) t1_keep = tn1;
    /* only ratios matter: rescale so that a long recurrence cannot overflow */
    if (n > 1 && fabsl(tn) > 1e2000L) { tn *= 1e-2000L; tn1 *= 1e-2000L; S *= 1e-2000L; }
  }
  const ld t0 = tn;
  *Ks = sqrtl(PI_L / (2 * x)) * t0 / S;
  const ld A1 = 0.25L - mu2;
  *K1s = *Ks * (0.5L + mu + x - A1 * t1_keep / t0) / x;
}

static void miller(ld mu, ld x, ld* Ks, ld* K1s) {
  int N = 32 + (int)(64 / x);
  ld a, b;
  miller_once(mu, x, N, &a, &b);
  for (int it = 0; it < 8; ++it) {
    N *= 2;
    ld a2, b2;
    miller_once(mu, x, N, &a2, &b2);
    /* 1e-17 relative: ~100 ulp of long double, still 10x below fp64 resolution (a 2e-19 test is
     * within rounding noise of the recurrence and fails at random) */
    const bool ok = fabsl(a2 - a) <= 1e-17L * fabsl(a2) && fabsl(b2 - b) <= 1e-17L * fabsl(b2);
    a = a2; b = b2;
    if (ok) break;
  }
  *Ks = a; *K1s = b;
}

/* Scaled modified Bessel function of the second kind, real order: returns e^x K_nu(x), x>0.
 * K_{-nu}=K_nu (A&S 9.6.6); |nu| = N + mu with |mu|<=1/2; forward recurrence
 * K_{v+1} = K_{v-1} + (2v/x) K_v (A&S 9.6.26), stable upward for K. */
static ld besselk_scaled_l(ld nu, ld x) {
  if (!(x > 0)) return std::numeric_limits<ld>::quiet_NaN();
  nu = fabsl(nu);
  const int N = (int)floorl(nu + 0.5L);
  const ld mu = nu - N;
  ld k0, k1;
  if (x <= 2) {
    temme_series(mu, x, &k0, &k1);
    const ld ex = expl(x);
    k0 *= ex; k1 *= ex;
  } else {
    miller(mu, x, &k0, &k1);
  }
  if (N == 0) return k0;
  for (int j = 1; j < N; ++j) {
    const ld k2 = k0 + 2 * (mu + j) / x * k1;
    k0 = k1; k1 = k2;
  }
  return k1;
}

/* ------------------------------------------------------------------------------------------
 * Ipatia shape (reading C1; ref. [10] of the paper, cited at PAPER.md:54, 450).
 * ---------------------------------------------------------------------------------------- */
struct Shape {
  ld mu, sigma, lambda, zeta, beta, a, n, a2, n2;
  ld nu, delta, alpha;
  int tcore;           /* 1: the zeta = 0 Student-t core below (no Bessel function) */
  ld sigpow;           /* G(d; sigma) = sigma^sigpow g(d/sigma) e^{beta d}: nu (Bessel core), 2 nu (Student-t core) */
  ld d0, d1;           /* joins: -a sigma, +a2 sigma */
  ld logG0, logG1;     /* log core value at the joins */
  ld L0, L1;           /* log-derivative of the core at the joins */
  int status;          /* 0 ok, 1 basic domain, 2 join slope sign */
};

/* zeta -> 0 limit of the core for lambda < 0 (reading D3; ref. [10] of the paper,
 * PAPER.md:450, and the Upsilon example's `Free('lb', -2.0, ...)` with no zeta).  With alpha -> 0,
 * K_nu(z) -> Gamma(|nu|) 2^{|nu|-1} z^{-|nu|} (A&S 9.6.9) and nu = lambda - 1/2 < 0, so up to a constant factor
 *     G(d) = (d^2 + delta^2)^{lambda - 1/2} e^{beta d}            (a Student-t core with -2 lambda degrees of freedom)
 *     L(d) = G'/G = beta + (2 lambda - 1) d / (d^2 + delta^2)
 * delta: the limit of sigma sqrt(zeta K_lambda(zeta)/K_{lambda+1}(zeta)) is sigma sqrt(-2 lambda - 2) for lambda < -1
 * (then sigma^2 is still the variance of the symmetric core); for -1 <= lambda < 0 that limit is 0 (the variance
 * diverges) and delta = sigma is taken as the scale (reading D3).  Tails, normalisation and likelihood are unchanged. */
static ld core_logG(const Shape& s, ld d) {
  if (s.tcore) return s.nu * logl(d * d + s.delta * s.delta) + s.beta * d;
  /* log G(d) = nu log r + beta d + log K_nu(alpha r),  r = sqrt(d^2+delta^2) */
  const ld r = sqrtl(d * d + s.delta * s.delta);
  const ld z = s.alpha * r;
  return s.nu * logl(r) + s.beta * d + logl(besselk_scaled_l(s.nu, z)) - z;
}

static ld core_logderiv(const Shape& s, ld d) {
  if (s.tcore) return s.beta + 2 * s.nu * d / (d * d + s.delta * s.delta);
  /* L(d) = beta - alpha (d/r) K_{nu-1}(z)/K_nu(z) */
  const ld r = sqrtl(d * d + s.delta * s.delta);
  const ld z = s.alpha * r;
  return s.beta - s.alpha * (d / r) * besselk_scaled_l(s.nu - 1, z) / besselk_scaled_l(s.nu, z);
}

static bool finite_all(const orc_params& p) {
  const double* v = &p.mu;
  for (int i = 0; i < 11; ++i) if (!std::isfinite(v[i])) return false;
  return true;
}

static Shape make_shape(const orc_params& p) {
  Shape s;
  s.mu = p.mu; s.sigma = p.sigma; s.lambda = p.lambda; s.zeta = p.zeta; s.beta = p.beta;
  s.a = p.a; s.n = p.n; s.a2 = p.a2; s.n2 = p.n2;
  s.status = 0;
  s.tcore = (p.zeta == 0) ? 1 : 0;
  if (!finite_all(p) || !(p.sigma > 0) || !(p.zeta > 0 || (p.zeta == 0 && p.lambda < 0)) || !(p.a > 0) || !(p.a2 > 0) ||
      !(p.n > 0) || !(p.n2 > 0) || !(p.f >= 0) || !(p.f <= 1)) {
    s.status = 1;
    return s;
  }
  s.nu = s.lambda - 0.5L;
  if (s.tcore) {
    s.delta = (s.lambda < -1) ? s.sigma * sqrtl(-2 * s.lambda - 2) : s.sigma;
    s.alpha = 0;
    s.sigpow = 2 * s.nu;
  } else {
    const ld Kl = besselk_scaled_l(s.lambda, s.zeta);
    const ld Kl1 = besselk_scaled_l(s.lambda + 1, s.zeta);
    s.delta = s.sigma * sqrtl(s.zeta * Kl / Kl1);
    s.alpha = sqrtl(s.zeta * Kl1 / Kl) / s.sigma;
    s.sigpow = s.nu;
  }
  s.d0 = -s.a * s.sigma;
  s.d1 = s.a2 * s.sigma;
  s.logG0 = core_logG(s, s.d0);
  s.logG1 = core_logG(s, s.d1);
  s.L0 = core_logderiv(s, s.d0);
  s.L1 = core_logderiv(s, s.d1);
  if (!(s.L0 > 0) || !(s.L1 < 0)) s.status = 2;
  return s;
}

/* log I(d): core inclusive of the joins (reading D8); power-law tails matching value and slope. */
static ld log_I(const Shape& s, ld d) {
  if (d < s.d0) return s.logG0 - s.n * logl(1 - (d - s.d0) * s.L0 / s.n);
  if (d > s.d1) return s.logG1 - s.n2 * logl(1 - (d - s.d1) * s.L1 / s.n2);
  return core_logG(s, d);
}

/* Gauss-Legendre nodes/weights on [-1,1] by Newton on P_n (A&S 25.4.29). */
static void gauss_legendre(int n, std::vector<ld>& x, std::vector<ld>& w) {
  x.resize(n); w.resize(n);
  for (int i = 0; i < n; ++i) {
    ld t = cosl(PI_L * (i + 0.75L) / (n + 0.5L));
    ld dp = 0;
    for (int it = 0; it < 100; ++it) {
      ld p0 = 1, p1 = t;
      for (int k = 2; k <= n; ++k) { const ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
      dp = n * (t * p1 - p0) / (t * t - 1);
      const ld dt = p1 / dp;
      t -= dt;
      if (fabsl(dt) < 1e-20L) break;
    }
    { ld p0 = 1, p1 = t;
      for (int k = 2; k <= n; ++k) { const ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
      dp = n * (t * p1 - p0) / (t * t - 1); }
    x[i] = t;
    w[i] = 2 / ((1 - t * t) * dp * dp);
  }
}

static ld core_integral_scaled(const Shape& s, ld A, ld B, ld logref) {
  /* int_A^B exp(logG(d)-logref) dd, composite 20-point Gauss-Legendre, panels doubled until stable */
  if (!(B > A)) return 0;
  /* the 20-point rule, computed once; C++11 initialises a function-local static exactly once even when
   * the timed multi-threaded wrapper (orc_nll, nthreads > 1) enters here from several threads */
  struct Rule { std::vector<ld> x, w; Rule() { gauss_legendre(20, x, w); } };
  static const Rule rule;
  const std::vector<ld>& gx = rule.x;
  const std::vector<ld>& gw = rule.w;
  ld prev = 0;
  for (int P = 4; P <= 8192; P *= 2) {
    ld tot = 0;
    const ld h = (B - A) / P;
    for (int j = 0; j < P; ++j) {
      const ld c = A + (j + 0.5L) * h;
      ld acc = 0;
      for (int i = 0; i < 20; ++i) acc += gw[i] * expl(core_logG(s, c + 0.5L * h * gx[i]) - logref);
      tot += acc * 0.5L * h;
    }
    if (P > 4 && fabsl(tot - prev) <= 1e-16L * fabsl(tot)) return tot;
    prev = tot;
  }
  return prev;
}

/* Tail integral between two points of the SAME tail (reading C5: the antiderivative of u^{-n} is
 * F(u) = (u^{1-n} - 1)/(1-n), log u at n = 1).  The difference F(ul) - F(ur), ul >= ur >= 1, is formed as
 *     ur^{1-n} expm1((1-n) log(ul/ur)) / (1-n)            (log(ul/ur) at n = 1)
 * -- the same closed form, without subtracting two numbers that both sit next to 1/(n-1) when the fit range lies
 * deep inside one tail and n is large (there the subtraction lost all digits: N_S = 0 for mu = 5700, sigma = 0.89,
 * n = 66; pinned against mpmath at 50 digits in tests/test_oracle_ipatia.py).  Returns the value without the
 * factor ur^{1-n}; *logscale = (1-n) log ur is added to the exponent of the prefactor by the caller. */
static ld powint_diff(ld ul, ld ur, ld n, ld* logscale) {
  const ld e = 1 - n;
  const ld lq = logl(ul / ur);
  *logscale = e * logl(ur);
  if (fabsl(e * lq) < 1e-12L) return lq * (1 + 0.5L * e * lq);
  return expm1l(e * lq) / e;
}

struct Norm { ld NS, core, left, right, NB, logref; };

/* N_S = int_lo^hi I(x-mu) dx (reading C5) and N_B = int_lo^hi e^{k(x-lo)} dx (shifted). */
static Norm make_norm(const Shape& s, ld k, ld lo, ld hi) {
  Norm N;
  const ld dl = lo - s.mu, dh = hi - s.mu;
  const ld dref = std::min(std::max((ld)0, dl), dh);
  N.logref = log_I(s, dref);
  N.left = N.right = N.core = 0;
  if (dl < s.d0) { /* left tail on [dl, min(d0,dh)] */
    const ld dr = std::min(s.d0, dh);
    const ld ul = 1 - (dl - s.d0) * s.L0 / s.n, ur = 1 - (dr - s.d0) * s.L0 / s.n;
    ld ls;
    const ld Fd = powint_diff(ul, ur, s.n, &ls);
    N.left = expl(s.logG0 - N.logref + ls) * (s.n / s.L0) * Fd;
  }
  if (dh > s.d1) { /* right tail on [max(d1,dl), dh] */
    const ld dL = std::max(s.d1, dl);
    const ld uh = 1 - (dh - s.d1) * s.L1 / s.n2, ul = 1 - (dL - s.d1) * s.L1 / s.n2;
    ld ls;
    const ld Fd = powint_diff(uh, ul, s.n2, &ls);
    N.right = expl(s.logG1 - N.logref + ls) * (s.n2 / (-s.L1)) * Fd;
  }
  const ld A = std::max(dl, s.d0), B = std::min(dh, s.d1);
  if (B > A) {
    if (A < 0 && B > 0) N.core = core_integral_scaled(s, A, 0, N.logref) + core_integral_scaled(s, 0, B, N.logref);
    else N.core = core_integral_scaled(s, A, B, N.logref);
  }
  N.NS = N.left + N.core + N.right; /* in units of exp(logref) */
  const ld w = hi - lo, t = k * w;
  N.NB = (fabsl(t) < 1e-8L) ? w * (1 + t / 2 + t * t / 6) : expm1l(t) / k;
  return N;
}

/* per-event log-likelihood (reading C3) */
static ld event_logpdf(const Shape& s, const Norm& N, ld f, ld k, ld lo, ld x) {
  const ld ES = (f > 0) ? logl(f) + log_I(s, x - s.mu) - N.logref - logl(N.NS) : -INFINITY;
  const ld EB = (f < 1) ? log1pl(-f) + k * (x - lo) - logl(N.NB) : -INFINITY;
  if (!(f > 0)) return EB;
  if (!(f < 1)) return ES;
  const ld m = std::max(ES, EB);
  return m + log1pl(expl(-fabsl(ES - EB)));
}

/* pairwise summation (north star; reading C3): recursive halving, leaves of <=64 left to right */
static ld pairwise(const double* v, int64_t i, int64_t j) {
  if (j - i <= 64) { ld s = 0; for (int64_t t = i; t < j; ++t) s += v[t]; return s; }
  const int64_t m = i + (j - i) / 2;
  return pairwise(v, i, m) + pairwise(v, m, j);
}

static ld nll_one(const double* x, int64_t n, const orc_params& p, ld lo, ld hi) {
  const Shape s = make_shape(p);
  if (s.status) return INFINITY;
  const Norm N = make_norm(s, p.k, lo, hi);
  std::vector<double> l((size_t)n);
  for (int64_t i = 0; i < n; ++i) l[i] = (double)event_logpdf(s, N, p.f, p.k, lo, x[i]);
  return -pairwise(l.data(), 0, n);
}

/* ------------------------------------------------------------------------------------------
 * Analytic gradient of the NLL with respect to (mu, sigma, f, k)  (the paper
 * offers analytic gradients through iminuit and generated derivative code, without
 * formulae).  Written out from the definition C1-C3 by the chain rule; nothing is approximated:
 *   w_S = f S / (f S + (1-f) B),  w_B = 1 - w_S
 *   d l / d f     = w_S / f - w_B / (1 - f)
 *   d l / d k     = w_B ( (x - lo) - d ln N_B / d k )
 *   d l / d mu    = w_S ( - dlogI/dd (x - mu) - d ln N_S / d mu )
 *   d l / d sigma = w_S ( dlogI/dsigma (x - mu) - d ln N_S / d sigma )
 * with (delta = sigma c1, alpha = c2 / sigma, d0 = -a sigma, d1 = a2 sigma; L = core log-derivative):
 * (nu below stands for the power of sigma in G(d; sigma) = sigma^p g(d/sigma) e^{beta d}: p = nu for the Bessel core,
 *  p = 2 nu for the zeta = 0 Student-t core -- Shape::sigpow)
 *   core   dlogI/dd = L(d)              dlogI/dsigma = nu/sigma + (d/sigma)(beta - L(d))
 *   left   dlogI/dd = L0 / u            dlogI/dsigma = nu/sigma - a beta + [ a L0 - (d-d0)(L0-beta)/sigma ] / u
 *   right  dlogI/dd = L1 / u            dlogI/dsigma = nu/sigma + a2 beta - [ a2 L1 + (d-d1)(L1-beta)/sigma ] / u
 *          u = 1 - (d - d_join) L_join / n_join
 *   d N_S / d mu    = I(lo - mu) - I(hi - mu)                      (Leibniz: the limits move with mu)
 *   d N_S / d sigma = int_lo^hi I dlogI/dsigma dx                  (composite Gauss-Legendre per region)
 *   d ln N_B / d k  = w e^{k w} / expm1(k w) - 1/k,  w = hi - lo   (-> w/2 as k -> 0)
 * beta (fifth component, round 2; SURVEY.md 8(f) f1 "(mu,sigma,f,k[,beta,...])"): delta and alpha do not depend on
 * beta, the core carries e^{beta d}, and the tails inherit beta through log G(d_join) and L_join (dL_join/dbeta = 1):
 *   d l / d beta = w_S ( dlogI/dbeta (x - mu) - d ln N_S / d beta )
 *   core   dlogI/dbeta = d        left   dlogI/dbeta = d0 + (d - d0)/u        right  dlogI/dbeta = d1 + (d - d1)/u
 *   d N_S / d beta = int_lo^hi I dlogI/dbeta dx                        (composite Gauss-Legendre per region)
 * ---------------------------------------------------------------------------------------- */
static ld dlogI_dd(const Shape& s, ld d) {
  if (d < s.d0) return s.L0 / (1 - (d - s.d0) * s.L0 / s.n);
  if (d > s.d1) return s.L1 / (1 - (d - s.d1) * s.L1 / s.n2);
  return core_logderiv(s, d);
}
static ld dlogI_dsigma(const Shape& s, ld d) {
  if (d < s.d0) {
    const ld u = 1 - (d - s.d0) * s.L0 / s.n;
    return s.sigpow / s.sigma - s.a * s.beta + (s.a * s.L0 - (d - s.d0) * (s.L0 - s.beta) / s.sigma) / u;
  }
  if (d > s.d1) {
    const ld u = 1 - (d - s.d1) * s.L1 / s.n2;
    return s.sigpow / s.sigma + s.a2 * s.beta - (s.a2 * s.L1 + (d - s.d1) * (s.L1 - s.beta) / s.sigma) / u;
  }
  return s.sigpow / s.sigma + (d / s.sigma) * (s.beta - core_logderiv(s, d));
}
static ld dlogI_dbeta(const Shape& s, ld d) {
  if (d < s.d0) return s.d0 + (d - s.d0) / (1 - (d - s.d0) * s.L0 / s.n);
  if (d > s.d1) return s.d1 + (d - s.d1) / (1 - (d - s.d1) * s.L1 / s.n2);
  return d;
}
/* int_A^B I(d) dlogI/dtheta(d) e^{-logref} dd inside ONE region (smooth integrand), theta = sigma (which = 0) or
 * beta (which = 1); composite 20-point Gauss-Legendre, panels doubled until stable */
static ld dsigma_integral_scaled(const Shape& s, ld A, ld B, ld logref, int which = 0) {
  if (!(B > A)) return 0;
  std::vector<ld> gx, gw;
  gauss_legendre(20, gx, gw);
  ld prev = 0;
  for (int P = 4; P <= 8192; P *= 2) {
    ld tot = 0;
    const ld h = (B - A) / P;
    for (int j = 0; j < P; ++j) {
      const ld c = A + (j + 0.5L) * h;
      ld acc = 0;
      for (int i = 0; i < 20; ++i) {
        const ld d = c + 0.5L * h * gx[i];
        acc += gw[i] * expl(log_I(s, d) - logref) * (which ? dlogI_dbeta(s, d) : dlogI_dsigma(s, d));
      }
      tot += acc * 0.5L * h;
    }
    if (P > 4 && fabsl(tot - prev) <= 1e-15L * (fabsl(tot) + 1e-300L)) return tot;
    prev = tot;
  }
  return prev;
}
/* d ln N_S / d mu, d ln N_S / d sigma, d ln N_B / d k  (N.NS is in units of exp(logref)) */
static void norm_derivs(const Shape& s, const Norm& N, ld k, ld lo, ld hi, ld* dlnNS_dmu, ld* dlnNS_dsig, ld* dlnNB_dk,
                        ld* dlnNS_dbeta = nullptr) {
  const ld dl = lo - s.mu, dh = hi - s.mu;
  const ld dNS_dmu = expl(log_I(s, dl) - N.logref) - expl(log_I(s, dh) - N.logref);
  ld dNS_dsig = 0;
  ld cuts[6]; int nc = 0;
  cuts[nc++] = dl;
  const ld inner[3] = {s.d0, 0, s.d1};
  for (int i = 0; i < 3; ++i) if (inner[i] > dl && inner[i] < dh) cuts[nc++] = inner[i];
  cuts[nc++] = dh;
  for (int i = 0; i + 1 < nc; ++i) dNS_dsig += dsigma_integral_scaled(s, cuts[i], cuts[i + 1], N.logref);
  if (dlnNS_dbeta) {
    ld dNS_dbeta = 0;
    for (int i = 0; i + 1 < nc; ++i) dNS_dbeta += dsigma_integral_scaled(s, cuts[i], cuts[i + 1], N.logref, 1);
    *dlnNS_dbeta = dNS_dbeta / N.NS;
  }
  *dlnNS_dmu = dNS_dmu / N.NS;
  *dlnNS_dsig = dNS_dsig / N.NS;
  const ld w = hi - lo, t = k * w;
  *dlnNB_dk = (fabsl(t) < 1e-6L) ? w * (0.5L + t / 12) : w * expl(t) / expm1l(t) - 1 / k;
}
extern "C" int orc_norm_derivs(const orc_params* pp, double lo, double hi, double* out /* [4]: mu, sigma, k, beta */) {
  const Shape s = make_shape(*pp);
  if (s.status) return s.status;
  const Norm N = make_norm(s, pp->k, lo, hi);
  ld a, b, c, e;
  norm_derivs(s, N, pp->k, lo, hi, &a, &b, &c, &e);
  out[0] = (double)a; out[1] = (double)b; out[2] = (double)c; out[3] = (double)e;
  return 0;
}
extern "C" int orc_nll_gradient(const double* x, int64_t n, const orc_params* pp, double lo_, double hi_, double* nll,
                                double* grad /* d NLL / d (mu, sigma, f, k, beta) */) {
  const orc_params& p = *pp;
  const Shape s = make_shape(p);
  if (s.status) return s.status;
  const ld lo = lo_, hi = hi_, f = p.f, k = p.k;
  const Norm N = make_norm(s, k, lo, hi);
  const ld dl = lo - s.mu, dh = hi - s.mu;
  ld dlnNS_dmu, dlnNS_dsig, dlnNB_dk, dlnNS_dbeta;
  norm_derivs(s, N, k, lo, hi, &dlnNS_dmu, &dlnNS_dsig, &dlnNB_dk, &dlnNS_dbeta);
  (void)dl; (void)dh;
  std::vector<double> g0((size_t)n), g1((size_t)n), g2((size_t)n), g3((size_t)n), g4((size_t)n), l((size_t)n);
  for (int64_t i = 0; i < n; ++i) {
    const ld d = (ld)x[i] - s.mu;
    const ld ES = (f > 0) ? logl(f) + log_I(s, d) - N.logref - logl(N.NS) : -INFINITY;
    const ld EB = (f < 1) ? log1pl(-f) + k * ((ld)x[i] - lo) - logl(N.NB) : -INFINITY;
    const ld li = event_logpdf(s, N, f, k, lo, x[i]);
    const ld wS = (f > 0) ? expl(ES - li) : 0, wB = (f < 1) ? expl(EB - li) : 0;
    l[i] = (double)li;
    g0[i] = (double)(wS * (-dlogI_dd(s, d) - dlnNS_dmu));
    g1[i] = (double)(wS * (dlogI_dsigma(s, d) - dlnNS_dsig));
    /* S/mix - B/mix written with the weights: w_S / f - w_B / (1 - f); the limits f -> 0, 1 use S/B directly */
    const ld SoverMix = (f > 0) ? wS / f : expl(log_I(s, d) - N.logref - logl(N.NS) - li);
    const ld BoverMix = (f < 1) ? wB / (1 - f) : expl(k * ((ld)x[i] - lo) - logl(N.NB) - li);
    g2[i] = (double)(SoverMix - BoverMix);
    g3[i] = (double)(wB * (((ld)x[i] - lo) - dlnNB_dk));
    g4[i] = (double)(wS * (dlogI_dbeta(s, d) - dlnNS_dbeta));
  }
  *nll = (double)(-pairwise(l.data(), 0, n));
  grad[0] = (double)(-pairwise(g0.data(), 0, n));
  grad[1] = (double)(-pairwise(g1.data(), 0, n));
  grad[2] = (double)(-pairwise(g2.data(), 0, n));
  grad[3] = (double)(-pairwise(g3.data(), 0, n));
  grad[4] = (double)(-pairwise(g4.data(), 0, n));
  return 0;
}
/* ------------------------------------------------------------------------------------------
 * Counter-based generator: Philox-4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), restated.
 * ---------------------------------------------------------------------------------------- */
static void philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { STREAM_COMP = 0, STREAM_SIG = 1, STREAM_BKG = 2, STREAM_YIELD = 3, STREAM_BIN = 4 };

/* two uniforms in (0,1) from one block: u = ((w>>5) 2^26 + (w'>>6) + 0.5) 2^-53  (reading D13) */
static void uniforms2(uint64_t seed, uint64_t slot, uint32_t attempt, uint32_t stream, double* u0, double* u1) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  const uint32_t ctr[4] = {(uint32_t)slot, (uint32_t)(slot >> 32), attempt, stream};
  uint32_t w[4];
  philox4x32_10(key, ctr, w);
  *u0 = ((double)(w[0] >> 5) * 67108864.0 + (double)(w[1] >> 6) + 0.5) * (1.0 / 9007199254740992.0);
  *u1 = ((double)(w[2] >> 5) * 67108864.0 + (double)(w[3] >> 6) + 0.5) * (1.0 / 9007199254740992.0);
}

/* Poisson(mean) on Philox uniforms (reading D14): sequential-search inversion for mean<10,
 * Hoermann's transformed rejection PTRS (Insurance: Math. & Econ. 12 (1993) 39) otherwise. */
/* diag (optional, tests only): diag[0] = attempts used, diag[1] = exit taken (0 inversion, 1 the quick
 * acceptance of the squeeze, 2 the full comparison with the probability function); no effect on the draw. */
static int64_t poisson_draw(uint64_t seed, uint64_t slot, uint32_t stream, double mean, int32_t* diag = nullptr) {
  if (diag) { diag[0] = 0; diag[1] = 0; }
  if (!(mean > 0)) return 0;
  if (mean < 10) {
    double u, v;
    uniforms2(seed, slot, 0, stream, &u, &v);
    int64_t k = 0;
    double p = std::exp(-mean), F = p;
    while (u > F && k < 1000) { ++k; p *= mean / (double)k; F += p; }
    return k;
  }
  const double smu = std::sqrt(mean);
  const double b = 0.931 + 2.53 * smu;
  const double a = -0.059 + 0.02483 * b;
  const double inv_alpha = 1.1239 + 1.1328 / (b - 3.4);
  const double vr = 0.9277 - 3.6224 / (b - 2.0);
  const double lmean = std::log(mean);
  for (uint32_t attempt = 0;; ++attempt) {
    double U, V;
    uniforms2(seed, slot, attempt, stream, &U, &V);
    U -= 0.5;
    const double us = 0.5 - std::fabs(U);
    const double kf = std::floor((2.0 * a / us + b) * U + mean + 0.43);
    if (diag) { diag[0] = (int32_t)attempt + 1; diag[1] = 1; }
    if (us >= 0.07 && V <= vr) return (int64_t)kf;
    if (kf < 0 || (us < 0.013 && V > us)) continue;
    if (diag) diag[1] = 2;
    if (std::log(V) + std::log(inv_alpha) - std::log(a / (us * us) + b) <= -mean + kf * lmean - std::lgamma(kf + 1.0))
      return (int64_t)kf;
  }
}

/* ------------------------------------------------------------------------------------------
 * Signal draws (reading D13, revised in round 2; PAPER.md:343-351 says only "accept-reject"): accept-reject under a
 * PIECEWISE envelope that is a true upper bound of I on the range [lo, hi] (d = x - mu in [dl, dh]):
 *   left tail  [dl, min(d0, dh)]   (if dl < d0):  envelope = I itself; weight = its exact integral (reading C5)
 *   core       [A, B] = [max(dl, d0), min(dh, d1)] cut into ENV_BOXES equal boxes; the core is unimodal (one sign
 *              change of L between the joins), so the maximum of G over a box is G at the point of the box closest
 *              to the mode d_m; box height h_j = that maximum times (1 + 2^-20); weight = h_j * width
 *   right tail [max(d1, dl), dh]   (if dh > d1):  envelope = I itself; weight = its exact integral
 * Mode d_m: 0 for beta = 0, else the root of L(d) = 0 between the joins by bisection.
 * Attempt t = 0, 1, ... of (seed, slot): (u1, u2) = uniforms2(seed, slot, t, STREAM_SIG); v = u1 * (total weight)
 * selects the region r (cumulative weights in the order left tail, boxes, right tail);
 *   tail:  the power law is sampled exactly by its inverse CDF with u2 (always accepted): with u = 1 - (d-d_j) L_j/n_j
 *          the mass from the region's left end is linear in t = u^{1-n} (in log u for n = 1), so
 *          t = t_a + u2 (t_b - t_a),  u = t^{1/(1-n)},  d = d_j - (u - 1) n_j / L_j
 *   box:   d = box_lo + width * (v - cum[r]) / weight_r  (the remainder of u1 is uniform);  accept iff u2 h_j < G(d).
 * All weights are in units of exp(logref) (the level make_norm uses).
 * ---------------------------------------------------------------------------------------- */
enum { ENV_BOXES = 16, ENV_MAXREG = ENV_BOXES + 2 };
struct Envelope {
  int nreg;
  int kind[ENV_MAXREG];          /* 0 left tail, 1 box, 2 right tail */
  ld cum[ENV_MAXREG + 1];        /* cumulative weights, cum[0] = 0 */
  ld blo[ENV_MAXREG], bw;        /* boxes: left edge, common width */
  ld logh[ENV_MAXREG];           /* boxes: log of the height (absolute, like log_I) */
  ld ta[ENV_MAXREG], tb[ENV_MAXREG]; /* tails: t (or log u for n = 1) at the left and right end of the region */
  ld logref;
};

static ld core_mode(const Shape& s) {
  if (s.beta == 0) return 0;
  ld a = s.d0, b = s.d1;                       /* L(d0) > 0 > L(d1) (status 0) */
  for (int it = 0; it < 200 && b - a > 1e-18L * (fabsl(a) + fabsl(b)); ++it) {
    const ld m = 0.5L * (a + b);
    if (core_logderiv(s, m) > 0) a = m; else b = m;
  }
  return 0.5L * (a + b);
}

static ld tail_t(ld u, ld n) { return (n == 1) ? logl(u) : powl(u, 1 - n); }

static Envelope make_envelope(const Shape& s, ld lo, ld hi) {
  Envelope E;
  const Norm N = make_norm(s, 0, lo, hi);
  const ld dl = lo - s.mu, dh = hi - s.mu;
  E.logref = N.logref;
  E.nreg = 0;
  E.cum[0] = 0;
  E.bw = 0;
  if (dl < s.d0) {
    const ld dr = std::min(s.d0, dh);
    const int r = E.nreg++;
    E.kind[r] = 0;
    E.ta[r] = tail_t(1 - (dl - s.d0) * s.L0 / s.n, s.n);
    E.tb[r] = tail_t(1 - (dr - s.d0) * s.L0 / s.n, s.n);
    E.cum[r + 1] = E.cum[r] + N.left;
  }
  const ld A = std::max(dl, s.d0), B = std::min(dh, s.d1);
  if (B > A) {
    const ld dm = core_mode(s);
    E.bw = (B - A) / ENV_BOXES;
    for (int j = 0; j < ENV_BOXES; ++j) {
      const int r = E.nreg++;
      E.kind[r] = 1;
      E.blo[r] = A + j * E.bw;
      const ld bhi = (j == ENV_BOXES - 1) ? B : A + (j + 1) * E.bw;
      const ld closest = std::min(std::max(dm, E.blo[r]), bhi);
      E.logh[r] = core_logG(s, closest) + log1pl(ldexpl(1, -20));
      E.cum[r + 1] = E.cum[r] + expl(E.logh[r] - N.logref) * E.bw;
    }
  }
  if (dh > s.d1) {
    const ld dL = std::max(s.d1, dl);
    const int r = E.nreg++;
    E.kind[r] = 2;
    E.ta[r] = tail_t(1 - (dL - s.d1) * s.L1 / s.n2, s.n2);
    E.tb[r] = tail_t(1 - (dh - s.d1) * s.L1 / s.n2, s.n2);
    E.cum[r + 1] = E.cum[r] + N.right;
  }
  return E;
}

/* diag (tests only): diag[0] += attempts used, diag[1] = 1 if an attempt saw G(d) above its box height */
static double draw_signal(const Shape& s, const Envelope& E, uint64_t seed, uint64_t slot, int64_t* diag = nullptr) {
  for (uint32_t attempt = 0;; ++attempt) {
    double u1, u2;
    uniforms2(seed, slot, attempt, STREAM_SIG, &u1, &u2);
    if (diag) diag[0] += 1;
    const ld v = (ld)u1 * E.cum[E.nreg];
    int r = 0;
    while (r + 1 < E.nreg && v >= E.cum[r + 1]) ++r;
    if (E.kind[r] != 1) {
      const ld n = (E.kind[r] == 0) ? s.n : s.n2, L = (E.kind[r] == 0) ? s.L0 : s.L1, dj = (E.kind[r] == 0) ? s.d0 : s.d1;
      const ld t = E.ta[r] + (ld)u2 * (E.tb[r] - E.ta[r]);
      const ld u = (n == 1) ? expl(t) : powl(t, 1 / (1 - n));
      return (double)(s.mu + (dj - (u - 1) * n / L));
    }
    const ld d = E.blo[r] + E.bw * ((v - E.cum[r]) / (E.cum[r + 1] - E.cum[r]));
    const ld lg = core_logG(s, d);
    if (diag && lg > E.logh[r]) diag[1] = 1;
    if ((ld)u2 < expl(lg - E.logh[r])) return (double)(s.mu + d);
    if (attempt > 100000u) return (double)(s.mu + d); /* unreachable: the acceptance is >= 1/2 for any unimodal core */
  }
}

static double draw_background(double k, uint64_t seed, uint64_t slot, double lo, double hi) {
  double u, v;
  uniforms2(seed, slot, 0, STREAM_BKG, &u, &v);
  const double w = hi - lo, t = k * w;
  if (std::fabs(t) < 1e-8) return lo + u * w;
  return lo + std::log1p(u * std::expm1(t)) / k; /* inverse CDF of the truncated exponential */
}

/* ========================================================================================== */
extern "C" {

double orc_besselk_scaled(double nu, double x) { return (double)besselk_scaled_l(nu, x); }
double orc_log_besselk(double nu, double x) { return (double)(logl(besselk_scaled_l(nu, x)) - (ld)x); }
double orc_zeta_int(int k) { return (double)zeta_int(k); }

/* out[8] = delta, alpha, d0, d1, logG0, logG1, L0, L1 ; returns status */
int orc_shape_consts(const orc_params* p, double* out) {
  const Shape s = make_shape(*p);
  if (s.status == 1) return 1;
  out[0] = (double)s.delta; out[1] = (double)s.alpha; out[2] = (double)s.d0; out[3] = (double)s.d1;
  out[4] = (double)s.logG0; out[5] = (double)s.logG1; out[6] = (double)s.L0; out[7] = (double)s.L1;
  return s.status;
}

/* log I(d) and L(d)=dlogG/dd of the core (for the join-continuity and derivative pins) */
double orc_log_I(const orc_params* p, double d) { const Shape s = make_shape(*p); return s.status ? NAN : (double)log_I(s, d); }
double orc_core_logG(const orc_params* p, double d) { const Shape s = make_shape(*p); return s.status == 1 ? NAN : (double)core_logG(s, d); }
double orc_core_logderiv(const orc_params* p, double d) { const Shape s = make_shape(*p); return s.status == 1 ? NAN : (double)core_logderiv(s, d); }

/* out[5] = N_S, core, left, right (all absolute, i.e. multiplied by exp(logref)), N_B */
int orc_norm(const orc_params* p, double lo, double hi, double* out) {
  const Shape s = make_shape(*p);
  if (s.status) { for (int i = 0; i < 5; ++i) out[i] = NAN; return s.status; }
  const Norm N = make_norm(s, p->k, lo, hi);
  const ld sc = expl(N.logref);
  out[0] = (double)(N.NS * sc); out[1] = (double)(N.core * sc); out[2] = (double)(N.left * sc);
  out[3] = (double)(N.right * sc); out[4] = (double)N.NB;
  return 0;
}

/* per-event log( f S(x) + (1-f) B(x) ) */
int orc_logpdf(const double* x, int64_t n, const orc_params* p, double lo, double hi, double* out) {
  const Shape s = make_shape(*p);
  if (s.status) { for (int64_t i = 0; i < n; ++i) out[i] = -INFINITY; return s.status; }
  const Norm N = make_norm(s, p->k, lo, hi);
  for (int64_t i = 0; i < n; ++i) out[i] = (double)event_logpdf(s, N, p->f, p->k, lo, x[i]);
  return 0;
}

/* normalised signal pdf S(x) alone (pins: integral = 1, worked example) */
double orc_signal_pdf(const orc_params* p, double lo, double hi, double x) {
  const Shape s = make_shape(*p);
  if (s.status) return NAN;
  const Norm N = make_norm(s, p->k, lo, hi);
  return (double)(expl(log_I(s, (ld)x - s.mu) - N.logref) / N.NS);
}

/* NLL_k = -sum_i l_ik for K parameter sets; nthreads==1 is THE oracle (pairwise sum in original
 * order); nthreads>1 gives each thread a contiguous chunk evaluated by the same routine and adds
 * the chunk sums in order (timing baseline, and large-N parity where stated). */
int orc_nll(const double* x, int64_t n, const orc_params* p, int K, double lo, double hi, double* nll, int nthreads) {
  for (int k = 0; k < K; ++k) {
    if (nthreads <= 1 || n < 4096) { nll[k] = (double)nll_one(x, n, p[k], lo, hi); continue; }
    std::vector<ld> part((size_t)nthreads, 0);
    std::vector<std::thread> th;
    for (int t = 0; t < nthreads; ++t) {
      const int64_t b = n * t / nthreads, e = n * (t + 1) / nthreads;
      th.emplace_back([&, t, b, e]() { part[(size_t)t] = nll_one(x + b, e - b, p[k], lo, hi); });
    }
    for (auto& h : th) h.join();
    ld s = 0;
    for (int t = 0; t < nthreads; ++t) s += part[(size_t)t];
    nll[k] = (double)s;
  }
  return 0;
}

/* Finite-difference gradient (reading C6): central differences over P floated parameters.
 * Set 0 = theta, sets 2j+1 / 2j+2 = theta with field idx[j] replaced by theta[idx[j]] +/- h[j] (each sum computed
 * once, in fp64), g_j = (NLL(theta + h_j e_j) - NLL(theta - h_j e_j)) / (2 h_j).  nll [2P+1] receives the NLLs of
 * the batch in that order, grad [P] the differences.  nthreads as in orc_nll. */
int orc_fd_gradient(const double* x, int64_t n, const orc_params* theta, int P, const int32_t* idx, const double* h,
                    double lo, double hi, int nthreads, double* nll, double* grad) {
  if (P < 1 || P > 11) return -1;
  std::vector<orc_params> batch((size_t)(2 * P + 1), *theta);
  for (int j = 0; j < P; ++j) {
    if (idx[j] < 0 || idx[j] > 10) return -1;
    const double base = (&theta->mu)[idx[j]];
    (&batch[(size_t)(2 * j + 1)].mu)[idx[j]] = base + h[j];
    (&batch[(size_t)(2 * j + 2)].mu)[idx[j]] = base - h[j];
  }
  orc_nll(x, n, batch.data(), 2 * P + 1, lo, hi, nll, nthreads);
  for (int j = 0; j < P; ++j) grad[j] = (nll[2 * j + 1] - nll[2 * j + 2]) / (2.0 * h[j]);
  return 0;
}

/* NLL per segment (toy), one parameter set per segment: offsets[T+1] */
int orc_nll_segmented(const double* x, const int64_t* offsets, int64_t T, const orc_params* p, double lo, double hi,
                      double* nll) {
  for (int64_t t = 0; t < T; ++t) nll[t] = (double)nll_one(x + offsets[t], offsets[t + 1] - offsets[t], p[t], lo, hi);
  return 0;
}

void orc_philox4x32_10(const uint32_t* key, const uint32_t* ctr, uint32_t* out) { philox4x32_10(key, ctr, out); }
void orc_uniforms2(uint64_t seed, uint64_t slot, uint32_t attempt, uint32_t stream, double* u) { uniforms2(seed, slot, attempt, stream, u, u + 1); }
int64_t orc_poisson(uint64_t seed, uint64_t slot, uint32_t stream, double mean) { return poisson_draw(seed, slot, stream, mean); }
/* n draws at slots slot0 .. slot0+n-1 (the same draws as n calls of orc_poisson); diag [2 n] optional: attempts and exit per draw */
void orc_poisson_array(uint64_t seed, uint64_t slot0, int64_t n, uint32_t stream, double mean, int64_t* out, int32_t* diag) {
  for (int64_t i = 0; i < n; ++i) out[i] = poisson_draw(seed, slot0 + (uint64_t)i, stream, mean, diag ? diag + 2 * i : nullptr);
}

/* configs 1-3: n events, component chosen per event by u<f (reading D13) */
int orc_generate_mixture(uint64_t seed, int64_t n, const orc_params* p, double lo, double hi, double* x) {
  const Shape s = make_shape(*p);
  if (s.status) return s.status;
  const Envelope env = make_envelope(s, lo, hi);
  for (int64_t i = 0; i < n; ++i) {
    double uc, v;
    uniforms2(seed, (uint64_t)i, 0, STREAM_COMP, &uc, &v);
    x[i] = (uc < p->f) ? draw_signal(s, env, seed, (uint64_t)i) : draw_background(p->k, seed, (uint64_t)i, lo, hi);
  }
  return 0;
}

/* tests only: n signal draws (slots 0..n-1) with the envelope diagnostics: diag[0] = total attempts, diag[1] = 1 if any
 * attempt found the core above its box height; env_out[0] = total envelope weight / N_S (1 / acceptance), env_out[1] below */
int orc_generate_signal_diag(uint64_t seed, int64_t n, const orc_params* p, double lo, double hi, double* x, int64_t* diag,
                             double* env_out) {
  const Shape s = make_shape(*p);
  if (s.status) return s.status;
  const Envelope env = make_envelope(s, lo, hi);
  const Norm N = make_norm(s, 0, lo, hi);
  diag[0] = diag[1] = 0;
  for (int64_t i = 0; i < n; ++i) x[i] = draw_signal(s, env, seed, (uint64_t)i, diag);
  env_out[0] = (double)(env.cum[env.nreg] / N.NS);
  /* env_out[1] = max over a dense grid of log G(d) - log h(box of d): the envelope is a bound iff this is <= 0 */
  ld worst = -INFINITY;
  for (int r = 0; r < env.nreg; ++r) {
    if (env.kind[r] != 1) continue;
    for (int i = 0; i <= 4000; ++i) worst = std::max(worst, core_logG(s, env.blo[r] + env.bw * i / 4000) - env.logh[r]);
  }
  env_out[1] = (double)worst;
  return 0;
}

/* config 4: T toys; toy t has Ns~Poisson(mean_sig), Nb~Poisson(mean_bkg) from seeds[t]; signal events
 * first, then background; offsets = exclusive scan. gen has T entries (gen_stride=1) or one (0).
 * Call with x==NULL to get the offsets only. Returns <0 if capacity is too small. */
int orc_toy_generate(const uint64_t* seeds, int64_t T, const orc_params* gen, int gen_stride, double mean_sig,
                     double mean_bkg, double lo, double hi, int64_t capacity, double* x, int64_t* offsets) {
  offsets[0] = 0;
  std::vector<int64_t> ns((size_t)T);
  for (int64_t t = 0; t < T; ++t) {
    ns[(size_t)t] = poisson_draw(seeds[t], 0, STREAM_YIELD, mean_sig);
    const int64_t nb = poisson_draw(seeds[t], 1, STREAM_YIELD, mean_bkg);
    offsets[t + 1] = offsets[t] + ns[(size_t)t] + nb;
  }
  if (!x) return 0;
  if (offsets[T] > capacity) return -1;
  for (int64_t t = 0; t < T; ++t) {
    const orc_params& p = gen[gen_stride ? t : 0];
    const Shape s = make_shape(p);
    if (s.status) return s.status;
    const Envelope env = make_envelope(s, lo, hi);
    const int64_t nt = offsets[t + 1] - offsets[t];
    for (int64_t j = 0; j < nt; ++j)
      x[offsets[t] + j] = (j < ns[(size_t)t]) ? draw_signal(s, env, seeds[t], (uint64_t)j)
                                               : draw_background(p.k, seeds[t], (uint64_t)j, lo, hi);
  }
  return 0;
}

/* B1: histogram, nbins uniform bins on [lo,hi]; bin = floor((x-lo)*nbins/(hi-lo)); x==hi goes to the
 * last bin; events outside the range are dropped. */
void orc_hist_fill(const double* x, int64_t n, double lo, double hi, int nbins, uint64_t* counts) {
  for (int b = 0; b < nbins; ++b) counts[b] = 0;
  const double scale = (double)nbins / (hi - lo);
  for (int64_t i = 0; i < n; ++i) {
    const double t = (x[i] - lo) * scale;
    if (!(t >= 0) || !(x[i] <= hi)) continue;
    int b = (int)t;
    if (b >= nbins) b = nbins - 1;
    counts[b]++;
  }
}

/* B2 (reading D15): s_b = I(c_b-mu)/sum I, b_b = e^{k(c_b-lo)}/sum e^{k(c_b'-lo)},
 * nu_b = ns s_b + nb b_b, NLL = sum_b [nu_b - n_b log nu_b]  (n_b=0 -> nu_b). */
int orc_binned_nll_scan(const uint64_t* counts, int nbins, double lo, double hi, const orc_params* shape,
                        const double* ns, const double* nb, const double* kk, int64_t npoints, double* nll) {
  const Shape s = make_shape(*shape);
  if (s.status) return s.status;
  std::vector<ld> sb((size_t)nbins), c((size_t)nbins);
  const ld w = ((ld)hi - lo) / nbins;
  ld ssum = 0;
  const ld ref = log_I(s, std::min(std::max((ld)0, (ld)lo - s.mu), (ld)hi - s.mu));
  for (int b = 0; b < nbins; ++b) {
    c[(size_t)b] = lo + (b + 0.5L) * w;
    sb[(size_t)b] = expl(log_I(s, c[(size_t)b] - s.mu) - ref);
    ssum += sb[(size_t)b];
  }
  for (int b = 0; b < nbins; ++b) sb[(size_t)b] /= ssum;
  std::vector<ld> bb((size_t)nbins);
  std::vector<double> terms((size_t)nbins);
  for (int64_t q = 0; q < npoints; ++q) {
    ld bsum = 0;
    for (int b = 0; b < nbins; ++b) { bb[(size_t)b] = expl((ld)kk[q] * (c[(size_t)b] - lo)); bsum += bb[(size_t)b]; }
    for (int b = 0; b < nbins; ++b) {
      const ld v = (ld)ns[q] * sb[(size_t)b] + (ld)nb[q] * bb[(size_t)b] / bsum;
      terms[(size_t)b] = (double)(counts[b] ? v - (ld)counts[b] * logl(v) : v);
    }
    nll[q] = (double)pairwise(terms.data(), 0, nbins);
  }
  return 0;
}

/* expected histogram nu_b for one (ns, nb, k) point (inputs of B3) */
int orc_expected_hist(int nbins, double lo, double hi, const orc_params* shape, double ns, double nb, double k, double* nu) {
  const Shape s = make_shape(*shape);
  if (s.status) return s.status;
  const ld w = ((ld)hi - lo) / nbins;
  std::vector<ld> sb((size_t)nbins), bb((size_t)nbins);
  ld ssum = 0, bsum = 0;
  const ld ref = log_I(s, std::min(std::max((ld)0, (ld)lo - s.mu), (ld)hi - s.mu));
  for (int b = 0; b < nbins; ++b) {
    const ld c = lo + (b + 0.5L) * w;
    sb[(size_t)b] = expl(log_I(s, c - s.mu) - ref); ssum += sb[(size_t)b];
    bb[(size_t)b] = expl((ld)k * (c - lo)); bsum += bb[(size_t)b];
  }
  for (int b = 0; b < nbins; ++b) nu[b] = (double)((ld)ns * sb[(size_t)b] / ssum + (ld)nb * bb[(size_t)b] / bsum);
  return 0;
}

/* B3: n_{t,b} ~ Poisson(mean_b), key = seeds[t], counter slot = b, stream STREAM_BIN */
void orc_poisson_hist_toys(const double* mean, int nbins, const uint64_t* seeds, int64_t T, uint32_t* counts) {
  for (int64_t t = 0; t < T; ++t)
    for (int b = 0; b < nbins; ++b) counts[t * nbins + b] = (uint32_t)poisson_draw(seeds[t], (uint64_t)b, STREAM_BIN, mean[b]);
}


/* ------------------------------------------------------------------------------------------
 * CLs on binned toys (CL.setData(fake_data),
 * CL.setExpected(HistoPdf), CL.CLs(ns, toys = 10000)).  The paper does not print its test statistic
 * (it cites its refs [11,12] for the CLs method) -> DESIGN.md reading F2: the likelihood ratio of the
 * two fixed expected histograms,
 *      q(n) = -2 ln [ L(n | nu_sb) / L(n | nu_b) ] = 2 sum_b [ (nu_sb_b - nu_b_b) - n_b ln(nu_sb_b / nu_b_b) ],
 * larger q = more background-like;  CL_sb = P(q >= q_obs | s+b toys),  CL_b = P(q >= q_obs | b toys),
 * CL_s = CL_sb / CL_b.  Plain left-to-right sums in long double.
 * ---------------------------------------------------------------------------------------- */
void orc_cls_teststat(const void* counts, int count_bytes, int64_t T, int nbins, const double* nu_sb,
                      const double* nu_b, double* q) {
  for (int64_t t = 0; t < T; ++t) {
    ld acc = 0;
    for (int b = 0; b < nbins; ++b) {
      const ld n = count_bytes == 8 ? (ld)((const uint64_t*)counts)[t * nbins + b]
                                    : (ld)((const uint32_t*)counts)[t * nbins + b];
      acc += ((ld)nu_sb[b] - (ld)nu_b[b]) - n * logl((ld)nu_sb[b] / (ld)nu_b[b]);
    }
    q[t] = (double)(2 * acc);
  }
}
int64_t orc_cls_count_ge(const double* q, int64_t T, double q_obs) {
  int64_t c = 0;
  for (int64_t t = 0; t < T; ++t) c += (q[t] >= q_obs) ? 1 : 0;
  return c;
}
/* out = {CL_sb, CL_b, CL_s}; CL_s is NaN when no background toy reaches q_obs */
void orc_cls_from_counts(int64_t count_sb, int64_t T_sb, int64_t count_b, int64_t T_b, double* out) {
  out[0] = (double)count_sb / (double)T_sb;
  out[1] = (double)count_b / (double)T_b;
  out[2] = count_b > 0 ? out[0] / out[1] : NAN;
}

/* ------------------------------------------------------------------------------------------
 * Gaussian-smeared signal shape on the bin grid (PAPER.md:291-312:
 * "SM = GaussSmear1(bins_cx, sigma0); sigf_gpu = SM.Smear(sigf_i_gpu)", an FFT convolution whose kernel,
 * normalisation and edge treatment the paper does not state) -> DESIGN.md reading F3:
 *   out_b = sum_j in_j g_{b-j},  g_m = exp(-(m w)^2 / (2 sigma0^2)) / sum_{|m'| <= M} g_{m'},  |m| <= M,
 *   w = (hi - lo)/nbins,  M = ceil(8 sigma0 / w)  (relative tail 1e-14),  in_j = 0 outside the grid
 * (linear convolution; the paper's FFT is circular, which is the same thing for a peak far from the edges).
 * sigma0 <= 0 copies the input.  Plain double loop in long double.
 * ---------------------------------------------------------------------------------------- */
void orc_gauss_smear(const double* in, int nbins, double lo, double hi, double sigma0, double* out) {
  if (!(sigma0 > 0)) { for (int b = 0; b < nbins; ++b) out[b] = in[b]; return; }
  const ld w = ((ld)hi - lo) / nbins;
  const int M = (int)ceill(8 * (ld)sigma0 / w);
  std::vector<ld> g((size_t)(2 * M + 1));
  ld norm = 0;
  for (int m = -M; m <= M; ++m) { g[(size_t)(m + M)] = expl(-(m * w) * (m * w) / (2 * (ld)sigma0 * sigma0)); norm += g[(size_t)(m + M)]; }
  for (int b = 0; b < nbins; ++b) {
    ld acc = 0;
    for (int j = std::max(0, b - M); j <= std::min(nbins - 1, b + M); ++j) acc += (ld)in[j] * g[(size_t)(b - j + M)];
    out[b] = (double)(acc / norm);
  }
}
/* binned path with a GIVEN signal shape sig[nbins] >= 0 (e.g. the smeared one), normalised to unit sum as
 * PAPER.md:311-312 does; otherwise exactly orc_expected_hist / orc_binned_nll_scan (reading D15) */
int orc_expected_hist_shape(int nbins, double lo, double hi, const double* sig, double ns, double nb, double k, double* nu) {
  const ld w = ((ld)hi - lo) / nbins;
  ld ssum = 0, bsum = 0;
  std::vector<ld> bb((size_t)nbins);
  for (int b = 0; b < nbins; ++b) { ssum += sig[b]; bb[(size_t)b] = expl((ld)k * ((b + 0.5L) * w)); bsum += bb[(size_t)b]; }
  if (!(ssum > 0)) return 3;
  for (int b = 0; b < nbins; ++b) nu[b] = (double)((ld)ns * sig[b] / ssum + (ld)nb * bb[(size_t)b] / bsum);
  return 0;
}
int orc_binned_nll_scan_shape(const uint64_t* counts, int nbins, double lo, double hi, const double* sig,
                              const double* ns, const double* nb, const double* kk, int64_t npoints, double* nll) {
  const ld w = ((ld)hi - lo) / nbins;
  ld ssum = 0;
  for (int b = 0; b < nbins; ++b) ssum += sig[b];
  if (!(ssum > 0)) return 3;
  std::vector<ld> bb((size_t)nbins);
  std::vector<double> terms((size_t)nbins);
  for (int64_t q = 0; q < npoints; ++q) {
    ld bsum = 0;
    for (int b = 0; b < nbins; ++b) { bb[(size_t)b] = expl((ld)kk[q] * ((b + 0.5L) * w)); bsum += bb[(size_t)b]; }
    for (int b = 0; b < nbins; ++b) {
      const ld v = (ld)ns[q] * sig[b] / ssum + (ld)nb[q] * bb[(size_t)b] / bsum;
      terms[(size_t)b] = (double)(counts[b] ? v - (ld)counts[b] * logl(v) : v);
    }
    nll[q] = (double)pairwise(terms.data(), 0, nbins);
  }
  return 0;
}
/* signal shape at the bin centres, I(c_b - mu) relative to its value at the reference point (what the
 * paper's Ipatia kernel writes before the smearing); not normalised */
int orc_signal_shape(int nbins, double lo, double hi, const orc_params* shape, double* out) {
  const Shape s = make_shape(*shape);
  if (s.status) return s.status;
  const ld w = ((ld)hi - lo) / nbins;
  const ld ref = log_I(s, std::min(std::max((ld)0, (ld)lo - s.mu), (ld)hi - s.mu));
  for (int b = 0; b < nbins; ++b) out[b] = (double)expl(log_I(s, lo + (b + 0.5L) * w - s.mu) - ref);
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * Extended likelihood (reading D4: the paper's FCN works with yields, "fs", "fb" and
 * "the sum, including normalization terms"):
 *     -log L_ext(ns, nb, shape) = (ns + nb) - sum_i log( ns S(x_i) + nb B(x_i) )
 * written out as such (not through the fraction form); the f field of the parameter set is ignored.
 * ---------------------------------------------------------------------------------------- */
int orc_nll_extended(const double* x, int64_t n, const orc_params* pp, double ns, double nb, double lo_, double hi_,
                     double* out) {
  orc_params p = *pp;
  p.f = 0.5;                                  /* only the shape and k are used */
  const Shape s = make_shape(p);
  if (s.status) return s.status;
  if (!(ns >= 0) || !(nb >= 0) || !(ns + nb > 0)) return 1;
  const ld lo = lo_, hi = hi_;
  const Norm N = make_norm(s, p.k, lo, hi);
  std::vector<double> l((size_t)n);
  for (int64_t i = 0; i < n; ++i) {
    const ld S = expl(log_I(s, (ld)x[i] - s.mu) - N.logref) / N.NS;
    const ld B = expl((ld)p.k * ((ld)x[i] - lo)) / N.NB;
    l[i] = (double)logl((ld)ns * S + (ld)nb * B);
  }
  *out = (double)(((ld)ns + (ld)nb) - pairwise(l.data(), 0, n));
  return 0;
}
} /* extern "C" */
