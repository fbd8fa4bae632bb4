// ipa_math.cuh -- scalar fp64 building blocks of the CUDA path (device code; the functions are
// also marked __host__ so that tests/devmath_host.cu can run the very same source on the CPU box,
// which has no GPU.  The product never calls them on the host).
//
// Nothing here is shared with oracle/: the Bessel function below is the trapezoid rule on the
// integral representation (the oracle uses Temme's series and Miller's recurrence in long double).
#pragma once
#include <math.h>
#include <stdint.h>

#define IPA_HD __host__ __device__ __forceinline__
#include "ipa_fastmath.cuh"

// ------------------------------------------------------------------------------------------------
// Scaled modified Bessel function of the second kind, real order:
//     e^x K_nu(x) = int_0^inf exp(-2 x sinh^2(t/2)) cosh(nu t) dt          (A&S 9.6.24, times e^x)
// by the trapezoid rule.  The integrand is entire and decays double-exponentially, so the rule
// converges geometrically: the error is governed by the Fourier transform of the integrand at
// 2 pi / h, i.e. by |K_{nu + 2 pi i/h}(x)| ~ exp(-pi^2/h) (x small) and exp(-2 pi^2/(h^2 x))
// (x large, Gaussian peak of width (x^2+nu^2)^(-1/4)).  h = min(0.2, 0.6 (x^2+nu^2)^(-1/4)) keeps
// both below 1e-21.  All terms are positive: no cancellation.
// ------------------------------------------------------------------------------------------------
IPA_HD double ipa_trap_step(double nu, double x) {
  return fmin(0.2, 0.6 / sqrt(sqrt(x * x + nu * nu)));
}

// term j >= 1 of the rule for order nu >= 0 (term 0 is 1 and carries the weight 1/2)
IPA_HD double ipa_trap_term(double nu, double x, double h, int j) {
  const double t = (double)j * h;
  const double s = sinh(0.5 * t);
  const double a = 2.0 * x * s * s;
  const double e = nu * t;
  return 0.5 * (exp(e - a) + exp(-e - a));
}

// serial evaluation (prologue fall-backs, direct mode, tests)
IPA_HD double ipa_besselk_scaled(double nu, double x) {
  nu = fabs(nu);
  const double h = ipa_trap_step(nu, x);
  double sum = 0.5, prev = 1.0;
  for (int j = 1; j < 8192; ++j) {
    const double term = ipa_trap_term(nu, x, h, j);
    sum += term;
    if (term <= prev && term < 1e-18 * sum) break;
    prev = term;
  }
  return h * sum;
}

// ------------------------------------------------------------------------------------------------
// Gauss-Legendre node i (0..n-1) and weight on [-1,1]: Newton on P_n (A&S 25.4.29-30).
// ------------------------------------------------------------------------------------------------
IPA_HD void ipa_gauss_legendre(int n, int i, double* node, double* weight) {
  double t = cos(3.14159265358979323846 * ((double)i + 0.75) / ((double)n + 0.5));
  double dp = 1.0;
  for (int it = 0; it < 8; ++it) {
    double p0 = 1.0, p1 = t;
    for (int k = 2; k <= n; ++k) {
      const double p2 = ((2.0 * k - 1.0) * t * p1 - (k - 1.0) * p0) / (double)k;
      p0 = p1;
      p1 = p2;
    }
    dp = (double)n * (t * p1 - p0) / (t * t - 1.0);
    t -= p1 / dp;
  }
  {
    double p0 = 1.0, p1 = t;
    for (int k = 2; k <= n; ++k) {
      const double p2 = ((2.0 * k - 1.0) * t * p1 - (k - 1.0) * p0) / (double)k;
      p0 = p1;
      p1 = p2;
    }
    dp = (double)n * (t * p1 - p0) / (t * t - 1.0);
  }
  *node = t;
  *weight = 2.0 / ((1.0 - t * t) * dp * dp);
}

// (u^(1-n) - 1)/(1-n), -> log u as n -> 1: the antiderivative factor of the power-law tails
IPA_HD double ipa_powint(double u, double n) {
  const double e = 1.0 - n;
  const double lu = log(u);
  const double y = e * lu;
  if (fabs(y) < 1e-9) return lu * (1.0 + 0.5 * y);
  return expm1(y) / e;
}

// F(ul) - F(ur), F(u) = (u^(1-n) - 1)/(1-n) (log u at n = 1), formed WITHOUT the cancellation of two nearly equal
// terms (range inside one tail, large n):  = ur^(1-n) expm1((1-n) log(ul/ur)) / (1-n).  Returned as the pair
// (value without the factor ur^(1-n), *logscale = (1-n) log ur) so that the caller can fold the scale into its
// log-reference before exponentiating.
IPA_HD double ipa_powint_diff(double ul, double ur, double n, double* logscale) {
  const double e = 1.0 - n;
  const double lq = log(ul / ur);
  const double y = e * lq;
  *logscale = e * log(ur);
  if (fabs(y) < 1e-9) return lq * (1.0 + 0.5 * y);
  return expm1(y) / e;
}

// error-free transformations for the double-double accumulation in the basis conversion
IPA_HD void ipa_two_sum(double a, double b, double* s, double* e) {
  const double t = a + b;
  const double bb = t - a;
  *e = (a - (t - bb)) + (b - bb);
  *s = t;
}
IPA_HD void ipa_two_prod(double a, double b, double* p, double* e) {
  const double t = a * b;
  *e = fma(a, b, -t);
  *p = t;
}

// ------------------------------------------------------------------------------------------------
// Counter-based generator Philox-4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), written from the
// published round function; reading D13 fixes key/counter layout and the uniform mapping.
// ------------------------------------------------------------------------------------------------
struct IpaU4 { uint32_t w0, w1, w2, w3; };

IPA_HD uint32_t ipa_mulhi32(uint32_t a, uint32_t b) {
#ifdef __CUDA_ARCH__
  return __umulhi(a, b);
#else
  return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32);
#endif
}

IPA_HD IpaU4 ipa_philox(uint64_t seed, uint64_t slot, uint32_t attempt, uint32_t stream) {
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  uint32_t c0 = (uint32_t)slot, c1 = (uint32_t)(slot >> 32), c2 = attempt, c3 = stream;
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t h0 = ipa_mulhi32(M0, c0), l0 = M0 * c0;
    const uint32_t h1 = ipa_mulhi32(M1, c2), l1 = M1 * c2;
    const uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
    c0 = n0; c1 = l1; c2 = n2; c3 = l0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  IpaU4 o; o.w0 = c0; o.w1 = c1; o.w2 = c2; o.w3 = c3;
  return o;
}

// two uniforms in (0,1): u = ((w >> 5) 2^26 + (w' >> 6) + 1/2) 2^-53
IPA_HD void ipa_uniforms2(uint64_t seed, uint64_t slot, uint32_t attempt, uint32_t stream, double* u0, double* u1) {
  const IpaU4 r = ipa_philox(seed, slot, attempt, stream);
  const double s = 1.0 / 9007199254740992.0;
  *u0 = ((double)(r.w0 >> 5) * 67108864.0 + (double)(r.w1 >> 6) + 0.5) * s;
  *u1 = ((double)(r.w2 >> 5) * 67108864.0 + (double)(r.w3 >> 6) + 0.5) * s;
}

enum { IPA_STREAM_COMP = 0, IPA_STREAM_SIG = 1, IPA_STREAM_BKG = 2, IPA_STREAM_YIELD = 3, IPA_STREAM_BIN = 4 };

// Poisson(mean) (reading D14): sequential-search inversion below 10, Hoermann's transformed
// rejection with squeeze (PTRS, Insurance: Math. & Econ. 12 (1993) 39-45) above.
// The constants of a mean (IpaPoissonConsts) are separate from the draw, so that a caller with many draws of one mean
// (a bin over many toys) forms them once; ipa_poisson is the two in a row -- same expressions, same values.
struct IpaPoissonConsts { double mean, p0, b, a, vr, lmean, linva; int kind; };   // kind: 0 zero, 1 inversion, 2 PTRS
IPA_HD IpaPoissonConsts ipa_poisson_consts(double mean) {
  IpaPoissonConsts c;
  c.mean = mean;
  c.p0 = c.b = c.a = c.vr = c.lmean = c.linva = 0.0;
  if (!(mean > 0.0)) { c.kind = 0; return c; }
  if (mean < 10.0) { c.kind = 1; c.p0 = exp(-mean); return c; }
  c.kind = 2;
  const double smu = sqrt(mean);
  c.b = 0.931 + 2.53 * smu;
  c.a = -0.059 + 0.02483 * c.b;
  const double inv_alpha = 1.1239 + 1.1328 / (c.b - 3.4);
  c.vr = 0.9277 - 3.6224 / (c.b - 2.0);
  c.lmean = log(mean);
  c.linva = log(inv_alpha);
  return c;
}
IPA_HD int64_t ipa_poisson_draw(const IpaPoissonConsts& c, uint64_t seed, uint64_t slot, uint32_t stream) {
  if (c.kind == 0) return 0;
  if (c.kind == 1) {
    double u, v;
    ipa_uniforms2(seed, slot, 0u, stream, &u, &v);
    int64_t k = 0;
    double p = c.p0, F = p;
    while (u > F && k < 1000) {
      ++k;
      p *= c.mean / (double)k;
      F += p;
    }
    return k;
  }
  const double mean = c.mean, b = c.b, a = c.a, vr = c.vr, lmean = c.lmean;
  for (uint32_t attempt = 0;; ++attempt) {
    double U, V;
    ipa_uniforms2(seed, slot, attempt, stream, &U, &V);
    U -= 0.5;
    const double us = 0.5 - fabs(U);
    const double kf = floor((2.0 * a / us + b) * U + mean + 0.43);
    if (us >= 0.07 && V <= vr) return (int64_t)kf;
    if (kf < 0.0 || (us < 0.013 && V > us)) continue;
    if (log(V) + c.linva - log(a / (us * us) + b) <= -mean + kf * lmean - lgamma(kf + 1.0)) return (int64_t)kf;
    if (attempt > 1000000u) return (int64_t)kf;
  }
}
IPA_HD int64_t ipa_poisson(uint64_t seed, uint64_t slot, uint32_t stream, double mean) {
  return ipa_poisson_draw(ipa_poisson_consts(mean), seed, slot, stream);
}
