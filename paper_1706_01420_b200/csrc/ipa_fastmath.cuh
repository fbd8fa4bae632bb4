// ipa_fastmath.cuh -- the streaming kernels' own fp64 sqrt / exp / log, written for the argument
// ranges of the hot path.  Polynomial coefficients live
// in __constant__ memory so that every DFMA takes its coefficient as a constant-bank operand (no
// register, no literal materialisation); the 33-entry log table is copied to shared memory by the
// kernels (per-lane index).  Marked __host__ __device__ so that tests/devmath_host.cu can run the
// same source on the GPU-less box (the rsqrt seed is emulated there with 20 good bits).
//
// Accuracy targets (checked in tests/test_abi_and_host_logic.py against mpmath):
//   ipa_fsqrt    relative error <= 2e-16 for normal positive arguments (seed truncated to 20 bits on the host)
//   ipa_fexp_neg relative error <= 3e-16 for a in [-90, 0]
//   ipa_flog     absolute error <= 2.5e-16 + 1.5e-16 |log u| for normal positive u
#pragma once
#include <math.h>
#include <stdint.h>
#include <string.h>
#include "ipa_fastmath_tables.inc"

#ifndef IPA_HD
#define IPA_HD __host__ __device__ __forceinline__
#endif

__constant__ double ipa_c_exp[IPA_EXP_DEG + 1] = IPA_EXP_COEFS;
__constant__ double ipa_c_log1p[IPA_LOG_DEG] = IPA_LOG1P_COEFS;
__constant__ double2 ipa_c_logtab[33] = IPA_LOG_TABLE;
// 16 KB table of the streaming kernels (layout: gen_fastmath_tables.py); the kernels copy it to shared memory
#define IPA_MATHTAB_DOUBLES 2048
__device__ const double ipa_d_mathtab[IPA_MATHTAB_DOUBLES] = IPA_MATHTAB_RAW;
static const double ipa_h_mathtab[IPA_MATHTAB_DOUBLES] = IPA_MATHTAB_RAW;
__constant__ double ipa_c_expq[4] = IPA_EXPQ_COEFS;
static const double ipa_h_expq[4] = IPA_EXPQ_COEFS;
__constant__ double ipa_c_expq2[3] = IPA_EXPQ2_COEFS;
static const double ipa_h_expq2[3] = IPA_EXPQ2_COEFS;
__device__ __align__(16) const long long ipa_d_chebT[IPA_CHEB_NC * IPA_CHEB_NC] = IPA_CHEB_TABLE;   // global memory (cp.async source)
static const long long ipa_h_chebT[IPA_CHEB_NC * IPA_CHEB_NC] = IPA_CHEB_TABLE;
__constant__ double ipa_c_gl16x[16] = IPA_GL16_X;
__constant__ double ipa_c_gl16w[16] = IPA_GL16_W;
// host copies (tests/devmath_host.cu only)
static const double ipa_h_gl16x[16] = IPA_GL16_X;
static const double ipa_h_gl16w[16] = IPA_GL16_W;
struct ipa_host_double2 { double x, y; };
static const double ipa_h_exp[IPA_EXP_DEG + 1] = IPA_EXP_COEFS;
static const double ipa_h_log1p[IPA_LOG_DEG] = IPA_LOG1P_COEFS;
static const ipa_host_double2 ipa_h_logtab[33] = IPA_LOG_TABLE;
#ifdef __CUDA_ARCH__
#define IPA_CEXP(j) ipa_c_exp[j]
#define IPA_CEXPQ(j) ipa_c_expq[j]
#define IPA_CEXPQ2(j) ipa_c_expq2[j]
#define IPA_CLOG(j) ipa_c_log1p[j]
#define IPA_GL16X(i) ipa_c_gl16x[i]
#define IPA_GL16W(i) ipa_c_gl16w[i]
#define IPA_CHEBT(j, k) ipa_d_chebT[(j) * IPA_CHEB_NC + (k)]
#else
#define IPA_CHEBT(j, k) ipa_h_chebT[(j) * IPA_CHEB_NC + (k)]
#define IPA_GL16X(i) ipa_h_gl16x[i]
#define IPA_GL16W(i) ipa_h_gl16w[i]
#define IPA_CEXP(j) ipa_h_exp[j]
#define IPA_CEXPQ(j) ipa_h_expq[j]
#define IPA_CEXPQ2(j) ipa_h_expq2[j]
#define IPA_CLOG(j) ipa_h_log1p[j]
#endif

// ---- bit access ---------------------------------------------------------------------------------
IPA_HD int ipa_hi(double v) {
#ifdef __CUDA_ARCH__
  return __double2hiint(v);
#else
  uint64_t b; memcpy(&b, &v, 8); return (int)(uint32_t)(b >> 32);
#endif
}
IPA_HD int ipa_lo(double v) {
#ifdef __CUDA_ARCH__
  return __double2loint(v);
#else
  uint64_t b; memcpy(&b, &v, 8); return (int)(uint32_t)b;
#endif
}
IPA_HD double ipa_mk(int hi, int lo) {
#ifdef __CUDA_ARCH__
  return __hiloint2double(hi, lo);
#else
  uint64_t b = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo; double v; memcpy(&v, &b, 8); return v;
#endif
}

// 1/sqrt(q) seed, about 20 good bits (MUFU.RSQ64H on the device)
IPA_HD double ipa_rsqrt_seed(double q) {
#ifdef __CUDA_ARCH__
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(q));
  return y;
#else
  const double y = 1.0 / sqrt(q);
  return ipa_mk(ipa_hi(y), 0);   // 20 mantissa bits, truncated: what the hardware seed guarantees
#endif
}

// sqrt(q), q > 0 normal: one third-order (Householder) step from the seed.  5 FP64 instructions.
//   e = 1 - q y^2,  sqrt(q) = q y (1 - e)^(-1/2) = q y (1 + e/2 + 3 e^2/8 + O(e^3))
IPA_HD double ipa_fsqrt(double q) {
  const double y = ipa_rsqrt_seed(q);
  const double g = q * y;
  const double e = fma(-g, y, 1.0);
  const double p = fma(0.375, e, 0.5) * e;
  return fma(g, p, g);
}

// sqrt(q) and 1/sqrt(q) from the same third-order step: 1/sqrt(q) = y (1 + p), one more FMA (the gradient kernel needs
// d/r beside r; a separate reciprocal of r cost a second seed and four FMAs)
IPA_HD double ipa_fsqrt_rsqrt(double q, double* rinv) {
  const double y = ipa_rsqrt_seed(q);
  const double g = q * y;
  const double e = fma(-g, y, 1.0);
  const double p = fma(0.375, e, 0.5) * e;
  *rinv = fma(y, p, y);
  return fma(g, p, g);
}

// 1/u, u > 0 normal: reciprocal seed (about 20 good bits, MUFU.RCP64H on the device) + ONE third-order step,
// y (1 + e + e^2), e = 1 - u y: the error e^3 is below 2^-58 (two Newton steps took one FMA more).
IPA_HD double ipa_frcp3(double u) {
#ifdef __CUDA_ARCH__
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(u));
#else
  double y = 1.0 / u;
  y = ipa_mk(ipa_hi(y), 0);
#endif
  const double e = fma(-u, y, 1.0);
  return fma(y, fma(e, e, e), y);
}

// e^a for a <= 0 (|a| is clamped to about 64 by the caller or here: results below 1e-27 are not
// distinguished).  n = round(a log2 e) by the 1.5 2^52 shift, Cody-Waite reduction with a 32-bit
// ln2_hi, degree-11 polynomial, scaling through the exponent field.  15 FP64 instructions.
IPA_HD double ipa_fexp_neg(double a) {
  const double SHIFT = 6755399441055744.0;
  const double t = fma(a, IPA_LOG2E, SHIFT);
  const int n = ipa_lo(t);
  const double nf = t - SHIFT;
  double r = fma(nf, -IPA_LN2_HI, a);
  r = fma(nf, -IPA_LN2_LO, r);
  double p = IPA_CEXP(IPA_EXP_DEG);
#pragma unroll
  for (int j = IPA_EXP_DEG - 1; j >= 0; --j) p = fma(p, r, IPA_CEXP(j));
  return ipa_mk(ipa_hi(p) + (n << 20), ipa_lo(p));
}

// -min(|D|, ~64) with the sign forced negative: integer work only
IPA_HD double ipa_neg_abs_clamped(double D) {
  int h = ipa_hi(D) & 0x7fffffff;
  h = h < 0x40500000 ? h : 0x40500000;
  return ipa_mk(h | (int)0x80000000, ipa_lo(D));
}
// max(D, 0) by the sign bit: integer work only (NaN with the sign clear passes through)
IPA_HD double ipa_relu_bits(double D) {
  const int m = ~(ipa_hi(D) >> 31);
  return ipa_mk(ipa_hi(D) & m, ipa_lo(D) & m);
}

// log(u), u > 0 normal.  tab[j] = {c_j, -log c_j}; u = 2^e m, j = top 5 mantissa bits,
// r = m c_j - 1 (|r| < 2^-6), log u = e ln2 + l_j + log1p(r).  11 FP64 instructions.
template <class Tab>
IPA_HD double ipa_flog(double u, const Tab* tab) {
  const int hu = ipa_hi(u);
  const int e = (hu >> 20) - 1023;
  const int j = (hu >> 15) & 31;
  const double m = ipa_mk((hu & 0x000fffff) | 0x3ff00000, ipa_lo(u));
  const double ef = ipa_mk(0x43300000, e ^ (int)0x80000000) - 4503601774854144.0;  // 2^52 + 2^31
  const double cj = tab[j].x, lj = tab[j].y;
  const double r = fma(m, cj, -1.0);
  double p = IPA_CLOG(IPA_LOG_DEG - 1);
#pragma unroll
  for (int k = IPA_LOG_DEG - 2; k >= 0; --k) p = fma(p, r, IPA_CLOG(k));
  return fma(ef, IPA_LN2, fma(p, r, lj));
}

// log(s) for s in [1, 2] (s = 1 + w, w in [0,1]): entry 32 of the table serves s == 2.  10 FP64.
template <class Tab>
IPA_HD double ipa_flog_1to2(double s, const Tab* tab) {
  unsigned j = (unsigned)((ipa_hi(s) - 0x3ff00000) >> 15);
  j = j < 32u ? j : 32u;   // s outside [1,2] (a NaN event) must not index past the table
  const double cj = tab[j].x, lj = tab[j].y;
  const double r = fma(s, cj, -1.0);
  double p = IPA_CLOG(IPA_LOG_DEG - 1);
#pragma unroll
  for (int k = IPA_LOG_DEG - 2; k >= 0; --k) p = fma(p, r, IPA_CLOG(k));
  return fma(p, r, lj);
}

// e^{-|D|}: -|D| enters through operand modifiers, the exponent shift is clamped instead of the argument.
// |D| < 1.4e9 (beyond that round(-|D| log2 e) leaves 32 bits).
IPA_HD double ipa_fexp_negabs(double D) {
  const double SHIFT = 6755399441055744.0;
  const double a = -fabs(D);
  const double t = fma(a, IPA_LOG2E, SHIFT);
  int n = ipa_lo(t);
  const double nf = t - SHIFT;
  double r = fma(nf, -IPA_LN2_HI, a);
  r = fma(nf, -IPA_LN2_LO, r);
  double p = IPA_CEXP(IPA_EXP_DEG);
#pragma unroll
  for (int j = IPA_EXP_DEG - 1; j >= 0; --j) p = fma(p, r, IPA_CEXP(j));
  n = n > -1000 ? n : -1000;
  return ipa_mk(ipa_hi(p) + (n << 20), ipa_lo(p));
}

// eb + log(1 + e^D) = eb + log(1 + e^{-|D|}) [+ D if D >= 0].  -|D| enters the exponential through operand
// modifiers, the exponent shift is clamped instead of the argument, and max(D,0) is a predicated add on
// the sign word: 2 integer instructions where the clamp / relu pair above needs 7.  |D| < 1.4e9.
template <class Tab>
IPA_HD double ipa_fsoftplus_add(double eb, double D, const Tab* tab) {
  const double SHIFT = 6755399441055744.0;
  const double a = -fabs(D);
  const double t = fma(a, IPA_LOG2E, SHIFT);
  int n = ipa_lo(t);
  const double nf = t - SHIFT;
  double r = fma(nf, -IPA_LN2_HI, a);
  r = fma(nf, -IPA_LN2_LO, r);
  double p = IPA_CEXP(IPA_EXP_DEG);
#pragma unroll
  for (int j = IPA_EXP_DEG - 1; j >= 0; --j) p = fma(p, r, IPA_CEXP(j));
  n = n > -1000 ? n : -1000;
  const double w = ipa_mk(ipa_hi(p) + (n << 20), ipa_lo(p));
  double l = eb + ipa_flog_1to2(1.0 + w, tab);
#ifdef __CUDA_ARCH__
  // predicated add on the sign word (the compiler would otherwise add and select: two more instructions)
  asm("{\n\t.reg .pred p;\n\tsetp.ge.s32 p, %2, 0;\n\t@p add.f64 %0, %0, %1;\n\t}" : "+d"(l) : "d"(D), "r"(ipa_hi(D)));
#else
  if (ipa_hi(D) >= 0) l += D;
#endif
  return l;
}

// log(1 + e^D) = max(D,0) + log(1 + e^{-|D|})
template <class Tab>
IPA_HD double ipa_fsoftplus(double D, const Tab* tab) {
  const double w = ipa_fexp_neg(ipa_neg_abs_clamped(D));
  return ipa_relu_bits(D) + ipa_flog_1to2(1.0 + w, tab);
}

// ================================================================================================
// Table-driven versions for the streaming kernels (round 2).  `mt` points to the 8 KB table
// (ipa_d_mathtab copied to shared memory; ipa_h_mathtab in the host build):
//   byte 0     {1/2, ln 2}                 log entry of s == 2
//   byte 16    2^(j/256), j = 0..255       e^a = 2^n 2^(j/256) e^r, |r| <= ln2/512, e^r = 1 + r q(r), q of degree 3
//   byte 4096  {c_j, -log c_j}, j = 0..255  log m = -log c_j + log1p(m c_j - 1), |m c_j - 1| < 2^-9,
//                                           log1p(r) = r (1 + r p(r)), p = -1/2 + r/3 - r^2/4 + r^3/5
// 9 FP64 instructions for the exponential (15 with the degree-11 polynomial), 6 for the logarithm on [1,2] (10),
// 8 for the general logarithm (12); each <= 3e-16 relative (exp) / 2.5e-16 + 1.5e-16 |log u| absolute (log),
// checked against mpmath on the host build.
// ================================================================================================
IPA_HD const double2* ipa_mt_at(const double* mt, unsigned byte_off) {
  return reinterpret_cast<const double2*>(reinterpret_cast<const char*>(mt) + byte_off);
}
IPA_HD double ipa_mt_d(const double* mt, unsigned byte_off) {
  return *reinterpret_cast<const double*>(reinterpret_cast<const char*>(mt) + byte_off);
}

// r (1 + r p(r)) + l  with p = -1/2 + r/3 - r^2/4 + r^3/5: log1p(r) + l for |r| < 2^-9.  5 FP64.
IPA_HD double ipa_log1p_small_add(double r, double l) {
  double p = fma(0.2, r, -0.25);
  p = fma(p, r, 0.33333333333333331);
  p = fma(p, r, -0.5);
  const double q = fma(p, r, 1.0);
  return fma(r, q, l);
}

// log(s) for s in [1, 2] (s = 1 + w, w in [0,1]).  Index = lowest exponent bit (1 on [1,2), 0 at s == 2) and the top
// 8 mantissa bits: byte offset 0 serves s == 2, 4096 + 16 j the rest; a NaN stays in bounds.  6 FP64, 3 integer.
IPA_HD double ipa_flog12_t(double s, const double* mt) {
  const unsigned off = ((unsigned)ipa_hi(s) >> 8) & 0x1ff0u;
  const double2 e = *ipa_mt_at(mt, off);
  return ipa_log1p_small_add(fma(s, e.x, -1.0), e.y);
}

// log(u), u > 0 normal: u = 2^e m, table entry of the top 8 mantissa bits.  8 FP64.
IPA_HD double ipa_flog_t(double u, const double* mt) {
  const int hu = ipa_hi(u);
  const int e = (hu >> 20) - 1023;
  const unsigned off = 4096u + (((unsigned)hu >> 8) & 0xff0u);
  const double ef = ipa_mk(0x43300000, e ^ (int)0x80000000) - 4503601774854144.0;  // 2^52 + 2^31
  const double2 t = *ipa_mt_at(mt, off);
  // m c_j - 1 with m = u 2^-e: the power of two goes into c_j's exponent field (exact, same bits as building m;
  // one integer instruction fewer; u < 2^1000)
  const double cs = ipa_mk(ipa_hi(t.x) - (hu & 0x7ff00000) + 0x3ff00000, ipa_lo(t.x));
  return fma(ef, IPA_LN2, ipa_log1p_small_add(fma(u, cs, -1.0), t.y));
}

// e^{-|D|}, any D with |D| < 5e6 (beyond that the integer part of -|D| 256/ln2 leaves 32 bits; the largest |Delta|
// the kernels produce on purpose is the f == 0 sentinel, 1e4).  9 FP64.
IPA_HD double ipa_fexp_negabs_t(double D, const double* mt) {
  const double SHIFT = 6755399441055744.0;
  const double a = -fabs(D);
  const double t = fma(a, IPA_LOG2E_256, SHIFT);
  int m = ipa_lo(t);                                    // round(a 256 / ln 2) = 256 n + j
  const double nf = t - SHIFT;
  double r = fma(nf, -IPA_LN2_256_HI, a);
  r = fma(nf, -IPA_LN2_256_LO, r);
  const double T = ipa_mt_d(mt, 16u + (((unsigned)m & 255u) << 3));
  double q = fma(IPA_CEXPQ(3), r, IPA_CEXPQ(2));
  q = fma(q, r, IPA_CEXPQ(1));
  q = fma(q, r, IPA_CEXPQ(0));
  const double w = fma(T * r, q, T);
  m = m > -256000 ? m : -256000;                        // 2^n stays a normal number (w < 1e-300 is not distinguished)
#ifdef __CUDA_ARCH__
  int hw;                                               // hi(w) + (m >> 8) 2^20 = hi(w) + (m & ~255) 4096: one mask, one multiply-add
  asm("mad.lo.s32 %0, %1, 4096, %2;" : "=r"(hw) : "r"(m & ~255), "r"(ipa_hi(w)));
  return ipa_mk(hw, ipa_lo(w));
#else
  return ipa_mk(ipa_hi(w) + ((m >> 8) << 20), ipa_lo(w));
#endif
}

// The softplus' own e^{-|D|}: 2^(j/1024) from the second half of the table (byte 8192), so that |r| <= ln2/2048 and
// e^r = 1 + r q(r) needs a q of degree 2 only (1.4e-16 relative).  The reduction r = a - m ln2/1024 takes ONE step with
// ln2/1024 rounded to fp64: the product is exact inside the FMA, so the only error is m times the representation error of
// the constant, < |a| 8e-17 relative in the result, i.e. < |a| e^{-|a|} 8e-17 < 3e-17 absolute in the softplus.
// The result enters the softplus as log(1 + w): its relative error counts times w / (1 + w) <= 1/2.  7 FP64.
// |D| < 1.4e6 (m = round(-|D| 1024 / ln 2) must fit 32 bits).
IPA_HD double ipa_fexp_negabs_sp(double D, const double* mt) {
  const double SHIFT = 6755399441055744.0;
  const double a = -fabs(D);
  const double t = fma(a, IPA_LOG2E_1024, SHIFT);
  int m = ipa_lo(t);                                    // round(a 1024 / ln 2) = 1024 n + j
  const double nf = t - SHIFT;
  const double r = fma(nf, -IPA_LN2_1024, a);
  const double T = ipa_mt_d(mt, 8192u + (((unsigned)m & 1023u) << 3));
  double q = fma(IPA_CEXPQ2(2), r, IPA_CEXPQ2(1));
  q = fma(q, r, IPA_CEXPQ2(0));
  const double w = fma(T * r, q, T);
  m = m > -1024000 ? m : -1024000;                      // 2^n stays a normal number
#ifdef __CUDA_ARCH__
  int hw;                                               // hi(w) + (m >> 10) 2^20 = hi(w) + (m & ~1023) 1024
  asm("mad.lo.s32 %0, %1, 1024, %2;" : "=r"(hw) : "r"(m & ~1023), "r"(ipa_hi(w)));
  return ipa_mk(hw, ipa_lo(w));
#else
  return ipa_mk(ipa_hi(w) + ((m >> 10) << 20), ipa_lo(w));
#endif
}

// eb + log(1 + e^D) = eb + log(1 + e^{-|D|}) + max(D, 0), and max(D, 0) = (D + |D|) / 2 with D + |D| EXACT (0 or 2 D): the
// final FMA rounds once, like the addition of D it replaces -- same bits, no compare and no select (ptxas turned a
// predicated add into an unconditional one plus two FSEL: 4 issue slots against 2 FP64 instructions here).
// (Folding D/2 + |D|/2 into the two FMAs of the sum instead cancels for D << 0: 3.5e-15 at D = -52 -- rejected.)
IPA_HD double ipa_fsoftplus_add_t(double eb, double D, const double* mt) {
  const double w = ipa_fexp_negabs_sp(D, mt);
  return fma(0.5, D + fabs(D), eb + ipa_flog12_t(1.0 + w, mt));
}
