// Branch-free FP64 elementary functions for the hot loops (sm_100a).
//
// The CUDA math library versions inline ~45 instructions per exp (16 FP64 operations, 22 UMOVs that materialise
// the 64-bit polynomial constants, a range check and a branch to a special-case tail) and call out-of-line slow
// paths for reciprocals and square roots of extreme operands.  In k_transfer these branches and the code volume
// cost more than the arithmetic (ncu: stall_no_instruction / branch_resolving grow with occupancy,
// profiles/r1_notes.md).  The versions below
//   * take their polynomial coefficients from __constant__ memory (LDCU.128 loads two per instruction),
//   * have no branches and no special-case tails,
//   * are accurate to <= 2 ulp on the stated domain (checked against mpmath in tests/test_gpu_stages.py through
//     ipole_eval_math), which is far inside the parity budget,
// and state the domain they are valid on.  Outside it the callers use the library function.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include "math_tables.inc"

namespace ipole {

// branch hints: the fallbacks for operands outside the fast paths are placed out of the hot instruction stream
#define IP_LIKELY(x) __builtin_expect(!!(x), 1)
#define IP_UNLIKELY(x) __builtin_expect(!!(x), 0)

__device__ __forceinline__ double mk_double(int hi, int lo) { return __hiloint2double(hi, lo); }

// 256-bit global accesses (sm_100: LDG/STG.E.ENL2.256), 32-byte aligned addresses
__device__ __forceinline__ void ld_global_v4(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p) : "memory");
}
__device__ __forceinline__ void ld_global_nc_v4(const double* p, double& a, double& b, double& c, double& d) {
  asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
__device__ __forceinline__ void st_global_v4(double* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// 1/x for normal x (1e-290 < |x| < 1e290): MUFU.RCP64H seed (>= 20 bits), one cubic and one quadratic Newton step
__device__ __forceinline__ double ip_rcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  e = fma(e, e, e);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}

// a/b with one residual correction (<= 1 ulp), b normal
__device__ __forceinline__ double ip_div(double a, double b) {
  const double y = ip_rcp(b);
  const double q = a * y;
  return fma(fma(-b, q, a), y, q);
}

// 1/sqrt(x) for normal x > 0: MUFU.RSQ64H seed, cubic then quadratic step
__device__ __forceinline__ double ip_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x * y, y, 1.0);                  // 1 - x y^2
  y = fma(y, e * fma(0.375, e, 0.5), y);           // y (1 + e/2 + 3 e^2/8)
  e = fma(-x * y, y, 1.0);
  return fma(0.5 * y, e, y);
}

// sqrt(x) for normal x > 0 (x = 0 must be handled by the caller)
__device__ __forceinline__ double ip_sqrt(double x) {
  const double y = ip_rsqrt(x);
  const double s = x * y;
  return fma(fma(-s, s, x), 0.5 * y, s);
}

// exp(r) - 1 = r + r^2 PE(r) on |r| <= ln2/2
__device__ __forceinline__ double expm1_poly(double r) {
  double p = c_pe[IPOLE_PE_N - 1];
#pragma unroll
  for (int j = IPOLE_PE_N - 2; j >= 0; --j) p = fma(p, r, c_pe[j]);
  return fma(r * r, p, r);
}

// x = k ln2 + r, k integer (returned as a double and as an int), |r| <= ln2/2 (+ rounding)
__device__ __forceinline__ double reduce_ln2(double x, int& ki) {
  const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);  // 1.5 * 2^52: round to nearest integer
  ki = __double2loint(t);
  const double k = t - 6755399441055744.0;
  double r = fma(k, -6.93147180369123816490e-01, x);   // ln2 hi (32 trailing zero bits: k * hi is exact)
  return fma(k, -1.90821492927058770002e-10, r);       // ln2 lo
}

// exp(x) for x <= 709 (any x below, including -inf; NaN gives 0).  Gradual underflow is kept: the scaling by 2^k is
// applied in two normal factors.
__device__ __forceinline__ double ip_exp(double x) {
  x = fmax(x, -746.0);
  int ki;
  const double r = reduce_ln2(x, ki);
  const double p = 1.0 + expm1_poly(r);
  const int k1 = ki >> 1, k2 = ki - k1;
  return (p * mk_double((k1 + 1023) << 20, 0)) * mk_double((k2 + 1023) << 20, 0);
}

// exp(x) - 1 for -inf <= x <= 709; relative accuracy kept for small |x| (k = 0 returns the polynomial itself)
__device__ __forceinline__ double ip_expm1(double x) {
  x = fmax(x, -60.0);                                   // exp(-60) - 1 rounds to -1
  int ki;
  const double r = reduce_ln2(x, ki);
  const double q = expm1_poly(r);
  const double s = mk_double((ki + 1023) << 20, 0);     // 2^k, k in [-87, 1023]
  return fma(s, q, s - 1.0);
}

// ln(x) for normal x > 0:  x = 2^e m, m in [sqrt(1/2), sqrt 2),  ln m = 2 f + f^3 PL(f^2),  f = (m - 1)/(m + 1)
__device__ __forceinline__ double ip_log(double x) {
  int hi = __double2hiint(x);
  const int lo = __double2loint(x);
  int e = (hi >> 20) - 1023;
  hi = (hi & 0x000fffff) | 0x3ff00000;                  // m in [1, 2)
  const int up = (hi >= 0x3ff6a09f) ? 1 : 0;            // m >= sqrt 2 (to 20 bits): halve it
  hi -= up << 20;
  e += up;
  const double m = mk_double(hi, lo);
  const double f = (m - 1.0) * ip_rcp(m + 1.0);
  const double w = f * f;
  double p = c_pl[IPOLE_PL_N - 1];
#pragma unroll
  for (int j = IPOLE_PL_N - 2; j >= 0; --j) p = fma(p, w, c_pl[j]);
  const double lm = fma(f * w, p, 2.0 * f);
  const double de = (double)e;
  return fma(de, 6.93147180369123816490e-01, fma(de, 1.90821492927058770002e-10, lm));
}

// sin and cos for |x| <= 1e5 (three-term Cody-Waite reduction by pi/2, then polynomials on |r| <= pi/4)
__device__ __forceinline__ void ip_sincos(double x, double* sp, double* cp) {
  const double t = fma(x, 6.36619772367581382433e-01, 6755399441055744.0);
  const int q = __double2loint(t);
  const double k = t - 6755399441055744.0;
  double r = fma(k, -1.57079632679489655800e+00, x);
  r = fma(k, -6.12323399573676603587e-17, r);
  r = fma(k, 1.49738490485916983293e-33, r);            // pi/2 = c1 + c2 - c3 to ~160 bits
  const double w = r * r;
  double ps = c_ps[IPOLE_PS_N - 1], pc = c_pc[IPOLE_PC_N - 1];
#pragma unroll
  for (int j = IPOLE_PS_N - 2; j >= 0; --j) ps = fma(ps, w, c_ps[j]);
#pragma unroll
  for (int j = IPOLE_PC_N - 2; j >= 0; --j) pc = fma(pc, w, c_pc[j]);
  const double s = fma(r * w, ps, r);
  const double c = fma(w * w, pc, fma(-0.5, w, 1.0));
  const double a = (q & 1) ? c : s, b = (q & 1) ? s : c;
  *sp = (q & 2) ? -a : a;
  *cp = ((q + 1) & 2) ? -b : b;
}

// any finite x: the library routine (Payne-Hanek) beyond the Cody-Waite range; the branch is never taken on the
// workloads of DESIGN.md section 5 (rotation angles per step are small)
__device__ __forceinline__ void ip_sincos_any(double x, double* sp, double* cp) {
  if (IP_LIKELY(fabs(x) <= 1e5)) ip_sincos(x, sp, cp);
  else sincos(x, sp, cp);
}
__device__ __forceinline__ double ip_cos_any(double x) {
  double s, c;
  ip_sincos_any(x, &s, &c);
  return c;
}

}  // namespace ipole
