// Thermal synchrotron emission / absorption / Faraday coefficients in the plasma frame (cgs) and the
// modified Bessel functions they need.  DESIGN.md R-7 ("synchrotron emission, synchrotron
// absorption and Faraday effects such as Faraday rotation and Faraday conversion"; PAPER.md:35 evaluated at
// every step).  In the tetrad with e_(2) along the projected field, j_U = alpha_U = rho_U = 0.
//
// K_n(z): power series (Abramowitz & Stegun 9.6.11-13) for z <= 2, Chebyshev series of e^z sqrt(z) K_n(z) in
// 4/z - 1 for z > 2 (bessel_tables.inc, written by gen_bessel_tables.py); K_2 = K_0 + (2/z) K_1.
#pragma once
#include "geom.cuh"
#include "bessel_tables.inc"
#include "pw_tables.inc"

namespace ipole {

// CGS constants, R-1 (literals held by this file only)
#define IP_EE   4.80320680e-10
#define IP_CL   2.99792458e10
#define IP_ME   9.1093826e-28
#define IP_MP   1.67262171e-24
#define IP_HPL  6.6260693e-27
#define IP_KBOL 1.3806505e-16
#define IP_GNEWT 6.6742e-8
#define IP_MSUN 1.989e33
#define IP_PC   3.085678e18

// e^z K_0(z), e^z K_1(z)
__device__ __forceinline__ void bessel_k01_scaled(double z, double& k0, double& k1) {
  if (z <= 2.0) {
    // t = z^2/4;  I0 = sum t^k/(k!)^2, I1 = (z/2) sum t^k/(k!(k+1)!)
    // K0 = -(ln(z/2)+gamma) I0 + sum_{k>=1} H_k t^k/(k!)^2
    // K1 = 1/z + ln(z/2) I1 - (z/4) sum_{k>=0} (psi(k+1)+psi(k+2)) t^k/(k!(k+1)!)
    const double EUL = 0.57721566490153286061;
    const double t = 0.25 * z * z;
    const double lg = ip_log(0.5 * z);
    double term0 = 1.0;   // t^k/(k!)^2
    double term1 = 1.0;   // t^k/(k!(k+1)!)
    double Hk = 0.0;      // harmonic number H_k
    double i0 = 1.0, s0 = 0.0;
    double i1 = 1.0, s1 = 1.0 - 2.0 * EUL;  // psi(1)+psi(2) = 1 - 2 gamma
#pragma unroll
    for (int k = 1; k <= 13; ++k) {
      const double ik = 1.0 / (double)k;
      Hk += ik;
      term0 *= t * ik * ik;
      term1 *= t * ik / (double)(k + 1);
      i0 += term0;
      s0 += term0 * Hk;
      i1 += term1;
      s1 += term1 * (2.0 * Hk + 1.0 / (double)(k + 1) - 2.0 * EUL);  // psi(k+1)+psi(k+2)
    }
    const double ez = ip_exp(z);
    k0 = ez * (-(lg + EUL) * i0 + s0);
    k1 = ez * (1.0 / z + lg * (0.5 * z) * i1 - 0.25 * z * s1);
  } else {
    const double xi = 4.0 / z - 1.0, x2 = 2.0 * xi;
    double b1 = 0.0, b2 = 0.0, d1 = 0.0, d2 = 0.0;  // Clenshaw
#pragma unroll
    for (int j = IPOLE_BESSEL_K0_NC - 1; j >= 1; --j) {
      const double b0 = c_bessel_k0[j] + x2 * b1 - b2; b2 = b1; b1 = b0;
    }
#pragma unroll
    for (int j = IPOLE_BESSEL_K1_NC - 1; j >= 1; --j) {
      const double d0 = c_bessel_k1[j] + x2 * d1 - d2; d2 = d1; d1 = d0;
    }
    const double rs = rsqrt(z);
    k0 = (c_bessel_k0[0] + xi * b1 - b2) * rs;
    k1 = (c_bessel_k1[0] + xi * d1 - d2) * rs;
  }
}

// Piecewise polynomial tables (pw_tables.inc, written by gen_pw_tables.py): every binary octave of x is cut into
// IPOLE_PW_NP = 8 pieces; on piece q the function is a polynomial in v = 16 m - (17 + 2 q), m = x 2^-e in [1, 2).
// Returns false when x is outside [2^e0, 2^e1) (or not a positive normal number): the caller evaluates the
// defining formula instead.
__device__ __forceinline__ bool pw_locate(double x, int e0, int e1, int& piece, double& v) {
  const int hi = __double2hiint(x);
  const int e = (hi >> 20) - 1023;
  const int q = (hi >> 17) & 7;
  piece = (e - e0) * IPOLE_PW_NP + q;
  const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(x));
  v = fma(m, 2.0 * IPOLE_PW_NP, -(double)(2 * IPOLE_PW_NP + 1 + 2 * q));
  return e >= e0 && e < e1;
}

__device__ __forceinline__ void bessel_ratios_series(double z, double Th, double& r0, double& r1);

// K_0/K_2 and K_1/K_2 at z = 1/Th
__device__ __forceinline__ void bessel_ratios(double z, double Th, double& r0, double& r1) {
  int piece; double v;
  if (IP_LIKELY(pw_locate(Th, IPOLE_PW_BESSEL_E0, IPOLE_PW_BESSEL_E1, piece, v))) {
    const double2* t = reinterpret_cast<const double2*>(&g_pw_bessel[piece][0][0]);
    double2 c = __ldg(t + IPOLE_PW_NC - 1);
    double a = c.x, b = c.y;
#pragma unroll
    for (int j = IPOLE_PW_NC - 2; j >= 0; --j) {
      c = __ldg(t + j);
      a = fma(a, v, c.x);
      b = fma(b, v, c.y);
    }
    r0 = a; r1 = b;
  } else {
    bessel_ratios_series(z, Th, r0, r1);
  }
}

// f(X) of the Faraday-conversion fit (R-7)
__device__ __forceinline__ double faraday_fX(double X) {
  int piece; double v;
  if (IP_LIKELY(pw_locate(X, IPOLE_PW_FX_E0, IPOLE_PW_FX_E1, piece, v))) {
    const double2* t = reinterpret_cast<const double2*>(&g_pw_fx[piece][0][0]);
    double p = 0.0;
#pragma unroll
    for (int j = IPOLE_PW_NC / 2 - 1; j >= 0; --j) {
      const double2 c = __ldg(t + j);
      p = fma(p, v, c.y);
      p = fma(p, v, c.x);
    }
    return p;
  }
  const double lX = ip_log(X);
  return 2.011 * ip_exp(-(1.0 / 4.7) * ip_exp(1.035 * lX)) - ip_cos_any(0.5 * X) * ip_exp(-(1.0 / 2.73) * ip_exp(1.2 * lX))
         - 0.011 * ip_exp(-(1.0 / 47.2) * X);
}

static_assert(IPOLE_PW_NC % 2 == 0, "faraday_fX reads its coefficients two at a time");

static_assert(IPOLE_BESSEL_K0_NC == IPOLE_BESSEL_K1_NC, "the two Chebyshev series are evaluated interleaved");

struct Coeff { double jI, jQ, jV, aI, aQ, aV, rQ, rV; };

__device__ __forceinline__ double finite_or_zero(double v) { return isfinite(v) ? v : 0.0; }

// K_0(z)/K_2(z) and K_1(z)/K_2(z): the e^z scaling of bessel_k01_scaled cancels in the ratios, so the series branch
// skips it here.
__device__ __forceinline__ void bessel_ratios_series(double z, double Th, double& r0, double& r1) {
  double k0, k1;
  if (z <= 2.0) {
    const double EUL = 0.57721566490153286061;
    const double t = 0.25 * z * z;
    const double lg = ip_log(0.5 * z);
    double term0 = 1.0, term1 = 1.0, Hk = 0.0;
    double i0 = 1.0, s0 = 0.0, i1 = 1.0, s1 = 1.0 - 2.0 * EUL;
#pragma unroll
    for (int k = 1; k <= 13; ++k) {
      const double ik = 1.0 / (double)k, ik1 = 1.0 / (double)(k + 1);  // folded at compile time
      Hk += ik;
      term0 *= t * (ik * ik);
      term1 *= t * (ik * ik1);
      i0 += term0;
      s0 = fma(term0, Hk, s0);
      i1 += term1;
      s1 = fma(term1, 2.0 * Hk + ik1 - 2.0 * EUL, s1);
    }
    k0 = s0 - (lg + EUL) * i0;
    k1 = Th + (0.5 * z) * (lg * i1 - 0.5 * s1);
  } else {
    const double xi = 4.0 * Th - 1.0, x2 = 2.0 * xi;
    double b1 = 0.0, b2 = 0.0, d1 = 0.0, d2 = 0.0;  // Clenshaw, the two series interleaved
#pragma unroll
    for (int j = IPOLE_BESSEL_K0_NC - 1; j >= 1; --j) {
      const double b0 = fma(x2, b1, c_bessel_k0[j] - b2); b2 = b1; b1 = b0;
      const double d0 = fma(x2, d1, c_bessel_k1[j] - d2); d2 = d1; d1 = d0;
    }
    k0 = fma(xi, b1, c_bessel_k0[0] - b2);   // common factor rsqrt(z) cancels in the ratios
    k1 = fma(xi, d1, c_bessel_k1[0] - d2);
  }
  const double ik2 = ip_rcp(fma(2.0 * Th, k1, k0));
  r0 = k0 * ik2;
  r1 = k1 * ik2;
}

// constants of the fits, folded at compile time (R-7)
#define IP_SQRT3 1.7320508075688772935
#define IP_C_NUC  (3.0 * IP_EE / (4.0 * M_PI * IP_ME * IP_CL))                 /* nu_c = C B sinT Th^2       */
#define IP_C_PRE  (IP_EE * IP_EE / (2.0 * IP_SQRT3 * IP_CL))                   /* j prefactor / (ne nu/Th^2) */
#define IP_C_HKT  (IP_HPL / (IP_ME * IP_CL * IP_CL))                           /* h nu / (me c^2 Th)         */
#define IP_C_IBNU (IP_CL * IP_CL / (2.0 * IP_HPL))                             /* 1/B_nu = C ip_expm1(.)/nu^3   */
#define IP_C_NUB  (IP_EE / (2.0 * M_PI * IP_ME * IP_CL))
#define IP_C_RV   (IP_EE * IP_EE * IP_EE / (M_PI * IP_ME * IP_ME * IP_CL * IP_CL))
#define IP_C_RQ   (IP_EE * IP_EE * IP_EE * IP_EE / (4.0 * M_PI * M_PI * IP_ME * IP_ME * IP_ME * IP_CL * IP_CL * IP_CL))

// INVARIANT: jI,jQ,jV are j/nu^2; aI,aQ,aV are alpha*nu; rQ,rV are rho*nu (R-1), the form the transfer
// step consumes; otherwise plain plasma-frame cgs coefficients (the form the stage parity test compares).  cosT = cosine of the angle between wave vector and field.  Divisions are replaced by a few
// shared reciprocals (1/nu, 1/Th, 1/nu_c, cube root reciprocal), pow(X,p) by exp(p ln X).
template <bool INVARIANT>
__device__ __forceinline__ Coeff synchrotron(double ne, double Th, double B, double cosT, double nu) {
  Coeff c;
  c.jI = c.jQ = c.jV = c.aI = c.aQ = c.aV = c.rQ = c.rV = 0.0;
  const double sin2 = 1.0 - cosT * cosT;
  if (!(sin2 > 0.0) || !(ne > 0.0) || !(B > 0.0) || !(Th > 0.0)) return c;
  const double isinT = ip_rsqrt(sin2), sinT = sin2 * isinT;
  const double inu = ip_rcp(nu), iTh = ip_rcp(Th);
  const double BsT = B * sinT;
  const double nuc = IP_C_NUC * BsT * (Th * Th);
  const double x = ip_div(nu, nuc);
  const double iy = rcbrt(x), iy2 = iy * iy;
  const double y = x * iy2;
  const double ex = ip_exp(-1.8899 * y);
  const double FI = 2.5651 * fma(fma(0.9977, iy, 1.92), iy, 1.0) * ex;
  const double FQ = 2.5651 * fma(fma(0.499873, iy, 0.93193), iy, 1.0) * ex;
  const double FV = (1.81348 * (iy2 * iy) + 3.42319 * iy2 + 0.0292545 * ip_rsqrt(x) + 2.03773 * iy) * ex;
  // j = C ne nu / Th^2 F
  const double pre0 = IP_C_PRE * ne * (iTh * iTh);
  const double pre = pre0 * (INVARIANT ? inu : nu);
  const double FVc = (4.0 / 3.0) * iTh * (cosT * isinT) * FV;
  c.jI = pre * FI;
  c.jQ = pre * FQ;
  c.jV = pre * FVc;
  // alpha = j / B_nu = j C expm1(h nu / (me c^2 Th)) / nu^3; the prefactors are multiplied first so that alpha
  // keeps full precision where j/nu^2 itself is subnormal (far Wien tail)
  const double prea = pre0 * (INVARIANT ? inu : inu * inu) * (IP_C_IBNU * ip_expm1(IP_C_HKT * nu * iTh));
  // Kirchhoff's law is applied to the emissivity as computed: where the cgs emissivity underflows to zero the
  // absorptivity is zero too (R-7: alpha_S = j_S / B_nu)
  const double prec = INVARIANT ? pre0 * nu : pre;
  c.aI = (prec * FI != 0.0) ? prea * FI : 0.0;
  c.aQ = (prec * FQ != 0.0) ? prea * FQ : 0.0;
  c.aV = (prec * FVc != 0.0) ? prea * FVc : 0.0;
  double r0, r1;
  bessel_ratios(iTh, Th, r0, r1);
  const double X = Th * ip_sqrt((1.4142135623730950488e3 * IP_C_NUB) * BsT * inu);
  const double fX = faraday_fX(X);
  const double neinu = ne * (INVARIANT ? inu : inu * inu);
  c.rV = IP_C_RV * neinu * B * cosT * r0;
  c.rQ = IP_C_RQ * neinu * inu * (BsT * BsT) * fX * (r1 + 6.0 * Th);
  c.jI = finite_or_zero(c.jI); c.jQ = finite_or_zero(c.jQ); c.jV = finite_or_zero(c.jV);
  c.aI = finite_or_zero(c.aI); c.aQ = finite_or_zero(c.aQ); c.aV = finite_or_zero(c.aV);
  c.rQ = finite_or_zero(c.rQ); c.rV = finite_or_zero(c.rV);
  return c;
}

__device__ __forceinline__ Coeff synchrotron_invariant(double ne, double Th, double B, double cosT, double nu) {
  return synchrotron<true>(ne, Th, B, cosT, nu);
}
__device__ __forceinline__ Coeff synchrotron_coefficients(double ne, double Th, double B, double cosT, double nu) {
  return synchrotron<false>(ne, Th, B, cosT, nu);
}

}  // namespace ipole
