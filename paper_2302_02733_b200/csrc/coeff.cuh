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
    const double lg = log(0.5 * z);
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
    const double ez = exp(z);
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

struct Coeff { double jI, jQ, jV, aI, aQ, aV, rQ, rV; };

__device__ __forceinline__ double finite_or_zero(double v) { return isfinite(v) ? v : 0.0; }

// plasma-frame cgs coefficients at frequency nu; cosT = cosine of the angle between wave vector and field
__device__ __forceinline__ Coeff synchrotron_coefficients(double ne, double Th, double B, double cosT, double nu) {
  Coeff c;
  c.jI = c.jQ = c.jV = c.aI = c.aQ = c.aV = c.rQ = c.rV = 0.0;
  const double sin2 = 1.0 - cosT * cosT;
  if (!(sin2 > 0.0) || !(ne > 0.0) || !(B > 0.0) || !(Th > 0.0)) return c;
  const double sinT = sqrt(sin2);
  const double nuc = 3.0 * IP_EE * B * sinT * Th * Th / (4.0 * M_PI * IP_ME * IP_CL);
  const double x = nu / nuc;
  const double y = cbrt(x);
  const double iy = 1.0 / y;
  const double ex = exp(-1.8899 * y);
  const double FI = 2.5651 * (1.0 + 1.92 * iy + 0.9977 * iy * iy) * ex;
  const double FQ = 2.5651 * (1.0 + 0.93193 * iy + 0.499873 * iy * iy) * ex;
  const double FV = (1.81348 / x + 3.42319 * iy * iy + 0.0292545 * rsqrt(x) + 2.03773 * iy) * ex;
  const double pre = ne * IP_EE * IP_EE * nu / (2.0 * sqrt(3.0) * IP_CL * Th * Th);
  c.jI = pre * FI;
  c.jQ = pre * FQ;
  c.jV = 2.0 * ne * IP_EE * IP_EE * nu * (cosT / sinT) / (3.0 * sqrt(3.0) * IP_CL * Th * Th * Th) * FV;
  const double iBnu = expm1(IP_HPL * nu / (IP_ME * IP_CL * IP_CL * Th)) / (2.0 * IP_HPL * nu * nu * nu / (IP_CL * IP_CL));
  c.aI = c.jI * iBnu;
  c.aQ = c.jQ * iBnu;
  c.aV = c.jV * iBnu;
  double k0, k1;
  bessel_k01_scaled(1.0 / Th, k0, k1);
  const double k2 = k0 + 2.0 * Th * k1;
  const double nuB = IP_EE * B / (2.0 * M_PI * IP_ME * IP_CL);
  const double X = Th * sqrt(sqrt(2.0) * sinT * 1e3 * nuB / nu);
  const double fX = 2.011 * exp(-pow(X, 1.035) / 4.7) - cos(0.5 * X) * exp(-pow(X, 1.2) / 2.73) - 0.011 * exp(-X / 47.2);
  c.rV = ne * IP_EE * IP_EE * IP_EE * B * cosT / (M_PI * IP_ME * IP_ME * IP_CL * IP_CL * nu * nu) * (k0 / k2);
  c.rQ = ne * IP_EE * IP_EE * IP_EE * IP_EE * B * B * sin2
         / (4.0 * M_PI * M_PI * IP_ME * IP_ME * IP_ME * IP_CL * IP_CL * IP_CL * nu * nu * nu) * fX * (k1 / k2 + 6.0 * Th);
  c.jI = finite_or_zero(c.jI); c.jQ = finite_or_zero(c.jQ); c.jV = finite_or_zero(c.jV);
  c.aI = finite_or_zero(c.aI); c.aQ = finite_or_zero(c.aQ); c.aV = finite_or_zero(c.aV);
  c.rQ = finite_or_zero(c.rQ); c.rV = finite_or_zero(c.rV);
  return c;
}

}  // namespace ipole
