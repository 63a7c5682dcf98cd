// ORACLE (test infrastructure).  Thermal synchrotron emission, absorption and Faraday coefficients.
//
// PAPER.md:33 names the processes ("synchrotron emission, synchrotron absorption and Faraday effects such
// as Faraday rotation and Faraday conversion") and PAPER.md:35 says they are evaluated "at every single
// step"; the formulas are not in the paper.  Reading DESIGN.md R-7: published
// ultra-relativistic thermal fits in the tetrad where j_U = alpha_U = rho_U = 0,
//   nu_c = 3 e B sin(thB) Th^2 / (4 pi m_e c),  x = nu/nu_c,  y = x^(1/3)
//   j_I = [n e^2 nu / (2 sqrt3 c Th^2)] 2.5651 (1 + 1.92/y + 0.9977/y^2) exp(-1.8899 y)
//   j_Q = [same]                        2.5651 (1 + 0.93193/y + 0.499873/y^2) exp(-1.8899 y)
//   j_V = [2 n e^2 nu cot(thB) / (3 sqrt3 c Th^3)] (1.81348/x + 3.42319/y^2 + 0.0292545/sqrt x + 2.03773/y) exp(-1.8899 y)
//   alpha_S = j_S / B_nu (Kirchhoff),  B_nu = (2 h nu^3/c^2) / expm1(h nu / (m_e c^2 Th))
//   rho_V = [n e^3 B cos(thB) / (pi m_e^2 c^2 nu^2)] K0(1/Th)/K2(1/Th)
//   rho_Q = [n e^4 B^2 sin^2(thB) / (4 pi^2 m_e^3 c^3 nu^3)] f(X) [K1(1/Th)/K2(1/Th) + 6 Th]
//   f(X) = 2.011 exp(-X^1.035/4.7) - cos(X/2) exp(-X^1.2/2.73) - 0.011 exp(-X/47.2)
//   X = Th [sqrt2 sin(thB) 1e3 nu_B/nu]^(1/2),  nu_B = e B / (2 pi m_e c)
// Modified Bessel functions K_n by trapezoid quadrature of the integral representation
//   e^z K_n(z) = int_0^inf exp(-z (cosh t - 1)) cosh(n t) dt     (exponentially convergent).
#pragma once
#include <cmath>

namespace iref {

// CGS constants, R-1
constexpr double EE = 4.80320680e-10;
constexpr double CL = 2.99792458e10;
constexpr double ME = 9.1093826e-28;
constexpr double MP = 1.67262171e-24;
constexpr double HPL = 6.6260693e-27;
constexpr double KBOL = 1.3806505e-16;
constexpr double GNEWT = 6.6742e-8;
constexpr double MSUN = 1.989e33;
constexpr double PC = 3.085678e18;

// out[n] = e^z K_n(z), n = 0,1,2
inline void bessel_k_scaled(double z, double out[3]) {
  // integrand negligible beyond z (cosh T - 1) = 50
  const double T = std::acosh(1.0 + 50.0 / z);
  int N = (int)std::ceil(T / 0.125);
  if (N < 96) N = 96;
  const double h = T / N;
  double s0 = 0.0, s1 = 0.0, s2 = 0.0;
  for (int i = 0; i <= N; ++i) {
    const double t = i * h;
    const double ch = std::cosh(t);
    // cosh t - 1 = 2 sinh^2(t/2): no cancellation at small t
    const double sh2 = std::sinh(0.5 * t);
    const double w = ((i == 0 || i == N) ? 0.5 : 1.0) * std::exp(-z * 2.0 * sh2 * sh2);
    s0 += w;
    s1 += w * ch;
    s2 += w * (2.0 * ch * ch - 1.0);
  }
  out[0] = h * s0; out[1] = h * s1; out[2] = h * s2;
}

struct CoeffCGS { double jI, jQ, jV, aI, aQ, aV, rQ, rV; };

inline double finite_or_zero(double v) { return std::isfinite(v) ? v : 0.0; }

// coefficients in the plasma frame, cgs, at frequency nu [Hz]; cosT = cos(angle between k and B)
inline CoeffCGS synchrotron_coefficients(double ne, double Th, double B, double cosT, double nu) {
  CoeffCGS c{0, 0, 0, 0, 0, 0, 0, 0};
  const double sin2 = 1.0 - cosT * cosT;
  if (!(sin2 > 0.0) || !(ne > 0.0) || !(B > 0.0) || !(Th > 0.0)) return c;
  const double sinT = std::sqrt(sin2);
  const double nuc = 3.0 * EE * B * sinT * Th * Th / (4.0 * M_PI * ME * CL);
  const double x = nu / nuc;
  const double y = std::cbrt(x);
  const double ex = std::exp(-1.8899 * y);
  const double FI = 2.5651 * (1.0 + 1.92 / y + 0.9977 / (y * y)) * ex;
  const double FQ = 2.5651 * (1.0 + 0.93193 / y + 0.499873 / (y * y)) * ex;
  const double FV = (1.81348 / x + 3.42319 / (y * y) + 0.0292545 / std::sqrt(x) + 2.03773 / y) * ex;
  const double pre = ne * EE * EE * nu / (2.0 * std::sqrt(3.0) * CL * Th * Th);
  c.jI = pre * FI;
  c.jQ = pre * FQ;
  c.jV = 2.0 * ne * EE * EE * nu * (cosT / sinT) / (3.0 * std::sqrt(3.0) * CL * Th * Th * Th) * FV;
  const double Bnu = (2.0 * HPL * nu * nu * nu / (CL * CL)) / std::expm1(HPL * nu / (ME * CL * CL * Th));
  c.aI = c.jI / Bnu;
  c.aQ = c.jQ / Bnu;
  c.aV = c.jV / Bnu;
  double k[3];
  bessel_k_scaled(1.0 / Th, k);
  const double nuB = EE * B / (2.0 * M_PI * ME * CL);
  const double X = Th * std::sqrt(std::sqrt(2.0) * sinT * 1e3 * nuB / nu);
  const double fX = 2.011 * std::exp(-std::pow(X, 1.035) / 4.7) - std::cos(0.5 * X) * std::exp(-std::pow(X, 1.2) / 2.73)
                    - 0.011 * std::exp(-X / 47.2);
  c.rV = ne * EE * EE * EE * B * cosT / (M_PI * ME * ME * CL * CL * nu * nu) * (k[0] / k[2]);
  c.rQ = ne * EE * EE * EE * EE * B * B * sin2 / (4.0 * M_PI * M_PI * ME * ME * ME * CL * CL * CL * nu * nu * nu) * fX
         * (k[1] / k[2] + 6.0 * Th);
  c.jI = finite_or_zero(c.jI); c.jQ = finite_or_zero(c.jQ); c.jV = finite_or_zero(c.jV);
  c.aI = finite_or_zero(c.aI); c.aQ = finite_or_zero(c.aQ); c.aV = finite_or_zero(c.aV);
  c.rQ = finite_or_zero(c.rQ); c.rV = finite_or_zero(c.rV);
  return c;
}

}  // namespace iref
