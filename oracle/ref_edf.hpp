// ORACLE (test infrastructure, not product code).  Synchrotron emissivities and absorptivities integrated numerically
// over an electron energy distribution function (eDF).
//
// PAPER.md:78 (Section 4, outlook): "The idea is to have eDFs for which accurate prescriptions ... do not exist and the
// integration of synchrotron emissivity over the electron energy distribution function requires numerical integration
// during ray tracing."  The paper gives no formulas; reading DESIGN.md R-13:
//
// eDF, isotropic, dn = n(gamma) dgamma, beta = sqrt(1 - 1/gamma^2):
//   kind 1  Maxwell-Juettner   n(gamma) = N gamma^2 beta exp(-(gamma-1)/Theta_e)
//   kind 2  kappa              n(gamma) = N gamma^2 beta [1 + (gamma - 1)/(kappa w)]^-(kappa+1),   w = Theta_e
//   N from  int n dgamma = n_e  by the quadrature stated below (the rule, not a closed form, defines the result).
// Single-electron synchrotron power in Stokes I, Q and the circular term (Rybicki & Lightman 6.31-6.35; Legg & Westfold
// 1968 as used in pin T8), pitch angle = angle theta between wave vector and field, nu_B = e B / (2 pi m c):
//   x = nu / nu_cr(gamma),   nu_cr = (3/2) gamma^2 nu_B sin(theta),   C = sqrt3 e^3 B sin(theta) / (4 pi m c^2)
//   j_I = C int n F(x) dgamma,   j_Q = C int n G(x) dgamma,   j_V = C (4 cot(theta)/3) int n H(x) / gamma dgamma
//   F(x) = x int_x^inf K_5/3,   G(x) = x K_2/3(x),   H(x) = x K_1/3(x) + int_x^inf K_1/3
// Absorption (Rybicki & Lightman 6.50 with E = gamma m c^2), same kernels:
//   alpha_S = -(C / (2 m nu^2)) int kernel_S(x, gamma) gamma^2 d/dgamma [ n(gamma) / gamma^2 ] dgamma
// with the derivative taken analytically:  d/dgamma[n/gamma^2] = N g(gamma) [ beta' - beta L(gamma) ],  beta' = 1/(gamma^3 beta),
//   Maxwell-Juettner g = exp(-(gamma-1)/Theta), L = 1/Theta;   kappa  g = q^-(kappa+1), L = (kappa+1)/(kappa w q), q = 1 + (gamma-1)/(kappa w).
// Quadrature (part of the definition of the result; the GPU follows the same rule):
//   * emission and absorption integrals in the variable x: n_nodes equal cells in ln x on [ln X_LO, ln X_HI] = [-16, 4],
//     midpoint rule, x_k = exp(ln X_HI - (k + 1/2) dlx), gamma_k = sqrt(xs / x_k) with xs = nu / ((3/2) nu_B sin(theta)),
//     dgamma = (gamma/2) dlx; cells with gamma_k <= 1 carry no electrons.  (The single-electron kernels are then the same
//     numbers F(x_k), G(x_k), H(x_k) for every plasma state -- which is what makes the rule cheap on the GPU; the range
//     covers 9 decades of x, e^-x F < 1e-22 above it and the eDF tail integrand falls like x^1.1 below it.)
//   * normalisation N = n_e / int_1^inf (n/N) dgamma in t = gamma - 1: 512 equal cells in ln t on [-16, 16], midpoint rule
//     (resolves cold, gamma - 1 ~ Theta_e << 1, and hot distributions alike).
//   Maxwell-Juettner is evaluated as g = exp(-(gamma - 1)/Theta_e): the common factor e^(-1/Theta_e) cancels against N.
// Faraday rotation and conversion keep the thermal expressions of ref_coeff.hpp with Theta_e (kappa: w) -- the paper's
// sentence is about the emissivity; stated as a reading.
//
// The kernels by the exponentially convergent trapezoid rule on
//   K_nu(x) = int_0^inf exp(-x cosh t) cosh(nu t) dt,   int_x^inf K_nu = int_0^inf exp(-x cosh t) cosh(nu t) / cosh t dt .
// Pins (tests/test_oracle_edf.py): F, G, H against mpmath/scipy; kind 1 against the thermal fits and Kirchhoff's law;
// kind 2 -> kind 1 for kappa -> infinity and the Rybicki & Lightman power-law closed forms (6.36, 6.53) in the tail;
// distance of the rule from adaptive quadrature; j_V, alpha_V of the kappa tail against the Mellin transform of H (E6).
#pragma once
#include <cmath>
#include "ref_coeff.hpp"

namespace iref {

struct EdfParams {
  int kind = 0;            // 0: the thermal fits of ref_coeff.hpp (default); 1: Maxwell-Juettner; 2: kappa
  double kappa = 3.5;
  int n_nodes = 128;       // cells of the x quadrature
};

constexpr double EDF_LNX_LO = -16.0, EDF_LNX_HI = 4.0;
constexpr int EDF_NORM_NODES = 512;
constexpr double EDF_LNT_LO = -16.0, EDF_LNT_HI = 16.0;

// F, G, H at x > 0
inline void synchrotron_kernels(double x, double& F, double& G, double& H) {
  // integrand < exp(-x) exp(-60) beyond x (cosh T - 1) = 60
  const double T = std::acosh(1.0 + 60.0 / x);
  int N = (int)std::ceil(T / 0.125);
  if (N < 64) N = 64;
  const double h = T / N;
  double sF = 0.0, sG = 0.0, sH = 0.0;
  for (int i = 0; i <= N; ++i) {
    const double t = i * h;
    const double ch = std::cosh(t);
    const double sh2 = std::sinh(0.5 * t);
    const double w = ((i == 0 || i == N) ? 0.5 : 1.0) * std::exp(-x * 2.0 * sh2 * sh2);   // exp(-x (cosh t - 1))
    sF += w * std::cosh(5.0 * t / 3.0) / ch;
    sG += w * std::cosh(2.0 * t / 3.0);
    sH += w * std::cosh(t / 3.0) * (x + 1.0 / ch);
  }
  const double ex = std::exp(-x);
  F = x * h * sF * ex;
  G = x * h * sG * ex;
  H = h * sH * ex;
}

// g(gamma) and L(gamma) = -dln g/dgamma of the two distributions
inline void edf_shape(const EdfParams& E, double Th, double gam, double& g, double& L) {
  if (E.kind == 1) { g = std::exp(-(gam - 1.0) / Th); L = 1.0 / Th; }
  else {
    const double q = 1.0 + (gam - 1.0) / (E.kappa * Th);
    g = std::pow(q, -(E.kappa + 1.0));
    L = (E.kappa + 1.0) / (E.kappa * Th * q);
  }
}

// int_1^inf gamma^2 beta g(gamma) dgamma
inline double edf_norm_integral(const EdfParams& E, double Th) {
  const double dlt = (EDF_LNT_HI - EDF_LNT_LO) / EDF_NORM_NODES;
  double s = 0.0;
  for (int k = 0; k < EDF_NORM_NODES; ++k) {
    const double t = std::exp(EDF_LNT_LO + (k + 0.5) * dlt);     // gamma - 1
    const double gam = 1.0 + t;
    double g, L;
    edf_shape(E, Th, gam, g, L);
    s += gam * std::sqrt(t * (t + 2.0)) * g * t * dlt;          // gamma^2 beta = gamma sqrt(gamma^2 - 1); dt = t dlt
  }
  return s;
}

// j_I, j_Q, j_V, alpha_I, alpha_Q, alpha_V by quadrature over the eDF; rho_Q, rho_V thermal.  cgs, plasma frame.
inline CoeffCGS synchrotron_coefficients_edf(const EdfParams& E, double ne, double Th, double B, double cosT, double nu) {
  CoeffCGS c = synchrotron_coefficients(ne, Th, B, cosT, nu);   // rho_Q, rho_V (and the early-outs) from here
  if (E.kind == 0) return c;
  c.jI = c.jQ = c.jV = c.aI = c.aQ = c.aV = 0.0;
  const double sin2 = 1.0 - cosT * cosT;
  if (!(sin2 > 0.0) || !(ne > 0.0) || !(B > 0.0) || !(Th > 0.0)) return c;
  const double sinT = std::sqrt(sin2);
  const double nuB = EE * B / (2.0 * M_PI * ME * CL);
  const double C = std::sqrt(3.0) * EE * EE * EE * B * sinT / (4.0 * M_PI * ME * CL * CL);
  const double xs = nu / (1.5 * nuB * sinT);
  const double dlx = (EDF_LNX_HI - EDF_LNX_LO) / E.n_nodes;
  double sI = 0.0, sQ = 0.0, sV = 0.0, aI = 0.0, aQ = 0.0, aV = 0.0;
  for (int k = 0; k < E.n_nodes; ++k) {
    const double x = std::exp(EDF_LNX_HI - (k + 0.5) * dlx);
    const double gam = std::sqrt(xs / x);
    if (!(gam > 1.0)) continue;
    const double beta = std::sqrt(1.0 - 1.0 / (gam * gam));
    const double dbeta = 1.0 / (gam * gam * gam * beta);
    double g, L;
    edf_shape(E, Th, gam, g, L);
    const double w = 0.5 * gam * dlx;                 // dgamma of the cell
    const double n = gam * gam * beta * g;            // n(gamma) / N
    const double dn = g * (dbeta - beta * L);         // d/dgamma [n / gamma^2] / N
    double F, G, H;
    synchrotron_kernels(x, F, G, H);
    sI += n * F * w;
    sQ += n * G * w;
    sV += n * H / gam * w;
    aI += F * gam * gam * dn * w;
    aQ += G * gam * gam * dn * w;
    aV += H / gam * gam * gam * dn * w;
  }
  const double Nn = ne / edf_norm_integral(E, Th);
  const double cot43 = 4.0 * (cosT / sinT) / 3.0;
  const double A = -C / (2.0 * ME * nu * nu);
  c.jI = finite_or_zero(C * Nn * sI);
  c.jQ = finite_or_zero(C * Nn * sQ);
  c.jV = finite_or_zero(C * Nn * cot43 * sV);
  c.aI = finite_or_zero(A * Nn * aI);
  c.aQ = finite_or_zero(A * Nn * aQ);
  c.aV = finite_or_zero(A * Nn * cot43 * aV);
  return c;
}

}  // namespace iref
