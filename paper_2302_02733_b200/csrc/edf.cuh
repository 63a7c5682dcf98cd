// Second physics workload ("eDFs for which accurate prescriptions ... do not exist and
// the integration of synchrotron emissivity over the electron energy distribution function requires numerical
// integration during ray tracing"): j_{I,Q,V} and alpha_{I,Q,V} of every transfer step by quadrature over the electron
// distribution.  Reading DESIGN.md R-13:
//   n(gamma) = N gamma^2 beta g(gamma),   g = exp(-gamma/Theta_e)  (Maxwell-Juettner)  |  [1 + (gamma-1)/(kappa w)]^-(kappa+1), w = Theta_e  (kappa)
//   j_I = C int n F(x) dgamma,  j_Q = C int n G(x) dgamma,  j_V = C (4 cot(theta)/3) int n H(x)/gamma dgamma,
//   alpha_S = -(C / (2 m nu^2)) int kernel_S gamma^2 d/dgamma[n/gamma^2] dgamma,  d/dgamma[n/gamma^2] = N g (beta' - beta L),
//   x = nu / ((3/2) gamma^2 nu_B sin(theta)),  C = sqrt3 e^3 B sin(theta) / (4 pi m c^2),  N from int n dgamma = n_e,
// all integrals by the midpoint rule in ln(gamma) on n_nodes equal cells of [0, ln gamma_max] -- the rule is part of the
// definition, the oracle (oracle/ref_edf.hpp) uses the same one.  rho_Q, rho_V stay the thermal expressions of coeff.cuh.
//
// The kernels F, G, H (x int K_5/3, x K_2/3, x K_1/3 + int K_1/3) come from piecewise degree-11 polynomials of their
// exponentially scaled forms (synch_tables.inc, written by gen_synch_tables.py); a node costs ~150 FP64 operations and a
// step 128 nodes: ~20 kflop per step, 13 times the whole thermal step.  It runs in k_apply (stepop.cuh), lane <-> ray.
#pragma once
#include "coeff.cuh"
#include "synch_tables.inc"

namespace ipole {

struct EdfDev {
  int kind;          // 0 thermal fits, 1 Maxwell-Juettner, 2 kappa
  int n_nodes;
  double kappa;
  double du;         // ln(gamma_max) / n_nodes
};

// e^x F(x), e^x G(x), e^x H(x) for 0 < x < 2^IPOLE_SYN_E1
__device__ __forceinline__ void synch_kernels_scaled(double x, double& F, double& G, double& H) {
  int piece; double v;
  if (IP_LIKELY(pw_locate(x, IPOLE_SYN_E0, IPOLE_SYN_E1, piece, v))) {
    const double* t = &g_syn[piece][0][0];
    double f, g, h, z;
    ld_global_nc_v4(t + 4 * (IPOLE_PW_NC - 1), f, g, h, z);
#pragma unroll
    for (int j = IPOLE_PW_NC - 2; j >= 0; --j) {
      double cf, cg, chh;
      ld_global_nc_v4(t + 4 * j, cf, cg, chh, z);
      f = fma(f, v, cf);
      g = fma(g, v, cg);
      h = fma(h, v, chh);
    }
    F = f; G = g; H = h;
  } else {
    // below the table: F, G ~ x^(1/3), H -> int_0^inf K_1/3 (never reached with gamma_max <= 1e6 at radio frequencies)
    const double s = cbrt(x * exp2(-(double)IPOLE_SYN_E0));
    F = IPOLE_SYN_F0 * s; G = IPOLE_SYN_G0 * s; H = IPOLE_SYN_H0;
  }
}

// plasma-frame cgs j_{I,Q,V}, alpha_{I,Q,V} into c (rho_Q, rho_V untouched)
__device__ __forceinline__ void synchrotron_edf_cgs(const EdfDev& E, double ne, double Th, double B, double cosT, double nu, Coeff& c) {
  c.jI = c.jQ = c.jV = c.aI = c.aQ = c.aV = 0.0;
  const double sin2 = 1.0 - cosT * cosT;
  if (!(sin2 > 0.0) || !(ne > 0.0) || !(B > 0.0) || !(Th > 0.0)) return;
  const double isinT = ip_rsqrt(sin2), sinT = sin2 * isinT;
  const double nuB = IP_C_NUB * B;
  const double xs = ip_div(nu, 1.5 * nuB * sinT);         // x = xs / gamma^2
  const double iTh = ip_rcp(Th);
  const double ikw = (E.kind == 2) ? ip_rcp(E.kappa * Th) : 0.0;
  const double kp1 = E.kappa + 1.0;
  double sN = 0.0, sI = 0.0, sQ = 0.0, sV = 0.0, aI = 0.0, aQ = 0.0, aV = 0.0;
  for (int k = 0; k < E.n_nodes; ++k) {
    const double gam = ip_exp(((double)k + 0.5) * E.du);
    const double ig = ip_rcp(gam), ig2 = ig * ig;
    const double b2 = 1.0 - ig2;
    const double ibeta = ip_rsqrt(b2), beta = b2 * ibeta;
    const double dbeta = ig2 * ig * ibeta;
    double g, L;
    if (E.kind == 1) { g = ip_exp(-gam * iTh); L = iTh; }
    else {
      const double q = fma(gam - 1.0, ikw, 1.0);
      g = ip_exp(-kp1 * ip_log(q));
      L = kp1 * ikw * ip_rcp(q);
    }
    const double w = gam * E.du;
    const double n = gam * gam * beta * g;
    sN = fma(n, w, sN);
    const double x = xs * ig2;
    if (x < 745.0) {                                    // beyond, e^-x is zero in double precision (and in the oracle)
      double F, G, H;
      synch_kernels_scaled(x, F, G, H);
      const double ex = ip_exp(-x) * w;
      F *= ex; G *= ex; H *= ex;
      const double dn = g * (dbeta - beta * L) * (gam * gam);
      sI = fma(n, F, sI);
      sQ = fma(n, G, sQ);
      sV = fma(n * ig, H, sV);
      aI = fma(F, dn, aI);
      aQ = fma(G, dn, aQ);
      aV = fma(H * ig, dn, aV);
    }
  }
  const double C = (IP_SQRT3 * IP_EE * IP_EE * IP_EE / (4.0 * M_PI * IP_ME * IP_CL * IP_CL)) * B * sinT;
  const double Nn = ip_div(ne, sN);
  const double cot43 = (4.0 / 3.0) * cosT * isinT;
  const double inu = ip_rcp(nu);
  const double A = -C * (1.0 / (2.0 * IP_ME)) * inu * inu;
  c.jI = finite_or_zero(C * Nn * sI);
  c.jQ = finite_or_zero(C * Nn * sQ);
  c.jV = finite_or_zero(C * Nn * cot43 * sV);
  c.aI = finite_or_zero(A * Nn * aI);
  c.aQ = finite_or_zero(A * Nn * aQ);
  c.aV = finite_or_zero(A * Nn * cot43 * aV);
}

// invariant forms (j/nu^2, alpha nu, rho nu) with the Faraday coefficients of the thermal expressions
__device__ __forceinline__ Coeff synchrotron_edf_invariant(const EdfDev& E, double ne, double Th, double B, double cosT, double nu) {
  Coeff c = synchrotron_invariant(ne, Th, B, cosT, nu);     // rho_Q nu, rho_V nu (the thermal j, alpha are replaced)
  Coeff e;
  synchrotron_edf_cgs(E, ne, Th, B, cosT, nu, e);
  const double inu = ip_rcp(nu), inu2 = inu * inu;
  c.jI = e.jI * inu2; c.jQ = e.jQ * inu2; c.jV = e.jV * inu2;
  c.aI = e.aI * nu; c.aQ = e.aQ * nu; c.aV = e.aV * nu;
  return c;
}

__global__ void k_eval_coefficients_edf(EdfDev E, int64_t n, const double* in, double* out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  Coeff c = synchrotron_coefficients(in[5 * i], in[5 * i + 1], in[5 * i + 2], in[5 * i + 3], in[5 * i + 4]);
  if (E.kind != 0) synchrotron_edf_cgs(E, in[5 * i], in[5 * i + 1], in[5 * i + 2], in[5 * i + 3], in[5 * i + 4], c);
  double* o = out + 8 * i;
  o[0] = c.jI; o[1] = c.jQ; o[2] = c.jV; o[3] = c.aI; o[4] = c.aQ; o[5] = c.aV; o[6] = c.rQ; o[7] = c.rV;
}

}  // namespace ipole
