// Second physics workload ("eDFs for which accurate prescriptions ... do not exist and
// the integration of synchrotron emissivity over the electron energy distribution function requires numerical
// integration during ray tracing"): j_{I,Q,V} and alpha_{I,Q,V} of every transfer step by quadrature over the electron
// distribution.  Reading DESIGN.md R-13:
//   n(gamma) = N gamma^2 beta g(gamma),   g = exp(-(gamma-1)/Theta_e)  (Maxwell-Juettner)  |  [1 + (gamma-1)/(kappa w)]^-(kappa+1), w = Theta_e  (kappa)
//   j_I = C int n F(x) dgamma,  j_Q = C int n G(x) dgamma,  j_V = C (4 cot(theta)/3) int n H(x)/gamma dgamma,
//   alpha_S = -(C / (2 m nu^2)) int kernel_S gamma^2 d/dgamma[n/gamma^2] dgamma,  d/dgamma[n/gamma^2] = N g (beta' - beta L),
//   x = nu / ((3/2) gamma^2 nu_B sin(theta)) = xs / gamma^2,  C = sqrt3 e^3 B sin(theta) / (4 pi m c^2),  N from int n dgamma = n_e.
// Quadrature (part of the definition; the oracle, oracle/ref_edf.hpp, uses the same rule): midpoint rule on n_nodes equal
// cells of ln x in [-16, 4], gamma_k = sqrt(xs / x_k), dgamma = (gamma/2) dln x; N by the midpoint rule on 512 cells of
// ln(gamma - 1) in [-16, 16].  rho_Q, rho_V stay the thermal expressions of coeff.cuh.
//
// With fixed x nodes the single-electron kernels F, G, H (x int K_5/3, x K_2/3, x K_1/3 + int K_1/3) are per-node
// constants: ipole_set_edf evaluates them once (k_edf_setup_nodes, from the piecewise degree-11 tables of their scaled
// forms in synch_tables.inc, written by gen_synch_tables.py) and k_apply stages them in shared memory, where all lanes of a
// warp read the same row.  (A first version integrated over ln gamma and looked the kernels up per node and lane: 36
// scattered 32-byte reads per node, which bound it by the L1 data pipe at 44 % FP64 -- profiles/r2_notes.md.)  The
// normalisation integral depends on Theta_e alone: ipole_set_edf tabulates its logarithm on a fine grid of ln Theta_e with
// the defining rule (k_edf_setup_norm) and the step interpolates it (4-point Lagrange, spacing 0.002: error < 1e-12).
// A node is then ~60 (Maxwell-Juettner) to ~90 (kappa) FP64 operations, all arithmetic: ~10 kflop per step with 128
// nodes, seven times the whole thermal step.  It runs in k_apply (stepop.cuh), lane <-> ray.
#pragma once
#include "coeff.cuh"
#include "synch_tables.inc"

namespace ipole {

#ifndef IPOLE_EDF_UNROLL
#define IPOLE_EDF_UNROLL 8
#endif
constexpr int EDF_UNROLL = IPOLE_EDF_UNROLL;
constexpr double EDF_LNX_LO = -16.0, EDF_LNX_HI = 4.0;
constexpr int EDF_NORM_NODES = 512;
constexpr double EDF_LNT_LO = -16.0, EDF_LNT_HI = 16.0;
constexpr int EDF_MAX_NODES = 1024;
// table of ln int (n/N) dgamma over ln Theta_e
constexpr double EDF_TAB_LNTH0 = -11.5, EDF_TAB_H = 0.002;   // Theta_e from 1e-5 ...
constexpr int EDF_TAB_N = 12001;                              // ... to 2.7e5

struct EdfDev {
  int kind;          // 0 thermal fits, 1 Maxwell-Juettner, 2 kappa
  int n_nodes;
  double kappa;
  double dlx;        // (EDF_LNX_HI - EDF_LNX_LO) / n_nodes
  const double4* nodes;   // device: per x node {x^-1/2, F(x), G(x), H(x)}
  const double* lnnorm;   // device: EDF_TAB_N values of ln int_1^inf gamma^2 beta g dgamma
};

// e^x F(x), e^x G(x), e^x H(x) for 0 < x < 2^IPOLE_SYN_E1 from the table `tab` (g_syn)
__device__ __forceinline__ void synch_kernels_scaled(const double* __restrict__ tab, double x, double& F, double& G, double& H) {
  int piece; double v;
  if (IP_LIKELY(pw_locate(x, IPOLE_SYN_E0, IPOLE_SYN_E1, piece, v))) {
    const double4* t = reinterpret_cast<const double4*>(tab) + (size_t)piece * IPOLE_PW_NC;
    double4 c = t[IPOLE_PW_NC - 1];
    double f = c.x, g = c.y, h = c.z;
#pragma unroll
    for (int j = IPOLE_PW_NC - 2; j >= 0; --j) {
      c = t[j];
      f = fma(f, v, c.x);
      g = fma(g, v, c.y);
      h = fma(h, v, c.z);
    }
    F = f; G = g; H = h;
  } else {
    // below the table: F, G ~ x^(1/3), H -> int_0^inf K_1/3 (never reached with gamma_max <= 1e6 at radio frequencies)
    const double s = cbrt(x * exp2(-(double)IPOLE_SYN_E0));
    F = IPOLE_SYN_F0 * s; G = IPOLE_SYN_G0 * s; H = IPOLE_SYN_H0;
  }
}

// g(gamma) and L = -dln g/dgamma at gamma - 1 = gm1
template <int KIND>
__device__ __forceinline__ void edf_shape(const EdfDev& E, double iTh, double ikw, double gm1, double& g, double& L) {
  if (KIND == 1) { g = ip_exp(-gm1 * iTh); L = iTh; }
  else {
    const double q = fma(gm1, ikw, 1.0);
    const double kp1 = E.kappa + 1.0;
    g = ip_exp(-kp1 * ip_log(q));
    L = kp1 * ikw * ip_rcp(q);
  }
}

// int_1^inf gamma^2 beta g(gamma) dgamma by the defining rule (library exp/sqrt: set-up and fall-back only)
__device__ __forceinline__ double edf_norm_integral(const EdfDev& E, double Th) {
  const double dlt = (EDF_LNT_HI - EDF_LNT_LO) / EDF_NORM_NODES;
  double s = 0.0;
  for (int k = 0; k < EDF_NORM_NODES; ++k) {
    const double t = exp(EDF_LNT_LO + ((double)k + 0.5) * dlt);
    double g;
    if (E.kind == 1) g = exp(-t / Th);
    else g = pow(1.0 + t / (E.kappa * Th), -(E.kappa + 1.0));
    s += (1.0 + t) * sqrt(t * (t + 2.0)) * g * t * dlt;
  }
  return s;
}

// ipole_set_edf: the per-node constants and the normalisation table
__global__ void k_edf_setup_nodes(EdfDev E, double4* nodes) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= E.n_nodes) return;
  const double x = exp(EDF_LNX_HI - ((double)k + 0.5) * E.dlx);
  double F, G, H;
  synch_kernels_scaled(&g_syn[0][0][0], x, F, G, H);
  const double ex = exp(-x);
  nodes[k] = make_double4(1.0 / sqrt(x), F * ex, G * ex, H * ex);
}
__global__ void k_edf_setup_norm(EdfDev E, double* lnnorm) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= EDF_TAB_N) return;
  lnnorm[i] = log(edf_norm_integral(E, exp(EDF_TAB_LNTH0 + i * EDF_TAB_H)));
}

// ln of the normalisation integral at Theta_e: 4-point Lagrange interpolation of the table (direct evaluation outside it)
__device__ __forceinline__ double edf_lnnorm(const EdfDev& E, double Th) {
  const double u = (ip_log(Th) - EDF_TAB_LNTH0) * (1.0 / EDF_TAB_H);
  const double fl = floor(u);
  const int i = (int)fl;
  if (IP_UNLIKELY(!(i >= 1 && i + 2 < EDF_TAB_N))) return log(edf_norm_integral(E, Th));
  const double t = u - fl;
  const double f0 = __ldg(E.lnnorm + i - 1), f1 = __ldg(E.lnnorm + i), f2 = __ldg(E.lnnorm + i + 1), f3 = __ldg(E.lnnorm + i + 2);
  const double w0 = -t * (t - 1.0) * (t - 2.0) * (1.0 / 6.0), w1 = (t + 1.0) * (t - 1.0) * (t - 2.0) * 0.5;
  const double w2 = -(t + 1.0) * t * (t - 2.0) * 0.5, w3 = (t + 1.0) * t * (t - 1.0) * (1.0 / 6.0);
  return w0 * f0 + w1 * f1 + w2 * f2 + w3 * f3;
}

// The node sums.  KIND is a template parameter so that the loop body holds no branch at all: the unrolled iterations then
// sit in one basic block and their reciprocal -> reciprocal square root -> exponential chains interleave.
template <int KIND>
__device__ __forceinline__ void edf_node_sums(const EdfDev& E, const double4* __restrict__ nodes, double sx, double iTh, double ikw,
                                              double& sI, double& sQ, double& sV, double& aI, double& aQ, double& aV) {
#pragma unroll EDF_UNROLL
  for (int k = 0; k < E.n_nodes; ++k) {
    const double4 nd = nodes[k];
    const double gam0 = sx * nd.x;
    const bool on = gam0 > 1.0;                        // cells below gamma = 1 carry no electrons (branch-free: the
    const double gam = on ? gam0 : 2.0;                // iterations of the unrolled loop interleave)
    const double ig = ip_rcp(gam), ig2 = ig * ig;
    const double b2 = 1.0 - ig2;
    const double ibeta = ip_rsqrt(b2), beta = b2 * ibeta;
    const double dbeta = ig2 * ig * ibeta;
    double g, L;
    edf_shape<KIND>(E, iTh, ikw, gam - 1.0, g, L);
    const double g3 = on ? gam * gam * gam * g : 0.0;             // gamma^3 g: n/N times the varying part of the cell width, over beta
    const double A1 = g3 * beta, A2 = g3 * (dbeta - beta * L);
    sI = fma(A1, nd.y, sI);
    sQ = fma(A1, nd.z, sQ);
    sV = fma(A1 * ig, nd.w, sV);
    aI = fma(A2, nd.y, aI);
    aQ = fma(A2, nd.z, aQ);
    aV = fma(A2 * ig, nd.w, aV);
  }
}

// plasma-frame cgs j_{I,Q,V}, alpha_{I,Q,V} into c (rho_Q, rho_V untouched).  `nodes`: E.nodes or a copy in shared memory.
__device__ __forceinline__ void synchrotron_edf_cgs(const EdfDev& E, const double4* __restrict__ nodes,
                                                    double ne, double Th, double B, double cosT, double nu, Coeff& c) {
  c.jI = c.jQ = c.jV = c.aI = c.aQ = c.aV = 0.0;
  const double sin2 = 1.0 - cosT * cosT;
  if (!(sin2 > 0.0) || !(ne > 0.0) || !(B > 0.0) || !(Th > 0.0)) return;
  const double isinT = ip_rsqrt(sin2), sinT = sin2 * isinT;
  const double nuB = IP_C_NUB * B;
  const double sx = ip_sqrt(ip_div(nu, 1.5 * nuB * sinT));       // gamma_k = sx x_k^-1/2
  const double iTh = ip_rcp(Th);
  const double ikw = ip_rcp(E.kappa * Th);
  double sI = 0.0, sQ = 0.0, sV = 0.0, aI = 0.0, aQ = 0.0, aV = 0.0;
  if (E.kind == 1) edf_node_sums<1>(E, nodes, sx, iTh, ikw, sI, sQ, sV, aI, aQ, aV);
  else edf_node_sums<2>(E, nodes, sx, iTh, ikw, sI, sQ, sV, aI, aQ, aV);
  const double C = (IP_SQRT3 * IP_EE * IP_EE * IP_EE / (4.0 * M_PI * IP_ME * IP_CL * IP_CL)) * B * sinT;
  const double Nn = ne * ip_exp(-edf_lnnorm(E, Th)) * (0.5 * E.dlx);   // N times the constant part of the cell width
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
__device__ __forceinline__ Coeff synchrotron_edf_invariant(const EdfDev& E, const double4* __restrict__ nodes, double ne, double Th,
                                                           double B, double cosT, double nu) {
  Coeff c = synchrotron_invariant(ne, Th, B, cosT, nu);     // rho_Q nu, rho_V nu (the thermal j, alpha are replaced)
  Coeff e;
  synchrotron_edf_cgs(E, nodes, ne, Th, B, cosT, nu, e);
  const double inu = ip_rcp(nu), inu2 = inu * inu;
  c.jI = e.jI * inu2; c.jQ = e.jQ * inu2; c.jV = e.jV * inu2;
  c.aI = e.aI * nu; c.aQ = e.aQ * nu; c.aV = e.aV * nu;
  return c;
}

__global__ void k_eval_coefficients_edf(EdfDev E, int64_t n, const double* in, double* out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  Coeff c = synchrotron_coefficients(in[5 * i], in[5 * i + 1], in[5 * i + 2], in[5 * i + 3], in[5 * i + 4]);
  if (E.kind != 0) synchrotron_edf_cgs(E, E.nodes, in[5 * i], in[5 * i + 1], in[5 * i + 2], in[5 * i + 3], in[5 * i + 4], c);
  double* o = out + 8 * i;
  o[0] = c.jI; o[1] = c.jQ; o[2] = c.jV; o[3] = c.aI; o[4] = c.aQ; o[5] = c.aV; o[6] = c.rQ; o[7] = c.rV;
}

}  // namespace ipole
