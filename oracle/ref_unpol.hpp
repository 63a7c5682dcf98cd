// ORACLE (test infrastructure, not product code): unpolarized transfer along a stored path.
//
// the model-fitting use case runs "nonpolarized images of moderate (to low) resolution of 128 x 128";
// polarized transfer is "far more complex and computationally demanding" than the unpolarized one.  The
// paper prints no equation for it; reading R-12: the scalar transfer equation in invariant form,
//   d(I/nu^3)/d(lambda) = j_I/nu^2 - (alpha_I nu) (I/nu^3),
// solved exactly over each step with the coefficients frozen at the step's midpoint -- the I row of the polarized
// step with alpha_Q = alpha_V = 0:
//   x = alpha_inv ds,   I <- I e^{-x} + j_inv ds (1 - e^{-x})/x      (the last factor is 1 at x = 0),
// on the same path, with the same midpoints (Xm, Km), the same plasma state, frequency nu = -k.u nu_obs, pitch angle
// and thermal synchrotron j_I, alpha_I as the polarized oracle.  No tetrad and no parallel transport are needed.
// It is NOT Stokes I of the polarized solution (there alpha_Q, alpha_V couple I to Q and V): pins U1-U3
// (tests/test_oracle_unpol.py) state the relation.
#pragma once
#include <cmath>
#include "ref_transfer.hpp"

namespace iref {

inline void unpolarized_step(const Geom& G, const Model& M, const Units& U, const double X[4], const double K[4], double dl,
                             double* I, double* tau) {
  Plasma p;
  plasma_at(G, M, U, X, p);
  if (!p.present) return;
  double g[4][4], kcov[4];
  gcov(G, X, g);
  lower(g, K, kcov);
  double om = 0.0;
  for (int m = 0; m < 4; ++m) om -= kcov[m] * p.u[m];
  if (!(om > 0.0)) return;
  const double nu = om * U.nu_obs;
  double jc, ac;
  if (p.direct) { jc = p.j[0]; ac = p.al[0]; }
  else {
    double bcov[4];
    lower(g, p.b, bcov);
    double bk = 0.0;
    for (int m = 0; m < 4; ++m) bk += bcov[m] * K[m];
    double cosT = bk / (om * p.B);
    if (cosT > 1.0) cosT = 1.0;
    if (cosT < -1.0) cosT = -1.0;
    const CoeffCGS c = synchrotron_coefficients_edf(M.edf, p.ne, p.Th, p.B, cosT, nu);
    jc = c.jI; ac = c.aI;
  }
  const double ji = jc / (nu * nu), ai = ac * nu;
  const double ds = dl * U.L_unit / U.nu_obs;
  const double x = ai * ds;
  const double em = std::expm1(-x);                     // e^{-x} - 1
  const double E = (x > 0.0) ? -em / x : 1.0;           // (1 - e^{-x}) / x
  *I = *I + *I * em + ji * ds * E;
  if (tau) *tau += x;
}

// Walk the stored path from its far end to the camera; returns I/nu^3 at the camera.
inline double transfer_unpolarized(const Geom& G, const Model& M, const Units& U, const Path& path, double* tau) {
  double I = 0.0;
  const int n = (int)path.dl.size();
  for (int s = n - 1; s >= 0; --s) {
    double Xm[4], Km[4];
    for (int m = 0; m < 4; ++m) {
      Xm[m] = 0.5 * (path.X[s][m] + path.X[s + 1][m]);
      Km[m] = 0.5 * (path.K[s][m] + path.K[s + 1][m]);
    }
    unpolarized_step(G, M, U, Xm, Km, path.dl[s], &I, tau);
  }
  return I;
}

}  // namespace iref
