// ORACLE (test infrastructure, not product code): the path-free bidirectional variant of the per-pixel loop.
//
// PAPER.md:43 (section 2.2): "The CPU code integrates the geodesics backwards in time (away from the observer) and
// saves the path to integrate radiative-transfer equation forward in time.  The GPU code does this integration in
// both directions, away from the observer (backwards in time) and toward the observer (forward in time), without
// saving the path in both cases. ... our geodesics integrator is not perfectly time-reversible so geodesic
// integrated forward in time may result in a slightly different path."
//
// The paper does not say how the forward pass chooses its steps, where it stops, or in which frame the result is
// read.  Reading R-10:
//   * the backward pass is trace() of ref_geodesic.hpp with nothing kept but its end point (X_n, K_n), its step
//     count n and its turning-point count;
//   * the forward pass starts at (X_n, K_n) and takes classical RK4 steps of +dl_j, dl_j = the same step rule
//     evaluated at the point the step starts from, until a step ends at r >= r_cam moving outward (the mirror image
//     of the backward pass's escape test), or at r <= the inner stop radius moving inward, or after max_steps steps.  Because the
//     rule is evaluated at the other end of each interval, the forward pass does not retrace the backward points
//     and in general takes a different number of steps;
//   * each forward step [hi -> lo] is one transfer step of transfer_along_path(): midpoint (Xm, Km) of its two end
//     points, half transport, plasma operator over dl_j, half transport;
//   * the forward pass ends within one step of the camera but not at it, so the tensor is read in the camera-type
//     tetrad built AT THE END POINT by the camera's own construction (static observer, e3 from d_X1, e2 from
//     -d_X2, e1 from d_X3; observer_tetrad()).  Reading the tensor with the tetrad of the camera position instead
//     is wrong by (r_cam/r_end)^2 in every Stokes parameter, since the angular coordinate components scale as 1/r.
// Step by step in that order; no other change to the stored-path oracle.
#pragma once
#include <array>
#include <vector>
#include "ref_geodesic.hpp"
#include "ref_transfer.hpp"

namespace iref {

// the camera construction of camera_setup() at an arbitrary point X (pin PF1: equals the camera tetrad at Xcam)
inline void observer_tetrad(const Geom& G, const double X[4], double e[4][4]) {
  double g[4][4];
  gcov(G, X, g);
  double basis[3][4], sg[3];
  double e0[4] = {1.0, 0.0, 0.0, 0.0};
  const double n0 = std::sqrt(-dot(g, e0, e0));
  for (int m = 0; m < 4; ++m) { e[0][m] = e0[m] / n0; basis[0][m] = e[0][m]; }
  sg[0] = -1.0;
  double e3[4] = {0.0, 1.0, 0.0, 0.0};
  gram_schmidt(g, e3, basis, sg, 1);
  for (int m = 0; m < 4; ++m) { e[3][m] = e3[m]; basis[1][m] = e3[m]; }
  sg[1] = 1.0;
  double e2[4] = {0.0, 0.0, -1.0, 0.0};
  gram_schmidt(g, e2, basis, sg, 2);
  for (int m = 0; m < 4; ++m) { e[2][m] = e2[m]; basis[2][m] = e2[m]; }
  sg[2] = 1.0;
  double e1[4] = {0.0, 0.0, 0.0, 1.0};
  gram_schmidt(g, e1, basis, sg, 3);
  for (int m = 0; m < 4; ++m) e[1][m] = e1[m];
}

struct Retrace {                               // optional record of the forward pass (index 0 = far end)
  std::vector<std::array<double, 4>> X, K;
  std::vector<double> dl;
};

// returns the number of forward steps; on return X, K hold the end point of the forward pass
inline int transfer_path_free(const Camera& C, const Model& M, const Units& U, const double Xn[4], const double Kn[4],
                              cplx N[4][4], double* tau, double* tauF, double Xend[4], Retrace* rec = nullptr) {
  double X[4], K[4];
  for (int m = 0; m < 4; ++m) { X[m] = Xn[m]; K[m] = Kn[m]; }
  if (rec) { rec->X.push_back({X[0], X[1], X[2], X[3]}); rec->K.push_back({K[0], K[1], K[2], K[3]}); }
  const double r_in = inner_stop_radius(C);
  int j = 0;
  while (true) {
    const double dl = stepsize(X, K, C.eps);
    double Xhi[4], Khi[4], Xm[4], Km[4], P[4][4];
    for (int m = 0; m < 4; ++m) { Xhi[m] = X[m]; Khi[m] = K[m]; }
    rk4_push(C.geom, X, K, +dl);
    ++j;
    for (int m = 0; m < 4; ++m) { Xm[m] = 0.5 * (X[m] + Xhi[m]); Km[m] = 0.5 * (K[m] + Khi[m]); }
    if (N) {
      transport_matrix(C.geom, Xm, Km, 0.5 * dl, P);
      congruence(P, N);
      plasma_operator(C.geom, M, U, Xm, Km, dl, N, tau, tauF);
      congruence(P, N);
    }
    if (rec) { rec->X.push_back({X[0], X[1], X[2], X[3]}); rec->K.push_back({K[0], K[1], K[2], K[3]}); rec->dl.push_back(dl); }
    if (X[1] >= C.Xcam[1] && X[1] > Xhi[1]) break;
    if (std::exp(X[1]) <= r_in && X[1] < Xhi[1]) break;
    if (j >= C.max_steps) break;
  }
  for (int m = 0; m < 4; ++m) Xend[m] = X[m];
  return j;
}

// Stokes (invariant I/nu^3 units) read in the observer tetrad at the end point of the forward pass
inline void end_point_stokes(const Camera& C, const double Xend[4], const cplx N[4][4], double S[4]) {
  Camera E = C;
  for (int m = 0; m < 4; ++m) E.Xcam[m] = Xend[m];
  observer_tetrad(C.geom, Xend, E.e);
  camera_stokes(C.geom, E, N, S);
}

}  // namespace iref
