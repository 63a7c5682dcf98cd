// ORACLE (test infrastructure).  Camera, step rule, RK4 null-geodesic push and ray tracing.
//
// Follows PAPER.md:35 ("the code launches photons from the point of the camera and integrates a null
// geodesic equation for every single pixel ... The step size of the integration is adaptive and
// parameterized") and PAPER.md:43 (backward integration away from the observer, the path saved; the
// integrator "is not perfectly time-reversible"; step parameter epsilon).  The paper gives neither the
// camera construction, the integrator nor the step rule: readings DESIGN.md R-3, R-4 (SURVEY.md 8(c)
// c-3, c-4):
//   camera tetrad by Gram-Schmidt at (r_cam, theta_cam, phi = 0): e0 || d_t, e3 from d_X1 (outward),
//   e2 from -d_X2 (up, toward the spin axis), e1 from d_X3 (right);
//   pixel (i,j): alpha = (i+1/2-nx/2) fov/nx, beta = (j+1/2-ny/2) fov/nx,
//   K = e0 + [-(alpha/r_cam) e1 - (beta/r_cam) e2 + e3] / sqrt(1 + (alpha^2+beta^2)/r_cam^2);
//   dX/dl = K, dK/dl = -Gamma(X) K K, classical RK4, step -dl with
//   dl = 1/(1/dl1 + 1/dl2 + 1/dl3), dl1 = eps/(|K1|+d), dl2 = eps min(X2,1-X2)/(|K2|+d), dl3 = eps/(|K3|+d).
#pragma once
#include <vector>
#include <array>
#include "ref_metric.hpp"

namespace iref {

struct Camera {
  Geom geom;
  double r_cam, fov, inclination_deg;
  int nx, ny;
  double eps, r_esc, stop_factor;
  int max_steps;
  double Xcam[4];
  double e[4][4];  // e[a][mu], contravariant components of the camera tetrad
};

inline void gram_schmidt(const double g[4][4], double v[4], const double (*basis)[4], const double* sign, int nb) {
  for (int b = 0; b < nb; ++b) {
    const double p = sign[b] * dot(g, v, basis[b]);
    for (int m = 0; m < 4; ++m) v[m] -= p * basis[b][m];
  }
  const double n = std::sqrt(std::fabs(dot(g, v, v)));
  for (int m = 0; m < 4; ++m) v[m] /= n;
}

inline void camera_setup(Camera& C) {
  const double th = C.inclination_deg * M_PI / 180.0;
  C.Xcam[0] = 0.0;
  C.Xcam[1] = std::log(C.r_cam);
  C.Xcam[2] = (C.geom.hslope == 1.0) ? th / M_PI : x2_of_theta(C.geom.hslope, th);
  C.Xcam[3] = 0.0;
  double g[4][4];
  gcov(C.geom, C.Xcam, g);
  const double sign[4] = {-1.0, 1.0, 1.0, 1.0};  // metric signature of the basis vectors already built
  // e0: static observer
  double e0[4] = {1.0, 0.0, 0.0, 0.0};
  const double n0 = std::sqrt(-dot(g, e0, e0));
  for (int m = 0; m < 4; ++m) C.e[0][m] = e0[m] / n0;
  // order of orthogonalisation: e0, e3, e2, e1
  double basis[4][4];
  double sg[4];
  for (int m = 0; m < 4; ++m) basis[0][m] = C.e[0][m];
  sg[0] = sign[0];
  double e3[4] = {0.0, 1.0, 0.0, 0.0};
  gram_schmidt(g, e3, basis, sg, 1);
  for (int m = 0; m < 4; ++m) { C.e[3][m] = e3[m]; basis[1][m] = e3[m]; }
  sg[1] = 1.0;
  double e2[4] = {0.0, 0.0, -1.0, 0.0};
  gram_schmidt(g, e2, basis, sg, 2);
  for (int m = 0; m < 4; ++m) { C.e[2][m] = e2[m]; basis[2][m] = e2[m]; }
  sg[2] = 1.0;
  double e1[4] = {0.0, 0.0, 0.0, 1.0};
  gram_schmidt(g, e1, basis, sg, 3);
  for (int m = 0; m < 4; ++m) C.e[1][m] = e1[m];
}

// impact parameters alpha (right) and beta (up) in GM/c^2
inline void camera_ray_ab(const Camera& C, double alpha, double beta, double X[4], double K[4]) {
  const double px = -alpha / C.r_cam, py = -beta / C.r_cam;
  const double nrm = std::sqrt(1.0 + px * px + py * py);
  for (int m = 0; m < 4; ++m) {
    X[m] = C.Xcam[m];
    K[m] = C.e[0][m] + (px * C.e[1][m] + py * C.e[2][m] + C.e[3][m]) / nrm;
  }
}

inline void camera_ray(const Camera& C, int i, int j, double X[4], double K[4]) {
  const double pix = C.fov / C.nx;  // square pixels
  camera_ray_ab(C, (i + 0.5 - 0.5 * C.nx) * pix, (j + 0.5 - 0.5 * C.ny) * pix, X, K);
}

inline double stepsize(const double X[4], const double K[4], double eps) {
  const double d = 1e-40;
  const double dl1 = eps / (std::fabs(K[1]) + d);
  const double dl2 = eps * std::fabs(std::fmin(X[2], 1.0 - X[2])) / (std::fabs(K[2]) + d);
  const double dl3 = eps / (std::fabs(K[3]) + d);
  return 1.0 / (1.0 / dl1 + 1.0 / dl2 + 1.0 / dl3);
}

inline void geodesic_rhs(const Geom& G, const double X[4], const double K[4], double dX[4], double dK[4]) {
  double Gam[4][4][4];
  connection(G, X, Gam);
  for (int l = 0; l < 4; ++l) {
    double s = 0.0;
    for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) s += Gam[l][m][n] * K[m] * K[n];
    dX[l] = K[l];
    dK[l] = -s;
  }
}

// classical 4th-order Runge-Kutta on (X,K), step dl (signed)
inline void rk4_push(const Geom& G, double X[4], double K[4], double dl) {
  double x1[4], k1[4], x2[4], k2[4], x3[4], k3[4], x4[4], k4[4], Xt[4], Kt[4];
  geodesic_rhs(G, X, K, x1, k1);
  for (int m = 0; m < 4; ++m) { Xt[m] = X[m] + 0.5 * dl * x1[m]; Kt[m] = K[m] + 0.5 * dl * k1[m]; }
  geodesic_rhs(G, Xt, Kt, x2, k2);
  for (int m = 0; m < 4; ++m) { Xt[m] = X[m] + 0.5 * dl * x2[m]; Kt[m] = K[m] + 0.5 * dl * k2[m]; }
  geodesic_rhs(G, Xt, Kt, x3, k3);
  for (int m = 0; m < 4; ++m) { Xt[m] = X[m] + dl * x3[m]; Kt[m] = K[m] + dl * k3[m]; }
  geodesic_rhs(G, Xt, Kt, x4, k4);
  for (int m = 0; m < 4; ++m) {
    X[m] += dl / 6.0 * (x1[m] + 2.0 * x2[m] + 2.0 * x3[m] + x4[m]);
    K[m] += dl / 6.0 * (k1[m] + 2.0 * k2[m] + 2.0 * k3[m] + k4[m]);
  }
}

struct Path {
  std::vector<std::array<double, 4>> X, K;  // points 0..n (0 = camera)
  std::vector<double> dl;                   // dl[s] > 0: step between point s and s+1
  int nturn = 0;                            // sign changes of K^2 between consecutive points
  int status = 0;                           // 1 horizon, 2 escaped, 3 max_steps
};

inline double inner_stop_radius(const Camera& C) {
  return C.geom.flat ? 1e-3 : C.stop_factor * horizon_radius(C.geom.a);
}

inline void trace(const Camera& C, const double X0[4], const double K0[4], Path& P) {
  P.X.clear(); P.K.clear(); P.dl.clear(); P.nturn = 0; P.status = 0;
  double X[4], K[4];
  for (int m = 0; m < 4; ++m) { X[m] = X0[m]; K[m] = K0[m]; }
  P.X.push_back({X[0], X[1], X[2], X[3]});
  P.K.push_back({K[0], K[1], K[2], K[3]});
  const double r_in = inner_stop_radius(C);
  int n = 0;
  while (true) {
    const double dl = stepsize(X, K, C.eps);
    const double x1_before = X[1];
    const double k2_before = K[2];
    rk4_push(C.geom, X, K, -dl);
    ++n;
    P.X.push_back({X[0], X[1], X[2], X[3]});
    P.K.push_back({K[0], K[1], K[2], K[3]});
    P.dl.push_back(dl);
    if ((K[2] < 0.0) != (k2_before < 0.0)) P.nturn++;
    const double r = std::exp(X[1]);
    if (r <= r_in) { P.status = 1; break; }
    if (r > C.r_esc && X[1] > x1_before) { P.status = 2; break; }
    if (n >= C.max_steps) { P.status = 3; break; }
  }
}

}  // namespace iref
