// ORACLE (test infrastructure).  Plasma models: what the fluid is at a point X of the ray.
//
// "For semianalytic models, the code calculates the model at the current geodesic
// position.  For GRMHD simulations we read out the plasma quantities from precomputed three 3D arrays
// ... and the code interpolates the plasma quantities to the point at every single step."
// The paper prints neither model; BASELINE.json configs[0] and configs[2] fix the parameters and the
// readings are DESIGN.md R-5:
//
// ADAF  n_e = n0 r^p_n, Theta_e = Th0 r^p_T, B = B0 r^p_B (r = Kerr-Schild radius, no theta
//       dependence); u: Keplerian u = u^t (1,0,0,Omega), Omega = 1/(r^1.5 + a) for r >= r_ISCO,
//       E = 1, L = 0 free fall inside: u_t = -1, u_theta = u_phi = 0,
//       u_r = -2r / (2r + sqrt(2r (r^2+a^2)))   [regular root of Delta u_r^2 - 4 r u_r - 2 r = 0];
//       b: d_phi projected orthogonal to u, scaled to b.b = B^2 (purely toroidal field).
// GRID  cell-centred MKS lattice, 8 planes rho,u,U1,U2,U3,B1,B2,B3, index (i N2 + j) N3 + k,
//       trilinear in index space, X3 periodic, X1/X2 clamped, empty for r > r_out or X1 < startx1;
//       primitives -> u^mu, b^mu the usual GRMHD way; Theta_e from the R_low/R_high prescription.
// SLAB  (tests) constant coefficients inside |r cos(theta)| < H, static fluid, uniform Cartesian
//       field direction cos(psi) x^ + sin(psi) y^; Cartesian x + i y = (r + i a) e^{i phi} sin(theta).
#pragma once
#include <cmath>
#include <vector>
#include "ref_metric.hpp"
#include "ref_coeff.hpp"

namespace iref {

enum ModelKind { MODEL_NONE = 0, MODEL_ADAF = 1, MODEL_SLAB = 2, MODEL_GRID = 3 };

struct AdafParams { double n0, p_n, Th0, p_T, B0, p_B; };
struct SlabParams { double H; int profile; double psi_deg; double j[4], alpha[4], rho[3]; };
struct GridParams {
  int N1, N2, N3;
  double startx[3], dx[3];
  double hslope, gam, M_unit, Rlow, Rhigh, r_out;
  std::vector<double> f[8];  // copies of the 8 planes
};

struct Plasma {
  bool present = false;
  double ne = 0, Th = 0, B = 0;  // cm^-3, dimensionless, Gauss
  double u[4] = {0, 0, 0, 0};    // fluid four-velocity, MKS contravariant
  double b[4] = {0, 0, 0, 0};    // field four-vector, MKS contravariant, |b| = B (direction only for the slab)
  bool direct = false;           // slab: cgs coefficients given directly
  double j[4] = {0, 0, 0, 0}, al[4] = {0, 0, 0, 0}, rh[3] = {0, 0, 0};
};

inline void plasma_adaf(const Geom& G, const AdafParams& M, const double X[4], Plasma& p) {
  const double a = G.a;
  const double r = std::exp(X[1]);
  double g[4][4], gi[4][4];
  gcov(G, X, g);
  p.ne = M.n0 * std::pow(r, M.p_n);
  p.Th = M.Th0 * std::pow(r, M.p_T);
  p.B = M.B0 * std::pow(r, M.p_B);
  if (r >= isco_radius(a)) {
    const double Om = 1.0 / (std::pow(r, 1.5) + a);
    const double ut = 1.0 / std::sqrt(-(g[0][0] + 2.0 * g[0][3] * Om + g[3][3] * Om * Om));
    p.u[0] = ut; p.u[1] = 0.0; p.u[2] = 0.0; p.u[3] = ut * Om;
  } else {
    invert4(g, gi);
    const double ur_ks = -2.0 * r / (2.0 * r + std::sqrt(2.0 * r * (r * r + a * a)));
    const double ucov[4] = {-1.0, r * ur_ks, 0.0, 0.0};  // u_X1 = (dr/dX1) u_r
    for (int m = 0; m < 4; ++m) {
      double s = 0.0;
      for (int n = 0; n < 4; ++n) s += gi[m][n] * ucov[n];
      p.u[m] = s;
    }
  }
  const double t[4] = {0.0, 0.0, 0.0, 1.0};
  const double tu = dot(g, t, p.u);
  double bb[4];
  for (int m = 0; m < 4; ++m) bb[m] = t[m] + tu * p.u[m];
  const double nrm = std::sqrt(dot(g, bb, bb));
  for (int m = 0; m < 4; ++m) p.b[m] = bb[m] * (p.B / nrm);
  p.present = true;
}

// solve the 3x3 system A x = y by Cramer's rule
inline void solve3(const double A[3][3], const double y[3], double x[3]) {
  auto det3 = [](const double M[3][3]) {
    return M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1]) - M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0])
           + M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0]);
  };
  const double D = det3(A);
  for (int c = 0; c < 3; ++c) {
    double B[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) B[i][j] = (j == c) ? y[i] : A[i][j];
    x[c] = det3(B) / D;
  }
}

inline void plasma_slab(const Geom& G, const SlabParams& M, const double X[4], Plasma& p) {
  const double a = G.a;
  const double r = std::exp(X[1]);
  const double th = theta_of_x2(G.hslope, X[2]);
  const double ph = X[3];
  const double z = r * std::cos(th);
  double w = 1.0;
  if (M.profile == 0) { if (!(std::fabs(z) < M.H)) return; }
  else w = std::exp(-z * z / (2.0 * M.H * M.H));
  double g[4][4];
  gcov(G, X, g);
  p.u[0] = 1.0 / std::sqrt(-g[0][0]); p.u[1] = p.u[2] = p.u[3] = 0.0;
  // Jacobian d(x,y,z)/d(r,theta,phi) of x = (r cos ph - a sin ph) sin th, y = (r sin ph + a cos ph) sin th, z = r cos th
  const double s = std::sin(th), c = std::cos(th), cp = std::cos(ph), sp = std::sin(ph);
  const double Jm[3][3] = {{cp * s, (r * cp - a * sp) * c, (-r * sp - a * cp) * s},
                           {sp * s, (r * sp + a * cp) * c, (r * cp - a * sp) * s},
                           {c, -r * s, 0.0}};
  const double psi = M.psi_deg * M_PI / 180.0;
  const double dir[3] = {std::cos(psi), std::sin(psi), 0.0};
  double v[3];
  solve3(Jm, dir, v);
  // KS (r,theta,phi) components -> MKS: divide by dr/dX1 = r and dtheta/dX2
  const double sp4[4] = {0.0, v[0] / r, v[1] / dtheta_dx2(G.hslope, X[2]), v[2]};
  // make it orthogonal to u (u is static, g_ti may be non-zero when the metric is not flat)
  const double su = dot(g, sp4, p.u);
  for (int m = 0; m < 4; ++m) p.b[m] = sp4[m] + su * p.u[m];
  const double nrm = std::sqrt(dot(g, p.b, p.b));
  for (int m = 0; m < 4; ++m) p.b[m] /= nrm;
  p.B = 1.0;
  p.direct = true;
  for (int i = 0; i < 4; ++i) { p.j[i] = w * M.j[i]; p.al[i] = w * M.alpha[i]; }
  for (int i = 0; i < 3; ++i) p.rh[i] = w * M.rho[i];
  p.present = true;
}

inline int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// L_unit = G M / c^2 [cm] enters through rho_unit = M_unit / L^3
inline void plasma_grid(const Geom& G, const GridParams& M, double L_unit, const double X[4], Plasma& p) {
  const double r = std::exp(X[1]);
  if (r > M.r_out || X[1] < M.startx[0]) return;
  // position in index space of the cell-centred lattice
  const double fi = (X[1] - M.startx[0]) / M.dx[0] - 0.5;
  const double fj = (X[2] - M.startx[1]) / M.dx[1] - 0.5;
  const double fk = (X[3] - M.startx[2]) / M.dx[2] - 0.5;
  const double i0f = std::floor(fi), j0f = std::floor(fj), k0f = std::floor(fk);
  const double di = fi - i0f, dj = fj - j0f, dk = fk - k0f;
  const int i0 = clampi((int)i0f, 0, M.N1 - 1), i1 = clampi((int)i0f + 1, 0, M.N1 - 1);
  const int j0 = clampi((int)j0f, 0, M.N2 - 1), j1 = clampi((int)j0f + 1, 0, M.N2 - 1);
  long kk = (long)k0f % M.N3; if (kk < 0) kk += M.N3;
  const int k0 = (int)kk, k1 = (int)((kk + 1) % M.N3);
  double prim[8];
  for (int q = 0; q < 8; ++q) {
    const double* F = M.f[q].data();
    auto at = [&](int i, int j, int k) { return F[((size_t)i * M.N2 + j) * M.N3 + k]; };
    prim[q] = (1 - di) * ((1 - dj) * ((1 - dk) * at(i0, j0, k0) + dk * at(i0, j0, k1))
                          + dj * ((1 - dk) * at(i0, j1, k0) + dk * at(i0, j1, k1)))
              + di * ((1 - dj) * ((1 - dk) * at(i1, j0, k0) + dk * at(i1, j0, k1))
                      + dj * ((1 - dk) * at(i1, j1, k0) + dk * at(i1, j1, k1)));
  }
  const double rho = prim[0], uu = prim[1];
  if (!(rho > 0.0) || !(uu > 0.0)) return;
  double g[4][4], gi[4][4];
  gcov(G, X, g);
  invert4(g, gi);
  const double alpha_l = 1.0 / std::sqrt(-gi[0][0]);
  double q2 = 0.0;
  for (int i = 1; i < 4; ++i) for (int j = 1; j < 4; ++j) q2 += g[i][j] * prim[1 + i] * prim[1 + j];
  const double gamma = std::sqrt(1.0 + q2);
  p.u[0] = gamma / alpha_l;
  for (int i = 1; i < 4; ++i) p.u[i] = prim[1 + i] - gamma * alpha_l * gi[0][i];
  double bt = 0.0;
  for (int i = 1; i < 4; ++i) for (int m = 0; m < 4; ++m) bt += g[i][m] * prim[4 + i] * p.u[m];
  double bc[4];
  bc[0] = bt;
  for (int i = 1; i < 4; ++i) bc[i] = (prim[4 + i] + bt * p.u[i]) / p.u[0];
  const double bsq = dot(g, bc, bc);
  if (!(bsq > 0.0)) return;
  const double rho_unit = M.M_unit / (L_unit * L_unit * L_unit);
  const double B_unit = CL * std::sqrt(4.0 * M_PI * rho_unit);
  p.ne = rho * rho_unit / (MP + ME);
  p.B = std::sqrt(bsq) * B_unit;
  const double beta = (M.gam - 1.0) * uu / (0.5 * bsq);
  const double b2 = beta * beta;
  const double R = (M.Rhigh * b2 + M.Rlow) / (1.0 + b2);
  p.Th = (MP / ME) * (M.gam - 1.0) * (uu / rho) / (1.0 + R);
  for (int m = 0; m < 4; ++m) p.b[m] = bc[m] * B_unit;
  p.present = true;
}

}  // namespace iref
