// Plasma models (what the fluid is at a point of the ray), the plasma-frame tetrad, and one application of the
// plasma operator to the polarization state.  DESIGN.md R-5, R-6 ("For semianalytic models, the code
// calculates the model at the current geodesic position.  For GRMHD simulations we read out the plasma quantities
// from precomputed three 3D arrays ... interpolates the plasma quantities to the point at every single step").
//
// Polarization state carried per ray ("factorised coherency tensor"): after every plasma
// step the coherency tensor of PAPER.md:37 is N^{mu nu} = sum_{a,b in {1,2}} n^{ab} f_a^mu f_b^nu with two REAL
// vectors f_1, f_2 (the transverse tetrad legs, parallel-transported since) and the 2x2 Hermitian n^{ab}, i.e. the
// four Stokes parameters S.  The congruence N <- P N P^T is f_a <- P f_a; projecting on a new tetrad is the real
// 2x2 congruence n <- M n M^T with M_{a'a} = e^(a')_mu f_a^mu.
#pragma once
#include "geom.cuh"
#include "coeff.cuh"
#include "stokes.cuh"

namespace ipole {

enum { MODEL_NONE = 0, MODEL_ADAF = 1, MODEL_SLAB = 2, MODEL_GRID = 3 };

struct AdafParams { double n0, p_n, Th0, p_T, B0, p_B, r_isco; };
struct SlabParams { double H; int profile; double cpsi, spsi; double j[4], al[4], rh[3]; };
struct GridParams {
  int N1, N2, N3;
  double startx[3], idx[3];      // idx = 1/dx
  double iN3;                    // 1/N3
  double gam, Rlow, Rhigh, r_out, lx_out;   // lx_out = ln r_out
  double ne_unit, B_unit;        // rho -> n_e [cm^-3], sqrt(b.b) -> Gauss
  const unsigned int* occ;       // device bitmap over stencil base cells (N1+1)(N2+1)N3: 1 = some corner has plasma
  const double* cells;           // device, cell-major: cells[((i*N2 + j)*N3 + k)*8 + field], fields rho,u,U1,U2,U3,B1,B2,B3
};
struct Units { double nu_obs, L_unit, D_cm, dl_unit; };
// the four numbers of GridParams a model-fitting sweep varies (ipole_make_images_grid)
struct GridScales { double ne_unit, B_unit, Rlow, Rhigh; };  // dl_unit = L_unit / nu_obs

struct Plasma {
  double ne, Th, B;
  double u[4], b[4];
  double j[4], al[4], rh[3];  // slab only
};

__device__ __forceinline__ double dotg(const Sym7& g, const double u[4], const double v[4]) {
  double l[4];
  g.mul(u, l);
  return dot4(l, v);
}

// the three power laws of the analytic flow at X1 = ln r
__device__ __forceinline__ void adaf_scalars(const AdafParams& M, double x1, double& ne, double& Th, double& B) {
  ne = M.n0 * ip_exp(M.p_n * x1);
  Th = M.Th0 * ip_exp(M.p_T * x1);
  B = M.B0 * ip_exp(M.p_B * x1);
}

// SCALARS = false: flow velocity and field DIRECTION only (b is a unit vector, P.B = 1; n_e, Theta_e are not set):
// what the tetrad and the pitch angle need (k_stepop; the scalars are evaluated where the coefficients are, k_apply)
template <bool SCALARS = true>
__device__ __forceinline__ bool plasma_adaf(const Geom& G, const AdafParams& M, const double X[4], const Point& p,
                                            const Sym7& g, const Inv6& gi, Plasma& P) {
  const double a = G.a, r = p.r;
  if (SCALARS) adaf_scalars(M, X[1], P.ne, P.Th, P.B);
  else { P.ne = 0.0; P.Th = 0.0; P.B = 1.0; }
  if (r >= M.r_isco) {
    const double Om = ip_rcp(r * ip_sqrt(r) + a);
    const double ut = ip_rsqrt(-(g.c00 + 2.0 * g.c03 * Om + g.c33 * Om * Om));
    P.u[0] = ut; P.u[1] = 0.0; P.u[2] = 0.0; P.u[3] = ut * Om;
  } else {
    const double ur_ks = -2.0 * r * ip_rcp(2.0 * r + ip_sqrt(2.0 * r * (r * r + a * a)));
    const double ucov[4] = {-1.0, r * ur_ks, 0.0, 0.0};
    gi.mul(ucov, P.u);
  }
  // d_phi projected orthogonal to u, scaled to b.b = B^2
  const double tu = g.c03 * P.u[0] + g.c13 * P.u[1] + g.c33 * P.u[3];
  double bb[4] = {tu * P.u[0], tu * P.u[1], tu * P.u[2], 1.0 + tu * P.u[3]};
  const double sc = P.B * ip_rsqrt(dotg(g, bb, bb));
#pragma unroll
  for (int m = 0; m < 4; ++m) P.b[m] = bb[m] * sc;
  return true;
}

__device__ __forceinline__ bool plasma_slab(const Geom& G, const SlabParams& M, const double X[4], const Point& p,
                                            const Sym7& g, Plasma& P) {
  const double a = G.a, r = p.r, s = p.s, c = p.c;
  const double z = r * c;
  double w = 1.0;
  if (M.profile == 0) { if (!(fabs(z) < M.H)) return false; }
  else w = ip_exp(-z * z / (2.0 * M.H * M.H));
  P.u[0] = rsqrt(-g.c00); P.u[1] = P.u[2] = P.u[3] = 0.0;
  double sp, cp;
  ip_sincos_any(X[3], &sp, &cp);
  // d(x,y,z)/d(r,theta,phi) of x = (r cos ph - a sin ph) sin th, y = (r sin ph + a cos ph) sin th, z = r cos th
  const double J[3][3] = {{cp * s, (r * cp - a * sp) * c, (-r * sp - a * cp) * s},
                          {sp * s, (r * sp + a * cp) * c, (r * cp - a * sp) * s},
                          {c, -r * s, 0.0}};
  const double dir[3] = {M.cpsi, M.spsi, 0.0};
  // Cramer's rule
  double col[3][3], v[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) { col[0][i] = J[i][0]; col[1][i] = J[i][1]; col[2][i] = J[i][2]; }
  double t[3];
  cross3(col[1], col[2], t); const double D = dot3(col[0], t);
  v[0] = dot3(dir, t) / D;
  cross3(col[2], col[0], t); v[1] = dot3(dir, t) / D;
  cross3(col[0], col[1], t); v[2] = dot3(dir, t) / D;
  const double sp4[4] = {0.0, v[0] / r, v[1] / p.tp, v[2]};
  const double su = dotg(g, sp4, P.u);
#pragma unroll
  for (int m = 0; m < 4; ++m) P.b[m] = sp4[m] + su * P.u[m];
  const double sc = rsqrt(dotg(g, P.b, P.b));
#pragma unroll
  for (int m = 0; m < 4; ++m) P.b[m] *= sc;
  P.B = 1.0; P.ne = 0.0; P.Th = 0.0;
#pragma unroll
  for (int i = 0; i < 4; ++i) { P.j[i] = w * M.j[i]; P.al[i] = w * M.al[i]; }
#pragma unroll
  for (int i = 0; i < 3; ++i) P.rh[i] = w * M.rh[i];
  return true;
}

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// The first two tests of grid_gather alone (same arithmetic, so it is false only where grid_gather is false): X inside
// the lattice in X1 and the stencil-occupancy bit set.  k_geodesic<true> marks with it the steps of a ray that may
// cross plasma.
__device__ __forceinline__ bool grid_occupied(const GridParams& M, const double X[4]) {
  if (X[1] > M.lx_out + 1e-9 || X[1] < M.startx[0]) return false;
  const double fi = (X[1] - M.startx[0]) * M.idx[0] - 0.5;
  const double fj = (X[2] - M.startx[1]) * M.idx[1] - 0.5;
  const double fk = (X[3] - M.startx[2]) * M.idx[2] - 0.5;
  const double i0f = floor(fi), j0f = floor(fj), k0f = floor(fk);
  int k0 = (int)(k0f - (double)M.N3 * floor(k0f * M.iN3));
  if (k0 >= M.N3) k0 -= M.N3;
  if (k0 < 0) k0 += M.N3;
  const int ib = clampi((int)i0f + 1, 0, M.N1), jb = clampi((int)j0f + 1, 0, M.N2);
  const size_t bit = ((size_t)ib * (M.N2 + 1) + jb) * M.N3 + k0;
  return ((__ldg(M.occ + (bit >> 5)) >> (bit & 31)) & 1u) != 0u;
}

// FP64 trilinear interpolation of the 8 fields.  The caller's SoA planes are re-tiled at load time into cell-major
// records of 8 doubles (64 B = two full sectors, 16-B aligned), so one corner of the stencil is two 256-bit
// read-only loads (ld.global.nc.v4.f64) instead of eight scattered 8-byte ones, and the two k-neighbours share a
// 128-B line: 8 lines per evaluation instead of up to 32 sectors in 32 different lines.
// Step 1 (needs no metric): the eight interpolated primitives at X.  Returns false where there is certainly no
// plasma (outside the lattice in X1, or rho <= 0 or u <= 0 after interpolation).
__device__ __forceinline__ bool grid_gather(const GridParams& M, const double X[4], double prim[8]) {
  if (X[1] > M.lx_out + 1e-9 || X[1] < M.startx[0]) return false;   // r_out itself is tested exactly in grid_state
  const double fi = (X[1] - M.startx[0]) * M.idx[0] - 0.5;
  const double fj = (X[2] - M.startx[1]) * M.idx[1] - 0.5;
  const double fk = (X[3] - M.startx[2]) * M.idx[2] - 0.5;
  const double i0f = floor(fi), j0f = floor(fj), k0f = floor(fk);
  const double di = fi - i0f, dj = fj - j0f, dk = fk - k0f;
  const int i0 = clampi((int)i0f, 0, M.N1 - 1), i1 = clampi((int)i0f + 1, 0, M.N1 - 1);
  const int j0 = clampi((int)j0f, 0, M.N2 - 1), j1 = clampi((int)j0f + 1, 0, M.N2 - 1);
  // k0f mod N3 in double arithmetic (a 64-bit integer remainder is ~100 emulated instructions); k0f is an exact
  // integer, so the only possible slip is the quotient being one off, which the two wrap tests repair
  int k0 = (int)(k0f - (double)M.N3 * floor(k0f * M.iN3));
  if (k0 >= M.N3) k0 -= M.N3;
  if (k0 < 0) k0 += M.N3;
  const int k1 = (k0 + 1 == M.N3) ? 0 : k0 + 1;
  // one bit says whether any of the eight corners holds plasma (built at load time by k_build_occupancy with the
  // same index rules): most steps inside r_out cross none, and then cost one 4-byte load instead of 512 bytes
  {
    const int ib = clampi((int)i0f + 1, 0, M.N1), jb = clampi((int)j0f + 1, 0, M.N2);
    const size_t bit = ((size_t)ib * (M.N2 + 1) + jb) * M.N3 + k0;
    if (!((__ldg(M.occ + (bit >> 5)) >> (bit & 31)) & 1u)) return false;
  }
  const size_t o00 = ((size_t)i0 * M.N2 + j0) * M.N3, o01 = ((size_t)i0 * M.N2 + j1) * M.N3;
  const size_t o10 = ((size_t)i1 * M.N2 + j0) * M.N3, o11 = ((size_t)i1 * M.N2 + j1) * M.N3;
  const double wi0 = 1.0 - di, wj0 = 1.0 - dj, wk0 = 1.0 - dk;
  const double w[8] = {wi0 * wj0 * wk0, wi0 * wj0 * dk, wi0 * dj * wk0, wi0 * dj * dk,
                       di * wj0 * wk0,  di * wj0 * dk,  di * dj * wk0,  di * dj * dk};
  const size_t off[8] = {o00 + k0, o00 + k1, o01 + k0, o01 + k1, o10 + k0, o10 + k1, o11 + k0, o11 + k1};
#pragma unroll
  for (int q = 0; q < 8; ++q) prim[q] = 0.0;
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    const double* rec = M.cells + off[c] * 8;
    double v[8];
    ld_global_nc_v4(rec, v[0], v[1], v[2], v[3]);
    ld_global_nc_v4(rec + 4, v[4], v[5], v[6], v[7]);
#pragma unroll
    for (int q = 0; q < 8; ++q) prim[q] = fma(w[c], v[q], prim[q]);
  }
  return prim[0] > 0.0 && prim[1] > 0.0;
}

// Step 2: fluid four-velocity, field four-vector, n_e, Theta_e, B from the primitives and the metric at X.
__device__ __forceinline__ bool grid_state(const Geom& G, const GridParams& M, const GridScales& S, const double prim[8],
                                           const Point& p, const Sym7& g, const Inv6& gi, Plasma& P) {
  if (p.r > M.r_out) return false;
  const double rho = prim[0], uu = prim[1];
  const double alpha_l = ip_rsqrt(-gi.c00);
  // q2 = g_ij U^i U^j (spatial block of the sparse metric)
  const double U1 = prim[2], U2 = prim[3], U3 = prim[4];
  const double q2 = g.c11 * U1 * U1 + 2.0 * g.c13 * U1 * U3 + g.c22 * U2 * U2 + g.c33 * U3 * U3;
  const double gamma = ip_sqrt(1.0 + q2);
  P.u[0] = gamma * ip_sqrt(-gi.c00);
  P.u[1] = U1 - gamma * alpha_l * gi.c01;
  P.u[2] = U2;
  P.u[3] = U3;
  double ul[4];
  g.mul(P.u, ul);
  const double B1 = prim[5], B2 = prim[6], B3 = prim[7];
  const double bt = B1 * ul[1] + B2 * ul[2] + B3 * ul[3];
  double bc[4];
  bc[0] = bt;
  const double iu0 = ip_rcp(P.u[0]);
  bc[1] = (B1 + bt * P.u[1]) * iu0;
  bc[2] = (B2 + bt * P.u[2]) * iu0;
  bc[3] = (B3 + bt * P.u[3]) * iu0;
  const double bsq = dotg(g, bc, bc);
  if (!(bsq > 0.0)) return false;
  P.ne = rho * S.ne_unit;
  P.B = ip_sqrt(bsq) * S.B_unit;
  const double beta = 2.0 * (M.gam - 1.0) * uu * ip_rcp(bsq);
  const double b2 = beta * beta;
  const double R = (S.Rhigh * b2 + S.Rlow) * ip_rcp(1.0 + b2);
  P.Th = (IP_MP / IP_ME) * (M.gam - 1.0) * uu * ip_rcp(rho * (1.0 + R));
#pragma unroll
  for (int m = 0; m < 4; ++m) P.b[m] = bc[m] * S.B_unit;
  return true;
}

__device__ __forceinline__ bool plasma_grid(const Geom& G, const GridParams& M, const double X[4], const Point& p,
                                            const Sym7& g, const Inv6& gi, Plasma& P) {
  double prim[8];
  const GridScales S = {M.ne_unit, M.B_unit, M.Rlow, M.Rhigh};
  return grid_gather(M, X, prim) && grid_state(G, M, S, prim, p, g, gi, P);
}

// eps^{mu a b c} p_a q_b w_c with [0123] = +1
__device__ __forceinline__ void levi4(const double p[4], const double q[4], const double w[4], double o[4]) {
  const double m01 = q[0] * w[1] - q[1] * w[0], m02 = q[0] * w[2] - q[2] * w[0], m03 = q[0] * w[3] - q[3] * w[0];
  const double m12 = q[1] * w[2] - q[2] * w[1], m13 = q[1] * w[3] - q[3] * w[1], m23 = q[2] * w[3] - q[3] * w[2];
  o[0] = p[1] * m23 - p[2] * m13 + p[3] * m12;
  o[1] = -(p[0] * m23 - p[2] * m03 + p[3] * m02);
  o[2] = p[0] * m13 - p[1] * m03 + p[3] * m01;
  o[3] = -(p[0] * m12 - p[1] * m02 + p[2] * m01);
}

// Stokes vector under the real 2x2 congruence n <- M n M^T
__device__ __forceinline__ void stokes_congruence(const double m11, const double m12, const double m21, const double m22,
                                                  double S[4]) {
  // Every rounding is spelt out (no contraction left to the compiler): kernels that walk the same ray in different ways
  // (k_apply, k_apply_wide) must reach the same bits.
  const double R11 = 0.5 * (S[0] + S[1]), R22 = 0.5 * (S[0] - S[1]), R12 = 0.5 * S[2];
  const double a11 = __dmul_rn(m11, m11), a12 = __dmul_rn(m11, m12), a22 = __dmul_rn(m12, m12);
  const double b11 = __dmul_rn(m21, m21), b12 = __dmul_rn(m21, m22), b22 = __dmul_rn(m22, m22);
  const double c11 = __dmul_rn(m11, m21), c22 = __dmul_rn(m12, m22);
  const double c12 = fma(m12, m21, __dmul_rn(m11, m22)), det = fma(-m12, m21, __dmul_rn(m11, m22));
  const double T11 = fma(a22, R22, fma(2.0 * a12, R12, __dmul_rn(a11, R11)));
  const double T22 = fma(b22, R22, fma(2.0 * b12, R12, __dmul_rn(b11, R11)));
  const double T12 = fma(c22, R22, fma(c12, R12, __dmul_rn(c11, R11)));
  S[0] = __dadd_rn(T11, T22);
  S[1] = __dadd_rn(T11, -T22);
  S[2] = 2.0 * T12;
  S[3] = __dmul_rn(det, S[3]);
}

struct PolState {
  double f1[4], f2[4];  // transverse legs, contravariant MKS components
  double S[4];          // invariant Stokes I/nu^3 ... in the (f1, f2) basis
  double tau, tauF;
};

// What the plasma operator needs once the tetrad has been dealt with: the fluid scalars, the frequency, the angle,
// and the 2x2 projection of the carried legs on the new ones.  Splitting the operator here lets the kernel finish
// the parallel transport of the new legs before the (register-hungry) coefficient and 4x4 step run.
struct PlasmaFrame {
  double ne, Th, B, cosT, nu;
  double m11, m12, m21, m22;     // M_{a'a} = e^(a')_mu f_a^mu
  double j[4], al[4], rh[3];     // slab only (cgs)
};

// Plasma state and plasma-frame tetrad at (X, K): what one step's plasma operator needs and what does NOT depend on
// the polarization state carried along the ray -- the two transverse legs e_(1), e_(2) (contravariant and covariant
// MKS components) and the fluid scalars, local frequency and pitch angle in F.  Returns false where there is no plasma.
// `lane` (model sweep only, else nullptr): the lane's own parameter set -- AdafParams, or GridScales overriding the four
// scale numbers of the shared GridParams.
template <int MODEL, bool SCALARS = true>
__device__ __forceinline__ bool plasma_tetrad(const Geom& G, const void* model, const void* lane, const Units& U, const double X[4],
                                              const double K[4], const Point& p, const Sym7& g, const Inv6& gi,
                                              const double* prim /* grid model: from grid_gather */, double e1[4], double e2[4],
                                              double e1c[4], double e2c[4], PlasmaFrame& F) {
  Plasma P;
  bool present;
  if (MODEL == MODEL_ADAF) present = plasma_adaf<SCALARS>(G, *(const AdafParams*)(lane ? lane : model), X, p, g, gi, P);
  else if (MODEL == MODEL_SLAB) present = plasma_slab(G, *(const SlabParams*)model, X, p, g, P);
  else {
    const GridParams& M = *(const GridParams*)model;
    if (lane) present = grid_state(G, M, *(const GridScales*)lane, prim, p, g, gi, P);
    else { const GridScales S = {M.ne_unit, M.B_unit, M.Rlow, M.Rhigh}; present = grid_state(G, M, S, prim, p, g, gi, P); }
  }
  if (!present) return false;

  double kcov[4], ucov[4];
  g.mul(K, kcov);
  g.mul(P.u, ucov);
  const double om = -dot4(kcov, P.u);
  if (!(om > 0.0)) return false;
  double e3[4], e3c[4];
  const double iom = ip_rcp(om);
#pragma unroll
  for (int m = 0; m < 4; ++m) e3[m] = K[m] * iom - P.u[m];
  g.mul(e3, e3c);
  const double n3 = dot4(e3c, e3);
  if (!(n3 > 1e-280)) return false;
  const double i3 = ip_rsqrt(n3);
#pragma unroll
  for (int m = 0; m < 4; ++m) { e3[m] *= i3; e3c[m] *= i3; }
  const double be3 = dot4(e3c, P.b);
#pragma unroll
  for (int m = 0; m < 4; ++m) e2[m] = P.b[m] - be3 * e3[m];
  g.mul(e2, e2c);
  const double n2 = dot4(e2c, e2);
  if (!(n2 > 1e-280)) return false;
  const double i2 = ip_rsqrt(n2);
#pragma unroll
  for (int m = 0; m < 4; ++m) { e2[m] *= i2; e2c[m] *= i2; }
  levi4(ucov, e2c, e3c, e1);
  const double isg = ip_rcp(p.sqrtmg);
#pragma unroll
  for (int m = 0; m < 4; ++m) e1[m] *= isg;
  g.mul(e1, e1c);

  F.nu = om * U.nu_obs;
  F.ne = P.ne; F.Th = P.Th; F.B = P.B;
  if (MODEL == MODEL_SLAB) {
#pragma unroll
    for (int i = 0; i < 4; ++i) { F.j[i] = P.j[i]; F.al[i] = P.al[i]; }
#pragma unroll
    for (int i = 0; i < 3; ++i) F.rh[i] = P.rh[i];
    F.cosT = 0.0;
  } else {
    double bcov[4];
    g.mul(P.b, bcov);
    F.cosT = fmin(1.0, fmax(-1.0, dot4(bcov, K) * iom * ip_rcp(P.B)));
  }
  return true;
}

// The same for the sequential kernels: on success the carried legs st.f1, st.f2 are REPLACED by the new transverse
// legs and F also holds the 2x2 projection of the old legs on the new ones.  Returns false where there is no plasma
// (nothing changed).
template <int MODEL>
__device__ __forceinline__ bool plasma_frame(const Geom& G, const void* model, const void* lane, const Units& U, const double X[4],
                                             const double K[4], const Point& p, const Sym7& g, const Inv6& gi,
                                             const double* prim /* grid model: from grid_gather */, PolState& st,
                                             PlasmaFrame& F) {
  double e1[4], e2[4], e1c[4], e2c[4];
  if (!plasma_tetrad<MODEL>(G, model, lane, U, X, K, p, g, gi, prim, e1, e2, e1c, e2c, F)) return false;
  F.m11 = dot4(e1c, st.f1); F.m12 = dot4(e1c, st.f2); F.m21 = dot4(e2c, st.f1); F.m22 = dot4(e2c, st.f2);
#pragma unroll
  for (int m = 0; m < 4; ++m) { st.f1[m] = e1[m]; st.f2[m] = e2[m]; }
  return true;
}

// Projection of the Stokes vector on the new legs, coefficients, analytic 4x4 step over affine length dl.
template <int MODEL>
__device__ __forceinline__ void plasma_apply(const Units& U, const PlasmaFrame& F, double dl, PolState& st) {
  const double ds = dl * U.dl_unit;
  stokes_congruence(F.m11, F.m12, F.m21, F.m22, st.S);
  double aI, rV;
  if (MODEL == MODEL_SLAB) {
    double ji[4], ai[4], ri[3];
    const double inu = ip_rcp(F.nu), inu2 = inu * inu;
#pragma unroll
    for (int i = 0; i < 4; ++i) { ji[i] = F.j[i] * inu2; ai[i] = F.al[i] * F.nu; }
#pragma unroll
    for (int i = 0; i < 3; ++i) ri[i] = F.rh[i] * F.nu;
    stokes_step(ai, ri, ds, ji, st.S);
    aI = ai[0]; rV = ri[2];
  } else {
    const Coeff c = synchrotron_invariant(F.ne, F.Th, F.B, F.cosT, F.nu);
    stokes_step_qv<MODEL != MODEL_GRID>(c.aI, c.aQ, c.aV, c.rQ, c.rV, ds, c.jI, c.jQ, c.jV, st.S);
    aI = c.aI; rV = c.rV;
  }
  st.tau += aI * ds;
  st.tauF += fabs(rV) * ds;
}

}  // namespace ipole
