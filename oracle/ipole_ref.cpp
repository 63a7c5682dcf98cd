// ORACLE (test infrastructure): C interface of the CPU reference, see ipole_ref.h.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
#include "ipole_ref.h"
#include <atomic>
#include <thread>
#include <vector>
#include <new>
#include "ref_metric.hpp"
#include "ref_geodesic.hpp"
#include "ref_coeff.hpp"
#include "ref_stokes_op.hpp"
#include "ref_plasma.hpp"
#include "ref_transfer.hpp"
#include "ref_pathfree.hpp"
#include "ref_unpol.hpp"

using namespace iref;

struct ipole_ref_ctx {
  Camera cam;
  Units units;
  Model model;
  std::atomic<int64_t> total_steps{0};
  int path_free = 0;   // 1: PAPER.md:43 bidirectional variant (ref_pathfree.hpp)
  int unpolarized = 0; // 1: scalar transfer of I alone (ref_unpol.hpp); takes precedence over path_free
};

static Geom mkgeom(double a, double h, int flat) { Geom G; G.a = a; G.hslope = h; G.flat = flat; return G; }

extern "C" {

int ipole_ref_init(const ipole_ref_camera* c, ipole_ref_ctx** out) {
  if (!c || !out) return -1;
  if (!(c->spin >= 0.0 && c->spin < 1.0) || !(c->inclination_deg > 0.0 && c->inclination_deg < 180.0)
      || !(c->r_cam > 0.0) || !(c->fov > 0.0) || c->nx <= 0 || c->ny <= 0 || !(c->freq_hz > 0.0))
    return -1;
  ipole_ref_ctx* x = new (std::nothrow) ipole_ref_ctx();
  if (!x) return -3;
  x->cam.geom = mkgeom(c->spin, c->hslope > 0.0 ? c->hslope : 1.0, c->flat_metric);
  x->cam.r_cam = c->r_cam;
  x->cam.fov = c->fov;
  x->cam.inclination_deg = c->inclination_deg;
  x->cam.nx = c->nx; x->cam.ny = c->ny;
  x->cam.eps = c->eps > 0.0 ? c->eps : 0.01;
  x->cam.r_esc = c->r_esc > 0.0 ? c->r_esc : c->r_cam;
  x->cam.stop_factor = c->stop_factor > 0.0 ? c->stop_factor : 1.05;
  x->cam.max_steps = c->max_steps > 0 ? c->max_steps : 50000;
  camera_setup(x->cam);
  const double M = (c->mbh_msun > 0.0 ? c->mbh_msun : 4.1e6) * MSUN;
  x->units.nu_obs = c->freq_hz;
  x->units.L_unit = GNEWT * M / (CL * CL);
  x->units.D_cm = (c->dsource_pc > 0.0 ? c->dsource_pc : 8000.0) * PC;
  *out = x;
  return 0;
}

int ipole_ref_load_model_adaf(ipole_ref_ctx* x, const ipole_ref_adaf* p) {
  if (!x || !p) return -1;
  if (x->cam.geom.flat) return -1;  // the flow is defined on Kerr only
  x->model.kind = MODEL_ADAF;
  x->model.adaf = AdafParams{p->n0, p->p_n, p->Th0, p->p_T, p->B0, p->p_B};
  return 0;
}

int ipole_ref_load_model_slab(ipole_ref_ctx* x, const ipole_ref_slab* p) {
  if (!x || !p || !(p->H > 0.0)) return -1;
  x->model.kind = MODEL_SLAB;
  SlabParams& s = x->model.slab;
  s.H = p->H; s.profile = p->profile; s.psi_deg = p->psi_deg;
  for (int i = 0; i < 4; ++i) { s.j[i] = p->j[i]; s.alpha[i] = p->alpha[i]; }
  for (int i = 0; i < 3; ++i) s.rho[i] = p->rho[i];
  return 0;
}

int ipole_ref_load_model_grid(ipole_ref_ctx* x, const ipole_ref_grid* p, const double* const fields[8]) {
  if (!x || !p || !fields) return -1;
  if (p->N1 < 1 || p->N2 < 1 || p->N3 < 1) return -1;
  if (p->hslope != x->cam.geom.hslope) return -1;  // camera and grid must share the coordinate map
  GridParams& g = x->model.grid;
  g.N1 = p->N1; g.N2 = p->N2; g.N3 = p->N3;
  for (int i = 0; i < 3; ++i) { g.startx[i] = p->startx[i]; g.dx[i] = p->dx[i]; }
  g.hslope = p->hslope; g.gam = p->gam; g.M_unit = p->M_unit; g.Rlow = p->Rlow; g.Rhigh = p->Rhigh; g.r_out = p->r_out;
  const size_t n = (size_t)p->N1 * p->N2 * p->N3;
  for (int q = 0; q < 8; ++q) {
    if (!fields[q]) return -1;
    g.f[q].assign(fields[q], fields[q] + n);
  }
  x->model.kind = MODEL_GRID;
  return 0;
}

static void one_pixel(ipole_ref_ctx* x, int64_t pix, double out[6], int32_t* nsteps, int32_t* nturn) {
  const Camera& C = x->cam;
  const int i = (int)(pix % C.nx), j = (int)(pix / C.nx);
  double X[4], K[4];
  camera_ray(C, i, j, X, K);
  Path path;
  trace(C, X, K, path);
  cplx N[4][4];
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) N[a][b] = 0.0;
  double tau = 0.0, tauF = 0.0, S[4];
  if (x->unpolarized) {
    S[0] = transfer_unpolarized(C.geom, x->model, x->units, path, &tau);
    S[1] = S[2] = S[3] = 0.0;
  } else if (x->path_free) {
    const int n = (int)path.dl.size();
    double Xend[4];
    transfer_path_free(C, x->model, x->units, path.X[n].data(), path.K[n].data(), N, &tau, &tauF, Xend);
    end_point_stokes(C, Xend, N, S);
  } else {
    transfer_along_path(C.geom, x->model, x->units, path, N, &tau, &tauF);
    camera_stokes(C.geom, C, N, S);
  }
  const double nu3 = x->units.nu_obs * x->units.nu_obs * x->units.nu_obs;
  for (int q = 0; q < 4; ++q) out[q] = S[q] * nu3;
  out[4] = tau; out[5] = tauF;
  *nsteps = (int32_t)path.dl.size();
  *nturn = path.nturn | (path.status == 3 ? 0x80 : 0);
}

int ipole_ref_make_pixels(ipole_ref_ctx* x, int64_t n, const int64_t* pixels, int nthreads, double* I, double* Q,
                          double* U, double* V, double* tau, double* tauF, int32_t* nsteps, int32_t* nturn) {
  if (!x || !I || !Q || !U || !V) return -1;
  if (x->model.kind == MODEL_NONE) return -2;
  const int64_t npix = (int64_t)x->cam.nx * x->cam.ny;
  if (!pixels) n = npix;
  if (nthreads < 1) nthreads = 1;
  std::atomic<int64_t> next{0};
  std::atomic<int64_t> steps{0};
  auto worker = [&]() {
    for (;;) {
      const int64_t q = next.fetch_add(1);
      if (q >= n) break;
      const int64_t pix = pixels ? pixels[q] : q;
      double out[6] = {0, 0, 0, 0, 0, 0};
      int32_t ns = 0, nt = 0;
      if (pix >= 0 && pix < npix) one_pixel(x, pix, out, &ns, &nt);
      I[q] = out[0]; Q[q] = out[1]; U[q] = out[2]; V[q] = out[3];
      if (tau) tau[q] = out[4];
      if (tauF) tauF[q] = out[5];
      if (nsteps) nsteps[q] = ns;
      if (nturn) nturn[q] = nt;
      steps.fetch_add(ns);
    }
  };
  if (nthreads == 1) worker();
  else {
    std::vector<std::thread> th;
    for (int t = 0; t < nthreads; ++t) th.emplace_back(worker);
    for (auto& t : th) t.join();
  }
  x->total_steps = steps.load();
  return 0;
}

void ipole_ref_free(ipole_ref_ctx* x) { delete x; }

int ipole_ref_set_unpolarized(ipole_ref_ctx* x, int on) {
  if (!x) return -1;
  x->unpolarized = on ? 1 : 0;
  return 0;
}

int ipole_ref_set_path_free(ipole_ref_ctx* x, int on) {
  if (!x) return -1;
  x->path_free = on ? 1 : 0;
  return 0;
}

int ipole_ref_retrace(ipole_ref_ctx* x, const double Xn[4], const double Kn[4], int cap, double* X, double* K, double* dl) {
  if (!x || !Xn || !Kn || cap < 0 || !X || !K || !dl) return -1;
  Retrace r;
  double Xend[4];
  const int n = transfer_path_free(x->cam, x->model, x->units, Xn, Kn, nullptr, nullptr, nullptr, Xend, &r);
  if (n > cap) return -n;
  for (int s = 0; s <= n; ++s) for (int m = 0; m < 4; ++m) { X[4 * s + m] = r.X[s][m]; K[4 * s + m] = r.K[s][m]; }
  for (int s = 0; s < n; ++s) dl[s] = r.dl[s];
  return n;
}

int ipole_ref_observer_tetrad(ipole_ref_ctx* x, const double X[4], double e[16]) {
  if (!x || !X || !e) return -1;
  double t[4][4];
  observer_tetrad(x->cam.geom, X, t);
  for (int a = 0; a < 4; ++a) for (int m = 0; m < 4; ++m) e[4 * a + m] = t[a][m];
  return 0;
}

int64_t ipole_ref_total_steps(ipole_ref_ctx* x) { return x ? x->total_steps.load() : 0; }

// ---- pieces ----
void ipole_ref_gcov(double a, double h, int flat, const double X[4], double g[16]) {
  double m[4][4];
  gcov(mkgeom(a, h, flat), X, m);
  std::memcpy(g, m, sizeof m);
}
void ipole_ref_gcon(double a, double h, int flat, const double X[4], double g[16]) {
  double m[4][4];
  gcon(mkgeom(a, h, flat), X, m);
  std::memcpy(g, m, sizeof m);
}
void ipole_ref_dgcov(double a, double h, int flat, const double X[4], double dg[64]) {
  double g[4][4], d[4][4][4];
  gcov_and_derivs(mkgeom(a, h, flat), X, g, d);
  std::memcpy(dg, d, sizeof d);
}
void ipole_ref_conn(double a, double h, int flat, const double X[4], double Gm[64]) {
  double c[4][4][4];
  connection(mkgeom(a, h, flat), X, c);
  std::memcpy(Gm, c, sizeof c);
}
double ipole_ref_x2_of_theta(double h, double th) { return x2_of_theta(h, th); }
double ipole_ref_theta_of_x2(double h, double x2) { return theta_of_x2(h, x2); }
double ipole_ref_isco(double a) { return isco_radius(a); }

int ipole_ref_camera_tetrad(ipole_ref_ctx* x, double Xcam[4], double e[16]) {
  if (!x) return -1;
  std::memcpy(Xcam, x->cam.Xcam, 4 * sizeof(double));
  std::memcpy(e, x->cam.e, 16 * sizeof(double));
  return 0;
}
int ipole_ref_camera_ray(ipole_ref_ctx* x, int i, int j, double X[4], double K[4]) {
  if (!x) return -1;
  camera_ray(x->cam, i, j, X, K);
  return 0;
}
int ipole_ref_camera_ray_ab(ipole_ref_ctx* x, double alpha, double beta, double X[4], double K[4]) {
  if (!x) return -1;
  camera_ray_ab(x->cam, alpha, beta, X, K);
  return 0;
}

int ipole_ref_trace(ipole_ref_ctx* x, const double X0[4], const double K0[4], int cap, double* X, double* K,
                    double* dl, int32_t* nturn, int32_t* status) {
  if (!x) return 0;
  Path p;
  trace(x->cam, X0, K0, p);
  const int n = (int)p.dl.size();
  if (nturn) *nturn = p.nturn;
  if (status) *status = p.status;
  if (n > cap) return -n;
  for (int s = 0; s <= n; ++s)
    for (int m = 0; m < 4; ++m) {
      if (X) X[4 * s + m] = p.X[s][m];
      if (K) K[4 * s + m] = p.K[s][m];
    }
  if (dl) for (int s = 0; s < n; ++s) dl[s] = p.dl[s];
  return n;
}

void ipole_ref_coefficients(double ne, double thetae, double B, double cosT, double nu, double out[8]) {
  const CoeffCGS c = synchrotron_coefficients(ne, thetae, B, cosT, nu);
  out[0] = c.jI; out[1] = c.jQ; out[2] = c.jV; out[3] = c.aI; out[4] = c.aQ; out[5] = c.aV; out[6] = c.rQ; out[7] = c.rV;
}
void ipole_ref_bessel_kscaled(double z, double out[3]) { bessel_k_scaled(z, out); }

int ipole_ref_set_edf(ipole_ref_ctx* x, int kind, double kappa, int n_nodes) {
  if (!x || kind < 0 || kind > 2 || (kind == 2 && !(kappa > 1.0)) || (kind != 0 && n_nodes < 1)) return -1;
  x->model.edf.kind = kind; x->model.edf.kappa = kappa; x->model.edf.n_nodes = n_nodes;
  return 0;
}
void ipole_ref_coefficients_edf(int kind, double kappa, int n_nodes, double ne, double thetae, double B,
                                double cosT, double nu, double out[8]) {
  EdfParams E; E.kind = kind; E.kappa = kappa; E.n_nodes = n_nodes;
  const CoeffCGS c = synchrotron_coefficients_edf(E, ne, thetae, B, cosT, nu);
  out[0] = c.jI; out[1] = c.jQ; out[2] = c.jV; out[3] = c.aI; out[4] = c.aQ; out[5] = c.aV; out[6] = c.rQ; out[7] = c.rV;
}
void ipole_ref_synchrotron_kernels(double x, double out[3]) { synchrotron_kernels(x, out[0], out[1], out[2]); }

void ipole_ref_stokes_operator(const double alpha[4], const double rho[3], double s, double O[16], double P[16]) {
  double o[4][4], p[4][4];
  stokes_operator(alpha, rho, s, o, p);
  std::memcpy(O, o, sizeof o);
  std::memcpy(P, p, sizeof p);
}

int ipole_ref_plasma(ipole_ref_ctx* x, const double X[4], double out[12]) {
  if (!x) return -1;
  if (x->model.kind == MODEL_NONE) return -2;
  Plasma p;
  plasma_at(x->cam.geom, x->model, x->units, X, p);
  out[0] = p.present ? 1.0 : 0.0; out[1] = p.ne; out[2] = p.Th; out[3] = p.B;
  for (int m = 0; m < 4; ++m) { out[4 + m] = p.u[m]; out[8 + m] = p.b[m]; }
  return 0;
}

int ipole_ref_plasma_tetrad(ipole_ref_ctx* x, const double X[4], const double K[4], const double u[4],
                            const double b[4], double econ[16], double ecov[16]) {
  if (!x) return -1;
  double g[4][4], ec[4][4], ev[4][4], om;
  gcov(x->cam.geom, X, g);
  if (!plasma_tetrad(g, K, u, b, ec, ev, &om)) return -4;
  std::memcpy(econ, ec, sizeof ec);
  std::memcpy(ecov, ev, sizeof ev);
  return 0;
}

int ipole_ref_transport_vacuum(ipole_ref_ctx* x, int n, const double* X, const double* K, const double* dl,
                               double N[32]) {
  if (!x || n < 0) return -1;
  cplx M[4][4];
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) M[a][b] = cplx(N[2 * (4 * a + b)], N[2 * (4 * a + b) + 1]);
  for (int s = n - 1; s >= 0; --s) {
    double Xm[4], Km[4], P[4][4];
    for (int m = 0; m < 4; ++m) { Xm[m] = 0.5 * (X[4 * s + m] + X[4 * (s + 1) + m]); Km[m] = 0.5 * (K[4 * s + m] + K[4 * (s + 1) + m]); }
    transport_matrix(x->cam.geom, Xm, Km, 0.5 * dl[s], P);
    congruence(P, M);
    congruence(P, M);
  }
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) { N[2 * (4 * a + b)] = M[a][b].real(); N[2 * (4 * a + b) + 1] = M[a][b].imag(); }
  return 0;
}

}  // extern "C"
