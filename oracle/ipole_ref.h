/* ipole_ref.h -- C interface of the CPU ORACLE (test infrastructure, not product code).
 *
 * A plain, slow, single-threaded-per-ray FP64 restatement of the per-pixel hot path of the
 * ipole-style imager of arXiv:2302.02733 ("launches photons from the point of the
 * camera ... integrates a null geodesic equation for every single pixel ... Once the geodesic
 * integration is over and saved the covariant fully polarized radiative-transfer equations are
 * integrated along the geodesic toward the observer"; PAPER.md:37 coherency matrix in the coordinate
 * frame).  The paper prints no equations; the readings taken are listed in DESIGN.md section 3 and
 * follow SURVEY.md section 8(c) (c-1 ... c-8).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use
 * this library.  It shares no source, header, table or constant generator with the CUDA path.
 *
 * Parity pins (tests/test_oracle_*.py, all -m "not gpu"): G1-G6 metric/connection/geodesic/shadow,
 * T1-T9 transport/operator/slab/absorption/Faraday/invariant/coefficients/frequency powers, E1-E5 numerically
 * integrated eDF coefficients.  Parity unpinned: the paper's Fig. 1 / Table 1 images (figures and data sets are not
 * available); the shape of the Faraday-conversion fit f(X) away from X -> 0; j_V, alpha_V of the kappa distribution.
 */
#ifndef IPOLE_REF_H
#define IPOLE_REF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ipole_ref_ctx ipole_ref_ctx;

/* Same field order and meaning as ipole_camera in include/ipole.h (declared independently). */
typedef struct {
  double spin, inclination_deg, r_cam, fov;
  int32_t nx, ny;
  double freq_hz, mbh_msun, dsource_pc;
  double eps, r_esc, stop_factor;
  int32_t max_steps;
  double hslope;
  int32_t flat_metric;
} ipole_ref_camera;

typedef struct { double n0, p_n, Th0, p_T, B0, p_B; } ipole_ref_adaf;
typedef struct {
  double H;        /* half thickness in GM/c^2: plasma where |r cos(theta)| < H (profile 0)      */
  int32_t profile; /* 0 top-hat; 1 Gaussian weight exp(-z^2/(2 H^2)) on every coefficient       */
  double psi_deg;  /* field direction cos(psi) x^ + sin(psi) y^ (Cartesian)                      */
  double j[4];     /* jI,jQ,jU,jV  erg s^-1 cm^-3 Hz^-1 sr^-1 in the plasma frame at freq_hz     */
  double alpha[4]; /* aI,aQ,aU,aV  cm^-1                                                          */
  double rho[3];   /* rQ,rU,rV     cm^-1                                                          */
} ipole_ref_slab;
typedef struct {
  int32_t N1, N2, N3;
  double startx[3], dx[3];
  double hslope, gam, M_unit, Rlow, Rhigh, r_out;
} ipole_ref_grid;

/* ---- whole path (mirror of the product ABI) ---- */
int  ipole_ref_init(const ipole_ref_camera*, ipole_ref_ctx** out);
int  ipole_ref_load_model_adaf(ipole_ref_ctx*, const ipole_ref_adaf*);
int  ipole_ref_load_model_slab(ipole_ref_ctx*, const ipole_ref_slab*);
int  ipole_ref_load_model_grid(ipole_ref_ctx*, const ipole_ref_grid*, const double* const fields[8]);
/* pixels: n flat indices j*nx+i (NULL => all nx*ny in order); outputs have n entries each
 * (tau, tauF, nsteps, nturn nullable); nthreads host threads shard the pixel list. */
int  ipole_ref_make_pixels(ipole_ref_ctx*, int64_t n, const int64_t* pixels, int nthreads,
                           double* I, double* Q, double* U, double* V, double* tau, double* tauF,
                           int32_t* nsteps, int32_t* nturn);
void ipole_ref_free(ipole_ref_ctx*);
/* Path-free bidirectional variant (reading R-10 in ref_pathfree.hpp): when on, make_pixels keeps only
 * the end point of the backward pass and re-integrates forward to r >= r_cam, one transfer step per forward step;
 * Stokes are read in the observer tetrad at the forward end point.  nsteps/nturn stay those of the backward pass.
 * Pins PF1-PF5 (tests/test_oracle_pathfree.py). */
int  ipole_ref_set_path_free(ipole_ref_ctx*, int on);
/* Unpolarized transfer ("nonpolarized images"; reading R-12 in ref_unpol.hpp): make_pixels solves the
 * scalar equation for I alone on the stored path; Q = U = V = 0, tauF = 0.  Pins U1-U3 (tests/test_oracle_unpol.py). */
int  ipole_ref_set_unpolarized(ipole_ref_ctx*, int on);
/* The forward pass alone, from (Xn, Kn): returns its step count n, points 0..n (0 = far end) and the n step sizes;
 * -(needed) if cap is too small. */
int  ipole_ref_retrace(ipole_ref_ctx*, const double Xn[4], const double Kn[4], int cap,
                       double* X /*[cap+1][4]*/, double* K /*[cap+1][4]*/, double* dl /*[cap]*/);
/* Second physics workload (eDFs whose synchrotron emissivity "requires numerical integration during ray
 * tracing"; reading R-13 in ref_edf.hpp): kind 0 thermal fits (default), 1 Maxwell-Juettner, 2 kappa distribution with
 * width w = Theta_e; j_{I,Q,V} and alpha_{I,Q,V} by the midpoint rule on n_nodes cells in ln x, x = nu/nu_cr(gamma) (ref_edf.hpp);
 * rho_Q, rho_V stay thermal.  Pins E1-E5 (tests/test_oracle_edf.py).  Returns -1 on bad arguments. */
int  ipole_ref_set_edf(ipole_ref_ctx*, int kind, double kappa, int n_nodes);
/* the coefficient stage on its own: out = (jI,jQ,jV,aI,aQ,aV,rQ,rV), cgs, plasma frame */
void ipole_ref_coefficients_edf(int kind, double kappa, int n_nodes, double ne, double thetae, double B,
                                double cosT, double nu, double out[8]);
/* F(x) = x int_x^inf K_5/3, G(x) = x K_2/3(x), H(x) = x K_1/3(x) + int_x^inf K_1/3 */
void ipole_ref_synchrotron_kernels(double x, double out[3]);
/* ---- stage entries used by the pins (tests/test_oracle_*.py) ---- */
void ipole_ref_gcov(double a, double hslope, int flat, const double X[4], double g[16]);
void ipole_ref_gcon(double a, double hslope, int flat, const double X[4], double g[16]);
void ipole_ref_dgcov(double a, double hslope, int flat, const double X[4], double dg[64]);
void ipole_ref_conn(double a, double hslope, int flat, const double X[4], double Gamma[64]);
void ipole_ref_coefficients(double ne, double thetae, double B, double cosT, double nu, double out[8]);
void ipole_ref_bessel_kscaled(double z, double out[3]);
void ipole_ref_stokes_operator(const double alpha[4], const double rho[3], double s, double O[16], double P[16]);
int64_t ipole_ref_total_steps(ipole_ref_ctx*);                       /* geodesic steps of the last make_pixels */
int  ipole_ref_camera_tetrad(ipole_ref_ctx*, double Xcam[4], double e[16]);
int  ipole_ref_camera_ray(ipole_ref_ctx*, int i, int j, double X[4], double K[4]);
int  ipole_ref_camera_ray_ab(ipole_ref_ctx*, double alpha, double beta, double X[4], double K[4]);
/* backward geodesic from (X0, K0): points 0..n, step sizes, theta turning points, stop status (1 horizon, 2 escape,
 * 3 step limit); returns n or -(needed) if cap is too small */
int  ipole_ref_trace(ipole_ref_ctx*, const double X0[4], const double K0[4], int cap, double* X, double* K, double* dl,
                     int32_t* nturn, int32_t* status);
int  ipole_ref_plasma(ipole_ref_ctx*, const double X[4], double out[12]);   /* present, ne, thetae, B, u[4], b[4] */
int  ipole_ref_plasma_tetrad(ipole_ref_ctx*, const double X[4], const double K[4], const double u[4], const double b[4],
                             double econ[16], double ecov[16]);
/* vacuum transport of a complex tensor N (32 doubles, re/im interleaved) along n stored steps, far end -> camera */
int  ipole_ref_transport_vacuum(ipole_ref_ctx*, int n, const double* X, const double* K, const double* dl, double N[32]);
/* camera-type tetrad e[a][mu] at an arbitrary point (static observer, e3 from d_X1, e2 from -d_X2, e1 from d_X3) */
int  ipole_ref_observer_tetrad(ipole_ref_ctx*, const double X[4], double e[16]);

#ifdef __cplusplus
}
#endif
#endif
