/* ipole.h -- C ABI of the B200-native polarized GR ray-tracing hot path (libipole_b200.so).
 *
 * What it computes (arXiv:2302.02733; citations are /root/reference/PAPER.md lines):
 *   PAPER.md:35  "the code launches photons from the point of the camera and integrates a null geodesic
 *                 equation for every single pixel ... The step size of the integration is adaptive and
 *                 parameterized ... Once the geodesic integration is over and saved the covariant fully
 *                 polarized radiative-transfer equations are integrated along the geodesic toward the
 *                 observer ... [at] every single step ... evaluate emission, self-absorption and Faraday
 *                 coefficients" (Section 2.1)
 *   PAPER.md:37  "the polarization state of light is described in a coordinate frame using a coherency
 *                 matrix N^{alpha beta}" (Section 2.1)
 *   PAPER.md:33  parameters: spin, viewing angle, frequency, field of view, resolution (Section 2.1)
 *   PAPER.md:56  output: Stokes I,Q,U,V images (Table 1 caption)
 * The paper prints no equations; the readings taken are DESIGN.md section 3 (R-1 ... R-9).
 *
 * Conventions
 *   - every function returns 0 on success or a negative IPOLE_E* code; nothing is written on error.
 *   - no global state; one ipole_ctx is not thread-safe, distinct contexts are independent.
 *   - pointers marked "host or device" are classified with cudaPointerGetAttributes; device outputs stay
 *     on the device (no hidden D2H); host outputs are copied back and the call synchronises the stream.
 *   - the caller owns every buffer it passes; the library copies what it needs to keep (grid fields).
 *   - all work is enqueued on the context's CUDA stream (ipole_set_stream; default: the legacy stream).
 *   - there is NO CPU fallback: without a CUDA device ipole_init returns IPOLE_ECUDA.
 */
#ifndef IPOLE_H
#define IPOLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define IPOLE_OK        0
#define IPOLE_EINVAL   -1   /* NULL pointer or parameter out of range                                  */
#define IPOLE_ENOMODEL -2   /* ipole_make_image before any ipole_load_model_*                          */
#define IPOLE_ENOMEM   -3   /* host or device allocation failed                                        */
#define IPOLE_ECUDA    -4   /* a CUDA call failed; ipole_last_cuda_error(ctx) has the cudaError_t      */
#define IPOLE_ENOIMAGE -5   /* ipole_get_stats / ipole_get_ray_info before ipole_make_image            */
#define IPOLE_ETOOBIG  -6   /* a size beyond the fixed maximum of an entry point that may not allocate  */

typedef struct ipole_ctx ipole_ctx; /* opaque; owns every device buffer it allocates */

/* Camera and integration parameters (PAPER.md:33 parameter list; step parameter eps PAPER.md:35, :43). */
typedef struct {
  double  spin;            /* a, 0 <= a < 1                                                            */
  double  inclination_deg; /* polar angle of the camera, in (0,180)                                    */
  double  r_cam;           /* camera radius ("distance"), GM/c^2                                       */
  double  fov;             /* full width of the image x axis, GM/c^2; pixels are square                */
  int32_t nx, ny;          /* pixels along x (right) and y (up, toward the spin axis)                  */
  double  freq_hz;         /* observing frequency                                                      */
  double  mbh_msun;        /* black-hole mass, Msun   (0 => 4.1e6); sets the length unit               */
  double  dsource_pc;      /* source distance, parsec (0 => 8000); only used for the flux in Jy        */
  double  eps;             /* step parameter (0 => 0.01)                                               */
  double  r_esc;           /* escape radius (0 => r_cam)                                               */
  double  stop_factor;     /* inner stop at stop_factor * r_horizon (0 => 1.05)                        */
  int32_t max_steps;       /* per-ray step limit (0 => 50000)                                          */
  double  hslope;          /* h of theta(X2) = pi X2 + (1-h)/2 sin(2 pi X2) (0 => 1)                   */
  int32_t flat_metric;     /* test switch: mass term off (Minkowski in the same coordinates)           */
} ipole_camera;

/* Analytic ADAF-like flow (BASELINE.json configs[0]): n_e = n0 r^p_n [cm^-3], Theta_e = Th0 r^p_T,
 * B = B0 r^p_B [G] purely toroidal; Keplerian outside the ISCO, E=1, L=0 free fall inside. */
typedef struct { double n0, p_n, Th0, p_T, B0, p_B; } ipole_adaf_params;

/* Test model: constant cgs coefficients in a slab |r cos(theta)| < H around the equatorial plane. */
typedef struct {
  double  H;        /* half thickness, GM/c^2 (> 0)                                                    */
  int32_t profile;  /* 0 top hat; 1 Gaussian weight exp(-z^2 / (2 H^2)) on every coefficient           */
  double  psi_deg;  /* field direction cos(psi) x^ + sin(psi) y^ in Cartesian Kerr-Schild axes         */
  double  j[4];     /* jI,jQ,jU,jV  erg s^-1 cm^-3 Hz^-1 sr^-1, plasma frame, at freq_hz               */
  double  alpha[4]; /* aI,aQ,aU,aV  cm^-1                                                              */
  double  rho[3];   /* rQ,rU,rV     cm^-1                                                              */
} ipole_slab_params;

/* GRMHD-like snapshot on a cell-centred MKS lattice ("precomputed ... 3D arrays ... the code
 * interpolates the plasma quantities to the point at every single step"). Cell (i,j,k) is centred at
 * X^d = startx[d] + (idx_d + 1/2) dx[d]; plane element index (i*N2 + j)*N3 + k. */
typedef struct {
  int32_t N1, N2, N3;
  double  startx[3], dx[3];
  double  hslope;   /* must equal the camera's hslope                                                  */
  double  gam;      /* adiabatic index of the fluid                                                    */
  double  M_unit;   /* mass unit [g]: rho_cgs = rho * M_unit / L^3                                     */
  double  Rlow, Rhigh; /* electron temperature prescription R = (Rhigh beta^2 + Rlow)/(1+beta^2)       */
  double  r_out;    /* no plasma beyond this radius                                                    */
} ipole_grid_desc;

typedef struct {
  double  flux_jy[4];      /* sum over pixels of I,Q,U,V times the pixel solid angle, in Jy            */
  double  lp, cp;          /* sqrt(Q^2+U^2)/I and V/I of the sums                                      */
  int64_t total_steps;     /* geodesic steps of all rays                                               */
  int32_t max_steps_seen;  /* longest ray                                                              */
  int32_t path_cap;        /* S_cap used for the bulk pass (from the probe pass)                       */
  int64_t n_ring;          /* rays with >= 2 theta turning points ("photon ring", configs[4])          */
  int64_t n_maxstep;       /* rays that ended on the step limit                                        */
  int64_t n_long;          /* rays that overflowed S_cap and went through the long-ray pass            */
  int32_t n_batches;       /* ray batches of the bulk pass                                             */
  int32_t n_launches;      /* kernels launched by the last ipole_make_image                            */
  float   ms_probe, ms_geodesic, ms_transfer, ms_total; /* CUDA-event times of the last image (0 until
                              ipole_get_stats synchronises them)                                       */
  float   ms_long;         /* long-ray passes (geodesic + transfer) on the side stream; they overlap the
                              bulk batches, so this is not part of a sum that gives ms_total            */
  int64_t total_steps_forward; /* path-free variant: steps of the forward passes of all rays (else 0)     */
  float   ms_stepop, ms_apply; /* split transfer (ipole_set_transfer_split): the step-parallel operator pass and
                              the per-ray apply pass; both are part of ms_transfer                      */
  int64_t n_retry;         /* rays that outgrew the path slots of their batch (sized from the predicted step count of the
                              batch's longest ray) and were traced again with S_cap slots                  */
  int32_t n_lanes;         /* 2: the batches alternated between two streams (ipole_set_batch_overlap) -- kernels of
                              consecutive batches then run side by side, their event times overlap, and ms_geodesic +
                              ms_transfer exceeds ms_total; 1: one batch after the other                   */
  int32_t plan_reused;     /* 1: the image was scheduled from the plan of the previous call (ipole_set_plan_reuse): no
                              probe pass (ms_probe = 0), no read-back, the call returned without waiting for the GPU */
} ipole_stats;

/* Create a context. Computes the camera tetrad on the device. IPOLE_EINVAL on bad parameters. */
int  ipole_init(const ipole_camera* cam, ipole_ctx** out);
/* Replace the camera of an existing context (keeps the loaded model and the device buffers). */
int  ipole_set_camera(ipole_ctx*, const ipole_camera* cam);
/* cuda_stream is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = legacy stream. */
int  ipole_set_stream(ipole_ctx*, void* cuda_stream);
/* Tunables: path_bytes = memory for the stored paths (and operator records) of a batch in HBM (0 => 50% of free
 * memory, at most 96 GiB); sort_rays: 0 = pixel order, 1 = order rays by predicted step count, longest first, when the
 * image has >= 32768 rays (default), 2 = always run the probe pass and sort (tests).
 * A budget far too small for the call makes the slots shorter than most rays, every ray then takes the long-ray pass a
 * few at a time, and a call that would need more than 8192 kernel work queues that way (e.g. a 128^2 eDF image with
 * 128 MiB) returns IPOLE_EINVAL without rendering: give it room for at least a few hundred full-length slots
 * ((max_steps + 1) x 128 B each). */
int  ipole_set_options(ipole_ctx*, uint64_t path_bytes, int32_t sort_rays);
/* Path-free bidirectional variant, the paper's own GPU design (section 2.2: "The GPU code does this
 * integration in both directions, away from the observer ... and toward the observer ..., without saving the path in
 * both cases"; reading R-10 in DESIGN.md).  on != 0: ipole_make_image / ipole_make_pixels keep only
 * the end point of each backward pass (64 B per ray), then re-integrate every ray forward with one RK4 push per
 * step (step rule evaluated at the point the step starts from), each push followed by the transfer step over its
 * two end points, until r >= r_cam moving outward; Stokes are read in the observer tetrad built at that end point.
 * No path buffer is allocated and the whole image is one geodesic launch and one transfer launch.  nsteps / nturn
 * remain those of the backward pass; ipole_stats.total_steps_forward counts the forward steps.  The image differs
 * from the stored-path one at the level the integrator is not time-reversible (paper: "negligible").
 * on == 0 (default): stored path.  Returns IPOLE_EINVAL for a NULL context. */
int  ipole_set_path_free(ipole_ctx*, int32_t on);
/* Transfer as two kernels (default on; "at every single step ... evaluate emission, self-absorption and
 * Faraday coefficients at a given point": everything of a step except the coefficients' action on the four Stokes
 * numbers depends on the stored path alone).  on != 0: on the stored path, for the analytic flow, a step-parallel kernel
 * turns every path step into a 64-byte operator record (the projection of the carried polarization basis on the step's
 * plasma tetrad; ln r, the angle to the field, the frequency in the plasma frame, the step length), and a per-ray
 * kernel evaluates the coefficients from it and applies them, from the far end to the camera.  on == 0: the single
 * per-ray transfer kernel does both (also used, whatever this switch says, for the
 * slab and grid models, the grid and unpolarized sweeps, the path-free and unpolarized variants, long rays, and rays with a step that
 * crosses no plasma).  The two give the same image up to rounding.  on == 2 is a test mode: as 1, but every seventh
 * ray of a batch is handed to the single kernel as if it had such a step.  Returns IPOLE_EINVAL for a NULL context. */
int  ipole_set_transfer_split(ipole_ctx*, int32_t on);
/* Batches side by side (default on).  A 4096 x 4096 image is 25-31 G steps of 64 (+ 64) bytes and goes through HBM in
 * tens of batches (PAPER.md:43 is the paper's answer to the same memory limit).  Every kernel of
 * a batch is persistent and ends in a tail of milliseconds while its last rays finish.  on != 0: consecutive batches
 * alternate between two streams, each with half of the path memory, so that the next batch's kernels fill those tails.
 * on == 0: one batch after the other on the context's stream (then the per-stage times of ipole_get_stats add up to
 * ms_total; bench.py measures its per-kernel figures this way).  Same image either way, bit for bit (a ray's arithmetic
 * does not depend on its batch).  Images of one or two batches and the sweeps always run on one stream.  IPOLE_EINVAL for NULL. */
int  ipole_set_batch_overlap(ipole_ctx*, int32_t on);
/* Asynchronous images by plan reuse (default on).  To schedule an image the host needs four facts from the device: the
 * longest probe ray (S_cap), the populations of the step-count bins (slots per batch), which rays outgrew their slots and
 * which are longer than S_cap.  Reading them back costs a probe pass and several host-device synchronisations, during
 * which ipole_make_image blocks.  All four depend on the geodesics alone -- camera, spin, eps, image size, scheduling
 * options -- not on the plasma model or its parameters (the geodesic is integrated first, "saved", and the
 * transfer then runs along it).  on != 0: the context keeps them from the last full-image call (and the ray order and
 * the two ray lists on the device); the next ipole_make_image with the SAME camera, image size, options and (to 1.5 %)
 * memory budget is scheduled from them: no probe pass, no read-back, the retried and the long rays start at once on
 * the side stream.  With device outputs such a call only enqueues work and RETURNS WHILE THE GPU IS STILL RUNNING
 * (ipole_stats.plan_reused = 1); outputs are valid once the context's stream reaches that point (stream order, an
 * event, or ipole_get_stats, which synchronises).  The model may be reloaded or its parameters changed in between (a
 * time series of GRMHD slices, a parameter fit at fixed geometry).  Any other call in between, a changed camera, stream or
 * option, or a different amount of free memory falls back to the planning call, which blocks as before and records a
 * new plan.  The image is the same, bit for bit, either way.  Not used for pixel lists, sweeps, many-camera calls, the
 * path-free variant and eDF coefficients.  on == 0: every call plans afresh.  IPOLE_EINVAL for a NULL context. */
int  ipole_set_plan_reuse(ipole_ctx*, int32_t on);
/* Second physics workload (outlook: electron distribution functions "for which accurate prescriptions ... do
 * not exist and the integration of synchrotron emissivity over the electron energy distribution function requires
 * numerical integration during ray tracing"; the paper gives no formulas: reading R-13 in DESIGN.md).
 * kind 0 (default): the thermal fits.  kind 1: Maxwell-Juettner, n(gamma) = N gamma^2 beta exp(-gamma/Theta_e).  kind 2: kappa
 * distribution, n(gamma) = N gamma^2 beta [1 + (gamma-1)/(kappa w)]^-(kappa+1) with w = Theta_e of the plasma model.  For
 * kind != 0 every transfer step evaluates j_{I,Q,V} = C int n {F, G, (4 cot/3) H/gamma} dgamma and alpha_{I,Q,V} =
 * -(C/(2 m nu^2)) int {..} gamma^2 d/dgamma[n/gamma^2] dgamma (single-electron synchrotron kernels F, G, H; x = nu / nu_cr(gamma))
 * by the midpoint rule on n_nodes equal cells of ln x in [-16, 4] (gamma = sqrt(xs/x), xs = nu / ((3/2) nu_B sin(theta)):
 * the kernels are then constants of the nodes); N from int n dgamma = n_e by the midpoint rule on 512 cells of ln(gamma-1)
 * in [-16, 16]; rho_Q, rho_V stay thermal.  Supported for the analytic flow on the stored path (ipole_make_image, _pixels,
 * _image_adaptive); those calls return IPOLE_EINVAL for another model, the sweeps, the path-free or the unpolarized
 * variant while kind != 0.  Zero fields take the defaults kappa 3.5, n_nodes 128.  The call enqueues two small set-up
 * kernels (node constants, normalisation table) on the context's stream.
 * IPOLE_EINVAL: NULL, kind outside 0..2, kappa <= 1, n_nodes > 1024. */
typedef struct { int32_t kind; int32_t n_nodes; double kappa; } ipole_edf;
int  ipole_set_edf(ipole_ctx*, const ipole_edf*);
/* FP32 STUDY switch, not a product path ("further code acceleration may be also obtained by switching to single
 * precision calculations").  on != 0: the geodesics of the analytic-flow and slab models on the stored
 * path are integrated in single precision (k_geodesic_f32: same step rule and stop rules), their path records widened to
 * FP64, and the transfer runs on them in FP64 as usual -- a mixed-precision image whose error and speed
 * profiles/r2_fp32_study.md reports (bench.py --fp32-geodesic).  Ignored for the grid model, the path-free variant and
 * ipole_make_images_cameras.  Returns IPOLE_EINVAL for a NULL context. */
int  ipole_set_geodesic_fp32(ipole_ctx*, int32_t on);
/* Unpolarized transfer (the model-fitting loop makes "nonpolarized images"; polarized
 * transfer is "far more complex and computationally demanding"; reading R-12 in DESIGN.md).  on != 0: every image
 * entry (ipole_make_image, _pixels, _images_adaf, _images_grid, _image_adaptive) solves the scalar equation
 * d(I/nu^3)/dlambda = j_I/nu^2 - alpha_I nu (I/nu^3) exactly per step on the stored path, with the same midpoints,
 * plasma state, frequency, pitch angle and thermal synchrotron j_I, alpha_I as the polarized path; no tetrad, no
 * parallel transport, no Faraday coefficients.  I is written, Q = U = V = 0, tau as usual, tauF = 0.  This is not
 * Stokes I of the polarized solution (alpha_Q, alpha_V couple I to Q and V there).  Takes precedence over
 * ipole_set_path_free.  Returns IPOLE_EINVAL for a NULL context. */
int  ipole_set_unpolarized(ipole_ctx*, int32_t on);

int  ipole_load_model_adaf(ipole_ctx*, const ipole_adaf_params*);
int  ipole_load_model_slab(ipole_ctx*, const ipole_slab_params*);
/* fields[0..7] = rho,u,U1,U2,U3,B1,B2,B3, each N1*N2*N3 doubles, host or device (all eight alike). */
int  ipole_load_model_grid(ipole_ctx*, const ipole_grid_desc*, const double* const fields[8]);

/* One full-Stokes image: I,Q,U,V [ny][nx] row-major, specific intensity in erg s^-1 cm^-2 Hz^-1 sr^-1.
 * tau (absorption optical depth) and tauF (Faraday depth, int |rho_V| dl) are optional [ny][nx] maps.
 * All non-NULL outputs must be of one kind (all host or all device).
 * Blocking: the FIRST image of a camera plans its batches from a probe pass and reads a few counters back, so the call
 * blocks for most of the image; with device outputs it returns with the last kernels still in flight.  Further images
 * of the same camera are scheduled from that plan and the call returns at once (ipole_set_plan_reuse, default on).
 * Either way the outputs are valid in stream order on the context's stream. */
int  ipole_make_image(ipole_ctx*, double* I, double* Q, double* U, double* V, double* tau, double* tauF);
/* Same for a list of n flat pixel indices j*nx+i (device or host int64); outputs have n entries. Used for
 * sampled parity checks at resolutions whose full image the CPU oracle cannot afford. pixels == NULL means
 * all nx*ny pixels in order (= ipole_make_image). nsteps/nturn optional (int32; nturn bit 7 = step limit). */
int  ipole_make_pixels(ipole_ctx*, int64_t n, const int64_t* pixels, double* I, double* Q, double* U, double* V,
                       double* tau, double* tauF, int32_t* nsteps, int32_t* nturn);
/* Many small images for model fitting ("we run the ipole code up to 10,000,000 times ... images of
 * moderate (to low) resolution of 128 x 128"): n_models analytic-flow parameter sets, optionally each
 * at its own observing frequency freq_hz[m] (NULL: the camera's), seen by the context's camera.  The geodesics
 * depend on the camera and the spin only, so they are integrated and stored ONCE and the stored paths are walked once
 * per parameter set: work item (ray, model), the lanes of a warp share a ray.  Every image is what
 * ipole_load_model_adaf(models[m]) + ipole_make_image would give at freq_hz[m].
 * Outputs: I,Q,U,V (and optional tau, tauF) are [n_models][ny][nx], all host or all device, caller-owned;
 * flux_jy (nullable, host or device) is [n_models][4] = sums of I,Q,U,V times the pixel solid angle in Jy.
 * The model loaded in the context, if any, is left as it was; ipole_get_stats afterwards describes the shared
 * geodesic pass and the image of models[0].  The stored-path design is used whatever ipole_set_path_free says.
 * IPOLE_EINVAL: NULL arguments, n_models < 1, a non-positive frequency, a flat-metric camera, mixed host/device
 * outputs, nx*ny*n_models > 2^31-1. */
int  ipole_make_images_adaf(ipole_ctx*, int32_t n_models, const ipole_adaf_params* models, const double* freq_hz,
                            double* I, double* Q, double* U, double* V, double* tau, double* tauF, double* flux_jy);
/* The same for the grid model loaded in the context (IPOLE_ENOMODEL otherwise): each set replaces the mass unit and
 * the electron-temperature parameters of ipole_grid_desc, optionally at its own frequency -- the parameters a GRMHD
 * fit varies at fixed snapshot and viewing angle.  Every image is what ipole_load_model_grid with those three numbers
 * + ipole_make_image would give.  The lanes of a warp share a ray, so the eight-cell gather of a step is one
 * broadcast load for up to 32 sets.  IPOLE_EINVAL also for M_unit <= 0. */
typedef struct { double M_unit, Rlow, Rhigh; } ipole_grid_scales;
int  ipole_make_images_grid(ipole_ctx*, int32_t n_models, const ipole_grid_scales* sets, const double* freq_hz,
                            double* I, double* Q, double* U, double* V, double* tau, double* tauF, double* flux_jy);
/* Many small images whose GEOMETRY differs (the fitting loop also varies viewing angle and spin): n_cams
 * cameras seen through the model loaded in the context (analytic flow or grid), all in one pass of the pipeline -- one probe and sort over
 * the union of their rays, geodesic / operator / apply launches over batches of that union -- so that 128 x 128 images
 * fill the GPU although each has only 16 k rays.  Every image is what ipole_set_camera(cams[k]) + ipole_make_image
 * would give.  The cameras may differ in spin, inclination, distance, field of view, frequency, mass, source distance,
 * escape radius and stop factor; they must agree in nx, ny, eps, max_steps and hslope, and none may be a flat-metric
 * camera.  The flow's ISCO follows each camera's spin.  Outputs I,Q,U,V (optional tau, tauF) are [n_cams][ny][nx], all
 * host or all device; flux_jy (nullable, host or device) is [n_cams][4].  The context's own camera and model are left
 * as they were; ipole_get_stats afterwards describes the union of the rays.  Works with ipole_set_edf; uses the split
 * transfer whatever ipole_set_transfer_split says.
 * Grid model: a grid was computed in one spacetime and scaled with one mass, so its cameras must ALSO share spin, mass
 * and hslope with the context's camera (the one the grid was loaded under); they differ in inclination, azimuth, field
 * of view, frequency, distance and source distance.  The geodesic kernel marks plasma-contact ranges per ray as for a
 * single camera; the lockstep transfer kernel takes frequency, length unit and the camera's transverse legs from each
 * ray's own camera.
 * IPOLE_ENOMODEL without a model, IPOLE_EINVAL for the slab model, for cameras that disagree in the fields above, for
 * the path-free or unpolarized variant, mixed host/device outputs, nx*ny*n_cams > 2^31-1. */
int  ipole_make_images_cameras(ipole_ctx*, int32_t n_cams, const ipole_camera* cams, double* I, double* Q, double* U, double* V,
                               double* tau, double* tauF, double* flux_jy);
/* Adaptive ray tracing ("another factor of 10 with adaptive ray tracing which reduces the number of light
 * rays to follow"; the paper gives no algorithm: reading R-11 in DESIGN.md).  Dyadic lattice levels
 * l = 0..levels of stride 2^(levels-l) (plus the last row and column): level 0 and 1 are traced everywhere; from then
 * on a new lattice point is traced only if it lies in a cell whose already traced points differ from the bilinear
 * interpolation of the cell's corners by more than rel_tol*|I| + abs_tol in some Stokes parameter (a cell narrower
 * than the stride, which gained no point at a level, keeps its flag), and is bilinearly interpolated otherwise.  The per-ray kernels are those of ipole_make_image (stored path or path-free as set).
 * I,Q,U,V: [ny][nx], all host or all device.  state (nullable, host or device): [ny][nx] bytes, 1 = traced,
 * 2 = interpolated.  info (nullable) is filled on return.  The call synchronises the stream once per level.
 * IPOLE_EINVAL: NULL outputs, levels outside 1..12, negative tolerances, an image with fewer than 2 pixels in x or y,
 * mixed host/device outputs. */
typedef struct {
  int64_t n_traced;            /* rays followed, all levels                                  */
  int64_t n_traced_level[16];  /* per level 0..levels                                        */
  int64_t total_steps;         /* geodesic steps of those rays                               */
  double  flux_jy[4];          /* sums of I,Q,U,V of the finished image times the pixel solid angle, Jy */
  float   ms_total;            /* CUDA-event time of the whole call (without the final copies to host buffers) */
  int32_t n_launches;          /* kernels launched                                           */
} ipole_adaptive_info;
int  ipole_make_image_adaptive(ipole_ctx*, int32_t levels, double rel_tol, double abs_tol, double* I, double* Q, double* U,
                               double* V, uint8_t* state, ipole_adaptive_info* info);
/* Per-ray step count and theta-turning-point count (bit 7 set: ended on max_steps) of the last image,
 * [ny][nx] or n entries; host or device; either may be NULL. */
int  ipole_get_ray_info(ipole_ctx*, int32_t* nsteps, int32_t* nturn);
/* Synchronises the stream and fills the statistics of the last image. */
int  ipole_get_stats(ipole_ctx*, ipole_stats*);

/* Totals of an image WITHOUT ANY ALLOCATION ("flux, polarization fractions"; the paper's images
 * are compared through their total flux and net polarization, Fig. 1) -- for callers that cannot call
 * cudaMalloc: code under CUDA graph capture, serving loops, harnesses that forbid it.  The same reduction as the one
 * ipole_make_image ends with, but its block partials live in a fixed array in the library's device image
 * (`static __device__`, 32 KiB; every GPU that loads the library holds it until the process exits) instead of a
 * cudaMalloc'ed buffer.  This call makes no cudaMalloc / cudaFree and calls no allocating library routine, does not
 * synchronise, and works on any four planes the caller has (not only the last image of the context).
 *   n            pixels, 1 <= n <= IPOLE_TOTALS_STATIC_MAX_PIXELS (4096 x 4096); more: IPOLE_ETOOBIG, nothing launched
 *   I, Q, U, V   DEVICE pointers, n doubles each, caller-owned, read only
 *   out6         DEVICE pointer, 6 doubles, caller-owned: sum of I, Q, U, V times the pixel solid angle of the
 *                context's camera in Jy (as ipole_stats.flux_jy), then lp = sqrt(Q^2+U^2)/I and cp = V/I of the sums
 * Two kernels on the context's stream (ipole_set_stream); the result is ready when the stream reaches that point.
 * The summation order is fixed (blocks of 16 384 pixels, folded in index order): a given image gives the same bits
 * every time; against ipole_stats.flux_jy, whose blocks are shaped differently, it agrees to rounding (~1e-15 rel.).
 * ALL CALLS SHARE THE ARRAY -- every context, every stream, every thread of the process on that GPU.  It keeps the
 * last call's contents; nothing in it has to start at zero (each call writes every partial it later reads).  Two calls
 * whose kernels overlap on the GPU (different streams or contexts without an ordering between them) RACE on it and
 * both results are undefined: order such calls with events, or keep them on one stream.
 * IPOLE_EINVAL: NULL argument, n < 1.  IPOLE_ECUDA: the array's device address could not be obtained at ipole_init
 * (cudaGetSymbolAddress; ipole_last_cuda_error has the code) or a launch failed. */
#define IPOLE_TOTALS_STATIC_MAX_PIXELS 16777216
int  ipole_image_totals_static(ipole_ctx*, int64_t n, const double* I, const double* Q, const double* U, const double* V,
                               double* out6);

/* ---- stages, exposed so that tests can check each against the oracle on its own ---- */
/* Camera tetrad: Xcam[4], e[a][mu] (16 doubles) to host memory. */
int  ipole_get_camera_tetrad(ipole_ctx*, double Xcam[4], double e[16]);
/* Trace the geodesic of pixel (i,j) on the device and return its stored path to HOST arrays:
 * X [cap+1][4], K [cap+1][4], dl [cap]; returns the number of steps n >= 0, or a negative error code
 * (IPOLE_EINVAL if cap is too small; *needed is always set when non-NULL). */
int  ipole_trace_pixel(ipole_ctx*, int32_t i, int32_t j, int32_t cap, double* X, double* K, double* dl,
                       int32_t* nturn, int32_t* status, int32_t* needed);
/* Device evaluation of the building blocks at n points (host arrays in and out):
 *   conn:  X[n][4] -> A-contracted connection Gamma^l_{mn} (64 doubles per point, [l][m][n])
 *   coeff: (ne, thetae, B, cos_thetaB, nu)[n][5] -> (jI,jQ,jV,aI,aQ,aV,rQ,rV)[n][8] in cgs
 *   stokes_step: (alpha[4], rho[3], s, S0[4], J[4])[n][16] -> S(s)[n][4] = O(s) S0 + P(s) J
 *   bessel: z[n] -> (e^z K0, e^z K1, e^z K2)[n][3] */
int  ipole_eval_connection(ipole_ctx*, int64_t n, const double* X, double* Gamma);
int  ipole_eval_coefficients(ipole_ctx*, int64_t n, const double* in5, double* out8);
/* as coeff, with j and alpha of the context's electron distribution (ipole_set_edf) */
int  ipole_eval_coefficients_edf(ipole_ctx*, int64_t n, const double* in5, double* out8);
int  ipole_eval_stokes_step(ipole_ctx*, int64_t n, const double* in16, double* out4);
int  ipole_eval_bessel(ipole_ctx*, int64_t n, const double* z, double* out3);
/* The branch-free elementary functions of the hot loops (csrc/fpmath.cuh) at n points x (host):
 * out[n][8] = exp(x), expm1(x), ln|x|, sin(x), cos(x), 1/x, 1/sqrt|x|, sqrt|x|.  Domains: see fpmath.cuh. */
int  ipole_eval_math(ipole_ctx*, int64_t n, const double* x, double* out8);
/* Plasma state of the loaded model at n points X[n][4] (host): out[n][12] = present, ne, thetae, B, u[4], b[4]. */
int  ipole_eval_plasma(ipole_ctx*, int64_t n, const double* X, double* out12);

/* FP64 FMA micro-benchmark (a chain-free DFMA loop on every SM) used as the measured ALU roofline
 * denominator: returns achieved TFLOP/s in *tflops and the kernel time in *ms. */
int  ipole_measure_fp64_peak(ipole_ctx*, double* tflops, float* ms);

int  ipole_last_cuda_error(const ipole_ctx*);  /* cudaError_t of the last failed CUDA call, 0 if none;
                                                * IPOLE_DEBUG=1 in the environment: its source line and text go to stderr */
void ipole_free(ipole_ctx*);
const char* ipole_strerror(int code);
const char* ipole_version(void);

#ifdef __cplusplus
}
#endif
#endif
