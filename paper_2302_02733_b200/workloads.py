"""Seeded synthetic inputs shaped like the paper's two workloads (Table 1).

This module is the ONLY thing the CUDA path's tests/bench and the CPU oracle have in common: it produces
inputs (camera / model parameter dictionaries and the GRMHD-like grid arrays).  It holds none of the imaging
method's arithmetic (no geodesics, no transfer, no coefficients) and imports neither side.

Stand-ins (the paper's own inputs -- the Vos et al. 2022 ADAF and the Moscibrodzka et al. 2014 GRMHD slice --
are not available): BASELINE.json configs[0..4]; recipe in DESIGN.md section 5.
"""
import numpy as np

SPIN = 0.9375
SEED = 230202733

#: camera shared by all configs (BASELINE.json configs[0]); the grid configs inherit r_cam, fov, M, D, eps
CAMERA = dict(spin=SPIN, r_cam=1000.0, fov=40.0, freq_hz=230e9, mbh_msun=4.1e6, dsource_pc=8000.0,
              eps=0.01, r_esc=1000.0, stop_factor=1.05, max_steps=50000, flat_metric=0)

ADAF = dict(n0=1.0e6, p_n=-1.5, Th0=30.0, p_T=-1.0, B0=30.0, p_B=-1.25)

#: frozen after a one-off calibration against the oracle at 64x64 (total flux ~ 1 Jy at 230 GHz, i = 20 deg)
GRID_M_UNIT = 1.5e20


def camera(kind, n, freq_hz=230e9, **over):
    """kind 'adaf' (inclination 60 deg, hslope 1) or 'grid' (20 deg, hslope 0.3); n x n pixels."""
    c = dict(CAMERA)
    c.update(nx=int(n), ny=int(n), freq_hz=float(freq_hz))
    if kind == "adaf":
        c.update(inclination_deg=60.0, hslope=1.0)
    elif kind == "grid":
        c.update(inclination_deg=20.0, hslope=0.3)
    else:
        raise ValueError(kind)
    c.update(over)
    return c


def _theta(h, x2):
    return np.pi * x2 + 0.5 * (1.0 - h) * np.sin(2.0 * np.pi * x2)


def _dtheta(h, x2):
    return np.pi * (1.0 + (1.0 - h) * np.cos(2.0 * np.pi * x2))


def _fm_lnh(a, l, r, th):
    """Fishbone & Moncrief (1976) ln(enthalpy) up to a constant, Kerr spin a, constant l = u^t u_phi."""
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2.0 * r + a * a
    AA = (r * r + a * a) ** 2 - Del * a * a * s2
    W = Sig * Sig * Del / (AA * AA * s2)
    root = np.sqrt(1.0 + 4.0 * l * l * W)
    return 0.5 * np.log((1.0 + root) / (Sig * Del / AA)) - 0.5 * root - 2.0 * a * r * l / AA


def _fm_l(a, r):
    """l = u^t u_phi of the prograde circular equatorial geodesic at radius r (Bardeen, Press & Teukolsky 1972)."""
    d = r ** 1.5 - 3.0 * np.sqrt(r) + 2.0 * a
    return (r ** 1.5 + a) * (r * r - 2.0 * a * np.sqrt(r) + a * a) / (r ** 1.5 * d)


def _normal_clamped(seed, field, shape):
    """xi ~ N(0,1) clamped to +-4, one independent Philox stream per (seed, field); cell order is C order."""
    g = np.random.Generator(np.random.Philox(key=[seed, field]))
    return np.clip(g.standard_normal(size=shape), -4.0, 4.0)


def fm_torus_grid(N1=288, N2=128, N3=128, seed=SEED, a=SPIN, hslope=0.3, r_in=6.0, r_max=12.0, r_out=50.0,
                  kappa=1.0e-3, gam=4.0 / 3.0, beta_norm=100.0, u_scale=20.0, noise=0.05, dtype=np.float64):
    """GRMHD-like snapshot: Fishbone-Moncrief torus with a poloidal-loop field on a cell-centred MKS lattice.

    Returns (desc, fields): desc is the grid descriptor dictionary of ipole_load_model_grid, fields a float64
    array [8][N1][N2][N3] = rho, u, U1, U2, U3, B1, B2, B3 (code units; primitives as in HARM-like codes)."""
    with np.errstate(invalid="ignore", divide="ignore"):  # cells inside the horizon (Delta < 0) are masked below
        return _fm_torus_grid(N1, N2, N3, seed, a, hslope, r_in, r_max, r_out, kappa, gam, beta_norm, u_scale, noise, dtype)


def _fm_torus_grid(N1, N2, N3, seed, a, hslope, r_in, r_max, r_out, kappa, gam, beta_norm, u_scale, noise, dtype):
    rh = 1.0 + np.sqrt(1.0 - a * a)
    startx = np.array([np.log(0.9 * rh), 0.0, 0.0])
    dx = np.array([(np.log(r_out) - startx[0]) / N1, 1.0 / N2, 2.0 * np.pi / N3])
    l = float(_fm_l(a, r_max))

    def torus(x1, x2):
        """rho, u (un-normalised) on the 2-D meshgrid of x1, x2"""
        r = np.exp(x1)[:, None]
        th = _theta(hslope, x2)[None, :]
        th = np.clip(th, 1e-12, np.pi - 1e-12)
        lnh = _fm_lnh(a, l, r, th) - _fm_lnh(a, l, np.array(r_in), np.array(np.pi / 2))
        inside = (lnh > 0.0) & (r > r_in)
        hm1 = np.where(inside, np.expm1(np.where(inside, lnh, 0.0)), 0.0)
        rho = (hm1 * (gam - 1.0) / (kappa * gam)) ** (1.0 / (gam - 1.0))
        u = kappa * rho ** gam / (gam - 1.0)
        return rho, u, inside

    x1c = startx[0] + (np.arange(N1) + 0.5) * dx[0]
    x2c = startx[1] + (np.arange(N2) + 0.5) * dx[1]
    x1f = startx[0] + np.arange(N1 + 1) * dx[0]
    x2f = startx[1] + np.arange(N2 + 1) * dx[1]
    rho, u, inside = torus(x1c, x2c)
    rho_max = rho.max()
    rho /= rho_max
    u /= rho_max

    # geometry at cell centres (Kerr-Schild functions, axisymmetric)
    r = np.exp(x1c)[:, None]
    th = _theta(hslope, x2c)[None, :]
    dth = _dtheta(hslope, x2c)[None, :]
    s2 = np.sin(th) ** 2
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2.0 * r + a * a
    AA = (r * r + a * a) ** 2 - Del * a * a * s2
    f = 2.0 * r / Sig
    sqrtg = r * dth * Sig * np.sin(th)

    # rotation: FM velocity in Boyer-Lindquist, which for u^r = 0 equals the Kerr-Schild (t, phi) components
    W = Sig * Sig * Del / (AA * AA * s2)
    up2 = 0.5 * (-1.0 + np.sqrt(1.0 + 4.0 * l * l * W))
    ut = np.sqrt(1.0 + up2) * np.sqrt(AA / (Sig * Del))
    uphi = 2.0 * a * r * np.sqrt(1.0 + up2) / np.sqrt(AA * Sig * Del) + np.sqrt(Sig / AA) * np.sqrt(up2) / np.sin(th)
    # primitive velocity utilde^i = u^i + u^t alpha^2 g^{ti}: alpha^2 = 1/(1+f), g^{t X1} = f/r, g^{t X2} = g^{t X3} = 0
    U1 = np.where(inside, ut * f / ((1.0 + f) * r), 0.0)
    U2 = np.zeros_like(U1)
    U3 = np.where(inside, uphi, 0.0)

    # poloidal loop: A_phi = max(rho/rho_max - 0.2, 0) at cell corners, B^1 = -d_2 A/sqrt(-g), B^2 = d_1 A/sqrt(-g)
    rho_f, _, _ = torus(x1f, x2f)
    Aphi = np.maximum(rho_f / rho_max - 0.2, 0.0)
    B1 = -(Aphi[:-1, 1:] - Aphi[:-1, :-1] + Aphi[1:, 1:] - Aphi[1:, :-1]) / (2.0 * dx[1] * sqrtg)
    B2 = (Aphi[1:, :-1] + Aphi[1:, 1:] - Aphi[:-1, :-1] - Aphi[:-1, 1:]) / (2.0 * dx[0] * sqrtg)
    # normalise to max(p_gas)/max(p_mag) = beta_norm, p_mag = b^2/2 with b^2 = (B^2 + (B.u)^2)/(u^t)^2 where the
    # products use the spatial Kerr-Schild metric in MKS components
    g11 = (1.0 + f) * r * r
    g22 = Sig * dth * dth
    g01 = f * r
    g13 = -a * s2 * (1.0 + f) * r
    g33 = s2 * (Sig + a * a * s2 * (1.0 + f))
    g03 = -a * f * s2
    # four-velocity of this flow: u^{X1} = u^{X2} = 0 exactly
    u1 = np.zeros_like(U1); u3 = np.where(inside, uphi, 0.0); u0 = np.where(inside, ut, 1.0)
    Bu = B1 * (g01 * u0 + g11 * u1 + g13 * u3) + B2 * (g22 * 0.0)
    BB = g11 * B1 * B1 + g22 * B2 * B2
    bsq = (BB + Bu * Bu) / (u0 * u0)
    pg_max = ((gam - 1.0) * u).max()
    pm_max = 0.5 * bsq.max()
    bnorm = np.sqrt(pg_max / (beta_norm * pm_max))
    B1 *= bnorm
    B2 *= bnorm
    u = u * u_scale

    fields = np.empty((8, N1, N2, N3), dtype=dtype)
    planes = [rho, u, U1, U2, U3, B1, B2, np.zeros_like(B1)]
    for q, p2 in enumerate(planes):
        fields[q] = p2[:, :, None]
    if noise > 0.0:
        for q in (0, 1, 5, 6, 7):
            fields[q] *= 1.0 + noise * _normal_clamped(seed, q, (N1, N2, N3))
    desc = dict(N1=int(N1), N2=int(N2), N3=int(N3), startx=[float(v) for v in startx], dx=[float(v) for v in dx],
                hslope=float(hslope), gam=float(gam), M_unit=float(GRID_M_UNIT), Rlow=1.0, Rhigh=40.0, r_out=float(r_out))
    return desc, fields


def config(i):
    """BASELINE.json configs[i] -> dict(name, camera(s), model).  Grid arrays are generated on demand by the caller
    with fm_torus_grid(*config['grid_shape'])."""
    if i == 0:
        return dict(name="W1", model="adaf", cameras=[camera("adaf", 32)], adaf=dict(ADAF))
    if i == 1:
        return dict(name="W2", model="adaf", cameras=[camera("adaf", 256, 230e9), camera("adaf", 256, 345e9)], adaf=dict(ADAF))
    if i == 2:
        return dict(name="W3", model="grid", cameras=[camera("grid", 256)], grid_shape=(288, 128, 128))
    if i == 3:
        return dict(name="W4", model="grid", cameras=[camera("grid", 1024)], grid_shape=(576, 256, 256), maps=True)
    if i == 4:
        return dict(name="W5", model="both", cameras=[camera("adaf", 4096), camera("grid", 4096)], adaf=dict(ADAF),
                    grid_shape=(576, 256, 256))
    raise IndexError(i)
