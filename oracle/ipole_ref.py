"""ORACLE (test infrastructure): ctypes loader for oracle/libipole_ref.so.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It builds the library with `make -C oracle` when it is missing or stale.  It shares
nothing with the CUDA path (paper_2302_02733_b200/).
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


class Camera(C.Structure):
    _fields_ = [("spin", C.c_double), ("inclination_deg", C.c_double), ("r_cam", C.c_double), ("fov", C.c_double),
                ("nx", C.c_int32), ("ny", C.c_int32), ("freq_hz", C.c_double), ("mbh_msun", C.c_double),
                ("dsource_pc", C.c_double), ("eps", C.c_double), ("r_esc", C.c_double), ("stop_factor", C.c_double),
                ("max_steps", C.c_int32), ("hslope", C.c_double), ("flat_metric", C.c_int32)]


class Adaf(C.Structure):
    _fields_ = [("n0", C.c_double), ("p_n", C.c_double), ("Th0", C.c_double), ("p_T", C.c_double),
                ("B0", C.c_double), ("p_B", C.c_double)]


class Slab(C.Structure):
    _fields_ = [("H", C.c_double), ("profile", C.c_int32), ("psi_deg", C.c_double), ("j", C.c_double * 4),
                ("alpha", C.c_double * 4), ("rho", C.c_double * 3)]


class Grid(C.Structure):
    _fields_ = [("N1", C.c_int32), ("N2", C.c_int32), ("N3", C.c_int32), ("startx", C.c_double * 3),
                ("dx", C.c_double * 3), ("hslope", C.c_double), ("gam", C.c_double), ("M_unit", C.c_double),
                ("Rlow", C.c_double), ("Rhigh", C.c_double), ("r_out", C.c_double)]


def build():
    subprocess.run(["make", "-s", "-C", _HERE], check=True)


def lib():
    global _LIB
    if _LIB is None:
        build()
        L = C.CDLL(os.path.join(_HERE, "libipole_ref.so"))
        dp = C.POINTER(C.c_double)
        L.ipole_ref_init.argtypes = [C.POINTER(Camera), C.POINTER(C.c_void_p)]
        L.ipole_ref_load_model_adaf.argtypes = [C.c_void_p, C.POINTER(Adaf)]
        L.ipole_ref_load_model_slab.argtypes = [C.c_void_p, C.POINTER(Slab)]
        L.ipole_ref_load_model_grid.argtypes = [C.c_void_p, C.POINTER(Grid), C.POINTER(dp)]
        L.ipole_ref_make_pixels.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_int] + [C.c_void_p] * 8
        L.ipole_ref_free.argtypes = [C.c_void_p]
        L.ipole_ref_free.restype = None
        for name in ("gcov", "gcon", "dgcov", "conn"):
            f = getattr(L, "ipole_ref_" + name)
            f.argtypes = [C.c_double, C.c_double, C.c_int, dp, dp]
            f.restype = None
        L.ipole_ref_x2_of_theta.argtypes = [C.c_double, C.c_double]
        L.ipole_ref_x2_of_theta.restype = C.c_double
        L.ipole_ref_theta_of_x2.argtypes = [C.c_double, C.c_double]
        L.ipole_ref_theta_of_x2.restype = C.c_double
        L.ipole_ref_isco.argtypes = [C.c_double]
        L.ipole_ref_isco.restype = C.c_double
        L.ipole_ref_camera_tetrad.argtypes = [C.c_void_p, dp, dp]
        L.ipole_ref_camera_ray.argtypes = [C.c_void_p, C.c_int, C.c_int, dp, dp]
        L.ipole_ref_camera_ray_ab.argtypes = [C.c_void_p, C.c_double, C.c_double, dp, dp]
        L.ipole_ref_trace.argtypes = [C.c_void_p, dp, dp, C.c_int, dp, dp, dp, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.ipole_ref_coefficients.argtypes = [C.c_double] * 5 + [dp]
        L.ipole_ref_coefficients.restype = None
        L.ipole_ref_bessel_kscaled.argtypes = [C.c_double, dp]
        L.ipole_ref_bessel_kscaled.restype = None
        L.ipole_ref_stokes_operator.argtypes = [dp, dp, C.c_double, dp, dp]
        L.ipole_ref_stokes_operator.restype = None
        L.ipole_ref_plasma.argtypes = [C.c_void_p, dp, dp]
        L.ipole_ref_plasma_tetrad.argtypes = [C.c_void_p, dp, dp, dp, dp, dp, dp]
        L.ipole_ref_transport_vacuum.argtypes = [C.c_void_p, C.c_int, dp, dp, dp, dp]
        L.ipole_ref_set_path_free.argtypes = [C.c_void_p, C.c_int]
        L.ipole_ref_set_unpolarized.argtypes = [C.c_void_p, C.c_int]
        L.ipole_ref_retrace.argtypes = [C.c_void_p, dp, dp, C.c_int, dp, dp, dp]
        L.ipole_ref_observer_tetrad.argtypes = [C.c_void_p, dp, dp]
        L.ipole_ref_total_steps.argtypes = [C.c_void_p]
        L.ipole_ref_total_steps.restype = C.c_int64
        L.ipole_ref_set_edf.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int]
        L.ipole_ref_coefficients_edf.argtypes = [C.c_int, C.c_double, C.c_int] + [C.c_double] * 5 + [dp]
        L.ipole_ref_coefficients_edf.restype = None
        L.ipole_ref_synchrotron_kernels.argtypes = [C.c_double, dp]
        L.ipole_ref_synchrotron_kernels.restype = None
        _LIB = L
    return _LIB


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _vec(v, n=4):
    a = np.ascontiguousarray(v, dtype=np.float64)
    assert a.size == n
    return a


def gcov(a, h, X, flat=0):
    out = np.zeros((4, 4)); lib().ipole_ref_gcov(a, h, flat, _dp(_vec(X)), _dp(out)); return out


def gcon(a, h, X, flat=0):
    out = np.zeros((4, 4)); lib().ipole_ref_gcon(a, h, flat, _dp(_vec(X)), _dp(out)); return out


def dgcov(a, h, X, flat=0):
    out = np.zeros((4, 4, 4)); lib().ipole_ref_dgcov(a, h, flat, _dp(_vec(X)), _dp(out)); return out


def conn(a, h, X, flat=0):
    out = np.zeros((4, 4, 4)); lib().ipole_ref_conn(a, h, flat, _dp(_vec(X)), _dp(out)); return out


def coefficients(ne, thetae, B, cosT, nu):
    out = np.zeros(8); lib().ipole_ref_coefficients(ne, thetae, B, cosT, nu, _dp(out)); return out


def coefficients_edf(kind, ne, thetae, B, cosT, nu, kappa=3.5, n_nodes=128):
    """(jI,jQ,jV,aI,aQ,aV,rQ,rV) with j, alpha integrated over the eDF (oracle/ref_edf.hpp): kind 1 Maxwell-Juettner, 2 kappa."""
    out = np.zeros(8)
    lib().ipole_ref_coefficients_edf(int(kind), float(kappa), int(n_nodes), ne, thetae, B, cosT, nu, _dp(out))
    return out


def synchrotron_kernels(x):
    """F(x), G(x), H(x) of the single-electron synchrotron power"""
    out = np.zeros(3); lib().ipole_ref_synchrotron_kernels(float(x), _dp(out)); return out


def bessel_kscaled(z):
    out = np.zeros(3); lib().ipole_ref_bessel_kscaled(z, _dp(out)); return out


def stokes_operator(alpha, rho, s):
    O = np.zeros((4, 4)); P = np.zeros((4, 4))
    lib().ipole_ref_stokes_operator(_dp(_vec(alpha)), _dp(_vec(rho, 3)), s, _dp(O), _dp(P))
    return O, P


class Ctx:
    """One oracle context: camera + model."""

    def __init__(self, **cam):
        c = Camera()
        for k, v in cam.items():
            setattr(c, k, v)
        self.cam = c
        self._h = C.c_void_p()
        rc = lib().ipole_ref_init(C.byref(c), C.byref(self._h))
        if rc != 0:
            raise ValueError("ipole_ref_init failed: %d" % rc)
        self._keep = None

    def close(self):
        if self._h:
            lib().ipole_ref_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def load_adaf(self, n0=1e6, p_n=-1.5, Th0=30.0, p_T=-1.0, B0=30.0, p_B=-1.25):
        p = Adaf(n0, p_n, Th0, p_T, B0, p_B)
        rc = lib().ipole_ref_load_model_adaf(self._h, C.byref(p))
        if rc != 0:
            raise ValueError("load_model_adaf failed: %d" % rc)

    def load_slab(self, H, j=(0, 0, 0, 0), alpha=(0, 0, 0, 0), rho=(0, 0, 0), psi_deg=0.0, profile=0):
        p = Slab()
        p.H = H; p.profile = profile; p.psi_deg = psi_deg
        p.j[:] = list(j); p.alpha[:] = list(alpha); p.rho[:] = list(rho)
        rc = lib().ipole_ref_load_model_slab(self._h, C.byref(p))
        if rc != 0:
            raise ValueError("load_model_slab failed: %d" % rc)

    def load_grid(self, desc, fields):
        g = Grid()
        g.N1, g.N2, g.N3 = desc["N1"], desc["N2"], desc["N3"]
        g.startx[:] = list(desc["startx"]); g.dx[:] = list(desc["dx"])
        for k in ("hslope", "gam", "M_unit", "Rlow", "Rhigh", "r_out"):
            setattr(g, k, desc[k])
        arrs = [np.ascontiguousarray(f, dtype=np.float64) for f in fields]
        ptrs = (C.POINTER(C.c_double) * 8)(*[_dp(a) for a in arrs])
        rc = lib().ipole_ref_load_model_grid(self._h, C.byref(g), ptrs)
        if rc != 0:
            raise ValueError("load_model_grid failed: %d" % rc)

    def make_pixels(self, pixels=None, nthreads=1):
        """Returns dict of arrays I,Q,U,V,tau,tauF (float64) and nsteps,nturn (int32) for the given flat pixel
        indices j*nx+i (all pixels, in order, when None)."""
        if pixels is None:
            n = self.cam.nx * self.cam.ny
            pp = None
        else:
            pix = np.ascontiguousarray(pixels, dtype=np.int64)
            n = pix.size
            pp = pix.ctypes.data_as(C.c_void_p)
        out = {k: np.zeros(n) for k in ("I", "Q", "U", "V", "tau", "tauF")}
        out["nsteps"] = np.zeros(n, dtype=np.int32)
        out["nturn"] = np.zeros(n, dtype=np.int32)
        args = [out[k].ctypes.data_as(C.c_void_p) for k in ("I", "Q", "U", "V", "tau", "tauF", "nsteps", "nturn")]
        rc = lib().ipole_ref_make_pixels(self._h, n, pp, int(nthreads), *args)
        if rc != 0:
            raise RuntimeError("ipole_ref_make_pixels failed: %d" % rc)
        return out

    def total_steps(self):
        return int(lib().ipole_ref_total_steps(self._h))

    def camera_tetrad(self):
        X = np.zeros(4); e = np.zeros((4, 4))
        lib().ipole_ref_camera_tetrad(self._h, _dp(X), _dp(e))
        return X, e

    def camera_ray(self, i, j):
        X = np.zeros(4); K = np.zeros(4)
        lib().ipole_ref_camera_ray(self._h, i, j, _dp(X), _dp(K))
        return X, K

    def camera_ray_ab(self, alpha, beta):
        X = np.zeros(4); K = np.zeros(4)
        lib().ipole_ref_camera_ray_ab(self._h, alpha, beta, _dp(X), _dp(K))
        return X, K

    def trace(self, X0, K0, cap=60000):
        X = np.zeros((cap + 1, 4)); K = np.zeros((cap + 1, 4)); dl = np.zeros(cap)
        nt = C.c_int32(); st = C.c_int32()
        n = lib().ipole_ref_trace(self._h, _dp(_vec(X0)), _dp(_vec(K0)), cap, _dp(X), _dp(K), _dp(dl), C.byref(nt), C.byref(st))
        if n < 0:
            raise RuntimeError("trace: cap too small, need %d" % -n)
        return X[:n + 1].copy(), K[:n + 1].copy(), dl[:n].copy(), nt.value, st.value

    def set_path_free(self, on=True):
        """PAPER.md:43 bidirectional variant: make_pixels re-integrates the geodesic forward instead of using a stored path."""
        rc = lib().ipole_ref_set_path_free(self._h, 1 if on else 0)
        if rc != 0:
            raise RuntimeError("set_path_free failed: %d" % rc)

    def set_edf(self, kind, kappa=3.5, n_nodes=128):
        """j, alpha by numerical integration over the eDF (0 thermal fits, 1 Maxwell-Juettner, 2 kappa)."""
        rc = lib().ipole_ref_set_edf(self._h, int(kind), float(kappa), int(n_nodes))
        if rc != 0:
            raise RuntimeError("set_edf failed: %d" % rc)

    def set_unpolarized(self, on=True):
        """Scalar transfer of I alone (oracle/ref_unpol.hpp)."""
        rc = lib().ipole_ref_set_unpolarized(self._h, 1 if on else 0)
        if rc != 0:
            raise RuntimeError("set_unpolarized failed: %d" % rc)

    def retrace(self, Xn, Kn, cap=60000):
        """Forward pass of the path-free variant from the far end (Xn, Kn): points 0..n (0 = far end), n step sizes."""
        X = np.zeros((cap + 1, 4)); K = np.zeros((cap + 1, 4)); dl = np.zeros(cap)
        n = lib().ipole_ref_retrace(self._h, _dp(_vec(Xn)), _dp(_vec(Kn)), cap, _dp(X), _dp(K), _dp(dl))
        if n < 0:
            raise RuntimeError("retrace failed: %d" % n)
        return X[:n + 1].copy(), K[:n + 1].copy(), dl[:n].copy()

    def observer_tetrad(self, X):
        e = np.zeros((4, 4))
        lib().ipole_ref_observer_tetrad(self._h, _dp(_vec(X)), _dp(e))
        return e

    def plasma(self, X):
        out = np.zeros(12)
        rc = lib().ipole_ref_plasma(self._h, _dp(_vec(X)), _dp(out))
        if rc != 0:
            raise RuntimeError("plasma failed: %d" % rc)
        return dict(present=bool(out[0]), ne=out[1], thetae=out[2], B=out[3], u=out[4:8].copy(), b=out[8:12].copy())

    def plasma_tetrad(self, X, K, u, b):
        ec = np.zeros((4, 4)); ev = np.zeros((4, 4))
        rc = lib().ipole_ref_plasma_tetrad(self._h, _dp(_vec(X)), _dp(_vec(K)), _dp(_vec(u)), _dp(_vec(b)), _dp(ec), _dp(ev))
        if rc != 0:
            raise RuntimeError("plasma_tetrad failed: %d" % rc)
        return ec, ev

    def transport_vacuum(self, X, K, dl, N):
        n = len(dl)
        Xc = np.ascontiguousarray(X, dtype=np.float64); Kc = np.ascontiguousarray(K, dtype=np.float64)
        dlc = np.ascontiguousarray(dl, dtype=np.float64)
        buf = np.zeros(32)
        Nc = np.asarray(N, dtype=np.complex128).reshape(16)
        buf[0::2] = Nc.real; buf[1::2] = Nc.imag
        rc = lib().ipole_ref_transport_vacuum(self._h, n, _dp(Xc), _dp(Kc), _dp(dlc), _dp(buf))
        if rc != 0:
            raise RuntimeError("transport_vacuum failed: %d" % rc)
        return (buf[0::2] + 1j * buf[1::2]).reshape(4, 4)
