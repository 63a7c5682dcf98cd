"""Thin ctypes binding of libipole_b200.so (the C ABI of include/ipole.h).

Argument marshalling only: every step of the hot path runs in the library's CUDA kernels.  PyTorch is used
for device memory and streams (outputs are torch CUDA tensors whose data_ptr() is handed to the library).
There is no CPU fallback: if the library is missing or no CUDA device is present this module raises.
It never imports anything under oracle/.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libipole_b200.so")
_LIB = None

OK, EINVAL, ENOMODEL, ENOMEM, ECUDA, ENOIMAGE, ETOOBIG = 0, -1, -2, -3, -4, -5, -6

#: every symbol include/ipole.h declares (checked by tests/test_abi.py)
SYMBOLS = ["ipole_init", "ipole_set_camera", "ipole_set_stream", "ipole_set_options", "ipole_set_path_free", "ipole_set_edf", "ipole_set_geodesic_fp32", "ipole_set_transfer_split", "ipole_set_batch_overlap", "ipole_set_plan_reuse", "ipole_image_totals_static", "ipole_set_unpolarized", "ipole_load_model_adaf",
           "ipole_load_model_slab", "ipole_load_model_grid", "ipole_make_image", "ipole_make_pixels", "ipole_make_images_adaf", "ipole_make_images_grid", "ipole_make_images_cameras", "ipole_make_image_adaptive",
           "ipole_get_ray_info", "ipole_get_stats", "ipole_get_camera_tetrad", "ipole_trace_pixel",
           "ipole_eval_connection", "ipole_eval_coefficients", "ipole_eval_coefficients_edf", "ipole_eval_stokes_step", "ipole_eval_bessel",
           "ipole_eval_plasma", "ipole_eval_math", "ipole_measure_fp64_peak", "ipole_last_cuda_error", "ipole_free", "ipole_strerror",
           "ipole_version"]


class Camera(C.Structure):
    _fields_ = [("spin", C.c_double), ("inclination_deg", C.c_double), ("r_cam", C.c_double), ("fov", C.c_double),
                ("nx", C.c_int32), ("ny", C.c_int32), ("freq_hz", C.c_double), ("mbh_msun", C.c_double),
                ("dsource_pc", C.c_double), ("eps", C.c_double), ("r_esc", C.c_double), ("stop_factor", C.c_double),
                ("max_steps", C.c_int32), ("hslope", C.c_double), ("flat_metric", C.c_int32)]


class AdafParams(C.Structure):
    _fields_ = [("n0", C.c_double), ("p_n", C.c_double), ("Th0", C.c_double), ("p_T", C.c_double),
                ("B0", C.c_double), ("p_B", C.c_double)]


class SlabParams(C.Structure):
    _fields_ = [("H", C.c_double), ("profile", C.c_int32), ("psi_deg", C.c_double), ("j", C.c_double * 4),
                ("alpha", C.c_double * 4), ("rho", C.c_double * 3)]


class GridDesc(C.Structure):
    _fields_ = [("N1", C.c_int32), ("N2", C.c_int32), ("N3", C.c_int32), ("startx", C.c_double * 3),
                ("dx", C.c_double * 3), ("hslope", C.c_double), ("gam", C.c_double), ("M_unit", C.c_double),
                ("Rlow", C.c_double), ("Rhigh", C.c_double), ("r_out", C.c_double)]


class Stats(C.Structure):
    _fields_ = [("flux_jy", C.c_double * 4), ("lp", C.c_double), ("cp", C.c_double), ("total_steps", C.c_int64),
                ("max_steps_seen", C.c_int32), ("path_cap", C.c_int32), ("n_ring", C.c_int64),
                ("n_maxstep", C.c_int64), ("n_long", C.c_int64), ("n_batches", C.c_int32), ("n_launches", C.c_int32),
                ("ms_probe", C.c_float), ("ms_geodesic", C.c_float), ("ms_transfer", C.c_float), ("ms_total", C.c_float),
                ("ms_long", C.c_float), ("total_steps_forward", C.c_int64), ("ms_stepop", C.c_float), ("ms_apply", C.c_float), ("n_retry", C.c_int64),
                ("n_lanes", C.c_int32), ("plan_reused", C.c_int32)]


class Edf(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_nodes", C.c_int32), ("kappa", C.c_double)]


class GridScales(C.Structure):
    _fields_ = [("M_unit", C.c_double), ("Rlow", C.c_double), ("Rhigh", C.c_double)]


class AdaptiveInfo(C.Structure):
    _fields_ = [("n_traced", C.c_int64), ("n_traced_level", C.c_int64 * 16), ("total_steps", C.c_int64),
                ("flux_jy", C.c_double * 4), ("ms_total", C.c_float), ("n_launches", C.c_int32)]


class IpoleError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        super().__init__("%s failed: %d (%s)" % (what, code, lib().ipole_strerror(code).decode()))


def lib():
    """Load libipole_b200.so (built in-tree by __graft_entry__.build()).  Raises if it is missing."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, dp = C.c_void_p, C.POINTER(C.c_double)
        L.ipole_init.argtypes = [C.POINTER(Camera), C.POINTER(vp)]
        L.ipole_set_camera.argtypes = [vp, C.POINTER(Camera)]
        L.ipole_set_stream.argtypes = [vp, vp]
        L.ipole_set_options.argtypes = [vp, C.c_uint64, C.c_int32]
        L.ipole_set_path_free.argtypes = [vp, C.c_int32]
        L.ipole_set_unpolarized.argtypes = [vp, C.c_int32]
        L.ipole_set_transfer_split.argtypes = [vp, C.c_int32]
        L.ipole_set_batch_overlap.argtypes = [vp, C.c_int32]
        L.ipole_set_plan_reuse.argtypes = [vp, C.c_int32]
        L.ipole_image_totals_static.argtypes = [vp, C.c_int64, vp, vp, vp, vp, vp]
        L.ipole_set_geodesic_fp32.argtypes = [vp, C.c_int32]
        L.ipole_set_edf.argtypes = [vp, C.POINTER(Edf)]
        L.ipole_eval_coefficients_edf.argtypes = [vp, C.c_int64, dp, dp]
        L.ipole_load_model_adaf.argtypes = [vp, C.POINTER(AdafParams)]
        L.ipole_load_model_slab.argtypes = [vp, C.POINTER(SlabParams)]
        L.ipole_load_model_grid.argtypes = [vp, C.POINTER(GridDesc), C.POINTER(vp)]
        L.ipole_make_image.argtypes = [vp] + [vp] * 6
        L.ipole_make_pixels.argtypes = [vp, C.c_int64, vp] + [vp] * 8
        L.ipole_make_images_adaf.argtypes = [vp, C.c_int32, C.POINTER(AdafParams), vp] + [vp] * 7
        L.ipole_make_image_adaptive.argtypes = [vp, C.c_int32, C.c_double, C.c_double, vp, vp, vp, vp, vp, C.POINTER(AdaptiveInfo)]
        L.ipole_make_images_grid.argtypes = [vp, C.c_int32, C.POINTER(GridScales), vp] + [vp] * 7
        L.ipole_make_images_cameras.argtypes = [vp, C.c_int32, C.POINTER(Camera)] + [vp] * 7
        L.ipole_get_ray_info.argtypes = [vp, vp, vp]
        L.ipole_get_stats.argtypes = [vp, C.POINTER(Stats)]
        L.ipole_get_camera_tetrad.argtypes = [vp, dp, dp]
        L.ipole_trace_pixel.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, dp, dp, dp, C.POINTER(C.c_int32),
                                        C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        for name in ("connection", "coefficients", "stokes_step", "bessel", "plasma", "math"):
            getattr(L, "ipole_eval_" + name).argtypes = [vp, C.c_int64, dp, dp]
        L.ipole_measure_fp64_peak.argtypes = [vp, dp, C.POINTER(C.c_float)]
        L.ipole_last_cuda_error.argtypes = [vp]
        L.ipole_free.argtypes = [vp]
        L.ipole_free.restype = None
        L.ipole_strerror.argtypes = [C.c_int]
        L.ipole_strerror.restype = C.c_char_p
        L.ipole_version.restype = C.c_char_p
        _LIB = L
    return _LIB


def _chk(rc, what):
    if rc < 0:
        raise IpoleError(rc, what)
    return rc


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ptr(t):
    """data pointer of a torch tensor / numpy array / None"""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return C.c_void_p(t.ctypes.data)
    return C.c_void_p(t.data_ptr())


class Ipole:
    """One context: camera + plasma model on the current CUDA device."""

    def __init__(self, **cam):
        self.cam = Camera()
        for k, v in cam.items():
            setattr(self.cam, k, v)
        self._h = C.c_void_p()
        _chk(lib().ipole_init(C.byref(self.cam), C.byref(self._h)), "ipole_init")
        self._keep = None

    # -- lifetime --
    def close(self):
        if getattr(self, "_h", None):
            lib().ipole_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def nx(self):
        return self.cam.nx

    @property
    def ny(self):
        return self.cam.ny

    # -- configuration --
    def set_camera(self, **cam):
        for k, v in cam.items():
            setattr(self.cam, k, v)
        _chk(lib().ipole_set_camera(self._h, C.byref(self.cam)), "ipole_set_camera")

    def set_stream(self, stream=None):
        """stream: a torch.cuda.Stream (None: torch's current stream)."""
        import torch
        s = stream if stream is not None else torch.cuda.current_stream()
        _chk(lib().ipole_set_stream(self._h, C.c_void_p(s.cuda_stream)), "ipole_set_stream")

    def set_options(self, path_bytes=0, sort_rays=True):
        _chk(lib().ipole_set_options(self._h, int(path_bytes), int(sort_rays)), "ipole_set_options")

    def set_path_free(self, on=True):
        """Path-free bidirectional variant: no stored path, forward re-integration (include/ipole.h)."""
        _chk(lib().ipole_set_path_free(self._h, 1 if on else 0), "ipole_set_path_free")

    def set_geodesic_fp32(self, on=True):
        """FP32 study switch (include/ipole.h ipole_set_geodesic_fp32): geodesics in single precision."""
        _chk(lib().ipole_set_geodesic_fp32(self._h, 1 if on else 0), "ipole_set_geodesic_fp32")

    def set_plan_reuse(self, on=True):
        """Schedule an image from the previous call's plan when camera and options are unchanged: the call then does not
        block (include/ipole.h ipole_set_plan_reuse)."""
        _chk(lib().ipole_set_plan_reuse(self._h, int(on)), "ipole_set_plan_reuse")

    def set_batch_overlap(self, on=True):
        """Consecutive batches side by side on two streams (include/ipole.h ipole_set_batch_overlap)."""
        _chk(lib().ipole_set_batch_overlap(self._h, int(on)), "ipole_set_batch_overlap")

    def set_transfer_split(self, on=True):
        """Transfer as a step-parallel operator pass + a per-ray apply pass (include/ipole.h ipole_set_transfer_split)."""
        _chk(lib().ipole_set_transfer_split(self._h, int(on)), "ipole_set_transfer_split")

    def set_edf(self, kind, kappa=3.5, n_nodes=128):
        """Electron distribution of the coefficient step (include/ipole.h ipole_set_edf): 0 thermal fits,
        1 Maxwell-Juettner, 2 kappa; j and alpha by numerical integration over it."""
        e = Edf(int(kind), int(n_nodes), float(kappa))
        _chk(lib().ipole_set_edf(self._h, C.byref(e)), "ipole_set_edf")

    def set_unpolarized(self, on=True):
        """Unpolarized transfer of I alone (include/ipole.h ipole_set_unpolarized)."""
        _chk(lib().ipole_set_unpolarized(self._h, 1 if on else 0), "ipole_set_unpolarized")

    def load_adaf(self, n0=1e6, p_n=-1.5, Th0=30.0, p_T=-1.0, B0=30.0, p_B=-1.25):
        p = AdafParams(n0, p_n, Th0, p_T, B0, p_B)
        _chk(lib().ipole_load_model_adaf(self._h, C.byref(p)), "ipole_load_model_adaf")

    def load_slab(self, H, j=(0, 0, 0, 0), alpha=(0, 0, 0, 0), rho=(0, 0, 0), psi_deg=0.0, profile=0):
        p = SlabParams()
        p.H = H; p.profile = profile; p.psi_deg = psi_deg
        p.j[:] = list(j); p.alpha[:] = list(alpha); p.rho[:] = list(rho)
        _chk(lib().ipole_load_model_slab(self._h, C.byref(p)), "ipole_load_model_slab")

    def load_grid(self, desc, fields):
        """fields: 8 planes (numpy float64 [8,N1,N2,N3] / list of arrays on the host, or torch CUDA tensors)."""
        g = GridDesc()
        g.N1, g.N2, g.N3 = desc["N1"], desc["N2"], desc["N3"]
        g.startx[:] = list(desc["startx"]); g.dx[:] = list(desc["dx"])
        for k in ("hslope", "gam", "M_unit", "Rlow", "Rhigh", "r_out"):
            setattr(g, k, desc[k])
        planes = []
        for f in fields:
            if isinstance(f, np.ndarray):
                f = np.ascontiguousarray(f, dtype=np.float64)
            else:
                f = f.contiguous()
            planes.append(f)
        ptrs = (C.c_void_p * 8)(*[_ptr(f) for f in planes])
        _chk(lib().ipole_load_model_grid(self._h, C.byref(g), ptrs), "ipole_load_model_grid")

    # -- the hot path --
    def make_image(self, maps=False, out=None):
        """One full-Stokes image on the device.  Returns dict of torch CUDA float64 tensors [ny, nx]
        (I, Q, U, V and, with maps=True, tau and tauF).  `out` may hold preallocated tensors to reuse."""
        import torch
        names = ["I", "Q", "U", "V"] + (["tau", "tauF"] if maps else [])
        if out is None:
            out = {k: torch.empty((self.ny, self.nx), dtype=torch.float64, device="cuda") for k in names}
        args = [_ptr(out.get(k)) for k in ("I", "Q", "U", "V", "tau", "tauF")]
        _chk(lib().ipole_make_image(self._h, *args), "ipole_make_image")
        return out

    def make_image_host(self, maps=False, out=None):
        """Same through HOST buffers (numpy or pinned torch CPU tensors): the library does the copies."""
        names = ["I", "Q", "U", "V"] + (["tau", "tauF"] if maps else [])
        if out is None:
            out = {k: np.empty((self.ny, self.nx), dtype=np.float64) for k in names}
        args = [_ptr(out.get(k)) for k in ("I", "Q", "U", "V", "tau", "tauF")]
        _chk(lib().ipole_make_image(self._h, *args), "ipole_make_image")
        return out

    def make_images_adaf(self, models, freqs=None, maps=False, out=None, host=False):
        """Many small images for model fitting (include/ipole.h ipole_make_images_adaf): `models` is a
        list of dicts with the keys of load_adaf; `freqs` an optional list of observing frequencies in Hz.  The
        geodesics are integrated once; returns dict of [n_models, ny, nx] arrays (torch CUDA tensors, or numpy with
        host=True) plus "flux_jy" [n_models, 4] (numpy)."""
        M = len(models)
        arr = (AdafParams * M)()
        for m, kw in enumerate(models):
            d = dict(n0=1e6, p_n=-1.5, Th0=30.0, p_T=-1.0, B0=30.0, p_B=-1.25); d.update(kw)
            arr[m] = AdafParams(d["n0"], d["p_n"], d["Th0"], d["p_T"], d["B0"], d["p_B"])
        return self._make_images(lib().ipole_make_images_adaf, "ipole_make_images_adaf", M, arr, freqs, maps, out, host)

    def make_images_grid(self, sets, freqs=None, maps=False, out=None, host=False):
        """The same for the loaded grid model: `sets` is a list of dicts M_unit, Rlow, Rhigh (include/ipole.h
        ipole_make_images_grid)."""
        M = len(sets)
        arr = (GridScales * M)()
        for m, kw in enumerate(sets):
            arr[m] = GridScales(kw["M_unit"], kw["Rlow"], kw["Rhigh"])
        return self._make_images(lib().ipole_make_images_grid, "ipole_make_images_grid", M, arr, freqs, maps, out, host)

    def make_images_cameras(self, cams, maps=False, out=None, host=False):
        """Many small images whose geometry differs (include/ipole.h ipole_make_images_cameras): `cams` is a
        list of camera dicts (the keys of the constructor); one pass of the pipeline over the union of their rays.
        Returns dict of [n_cams, ny, nx] arrays plus "flux_jy" [n_cams, 4]."""
        M = len(cams)
        arr = (Camera * M)()
        for m, kw in enumerate(cams):
            for k, v in kw.items():
                setattr(arr[m], k, v)
        ny, nx = arr[0].ny, arr[0].nx
        names = ["I", "Q", "U", "V"] + (["tau", "tauF"] if maps else [])
        if out is None:
            if host:
                out = {k: np.empty((M, ny, nx), dtype=np.float64) for k in names}
            else:
                import torch
                out = {k: torch.empty((M, ny, nx), dtype=torch.float64, device="cuda") for k in names}
        flux = np.zeros((M, 4))
        args = [_ptr(out.get(k)) for k in ("I", "Q", "U", "V", "tau", "tauF")]
        _chk(lib().ipole_make_images_cameras(self._h, M, arr, *args, _ptr(flux)), "ipole_make_images_cameras")
        out = dict(out)
        out["flux_jy"] = flux
        return out

    def _make_images(self, fn, what, M, arr, freqs, maps, out, host):
        fr = None if freqs is None else np.ascontiguousarray(freqs, dtype=np.float64)
        assert fr is None or fr.size == M
        names = ["I", "Q", "U", "V"] + (["tau", "tauF"] if maps else [])
        if out is None:
            if host:
                out = {k: np.empty((M, self.ny, self.nx), dtype=np.float64) for k in names}
            else:
                import torch
                out = {k: torch.empty((M, self.ny, self.nx), dtype=torch.float64, device="cuda") for k in names}
        flux = np.zeros((M, 4))
        args = [_ptr(out.get(k)) for k in ("I", "Q", "U", "V", "tau", "tauF")]
        _chk(fn(self._h, M, arr, _ptr(fr), *args, _ptr(flux)), what)
        out = dict(out)
        out["flux_jy"] = flux
        return out

    def make_image_adaptive(self, levels=3, rel_tol=1e-2, abs_tol=0.0, out=None, host=False):
        """Adaptive ray tracing (include/ipole.h ipole_make_image_adaptive).  Returns (dict of I,Q,U,V
        [ny, nx] and "state" uint8 [ny, nx]: 1 traced, 2 interpolated; info dict)."""
        names = ["I", "Q", "U", "V"]
        if out is None:
            if host:
                out = {k: np.empty((self.ny, self.nx), dtype=np.float64) for k in names}
            else:
                import torch
                out = {k: torch.empty((self.ny, self.nx), dtype=torch.float64, device="cuda") for k in names}
        state = np.zeros((self.ny, self.nx), dtype=np.uint8)
        info = AdaptiveInfo()
        _chk(lib().ipole_make_image_adaptive(self._h, int(levels), float(rel_tol), float(abs_tol), *[_ptr(out[k]) for k in names],
                                             _ptr(state), C.byref(info)), "ipole_make_image_adaptive")
        out = dict(out)
        out["state"] = state
        d = dict(n_traced=info.n_traced, n_traced_level=[info.n_traced_level[i] for i in range(levels + 1)],
                 total_steps=info.total_steps, flux_jy=[info.flux_jy[i] for i in range(4)], ms_total=info.ms_total,
                 n_launches=info.n_launches)
        return out, d

    def make_pixels(self, pixels):
        """Stokes, maps and ray info for a list of flat pixel indices j*nx+i (host numpy in, host numpy out)."""
        pix = np.ascontiguousarray(pixels, dtype=np.int64)
        n = pix.size
        out = {k: np.zeros(n) for k in ("I", "Q", "U", "V", "tau", "tauF")}
        out["nsteps"] = np.zeros(n, dtype=np.int32)
        out["nturn"] = np.zeros(n, dtype=np.int32)
        args = [_ptr(out[k]) for k in ("I", "Q", "U", "V", "tau", "tauF", "nsteps", "nturn")]
        _chk(lib().ipole_make_pixels(self._h, n, _ptr(pix), *args), "ipole_make_pixels")
        return out

    def ray_info(self):
        n = self.nx * self.ny
        ns = np.zeros(n, dtype=np.int32); nt = np.zeros(n, dtype=np.int32)
        _chk(lib().ipole_get_ray_info(self._h, _ptr(ns), _ptr(nt)), "ipole_get_ray_info")
        return ns.reshape(self.ny, self.nx), nt.reshape(self.ny, self.nx)

    def image_totals_static(self, I, Q, U, V, out):
        """Totals of four CUDA FP64 planes into the CUDA tensor `out` (6 doubles: flux_jy[4], lp, cp) through the entry point
        that allocates nothing (include/ipole.h ipole_image_totals_static).  Asynchronous on the context's stream."""
        for t in (I, Q, U, V, out):
            if not (t.is_cuda and t.is_contiguous() and str(t.dtype) == "torch.float64"):
                raise ValueError("image_totals_static takes contiguous CUDA float64 tensors")
        if out.numel() < 6 or not (I.numel() == Q.numel() == U.numel() == V.numel()):
            raise ValueError("image_totals_static: out needs 6 doubles, the planes equal sizes")
        _chk(lib().ipole_image_totals_static(self._h, I.numel(), I.data_ptr(), Q.data_ptr(), U.data_ptr(), V.data_ptr(),
                                             out.data_ptr()), "ipole_image_totals_static")
        return out

    def stats(self):
        s = Stats()
        _chk(lib().ipole_get_stats(self._h, C.byref(s)), "ipole_get_stats")
        d = {k: getattr(s, k) for k, _ in Stats._fields_ if k != "flux_jy"}
        d["flux_jy"] = [s.flux_jy[i] for i in range(4)]
        return d

    # -- stages --
    def camera_tetrad(self):
        X = np.zeros(4); e = np.zeros((4, 4))
        _chk(lib().ipole_get_camera_tetrad(self._h, _dp(X), _dp(e)), "ipole_get_camera_tetrad")
        return X, e

    def trace_pixel(self, i, j, cap=60000):
        X = np.zeros((cap + 1, 4)); K = np.zeros((cap + 1, 4)); dl = np.zeros(cap)
        nt = C.c_int32(); st = C.c_int32(); need = C.c_int32()
        n = _chk(lib().ipole_trace_pixel(self._h, i, j, cap, _dp(X), _dp(K), _dp(dl), C.byref(nt), C.byref(st),
                                         C.byref(need)), "ipole_trace_pixel")
        return X[:n + 1].copy(), K[:n + 1].copy(), dl[:n].copy(), nt.value, st.value

    def _eval(self, name, x, nin, nout):
        a = np.ascontiguousarray(x, dtype=np.float64).reshape(-1, nin)
        o = np.zeros((a.shape[0], nout))
        _chk(getattr(lib(), "ipole_eval_" + name)(self._h, a.shape[0], _dp(a), _dp(o)), "ipole_eval_" + name)
        return o

    def eval_connection(self, X):
        return self._eval("connection", X, 4, 64).reshape(-1, 4, 4, 4)

    def eval_coefficients(self, ne, thetae, B, cosT, nu):
        x = np.stack(np.broadcast_arrays(ne, thetae, B, cosT, nu), axis=-1).astype(np.float64)
        return self._eval("coefficients", x, 5, 8)

    def eval_coefficients_edf(self, ne, thetae, B, cosT, nu):
        x = np.stack(np.broadcast_arrays(ne, thetae, B, cosT, nu), axis=-1).astype(np.float64)
        return self._eval("coefficients_edf", x, 5, 8)

    def eval_stokes_step(self, alpha, rho, s, S0, J):
        x = np.concatenate([np.asarray(alpha, float).reshape(-1, 4), np.asarray(rho, float).reshape(-1, 3),
                            np.asarray(s, float).reshape(-1, 1), np.asarray(S0, float).reshape(-1, 4),
                            np.asarray(J, float).reshape(-1, 4)], axis=1)
        return self._eval("stokes_step", x, 16, 4)

    def eval_bessel(self, z):
        return self._eval("bessel", z, 1, 3)

    def eval_math(self, x):
        """exp, expm1, ln|x|, sin, cos, 1/x, 1/sqrt|x|, sqrt|x| of csrc/fpmath.cuh"""
        return self._eval("math", x, 1, 8)

    def eval_plasma(self, X):
        return self._eval("plasma", X, 4, 12)

    def fp64_peak(self):
        t = C.c_double(); ms = C.c_float()
        _chk(lib().ipole_measure_fp64_peak(self._h, C.byref(t), C.byref(ms)), "ipole_measure_fp64_peak")
        return t.value, ms.value
