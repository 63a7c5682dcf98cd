"""Many cameras per call (the camera half; include/ipole.h ipole_make_images_cameras), pytest -m gpu:
one pass of the pipeline over the union of the rays of cameras that differ in inclination, spin, frequency, field of view
and mass.  Every image must be the image a single call with that camera gives, and must match the oracle."""
import numpy as np
import pytest

from paper_2302_02733_b200 import workloads as W
from test_gpu_parity import check_parity, to_np, ipole, small_grid, NTHREADS  # noqa: F401

pytestmark = pytest.mark.gpu


def cameras(n, npix=32):
    out = []
    for k in range(n):
        out.append(W.camera("adaf", npix, inclination_deg=17.0 + 146.0 * k / max(1, n - 1), spin=[0.9375, 0.5, 0.0, 0.99][k % 4],
                            freq_hz=[230e9, 345e9, 86e9][k % 3], fov=[40.0, 60.0][k % 2], mbh_msun=[4.1e6, 6.5e9][k % 2],
                            dsource_pc=[8000.0, 16.8e6][k % 2]))
    return out


def test_cameras_equal_single_calls_and_oracle(ipole, ref):
    cams = cameras(6)
    g = ipole.Ipole(**cams[0]); g.load_adaf(**W.ADAF)
    out = g.make_images_cameras(cams, maps=True)
    for m, cam in enumerate(cams):
        f = ipole.Ipole(**cam); f.load_adaf(**W.ADAF)
        one = to_np(f.make_image(maps=True)); st = f.stats()
        sc = np.abs(one["I"]).max()
        for k in ("I", "Q", "U", "V"):
            assert np.abs(out[k][m].cpu().numpy().ravel() - one[k]).max() <= 1e-11 * sc, (m, k)
        for k in ("tau", "tauF"):
            assert np.allclose(out[k][m].cpu().numpy().ravel(), one[k], rtol=1e-11, atol=0), (m, k)
        assert np.allclose(out["flux_jy"][m], st["flux_jy"], rtol=1e-10, atol=1e-12 * abs(st["flux_jy"][0]))
        if m in (1, 4):
            r = ref.Ctx(**cam); r.load_adaf(**W.ADAF)
            want = r.make_pixels(nthreads=NTHREADS)
            got = {k: out[k][m].cpu().numpy().ravel() for k in ("I", "Q", "U", "V", "tau", "tauF")}
            check_parity(got, want, "camera %d" % m, min_lit=0.9)
    # the context's own camera and model are untouched
    a = to_np(g.make_image())
    f = ipole.Ipole(**cams[0]); f.load_adaf(**W.ADAF)
    b = to_np(f.make_image())
    for k in a:
        assert np.array_equal(a[k], b[k]), k


def test_cameras_probe_sort_batches_long_rays_and_host_buffers(ipole):
    cams = cameras(40, npix=32)                       # 40 960 rays: the union is probed and sorted
    cams = [dict(c, max_steps=6000) for c in cams]
    g = ipole.Ipole(**cams[0]); g.load_adaf(**W.ADAF)
    a = g.make_images_cameras(cams)
    st = g.stats()
    assert st["ms_probe"] > 0
    A = {k: a[k].cpu().numpy() for k in ("I", "Q", "U", "V")}
    g.set_options(64 << 20, 1)                        # many batches; some rays outgrow their slots and S_cap
    b = g.make_images_cameras(cams, host=True)
    st2 = g.stats()
    assert st2["n_batches"] > 3
    for k in A:
        assert np.array_equal(A[k], b[k]), k
    assert np.allclose(a["flux_jy"], b["flux_jy"], rtol=1e-13)
    g.set_options(0, 1)
    g.set_edf(2)                                      # and with the numerically integrated coefficients
    e = g.make_images_cameras(cams[:3])
    f = ipole.Ipole(**cams[1]); f.load_adaf(**W.ADAF); f.set_edf(2)
    one = to_np(f.make_image())
    assert np.abs(e["I"][1].cpu().numpy().ravel() - one["I"]).max() <= 1e-11 * one["I"].max()


def test_cameras_errors(ipole):
    cams = cameras(3)
    g = ipole.Ipole(**cams[0])
    with pytest.raises(ipole.IpoleError) as e:
        g.make_images_cameras(cams)
    assert e.value.code == ipole.ENOMODEL
    g.load_adaf(**W.ADAF)
    with pytest.raises(ipole.IpoleError):
        g.make_images_cameras([cams[0], dict(cams[1], nx=16)])
    with pytest.raises(ipole.IpoleError):
        g.make_images_cameras([cams[0], dict(cams[1], eps=0.02)])
    g.set_path_free(True)
    with pytest.raises(ipole.IpoleError):
        g.make_images_cameras(cams)
    g.set_path_free(False)
    g.make_images_cameras(cams)


def test_grid_cameras_equal_single_calls_and_oracle(ipole, ref, small_grid):
    """The grid model through ipole_make_images_cameras: cameras that share spin, mass and hslope with the context's and
    differ in inclination, frequency, field of view and distance; k_geodesic<true, MC> + k_transfer_group<grid, MC>."""
    desc, fields = small_grid
    base = W.camera("grid", 40)
    cams = []
    for k, (inc, fr, fov, dist) in enumerate(((20.0, 230e9, 40.0, 8000.0), (60.0, 345e9, 40.0, 8000.0), (85.0, 86e9, 60.0, 8000.0),
                                              (140.0, 230e9, 30.0, 16000.0), (20.0, 690e9, 40.0, 8000.0))):
        cam = dict(base); cam.update(inclination_deg=inc, freq_hz=fr, fov=fov, dsource_pc=dist)
        cams.append(cam)
    g = ipole.Ipole(**base); g.load_grid(desc, fields)
    out = g.make_images_cameras(cams, maps=True)
    for m, cam in enumerate(cams):
        f = ipole.Ipole(**cam); f.load_grid(desc, fields)
        one = to_np(f.make_image(maps=True)); st = f.stats()
        f.close()
        sc = np.abs(one["I"]).max()
        assert sc > 0
        for k in ("I", "Q", "U", "V"):
            # (another instantiation of the same kernels: rounding-level differences, amplified where the Faraday depth is large)
            assert np.abs(out[k][m].cpu().numpy().ravel() - one[k]).max() <= 1e-9 * sc, (m, k)
        for k in ("tau", "tauF"):
            assert np.allclose(out[k][m].cpu().numpy().ravel(), one[k], rtol=1e-9, atol=1e-12 * np.abs(one[k]).max()), (m, k)
        assert np.allclose(out["flux_jy"][m], st["flux_jy"], rtol=1e-9, atol=1e-11 * abs(st["flux_jy"][0]))
        if m == 2:
            r = ref.Ctx(**cam); r.load_grid(desc, fields)
            want = r.make_pixels(nthreads=NTHREADS)
            got = {k: out[k][m].cpu().numpy().ravel() for k in ("I", "Q", "U", "V", "tau", "tauF")}
            check_parity(got, want, "grid camera %d" % m, min_lit=0.2)
    # many batches, per-batch slots, retry level and long rays with cameras
    g.set_options(24 << 20, 2)
    out2 = g.make_images_cameras(cams, maps=True)
    assert g.stats()["n_batches"] > 3
    for k in ("I", "Q", "U", "V", "tau", "tauF"):
        assert np.array_equal(out2[k].cpu().numpy(), out[k].cpu().numpy()), k
    # the context's own camera is untouched, and a camera of another spin or mass is refused
    again = to_np(g.make_image(maps=True))
    f = ipole.Ipole(**base); f.load_grid(desc, fields); f.set_options(24 << 20, 2)
    want = to_np(f.make_image(maps=True))
    for k in want:
        assert np.array_equal(again[k], want[k]), k
    bad = dict(cams[1]); bad["spin"] = 0.5
    with pytest.raises(ipole.IpoleError) as ei:
        g.make_images_cameras([cams[0], bad])
    assert ei.value.code == ipole.EINVAL
