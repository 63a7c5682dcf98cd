"""Unpolarized transfer on the GPU (R-12), pytest -m gpu: ipole_set_unpolarized(1) against the
oracle's scalar transfer (oracle/ref_unpol.hpp, pins U1-U3), north-star tolerances."""
import numpy as np
import pytest

from paper_2302_02733_b200 import workloads as W
from test_gpu_parity import check_parity, gpu_full_then_sample, sample_pixels, to_np, ipole, NTHREADS  # noqa: F401

pytestmark = pytest.mark.gpu


def pair(ipole, ref, cam, load):
    g = ipole.Ipole(**cam); load(g); g.set_unpolarized(True)
    r = ref.Ctx(**cam); load(r); r.set_unpolarized(True)
    return g, r


def test_unpol_w1_and_scheduling(ipole, ref):
    cam = W.camera("adaf", 32, max_steps=6000)
    g, r = pair(ipole, ref, cam, lambda c: c.load_adaf(**W.ADAF))
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(1024))
    info = check_parity(got, want, "unpol W1", min_lit=0.99)
    assert info["max_err"] < 1e-9
    assert all((got[k] == 0).all() for k in ("Q", "U", "V", "tauF"))
    # batches, forced sort, long-ray pass, host buffers: same bits
    for opts in ((0, 2), (8 << 20, 2), (12 << 20, 0)):
        g.set_options(*opts)
        again, _ = gpu_full_then_sample(g, np.arange(1024))
        for k in got:
            assert np.array_equal(got[k], again[k]), (opts, k)
    host = g.make_image_host(maps=True)
    for k in host:
        assert np.array_equal(host[k].ravel(), got[k]), k
    # switching it off restores the polarized image
    g.set_options(0, 1); g.set_unpolarized(False)
    pol = to_np(g.make_image())
    assert np.abs(pol["Q"]).max() > 0 and np.all(np.abs(pol["I"] / got["I"] - 1) < 1e-2)


def test_unpol_slab_closed_form_and_grid(ipole, ref):
    L = 6.6742e-8 * 4.1e6 * 1.989e33 / 2.99792458e10 ** 2
    cam = W.camera("adaf", 16, spin=0.0, flat_metric=1, inclination_deg=40.0, fov=2.0, r_cam=500.0, r_esc=500.0)
    H, j = 2.0, 1e-20
    path = 2 * H / np.cos(np.radians(40.0)) * L
    a = 3.0 / path
    g, r = pair(ipole, ref, cam, lambda c: c.load_slab(H, j=(j, 0.3 * j, 0, 0.1 * j), alpha=(a, 0.2 * a, 0, 0), rho=(a, 0, 2 * a)))
    img = to_np(g.make_image(maps=True)); want = r.make_pixels(nthreads=NTHREADS)
    assert np.allclose(img["I"], j / a * (1 - np.exp(-a * path)), rtol=5e-3, atol=0)   # scalar closed form: alpha_Q ignored
    assert np.abs(img["I"] - want["I"]).max() <= 1e-9 * want["I"].max() and np.allclose(img["tau"], want["tau"], rtol=1e-9)
    desc, fields = W.fm_torus_grid(72, 32, 32)
    cam = W.camera("grid", 32)
    g, r = pair(ipole, ref, cam, lambda c: c.load_grid(desc, fields))
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(1024))
    info = check_parity(got, want, "unpol grid", min_lit=0.2)
    assert info["lit"] < 1.0


def test_unpol_w2_sampled_and_sweeps(ipole, ref):
    cam = W.camera("adaf", 256)
    g, r = pair(ipole, ref, cam, lambda c: c.load_adaf(**W.ADAF))
    pix = sample_pixels(256, 256, 8, window=(150, 120, 48, 16))
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, pix)
    check_parity(got, want, "unpol W2", min_lit=0.99)
    # the model sweep in unpolarized mode: the paper's fitting case
    cam = W.camera("adaf", 32)
    models = [dict(n0=1e6, Th0=30.0, B0=30.0), dict(n0=3e5, Th0=45.0, B0=20.0), dict(n0=4e6, Th0=10.0, B0=70.0)]
    freqs = [230e9, 86e9, 345e9]
    g = ipole.Ipole(**cam); g.set_unpolarized(True)
    out = g.make_images_adaf(models, freqs, maps=True)
    for m, (mod, fr) in enumerate(zip(models, freqs)):
        rr = ref.Ctx(**dict(cam, freq_hz=fr)); rr.load_adaf(**mod); rr.set_unpolarized(True)
        want = rr.make_pixels(nthreads=NTHREADS)
        gm = {k: out[k][m].cpu().numpy().ravel() for k in ("I", "Q", "U", "V", "tau", "tauF")}
        check_parity(gm, want, "unpol sweep %d" % m, min_lit=0.99)
    desc, fields = W.fm_torus_grid(72, 32, 32)
    camg = W.camera("grid", 32)
    gg = ipole.Ipole(**camg); gg.load_grid(desc, fields); gg.set_unpolarized(True)
    sets = [dict(M_unit=desc["M_unit"], Rlow=1.0, Rhigh=40.0), dict(M_unit=2.5 * desc["M_unit"], Rlow=1.0, Rhigh=5.0)]
    out = gg.make_images_grid(sets, maps=True)
    for m, st_ in enumerate(sets):
        d = dict(desc); d.update(st_)
        rr = ref.Ctx(**camg); rr.load_grid(d, fields); rr.set_unpolarized(True)
        want = rr.make_pixels(nthreads=NTHREADS)
        gm = {k: out[k][m].cpu().numpy().ravel() for k in ("I", "Q", "U", "V", "tau", "tauF")}
        check_parity(gm, want, "unpol grid sweep %d" % m, min_lit=0.2)
