"""GPU parity of the path-free bidirectional variant (R-10), pytest -m gpu:
ipole_set_path_free(1) through the C ABI against the oracle's path-free variant (oracle/ref_pathfree.hpp) on the same
synthetic inputs, with the tolerances of BASELINE.json north_star (tests/test_gpu_parity.py::check_parity).
"""
import os

import numpy as np
import pytest

from paper_2302_02733_b200 import workloads as W
from test_gpu_parity import check_parity, gpu_full_then_sample, sample_pixels, to_np, ipole, NTHREADS  # noqa: F401

pytestmark = pytest.mark.gpu


def pair(ipole, ref, cam, load):
    g = ipole.Ipole(**cam); load(g); g.set_path_free(True)
    r = ref.Ctx(**cam); load(r); r.set_path_free(True)
    return g, r


def test_pf_w1_adaf_32_full_image(ipole, ref):
    cam = W.camera("adaf", 32)
    g, r = pair(ipole, ref, cam, lambda c: c.load_adaf(**W.ADAF))
    want = r.make_pixels(nthreads=NTHREADS)
    got, img = gpu_full_then_sample(g, np.arange(1024))
    info = check_parity(got, want, "PF W1", min_lit=0.99)
    assert info["max_err"] < 1e-8
    st = g.stats()
    assert st["n_batches"] == 1 and st["path_cap"] == 0 and st["n_long"] == 0
    assert st["total_steps"] == int(want["nsteps"].sum())                 # backward pass
    assert abs(st["total_steps_forward"] / st["total_steps"] - 1) < 0.01  # forward pass: about as many, not the same
    # host buffers: bit-identical
    host = g.make_image_host(maps=True)
    for k in host:
        assert np.array_equal(host[k].ravel(), got[k]), k
    # the pixel-list entry gives the same bits
    pix = np.arange(0, 1024, 7, dtype=np.int64)
    lst = g.make_pixels(pix)
    for k in ("I", "Q", "U", "V", "tau", "tauF", "nsteps", "nturn"):
        assert np.array_equal(lst[k], got[k][pix]), k
    # switching the variant off restores the stored-path image bit for bit
    g2 = ipole.Ipole(**cam); g2.load_adaf(**W.ADAF)
    stored = to_np(g2.make_image(maps=True))
    g.set_path_free(False)
    back = to_np(g.make_image(maps=True))
    for k in stored:
        assert np.array_equal(stored[k], back[k]), k
    assert g.stats()["total_steps_forward"] == 0
    # and the two variants differ "negligibly" but not by nothing
    d = abs(got["I"].sum() - stored["I"].sum()) / stored["I"].sum()
    assert 0 < d < 5e-4


def test_pf_ragged_image_other_camera_and_forced_sort(ipole, ref):
    cam = W.camera("adaf", 8, freq_hz=345e9, inclination_deg=33.0, spin=0.5, hslope=0.7)
    cam.update(nx=37, ny=23, fov=30.0)
    g, r = pair(ipole, ref, cam, lambda c: c.load_adaf(**W.ADAF))
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(37 * 23))
    check_parity(got, want, "PF ragged", min_lit=0.99)
    g.set_options(0, 2)   # probe + sort: the order of the rays must not change a bit
    again, _ = gpu_full_then_sample(g, np.arange(37 * 23))
    for k in got:
        assert np.array_equal(got[k], again[k]), k


def test_pf_large_eps_and_step_limit(ipole, ref):
    # eps > 0.04: the general RK4 form (k_transfer<., 2>)
    cam = W.camera("adaf", 16, eps=0.05)
    g, r = pair(ipole, ref, cam, lambda c: c.load_adaf(**W.ADAF))
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(256))
    check_parity(got, want, "PF eps 0.05", min_lit=0.99)
    # step limit: the backward pass ends on max_steps somewhere mid-flight, the forward pass starts there
    cam = W.camera("adaf", 16, max_steps=900)
    g, r = pair(ipole, ref, cam, lambda c: c.load_adaf(**W.ADAF))
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(256))
    assert ((want["nturn"] & 0x80) != 0).all() and (got["nturn"] == want["nturn"]).all() and (got["nsteps"] == 900).all()
    check_parity(got, want, "PF max_steps")


def test_pf_slab_flat_space(ipole, ref):
    L = 6.6742e-8 * 4.1e6 * 1.989e33 / 2.99792458e10 ** 2
    cam = W.camera("adaf", 16, spin=0.0, flat_metric=1, inclination_deg=40.0, fov=2.0, r_cam=500.0, r_esc=500.0)
    H, j = 2.0, 1e-20
    path = 2 * H / np.cos(np.radians(40.0)) * L
    a = 3.0 / path
    g, r = pair(ipole, ref, cam, lambda c: c.load_slab(H, j=(j, 0, 0, 0), alpha=(a, 0, 0, 0)))
    img = to_np(g.make_image(maps=True)); want = r.make_pixels(nthreads=NTHREADS)
    assert np.allclose(img["I"], j / a * (1 - np.exp(-a * path)), rtol=5e-3, atol=0)   # closed form
    assert np.abs(img["I"] - want["I"]).max() <= 1e-9 * want["I"].max()
    kw = dict(H=H, j=(j, 0.3 * j, -0.2 * j, 0.1 * j), alpha=(a, 0.2 * a, 0.1 * a, -0.05 * a), rho=(4 * a, -2 * a, 9 * a),
              psi_deg=20.0, profile=1)
    g, r = pair(ipole, ref, cam, lambda c: c.load_slab(**kw))
    got, _ = gpu_full_then_sample(g, np.arange(256))
    want = r.make_pixels(nthreads=NTHREADS)
    check_parity(got, want, "PF slab", min_lit=1.0)


def test_pf_grid_small_full_image(ipole, ref):
    desc, fields = W.fm_torus_grid(72, 32, 32)
    cam = W.camera("grid", 32)
    g, r = pair(ipole, ref, cam, lambda c: c.load_grid(desc, fields))
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(1024))
    info = check_parity(got, want, "PF grid small", min_lit=0.2)
    assert info["lit"] < 1.0


def test_pf_w2_adaf_256_sampled(ipole, ref):
    cam = W.camera("adaf", 256)
    g, r = pair(ipole, ref, cam, lambda c: c.load_adaf(**W.ADAF))
    pix = sample_pixels(256, 256, 8, window=(150, 120, 48, 16))
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, pix)
    info = check_parity(got, want, "PF W2", min_lit=0.99)
    assert info["ring_frac"] > 0.02


def test_pf_w4_grid_1024_sampled_with_maps(ipole, ref):
    desc, fields = W.fm_torus_grid(576, 256, 256)
    cam = W.camera("grid", 1024)
    g, r = pair(ipole, ref, cam, lambda c: c.load_grid(desc, fields))
    pix = sample_pixels(1024, 1024, 32, window=(560, 508, 128, 4))
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, pix, maps=True)
    check_parity(got, want, "PF W4", min_lit=0.3)


def test_pf_w5_adaf_4096_sampled(ipole, ref):
    """Full size, in the configuration `bench.py --workload adaf4096 --path-free` times."""
    cam = W.camera("adaf", 4096)
    g, r = pair(ipole, ref, cam, lambda c: c.load_adaf(**W.ADAF))
    pix = sample_pixels(4096, 4096, 128, window=(2400, 2040, 256, 2))
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, img = gpu_full_then_sample(g, pix, maps=False)
    check_parity(got, want, "PF W5 adaf", min_lit=0.99)
    st = g.stats()
    assert st["n_batches"] == 1 and st["n_maxstep"] == 0
    import torch
    pol = torch.sqrt(img["Q"] ** 2 + img["U"] ** 2 + img["V"] ** 2)
    assert bool((pol <= img["I"] * (1 + 1e-12)).all()) and bool(torch.isfinite(img["I"]).all())


def test_pf_difference_from_stored_path_vs_eps(ipole, capsys):
    """"for a typically adopted value of epsilon the differences in all Stokes parameter images produced
    by CPU and GPU codes are negligible" -- measured here on the GPU for both variants (W2 geometry, 256^2, 230 GHz).
    `pytest tests/test_gpu_pathfree.py -m gpu -k vs_eps -s` prints the table kept in profiles/r1_pathfree.md."""
    rows = []
    for eps in (0.04, 0.02, 0.01, 0.005):
        cam = W.camera("adaf", 256, eps=eps)
        g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
        a = to_np(g.make_image())
        ns, nt = g.ray_info()
        g.set_path_free(True)
        b = to_np(g.make_image())
        tot = a["I"].sum()
        dtot = [abs(b[k].sum() - a[k].sum()) / tot for k in "IQUV"]
        lit = a["I"] > 1e-6 * a["I"].max()
        rel = np.abs(b["I"] - a["I"])[lit] / a["I"][lit]
        pol = np.maximum.reduce([np.abs(b[k] - a[k])[lit] / a["I"][lit] for k in "QUV"])
        rows.append((eps, dtot, np.median(rel), np.percentile(rel, 99), rel.max(), np.median(pol), np.percentile(pol, 99)))
    with capsys.disabled():
        print("\neps    |dI|/I    |dQ|/I    |dU|/I    |dV|/I   pixel I: median   p99      max     pixel Q,U,V/I: median  p99")
        for eps, dtot, med, p99, mx, pmed, pp99 in rows:
            print("%.3f  %.2e  %.2e  %.2e  %.2e   %.2e  %.2e  %.2e   %.2e  %.2e" % ((eps,) + tuple(dtot) + (med, p99, mx, pmed, pp99)))
    for eps, dtot, med, p99, mx, pmed, pp99 in rows:
        if eps <= 0.02:
            assert max(dtot) < 1e-3 and med < 1e-4 and pmed < 1e-4
    assert rows[-1][2] < rows[0][2]   # the typical pixel difference shrinks with eps
