"""Second physics workload (reading R-13), pytest -m gpu: j and alpha of every transfer step
integrated numerically over a Maxwell-Juettner or kappa electron distribution, against the oracle (oracle/ref_edf.hpp) --
the coefficient stage on its own and whole images through ipole_make_image."""
import numpy as np
import pytest

from paper_2302_02733_b200 import workloads as W
from test_gpu_parity import check_parity, to_np, ipole, NTHREADS  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kind,kappa", [(1, 3.5), (2, 3.5), (2, 5.0)])
def test_edf_coefficients_match_the_oracle(ipole, ref, kind, kappa):
    rng = np.random.default_rng(78 + kind)
    n = 160
    ne = 10 ** rng.uniform(1.5, 6, n); Th = 10 ** rng.uniform(-1.2, 1.5, n); B = 10 ** rng.uniform(-2.3, 1.4, n)
    cosT = rng.uniform(-0.999, 0.999, n); nu = 10 ** rng.uniform(10.5, 12.2, n)
    # the value ranges of W1 (SURVEY c-9): cold, weakly magnetised outskirts where everything underflows included
    g = ipole.Ipole(**W.camera("adaf", 8))
    g.set_edf(kind, kappa=kappa)
    got = g.eval_coefficients_edf(ne, Th, B, cosT, nu)
    want = np.array([ref.coefficients_edf(kind, ne[i], Th[i], B[i], cosT[i], nu[i], kappa=kappa) for i in range(n)])
    for k in range(8):
        scale = np.maximum(np.abs(want[:, k]), 1e-300)
        big = np.abs(want[:, k]) > 1e-250            # far below anything that reaches an image
        err = np.abs(got[:, k] - want[:, k])[big] / scale[big]
        assert err.max() < 2e-10, (k, err.max())
    assert (np.abs(want[:, 0]) > 1e-30).sum() > n // 8
    # kind 0 is the thermal-fit stage
    g.set_edf(0)
    assert np.array_equal(g.eval_coefficients_edf(ne, Th, B, cosT, nu), g.eval_coefficients(ne, Th, B, cosT, nu))


@pytest.mark.parametrize("kind", [1, 2])
def test_edf_image_matches_the_oracle(ipole, ref, kind):
    cam = W.camera("adaf", 12)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF); g.set_edf(kind)
    got = to_np(g.make_image(maps=True))
    ns, nt = g.ray_info()
    got["nsteps"], got["nturn"] = ns.ravel(), nt.ravel()
    r = ref.Ctx(**cam); r.load_adaf(**W.ADAF); r.set_edf(kind)
    want = r.make_pixels(nthreads=NTHREADS)
    check_parity(got, want, "edf kind %d" % kind, min_lit=0.99)
    assert np.allclose(got["tau"], want["tau"], rtol=1e-7, atol=0) and np.allclose(got["tauF"], want["tauF"], rtol=1e-7, atol=0)
    # and it is a different image from the thermal-fit one (kappa: a brighter, flatter-spectrum source)
    g.set_edf(0)
    fit = to_np(g.make_image())
    if kind == 2:
        assert got["I"].sum() > 1.3 * fit["I"].sum()
    else:
        assert got["I"].sum() == pytest.approx(fit["I"].sum(), rel=0.05)


def test_edf_long_rays_batches_and_unsupported_combinations(ipole):
    cam = W.camera("adaf", 24, max_steps=6000)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF); g.set_edf(2)
    base = to_np(g.make_image())
    g.set_options(40 << 20, 0)           # slots far shorter than the rays: every ray takes the third level (split kernels, max_steps slots)
    a = to_np(g.make_image()); st = g.stats()
    assert st["n_long"] == 24 * 24
    for k in base:
        assert np.array_equal(base[k], a[k]), k
    g.set_options(0, 1)
    g.set_path_free(True)
    with pytest.raises(ipole.IpoleError):
        g.make_image()
    g.set_path_free(False); g.set_unpolarized(True)
    with pytest.raises(ipole.IpoleError):
        g.make_image()
    g.set_unpolarized(False)
    with pytest.raises(ipole.IpoleError):
        g.make_images_adaf([dict(n0=1e6)])
    with pytest.raises(ipole.IpoleError):
        g.set_edf(2, kappa=0.5)
    g.set_edf(0)
    g.make_images_adaf([dict(n0=1e6)])


def test_fp32_geodesic_study_switch(ipole):
    """ipole_set_geodesic_fp32 (PAPER.md:70 study, profiles/r2_fp32_study.md): single-precision geodesics give the image to
    ~1e-5..1e-3 per pixel, not to 1e-7; switching back restores the FP64 image bit for bit."""
    cam = W.camera("adaf", 48)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    a = to_np(g.make_image())
    g.set_geodesic_fp32(True)
    b = to_np(g.make_image())
    g.set_geodesic_fp32(False)
    c = to_np(g.make_image())
    for k in a:
        assert np.array_equal(a[k], c[k]), k
    lit = a["I"] > 1e-6 * a["I"].max()
    rel = np.abs(b["I"] - a["I"])[lit] / a["I"][lit]
    assert 1e-7 < np.median(rel) < 1e-3 and abs(b["I"].sum() / a["I"].sum() - 1) < 1e-3
