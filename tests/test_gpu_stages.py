"""GPU stage-by-stage parity (pytest -m gpu): each building block of the CUDA path, called through the C ABI,
against the CPU oracle on the same seeded inputs, plus independent references where one exists (scipy Bessel)."""
import numpy as np
import pytest

from paper_2302_02733_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ipole():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import __graft_entry__ as ge
    ge.build()
    from paper_2302_02733_b200 import ipole as m
    return m


@pytest.mark.parametrize("kind,n", [("adaf", 32), ("grid", 32)])
def test_camera_tetrad(ipole, ref, kind, n):
    cam = W.camera(kind, n)
    g = ipole.Ipole(**cam)
    r = ref.Ctx(**cam)
    Xg, eg = g.camera_tetrad()
    Xr, er = r.camera_tetrad()
    assert np.allclose(Xg, Xr, rtol=0, atol=1e-15)
    assert np.allclose(eg, er, rtol=1e-14, atol=1e-18)


@pytest.mark.parametrize("a,h,flat", [(0.9375, 1.0, 0), (0.9375, 0.3, 0), (0.0, 1.0, 0), (0.5, 0.3, 1), (0.0, 1.0, 1)])
def test_connection(ipole, ref, a, h, flat):
    cam = W.camera("adaf", 8, spin=a, hslope=h, flat_metric=flat)
    g = ipole.Ipole(**cam)
    rng = np.random.default_rng(11)
    n = 200
    X = np.stack([rng.normal(size=n), rng.uniform(0.35, 7.0, n), rng.uniform(0.005, 0.995, n), rng.uniform(0, 2 * np.pi, n)], 1)
    G = g.eval_connection(X)
    Gr = np.stack([ref.conn(a, h, x, flat) for x in X])
    scale = np.abs(Gr).max(axis=(1, 2, 3), keepdims=True)
    assert (np.abs(G - Gr) / scale).max() < 1e-10
    assert np.abs(G - np.swapaxes(G, 2, 3)).max() / scale.max() < 1e-12  # symmetric in the lower indices


def test_bessel(ipole, ref):
    from scipy.special import kve
    g = ipole.Ipole(**W.camera("adaf", 8))
    z = np.concatenate([10 ** np.random.default_rng(3).uniform(-3, 4, 2000), [2.0, 2.0 + 1e-12, 2.0 - 1e-12, 1e-3, 1e4]])
    b = g.eval_bessel(z)
    for n in range(3):
        assert np.abs(b[:, n] / kve(n, z) - 1).max() < 1e-14
    br = np.stack([ref.bessel_kscaled(v) for v in z[:300]])
    assert (np.abs(b[:300] - br) / br).max() < 1e-13


def test_coefficients(ipole, ref):
    g = ipole.Ipole(**W.camera("adaf", 8))
    rng = np.random.default_rng(5)
    n = 3000
    ne = 10 ** rng.uniform(0, 7, n)
    Th = 10 ** rng.uniform(-2, 2, n)
    B = 10 ** rng.uniform(-3, 2, n)
    cosT = rng.uniform(-1, 1, n)
    nu = 10 ** rng.uniform(10.5, 12.5, n)
    # the degenerate cases of the method: field along the ray, no field, no electrons, cold plasma
    cosT[:4] = [1.0, -1.0, 0.0, 1.0 - 1e-16]
    B[4] = 0.0; ne[5] = 0.0; Th[6] = 1e-6; Th[7] = 1e-3
    out = g.eval_coefficients(ne, Th, B, cosT, nu)
    want = np.stack([ref.coefficients(*v) for v in zip(ne, Th, B, cosT, nu)])
    assert np.isfinite(out).all()
    assert (out[[0, 1, 4, 5]] == 0).all()
    scale = np.abs(want) + 1e-300
    err = np.abs(out - want) / scale
    # exp(-1.8899 x^(1/3)) amplifies the rounding of x^(1/3): allow 1e-11 relative
    assert err[want != 0].max() < 1e-11
    assert (out[want == 0] == 0).all()


def test_stokes_step(ipole, ref):
    g = ipole.Ipole(**W.camera("adaf", 8))
    rng = np.random.default_rng(9)
    n = 2000
    al = rng.normal(size=(n, 4)); al[:, 0] = np.abs(al[:, 0]) + np.linalg.norm(al[:, 1:], axis=1)
    rh = rng.normal(size=(n, 3)) * 10 ** rng.uniform(-2, 1.5, (n, 1))
    scale = 10 ** rng.uniform(-12, 0.5, (n, 1))
    al *= scale; rh *= scale
    s = 10 ** rng.uniform(-3, 1, n) / scale[:, 0] * 10 ** rng.uniform(-3, 0, n)
    S0 = rng.normal(size=(n, 4)); S0[:, 0] = np.linalg.norm(S0[:, 1:], axis=1) * (1 + rng.uniform(0, 1, n))
    J = rng.normal(size=(n, 4)) * scale
    # degenerate cases: no Faraday, no polarized absorption, nothing at all, aU = rU = 0
    rh[:50] = 0; al[50:100, 1:] = 0; al[100:120] = 0; rh[100:120] = 0; al[120:400, 2] = 0; rh[120:400, 1] = 0
    J[120:300, 2] = 0; J[:10, 2] = 0; J[50:60, 2] = 0; J[100:110, 2] = 0  # aU = rU = jU = 0: the specialised step of the transfer kernel
    out = g.eval_stokes_step(al, rh, s, S0, J)
    want = np.zeros((n, 4))
    for i in range(n):
        O, P = ref.stokes_operator(al[i], rh[i], s[i])
        want[i] = O @ S0[i] + P @ J[i]
    norm = np.abs(want).max(axis=1, keepdims=True)
    assert (np.abs(out - want) / norm).max() < 1e-11


@pytest.mark.parametrize("model", ["adaf", "slab", "grid"])
def test_plasma_models(ipole, ref, model):
    rng = np.random.default_rng(21)
    n = 400
    if model == "grid":
        cam = W.camera("grid", 8)
        desc, fields = W.fm_torus_grid(48, 24, 16)
        g = ipole.Ipole(**cam); r = ref.Ctx(**cam)
        g.load_grid(desc, fields); r.load_grid(desc, fields)
        X = np.stack([np.zeros(n), rng.uniform(0.0, 4.2, n), rng.uniform(0.0, 1.0, n), rng.uniform(-7, 14, n)], 1)
    elif model == "adaf":
        cam = W.camera("adaf", 8)
        g = ipole.Ipole(**cam); r = ref.Ctx(**cam)
        g.load_adaf(**W.ADAF); r.load_adaf(**W.ADAF)
        X = np.stack([np.zeros(n), rng.uniform(0.3, 6.9, n), rng.uniform(0.01, 0.99, n), rng.uniform(0, 6.28, n)], 1)
    else:
        cam = W.camera("adaf", 8, spin=0.3, flat_metric=1)
        kw = dict(H=3.0, j=(1e-20, 2e-21, -1e-21, 5e-22), alpha=(1e-13, 2e-14, 1e-14, -5e-15), rho=(3e-13, 1e-13, -2e-13), psi_deg=25.0, profile=1)
        g = ipole.Ipole(**cam); r = ref.Ctx(**cam)
        g.load_slab(**kw); r.load_slab(**kw)
        X = np.stack([np.zeros(n), rng.uniform(0.0, 3.0, n), rng.uniform(0.05, 0.95, n), rng.uniform(0, 6.28, n)], 1)
    out = g.eval_plasma(X)
    n_present = 0
    for i in range(n):
        p = r.plasma(X[i])
        assert bool(out[i, 0]) == p["present"], i
        if not p["present"]:
            continue
        n_present += 1
        want = np.concatenate([[p["ne"], p["thetae"], p["B"]], p["u"], p["b"]])
        got = out[i, 1:]
        tol = 1e-11 * max(np.abs(want[3:7]).max(), 1.0)
        assert np.allclose(got[:3], want[:3], rtol=1e-11, atol=0), (i, got[:3], want[:3])
        assert np.allclose(got[3:7], want[3:7], rtol=0, atol=tol)
        assert np.allclose(got[7:], want[7:], rtol=0, atol=1e-11 * max(np.abs(want[7:]).max(), 1e-300))
    assert n_present > n // 10


@pytest.mark.parametrize("kind,pix", [("adaf", (3, 5)), ("adaf", (16, 16)), ("adaf", (20, 14)), ("adaf", (12, 17)),
                                      ("grid", (16, 15)), ("grid", (9, 22)), ("grid", (21, 16))])
def test_geodesic_path(ipole, ref, kind, pix):
    """a-2/a-3: the stored path (X, K, dl at every point) of single rays, incl. ring rays and captured rays."""
    cam = W.camera(kind, 32)
    g = ipole.Ipole(**cam); r = ref.Ctx(**cam)
    Xg, Kg, dg, ntg, stg = g.trace_pixel(*pix)
    X0, K0 = r.camera_ray(*pix)
    Xo, Ko, do, nto, sto = r.trace(X0, K0)
    assert len(dg) == len(do) and ntg == nto and stg == sto
    tol = 1e-9 if nto >= 2 else 1e-11
    assert np.abs(Xg[:, 1:] - Xo[:, 1:]).max() < tol
    assert (np.abs(Kg - Ko) / np.abs(Ko).max(axis=1, keepdims=True)).max() < tol
    assert np.allclose(dg, do, rtol=tol)


@pytest.mark.parametrize("kind,eps", [("adaf", 0.04), ("grid", 0.04), ("adaf", 0.08), ("grid", 0.08), ("grid", 0.0025)])
def test_geodesic_path_other_step_parameters(ipole, ref, kind, eps):
    """The RK4 push has two forms (kernels.cuh rk4_push<SMALL>): stage points by short Taylor shifts from the start
    point for eps <= 0.04 (the 4-eps probe pass runs at that edge), from scratch above.  Both against the oracle."""
    cam = W.camera(kind, 32, eps=eps)
    g = ipole.Ipole(**cam); r = ref.Ctx(**cam)
    for pix in ((5, 7), (16, 16), (20, 14)):
        Xg, Kg, dg, ntg, stg = g.trace_pixel(*pix)
        X0, K0 = r.camera_ray(*pix)
        Xo, Ko, do, nto, sto = r.trace(X0, K0)
        assert len(dg) == len(do) and ntg == nto and stg == sto
        tol = 1e-9 if nto >= 2 else 1e-11
        assert np.abs(Xg[:, 1:] - Xo[:, 1:]).max() < tol
        assert (np.abs(Kg - Ko) / np.abs(Ko).max(axis=1, keepdims=True)).max() < tol
        assert np.allclose(dg, do, rtol=tol)


def test_fp64_peak_microbenchmark(ipole):
    g = ipole.Ipole(**W.camera("adaf", 8))
    tf, ms = g.fp64_peak()
    assert 10.0 < tf < 60.0 and ms > 0


def test_fpmath_against_mpmath(ipole):
    """The branch-free elementary functions of csrc/fpmath.cuh (exp, expm1, log, sincos, rcp, rsqrt, sqrt) against
    40-digit mpmath values: <= 2 ulp on the domains stated there, exact limits at the ends."""
    import mpmath as mp
    mp.mp.dps = 40
    g = ipole.Ipole(**W.camera("adaf", 8))
    rng = np.random.default_rng(17)
    x = np.concatenate([rng.uniform(-745, 709, 600), rng.uniform(-2, 2, 600), 10 ** rng.uniform(-300, -1, 300),
                        -10 ** rng.uniform(-300, -1, 300), rng.uniform(-1e5, 1e5, 600), 10 ** rng.uniform(-280, 280, 600),
                        [0.5, 1.0, 2.0, np.sqrt(2.0), 1.0 / np.sqrt(2.0), 1e-300, -1e-300, 709.0, -745.0, -708.4, 1e5]])
    out = g.eval_math(x)
    ulp = lambda got, want: np.abs(got - want) / np.spacing(np.abs(want))
    f = lambda fn, v: np.array([float(fn(mp.mpf(float(t)))) for t in v])
    m = x <= 709
    assert ulp(out[m, 0], f(mp.exp, x[m])).max() <= 2.0                       # includes the subnormal range below -708
    assert ulp(out[m, 1], f(mp.expm1, x[m])).max() <= 2.0
    nz = np.abs(x) > 1e-290
    assert ulp(out[nz, 2], f(mp.log, np.abs(x[nz]))).max() <= 2.0
    m = np.abs(x) <= 1e5
    # sin/cos: absolute error <= 1 ulp of 1 near the zeros of the function, <= 2 ulp elsewhere
    for col, fn in ((3, mp.sin), (4, mp.cos)):
        want = f(fn, x[m])
        assert (np.abs(out[m, col] - want) <= 2.0 * np.maximum(np.spacing(np.abs(want)), 1e-22)).all()
    big = np.array([1e6, 1e9, 3e15])
    ob = g.eval_math(big)
    assert np.abs(ob[:, 3] - np.sin(big)).max() < 1e-15 and np.abs(ob[:, 4] - np.cos(big)).max() < 1e-15  # library fallback
    m = (np.abs(x) > 1e-290) & (np.abs(x) < 1e290)
    assert ulp(out[m, 5], 1.0 / x[m]).max() <= 1.0
    assert ulp(out[m, 6], f(lambda t: 1 / mp.sqrt(t), np.abs(x[m]))).max() <= 2.0
    assert ulp(out[m, 7], np.sqrt(np.abs(x[m]))).max() <= 1.0
    edge = g.eval_math(np.array([-np.inf, -1e4, -800.0]))
    assert (edge[:, 0] == 0).all() and (edge[:, 1] == -1).all()
