"""Adaptive ray tracing on the GPU (R-11), pytest -m gpu:
ipole_make_image_adaptive against the oracle's algorithm (oracle/adaptive_ref.py) driven by the oracle's own rays."""
import numpy as np
import pytest

from oracle import adaptive_ref
from paper_2302_02733_b200 import workloads as W
from test_gpu_parity import to_np, ipole, NTHREADS  # noqa: F401

pytestmark = pytest.mark.gpu


def oracle_tracer(r):
    def trace(pix):
        o = r.make_pixels(pix, nthreads=NTHREADS)
        return np.stack([o[k] for k in "IQUV"], axis=1)
    return trace


def compare(got, state, img_ref, state_ref, label):
    same = state == state_ref
    assert same.mean() >= 0.999, (label, "refinement decisions", same.mean())
    I0 = img_ref[0]
    lit = (I0 > 0) & same
    err = np.zeros(I0.shape)
    for k, name in enumerate("IQUV"):
        g = got[name].reshape(I0.shape)
        assert (g[(I0 == 0) & same] == 0).all(), (label, "dark", name)
        err[lit] = np.maximum(err[lit], np.abs(g - img_ref[k])[lit] / I0[lit])
    assert (err <= 1e-7).mean() >= 0.999 and err.max() <= 1e-4, (label, np.sort(err.ravel())[-5:])
    return err.max()


@pytest.mark.parametrize("nx,ny,L,tol", [(64, 64, 3, 2e-2), (37, 23, 2, 5e-3), (5, 3, 3, 1e-2), (2, 2, 1, 1e-2), (9, 2, 2, 0.0)])
def test_adaptive_matches_the_oracle_algorithm(ipole, ref, nx, ny, L, tol):
    cam = W.camera("adaf", 8); cam.update(nx=nx, ny=ny)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    r = ref.Ctx(**cam); r.load_adaf(**W.ADAF)
    # the image spans many decades (thermal cut-off): a purely relative test would refine the faint outskirts for
    # ever, so the absolute floor is 1e-3 of the brightest pixel
    atol = 1e-3 * float(g.make_image()["I"].max())
    img_ref, state_ref, counts = adaptive_ref.adaptive_image(oracle_tracer(r), nx, ny, L, tol, atol)
    out, info = g.make_image_adaptive(L, tol, atol)
    got = to_np({k: out[k] for k in "IQUV"})
    compare(got, out["state"], img_ref, state_ref, "adaptive %dx%d" % (nx, ny))
    assert info["n_traced_level"] == counts and info["n_traced"] == sum(counts) == int((out["state"] == 1).sum())
    assert 0 < info["n_traced"] <= nx * ny and (out["state"] > 0).all()
    assert info["n_traced"] < nx * ny or nx * ny < 100
    # host buffers: same bits
    h, _ = g.make_image_adaptive(L, tol, atol, host=True)
    for k in "IQUV":
        assert np.array_equal(h[k].ravel(), got[k]), k
    assert np.array_equal(h["state"], out["state"])
    # flux of the finished image
    L_ = 6.6742e-8 * 4.1e6 * 1.989e33 / 2.99792458e10 ** 2
    dom = (cam["fov"] / nx * L_ / (8000.0 * 3.085678e18)) ** 2 * 1e23
    assert np.allclose(info["flux_jy"], [got[k].sum() * dom for k in "IQUV"], rtol=1e-12, atol=1e-12 * got["I"].sum() * dom)
    # the path-free variant goes through the same entry
    g.set_path_free(True)
    out2, info2 = g.make_image_adaptive(L, tol, atol)
    assert info2["n_traced"] > 0 and np.isfinite(out2["I"].cpu().numpy()).all()
    assert abs(float(out2["I"].sum()) / got["I"].sum() - 1) < 2e-3


def test_adaptive_limits_and_quality(ipole):
    cam = W.camera("adaf", 128)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    full = to_np(g.make_image())
    # zero tolerance: every pixel is traced and equals the full image bit for bit
    out, info = g.make_image_adaptive(3, 0.0)
    assert (out["state"] == 1).all() and info["n_traced"] == 128 * 128
    for k in "IQUV":
        assert np.array_equal(out[k].cpu().numpy().ravel(), full[k]), k
    # infinite tolerance: only the two coarsest levels are traced (stride 4 lattice + last row/column)
    out, info = g.make_image_adaptive(3, 1e300)
    assert info["n_traced"] == 33 * 33 and info["n_traced_level"][2:] == [0, 0]
    # a useful tolerance: far fewer rays, small error; traced pixels carry the exact values
    out, info = g.make_image_adaptive(3, 2e-2, 1e-3 * full["I"].max())
    frac = info["n_traced"] / (128 * 128)
    I = out["I"].cpu().numpy().ravel()
    err = np.abs(I - full["I"]) / full["I"].max()
    tr = out["state"].ravel() == 1
    assert np.array_equal(I[tr], full["I"][tr])
    assert frac < 0.2 and err.max() < 5e-3 and np.percentile(err, 99) < 1e-3
    assert abs(I.sum() / full["I"].sum() - 1) < 3e-3


def test_adaptive_grid_dark_regions_and_errors(ipole, ref):
    desc, fields = W.fm_torus_grid(72, 32, 32)
    cam = W.camera("grid", 48)
    g = ipole.Ipole(**cam); g.load_grid(desc, fields)
    r = ref.Ctx(**cam); r.load_grid(desc, fields)
    atol = 1e-3 * float(g.make_image()["I"].max())
    img_ref, state_ref, counts = adaptive_ref.adaptive_image(oracle_tracer(r), 48, 48, 2, 1e-2, atol)
    out, info = g.make_image_adaptive(2, 1e-2, atol)
    compare(to_np({k: out[k] for k in "IQUV"}), out["state"], img_ref, state_ref, "adaptive grid")
    assert info["n_traced"] < 48 * 48          # the dark corners are not refined
    for bad in (dict(levels=0), dict(levels=13), dict(rel_tol=-1.0)):
        with pytest.raises(ipole.IpoleError):
            g.make_image_adaptive(**bad)
    g.set_camera(nx=9, ny=1)            # a lattice cell needs two lines each way
    with pytest.raises(ipole.IpoleError):
        g.make_image_adaptive()
    g0 = ipole.Ipole(**cam)
    with pytest.raises(ipole.IpoleError) as ei:
        g0.make_image_adaptive()
    assert ei.value.code == ipole.ENOMODEL
