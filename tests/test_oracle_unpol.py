"""Pins U1-U3 of the oracle's unpolarized transfer (oracle/ref_unpol.hpp; reading R-12)."""
import os
import numpy as np

from test_oracle_transfer import CAM, L_UNIT


def _slab(ref, inc, unpol, eps=0.01, **slab):
    c = ref.Ctx(**dict(CAM, spin=0.0, flat_metric=1, inclination_deg=inc, nx=2, ny=2, fov=8.0, eps=eps))
    c.load_slab(**slab)
    c.set_unpolarized(unpol)
    return c.make_pixels()


def test_U1_closed_forms_of_the_scalar_equation(ref):
    # optically thin Gaussian slab: I = j sqrt(2 pi) H / cos(angle), second order in eps
    inc, H, j = 40.0, 3.0, 2.5e-18
    al = np.array([-2.0, 2.0, -2.0, 2.0]); be = np.array([-2.0, -2.0, 2.0, 2.0])
    ci, si = np.cos(np.radians(inc)), np.sin(np.radians(inc))
    exact = j * np.sqrt(2 * np.pi) * H * L_UNIT * np.sqrt(1 + (al ** 2 + be ** 2) / 1e6) / (ci - be / 1000.0 * si)
    e = {eps: _slab(ref, inc, True, eps=eps, H=H, profile=1, j=(j, 0, 0, 0))["I"] / exact - 1 for eps in (0.02, 0.01)}
    assert np.all(np.abs(e[0.01]) < 1.5e-4) and np.all((e[0.02] / e[0.01] > 3.5) & (e[0.02] / e[0.01] < 4.5))
    # emission and absorption: I = (j/alpha)(1 - e^-tau) with the code's own tau; thick limit j/alpha
    inc, H, j, a = 30.0, 2.0, 4.0e-17, 6.0e-13
    o = _slab(ref, inc, True, H=H, profile=1, j=(j, 0, 0, 0), alpha=(a, 0, 0, 0))
    tau = a * np.sqrt(2 * np.pi) * H * L_UNIT / np.cos(np.radians(inc))
    assert np.allclose(o["tau"], tau, rtol=4e-3)
    assert np.allclose(o["I"], j / a * (1 - np.exp(-o["tau"])), rtol=1e-12)   # exact for a shared profile, any steps
    o = _slab(ref, inc, True, H=H, profile=1, j=(j, 0, 0, 0), alpha=(40 * a, 0, 0, 0))
    assert np.allclose(o["I"], j / (40 * a), rtol=1e-12)
    assert all(np.all(o[k] == 0) for k in ("Q", "U", "V", "tauF"))


def test_U2_equals_the_polarized_I_when_nothing_couples_to_it(ref):
    # alpha_Q = alpha_U = alpha_V = 0: the I row of the 4x4 system is the scalar equation, whatever j_QUV and rho do
    kw = dict(H=2.0, profile=1, psi_deg=25.0, j=(3e-17, 1e-17, -5e-18, 2e-18), alpha=(5e-13, 0, 0, 0), rho=(3e-12, -1e-12, 6e-12))
    a = _slab(ref, 35.0, False, **kw)
    b = _slab(ref, 35.0, True, **kw)
    assert np.allclose(a["I"], b["I"], rtol=1e-12) and np.array_equal(a["tau"], b["tau"])
    assert np.abs(a["Q"]).max() > 0 and np.all(b["Q"] == 0)
    # ... and differs once alpha_Q couples I to Q
    kw["alpha"] = (5e-13, 3e-13, 0, 0)
    a = _slab(ref, 35.0, False, **kw); b = _slab(ref, 35.0, True, **kw)
    assert np.all(np.abs(a["I"] / b["I"] - 1) > 1e-3)


def test_U3_adaf_image_close_to_polarized_I_and_same_geodesics(ref):
    nt = os.cpu_count() or 1
    c = ref.Ctx(**CAM); c.load_adaf()
    a = c.make_pixels(nthreads=nt)
    c.set_unpolarized(True)
    b = c.make_pixels(nthreads=nt)
    assert np.array_equal(a["nsteps"], b["nsteps"]) and np.array_equal(a["nturn"], b["nturn"])
    assert np.allclose(a["tau"], b["tau"], rtol=1e-12, atol=0)
    # the polarized I differs by the coupling terms alpha_Q Q + alpha_V V <= alpha_I I: a fraction of the (small)
    # optical depth, plus the norm defect of the discrete parallel transport that only the polarized solution
    # carries (second-order scheme: pin T1 bounds it by 2e-3 at eps = 0.01)
    rel = np.abs(a["I"] - b["I"]) / a["I"]
    assert np.all(rel <= a["tau"] + 3e-3) and abs(a["I"].sum() / b["I"].sum() - 1) < 2e-3
    assert np.all(b["I"] > 0) and np.all(b["Q"] == 0) and np.all(b["V"] == 0)
    c.set_unpolarized(False)
    again = c.make_pixels(nthreads=nt)
    assert all(np.array_equal(a[k], again[k]) for k in a)
