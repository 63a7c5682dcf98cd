"""Pins PF1-PF5 of the oracle's path-free bidirectional variant (reading R-10, oracle/ref_pathfree.hpp).

What fixes the variant from outside the oracle: the geodesic through the backward end point is unique, so the forward
pass must carry the same constants of motion back to the camera radius (PF2); the closed-form slab solutions hold for
any partition of the ray, so they hold for the forward pass and its end-point tetrad too (PF3); and the paper's own
statement that stored-path and path-free images differ negligibly at the usual epsilon (PF4).
"""
import os
import numpy as np
import pytest

from test_oracle_geodesic import constants
from test_oracle_transfer import CAM, A, L_UNIT


def test_PF1_observer_tetrad_is_the_camera_construction(ref):
    for h, inc in ((1.0, 60.0), (0.3, 20.0)):
        c = ref.Ctx(**dict(CAM, inclination_deg=inc, hslope=h))
        Xc, e = c.camera_tetrad()
        assert np.array_equal(c.observer_tetrad(Xc), e)
        # anywhere else: orthonormal, static, e3 outward, e2 toward the axis, e1 along +phi, right-handed
        X = np.array([0.0, np.log(37.0), 0.31, 2.0])
        t = c.observer_tetrad(X)
        g = ref.gcov(A, h, X)
        assert np.allclose(t @ g @ t.T, np.diag([-1, 1, 1, 1]), atol=1e-13)
        assert t[0, 1] == 0 and t[0, 2] == 0 and t[0, 3] == 0 and t[0, 0] > 0
        assert t[3, 1] > 0 and t[2, 2] < 0 and t[1, 3] > 0 and np.linalg.det(t) > 0


def test_PF2_forward_pass_is_the_same_geodesic_and_stops_at_the_camera_radius(ref):
    drift = {}
    for eps in (0.01, 0.005):
        c = ref.Ctx(**dict(CAM, eps=eps))
        worst = 0.0
        for (i, j) in ((3, 4), (12, 15), (13, 14), (20, 16), (16, 20), (25, 28)):
            X0, K0 = c.camera_ray(i, j)
            X, K, dl, nt, st = c.trace(X0, K0)
            n = len(dl)
            Xf, Kf, dlf = c.retrace(X[n], K[n])
            m = len(dlf)
            assert np.array_equal(Xf[0], X[n]) and np.array_equal(Kf[0], K[n])
            # stop rule: the last step, and only the last, ends at r >= r_cam moving outward
            assert Xf[m, 1] >= X0[1] and Xf[m, 1] > Xf[m - 1, 1]
            out = (Xf[1:m, 1] >= X0[1]) & (Xf[1:m, 1] > Xf[0:m - 1, 1])
            assert not out.any()
            # it overshoots the camera by less than its last step (dr <= r K^1 dl)
            assert np.exp(Xf[m, 1]) - 1000.0 <= 1000.0 * abs(Kf[m - 1, 1]) * dlf[m - 1] * 1.01
            # steps are taken forward (+dl) with the rule evaluated at the point they start from
            assert np.all(dlf > 0)
            # the step counts may differ (rule evaluated at the other end of every interval) but only slightly
            assert abs(m - n) < 0.02 * n
            # same constants of motion as the camera ray all the way: the forward pass retraces that geodesic
            E0, L0, Q0, _ = constants(ref, A, 1.0, X0, K0)
            for s in (m // 3, m):
                E, L, Q, kk = constants(ref, A, 1.0, Xf[s], Kf[s])
                worst = max(worst, abs(E / E0 - 1), abs(L - L0) / max(abs(L0), E0), abs(Q - Q0) / max(abs(Q0), E0 ** 2), abs(kk))
            # ... and arrives on the camera's line of sight: at the end radius the angular offset from the camera
            # is what the ray's own slope gives over the overshoot, not more
            over = Xf[m, 1] - X0[1]
            assert abs(Xf[m, 2] - X0[2]) <= abs(Kf[m, 2] / Kf[m, 1]) * over * 1.05 + 1e-9
        drift[eps] = worst
    assert drift[0.01] < 2e-6
    assert drift[0.01] / drift[0.005] > 10.0   # fourth order, as for the backward pass (pin G3)


def _slab(ref, inc, eps=0.01, **slab):
    c = ref.Ctx(**dict(CAM, spin=0.0, flat_metric=1, inclination_deg=inc, nx=2, ny=2, fov=8.0, eps=eps))
    c.load_slab(**slab)
    c.set_path_free(True)
    return c.make_pixels()


def test_PF3_closed_form_slabs_through_the_forward_pass(ref):
    # optically thin Gaussian slab: I = j sqrt(2 pi) H / cos(angle to the normal), second-order convergence
    inc, H, j = 40.0, 3.0, 2.5e-18
    al = np.array([-2.0, 2.0, -2.0, 2.0]); be = np.array([-2.0, -2.0, 2.0, 2.0])
    ci, si = np.cos(np.radians(inc)), np.sin(np.radians(inc))
    exact = j * np.sqrt(2 * np.pi) * H * L_UNIT * np.sqrt(1 + (al ** 2 + be ** 2) / 1e6) / (ci - be / 1000.0 * si)
    err = {}
    for eps in (0.02, 0.01):
        o = _slab(ref, inc, eps=eps, H=H, profile=1, j=(j, 0, 0, 0))
        err[eps] = o["I"] / exact - 1
        assert np.all(o["V"] == 0)
    # a tetrad taken at the camera instead of the end point would be off by 2 (r_end - r_cam)/r_cam ~ 1e-2 here
    assert np.all(np.abs(err[0.01]) < 2e-4)
    assert np.all((err[0.02] / err[0.01] > 3.3) & (err[0.02] / err[0.01] < 4.7))
    # absorption: I = (j/alpha)(1 - e^-tau) with the code's own tau; optically thick limit j/alpha
    inc, H, j, a = 30.0, 2.0, 4.0e-17, 6.0e-13
    o = _slab(ref, inc, H=H, profile=1, j=(j, 0, 0, 0), alpha=(a, 0, 0, 0))
    tau = a * np.sqrt(2 * np.pi) * H * L_UNIT / np.cos(np.radians(inc))
    assert np.allclose(o["tau"], tau, rtol=4e-3)
    assert np.allclose(o["I"], j / a * (1 - np.exp(-o["tau"])), rtol=1e-5)
    o = _slab(ref, inc, H=H, profile=1, j=(j, 0, 0, 0), alpha=(40 * a, 0, 0, 0))
    assert np.allclose(o["I"], j / (40 * a), rtol=1e-9)
    # Faraday rotation: Q = jQ sin(rV x)/rV, U = jQ (1 - cos(rV x))/rV -- fixes the sense of the forward transport and
    # the orientation of the end-point tetrad
    inc, H, jQ = 50.0, 2.0, 1.0e-18
    x = np.sqrt(2 * np.pi) * H * L_UNIT / np.cos(np.radians(inc))
    rV = 2.2 / x
    o = _slab(ref, inc, H=H, profile=1, psi_deg=0.0, j=(2 * jQ, jQ, 0, 0), rho=(0, 0, rV))
    assert abs(o["Q"].mean() / (jQ * np.sin(2.2) / rV) - 1) < 2e-3
    assert abs(o["U"].mean() / (jQ * (1 - np.cos(2.2)) / rV) - 1) < 2e-3
    assert np.all(np.abs(o["V"]) < 1e-12 * o["I"])
    # Faraday conversion: U = jU sin(rQ x)/rQ, V = jU (1 - cos(rQ x))/rQ
    rQ = 1.3 / x
    o = _slab(ref, inc, H=H, profile=1, psi_deg=0.0, j=(2 * jQ, 0, jQ, 0), rho=(rQ, 0, 0))
    assert abs(o["U"].mean() / (jQ * np.sin(1.3) / rQ) - 1) < 2e-3
    assert abs(o["V"].mean() / (jQ * (1 - np.cos(1.3)) / rQ) - 1) < 2e-3


def test_PF4_images_differ_negligibly_from_the_stored_path(ref):
    """"for a typically adopted value of epsilon the differences in all Stokes parameter images produced
    by CPU and GPU codes are negligible"."""
    nt = os.cpu_count() or 1
    c = ref.Ctx(**CAM)   # W1: eps = 0.01
    c.load_adaf()
    a = c.make_pixels(nthreads=nt)
    c.set_path_free(True)
    b = c.make_pixels(nthreads=nt)
    assert np.array_equal(a["nsteps"], b["nsteps"]) and np.array_equal(a["nturn"], b["nturn"])   # backward pass unchanged
    tot = a["I"].sum()
    for k in "IQUV":
        assert np.all(np.isfinite(b[k]))
        assert abs(b[k].sum() - a[k].sum()) < 5e-4 * tot
    lit = a["I"] > 1e-6 * a["I"].max()
    rel = np.abs(b["I"] - a["I"])[lit] / a["I"][lit]
    assert np.median(rel) < 1e-5 and rel.max() < 2e-2
    rt = np.abs(b["tau"] - a["tau"]) / a["tau"]
    assert np.median(rt) < 1e-5 and rt.max() < 2e-2
    # invariant of the transfer equation holds for the variant as well
    assert np.all(b["I"] * (1 + 1e-12) >= np.sqrt(b["Q"] ** 2 + b["U"] ** 2 + b["V"] ** 2))


def test_PF5_vacuum_and_switch(ref):
    c = ref.Ctx(**dict(CAM, nx=2, ny=2, flat_metric=1, spin=0.0))
    c.load_slab(H=1e-9, j=(1, 0, 0, 0))
    c.set_path_free(True)
    o = c.make_pixels()
    assert np.all(o["I"] == 0) and np.all(o["tau"] == 0)
    # switching the variant off restores the stored-path result bit for bit
    c2 = ref.Ctx(**dict(CAM, nx=4, ny=4))
    c2.load_adaf()
    a = c2.make_pixels()
    c2.set_path_free(True); c2.make_pixels(); c2.set_path_free(False)
    b = c2.make_pixels()
    assert all(np.array_equal(a[k], b[k]) for k in a)
