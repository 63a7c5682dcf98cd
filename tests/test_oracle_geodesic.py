"""Pins G3-G6 for the oracle's camera and geodesic integrator.

Checks against what the mathematics fixes: the Killing/Carter constants of Kerr geodesics and the null
condition (with the 4th-order convergence of RK4), Synge's closed form for the Schwarzschild shadow seen
from a finite distance, Bardeen's capture criterion for Kerr, Einstein's weak-field deflection 4/b.
"""
import numpy as np
import pytest

A = 0.9375
CAM = dict(spin=A, inclination_deg=60.0, r_cam=1000.0, fov=40.0, nx=32, ny=32, freq_hz=230e9)


def constants(ref, a, h, X, K):
    g = ref.gcov(a, h, X)
    kc = g @ K
    th = ref.lib().ipole_ref_theta_of_x2(h, X[2])
    dth = np.pi * (1 + (1 - h) * np.cos(2 * np.pi * X[2]))
    E, L = -kc[0], kc[3]
    kth = kc[2] / dth
    Q = kth ** 2 + np.cos(th) ** 2 * (L * L / np.sin(th) ** 2 - a * a * E * E)
    terms = np.abs(np.outer(K, K) * g).sum()
    return E, L, Q, (K @ kc) / terms


def test_camera_tetrad_orthonormal_and_ray_null(ref):
    for h, inc in ((1.0, 60.0), (0.3, 20.0)):
        c = ref.Ctx(**dict(CAM, inclination_deg=inc, hslope=h))
        X, e = c.camera_tetrad()
        g = ref.gcov(A, h, X)
        eta = e @ g @ e.T
        assert np.allclose(eta, np.diag([-1, 1, 1, 1]), atol=1e-13)
        assert np.exp(X[1]) == pytest.approx(1000.0) and ref.lib().ipole_ref_theta_of_x2(h, X[2]) == pytest.approx(np.radians(inc))
        # static observer; e3 radial outward, e2 toward the axis (decreasing X2), e1 along +phi; right-handed
        assert e[0, 1] == 0 and e[0, 2] == 0 and e[0, 3] == 0 and e[0, 0] > 0
        assert e[3, 1] > 0 and e[2, 2] < 0 and e[1, 3] > 0
        assert np.linalg.det(e) > 0  # (e0,e1,e2,e3) vs (t,X1,X2,X3): e1~phi, e2~-theta, e3~r  => even permutation * (-1)^... > 0
        for (i, j) in ((0, 0), (31, 5), (16, 16)):
            Xr, K = c.camera_ray(i, j)
            assert abs(K @ g @ K) < 1e-14
            assert -(K @ g @ e[0]) == pytest.approx(1.0, abs=1e-14)  # unit energy in the camera frame
        # pixel (i,j) -> offsets: alpha = (i + 1/2 - nx/2) fov/nx.  Bardeen: L_z/E = -alpha sin(i); the image
        # centre (alpha = 0) looks along the Kerr-Schild radial direction d_X1, which carries L_z = g_{r phi} =
        # -a sin^2(i): the Kerr-Schild camera sits at Cartesian y = a sin(i), so the image is shifted by that much
        Xr, K = c.camera_ray(31, 16)
        E, L, Q, _ = constants(ref, A, h, Xr, K)
        alpha = (31 + 0.5 - 16) * 40.0 / 32
        si = np.sin(np.radians(inc))
        assert L / E == pytest.approx(-(alpha * si + A * si * si), rel=2e-3)
        Xr, K = c.camera_ray(16, 31)  # beta > 0 shows what lies above the axis: that photon arrives moving down
        assert K[2] > 0


def test_G3_constants_of_motion_converge_at_fourth_order(ref):
    drift = {}
    for eps in (0.01, 0.005, 0.00125):
        c = ref.Ctx(**dict(CAM, eps=eps, max_steps=200000))
        worst = 0.0
        for (i, j) in ((3, 4), (12, 15), (15, 17), (20, 16), (16, 20), (18, 14), (25, 28), (14, 14)):
            X0, K0 = c.camera_ray(i, j)
            X, K, dl, nt, st = c.trace(X0, K0, cap=200000)
            E0, L0, Q0, _ = constants(ref, A, 1.0, X[0], K[0])
            for s in (len(dl) // 2, len(dl)):
                E, L, Q, kk = constants(ref, A, 1.0, X[s], K[s])
                worst = max(worst, abs(E / E0 - 1), abs(L - L0) / max(abs(L0), E0), abs(Q - Q0) / max(abs(Q0), E0 ** 2), abs(kk))
        drift[eps] = worst
    # 4th order: halving eps gains ~16x; at eps_chk = 1.25e-3 the north-star level 1e-10 is met
    assert drift[0.01] / drift[0.005] > 10.0
    assert drift[0.005] / drift[0.00125] > 100.0
    assert drift[0.00125] < 1e-10
    assert drift[0.01] < 1e-6


def captured(c, alpha, beta):
    X0, K0 = c.camera_ray_ab(alpha, beta)
    X, K, dl, nt, st = c.trace(X0, K0)
    return st == 1


def test_G4_schwarzschild_shadow_radius_synge(ref):
    # Synge (1966): a static observer at r_cam sees the shadow edge at sin(psi) = sqrt(27) sqrt(1 - 2/r_cam) / r_cam;
    # the pin-hole camera maps it to alpha_c = r_cam tan(psi) (-> sqrt(27) as r_cam -> infinity)
    c = ref.Ctx(**dict(CAM, spin=0.0, inclination_deg=90.0))
    rc = 1000.0
    synge = rc * np.tan(np.arcsin(np.sqrt(27.0 * (1 - 2 / rc)) / rc))
    lo, hi = 4.0, 6.0
    for _ in range(36):
        mid = 0.5 * (lo + hi)
        if captured(c, mid, 0.0):
            lo = mid
        else:
            hi = mid
    assert 0.5 * (lo + hi) == pytest.approx(synge, abs=2e-6)
    assert abs(synge - np.sqrt(27)) < 2e-2
    # a = 0: the edge is a circle (same radius along beta and along the diagonal)
    for ang in (np.pi / 3, np.pi / 4, -2.0):  # not along the polar axis, where the coordinates are singular
        assert captured(c, (synge - 1e-4) * np.cos(ang), (synge - 1e-4) * np.sin(ang))
        assert not captured(c, (synge + 1e-4) * np.cos(ang), (synge + 1e-4) * np.sin(ang))


def test_G5_kerr_shadow_matches_bardeen_capture_criterion(ref):
    # A photon with xi = L/E, eta = Q/E^2 coming from infinity is captured iff the radial potential
    # R(r) = (r^2 + a^2 - a xi)^2 - Delta [eta + (xi - a)^2] has no zero outside the horizon (Bardeen 1973).
    c = ref.Ctx(**CAM)
    rh = 1 + np.sqrt(1 - A * A)
    rr = np.concatenate([np.linspace(rh, 12.0, 200001), np.linspace(12.0, 1000.0, 20001)])
    Del = rr * rr - 2 * rr + A * A
    rng = np.random.default_rng(5)
    n_cap = 0
    for _ in range(160):
        al, be = rng.uniform(-9, 9, 2)
        X0, K0 = c.camera_ray_ab(al, be)
        E, L, Q, _ = constants(ref, A, 1.0, X0, K0)
        xi, eta = L / E, Q / E ** 2
        Rmin = (((rr * rr + A * A - A * xi) ** 2 - Del * (eta + (xi - A) ** 2)) / rr ** 4).min()
        if abs(Rmin) < 2e-4:
            continue  # too close to the critical curve for the sampled minimum to decide
        cap = captured(c, al, be)
        n_cap += cap
        assert cap == (Rmin > 0), (al, be, Rmin)
    assert 20 < n_cap < 140
    # prograde side (alpha < 0 for a > 0 with L/E = -alpha sin i) lies closer to the centre: the D-shape
    def edge(sign):
        lo, hi = 0.0, 9.0
        for _ in range(30):
            mid = 0.5 * (lo + hi)
            if captured(c, sign * mid, 0.0):
                lo = mid
            else:
                hi = mid
        return lo
    assert edge(-1.0) < edge(+1.0) - 1.0


def test_G6_weak_field_deflection(ref):
    # Einstein: deflection 4/b for b >> 1 (next order 15 pi / (4 b^2)); straight line from r_cam back to r_cam
    # sweeps pi - 2 asin(b/r_cam) in azimuth
    rc, b = 1.0e5, 1000.0
    c = ref.Ctx(**dict(CAM, spin=0.0, inclination_deg=90.0, r_cam=rc, eps=0.005))
    X0, K0 = c.camera_ray_ab(b, 0.0)
    X, K, dl, nt, st = c.trace(X0, K0)
    assert st == 2
    # interpolate the last step to r = rc exactly
    x1a, x1b = X[-2, 1], X[-1, 1]
    w = (np.log(rc) - x1a) / (x1b - x1a)
    dphi = abs((1 - w) * X[-2, 3] + w * X[-1, 3] - X[0, 3])
    defl = dphi - (np.pi - 2 * np.arcsin(b / rc))
    assert defl == pytest.approx(4 / b + 15 * np.pi / (4 * b * b), rel=3e-3)
    assert abs(X[:, 2] - 0.5).max() < 1e-12  # stays in the equatorial plane


def test_step_rule_stop_conditions_and_turning_points(ref):
    c = ref.Ctx(**CAM)
    rh = 1 + np.sqrt(1 - A * A)
    X0, K0 = c.camera_ray(16, 17)  # inside the shadow
    X, K, dl, nt, st = c.trace(X0, K0)
    assert st == 1 and np.exp(X[-1, 1]) <= 1.05 * rh < np.exp(X[-2, 1])
    X0, K0 = c.camera_ray(2, 29)
    X, K, dl, nt, st = c.trace(X0, K0)
    assert st == 2 and np.exp(X[-1, 1]) > 1000.0 >= np.exp(X[-2, 1]) and nt == 1
    # the documented step rule: 1/dl = (|K1| + |K3| + |K2|/min(X2,1-X2)) / eps
    for s in (0, len(dl) // 2, len(dl) - 1):
        inv = (abs(K[s, 1]) + abs(K[s, 3]) + abs(K[s, 2]) / min(X[s, 2], 1 - X[s, 2])) / 0.01
        assert dl[s] == pytest.approx(1 / inv, rel=1e-12)
    assert np.all(dl > 0) and np.all(np.diff(X[:, 0]) < 0)  # integrated backward in time
    # max_steps: the ray ends there and is flagged
    c2 = ref.Ctx(**dict(CAM, max_steps=100, nx=2, ny=2))
    c2.load_adaf()
    o = c2.make_pixels()
    assert np.all(o["nsteps"] == 100) and np.all(o["nturn"] & 0x80)
