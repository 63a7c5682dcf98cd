"""Pins G1, G2 for the oracle's metric and connection.

Nothing here retypes the oracle's formulas: the checks are textbook special cases (Schwarzschild in
ingoing Eddington-Finkelstein form, Minkowski), the vacuum Einstein equations R_mn = 0 for a != 0,
metric compatibility of the connection against finite differences, and the horizon / determinant.
"""
import numpy as np
import pytest

A = 0.9375
PTS = [(np.log(3.0), 0.31, 0.4), (np.log(1.6), 0.52, 2.0), (np.log(40.0), 0.11, 5.0), (np.log(7.0), 0.77, 1.0)]


def fd(fun, X, k, h):
    Xp = np.array(X, float); Xm = np.array(X, float)
    Xp[k] += h; Xm[k] -= h
    return (fun(Xp) - fun(Xm)) / (2 * h)


def test_G1_schwarzschild_is_ingoing_eddington_finkelstein(ref):
    # textbook: ds^2 = -(1-2/r) dt^2 + (4/r) dt dr + (1+2/r) dr^2 + r^2 dOmega^2, with r = e^X1, theta = pi X2 (h = 1)
    for (x1, x2, x3) in PTS:
        r, th = np.exp(x1), np.pi * x2
        g = ref.gcov(0.0, 1.0, [0, x1, x2, x3])
        J = np.array([1.0, r, np.pi, 1.0])
        ef = np.zeros((4, 4))
        ef[0, 0] = -(1 - 2 / r); ef[0, 1] = ef[1, 0] = 2 / r; ef[1, 1] = 1 + 2 / r
        ef[2, 2] = r * r; ef[3, 3] = (r * np.sin(th)) ** 2
        assert np.allclose(g, ef * np.outer(J, J), rtol=1e-14, atol=1e-14)


def test_G1_flat_switch_is_minkowski(ref):
    # with f = 0 and a = 0 the line element is flat: dr^2 + r^2 dth^2 + r^2 sin^2 dphi^2 - dt^2
    x1, x2, x3 = np.log(5.0), 0.3, 1.0
    r, th = 5.0, np.pi * 0.3
    g = ref.gcov(0.0, 1.0, [0, x1, x2, x3], flat=1)
    expect = np.diag([-1.0, r * r, (np.pi * r) ** 2, (r * np.sin(th)) ** 2])
    assert np.allclose(g, expect, rtol=1e-14, atol=1e-14)
    # and its Riemann-free connection still has the textbook spherical entries, e.g. Gamma^r_thth = -r
    G = ref.conn(0.0, 1.0, [0, x1, x2, x3], flat=1)
    # in (X1,X2): Gamma^X1_X2X2 = (dth/dX2)^2 Gamma^r_thth / (dr/dX1) = -pi^2
    assert abs(G[1, 2, 2] + np.pi ** 2) < 1e-12
    assert abs(G[2, 1, 2] - 1.0) < 1e-12  # Gamma^th_r th = 1/r  ->  Gamma^X2_X1X2 = r * 1/r


@pytest.mark.parametrize("h", [1.0, 0.3])
def test_G1_inverse_determinant_horizon(ref, h):
    for (x1, x2, x3) in PTS:
        X = [0, x1, x2, x3]
        g = ref.gcov(A, h, X); gi = ref.gcon(A, h, X)
        assert np.allclose(g @ gi, np.eye(4), atol=1e-12)
        assert np.allclose(g, g.T) and np.allclose(gi, gi.T, atol=1e-13)
        # Kerr: sqrt(-g) = Sigma sin(theta) in (t,r,theta,phi); times the Jacobian r * dtheta/dX2
        r = np.exp(x1); th = ref.lib().ipole_ref_theta_of_x2(h, x2)
        dth = (ref.lib().ipole_ref_theta_of_x2(h, x2 + 1e-6) - ref.lib().ipole_ref_theta_of_x2(h, x2 - 1e-6)) / 2e-6
        Sig = r * r + A * A * np.cos(th) ** 2
        assert np.sqrt(-np.linalg.det(g)) == pytest.approx(Sig * np.sin(th) * r * dth, rel=1e-8)
    # the horizon is where g^{rr} = Delta/Sigma vanishes: r_h = 1 + sqrt(1 - a^2)
    rh = 1 + np.sqrt(1 - A * A)
    gi = ref.gcon(A, h, [0, np.log(rh), 0.37, 0.0])
    assert abs(gi[1, 1]) < 1e-13
    assert ref.gcon(A, h, [0, np.log(rh * 1.01), 0.37, 0.0])[1, 1] > 0


@pytest.mark.parametrize("h", [1.0, 0.3])
def test_G2_connection_metric_compatible_and_symmetric(ref, h):
    for (x1, x2, x3) in PTS:
        X = np.array([0, x1, x2, x3])
        G = ref.conn(A, h, X); g = ref.gcov(A, h, X); dg = ref.dgcov(A, h, X)
        assert np.allclose(G, np.transpose(G, (0, 2, 1)), atol=1e-14)
        Glow = np.einsum("lk,kmn->lmn", g, G)  # Gamma_{l m n}
        # d_k g_{mn} = Gamma_{m k n} + Gamma_{n k m}
        ident = np.transpose(Glow, (1, 0, 2)) + np.transpose(Glow, (1, 2, 0))
        assert np.allclose(dg, ident, rtol=1e-11, atol=1e-11 * np.abs(dg).max())
        for k in range(4):
            num = fd(lambda Y: ref.gcov(A, h, Y), X, k, 1e-5)
            assert np.allclose(num, dg[k], rtol=1e-7, atol=1e-7 * max(1.0, np.abs(dg).max()))


def ricci(ref, a, h, X, flat=0):
    hh = 2e-4
    G = ref.conn(a, h, X, flat)
    dG = np.zeros((4, 4, 4, 4))  # dG[k][l][m][n] = d_k Gamma^l_mn
    for k in (1, 2):
        Xp = np.array(X, float); Xm = np.array(X, float); Xp2 = np.array(X, float); Xm2 = np.array(X, float)
        Xp[k] += hh; Xm[k] -= hh; Xp2[k] += 2 * hh; Xm2[k] -= 2 * hh
        dG[k] = (8 * (ref.conn(a, h, Xp, flat) - ref.conn(a, h, Xm, flat))
                 - (ref.conn(a, h, Xp2, flat) - ref.conn(a, h, Xm2, flat))) / (12 * hh)
    R = np.einsum("llmn->mn", dG) - np.einsum("nlml->mn", dG) \
        + np.einsum("lls,smn->mn", G, G) - np.einsum("lns,sml->mn", G, G)
    return R, G


@pytest.mark.parametrize("h", [1.0, 0.3])
def test_G2_kerr_is_a_vacuum_solution(ref, h):
    # R_mn = 0 (Kerr 1963): fails for any wrong component, sign, or derivative in metric or connection
    for (x1, x2, x3) in PTS:
        X = [0, x1, x2, x3]
        R, G = ricci(ref, A, h, X)
        scale = np.abs(G).max() ** 2
        assert np.abs(R).max() < 1e-8 * scale, (X, np.abs(R).max(), scale)
    R, G = ricci(ref, 0.5, h, [0, np.log(4.0), 0.4, 0.0], flat=1)
    assert np.abs(R).max() < 1e-8 * np.abs(G).max() ** 2


def test_isco_radius_textbook_values(ref):
    # Bardeen, Press & Teukolsky 1972: r_isco = 6 (a=0), 1 (a->1); 2.0442 for a = 0.9375 (SURVEY c-5)
    assert ref.lib().ipole_ref_isco(0.0) == pytest.approx(6.0, abs=1e-12)
    assert ref.lib().ipole_ref_isco(1.0 - 1e-12) == pytest.approx(1.0, abs=2e-4)
    r = ref.lib().ipole_ref_isco(A)
    assert r == pytest.approx(2.0442, abs=1e-4)
    # circular equatorial orbit marginally stable: d^2 V/dr^2 = 0  <=>  r^2 - 6 r + 8 a sqrt(r) - 3 a^2 = 0
    assert abs(r * r - 6 * r + 8 * A * np.sqrt(r) - 3 * A * A) < 1e-12


def test_theta_map_roundtrip(ref):
    L = ref.lib()
    for h in (1.0, 0.3):
        for th in (0.2, 1.0, np.pi / 3, 2.9):
            assert L.ipole_ref_theta_of_x2(h, L.ipole_ref_x2_of_theta(h, th)) == pytest.approx(th, abs=1e-14)
    assert L.ipole_ref_theta_of_x2(0.3, 0.5) == pytest.approx(np.pi / 2)
