"""Pins E1-E6 of the oracle's numerically integrated eDF coefficients (oracle/ref_edf.hpp; reading R-13).

References outside the oracle: scipy's K_nu and adaptive quadrature for the kernels F, G, H; the published thermal fits
and Kirchhoff's law (Rayleigh-Jeans) for the Maxwell-Juettner case; the Rybicki & Lightman power-law closed forms
(6.36 emission, 6.53 absorption) for the tail of the kappa distribution; scipy quadrature of the same integrands with an
independent rule for the convergence of the midpoint rule; Mellin transforms of the kernel H (Gamma functions) for j_V and
alpha_V of the power-law tail."""
import numpy as np
import pytest
from scipy import integrate, special

EE, CL, ME, KB, HPL = 4.80320680e-10, 2.99792458e10, 9.1093826e-28, 1.3806505e-16, 6.6260693e-27


def _tail(nu, x):
    """int_x^inf K_nu(t) dt with mpmath (20 digits), the range cut at every decade: K_nu ~ t^-nu near 0"""
    import mpmath as mp
    mp.mp.dps = 20
    pts = [mp.mpf(x)]
    d = 10.0 ** np.floor(np.log10(x) + 1)
    while d < 50.0:
        if d > x:
            pts.append(mp.mpf(d))
        d *= 10.0
    pts.append(mp.inf)
    return float(mp.quad(lambda t: mp.besselk(nu, t), pts))


def _F(x):
    return x * _tail(5.0 / 3.0, x)


def _H(x):
    return x * special.kv(1.0 / 3.0, x) + _tail(1.0 / 3.0, x)


@pytest.mark.parametrize("x", [1e-6, 1e-3, 0.03, 0.29, 1.0, 4.0, 30.0, 300.0])
def test_E1_kernels_vs_scipy(ref, x):
    F, G, H = ref.synchrotron_kernels(x)
    assert F == pytest.approx(_F(x), rel=2e-10)
    assert G == pytest.approx(x * special.kv(2.0 / 3.0, x), rel=2e-12)
    assert H == pytest.approx(_H(x), rel=2e-10)


@pytest.mark.parametrize("Th,x", [(10.0, 1.0), (30.0, 30.0), (3.0, 100.0), (20.0, 1e3)])
def test_E2_maxwell_juettner_reproduces_the_thermal_fits_and_kirchhoff(ref, Th, x):
    ne, B, th = 2.0e5, 9.0, 1.05
    nuB = EE * B / (2 * np.pi * ME * CL)
    nu = x * 1.5 * Th * Th * nuB * np.sin(th)
    fit = ref.coefficients(ne, Th, B, np.cos(th), nu)
    num = ref.coefficients_edf(1, ne, Th, B, np.cos(th), nu)
    # the fits are good to ~1 % (pin T8); at Theta_e = 3 they also carry their ultra-relativistic approximation
    tol = 0.02 if Th >= 10 else 0.08
    assert num[0] == pytest.approx(fit[0], rel=tol)
    assert num[1] == pytest.approx(fit[1], rel=tol)
    assert num[2] == pytest.approx(fit[2], rel=2 * tol)
    # Kirchhoff in the Rayleigh-Jeans limit (h nu << k T_e): alpha_S = j_S c^2 / (2 nu^2 Theta_e m c^2), to the accuracy of
    # the classical absorption formula, O(h nu / k T) ~ 1e-9 here, and of the quadrature
    for s in range(3):
        assert num[3 + s] == pytest.approx(num[s] / (2 * nu * nu * Th * ME), rel=2e-6)
    # Faraday coefficients are the thermal ones
    assert num[6] == fit[6] and num[7] == fit[7]


def test_E3_kappa_tends_to_maxwell_juettner(ref):
    ne, Th, B, th, nu = 1.0e5, 12.0, 15.0, 0.8, 230e9
    mj = ref.coefficients_edf(1, ne, Th, B, np.cos(th), nu)
    k6 = ref.coefficients_edf(2, ne, Th, B, np.cos(th), nu, kappa=1e6)
    assert np.allclose(k6[:6], mj[:6], rtol=2e-4, atol=0)
    k4 = ref.coefficients_edf(2, ne, Th, B, np.cos(th), nu, kappa=4.0)
    assert k4[0] > 2.0 * mj[0]                    # a real tail changes the answer (nu is above the thermal peak here)


def test_E4_kappa_tail_matches_the_power_law_closed_forms(ref):
    """gamma >> kappa w: n(gamma) -> N (kappa w)^(kappa+1) gamma^-p with p = kappa - 1.  Where the emission comes from that
    tail, j_I and alpha_I are the Rybicki & Lightman power-law results (6.36, 6.53) with that normalisation."""
    kappa, w, ne, B, th = 3.5, 3.0, 1.0e4, 0.5, 1.2
    p = kappa - 1.0
    nuB = EE * B / (2 * np.pi * ME * CL)
    # N from the normalisation integral (scipy, not the oracle's rule)
    nrm = integrate.quad(lambda g: g * np.sqrt(g * g - 1) * (1 + (g - 1) / (kappa * w)) ** -(kappa + 1), 1, np.inf, limit=400)[0]
    Kpl = ne / nrm * (kappa * w) ** (kappa + 1)       # n(gamma) ~ Kpl gamma^-p
    from scipy.special import gamma as Gm
    prev = None
    for gstar in (1e3, 3e3):                          # emission from gamma ~ gstar >> kappa w = 10.5
        nu = 1.5 * gstar ** 2 * nuB * np.sin(th)
        c = ref.coefficients_edf(2, ne, w, B, np.cos(th), nu, kappa=kappa, n_nodes=400)
        # R&L 6.36 divided by 4 pi (per steradian), with omega = 2 pi nu and N(E) dE = n(gamma) dgamma
        jpl = (np.sqrt(3) * EE ** 3 * Kpl * B * np.sin(th) / (4 * np.pi * ME * CL ** 2 * (p + 1)) * Gm(p / 4 + 19 / 12) * Gm(p / 4 - 1 / 12)
               * (2 * np.pi * ME * CL * nu / (3 * EE * B * np.sin(th))) ** (-(p - 1) / 2))
        # R&L 6.53 in the same variables
        apl = (np.sqrt(3) * EE ** 3 / (8 * np.pi * ME) * (3 * EE / (2 * np.pi * ME ** 3 * CL ** 5)) ** (p / 2) * Kpl * (ME * CL ** 2) ** (p - 1)
               * (B * np.sin(th)) ** ((p + 2) / 2) * Gm((3 * p + 2) / 12) * Gm((3 * p + 22) / 12) * nu ** (-(p + 4) / 2))
        dj, da = c[0] / jpl - 1, c[3] / apl - 1
        # the kappa distribution approaches the pure power law like (kappa+1) kappa w / gamma: -4 % at gamma* = 1000, -1.5 % at 3000
        assert abs(dj) < 0.08 and abs(da) < 0.08
        if prev is not None:
            assert abs(dj) < 0.45 * abs(prev[0]) and abs(da) < 0.45 * abs(prev[1])
        prev = (dj, da)
        # linear-polarization fraction of a power law: (p + 1) / (p + 7/3)
        assert c[1] / c[0] == pytest.approx((p + 1) / (p + 7.0 / 3.0), rel=0.03)
    assert abs(prev[0]) < 0.025 and abs(prev[1]) < 0.03


def _mellin_H(s):
    """int_0^inf x^(s-1) H(x) dx for H(x) = x K_1/3(x) + int_x^inf K_1/3, from int_0^inf x^(mu-1) K_nu = 2^(mu-2) Gamma((mu-nu)/2)
    Gamma((mu+nu)/2) (Gradshteyn & Ryzhik 6.561.16) and one integration by parts for the tail term."""
    from scipy.special import gamma as Gm
    return 2.0 ** (s - 1.0) * (1.0 + 1.0 / s) * Gm(0.5 * s + 1.0 / 3.0) * Gm(0.5 * s + 2.0 / 3.0)


def test_E6_kappa_tail_circular_coefficients_match_the_power_law_closed_forms(ref):
    """j_V and alpha_V of the kappa distribution where the tail n -> K gamma^-p emits: with x = nu/nu_c(gamma) the gamma
    integrals become Mellin transforms of H,
      j_V     = C (4 cot th / 3) K (1/2) xs^(-p/2)     M_H(p/2),
      alpha_V = C/(2 m_e nu^2) (4 cot th / 3) K (p+2) (1/2) xs^(-(p+1)/2) M_H((p+1)/2),      xs = nu / (1.5 nu_B sin th),
    products of Gamma functions -- no quadrature of the oracle's enters (the Mellin transform itself is checked here against
    scipy quadrature of the mpmath kernel)."""
    K13 = lambda t: special.kv(1.0 / 3.0, t)
    def Hq(x):      # (the tail in u = ln t below 1: K_1/3 ~ t^-1/3 there)
        lo = integrate.quad(lambda u: K13(np.exp(u)) * np.exp(u), np.log(x), 0.0, epsabs=0, epsrel=1e-10)[0] if x < 1.0 else 0.0
        return x * K13(x) + lo + integrate.quad(K13, max(x, 1.0), np.inf, epsabs=0, epsrel=1e-10)[0]
    assert Hq(0.29) == pytest.approx(_H(0.29), rel=1e-8)
    for s in (1.25, 1.75):
        num = integrate.quad(lambda u: np.exp(u * s) * Hq(np.exp(u)), np.log(1e-9), np.log(80.0), limit=200, epsabs=0, epsrel=1e-8)[0]
        assert num == pytest.approx(_mellin_H(s), rel=1e-6)
    kappa, w, ne, B, th = 3.5, 3.0, 1.0e4, 0.5, 1.2
    p = kappa - 1.0
    nuB = EE * B / (2 * np.pi * ME * CL)
    nrm = integrate.quad(lambda g: g * np.sqrt(g * g - 1) * (1 + (g - 1) / (kappa * w)) ** -(kappa + 1), 1, np.inf, limit=400)[0]
    Kpl = ne / nrm * (kappa * w) ** (kappa + 1)
    C = np.sqrt(3) * EE ** 3 * B * np.sin(th) / (4 * np.pi * ME * CL ** 2)
    cot43 = 4.0 / (3.0 * np.tan(th))
    prev = None
    for gstar in (1e3, 3e3):
        nu = 1.5 * gstar ** 2 * nuB * np.sin(th)
        xs = nu / (1.5 * nuB * np.sin(th))
        c = ref.coefficients_edf(2, ne, w, B, np.cos(th), nu, kappa=kappa, n_nodes=400)
        jV = C * cot43 * Kpl * 0.5 * xs ** (-p / 2) * _mellin_H(p / 2)
        aV = C / (2 * ME * nu * nu) * cot43 * Kpl * (p + 2) * 0.5 * xs ** (-(p + 1) / 2) * _mellin_H((p + 1) / 2)
        dj, da = c[2] / jV - 1, c[5] / aV - 1
        assert abs(dj) < 0.08 and abs(da) < 0.08, (dj, da)
        if prev is not None:
            assert abs(dj) < 0.45 * abs(prev[0]) and abs(da) < 0.45 * abs(prev[1])
        prev = (dj, da)
        # circular over total emission of a power law falls like 1/gamma*: j_V / j_I ~ cot th / gamma*
        assert 0.3 < (c[2] / c[0]) * gstar * np.tan(th) < 3.0
    assert abs(prev[0]) < 0.03 and abs(prev[1]) < 0.03
    # the sign follows cos th (the handedness of the gyration seen from the two sides of the field)
    cm = ref.coefficients_edf(2, ne, w, B, -np.cos(th), nu, kappa=kappa, n_nodes=400)
    assert cm[2] == pytest.approx(-c[2], rel=1e-12) and cm[5] == pytest.approx(-c[5], rel=1e-12)


def test_E5_midpoint_rule_converges_to_adaptive_quadrature(ref):
    """The rule (midpoint in ln x, 128 cells on [e^-16, e^4]; normalisation in ln(gamma-1)) defines the result; this pin says
    how far that is from the continuum integral: < 1e-5, converging with the number of cells -- far below the ~1 %
    accuracy of the thermal fits it stands in for."""
    ne, Th, B, th, nu, kappa = 3.0e4, 8.0, 6.0, 0.9, 230e9, 3.5
    nuB = EE * B / (2 * np.pi * ME * CL)
    C = np.sqrt(3) * EE ** 3 * B * np.sin(th) / (4 * np.pi * ME * CL ** 2)
    n_of = lambda g: g * np.sqrt(g * g - 1) * (1 + (g - 1) / (kappa * Th)) ** -(kappa + 1)
    nrm = integrate.quad(n_of, 1, np.inf, limit=400)[0]
    # F here by adaptive quadrature of the cosh representation (the kernels themselves are pinned against mpmath in E1)
    def Fi(x):
        if x > 200.0:
            return 0.0
        T = np.arccosh(1.0 + 45.0 / x)
        return x * np.exp(-x) * integrate.quad(lambda t: np.exp(-2.0 * x * np.sinh(0.5 * t) ** 2) * np.cosh(5.0 * t / 3.0) / np.cosh(t),
                                               0.0, T, limit=200, epsabs=0, epsrel=1e-10)[0]
    assert Fi(0.29) == pytest.approx(_F(0.29), rel=1e-9) and Fi(1e-5) == pytest.approx(_F(1e-5), rel=1e-9)
    f = lambda u: n_of(np.exp(u)) * Fi(nu / (1.5 * np.exp(2 * u) * nuB * np.sin(th))) * np.exp(u)
    jI = C * ne / nrm * integrate.quad(f, 0.0, np.log(1e6), limit=800, epsabs=0, epsrel=1e-8)[0]
    err = []
    for n in (16, 32, 128):
        c = ref.coefficients_edf(2, ne, Th, B, np.cos(th), nu, kappa=kappa, n_nodes=n)
        err.append(abs(c[0] / jI - 1))
    assert err[2] < 1e-5 and err[0] > 3 * err[2]
    a = ref.coefficients_edf(2, ne, Th, B, np.cos(th), nu, kappa=kappa, n_nodes=128)
    b = ref.coefficients_edf(2, ne, Th, B, np.cos(th), nu, kappa=kappa, n_nodes=512)
    assert np.allclose(a[:6], b[:6], rtol=1e-5, atol=0)
