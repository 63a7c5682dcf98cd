"""Pins T2, T8 for the oracle's synchrotron coefficients, Bessel functions and the 4x4 evolution operator.

Independent references: scipy's exponentially scaled K_n; the first-principles synchrotron integrals over a
relativistic Maxwellian (Rybicki & Lightman 6.31-6.35 single-electron power with F, G and Legg & Westfold's
circular term) evaluated by quadrature; the cold-plasma Faraday rotation / conversion laws; a 40-digit matrix
exponential (mpmath) for the operator.
"""
import numpy as np
import pytest
from scipy import integrate, special
import mpmath as mp

EE, CL, ME, HPL = 4.80320680e-10, 2.99792458e10, 9.1093826e-28, 6.6260693e-27


def test_bessel_scaled_vs_scipy(ref):
    for z in (1e-3, 0.03, 0.5, 1.0, 2.0, 7.0, 33.0, 300.0, 3000.0):
        k = ref.bessel_kscaled(z)
        for n in range(3):
            assert k[n] == pytest.approx(special.kve(n, z), rel=2e-13)


def _F(y):
    return y * integrate.quad(lambda t: special.kv(5.0 / 3.0, t), y, np.inf, limit=400)[0]


def _G(y):
    return y * special.kv(2.0 / 3.0, y)


def _H(y):
    return y * special.kv(1.0 / 3.0, y) + integrate.quad(lambda t: special.kv(1.0 / 3.0, t), y, np.inf, limit=400)[0]


@pytest.mark.parametrize("x", [0.1, 1.0, 10.0, 100.0, 1000.0])
def test_T8_emissivities_vs_first_principles(ref, x):
    # j_S = (1/4pi) int n(gamma) P_S(nu,gamma) dgamma, n(gamma) = n gamma^2 e^{-gamma/Th} / (2 Th^3) (Th >> 1),
    # P_I = sqrt3 e^3 B sin / (m c^2) F(nu/nu_cr), P_Q likewise with G, P_V = P-prefactor * (4 cot / (3 gamma)) H,
    # nu_cr = (3/2) gamma^2 nu_B sin.
    ne, Th, B, th = 1.0e5, 25.0, 12.0, 1.1
    nuB = EE * B / (2 * np.pi * ME * CL)
    nuc = 1.5 * Th * Th * nuB * np.sin(th)
    nu = x * nuc
    pref = np.sqrt(3.0) * EE ** 3 * B * np.sin(th) / (ME * CL * CL) / (4 * np.pi) * ne / 2.0

    def integ(fn, power):
        f = lambda z: z ** power * np.exp(-z) * fn(x / (z * z))
        return integrate.quad(f, 0, 2.0, limit=400)[0] + integrate.quad(f, 2.0, 60.0, limit=400)[0]

    jI = pref * integ(_F, 2)
    jQ = pref * integ(_G, 2)
    jV = pref * (4.0 / (3.0 * Th * np.tan(th))) * integ(_H, 1)
    c = ref.coefficients(ne, Th, B, np.cos(th), nu)
    assert c[0] == pytest.approx(jI, rel=0.01)
    assert c[1] == pytest.approx(jQ, rel=0.015)
    assert c[2] == pytest.approx(jV, rel=0.01)
    # Kirchhoff: alpha_S = j_S / B_nu(T_e)
    Bnu = 2 * HPL * nu ** 3 / CL ** 2 / np.expm1(HPL * nu / (ME * CL * CL * Th))
    assert np.allclose(c[3:6], c[0:3] / Bnu, rtol=1e-13)


def test_T8_faraday_cold_limits_and_parities(ref):
    ne, B, nu, th = 3.0e4, 8.0, 230e9, 0.7
    # Theta_e -> 0: textbook rotation measure law and cold-plasma conversion
    c = ref.coefficients(ne, 1e-3, B, np.cos(th), nu)
    rV = EE ** 3 * ne * B * np.cos(th) / (np.pi * ME ** 2 * CL ** 2 * nu ** 2)
    rQ = EE ** 4 * ne * B ** 2 * np.sin(th) ** 2 / (4 * np.pi ** 2 * ME ** 3 * CL ** 3 * nu ** 3)
    assert c[7] == pytest.approx(rV, rel=2e-3)
    assert c[6] == pytest.approx(rQ, rel=1e-2)
    # hot plasma suppresses rotation like K0/K2 ~ ln(Th)/(2 Th^2)
    c_hot = ref.coefficients(ne, 20.0, B, np.cos(th), nu)
    assert c_hot[7] / rV == pytest.approx(special.kve(0, 0.05) / special.kve(2, 0.05), rel=1e-12)
    # hot plasma, high frequency (X -> 0, f(X) -> 1): the conversion coefficient of an isotropic distribution is the cold
    # one times <gamma (1 + beta^2)> = <2 gamma - 1/gamma> (Melrose 1997; Shcherbakov 2008), which for Maxwell-Juettner
    # electrons is K1/K2 + 6 Theta_e.  The average is taken here by quadrature over n(gamma) ~ gamma^2 beta e^(-gamma/Theta):
    # a dropped 6 Theta_e, a wrong Bessel order or a wrong constant in the bracket fails this.
    for Th_hot in (1.0, 10.0, 30.0):
        nu_hi = 1e21                                   # X = Th [sqrt2 sin 1e3 nu_B/nu]^(1/2) ~ 4e-6 Th: f(X) = 1 - O(1e-5)
        w = lambda g: g * np.sqrt(g * g - 1.0) * np.exp(-(g - 1.0) / Th_hot)
        num = integrate.quad(lambda g: w(g) * (2.0 * g - 1.0 / g), 1.0, np.inf, limit=400)[0]
        den = integrate.quad(w, 1.0, np.inf, limit=400)[0]
        c_h = ref.coefficients(ne, Th_hot, B, np.cos(th), nu_hi)
        rQ_cold = EE ** 4 * ne * B ** 2 * np.sin(th) ** 2 / (4 * np.pi ** 2 * ME ** 3 * CL ** 3 * nu_hi ** 3)
        assert c_h[6] / rQ_cold == pytest.approx(num / den, rel=2e-4)
    # f(X) itself (a published fit to a numerical integral, Shcherbakov 2008) is pinned only at X -> 0 (above): "parity
    # unpinned" for its shape at X >~ 0.1
    # parities under theta_B -> pi - theta_B: j_V, alpha_V, rho_V odd; the rest even
    cp = ref.coefficients(ne, 5.0, B, np.cos(th), nu)
    cm = ref.coefficients(ne, 5.0, B, -np.cos(th), nu)
    for i in (0, 1, 3, 4, 6):
        assert cm[i] == cp[i]
    for i in (2, 5, 7):
        assert cm[i] == -cp[i]
    assert cp[0] > cp[1] > 0 and cp[0] > abs(cp[2])
    # degenerate inputs give zeros, never NaN; underflow of exp(-1.89 x^(1/3)) gives exact zero emission
    assert np.all(ref.coefficients(ne, 5.0, B, 1.0, nu) == 0)
    assert np.all(ref.coefficients(0.0, 5.0, B, 0.3, nu) == 0)
    far = ref.coefficients(30.0, 0.03, 5e-3, 0.3, nu)
    assert np.all(np.isfinite(far)) and far[0] == 0.0 and far[7] != 0.0


def _expm_ref(al, rh, s, J=None):
    mp.mp.dps = 40
    aI, aQ, aU, aV = [mp.mpf(float(v)) for v in al]
    rQ, rU, rV = [mp.mpf(float(v)) for v in rh]
    K = mp.matrix([[aI, aQ, aU, aV], [aQ, aI, rV, -rU], [aU, -rV, aI, rQ], [aV, rU, -rQ, aI]])
    O = mp.expm(-K * mp.mpf(float(s)))
    # P = int_0^s exp(-K x) dx from the augmented matrix [[-K, 1],[0,0]]
    Aug = mp.zeros(8, 8)
    for i in range(4):
        for j in range(4):
            Aug[i, j] = -K[i, j]
        Aug[i, 4 + i] = 1
    E = mp.expm(Aug * mp.mpf(float(s)))
    to = lambda M, r0, c0: np.array([[float(M[r0 + i, c0 + j]) for j in range(4)] for i in range(4)])
    return to(O, 0, 0), to(E, 0, 4)


def test_T2_operator_vs_high_precision_matrix_exponential(ref):
    rng = np.random.default_rng(11)
    cases = []
    for scale in (1.0, 1e-3, 1e-30, 1e-90):
        for _ in range(4):
            aI = rng.uniform(0.5, 2.0)
            a = rng.normal(size=3) * rng.uniform(0, 0.5)
            r = rng.normal(size=3) * rng.choice([0.0, 1.0, 30.0])
            cases.append((np.concatenate([[aI], a]) * scale, r * scale, rng.uniform(0.1, 2.0) / scale))
    cases.append((np.array([0.3, 0.0, 0.0, 0.0]), np.zeros(3), 1.7))                 # no polarised terms
    cases.append((np.array([0.0, 0.0, 0.0, 0.0]), np.array([0.0, 0.0, 2.0]), 1.0))   # pure rotation
    cases.append((np.array([0.0, 0.0, 0.0, 0.0]), np.zeros(3), 2.5))                 # vacuum
    cases.append((np.array([1.0, 0.2, 0.0, 0.1]), np.array([0.4, 0.0, -3.0]), 1e-9))  # tiny step
    cases.append((np.array([1.0, 0.3, 0.1, -0.2]), np.array([0.3, 0.1, -0.2]) * 2, 0.9))  # alpha parallel rho
    for al, rh, s in cases:
        O, P = ref.stokes_operator(al, rh, s)
        Oe, Pe = _expm_ref(al, rh, s)
        assert np.allclose(O, Oe, rtol=0, atol=2e-13 * max(1.0, np.abs(Oe).max())), (al, rh, s)
        assert np.allclose(P, Pe, rtol=0, atol=2e-13 * np.abs(Pe).max()), (al, rh, s)


def test_T2_operator_semigroup_and_closed_forms(ref):
    al = np.array([0.7, 0.2, -0.1, 0.05]); rh = np.array([0.5, 0.3, -2.0])
    O1, P1 = ref.stokes_operator(al, rh, 0.4)
    O2, P2 = ref.stokes_operator(al, rh, 0.9)
    O3, P3 = ref.stokes_operator(al, rh, 1.3)
    assert np.allclose(O2 @ O1, O3, atol=1e-14)
    assert np.allclose(P2 + O2 @ P1, P3, atol=1e-14)  # int_0^{s1+s2} = int_0^{s2} + O(s2) int_0^{s1}
    # rho_V only: rotation of (Q,U) by rho_V s with dQ/ds = -rho_V U, dU/ds = +rho_V Q
    O, P = ref.stokes_operator([0, 0, 0, 0], [0, 0, 0.8], 1.5)
    c, s = np.cos(1.2), np.sin(1.2)
    assert np.allclose(O, [[1, 0, 0, 0], [0, c, -s, 0], [0, s, c, 0], [0, 0, 0, 1]], atol=1e-15)
    # rho_Q only: rotation of (U,V): dU/ds = -rho_Q V, dV/ds = +rho_Q U
    O, P = ref.stokes_operator([0, 0, 0, 0], [0.8, 0, 0], 1.5)
    assert np.allclose(O, [[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, c, -s], [0, 0, s, c]], atol=1e-15)
    # alpha_I only: e^{-tau}, (1 - e^{-tau})/alpha
    O, P = ref.stokes_operator([2.0, 0, 0, 0], [0, 0, 0], 0.3)
    assert np.allclose(O, np.exp(-0.6) * np.eye(4), atol=1e-16) and np.allclose(P, (1 - np.exp(-0.6)) / 2 * np.eye(4), atol=1e-16)
