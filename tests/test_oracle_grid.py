"""Pins for the oracle's grid plasma model and checks of the synthetic GRMHD-like input."""
import numpy as np
import pytest
from paper_2302_02733_b200 import workloads as W

A = W.SPIN
ME, MP, CL = 9.1093826e-28, 1.67262171e-24, 2.99792458e10
L_UNIT = 6.6742e-8 * 4.1e6 * 1.989e33 / CL ** 2


def small_desc(N1=12, N2=10, N3=8):
    rh = 1 + np.sqrt(1 - A * A)
    sx = [np.log(0.9 * rh), 0.0, 0.0]
    return dict(N1=N1, N2=N2, N3=N3, startx=sx, dx=[(np.log(50.0) - sx[0]) / N1, 1.0 / N2, 2 * np.pi / N3],
                hslope=0.3, gam=4.0 / 3.0, M_unit=1.5e20, Rlow=1.0, Rhigh=40.0, r_out=50.0)


def test_trilinear_reproduces_linear_fields_and_wraps(ref):
    d = small_desc()
    N1, N2, N3 = d["N1"], d["N2"], d["N3"]
    i, j, k = np.meshgrid(np.arange(N1), np.arange(N2), np.arange(N3), indexing="ij")
    f = np.zeros((8, N1, N2, N3))
    f[0] = 1.0 + 0.5 * i + 0.25 * j          # linear in the two non-periodic indices
    f[1] = 2.0 + np.cos(2 * np.pi * k / N3)  # periodic in k
    f[5] = 1e-3
    c = ref.Ctx(**W.camera("grid", 4))
    c.load_grid(d, f)
    rho_unit = d["M_unit"] / L_UNIT ** 3
    rng = np.random.default_rng(3)
    for _ in range(50):
        fi, fj, fk = rng.uniform(0, N1 - 1), rng.uniform(0, N2 - 1), rng.uniform(-3 * N3, 3 * N3)
        X = [0.0, d["startx"][0] + (fi + 0.5) * d["dx"][0], (fj + 0.5) * d["dx"][1], (fk + 0.5) * d["dx"][2]]
        p = c.plasma(X)
        assert p["present"]
        assert p["ne"] == pytest.approx((1.0 + 0.5 * fi + 0.25 * fj) * rho_unit / (MP + ME), rel=1e-12)
    # periodic wrap: identical state at X3 and X3 + 2 pi; piecewise-linear in k between nodes
    X = [0.0, d["startx"][0] + 4.2 * d["dx"][0], 0.43, 1.234]
    p1 = c.plasma(X); p2 = c.plasma([X[0], X[1], X[2], X[3] + 2 * np.pi]); p3 = c.plasma([X[0], X[1], X[2], X[3] - 4 * np.pi])
    assert p1["thetae"] == pytest.approx(p2["thetae"], rel=1e-12) and p1["thetae"] == pytest.approx(p3["thetae"], rel=1e-12)
    # clamped (constant) extrapolation in the half cell next to the pole and the inner edge
    pa = c.plasma([0.0, d["startx"][0] + 3.5 * d["dx"][0], 0.2 * d["dx"][1], 0.5 * d["dx"][2]])
    pb = c.plasma([0.0, d["startx"][0] + 3.5 * d["dx"][0], 0.5 * d["dx"][1], 0.5 * d["dx"][2]])
    assert pa["ne"] == pytest.approx(pb["ne"], rel=1e-13)
    # outside the domain: no plasma
    assert not c.plasma([0.0, np.log(50.1), 0.4, 0.0])["present"]
    assert not c.plasma([0.0, d["startx"][0] - 1e-3, 0.4, 0.0])["present"]


def test_primitives_to_four_vectors(ref):
    d = small_desc()
    f = np.zeros((8, d["N1"], d["N2"], d["N3"]))
    prim = np.array([0.7, 0.02, 0.05, -0.03, 0.11, 2e-3, -1e-3, 3e-3])
    for q in range(8):
        f[q] = prim[q]
    c = ref.Ctx(**W.camera("grid", 4))
    c.load_grid(d, f)
    for X in ([0.0, np.log(3.0), 0.3, 1.0], [0.0, np.log(12.0), 0.52, 4.0]):
        p = c.plasma(X)
        g = ref.gcov(A, 0.3, X); gi = ref.gcon(A, 0.3, X)
        u, b = p["u"], p["b"]
        assert u @ g @ u == pytest.approx(-1.0, abs=1e-13)
        assert abs(u @ g @ b) < 1e-12 * np.sqrt(b @ g @ b)
        # inverse relations (Gammie, McKinney & Toth 2003): utilde^i = u^i - u^t g^{ti}/g^{tt};  B^i = b^i u^t - b^t u^i
        ut_rec = u[1:] - u[0] * gi[0, 1:] / gi[0, 0]
        assert np.allclose(ut_rec, prim[2:5], rtol=1e-12)
        B_unit = CL * np.sqrt(4 * np.pi * d["M_unit"] / L_UNIT ** 3)
        bc = b / B_unit
        assert np.allclose(bc[1:] * u[0] - bc[0] * u[1:], prim[5:8], rtol=1e-11)
        assert p["B"] == pytest.approx(np.sqrt(b @ g @ b), rel=1e-13)
        # R_low/R_high electron temperature: bounded by the single-fluid value over (1 + R), R in [R_low, R_high]
        Tgas = (MP / ME) * (d["gam"] - 1) * prim[1] / prim[0]
        assert Tgas / (1 + d["Rhigh"]) < p["thetae"] < Tgas / (1 + d["Rlow"])
        beta = (d["gam"] - 1) * prim[1] / (0.5 * (bc @ g @ bc))
        assert p["thetae"] == pytest.approx(Tgas / (1 + (d["Rhigh"] * beta ** 2 + d["Rlow"]) / (1 + beta ** 2)), rel=1e-12)
    # empty cells: skipped, not fed into the tetrad
    f[0] = 0.0
    c.load_grid(d, f)
    assert not c.plasma([0.0, np.log(3.0), 0.3, 1.0])["present"]


def test_synthetic_torus_properties():
    d, f = W.fm_torus_grid(96, 64, 4)
    assert f.shape == (8, 96, 64, 4) and np.all(np.isfinite(f))
    d0, f0 = W.fm_torus_grid(96, 64, 4, noise=0.0)
    rho = f0[0][:, :, 0]
    i, j = np.unravel_index(rho.argmax(), rho.shape)
    r = np.exp(d["startx"][0] + (np.arange(96) + 0.5) * d["dx"][0])
    assert abs(r[i] - 12.0) < 0.5 and j in (31, 32)          # pressure maximum at r_max in the equatorial plane
    on = rho.max(axis=1) > 0
    assert 5.9 < r[on].min() < 6.6 and 38.0 < r[on].max() < 45.0  # inner edge r_in = 6, outer edge ~ 42
    assert rho.max() == pytest.approx(1.0)
    assert np.all(f0[3] == 0) and np.all(f0[7] == 0)
    assert np.allclose(f0[0][:, ::-1, 0], f0[0][:, :, 0], rtol=1e-9, atol=1e-12)  # reflection symmetric
    # 5 % multiplicative noise, deterministic in the seed, independent per field
    d1, f1 = W.fm_torus_grid(96, 64, 4)
    assert np.array_equal(f, f1)
    m = f0[0] > 0
    ratio = f[0][m] / f0[0][m] - 1
    assert abs(ratio.std() - 0.05) < 5e-3 and np.abs(ratio).max() <= 0.2 + 1e-12
    assert not np.allclose(f[0][m] / f0[0][m], f[1][m] / f0[1][m])
    d2, f2 = W.fm_torus_grid(96, 64, 4, seed=1)
    assert not np.array_equal(f, f2)
    assert [W.config(k)["name"] for k in range(5)] == ["W1", "W2", "W3", "W4", "W5"]
