"""Pins A1-A4 of the oracle's adaptive ray tracing (oracle/adaptive_ref.py; reading R-11).

The refinement rule is a heuristic, so what pins it from outside are the cases where its result is fixed by
mathematics: an affine image is reproduced exactly from the two coarsest levels; with zero tolerance on a curved
image every pixel is traced; with an infinite tolerance the image is the library's multilinear interpolation of the
level-1 lattice; on a thin ring the traced pixels hug the ring and the error stays at the tolerance."""
import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

from oracle import adaptive_ref as A


def tracer(fn, nx, calls=None):
    def trace(pix):
        if calls is not None:
            calls.append(np.array(pix))
        i, j = pix % nx, pix // nx
        return np.stack(fn(i.astype(float), j.astype(float)), axis=1)
    return trace


def test_A1_affine_image_needs_two_levels_and_is_exact():
    nx, ny, L = 61, 45, 3      # neither size is 1 modulo the base stride: the last cells are narrower
    f = lambda x, y: (3.0 + 0.01 * x + 0.02 * y, 0.5 - 0.003 * x, 0.1 * y / 45, -0.2 + 0.001 * (x + y))
    calls = []
    img, state, counts = A.adaptive_image(tracer(f, nx, calls), nx, ny, L, rel_tol=1e-9)
    n0 = len(A.lines(nx, 8)) * len(A.lines(ny, 8)); n1 = len(A.lines(nx, 4)) * len(A.lines(ny, 4))
    # the corner cell [56,60]x[40,44] is narrower than the level-1 stride both ways: it gains no point at level 1, keeps
    # its flag, and is examined with its five level-2 points instead (which the affine image passes)
    assert counts == [n0, n1 - n0, 5, 0]
    assert (state == 1).sum() == n1 + 5 and (state == 2).sum() == nx * ny - n1 - 5
    jj, ii = np.mgrid[0:ny, 0:nx]
    want = np.stack(f(ii.astype(float), jj.astype(float)))
    assert np.abs(img - want).max() < 1e-13
    allpix = np.concatenate(calls)
    assert np.unique(allpix).size == allpix.size                      # no pixel traced twice
    assert A.lines(16, 8) == [0, 8, 15] and A.lines(17, 8) == [0, 8, 16] and A.lines(9, 1) == list(range(9))


def test_A2_zero_tolerance_traces_every_pixel():
    nx, ny, L = 33, 26, 3
    f = lambda x, y: (2.0 + np.sin(0.3 * x) * np.cos(0.2 * y), 0.3 * np.sin(0.11 * x * y + 1.0), 0.1 * np.cos(0.7 * x + 0.1 * y * y), 0.05 * np.sin(x + y))
    img, state, counts = A.adaptive_image(tracer(f, nx), nx, ny, L, rel_tol=0.0, abs_tol=0.0)
    assert (state == 1).all() and sum(counts) == nx * ny
    jj, ii = np.mgrid[0:ny, 0:nx]
    assert np.array_equal(img, np.stack(f(ii.astype(float), jj.astype(float))))


def test_A3_without_refinement_it_is_the_multilinear_interpolant_of_level_1():
    nx, ny, L = 50, 39, 3
    f = lambda x, y: (1.0 + 0.05 * x * y / 50 + np.sin(0.2 * x), np.cos(0.15 * y), 0.01 * x * x, np.sin(0.1 * x) * np.sin(0.1 * y))
    img, state, counts = A.adaptive_image(tracer(f, nx), nx, ny, L, rel_tol=1e30)
    lx, ly = np.array(A.lines(nx, 4), float), np.array(A.lines(ny, 4), float)
    assert sum(counts) == lx.size * ly.size and counts[2:] == [0, 0]
    jj, ii = np.mgrid[0:ny, 0:nx]
    for k in range(4):
        vals = f(*np.meshgrid(lx, ly))[k]                                    # [ly, lx]
        want = RegularGridInterpolator((ly, lx), vals, method="linear")(np.stack([jj.ravel(), ii.ravel()], axis=1)).reshape(ny, nx)
        assert np.abs(img[k] - want).max() < 1e-12 * np.abs(vals).max()
    # levels 2 and 3 interpolate from level-1 values that are themselves exact at the level-1 lattice
    assert np.array_equal(state[::4, ::4], np.ones_like(state[::4, ::4]))


def test_A4_thin_ring_is_resolved_where_it_is_and_nowhere_else():
    n, L, tol = 128, 3, 1e-2
    def f(x, y):
        r = np.hypot(x - 63.3, y - 64.1)
        I = 0.05 + 0.002 * x / n + np.exp(-0.5 * ((r - 30.0) / 1.2) ** 2)
        return (I, 0.3 * I * np.cos(2 * np.arctan2(y - 64.1, x - 63.3)), 0.3 * I * np.sin(2 * np.arctan2(y - 64.1, x - 63.3)), 0.01 * I)
    img, state, counts = A.adaptive_image(tracer(f, n), n, n, L, rel_tol=tol)
    jj, ii = np.mgrid[0:n, 0:n]
    want = np.stack(f(ii.astype(float), jj.astype(float)))
    traced = state == 1
    assert 0.15 < traced.mean() < 0.45
    r = np.hypot(ii - 63.3, jj - 64.1)
    assert traced[np.abs(r - 30.0) < 2.5].all()                   # the ring itself is fully traced
    assert traced[r > 46].mean() < 0.08                           # far outside it only the two coarse levels are
    assert np.array_equal(img[:, traced], want[:, traced])
    err = np.abs(img - want).max(axis=0) / want[0]
    assert err.max() < 5 * tol and np.percentile(err, 99) < tol
    # a looser tolerance traces fewer pixels, a tighter one more
    c_loose = sum(A.adaptive_image(tracer(f, n), n, n, L, rel_tol=5e-2)[2])
    c_tight = sum(A.adaptive_image(tracer(f, n), n, n, L, rel_tol=2e-3)[2])
    assert c_loose < sum(counts) < c_tight
