"""ORACLE (test infrastructure, not product code): adaptive ray tracing, step by step.

PAPER.md:70: "Our GPU code could be further sped up by another factor of 10 with adaptive ray tracing which reduces the
number of light rays to follow (following e.g., Gelles et al. 2021)"; PAPER.md:25 lists it among the ways to cut the
cost of an image.  The paper gives no algorithm (it is future work there), so this is a heuristic of our own, stated
here in full and followed literally by the CUDA path (reading R-11 in DESIGN.md):

  lattice of level l (l = 0..L, stride s_l = 2^(L-l)): the pixel indices {0, s_l, 2 s_l, ...} and n-1, in x and in y.
  A cell of level l is the rectangle between consecutive lattice lines in x and in y (the last one may be narrower).
  * level 0: every lattice point is traced; every level-0 cell is flagged.
  * level l >= 1: the new points are the level-l lattice points that are not level-(l-1) lattice points.  A new point
    is traced if at least one level-(l-1) cell whose closed rectangle contains it is flagged; otherwise its four
    Stokes values are the bilinear interpolation of the corners of the level-(l-1) cell that contains it (for a
    point on an edge shared by two cells, the one to its right / above it, the other one at the image border).
    Then every flagged level-(l-1) cell P is examined: it needs refinement if, for some new point p in its closed
    rectangle and some Stokes parameter k, |S_k(p) - B_P,k(p)| > rel_tol * |I(p)| + abs_tol, with B_P the bilinear
    interpolant of P's four corners; a flagged cell that gains no new point at this level (it is narrower than the
    stride both ways) also counts as needing refinement, i.e. its flag is carried down.  The level-l cells inside P
    are flagged iff P needs refinement; the cells inside an unflagged P are unflagged.
  After level L (stride 1) every pixel has a value.  Bilinear weights use the actual corner coordinates.

`trace(pixels) -> array [n, 4]` is any per-pixel function (the CPU oracle's make_pixels in the parity tests, closed
forms in the pins).  Pins A1-A4: tests/test_oracle_adaptive.py.  Plain loops; nothing shared with the CUDA path.
"""
import numpy as np


def lines(n, s):
    """lattice lines of stride s on n pixels: multiples of s, and n-1"""
    out = list(range(0, n, s))
    if out[-1] != n - 1:
        out.append(n - 1)
    return out


def bilinear(img, i0, i1, j0, j1, i, j):
    """bilinear interpolant of the four corners (i0|i1, j0|j1) of img[:, j, i] at (i, j)"""
    t = (i - i0) / (i1 - i0) if i1 > i0 else 0.0
    u = (j - j0) / (j1 - j0) if j1 > j0 else 0.0
    return ((1 - t) * (1 - u)) * img[:, j0, i0] + (t * (1 - u)) * img[:, j0, i1] + ((1 - t) * u) * img[:, j1, i0] + (t * u) * img[:, j1, i1]


def adaptive_image(trace, nx, ny, L, rel_tol, abs_tol=0.0):
    """Returns img [4, ny, nx], state [ny, nx] (1 traced, 2 interpolated), and the number of traced pixels per level."""
    assert nx >= 2 and ny >= 2 and L >= 1
    img = np.zeros((4, ny, nx))
    state = np.zeros((ny, nx), dtype=np.uint8)
    S = 1 << L

    def do_trace(pts):
        if not pts:
            return
        pix = np.array([j * nx + i for (i, j) in pts], dtype=np.int64)
        val = np.asarray(trace(pix), dtype=np.float64).reshape(len(pts), 4)
        for (i, j), v in zip(pts, val):
            img[:, j, i] = v
            state[j, i] = 1

    lx, ly = lines(nx, S), lines(ny, S)
    do_trace([(i, j) for j in ly for i in lx])
    counts = [len(lx) * len(ly)]
    # flagged cells of the previous level, keyed by their lower-left corner
    flagged = {(lx[a], ly[b]) for a in range(len(lx) - 1) for b in range(len(ly) - 1)}
    for l in range(1, L + 1):
        s = S >> l
        px, py = lx, ly                      # lines of level l-1
        lx, ly = lines(nx, s), lines(ny, s)  # lines of level l
        cells = [(px[a], px[a + 1], py[b], py[b + 1]) for a in range(len(px) - 1) for b in range(len(py) - 1)]
        pxs, pys = set(px), set(py)
        new = [(i, j) for j in ly for i in lx if not (i in pxs and j in pys)]

        def parents(i, j):
            xs = [a for a in range(len(px) - 1) if px[a] <= i <= px[a + 1]]
            ys = [b for b in range(len(py) - 1) if py[b] <= j <= py[b + 1]]
            return [(px[a], px[a + 1], py[b], py[b + 1]) for a in xs for b in ys]

        to_trace, to_interp = [], []
        for (i, j) in new:
            par = parents(i, j)
            if any((c[0], c[2]) in flagged for c in par):
                to_trace.append((i, j))
            else:
                to_interp.append(((i, j), par[-1]))   # the cell to the right / above when there are two
        for (i, j), (i0, i1, j0, j1) in to_interp:
            img[:, j, i] = bilinear(img, i0, i1, j0, j1, i, j)
            state[j, i] = 2
        do_trace(to_trace)
        counts.append(len(to_trace))
        new_flagged = set()
        lxs, lys = set(lx), set(ly)
        for (i0, i1, j0, j1) in cells:
            if (i0, j0) not in flagged:
                continue
            xs = [i for i in range(i0, i1 + 1) if i in lxs]
            ys = [j for j in range(j0, j1 + 1) if j in lys]
            refine = len(xs) == 2 and len(ys) == 2   # no new point in P: the flag is carried down
            for j in ys:
                for i in xs:
                    if i in pxs and j in pys:
                        continue            # a corner of P
                    b = bilinear(img, i0, i1, j0, j1, i, j)
                    if np.any(np.abs(img[:, j, i] - b) > rel_tol * abs(img[0, j, i]) + abs_tol):
                        refine = True
            if refine:
                for a in range(len(xs) - 1):
                    for c in range(len(ys) - 1):
                        new_flagged.add((xs[a], ys[c]))
        flagged = new_flagged
    assert (state > 0).all()
    return img, state, counts
