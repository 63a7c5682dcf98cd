"""Writes pw_tables.inc: piecewise polynomial tables of two special functions of the coefficient step.

Used by the CUDA path only (coeff.cuh).  The CPU oracle evaluates the defining formulas (quadrature for K_n,
exp/pow/cos for f) and shares nothing with this file.

  bessel : R0(Th) = K_0(1/Th)/K_2(1/Th),  R1(Th) = K_1(1/Th)/K_2(1/Th)          2^-8 <= Th < 2^12
  fx     : f(X) = 2.011 exp(-X^1.035/4.7) - cos(X/2) exp(-X^1.2/2.73) - 0.011 exp(-X/47.2)   2^-30 <= X < 2^9
           (R-7; the Faraday-conversion fit)

Every binary octave [2^e, 2^(e+1)) is cut into NP = 8 equal pieces; on piece q the function is a degree-11
polynomial in v = 2 NP m - (2 NP + 1 + 2 q) in [-1, 1], m = x 2^-e in [1, 2).  The nearest singularity (x = 0) is
at least 17 piece half-widths away, so the Chebyshev coefficients decay like 34^-n or faster and degree 11 reaches
double precision (the generator checks the first dropped term).
Coefficients come from a Chebyshev interpolant computed with mpmath at 30 digits, are stored in ascending order, and are checked here in
double arithmetic against mpmath at random points of every piece.

Run:  python paper_2302_02733_b200/csrc/gen_pw_tables.py   (rewrites pw_tables.inc beside it; about a minute)
"""
import os
import mpmath as mp
import numpy as np

mp.mp.dps = 30
NC = 12  # coefficients per piece (degree 11)
NP = 8   # pieces per binary octave

BESSEL_E0, BESSEL_E1 = -8, 12
FX_E0, FX_E1 = -30, 9


def r01(th):
    z = 1 / th
    k0, k1 = mp.besselk(0, z), mp.besselk(1, z)
    k2 = k0 + 2 * th * k1
    return k0 / k2, k1 / k2


def fx(x):
    return (mp.mpf("2.011") * mp.exp(-x ** mp.mpf("1.035") / mp.mpf("4.7"))
            - mp.cos(x / 2) * mp.exp(-x ** mp.mpf("1.2") / mp.mpf("2.73"))
            - mp.mpf("0.011") * mp.exp(-x / mp.mpf("47.2")))


NNODE = 20  # Chebyshev nodes per piece (interpolant of degree 19, truncated to NC terms)
_NODES = [mp.cos(mp.pi * (mp.mpf(j) + mp.mpf(1) / 2) / NNODE) for j in range(NNODE)]
_COS = [[mp.cos(mp.pi * n * (mp.mpf(j) + mp.mpf(1) / 2) / NNODE) for j in range(NNODE)] for n in range(NNODE)]


def _cheb_T(n):
    """integer monomial coefficients (ascending) of T_n"""
    a, b = [1], [0, 1]
    if n == 0:
        return a
    for _ in range(n - 1):
        c = [0] + [2 * t for t in b]
        for i, t in enumerate(a):
            c[i] -= t
        a, b = b, c
    return b


_TN = [_cheb_T(n) for n in range(NC)]


def piece_fit(fvec, nf, e, q):
    """fvec(x) -> nf values.  Ascending monomial coefficients in v of each, x = 2^e (2 NP + 1 + 2 q + v)/(2 NP), v in [-1, 1];
    also returns the size of the first dropped Chebyshev coefficient relative to the largest kept one."""
    vals = [fvec(mp.ldexp(1, e) * (2 * NP + 1 + 2 * q + v) / (2 * NP)) for v in _NODES]
    out, drop = [], 0.0
    for k in range(nf):
        cheb = []
        for n in range(NC + 1):
            sacc = mp.mpf(0)
            for j in range(NNODE):
                sacc += vals[j][k] * _COS[n][j]
            cheb.append(sacc * 2 / NNODE)
        cheb[0] /= 2
        drop = max(drop, float(abs(cheb[NC]) / max(abs(c) for c in cheb[:NC])))
        mono = [mp.mpf(0)] * NC
        for n in range(NC):
            for i, t in enumerate(_TN[n]):
                mono[i] += cheb[n] * t
        out.append([float(m) for m in mono])
    return out, drop


def horner(c, v):
    p = np.full_like(v, c[-1])
    for a in c[-2::-1]:
        p = p * v + a
    return p


def build(fvec, nf, e0, e1, label, rng):
    """Returns array [pieces][NC][nf]."""
    npieces = (e1 - e0) * NP
    tab = np.zeros((npieces, NC, nf))
    worst, worst_at, wdrop = 0.0, None, 0.0
    for e in range(e0, e1):
        for q in range(NP):
            i = (e - e0) * NP + q
            cs, drop = piece_fit(fvec, nf, e, q)
            wdrop = max(wdrop, drop)
            v = rng.uniform(-1, 1, 4)
            ref = np.array([[float(t) for t in fvec(mp.ldexp(1, e) * (2 * NP + 1 + 2 * q + mp.mpf(float(u))) / (2 * NP))] for u in v])
            for k in range(nf):
                tab[i, :, k] = cs[k]
                got = horner(cs[k], v)
                scale = np.maximum(np.abs(ref[:, k]), 1e-3 * np.max(np.abs(cs[k])))  # absolute near a zero crossing
                err = float(np.max(np.abs(got - ref[:, k]) / scale))
                if err > worst:
                    worst, worst_at = err, (e, q, k)
    print("%s: %d pieces, worst error in double evaluation %.2e at %s, first dropped Chebyshev term %.1e"
          % (label, npieces, worst, worst_at, wdrop))
    assert worst < 1e-15 and wdrop < 3e-16, (worst, wdrop)  # both relative to the piece's largest coefficient
    return tab


def emit(out, name, tab):
    n, nc, nf = tab.shape
    out.append("__device__ const double g_pw_%s[%d][%d][%d] = {" % (name, n, nc, nf))
    for i in range(n):
        rows = ", ".join("{" + ", ".join(repr(float(tab[i, j, k])) for k in range(nf)) + "}" for j in range(nc))
        out.append("  {" + rows + "},")
    out.append("};")


def main():
    rng = np.random.default_rng(23)
    out = ["// generated by gen_pw_tables.py -- do not edit.  [piece][coefficient (ascending)][function]; see coeff.cuh."]
    out.append("#define IPOLE_PW_NC %d\n#define IPOLE_PW_NP %d" % (NC, NP))
    out.append("#define IPOLE_PW_BESSEL_E0 %d\n#define IPOLE_PW_BESSEL_E1 %d" % (BESSEL_E0, BESSEL_E1))
    out.append("#define IPOLE_PW_FX_E0 %d\n#define IPOLE_PW_FX_E1 %d" % (FX_E0, FX_E1))
    tb = build(r01, 2, BESSEL_E0, BESSEL_E1, "bessel ratios", rng)
    emit(out, "bessel", tb)
    tf = build(lambda x: (fx(x),), 1, FX_E0, FX_E1, "f(X)", rng)
    emit(out, "fx", tf)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "pw_tables.inc")
    with open(path, "w") as fh:
        fh.write("\n".join(out) + "\n")


if __name__ == "__main__":
    main()
