"""Writes tests/golden/t7_adaf32_totals.txt: REGRESSION values of the oracle for BASELINE.json configs[0] (W1: the
analytic ADAF image at 32x32, 230 GHz).  Calls only oracle/.  These are not the paper's numbers (the paper prints none
for this synthetic stand-in) and not an independent pin: they freeze the oracle, which is pinned by G1-G6 / T1-T9, so
that an unintended change of its arithmetic fails tests/test_oracle_transfer.py::test_T7.

    python tests/golden/make_t7_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import ipole_ref  # noqa: E402

CAM = dict(spin=0.9375, inclination_deg=60.0, r_cam=1000.0, fov=40.0, nx=32, ny=32, freq_hz=230e9, mbh_msun=4.1e6, dsource_pc=8000.0)
L_UNIT = 6.6742e-8 * 4.1e6 * 1.989e33 / 2.99792458e10 ** 2
PC = 3.085678e18


def main():
    c = ipole_ref.Ctx(**CAM)
    c.load_adaf()
    o = c.make_pixels(nthreads=os.cpu_count() or 1)
    sc = (40.0 * L_UNIT / (8000.0 * PC)) ** 2 / 32 ** 2 * 1e23
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "t7_adaf32_totals.txt")
    with open(out, "w") as f:
        f.write("# regression values of the CPU oracle, W1 (configs[0]): written by tests/golden/make_t7_golden.py\n")
        for k in "IQUV":
            f.write("flux_%s_jy %.17e\n" % (k, float(np.sum(o[k])) * sc))
        f.write("total_steps %d\n" % int(o["nsteps"].sum()))
        f.write("max_steps %d\n" % int(o["nsteps"].max()))
    print(open(out).read())


if __name__ == "__main__":
    main()
