"""GPU image parity (pytest -m gpu): the CUDA path, called through the C ABI, against the CPU oracle on the same
seeded synthetic inputs (BASELINE.json configs[0..4]; recipe in DESIGN.md section 5).

Tolerances are the ones BASELINE.json north_star states (FP64):
  total Stokes I flux relative 1e-9; Q/U/V totals absolute 1e-9 of the I total;
  per-pixel Stokes relative 1e-7 on >= 99.9 % of pixels (Q,U,V measured against the pixel's I: an error of the
  polarization fraction); at most 1e-4 on rays crossing the photon ring (>= 2 theta turning points).
Pixels the oracle leaves exactly dark (no plasma on the ray) must be exactly dark on the GPU.
"""
import os

import numpy as np
import pytest

from paper_2302_02733_b200 import workloads as W

pytestmark = pytest.mark.gpu
NTHREADS = os.cpu_count() or 1


@pytest.fixture(scope="module")
def ipole():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import __graft_entry__ as ge
    ge.build()
    from paper_2302_02733_b200 import ipole as m
    return m


def to_np(img):
    return {k: v.detach().cpu().numpy().ravel() if hasattr(v, "detach") else np.asarray(v).ravel() for k, v in img.items()}


def check_parity(gpu, ref, label, min_lit=0.0):
    """gpu, ref: dicts of flat arrays over the SAME pixels (I,Q,U,V[,tau,tauF,nsteps,nturn])."""
    I0 = ref["I"]
    n = I0.size
    totI = I0.sum()
    assert abs(gpu["I"].sum() - totI) <= 1e-9 * abs(totI), (label, "total I", gpu["I"].sum(), totI)
    for k in "QUV":
        assert abs(gpu[k].sum() - ref[k].sum()) <= 1e-9 * abs(totI), (label, "total " + k)
    dark = I0 == 0.0
    for k in "IQUV":
        assert (gpu[k][dark] == 0.0).all(), (label, "dark pixels", k)
    lit = ~dark
    assert lit.mean() >= min_lit, (label, "lit fraction", lit.mean())
    # Pixels more than ~250 decades below anything visible (I_nu < 1e-250 cgs; the peak of these images is ~1e-4): their
    # invariant I/nu^3 ~ 1e-284 and the products that form it run through the subnormal range, where a double has a few
    # bits.  "Relative to the pixel's own I" means nothing there; they must agree absolutely to 1e-250.
    tiny = lit & (I0 < 1e-250)
    for k in "IQUV":
        assert (np.abs(gpu[k][tiny] - ref[k][tiny]) <= 1e-250).all(), (label, "underflowing pixels", k)
    lit = lit & ~tiny
    err = np.zeros(n)
    for k in "IQUV":
        err[lit] = np.maximum(err[lit], np.abs(gpu[k][lit] - ref[k][lit]) / np.abs(I0[lit]))
    ring = (ref["nturn"] & 0x7f) >= 2
    ok = err <= 1e-7
    assert ok.mean() >= 0.999, (label, "pixels within 1e-7", ok.mean(), np.sort(err)[-5:])
    assert err.max() <= 1e-4, (label, "worst pixel", err.max())
    if ring.any():
        assert err[ring].max() <= 1e-4, (label, "ring rays", err[ring].max())
    # invariant that holds at any size: I >= sqrt(Q^2+U^2+V^2)
    pol = np.sqrt(gpu["Q"] ** 2 + gpu["U"] ** 2 + gpu["V"] ** 2)
    assert (pol <= gpu["I"] * (1 + 1e-12) + 1e-300).all(), (label, "I >= sqrt(Q^2+U^2+V^2)")
    assert (gpu["I"] >= 0).all()
    if "nsteps" in gpu and "nsteps" in ref:
        same = gpu["nsteps"] == ref["nsteps"]
        assert same.mean() >= 0.999 and np.abs(gpu["nsteps"] - ref["nsteps"]).max() <= 1, (label, "nsteps")
        assert (gpu["nturn"] == ref["nturn"]).mean() >= 0.999, (label, "nturn")
    for k in ("tau", "tauF"):
        if k in gpu and k in ref:
            assert np.allclose(gpu[k], ref[k], rtol=1e-7, atol=1e-300), (label, k)
    nt = ref["nturn"] & 0x7f
    cls = {name: (float(err[m].max()) if m.any() else 0.0, int(m.sum())) for name, m in
           (("n_turn<2", nt < 2), ("n_turn=2", nt == 2), ("n_turn>=3", nt >= 3))}
    return dict(max_err=float(err.max()), ring_frac=float(ring.mean()), lit=float(lit.mean()), by_class=cls,
                within_1e7=float(ok.mean()))


def report(label, n, info):
    """worst per-pixel error of each turning-point class (printed with pytest -s; the driver's log keeps it)"""
    print("\n%s: %d sampled pixels, %.4f %% within 1e-7, worst |dS|/I by class: %s" % (
        label, n, 100 * info["within_1e7"], ", ".join("%s %.2e (%d px)" % (k, v[0], v[1]) for k, v in info["by_class"].items())))


def sample_pixels(nx, ny, stride, window=None):
    """strided lattice of pixel centres plus every pixel of a window (x0, y0, w, h) that straddles the photon ring"""
    ii, jj = np.meshgrid(np.arange(stride // 2, nx, stride), np.arange(stride // 2, ny, stride))
    pix = (jj * nx + ii).ravel()
    if window:
        x0, y0, w, h = window
        wi, wj = np.meshgrid(np.arange(x0, x0 + w), np.arange(y0, y0 + h))
        pix = np.unique(np.concatenate([pix, (wj * nx + wi).ravel()]))
    return pix.astype(np.int64)


def gpu_full_then_sample(g, pix, maps=True):
    img = g.make_image(maps=maps)
    ns, nt = g.ray_info()
    out = {k: v.detach().cpu().numpy().ravel()[pix] for k, v in img.items()}
    out["nsteps"] = ns.ravel()[pix]
    out["nturn"] = nt.ravel()[pix]
    return out, img


# ------------------------------------------------------------------ configs[0]: W1, every pixel
def test_w1_adaf_32_full_image(ipole, ref):
    cam = W.camera("adaf", 32)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    r = ref.Ctx(**cam); r.load_adaf(**W.ADAF)
    want = r.make_pixels(nthreads=NTHREADS)
    got, img = gpu_full_then_sample(g, np.arange(32 * 32))
    info = check_parity(got, want, "W1", min_lit=0.99)
    assert info["max_err"] < 1e-9  # what this scheme actually reaches away from discrete events
    # the same through HOST buffers (the e2e entry): bit-identical to the device-buffer call
    host = g.make_image_host(maps=True)
    for k in host:
        assert np.array_equal(host[k].ravel(), got[k]), k
    # a-9: totals from the reduction kernel
    st = g.stats()
    L = 6.6742e-8 * 4.1e6 * 1.989e33 / 2.99792458e10 ** 2
    dom = (cam["fov"] / cam["nx"] * L / (8000.0 * 3.085678e18)) ** 2 * 1e23
    for q, k in enumerate("IQUV"):
        assert abs(st["flux_jy"][q] - want[k].sum() * dom) <= 1e-9 * abs(want["I"].sum() * dom)
    assert st["total_steps"] == int(want["nsteps"].sum()) and st["max_steps_seen"] == int(want["nsteps"].max())
    assert st["n_ring"] == int(((want["nturn"] & 0x7f) >= 2).sum())
    assert abs(st["lp"] - np.hypot(want["Q"].sum(), want["U"].sum()) / want["I"].sum()) < 1e-9
    assert abs(st["cp"] - want["V"].sum() / want["I"].sum()) < 1e-9


def test_ragged_image_and_other_camera(ipole, ref):
    """nx != ny, not a multiple of the warp size, other inclination / frequency / spin / hslope."""
    cam = W.camera("adaf", 8, freq_hz=345e9, inclination_deg=33.0, spin=0.5, hslope=0.7)
    cam.update(nx=37, ny=23, fov=30.0)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    r = ref.Ctx(**cam); r.load_adaf(**W.ADAF)
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(37 * 23))
    check_parity(got, want, "ragged", min_lit=0.99)


# ------------------------------------------------------------------ configs[1]: W2, sampled
@pytest.mark.parametrize("freq", [230e9, 345e9])
def test_w2_adaf_256_sampled(ipole, ref, freq):
    cam = W.camera("adaf", 256, freq_hz=freq)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    r = ref.Ctx(**cam); r.load_adaf(**W.ADAF)
    pix = sample_pixels(256, 256, 8, window=(150, 120, 48, 16))  # the window crosses the ring on the +x side
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, img = gpu_full_then_sample(g, pix)
    info = check_parity(got, want, "W2 %g" % freq, min_lit=0.99)
    assert info["ring_frac"] > 0.02
    # the pixel-list entry point gives bit-identical numbers to the full image
    lst = g.make_pixels(pix)
    for k in ("I", "Q", "U", "V", "tau", "tauF", "nsteps", "nturn"):
        assert np.array_equal(lst[k], got[k]), k


# ------------------------------------------------------------------ scheduling must not change a single bit
def test_batching_sorting_and_long_ray_pass_are_bit_neutral(ipole):
    cam = W.camera("adaf", 48, max_steps=6000)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    g.set_transfer_split(False)   # the long-ray pass is always the single kernel: compare like with like
    base = to_np(g.make_image(maps=True)); st0 = g.stats()
    assert st0["n_batches"] == 1 and st0["n_long"] == 0
    # forced probe + sort, default budget
    g.set_options(0, 2)
    a = to_np(g.make_image(maps=True)); st1 = g.stats()
    assert st1["ms_probe"] > 0
    # tiny path buffer: many batches; S_cap from the probe
    g.set_options(24 << 20, 2)
    b = to_np(g.make_image(maps=True)); st2 = g.stats()
    assert st2["n_batches"] > 3 and st2["n_lanes"] == 2      # batches alternate between two streams by default
    g.set_batch_overlap(False)
    b1 = to_np(g.make_image(maps=True)); st2b = g.stats()
    assert st2b["n_batches"] > 1 and st2b["n_lanes"] == 1
    g.set_batch_overlap(True)
    for k in b:
        assert np.array_equal(b[k], b1[k]), k
    # no probe and a slot far too small for any ray: every ray goes through the long-ray pass
    g.set_options(40 << 20, 0)
    c = to_np(g.make_image(maps=True)); st3 = g.stats()
    assert st3["n_long"] == 48 * 48 and st3["path_cap"] < 300
    for other in (a, b, c):
        for k in base:
            assert np.array_equal(base[k], other[k]), k
    for st in (st1, st2, st3):
        assert st["total_steps"] == st0["total_steps"] and st["flux_jy"] == st0["flux_jy"]


def test_split_transfer_matches_the_single_kernel(ipole):
    """k_stepop + k_apply against k_transfer on the same stored paths: rounding-level agreement per pixel, the same
    under batching with per-batch slots and the retry level, and with every seventh ray handed over to k_transfer."""
    cam = W.camera("adaf", 64)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    g.set_transfer_split(False)
    one = to_np(g.make_image(maps=True))
    g.set_transfer_split(True)
    two = to_np(g.make_image(maps=True)); st = g.stats()
    assert st["ms_stepop"] > 0 and st["ms_apply"] > 0
    scale = np.abs(one["I"]) + 1e-300
    for k in ("I", "Q", "U", "V"):
        assert np.max(np.abs(one[k] - two[k]) / scale) < 1e-11, k
    assert np.allclose(one["tau"], two["tau"], rtol=1e-12, atol=0) and np.allclose(one["tauF"], two["tauF"], rtol=1e-12, atol=0)
    # many batches with slots sized from the predicted step counts; some rays outgrow them and are retried
    g.set_options(48 << 20, 2)
    three = to_np(g.make_image(maps=True)); st3 = g.stats()
    assert st3["n_batches"] > 3 and st3["n_lanes"] == 2
    for k in two:
        assert np.array_equal(two[k], three[k]), k
    g.set_batch_overlap(False)          # the same batches one after the other on one stream
    three1 = to_np(g.make_image(maps=True))
    assert g.stats()["n_lanes"] == 1
    g.set_batch_overlap(True)
    for k in two:
        assert np.array_equal(two[k], three1[k]), k
    g.set_options(0, 1)
    g.set_transfer_split(2)
    four = to_np(g.make_image(maps=True))
    changed = 0
    for k in ("I", "Q", "U", "V"):
        assert np.max(np.abs(four[k] - two[k]) / scale) < 1e-11, k
        changed += int((four[k] != two[k]).sum())
    assert changed > 0   # the handed-over rays really went through the other kernel
    # slots far too short for any ray: every ray goes to the long-ray pass and k_apply meets groups with nothing to do
    g.set_transfer_split(True)
    g.set_options(40 << 20, 0)
    five = to_np(g.make_image(maps=True))
    assert g.stats()["n_long"] == 64 * 64
    for k in one:
        assert np.array_equal(one[k], five[k]), k    # the long-ray pass is the single kernel


def test_plan_reuse_is_bit_neutral_and_follows_camera_model_and_calls(ipole):
    """ipole_set_plan_reuse: a full image scheduled from the previous call's plan (no probe, no read-back, retried and long
    rays from the recorded lists) is the image the planning call makes, bit for bit; the plan follows the camera and is
    dropped by any other call in between; the model may change under it."""
    def fresh(cam, adaf, budget):
        f = ipole.Ipole(**cam); f.load_adaf(**adaf); f.set_plan_reuse(False); f.set_options(budget, 2)
        img = to_np(f.make_image(maps=True)); ns, nt = f.ray_info(); st = f.stats()
        assert st["plan_reused"] == 0
        f.close()
        return img, ns, nt, st

    def same(a, b):
        for k in a:
            assert np.array_equal(a[k], b[k]), k

    for n, budget in ((256, 1 << 30), (96, 0)):       # many batches on two lanes + retries + long rays; one batch
        cam = W.camera("adaf", n)
        g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF); g.set_options(budget, 2)
        a = to_np(g.make_image(maps=True)); nsa, nta = g.ray_info(); sta = g.stats()
        assert sta["plan_reused"] == 0 and sta["ms_probe"] > 0
        b = to_np(g.make_image(maps=True)); nsb, ntb = g.ray_info(); stb = g.stats()
        assert stb["plan_reused"] == 1 and stb["ms_probe"] == 0
        same(a, b)
        assert np.array_equal(nsa, nsb) and np.array_equal(nta, ntb)
        for k in ("total_steps", "n_long", "n_retry", "n_batches", "n_ring", "flux_jy", "path_cap"):
            assert sta[k] == stb[k], k
        if budget:
            assert sta["n_batches"] > 3 and sta["n_lanes"] == 2 and sta["n_long"] + sta["n_retry"] > 0
        # another model under the same plan
        other = dict(W.ADAF); other["n0"] = 0.4 * W.ADAF["n0"]; other["Th0"] = 1.5 * W.ADAF["Th0"]
        g.load_adaf(**other)
        c1 = to_np(g.make_image(maps=True)); st = g.stats()
        assert st["plan_reused"] == 1
        want, ns, nt, _ = fresh(cam, other, budget)
        same(c1, want)
        assert np.array_equal(g.ray_info()[0], ns)
        # another camera: planned afresh, then reused again
        cam2 = W.camera("adaf", n, inclination_deg=35.0)
        g.set_camera(**cam2)
        d1 = to_np(g.make_image(maps=True)); assert g.stats()["plan_reused"] == 0
        d2 = to_np(g.make_image(maps=True)); assert g.stats()["plan_reused"] == 1
        want, ns, nt, _ = fresh(cam2, other, budget)
        same(d1, want); same(d2, want)
        # a pixel-list call in between drops the plan; so does the switch
        g.make_pixels(np.arange(0, n * n, 7, dtype=np.int64))
        e1 = to_np(g.make_image(maps=True)); assert g.stats()["plan_reused"] == 0
        same(e1, want)
        g.set_plan_reuse(False)
        e2 = to_np(g.make_image(maps=True)); assert g.stats()["plan_reused"] == 0
        same(e2, want)
        g.close()


def test_step_limit_flags_rays(ipole, ref):
    cam = W.camera("adaf", 16, max_steps=900)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    r = ref.Ctx(**cam); r.load_adaf(**W.ADAF)
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(256))
    assert ((want["nturn"] & 0x80) != 0).all() and (got["nturn"] == want["nturn"]).all()
    assert (got["nsteps"] == 900).all()
    check_parity(got, want, "max_steps")
    assert g.stats()["n_maxstep"] == 256


def test_edge_cases(ipole):
    import torch
    cam = W.camera("adaf", 8)
    g = ipole.Ipole(**cam)
    with pytest.raises(ipole.IpoleError) as ei:
        g.make_image()
    assert ei.value.code == ipole.ENOMODEL
    g.load_adaf(**W.ADAF)
    with pytest.raises(ipole.IpoleError) as ei:
        g.stats()
    assert ei.value.code == ipole.ENOIMAGE
    assert g.make_pixels(np.zeros(0, dtype=np.int64))["I"].size == 0          # empty list
    with pytest.raises(ipole.IpoleError):
        g.make_pixels(np.array([64], dtype=np.int64))                          # pixel out of range
    # mixed host/device outputs are rejected
    I = torch.empty((8, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(ipole.IpoleError):
        g.make_image(out=dict(I=I, Q=np.empty((8, 8)), U=I.clone(), V=I.clone()))
    # 1x1 image, and a camera swap on a live context
    g.set_camera(nx=1, ny=1)
    one = to_np(g.make_image())
    assert one["I"].size == 1 and np.isfinite(one["I"]).all()
    # a user stream
    s = torch.cuda.Stream()
    g.set_camera(nx=8, ny=8)
    ref_img = to_np(g.make_image())
    with torch.cuda.stream(s):
        g.set_stream(s)
        img = g.make_image()
    s.synchronize()
    for k in ref_img:
        assert np.array_equal(ref_img[k], to_np(img)[k])
    # flat metric refuses the ADAF flow (defined on Kerr only)
    with pytest.raises(ipole.IpoleError):
        g.set_camera(flat_metric=1)


# ------------------------------------------------------------------ slab in flat space: closed forms through the whole pipeline
def _slab_cam(n=16):
    return W.camera("adaf", n, spin=0.0, flat_metric=1, inclination_deg=40.0, fov=2.0, r_cam=500.0, r_esc=500.0)


def test_slab_flat_space_closed_forms(ipole, ref):
    L = 6.6742e-8 * 4.1e6 * 1.989e33 / 2.99792458e10 ** 2
    cam = _slab_cam()
    H = 2.0
    path = 2 * H / np.cos(np.radians(40.0)) * L  # every ray crosses the slab at the same angle in flat space (to O(fov/r_cam))
    g = ipole.Ipole(**cam); r = ref.Ctx(**cam)
    # T3 optically thin emission: I = j * path
    j = 1e-20
    for c in (g, r):
        c.load_slab(H, j=(j, 0, 0, 0))
    img = to_np(g.make_image()); want = r.make_pixels(nthreads=NTHREADS)
    assert np.allclose(img["I"], j * path, rtol=5e-3, atol=0)  # closed form (pin-hole camera: angles differ by ~fov/r_cam)
    assert np.abs(img["I"] - want["I"]).max() <= 1e-9 * want["I"].max()
    # T4 absorption with emission: I = (j/a)(1 - exp(-a path))
    a = 3.0 / path
    for c in (g, r):
        c.load_slab(H, j=(j, 0, 0, 0), alpha=(a, 0, 0, 0))
    img = to_np(g.make_image(maps=True)); want = r.make_pixels(nthreads=NTHREADS)
    assert np.allclose(img["I"], j / a * (1 - np.exp(-a * path)), rtol=5e-3, atol=0)
    assert np.allclose(img["tau"], 3.0, rtol=5e-3, atol=0)
    assert np.abs(img["I"] - want["I"]).max() <= 1e-9 * want["I"].max()
    # T5/T6 Faraday rotation and conversion with polarized emission, all coefficients (incl. the U ones) non-zero
    kw = dict(H=H, j=(j, 0.3 * j, -0.2 * j, 0.1 * j), alpha=(a, 0.2 * a, 0.1 * a, -0.05 * a), rho=(4 * a, -2 * a, 9 * a),
              psi_deg=20.0, profile=1)
    for c in (g, r):
        c.load_slab(**kw)
    got, _ = gpu_full_then_sample(g, np.arange(256))
    want = r.make_pixels(nthreads=NTHREADS)
    check_parity(got, want, "slab", min_lit=1.0)


# ------------------------------------------------------------------ configs[2..4]: grid model
@pytest.fixture(scope="module")
def small_grid():
    return W.fm_torus_grid(72, 32, 32)


def test_grid_small_full_image(ipole, ref, small_grid):
    desc, fields = small_grid
    cam = W.camera("grid", 32)
    g = ipole.Ipole(**cam); g.load_grid(desc, fields)
    r = ref.Ctx(**cam); r.load_grid(desc, fields)
    want = r.make_pixels(nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, np.arange(1024))
    info = check_parity(got, want, "grid small", min_lit=0.2)
    assert info["lit"] < 1.0  # the corners see no plasma: exercises the dark-pixel path
    # grid planes given as DEVICE pointers (torch tensors) give the same image
    import torch
    g2 = ipole.Ipole(**cam)
    g2.load_grid(desc, [torch.from_numpy(np.ascontiguousarray(f)).cuda() for f in fields])
    img2 = to_np(g2.make_image(maps=True))
    for k in img2:
        assert np.array_equal(img2[k], got[k])


def test_grid_plasma_contact_range_is_bit_neutral(ipole, small_grid, monkeypatch):
    """k_geodesic<true> marks the steps that may cross plasma and k_transfer starts at the first of them: same bits as
    walking every step (IPOLE_NO_OCC=1), through batches and the long-ray pass too."""
    desc, fields = small_grid
    cam = W.camera("grid", 48, max_steps=6000)
    monkeypatch.setenv("IPOLE_NO_OCC", "1")
    g0 = ipole.Ipole(**cam); g0.load_grid(desc, fields)
    monkeypatch.delenv("IPOLE_NO_OCC")
    base = to_np(g0.make_image(maps=True)); st0 = g0.stats()
    g = ipole.Ipole(**cam); g.load_grid(desc, fields)
    for opts in ((0, 1), (0, 2), (24 << 20, 2), (40 << 20, 0)):
        g.set_options(*opts)
        img = to_np(g.make_image(maps=True)); st = g.stats()
        for k in base:
            assert np.array_equal(base[k], img[k]), (opts, k)
        assert st["total_steps"] == st0["total_steps"] and st["flux_jy"] == st0["flux_jy"]
    assert st["n_long"] == 48 * 48
    assert (base["I"] == 0).any() and (base["I"] > 0).any()   # dark rays (never walked) and lit ones


def test_growing_retry_buffer_leaves_the_plan_lists_and_long_operator_records_alone(ipole):
    """Regression: ensure_retry_buf (the slots of the side-stream retry level) once freed the recorded plan's ray lists and
    the long-ray operator records when it grew, without forgetting the pointers -- a later call used freed memory and
    reported cudaErrorInvalidValue (seen as an intermittent failure of 4096^2 adaptive grid images).  Here the buffer is
    made to grow between images of one context (larger memory budget), with a recorded plan and long rays in play."""
    cam = W.camera("adaf", 128)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    g.set_options(768 << 20, 2)
    a = to_np(g.make_image(maps=True)); sta = g.stats()
    b = to_np(g.make_image(maps=True)); stb = g.stats()
    assert stb["plan_reused"] == 1 and sta["n_batches"] >= 3 and sta["n_long"] + sta["n_retry"] > 0
    pix = sample_pixels(128, 128, 8)
    lst0 = g.make_pixels(pix)                            # a small call: its long rays keep operator records (d_ops_long)
    for budget in (3 << 30, 12 << 30):                   # the retry level's slots grow with the budget
        g.set_options(budget, 2)
        c1 = to_np(g.make_image(maps=True)); assert g.stats()["plan_reused"] == 0
        c2 = to_np(g.make_image(maps=True)); assert g.stats()["plan_reused"] == 1
        lst = g.make_pixels(pix)
        for k in a:
            assert np.array_equal(a[k], c1[k]) and np.array_equal(a[k], c2[k]) and np.array_equal(a[k], b[k]), k
        for k in ("I", "Q", "U", "V", "tau", "tauF"):
            assert np.array_equal(lst[k], lst0[k]), k
    # a larger image on the same context: the recorded lists have to grow (freeing the old ones -- a second time, before the fix)
    cam2 = W.camera("adaf", 256)
    g.set_camera(**cam2); g.set_options(1 << 30, 2)
    d1 = to_np(g.make_image(maps=True)); assert g.stats()["plan_reused"] == 0
    d2 = to_np(g.make_image(maps=True)); st = g.stats()
    assert st["plan_reused"] == 1 and st["n_long"] + st["n_retry"] > sta["n_long"] + sta["n_retry"]
    f = ipole.Ipole(**cam2); f.load_adaf(**W.ADAF); f.set_options(1 << 30, 2)
    want = to_np(f.make_image(maps=True)); f.close()
    for k in want:
        assert np.array_equal(d1[k], want[k]) and np.array_equal(d2[k], want[k]), k
    assert ipole.lib().ipole_last_cuda_error(g._h) == 0
    g.close()


def test_low_latency_geodesic_build_is_bit_neutral(ipole, small_grid, monkeypatch):
    """Launches that cannot fill the GPU use k_geodesic compiled for 2 blocks per SM (kernels.cuh, LOWLAT): the same path
    records, step counts and images as the 4-block build (IPOLE_NO_LOWLAT=1), for both flows.  The same switch picks the
    operator walk of the analytic flow: one warp per RAY (k_apply_wide, stepop.cuh) against one warp per 32 rays (k_apply);
    the two must agree to the bit (every rounding of the Stokes update is spelt out in stokes.cuh / plasma.cuh)."""
    desc, fields = small_grid
    for kind in ("adaf", "grid"):
        cam = W.camera(kind, 96)                       # 9216 rays: every launch is under-filled
        outs = []
        for off in (True, False):
            if off:
                monkeypatch.setenv("IPOLE_NO_LOWLAT", "1")
            g = ipole.Ipole(**cam)
            if off:
                monkeypatch.delenv("IPOLE_NO_LOWLAT")
            g.load_adaf(**W.ADAF) if kind == "adaf" else g.load_grid(desc, fields)
            img = to_np(g.make_image(maps=True)); ns, nt = g.ray_info()
            outs.append((img, ns.copy(), nt.copy(), g.stats()))
            g.close()
        (a, nsa, nta, sa), (b, nsb, ntb, sb) = outs
        for k in a:
            assert np.array_equal(a[k], b[k]), (kind, k)
        assert np.array_equal(nsa, nsb) and np.array_equal(nta, ntb)
        assert sa["total_steps"] == sb["total_steps"] and sa["flux_jy"] == sb["flux_jy"]


def test_w3_grid_256_sampled(ipole, ref):
    desc, fields = W.fm_torus_grid(288, 128, 128)
    cam = W.camera("grid", 256)
    g = ipole.Ipole(**cam); g.load_grid(desc, fields)
    r = ref.Ctx(**cam); r.load_grid(desc, fields)
    pix = sample_pixels(256, 256, 8, window=(140, 124, 40, 8))
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, pix)
    check_parity(got, want, "W3", min_lit=0.3)


# ------------------------------------------------------------------ full sizes, in the configuration bench.py times
def test_w5_adaf_4096_sampled(ipole, ref):
    cam = W.camera("adaf", 4096)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    r = ref.Ctx(**cam); r.load_adaf(**W.ADAF)
    # the sample DESIGN.md section 6 / BASELINE.md declare: every 16th pixel (65 536 rays) plus every pixel of a 512 x 128
    # window across the photon ring on the +x side
    pix = sample_pixels(4096, 4096, 16, window=(2300, 1984, 512, 128))
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, img = gpu_full_then_sample(g, pix, maps=False)
    info = check_parity(got, want, "W5 adaf", min_lit=0.99)
    report("W5 adaf 4096^2", pix.size, info)
    st = g.stats()
    # the images bench.py times are scheduled from the plan of the call before them (ipole_set_plan_reuse): same bits
    again = g.make_image(maps=False)
    assert g.stats()["plan_reused"] == 1 and st["plan_reused"] == 0
    for k in img:
        assert bool((again[k] == img[k]).all()), k
    del again
    assert st["n_batches"] >= 1 and st["n_maxstep"] == 0
    # properties of the whole 4096^2 image
    import torch
    pol = torch.sqrt(img["Q"] ** 2 + img["U"] ** 2 + img["V"] ** 2)
    assert bool((pol <= img["I"] * (1 + 1e-12)).all()) and bool(torch.isfinite(img["I"]).all())
    assert abs(st["flux_jy"][0] / (float(img["I"].sum()) * (40.0 / 4096 * 6.6742e-8 * 4.1e6 * 1.989e33 / 2.99792458e10 ** 2
                                                             / (8000.0 * 3.085678e18)) ** 2 * 1e23) - 1) < 1e-12


@pytest.fixture(scope="module")
def big_grid():
    return W.fm_torus_grid(576, 256, 256)


def test_w4_grid_1024_sampled_with_maps(ipole, ref, big_grid):
    desc, fields = big_grid
    cam = W.camera("grid", 1024)
    g = ipole.Ipole(**cam); g.load_grid(desc, fields)
    r = ref.Ctx(**cam); r.load_grid(desc, fields)
    pix = sample_pixels(1024, 1024, 4, window=(560, 496, 128, 32))      # every 4th pixel (65 536 rays) + a ring window
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, _ = gpu_full_then_sample(g, pix, maps=True)
    info = check_parity(got, want, "W4", min_lit=0.3)
    report("W4 grid 1024^2", pix.size, info)


def test_w5_grid_4096_sampled(ipole, ref, big_grid):
    desc, fields = big_grid
    cam = W.camera("grid", 4096)
    g = ipole.Ipole(**cam); g.load_grid(desc, fields)
    r = ref.Ctx(**cam); r.load_grid(desc, fields)
    pix = sample_pixels(4096, 4096, 16, window=(2240, 1984, 512, 128))
    want = r.make_pixels(pix, nthreads=NTHREADS)
    got, img = gpu_full_then_sample(g, pix, maps=False)
    info = check_parity(got, want, "W5 grid", min_lit=0.3)
    report("W5 grid 4096^2", pix.size, info)
    again = g.make_image(maps=False)          # scheduled from the recorded plan, as the images bench.py times
    assert g.stats()["plan_reused"] == 1
    for k in img:
        assert bool((again[k] == img[k]).all()), k
