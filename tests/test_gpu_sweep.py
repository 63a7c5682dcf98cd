"""Many-small-images mode, pytest -m gpu: ipole_make_images_adaf walks the stored
paths of one geodesic pass once per parameter set.  Every image of the batch must be the image ipole_make_image gives
for that parameter set and frequency, and must match the oracle to the north-star tolerances."""
import numpy as np
import pytest

from paper_2302_02733_b200 import workloads as W
from test_gpu_parity import check_parity, to_np, ipole, NTHREADS  # noqa: F401

pytestmark = pytest.mark.gpu

MODELS = [dict(n0=1e6, Th0=30.0, B0=30.0), dict(n0=3e5, Th0=45.0, B0=20.0, p_n=-1.3), dict(n0=2e6, Th0=12.0, B0=55.0, p_T=-0.8),
          dict(n0=5e6, Th0=8.0, B0=80.0, p_B=-1.1), dict(n0=1e5, Th0=60.0, B0=10.0)]
FREQS = [230e9, 345e9, 86e9, 230e9, 690e9]


def single(ipole, cam, model, freq, maps=True):
    g = ipole.Ipole(**dict(cam, freq_hz=freq)); g.load_adaf(**model)
    img = to_np(g.make_image(maps=maps))
    return img, g.stats()


def close(a, b, scale):
    return np.abs(a - b).max() <= 1e-12 * scale


def test_sweep_equals_single_images_and_oracle(ipole, ref):
    cam = W.camera("adaf", 32)
    g = ipole.Ipole(**cam)
    out = g.make_images_adaf(MODELS, FREQS, maps=True)
    st = g.stats()
    assert st["n_batches"] == 1
    for m, (mod, fr) in enumerate(zip(MODELS, FREQS)):
        img, st1 = single(ipole, cam, mod, fr)
        sc = img["I"].max()
        for k in ("I", "Q", "U", "V"):
            assert close(out[k][m].cpu().numpy().ravel(), img[k], sc), (m, k)
        for k in ("tau", "tauF"):
            assert np.allclose(out[k][m].cpu().numpy().ravel(), img[k], rtol=1e-12, atol=0), (m, k)
        assert np.allclose(out["flux_jy"][m], st1["flux_jy"], rtol=1e-12, atol=1e-12 * abs(st1["flux_jy"][0]))
        # against the oracle, north-star tolerances
        r = ref.Ctx(**dict(cam, freq_hz=fr)); r.load_adaf(**mod)
        want = r.make_pixels(nthreads=NTHREADS)
        got = {k: out[k][m].cpu().numpy().ravel() for k in ("I", "Q", "U", "V", "tau", "tauF")}
        check_parity(got, want, "sweep model %d" % m, min_lit=0.99)
    # the shared geodesic pass is the ordinary one
    assert st["total_steps"] == int(want["nsteps"].sum())


def test_sweep_chunks_batches_long_rays_and_host_buffers(ipole):
    cam = W.camera("adaf", 24, max_steps=6000)
    g = ipole.Ipole(**cam)
    g.load_adaf(n0=7e5)                          # a loaded model must survive the sweep untouched
    before = to_np(g.make_image())
    models = [dict(n0=1e6 * (1 + 0.03 * (m % 64)), Th0=30.0 - 0.2 * (m % 64)) for m in range(70)]   # > 64: two chunks
    a = g.make_images_adaf(models, maps=True)
    A = {k: a[k].cpu().numpy() for k in ("I", "Q", "U", "V", "tau", "tauF")}
    for k in A:
        assert np.array_equal(A[k][0:6], A[k][64:70]), k      # same parameters in both chunks: same bits
    assert not np.array_equal(A["I"][0], A["I"][1])
    after = to_np(g.make_image())
    for k in before:
        assert np.array_equal(before[k], after[k])
    # spot-check two images of the batch against single calls
    for m in (3, 69):
        img, _ = single(ipole, cam, models[m], cam["freq_hz"])
        for k in ("I", "Q", "U", "V"):
            assert close(A[k][m].ravel(), img[k], img["I"].max()), (m, k)
    # host buffers: the same bits as device buffers
    h = g.make_images_adaf(models, maps=True, host=True)
    for k in A:
        assert np.array_equal(h[k], A[k]), k
    assert np.array_equal(h["flux_jy"], a["flux_jy"])
    # tiny path buffer: several ray batches, S_cap from the probe; then a slot too small for any ray (long-ray pass).
    # The bulk of a sweep runs k_stepop once + k_apply per parameter set, its long rays the single sweep kernel: the two
    # agree to rounding (as for single images), and each is bit-neutral to batching on its own.
    peak = A["I"][:9].max()
    for opts in ((8 << 20, 2), (12 << 20, 0)):
        g.set_options(*opts)
        b = g.make_images_adaf(models[:9], maps=True)
        st = g.stats()
        assert st["n_batches"] > 1 or st["n_long"] > 0
        for k in ("I", "Q", "U", "V"):
            assert np.abs(b[k].cpu().numpy() - A[k][:9]).max() <= 1e-11 * peak, (opts, k)
        for k in ("tau", "tauF"):
            assert np.allclose(b[k].cpu().numpy(), A[k][:9], rtol=1e-11, atol=0), (opts, k)
    g.set_options(0, 1); g.set_transfer_split(False)          # the single sweep kernel everywhere: same bits whatever the batching
    a0 = g.make_images_adaf(models[:9], maps=True)
    A0 = {k: a0[k].cpu().numpy() for k in A}
    for k in ("I", "Q", "U", "V"):
        assert np.abs(A0[k] - A[k][:9]).max() <= 1e-11 * peak, k
    for opts in ((8 << 20, 2), (12 << 20, 0)):
        g.set_options(*opts)
        b = g.make_images_adaf(models[:9], maps=True)
        for k in A:
            assert np.array_equal(b[k].cpu().numpy(), A0[k]), (opts, k)
    g.set_transfer_split(True)
    # the path-free switch does not apply to the sweep (the shared stored path is its point)
    g.set_options(0, 1); g.set_path_free(True)
    c = g.make_images_adaf(models[:3])
    for k in ("I", "Q", "U", "V"):
        assert np.array_equal(c[k].cpu().numpy(), A[k][:3])


def test_sweep_errors(ipole):
    g = ipole.Ipole(**W.camera("adaf", 8))
    with pytest.raises(ipole.IpoleError):
        g.make_images_adaf([])
    with pytest.raises(ipole.IpoleError):
        g.make_images_adaf([dict()], freqs=[0.0])
    flat = ipole.Ipole(**W.camera("adaf", 8, spin=0.0, flat_metric=1))
    with pytest.raises(ipole.IpoleError):
        flat.make_images_adaf([dict()])
    out = g.make_images_adaf([dict()])        # one model, default parameters = W1's flow
    g.load_adaf(**W.ADAF)
    img = to_np(g.make_image())
    assert close(out["I"][0].cpu().numpy().ravel(), img["I"], img["I"].max())


def test_grid_sweep_equals_single_images_and_oracle(ipole, ref):
    desc, fields = W.fm_torus_grid(72, 32, 32)
    cam = W.camera("grid", 32)
    sets = [dict(M_unit=desc["M_unit"], Rlow=desc["Rlow"], Rhigh=desc["Rhigh"]),
            dict(M_unit=3.0 * desc["M_unit"], Rlow=1.0, Rhigh=10.0), dict(M_unit=0.2 * desc["M_unit"], Rlow=2.0, Rhigh=80.0),
            dict(M_unit=desc["M_unit"], Rlow=1.0, Rhigh=1.0)]
    freqs = [230e9, 230e9, 86e9, 345e9]
    g = ipole.Ipole(**cam); g.load_grid(desc, fields)
    before = to_np(g.make_image(maps=True))
    out = g.make_images_grid(sets, freqs, maps=True)
    after = to_np(g.make_image(maps=True))
    for k in before:
        assert np.array_equal(before[k], after[k]), k      # the loaded model is untouched
    for m, (st_, fr) in enumerate(zip(sets, freqs)):
        d = dict(desc); d.update(st_)
        g1 = ipole.Ipole(**dict(cam, freq_hz=fr)); g1.load_grid(d, fields)
        img = to_np(g1.make_image(maps=True)); s1 = g1.stats()
        sc = img["I"].max()
        for k in ("I", "Q", "U", "V"):
            assert close(out[k][m].cpu().numpy().ravel(), img[k], sc), (m, k)
        for k in ("tau", "tauF"):
            assert np.allclose(out[k][m].cpu().numpy().ravel(), img[k], rtol=1e-12, atol=0), (m, k)
        assert np.allclose(out["flux_jy"][m], s1["flux_jy"], rtol=1e-12, atol=1e-12 * abs(s1["flux_jy"][0]))
        r = ref.Ctx(**dict(cam, freq_hz=fr)); r.load_grid(d, fields)
        want = r.make_pixels(nthreads=NTHREADS)
        got = {k: out[k][m].cpu().numpy().ravel() for k in ("I", "Q", "U", "V", "tau", "tauF")}
        check_parity(got, want, "grid sweep set %d" % m, min_lit=0.2)
    assert np.array_equal(out["I"][0].cpu().numpy().ravel(), before["I"]) or close(out["I"][0].cpu().numpy().ravel(), before["I"], before["I"].max())
    # 70 sets: two chunks; host buffers
    many = [dict(M_unit=desc["M_unit"] * (1 + 0.05 * (m % 64)), Rlow=1.0, Rhigh=40.0) for m in range(70)]
    a = g.make_images_grid(many)
    h = g.make_images_grid(many, host=True)
    for k in ("I", "Q", "U", "V"):
        A = a[k].cpu().numpy()
        assert np.array_equal(A[0:6], A[64:70]) and np.array_equal(h[k], A), k
    # The bulk of a grid sweep runs k_gridop once + k_gridapply_sweep per set (gridsweep.cuh), long rays the single sweep
    # kernel.  Several ray batches, then slots too short for any ray (every ray a long ray), then the single kernel
    # everywhere (ipole_set_transfer_split(0)): the same images to rounding, amplified where the Faraday depth is large.
    A = {k: a[k].cpu().numpy()[:9] for k in ("I", "Q", "U", "V")}
    peak = A["I"].max()
    for opts, split in (((8 << 20, 2), True), ((12 << 20, 0), True), ((0, 1), False)):
        g.set_options(*opts); g.set_transfer_split(split)
        b = g.make_images_grid(many[:9])
        st = g.stats()
        if split:
            assert st["n_batches"] > 1 or st["n_long"] > 0
        else:
            assert st["ms_stepop"] == 0
        for k in A:
            assert np.abs(b[k].cpu().numpy() - A[k]).max() <= 1e-9 * peak, (opts, split, k)
    g.set_options(0, 1); g.set_transfer_split(True)
    assert g.make_images_grid(many[:2]) is not None and g.stats()["ms_stepop"] > 0
    # errors
    with pytest.raises(ipole.IpoleError):
        g.make_images_grid([dict(M_unit=0.0, Rlow=1.0, Rhigh=1.0)])
    g0 = ipole.Ipole(**cam)
    with pytest.raises(ipole.IpoleError) as ei:
        g0.make_images_grid(sets)
    assert ei.value.code == ipole.ENOMODEL


def test_independent_contexts_side_by_side(ipole):
    """include/ipole.h: distinct contexts are independent.  Four cameras on four contexts, streams and host threads
    give the same bits as one after the other (bench.py --workload cams128 measures the gain)."""
    import threading
    import torch
    incl = [25.0, 45.0, 60.0, 75.0]
    cams = [W.camera("adaf", 40, inclination_deg=a) for a in incl]
    want = []
    for cam in cams:
        g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
        want.append(to_np(g.make_image(maps=True)))
    ctxs, streams, outs = [], [], [None] * 4
    for cam in cams:
        g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF); g.set_options(1 << 30, 1)
        s = torch.cuda.Stream(); g.set_stream(s)
        ctxs.append(g); streams.append(s)

    def work(k):
        outs[k] = ctxs[k].make_image(maps=True)
    for _ in range(3):
        ts = [threading.Thread(target=work, args=(k,)) for k in range(4)]
        for t in ts: t.start()
        for t in ts: t.join()
        for s in streams: s.synchronize()
        for k in range(4):
            got = to_np(outs[k])
            for name in want[k]:
                assert np.array_equal(got[name], want[k][name]), (k, name)


def test_sweep_of_more_than_one_chunk_with_long_rays(ipole):
    """70 parameter sets (two table chunks) AND a path budget so small that rays overflow their slots: the long-ray
    passes walk the same chunks on the side stream while the main stream walks them for the bulk; each stream has its
    own parameter tables (a shared one could hand a kernel the other chunk's parameters)."""
    cam = W.camera("adaf", 24, max_steps=6000)
    models = [dict(n0=1e6 * (1 + 0.03 * m), Th0=30.0 - 0.2 * (m % 64), B0=30.0 + 0.1 * m) for m in range(70)]
    g = ipole.Ipole(**cam)
    split = g.make_images_adaf(models)         # bulk through k_stepop + k_apply<sweep>
    g.set_transfer_split(False)                # long rays take the single sweep kernel: compare like with like
    want = g.make_images_adaf(models)
    assert g.stats()["n_long"] == 0
    W_ = {k: want[k].cpu().numpy() for k in ("I", "Q", "U", "V")}
    for k in W_:
        assert np.abs(split[k].cpu().numpy() - W_[k]).max() <= 1e-11 * W_["I"].max(), k
    # a batch in which k_stepop meets a ray it cannot express falls back to the single sweep kernel as a whole (test mode 2
    # of the switch declares every seventh ray such a ray)
    g.set_transfer_split(2)
    fb = g.make_images_adaf(models)
    for k in W_:
        assert np.array_equal(fb[k].cpu().numpy(), W_[k]), k
    g.set_transfer_split(False)
    for rep in range(3):                       # a race would not show every time
        g.set_options(6 << 20, 0)              # no probe, slots far shorter than the rays: every ray is a long ray
        got = g.make_images_adaf(models)
        assert g.stats()["n_long"] > 0
        for k in W_:
            assert np.array_equal(got[k].cpu().numpy(), W_[k]), (rep, k)


def test_adaptive_sweep_adaptive_on_one_context(ipole):
    """The sweep entry must leave the adaptive entry's buffers and events alone (it used to free them when its own
    staging buffer grew): adaptive -> sweep with growing n_models -> adaptive gives the same image twice."""
    cam = W.camera("adaf", 48)
    g = ipole.Ipole(**cam); g.load_adaf(**W.ADAF)
    a1, i1 = g.make_image_adaptive(2, 0.05, 0.0, host=True)
    for M in (2, 9, 33):                       # host outputs: the staging buffer grows with every call
        g.make_images_adaf([dict(n0=1e6 * (1 + 0.1 * m)) for m in range(M)], host=True)
    a2, i2 = g.make_image_adaptive(2, 0.05, 0.0, host=True)
    for k in ("I", "Q", "U", "V", "state"):
        assert np.array_equal(a1[k], a2[k]), k
    assert i1["n_traced"] == i2["n_traced"]


def test_set_camera_with_a_new_mass_rescales_the_grid_units(ipole):
    """ipole_set_camera keeps the loaded grid model; its density and field units contain GM/c^2, so a new mass must give
    the image a fresh context with that mass gives (they used to keep the old length unit)."""
    desc, fields = W.fm_torus_grid(48, 24, 16)
    cam1, cam2 = W.camera("grid", 24), W.camera("grid", 24, mbh_msun=6.5e9, dsource_pc=16.8e6)
    g = ipole.Ipole(**cam1); g.load_grid(desc, fields)
    g.make_image()
    g.set_camera(**cam2)
    a = to_np(g.make_image())
    f = ipole.Ipole(**cam2); f.load_grid(desc, fields)
    b = to_np(f.make_image())
    assert (b["I"] > 0).any()
    for k in ("I", "Q", "U", "V"):
        assert np.array_equal(a[k], b[k]), k
