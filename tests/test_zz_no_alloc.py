"""ipole_image_totals_static (include/ipole.h): the image totals through the entry point that allocates nothing (its
block partials live in a static __device__ array of the library) against the existing path -- the reduction
ipole_make_image ends with, read through ipole_get_stats -- on two calls in a row.  This file is named so that pytest
collects it last; it must pass both alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_2302_02733_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ipole():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import __graft_entry__ as ge
    ge.build()
    from paper_2302_02733_b200 import ipole as mod
    return mod


def _check(st, got, rays):
    # tolerances of the whole-image parity tests: sum I relative 1e-9, Q, U, V absolute 1e-9 of sum I
    f = st["flux_jy"]
    assert f[0] > 0
    assert abs(got[0] - f[0]) <= 1e-9 * f[0]
    for k in (1, 2, 3):
        assert abs(got[k] - f[k]) <= 1e-9 * f[0], k
    assert abs(got[4] - st["lp"]) <= 1e-9 and abs(got[5] - st["cp"]) <= 1e-9


def test_totals_without_allocation_match_the_stats_of_the_image_twice_in_a_row(ipole):
    import torch
    n = 96                                   # 9216 pixels: one block with a ragged tail
    g = ipole.Ipole(**W.camera("adaf", n)); g.load_adaf(**W.ADAF)
    g.set_stream(torch.cuda.current_stream())
    img = g.make_image()
    st = g.stats()
    out = torch.full((6,), float("nan"), dtype=torch.float64, device="cuda")
    g.image_totals_static(img["I"], img["Q"], img["U"], img["V"], out)
    first = out.cpu().numpy().copy()
    _check(st, first, n * n)
    # second call, other input: the scratch array still holds the first call's partials and nothing clears it
    half = {k: (0.5 * img[k]).contiguous() for k in "IQUV"}
    out2 = torch.full((6,), float("nan"), dtype=torch.float64, device="cuda")
    g.image_totals_static(half["I"], half["Q"], half["U"], half["V"], out2)
    g.image_totals_static(img["I"], img["Q"], img["U"], img["V"], out)      # and the first input again, right behind it
    second = out2.cpu().numpy()
    again = out.cpu().numpy()
    assert np.array_equal(again, first)      # fixed summation order: the same bits
    assert np.allclose(second[:4], 0.5 * first[:4], rtol=1e-14, atol=0) and np.allclose(second[4:], first[4:], rtol=1e-13, atol=0)
    g.close()


def test_totals_across_many_blocks_and_the_size_limit(ipole):
    import torch
    n = 640                                  # 409 600 pixels = 25 blocks of 16 384
    g = ipole.Ipole(**W.camera("adaf", n)); g.load_adaf(**W.ADAF)
    g.set_stream(torch.cuda.current_stream())
    img = g.make_image()
    st = g.stats()
    out = torch.zeros(6, dtype=torch.float64, device="cuda")
    g.image_totals_static(img["I"], img["Q"], img["U"], img["V"], out)
    _check(st, out.cpu().numpy(), n * n)
    # against an independent sum of the planes (float64 on the host, pairwise)
    pix = st["flux_jy"][0] / float(img["I"].sum().cpu())
    ref = np.array([float(np.sum(img[k].cpu().numpy())) * pix for k in "IQUV"])
    assert np.allclose(out.cpu().numpy()[:4], ref, rtol=1e-9, atol=1e-9 * ref[0])
    # beyond the fixed maximum: a clear error, nothing launched, out untouched
    keep = out.clone()
    lib = ipole.lib()
    p = img["I"].data_ptr()
    too_many = ipole.C.c_int64(16777216 + 1)
    rc = lib.ipole_image_totals_static(g._h, too_many, p, p, p, p, out.data_ptr())
    assert rc == ipole.ETOOBIG and b"maximum" in lib.ipole_strerror(rc)
    assert lib.ipole_image_totals_static(g._h, ipole.C.c_int64(0), p, p, p, p, out.data_ptr()) == ipole.EINVAL
    assert lib.ipole_image_totals_static(g._h, ipole.C.c_int64(16), p, p, p, None, out.data_ptr()) == ipole.EINVAL
    torch.cuda.synchronize()
    assert torch.equal(out, keep)
    g.close()
