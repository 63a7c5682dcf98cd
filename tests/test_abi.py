"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/ipole.h
declares; the ctypes structures mirror the header; the product path fails loudly without a GPU / library."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ipole.h")


@pytest.fixture(scope="module")
def built():
    import __graft_entry__ as ge
    ge.build()
    from paper_2302_02733_b200 import ipole
    return ipole


def _declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ipole_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(built):
    lib = ctypes.CDLL(built.LIB_PATH)
    names = _declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), "missing export: " + n
    assert sorted(built.SYMBOLS) == names  # the binding knows exactly the header's entry points


def test_no_torch_or_cxx_types_in_header():
    src = open(HEADER).read()
    assert 'extern "C"' in src
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)  # declarations only
    for bad in ("torch", "at::", "std::", "Tensor", "class ", "template"):
        assert bad not in src


def test_struct_layouts_match_header(built, tmp_path):
    """sizeof/offsetof of the ABI structs as the C compiler sees them == the ctypes mirrors."""
    prog = tmp_path / "layout.c"
    prog.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "ipole.h"\nint main(void){\n'
                    'printf("%zu %zu %zu %zu %zu\\n", sizeof(ipole_camera), sizeof(ipole_adaf_params), '
                    'sizeof(ipole_slab_params), sizeof(ipole_grid_desc), sizeof(ipole_stats));\n'
                    'printf("%zu %zu %zu %zu\\n", offsetof(ipole_camera, freq_hz), offsetof(ipole_camera, hslope), '
                    'offsetof(ipole_grid_desc, startx), offsetof(ipole_stats, ms_probe));\nreturn 0;}\n')
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(prog), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()
    got = [int(v) for v in out]
    I = built
    want = [ctypes.sizeof(I.Camera), ctypes.sizeof(I.AdafParams), ctypes.sizeof(I.SlabParams), ctypes.sizeof(I.GridDesc),
            ctypes.sizeof(I.Stats), I.Camera.freq_hz.offset, I.Camera.hslope.offset, I.GridDesc.startx.offset,
            I.Stats.ms_probe.offset]
    assert got == want


def test_strerror_and_version(built):
    L = built.lib()
    assert L.ipole_strerror(0) == b"ok"
    assert b"invalid" in L.ipole_strerror(built.EINVAL)
    assert b"sm_100a" in L.ipole_version()


def test_init_rejects_bad_arguments_without_touching_the_gpu(built):
    L = built.lib()
    h = ctypes.c_void_p()
    assert L.ipole_init(None, ctypes.byref(h)) == built.EINVAL
    cam = built.Camera(spin=1.5, inclination_deg=60, r_cam=1000, fov=40, nx=8, ny=8, freq_hz=230e9)
    assert L.ipole_init(ctypes.byref(cam), ctypes.byref(h)) == built.EINVAL
    cam = built.Camera(spin=0.5, inclination_deg=0.0, r_cam=1000, fov=40, nx=8, ny=8, freq_hz=230e9)
    assert L.ipole_init(ctypes.byref(cam), ctypes.byref(h)) == built.EINVAL
    cam = built.Camera(spin=0.5, inclination_deg=60, r_cam=1000, fov=40, nx=0, ny=8, freq_hz=230e9)
    assert L.ipole_init(ctypes.byref(cam), ctypes.byref(h)) == built.EINVAL
    assert not h.value


def test_no_cpu_fallback(built):
    """Without a CUDA device the product path must fail loudly (IPOLE_ECUDA), never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(built.IpoleError) as ei:
        built.Ipole(spin=0.9, inclination_deg=60.0, r_cam=1000.0, fov=40.0, nx=8, ny=8, freq_hz=230e9)
    assert ei.value.code == built.ECUDA


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2302_02733_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                text = open(os.path.join(dirpath, f)).read()
                assert "ipole_ref" not in text and "from oracle" not in text and "import oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".hpp", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libipole_b200" not in text and "csrc" not in text, f


def test_binding_missing_library_raises(built, monkeypatch):
    monkeypatch.setattr(built, "_LIB", None)
    monkeypatch.setattr(built, "LIB_PATH", "/nonexistent/libipole_b200.so")
    with pytest.raises(ImportError):
        built.lib()
