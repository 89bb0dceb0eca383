"""CPU-only: the C-ABI library builds, loads and exports every symbol include/gbe.h declares (no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1603_00937_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "gbe.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gbe_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    assert "gbe_build_graph" in syms and "gbe_density" in syms and "gbe_free_graph" in syms
    assert len(syms) >= 10


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    for s in declared_symbols():
        assert hasattr(lib, s), s


def test_binding_lists_the_same_symbols(libpath):
    import paper_1603_00937_b200 as pkg
    assert sorted(pkg.EXPORTS) == declared_symbols()
    l = pkg.lib()
    assert l.gbe_strerror(0) == b"ok"
    assert b"invalid" in l.gbe_strerror(-1)
    assert b"sm_100a" in l.gbe_version()


def test_null_arguments_are_rejected_without_a_gpu(libpath):
    lib = ctypes.CDLL(libpath)
    assert lib.gbe_graph_get_info(None, None) == -1
    out = ctypes.c_void_p()
    assert lib.gbe_build_graph(None, None, None, 1, None, ctypes.byref(out)) == -1
    assert lib.gbe_density(None, None, ctypes.c_double(0), 1, ctypes.c_double(-1), None, 0, None, None, None) == -1
    lib.gbe_free_graph(None)  # no-op


def test_sass_uses_fp64_tensor_cores_and_async_copies(libpath):
    import shutil
    import subprocess
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    sass = subprocess.run(["cuobjdump", "-sass", libpath], capture_output=True, text=True).stdout
    assert "DMMA.8x8x4" in sass      # mma.sync f64 -> FP64 tensor pipe
    assert "LDGSTS" in sass          # cp.async staging of the X panels
    assert "UTMALDG" in sass         # 2-D tensor-map TMA loads of the X^2 panels (cp.async.bulk.tensor)
    assert "UBLKCP" in sass          # TMA bulk copies (cp.async.bulk) of the packed small-m kernel
    assert "ACQBULK" in sass and "PREEXIT" in sass  # griddepcontrol.wait / .launch_dependents (dependent launch)
    assert "sm_100a" in sass


def test_sources_take_the_current_device_not_a_literal_one():
    """include/gbe.h: every call works on the CURRENT device.  No CUDA runtime query in the sources may name a device by a
    literal index, none may assume the SM count of one product, and one-time set-up must not hang on a process-wide flag."""
    import glob
    bad = []
    for path in sorted(glob.glob(os.path.join(ROOT, "paper_1603_00937_b200", "csrc", "*.cu*"))):
        text = open(path).read()
        code = re.sub(r"//[^\n]*", "", text)
        for m in re.finditer(r"cudaDeviceGetAttribute\s*\(([^;]*?)\)\s*[;)]", code, flags=re.S):
            last = m.group(1).split(",")[-1].strip()
            if re.fullmatch(r"\d+", last):
                bad.append((os.path.basename(path), "cudaDeviceGetAttribute(..., %s)" % last))
        for m in re.finditer(r"\b148\b", code):
            bad.append((os.path.basename(path), "literal SM count 148"))
        for m in re.finditer(r"static\s+bool\s+\w+\s*=\s*false", code):
            bad.append((os.path.basename(path), m.group(0)))
        for m in re.finditer(r"cudaSetDevice\s*\(\s*\d+\s*\)|cudaDeviceGetDefaultMemPool\s*\([^,]*,\s*\d+\s*\)", code):
            bad.append((os.path.basename(path), m.group(0)))
    assert not bad, bad
