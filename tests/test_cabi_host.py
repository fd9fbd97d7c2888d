"""CPU-side checks of the CUDA product path (no GPU): the C-ABI library builds for sm_100a, loads, exports every
symbol include/mdwf.h declares, its host logic passes its self-test, and it fails loudly without a device."""
import ctypes
import os
import re
import subprocess
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1810_01609_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "mdwf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mdwf_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(libpath):
    L = ctypes.CDLL(libpath)
    names = declared_symbols()
    assert {"mdwf_create", "mdwf_load_gauge", "mdwf_dslash", "mdwf_solve", "mdwf_seq_source", "mdwf_nucleon_2pt"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
    import paper_1810_01609_b200 as mdwf
    assert sorted(mdwf.EXPORTS) == names          # the binding covers exactly the header


def test_host_selftest(libpath):
    import paper_1810_01609_b200 as mdwf
    assert mdwf.mdwf_selftest_host(1.3, 1.5, 0.5, 0.05) == 0
    assert mdwf.mdwf_selftest_host(1.8, 1.0, 0.0, 0.3) == 0     # Shamir


def test_product_sass_is_sm100a(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out, out[:400]


def test_fp16_stencil_runs_on_tensor_cores(libpath):
    """the 16-bit stencil is an MMA kernel: its SASS holds HMMA (mma.sync f16 -> f32) instructions"""
    sass = subprocess.run(["cuobjdump", "-sass", libpath], capture_output=True, text=True).stdout
    in_hop16, hmma = False, 0
    for line in sass.splitlines():
        if "Function :" in line:
            in_hop16 = "hop16_kernel" in line
        elif in_hop16 and "HMMA." in line:
            hmma += 1
    assert hmma > 100, hmma


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback(libpath):
    import paper_1810_01609_b200 as mdwf
    with pytest.raises(RuntimeError):
        mdwf.Context((4, 4, 4, 4), 4, 1.3, 1.5, 0.5, 0.1)
    # and the C entry point itself reports the missing device instead of computing anything
    L = mdwf.lib()
    g = mdwf.binding.Geometry()
    for i in range(4):
        g.dims[i] = 4
        g.bc[i] = 1
    g.Ls, g.device = 4, 0
    h = ctypes.c_void_p()
    rc = L.mdwf_create(ctypes.byref(h), ctypes.byref(g), 1.3, 1.5, 0.5, 0.1)
    assert rc == mdwf.binding.ECUDA
    assert b"no CPU fallback" in L.mdwf_last_error(h)
    L.mdwf_destroy(h)


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1810_01609_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "mdwf_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            # the product is only ever NAMED in header comments that say the two share nothing
            code = "\n".join(l for l in text.splitlines() if not l.lstrip().startswith(("//", "#", "*", "/*", "this package", '"""')))
            assert "paper_1810_01609_b200" not in code, f
            assert "import paper_1810_01609_b200" not in text and '#include "../paper' not in text, f
