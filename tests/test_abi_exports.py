"""CPU-side checks of the boundary: the CUDA library builds for sm_100a, loads, and exports every symbol that
include/gfcc.h declares; the binding refuses to compute without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "gfcc.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(gfcc_[a-z_0-9]+)\s*\(", txt)))


def test_library_builds_and_exports_all_declared_symbols():
    from paper_2010_04768_b200 import build, EXPORTS
    path = build.build()
    lib = ctypes.CDLL(path)
    decl = declared_symbols()
    assert len(decl) >= 12
    for name in decl:
        assert hasattr(lib, name), f"{name} declared in gfcc.h but not exported"
    assert sorted(EXPORTS) == decl


def test_sass_is_sm100a_dmma():
    import subprocess
    from paper_2010_04768_b200 import build
    path = build.build()
    out = subprocess.run(["cuobjdump", "-sass", path], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert "DMMA.8x8x4" in out            # FP64 tensor-core MMA
    assert "LDGSTS" in out                # cp.async shared-memory staging
    assert "UTCIMMA" in out               # tcgen05.mma kind::i8 (INT8 engine)
    assert "UTMALDG" in out               # TMA loads
    assert "LDTM" in out                  # tcgen05.ld (TMEM -> registers)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2010_04768_b200 as g
    with pytest.raises(g.GfccError):
        g.gfcc_create(2, 2, 1, *[torch.zeros(1, dtype=torch.float64)] * 6)
    # the C entry point itself also refuses: null handle / no device
    lib = g.lib()
    out = ctypes.c_void_p()
    z = (ctypes.c_double * 64)()
    rc = lib.gfcc_create(2, 2, 1, z, z, z, z, z, z, ctypes.byref(out))
    assert rc == g.GFCC_ECUDA and not out.value
    assert b"no CUDA device" in lib.gfcc_last_error(None)
    assert lib.gfcc_create(1, 2, 1, z, z, z, z, z, z, ctypes.byref(out)) == g.GFCC_EINVAL


def test_product_does_not_import_oracle():
    import sys
    import subprocess
    code = "import sys; import paper_2010_04768_b200, gfcc_inputs; assert 'oracle' not in sys.modules; print('ok')"
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, capture_output=True, text=True)
    assert out.stdout.strip() == "ok", out.stderr
    for fn in os.listdir(os.path.join(ROOT, "paper_2010_04768_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_2010_04768_b200", "csrc", fn)).read().lower().replace("no oracle", "")
