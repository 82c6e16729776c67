"""C-ABI boundary (-m "not gpu"): libargus.so loads without a GPU and exports every symbol include/argus.h
declares; host-side validation answers without touching a device; the binding refuses to run without CUDA
(no CPU fallback); the product package never imports the oracle."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "argus.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(argus_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    import paper_2207_14304_b200 as argus
    return argus.load_library()


def test_header_symbols_are_exported(lib):
    names = _declared()
    assert {"argus_calibrate", "argus_healpix_footprint", "argus_resample", "argus_coadd_accumulate"} <= set(names)
    for n in names:
        assert getattr(lib, n) is not None, n
    from paper_2207_14304_b200.binding import EXPORTS
    assert sorted(EXPORTS) == names


def test_dynamic_symbol_table_is_c_abi():
    import paper_2207_14304_b200 as argus
    out = subprocess.run(["nm", "-D", "--defined-only", argus.library_path()], capture_output=True, text=True, check=True).stdout
    syms = {line.split()[-1] for line in out.splitlines() if " T " in line}
    for n in _declared():
        assert n in syms, n + " is not an unmangled extern \"C\" symbol"


def test_host_side_validation_without_device(lib):
    lib.argus_strerror.restype = C.c_char_p
    assert lib.argus_strerror(0) == b"ok"
    assert b"nside" in lib.argus_strerror(-3)
    assert lib.argus_version() >= 100
    assert lib.argus_ctx_create(None, 0, 0) == -1            # ARGUS_ERR_NULL before any CUDA call
    h = C.c_void_p()
    assert lib.argus_ctx_create(C.byref(h), 0, 5) == -2      # max_tiles out of range: ARGUS_ERR_SHAPE
    assert lib.argus_ctx_destroy(None) == -1
    assert lib.argus_calibrate(None, None, None, None, None, None, 4, 4, 1.0, 65535, 0.1, None, None, None) == -1
    n = C.c_size_t()
    assert lib.argus_healpix_footprint(None, None, 4, 4, 1 << 17, None, 0, C.byref(n), None) == -1
    n.value = 77
    assert lib.argus_segment_products(None, 1 << 17, 1 << 14, None, None, None, 0, None, 0, None, None, None, None, None,
                                      None, 0, None, C.byref(n), None) == -1
    # background map / source detection: NULL context before any CUDA call, count reset
    assert lib.argus_background_map(None, None, 64, 64, 64, 16, None, None, None, None, None, None) == -1
    n.value = 77
    assert lib.argus_detect_sources(None, None, 64, 64, 64, None, None, C.c_float(5.0), None, 0, None, C.byref(n), None) == -1
    assert n.value == 77                                      # a NULL context touches nothing


def test_argus_source_record_layout_matches_binding():
    """argus_source (argus.h) is 32 bytes: int32 x, y; float peak, flux, cx, cy, bkg, nse -- the binding's SOURCE_DTYPE."""
    import numpy as np

    from paper_2207_14304_b200.binding import SOURCE_DTYPE
    dt = np.dtype(SOURCE_DTYPE)
    assert dt.itemsize == 32 and dt.names == ("x", "y", "peak", "flux", "cx", "cy", "bkg", "nse")
    text = open(os.path.join(ROOT, "include", "argus.h")).read()
    body = text[text.index("typedef struct argus_source {"):text.index("} argus_source;")]
    fields = [w.strip(" ,;") for line in body.splitlines()[1:] for w in line.split("/*")[0].replace("int32_t", "").replace("float", "").split(",")]
    assert [f for f in fields if f] == list(dt.names)


def test_no_cpu_fallback():
    import torch

    import paper_2207_14304_b200 as argus
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        argus.Context(0)


def test_product_does_not_import_oracle():
    code = "import sys; import paper_2207_14304_b200 as a; a.load_library(); assert 'oracle' not in sys.modules"
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)
    pkg = os.path.join(ROOT, "paper_2207_14304_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dp, f)).read()
                for needle in ("import oracle", "from oracle", "argus_oracle", "orc_"):
                    assert needle not in text, "%s mentions %s" % (f, needle)
