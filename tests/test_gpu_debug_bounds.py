"""-m gpu: the ARGUS_DEBUG_BOUNDS build of the library (every shared-memory gather of the staged kernels checked on the
device against its staged box) over config 0, the special pointings and 8 fuzz geometries -- the out-of-bounds evidence
compute-sanitizer would give, which is not available on the GPU pool.  Runs in a subprocess with the debug library, so
that the product library stays the one every other test loads."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_no_gather_leaves_its_staged_box():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    sys.path.insert(0, ROOT)
    from paper_2207_14304_b200 import _build
    lib = _build.build(debug_bounds=True)
    env = dict(os.environ, ARGUS_LIBRARY=lib)
    out = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "debug_bounds_run.py")], env=env, capture_output=True,
                         text=True, timeout=900)
    assert out.returncode == 0, out.stdout[-2000:] + out.stderr[-4000:]
    assert "debug bounds ok" in out.stdout
    print(out.stdout.strip().splitlines()[-1])
    # the check itself fires when the staged box is pretended narrower than it is
    out = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "debug_bounds_run.py"), "--expect-violation"], env=env,
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and "violation detected" in out.stdout, out.stdout[-2000:] + out.stderr[-2000:]


def test_forced_margins_produce_strays_served_exactly():
    """ARGUS_OPT_UNIT_MARGIN < 0 makes the unit boxes too small for some sub-blocks: plan_units_kernel must find them
    (n_stray > 0) and the stray kernel must serve them within the tolerance; margin 0 has no stray at this geometry."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    sys.path.insert(0, ROOT)
    import numpy as np
    import oracle
    import paper_2207_14304_b200 as argus
    import synth
    from gpu_util import assert_values_match, upload
    fr = synth.config0()
    ctx = argus.Context(0)
    try:
        ctx.set_fast_path(3)
        d = upload(fr)
        idx_or, _ = oracle.footprint(fr.wcs, 512, 512, fr.nside)
        cal, mask = oracle.calibrate_frame(fr)
        vo, wo, fl = oracle.resample(cal, mask, fr.wcs, fr.nside, idx_or, oracle.BILINEAR)
        for margin in (0, -1, -2, -8):
            ctx.set_unit_margin(margin)
            v = torch.full((len(idx_or),), float("nan"), dtype=torch.float32, device="cuda")
            w = torch.full_like(v, float("nan"))
            argus.argus_resample(ctx, fr.wcs, 512, 512, fr.nside, "bilinear", v, w, **d)
            torch.cuda.synchronize()
            info = argus.argus_plan_info(ctx)
            assert info["n_units"] > 0
            assert (info["n_stray"] > 0) == (margin < 0), info
            assert_values_match(v.cpu().numpy(), w.cpu().numpy(), vo, wo, fl, "unit kernel, margin %d (%d strays)" % (margin, info["n_stray"]))
    finally:
        ctx.close()
