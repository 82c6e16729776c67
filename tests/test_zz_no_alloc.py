"""GPU test (-m gpu) of argus_background_map_static, the entry point that allocates nothing (include/argus.h): its cell
scratch is a file-scope device array of the library.  Collected last on purpose (the suite runs with pytest -x).

It runs the same two kernels as argus_background_map (R-D1, R-D2 of DESIGN.md section 11), so its outputs are compared
with that path's BIT FOR BIT (the medians are exact selections: tests/test_gpu_background.py holds the existing path to
the oracle), on two calls in a row that share the array: the second call, on a different and smaller frame, must not see
anything of the first, and a third call repeats the first.  Passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import synth  # noqa: E402,F401
from synth import frames as sf  # noqa: E402
from gpu_util import upload  # noqa: E402

DEV = "cuda:0"


@pytest.fixture(scope="module")
def argus():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2207_14304_b200 as a
    a.load_library()
    torch.cuda.set_device(0)
    return a


def _grids(W, H, B):
    g = -(-H // B) * -(-W // B)
    return (torch.full((g,), float("nan"), dtype=torch.float32, device=DEV),
            torch.full((g,), float("nan"), dtype=torch.float32, device=DEV))


def _existing(argus, W, H, B, n_min, frame):
    ctx = argus.Context(0)
    try:
        bkg, nse = _grids(W, H, B)
        argus.argus_background_map(ctx, W, H, bkg, nse, cell=B, n_min=n_min, **frame)
        torch.cuda.synchronize()
        return bkg.cpu().numpy(), nse.cpu().numpy()
    finally:
        ctx.close()


def _static(argus, W, H, B, n_min, frame):
    bkg, nse = _grids(W, H, B)
    argus.argus_background_map_static(W, H, bkg, nse, cell=B, n_min=n_min, **frame)
    torch.cuda.synchronize()
    return bkg.cpu().numpy(), nse.cpu().numpy()


def _same(a, b):
    # bit patterns: +inf noise of cells without a valid neighbour and signed zeros included
    return np.array_equal(a.view(np.uint32), b.view(np.uint32))


def test_static_scratch_matches_existing_path_on_two_calls_in_a_row(argus):
    # call 1: config 0 with fused calibration (raw + masters, defects, saturated stars), 64-pixel cells
    fr = sf.config0()
    H1, W1 = fr.shape
    f1 = upload(fr)
    # call 2: a smaller ragged calibrated frame with a hole of invalid cells, 16-pixel cells: fewer cells than call 1
    # left behind in the array, other values
    rng = np.random.default_rng(2207)
    H2, W2 = 130, 333
    cal = rng.normal(150.0, 9.0, (H2, W2)).astype(np.float32)
    mask = (rng.random((H2, W2)) > 0.03).astype(np.uint8)
    mask[10:90, 20:120] = 0
    cal[mask == 0] = 0.0
    f2 = dict(cal=torch.from_numpy(cal).to(DEV), mask=torch.from_numpy(mask).to(DEV))

    want1 = _existing(argus, W1, H1, 64, 16, f1)
    want2 = _existing(argus, W2, H2, 16, 8, f2)
    assert np.isfinite(want1[0]).all() and np.isinf(want2[1]).any() and np.isfinite(want2[1]).any()

    got1 = _static(argus, W1, H1, 64, 16, f1)
    got2 = _static(argus, W2, H2, 16, 8, f2)
    got3 = _static(argus, W1, H1, 64, 16, f1)
    for got, want, what in ((got1, want1, "first call"), (got2, want2, "second call"), (got3, want1, "third call")):
        assert _same(got[0], want[0]), what + ": bkg differs from argus_background_map"
        assert _same(got[1], want[1]), what + ": nse differs from argus_background_map"


def test_static_scratch_allocates_nothing(argus):
    """Device memory in use (driver view) does not move over repeated calls.  One call first: the CUDA runtime loads a
    kernel's module at its first launch in the process (lazy loading), which is not an allocation of the entry point's.
    torch's caching allocator is not involved: the outputs exist before the first reading."""
    fr = sf.config0()
    H, W = fr.shape
    f = upload(fr)
    bkg, nse = _grids(W, H, 8)
    argus.argus_background_map_static(W, H, bkg, nse, cell=8, n_min=1, **f)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(0)
    for _ in range(3):
        argus.argus_background_map_static(W, H, bkg, nse, cell=8, n_min=1, **f)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(0)
    assert free1 == free0
    assert torch.isfinite(bkg).all()


def test_static_scratch_rejects_grids_beyond_its_maximum(argus):
    from paper_2207_14304_b200 import binding
    W = H = 8 * 1025                       # 1025 x 1025 cells of 8 pixels > 2^20
    assert (W // 8) * (H // 8) > binding.ARGUS_BG_STATIC_MAX_CELLS
    cal = torch.zeros((H, W), dtype=torch.float32, device=DEV)
    mask = torch.ones((H, W), dtype=torch.uint8, device=DEV)
    bkg, nse = _grids(W, H, 8)
    with pytest.raises(argus.ArgusError) as e:
        argus.argus_background_map_static(W, H, bkg, nse, cell=8, n_min=1, cal=cal, mask=mask)
    assert e.value.status == -6 and "ARGUS_BG_STATIC_MAX_CELLS" in str(e.value)
    torch.cuda.synchronize()
    assert torch.isnan(bkg).all() and torch.isnan(nse).all()      # nothing was launched
    # exactly at the maximum it runs: 1024 x 1024 cells
    W = H = 8 * 1024
    bkg, nse = _grids(W, H, 8)
    argus.argus_background_map_static(W, H, bkg, nse, cell=8, n_min=1, cal=cal[:H, :W].contiguous(),
                                      mask=mask[:H, :W].contiguous())
    torch.cuda.synchronize()
    assert (bkg == 0).all() and (nse == 0).all()
