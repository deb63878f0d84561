"""pdrt_objective_noalloc (include/pdrt.h): the objective on the library's static device scratch, for callers that cannot
call cudaMalloc.  Checked against the existing path (pdrt_objective) through the C ABI on two calls in a row with different
inputs — the scratch is shared and keeps the last call's contents — at a size with several blocks and a ragged tail, at the
largest size the scratch serves, and one voxel slice beyond it (rejected).  The file name sorts last on purpose: the
run is `pytest -x`, and a failure here must not hide another test."""
import pytest

from paper_2512_18863_b200 import workloads as W

pytestmark = pytest.mark.gpu

MAX_VOXELS = 1 << 25          # PDRT_NOALLOC_MAX_VOXELS of include/pdrt.h
LOSS_RTOL = 1e-9              # the tolerance of tests/test_gpu_planning.py for the float64 loss


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _inputs(torch, shape, seed, n_struct=3):
    """Seeded dose and overlapping structures on the device: about half of the voxels in some structure."""
    gen = torch.Generator(device="cuda")
    gen.manual_seed(seed)
    dose = torch.rand(shape, generator=gen, device="cuda", dtype=torch.float32) * 4.0
    bits = torch.zeros(shape, dtype=torch.int32, device="cuda")
    for s in range(n_struct):
        bits |= (torch.rand(shape, generator=gen, device="cuda") < 0.25).to(torch.int32) << s
    return dose, bits


def _both(torch, eng, dose, bits, lam, presc, power, out):
    want_loss, want_g = eng.objective(dose, bits, lam, presc, power)
    loss, g = eng.objective_noalloc(dose, bits, lam, presc, power, out)
    torch.cuda.synchronize()
    assert float(loss[0]) == pytest.approx(float(want_loss[0]), rel=LOSS_RTOL)
    assert float(want_loss[0]) > 0.0
    assert torch.equal(g, want_g), "dL/dDose: same arithmetic per voxel, so bit-identical"


def test_two_calls_in_a_row_match_the_existing_path(torch):
    from paper_2512_18863_b200 import Engine
    wl = W.tiny(seed=61, nx=37, ny=29, nz=17)                 # 18 241 voxels: 5 blocks of 4096, ragged tail
    eng = Engine(wl.grid, wl.model, wl.density)
    lam, presc = [0.7, 1.9, 0.3], [2.0, 0.0, 1.0]
    shape = eng.dose_shape
    out = (torch.full((1,), -1.0, dtype=torch.float64, device="cuda"), torch.empty(shape, dtype=torch.float32, device="cuda"))
    a = _inputs(torch, shape, 1)
    b = _inputs(torch, shape, 2)
    calls = (a + (2,), b + (1,), b + (2,), a + (1,))
    kept = [torch.empty_like(out[1]) for _ in calls]          # everything the loop below needs exists before it starts
    eng.objective_noalloc(*a, lam, presc, 2, out)             # resolves the symbol address, loads the kernel
    torch.cuda.synchronize()
    scratch0, free0 = eng.get_info().scratch_bytes, torch.cuda.mem_get_info()[0]
    res = []
    for (dose, bits, power), keep in zip(calls, kept):
        loss, g = eng.objective_noalloc(dose, bits, lam, presc, power, out)
        keep.copy_(g)
        res.append((loss.item(), keep))
    torch.cuda.synchronize()
    assert eng.get_info().scratch_bytes == scratch0 and torch.cuda.mem_get_info()[0] == free0, "the calls allocate no device memory"
    for (dose, bits, power), (loss, g) in zip(calls, res):
        want_loss, want_g = eng.objective(dose, bits, lam, presc, power)
        assert loss == pytest.approx(float(want_loss[0]), rel=LOSS_RTOL) and loss > 0.0
        assert torch.equal(g, want_g)
    # back to back on one stream without a synchronise in between: stream order is enough
    out2 = (torch.empty(1, dtype=torch.float64, device="cuda"), torch.empty_like(out[1]))
    eng.objective_noalloc(*a, lam, presc, 2, out)
    eng.objective_noalloc(*b, lam, presc, 2, out2)
    torch.cuda.synchronize()
    assert float(out[0][0]) == res[0][0] and float(out2[0][0]) == res[2][0], "bit-reproducible: the summation order is fixed"


def test_second_engine_and_a_one_block_grid_share_the_scratch(torch):
    from paper_2512_18863_b200 import Engine
    small = W.tiny(seed=62, nx=9, ny=7, nz=5)                 # 315 voxels: one partly filled block
    wide = W.tiny(seed=63, nx=64, ny=64, nz=33)               # 135 168 voxels = 33 whole blocks
    e1, e2 = Engine(small.grid, small.model, small.density), Engine(wide.grid, wide.model, wide.density)
    lam, presc = [1.0, 0.5, 2.0], [1.5, 0.0, 3.0]
    for rnd in range(2):
        for eng in (e2, e1):                                  # the larger grid first: its partials stay behind in the scratch
            dose, bits = _inputs(torch, eng.dose_shape, 10 * rnd + eng.dose_shape[0])
            out = (torch.empty(1, dtype=torch.float64, device="cuda"), torch.empty(eng.dose_shape, dtype=torch.float32, device="cuda"))
            _both(torch, eng, dose, bits, lam, presc, 1 + rnd, out)


def test_largest_grid_is_served_and_one_slice_more_is_rejected(torch):
    from paper_2512_18863_b200 import Engine, PdrtError
    lam, presc = [0.25, 1.0, 4.0], [0.0, 2.0, 1.0]
    wl = W.tiny(seed=64, nx=512, ny=512, nz=128, spacing=1.0)   # exactly PDRT_NOALLOC_MAX_VOXELS: 8192 blocks
    assert wl.grid["nx"] * wl.grid["ny"] * wl.grid["nz"] == MAX_VOXELS
    eng = Engine(wl.grid, wl.model, wl.density)
    dose, bits = _inputs(torch, eng.dose_shape, 5)
    out = (torch.empty(1, dtype=torch.float64, device="cuda"), torch.empty(eng.dose_shape, dtype=torch.float32, device="cuda"))
    for power in (2, 1):
        _both(torch, eng, dose, bits, lam, presc, power, out)
    del eng, dose, bits, out
    wl = W.tiny(seed=65, nx=512, ny=512, nz=129, spacing=1.0)
    eng = Engine(wl.grid, wl.model, wl.density)
    dose, bits = _inputs(torch, eng.dose_shape, 6)
    out = (torch.full((1,), -7.0, dtype=torch.float64, device="cuda"), torch.zeros(eng.dose_shape, dtype=torch.float32, device="cuda"))
    with pytest.raises(PdrtError) as err:
        eng.objective_noalloc(dose, bits, lam, presc, 2, out)
    assert err.value.code == -1 and str(MAX_VOXELS) in str(err.value) and str(512 * 512 * 129) in str(err.value)
    torch.cuda.synchronize()
    assert float(out[0][0]) == -7.0 and not bool(out[1].any()), "a rejected call launches nothing"
    loss, _ = eng.objective(dose, bits, lam, presc, 2)        # the existing path still serves that grid
    assert float(loss[0]) > 0.0
