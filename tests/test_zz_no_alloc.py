"""flare_virial_static: the virial read-out for callers that may not allocate device memory.

Some programs that embed this library cannot call cudaMalloc once they are running: their own pool already holds
the GPU's memory, an allocation would stall every stream of the device, or their rules forbid it (a pressure
coupling or monitor that runs every MD step).  For them `flare_virial_static` keeps its partial sums in a fixed
array inside the library instead of in caller-provided scratch, and writes the 3 x 3 result to a device buffer the
caller owns.  These tests check, through the C ABI on a GPU, that it gives what the existing path
(`flare_get_virial`, scratch in the bound workspace) gives, at the tolerance the virial parity test uses
(1e-10 of the largest component), on calls that follow one another and therefore share that array: first a system
that fills several rows of it (with a ragged last tile), then a smaller one that leaves the first call's rows
behind it, then the first again.  Also: repeated calls are bit-identical, the calls take no device memory, and a
context above the stated limit is refused with a message that names the limit.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process and after the rest of the suite (nothing here depends on what
ran before: the array needs no initial contents)."""
import numpy as np
import pytest

from paper_2204_12573_b200 import workloads as w

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch

    return torch


@pytest.fixture(scope="module")
def flare():
    from paper_2204_12573_b200 import flare as fl

    fl.load_library()
    return fl


def _evaluated(torch, flare, s):
    ctx = flare.from_system(s).bind(s.n_atoms)
    pos = torch.as_tensor(s.pos, dtype=torch.float64, device="cuda")
    types = torch.as_tensor(s.types, dtype=torch.int32, device="cuda")
    ctx.compute(pos, types, s.box, s.pbc, variances=False)
    torch.cuda.synchronize()
    return ctx


def _static(torch, ctx):
    out = torch.full((9,), float("nan"), dtype=torch.float64, device="cuda")  # the caller's output buffer
    ctx.virial_static(out)
    torch.cuda.synchronize()
    return out.cpu().numpy().reshape(3, 3)


def test_static_virial_matches_existing_path_on_consecutive_calls(torch, flare):
    big = w.tile_like_c3(30, 15, n_max=4, l_max=2)   # several 2048-atom tiles and a ragged tail
    small = w.config2()                              # 1264 atoms: one tile; rows above it keep the big call's sums
    assert big.n_atoms > 2 * 2048 and big.n_atoms % 2048 != 0 and small.n_atoms < 2048
    ctx_big, ctx_small = _evaluated(torch, flare, big), _evaluated(torch, flare, small)
    ref_big, ref_small = ctx_big.virial(), ctx_small.virial()   # existing path: scratch in the bound workspace
    for ref in (ref_big, ref_small):
        assert np.abs(ref).max() > 1e-3

    # calls in a row, all through the one shared array
    got = [_static(torch, ctx_big), _static(torch, ctx_small), _static(torch, ctx_big), _static(torch, ctx_small)]
    for g, ref in zip(got, (ref_big, ref_small, ref_big, ref_small)):
        assert np.all(np.isfinite(g))
        assert np.abs(g - ref).max() <= 1e-10 * np.abs(ref).max()
    # fixed summation order: a repeat is bit-identical, whatever ran in between
    assert np.array_equal(got[0], got[2]) and np.array_equal(got[1], got[3])
    # the existing path is unaffected by the new one
    assert np.array_equal(ctx_big.virial(), ref_big) and np.array_equal(ctx_small.virial(), ref_small)


def test_static_virial_takes_no_device_memory(torch, flare):
    s = w.config1()
    ctx = _evaluated(torch, flare, s)
    ref = ctx.virial()
    out = torch.empty(9, dtype=torch.float64, device="cuda")
    ctx.virial_static(out)          # first use: address lookup, kernels loaded
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        ctx.virial_static(out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0           # device-wide figure: a cudaMalloc inside the call would show here
    assert np.abs(out.cpu().numpy().reshape(3, 3) - ref).max() <= 1e-10 * np.abs(ref).max()


def test_static_virial_argument_errors(torch, flare):
    s = w.config1()
    ctx = flare.from_system(s).bind(s.n_atoms)
    out = torch.zeros(9, dtype=torch.float64, device="cuda")
    with pytest.raises(flare.FlareError) as ei:
        ctx.virial_static(out)      # nothing evaluated yet
    assert ei.value.code == -9
    with pytest.raises(ValueError):
        ctx.virial_static(torch.zeros(9, dtype=torch.float32, device="cuda"))

    # one atom above the limit: refused before anything is launched (a small-footprint binding, never evaluated)
    too_many = flare.VIRIAL_STATIC_MAX_ATOMS + 1
    lean = flare.from_system(s, max_neighbors=4, chunk_atoms=256, skin=0.0)
    assert lean.workspace_bytes(too_many) < 16 << 30
    lean.bind(too_many)
    with pytest.raises(flare.FlareError) as ei:
        lean.virial_static(out)
    assert ei.value.code == -1 and str(flare.VIRIAL_STATIC_MAX_ATOMS) in str(ei.value)
    assert "flare_get_virial" in str(ei.value)
    assert np.array_equal(out.cpu().numpy(), np.zeros(9))   # the output was not touched
