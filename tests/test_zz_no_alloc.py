"""cos_det_eval_static: the determinant route for callers that are not allowed to allocate device memory.

Who that is: a Monte-Carlo loop that cannot afford the device-wide stall of a cudaMalloc / cudaFree in steady state, a
plug-in inside a program whose own memory pool has taken all of HBM (so a further cudaMalloc fails), a service with a
latency bound on its request path.  For them the library carries its own scratch -- a 16 MiB array compiled into
libcos_b200.so -- and the entry point promises to call no allocator (include/cos.h).

What is checked here, through the C-ABI on a real GPU:
  * two calls in a row (the second on a different, smaller problem, so the scratch still holds the first call's data)
    return exactly what the existing cos_det_eval returns with a freshly allocated work buffer -- same kernels and
    summation order, so the comparison is bit-for-bit, which is tighter than the 1e-10 * R the parity tests allow;
  * the first problem again after the second: stale scratch contents change nothing;
  * the device's free memory does not shrink across the calls;
  * a problem beyond COS_DET_STATIC_SCRATCH_BYTES is refused with COS_EUNSUPPORTED and leaves the output untouched;
    an empty batch is a no-op.

This file is named so that pytest collects it last: under `pytest -x` a failure here cannot hide another test.  It builds
its own fixture and inputs, so it passes alone in a fresh process (where its first call performs the one-time address
look-up) as well as after the rest of the suite.
"""
import numpy as np
import pytest

from cos_workloads import random_matrices

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cos():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    torch.cuda.set_device(0)
    import paper_2507_12349_b200 as cos_mod
    cos_mod.load_library()
    return cos_mod


def _problem(seed, n, nf, B):
    import torch
    G = random_matrices(seed, nf, n, B, scale=0.8)
    Gd = torch.from_numpy(np.ascontiguousarray(G.reshape(-1, B))).cuda()
    sig = [0.5, -1.0 / 3.0, 0.25][:nf]
    return Gd, sig


def _existing_path(cos, Gd, n, nf, sig, prec, B):
    """cos_det_eval with a caller-allocated work buffer: the path that is already under parity test."""
    import torch
    out = torch.full(((1 << n) - 1, B), float("nan"), dtype=torch.float64, device="cuda")
    nbytes = cos.cos_det_workspace_bytes(n, nf, prec, B)
    work = torch.empty((nbytes + 7) // 8, dtype=torch.float64, device="cuda")
    cos.cos_det_eval(n, nf, nf, sig, prec, Gd, B, out, work)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_static_scratch_matches_existing_path_on_consecutive_calls(cos):
    import torch
    # (n, flavours, precision, batch): a three-flavour fp64 problem of 70 configurations (two full tiles and a ragged
    # one), then a smaller two-flavour double-double one that reuses the same scratch bytes with another layout
    first, second = (6, 3, cos.COS_DET_FP64, 70), (4, 2, cos.COS_DET_DD, 33)
    cases = []
    for seed, (n, nf, prec, B) in zip((4101, 4102), (first, second)):
        assert 0 < cos.cos_det_workspace_bytes(n, nf, prec, B) <= cos.COS_DET_STATIC_SCRATCH_BYTES
        Gd, sig = _problem(seed, n, nf, B)
        ref = _existing_path(cos, Gd, n, nf, sig, prec, B)
        assert np.all(np.isfinite(ref)) and np.any(ref != 0.0)
        out = torch.full(((1 << n) - 1, B), float("nan"), dtype=torch.float64, device="cuda")
        cases.append((n, nf, prec, B, Gd, sig, ref, out))

    # one-time set-up happens inside the first call on this device; do it before looking at the free memory
    n, nf, prec, B, Gd, sig, ref, out = cases[0]
    cos.cos_det_eval_static(n, nf, nf, sig, prec, Gd, B, out)
    torch.cuda.synchronize()
    out.fill_(float("nan"))
    torch.cuda.synchronize()

    free_before, _ = torch.cuda.mem_get_info()
    for n, nf, prec, B, Gd, sig, ref, out in cases:                 # two calls in a row, same stream, no sync between
        cos.cos_det_eval_static(n, nf, nf, sig, prec, Gd, B, out)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, "the no-allocation entry point took device memory"

    for n, nf, prec, B, Gd, sig, ref, out in cases:
        got = out.cpu().numpy()
        assert np.array_equal(got, ref), ("static scratch vs cos_det_eval", n, nf, prec, np.abs(got - ref).max())

    # the first problem once more, now on top of the second call's leftovers
    n, nf, prec, B, Gd, sig, ref, out = cases[0]
    out.fill_(float("nan"))
    cos.cos_det_eval_static(n, nf, nf, sig, prec, Gd, B, out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)


def test_static_scratch_limit_and_empty_batch(cos):
    import torch
    n, nf, prec = 10, 3, cos.COS_DET_FP64
    B = 410                                                         # 409 is the last batch that fits (include/cos.h)
    assert cos.cos_det_workspace_bytes(n, nf, prec, B - 1) <= cos.COS_DET_STATIC_SCRATCH_BYTES
    assert cos.cos_det_workspace_bytes(n, nf, prec, B) > cos.COS_DET_STATIC_SCRATCH_BYTES
    Gd = torch.zeros(nf * n * n, B, dtype=torch.float64, device="cuda")
    out = torch.full(((1 << n) - 1, B), float("nan"), dtype=torch.float64, device="cuda")
    with pytest.raises(cos.CosError) as ei:
        cos.cos_det_eval_static(n, nf, nf, None, prec, Gd, B, out)
    assert ei.value.code == cos.COS_EUNSUPPORTED
    msg = str(ei.value)
    assert str(cos.COS_DET_STATIC_SCRATCH_BYTES) in msg and str(cos.cos_det_workspace_bytes(n, nf, prec, B)) in msg
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all()), "a refused call must not launch anything"
    # argument errors are cos_det_eval's own
    with pytest.raises(cos.CosError) as ei:
        cos.cos_det_eval_static(4, 5, 5, None, prec, Gd, 8, out)
    assert ei.value.code == cos.COS_EUNSUPPORTED
    cos.cos_det_eval_static(4, 3, 3, None, prec, Gd, 0, out)        # empty batch: nothing to do, no error
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all())
