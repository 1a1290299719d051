"""das_beamform_static: the raw -> volume call for users who cannot allocate device memory -- run with -m gpu.

Why the call exists (include/das.h): das_convert + das_execute want a converted buffer from the caller, and
das_beamform_host allocates staging buffers on first use.  A real-time acquisition loop (an allocation stalls the
device: a dropped frame), a plug-in inside an application whose own pool already holds the whole GPU (cudaMalloc
fails there) or software that may not allocate after set-up can use neither.  das_beamform_static runs the same
two kernels through a 16 MiB scratch array that is built into the library image, so nobody allocates anything.

What is checked here: its volume equals the one das_convert + das_execute give for the same plan and data (the
existing path, itself compared with the CPU oracle in test_gpu_parity.py), at the fp32 gate of those tests,
on two calls in a row with DIFFERENT data -- the array is shared by all calls and keeps the last call's bytes, so
the second call would show anything stale -- and for the tiled, general and tensor-core plans; that free device
memory does not shrink across a call once the one-time address look-up of the first call is done; and that a plan
whose converted data exceeds the array is refused with DAS_ERR_SIZE before anything is enqueued.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (the first call then does the look-up) and after the others.
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

TOL_MAX = 1e-5          # the fp32 gate of tests/test_gpu_parity.py; the two paths run the same kernels


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (torch.cuda.is_available() is False)")
    return torch


def _frames(w, seeds, n_frames):
    """Distinct seeded channel data per call: the workload's echoes rescaled plus fresh noise."""
    out = []
    for s in seeds:
        rng = np.random.default_rng(s)
        shape = ((n_frames,) if n_frames > 1 else ()) + w.y.shape
        noise = (rng.normal(0, 0.05, shape) + 1j * rng.normal(0, 0.05, shape)).astype(np.complex64)
        out.append(np.ascontiguousarray((w.y * np.float32(1.0 + 0.25 * s) + noise).astype(np.complex64)))
    return out


@pytest.mark.parametrize("algo,storage,n_frames", [
    ("TILED", "FP32", 0), ("TILED", "FP16", 0), ("GENERAL", "FP32", 0), ("TC", "FP16", 8)])
def test_static_scratch_equals_convert_execute_on_two_calls(das_lib, algo, storage, n_frames):
    das, torch = das_lib, _torch()
    w = wl.config(1)
    plan = das.Plan.from_workload(w, storage=getattr(das, "STORE_" + storage), algo=getattr(das, "ALGO_" + algo),
                                  n_frames=n_frames)
    assert plan.algo == getattr(das, "ALGO_" + algo)
    assert plan.converted_bytes <= das.STATIC_SCRATCH_BYTES
    stream = torch.cuda.current_stream().cuda_stream
    raws = [torch.from_numpy(y).cuda() for y in _frames(w, (3, 4), n_frames)]
    shape = plan.grid_shape if plan.frames == 1 else (plan.frames,) + tuple(plan.grid_shape)
    outs = [torch.full(shape, float("nan"), dtype=torch.complex64, device="cuda") for _ in raws]
    refs = [das.beamform_torch(plan, raw)[0] for raw in raws]           # existing path, caller-owned buffer
    torch.cuda.synchronize()
    free = []
    for raw, out in zip(raws, outs):                                    # two calls in a row, nothing in between
        plan.beamform_static(raw.data_ptr(), out.data_ptr(), 1.0, stream)
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
    assert free[1] >= free[0], "free device memory shrank across the second call: something allocated"
    assert not torch.equal(refs[0], refs[1])                            # the two calls really differ
    for i, (out, ref) in enumerate(zip(outs, refs)):
        got, exp = out.cpu().numpy(), ref.cpu().numpy()
        assert np.isfinite(got.view(np.float32)).all(), f"call {i}: output not fully written"
        err = np.abs(got.astype(np.complex128) - exp).max() / np.abs(exp).max()
        assert err <= TOL_MAX, f"call {i}: static-scratch path differs from das_convert + das_execute by {err:.3e}"
    plan.destroy()


def test_static_scratch_refuses_what_does_not_fit(das_lib):
    das, torch = das_lib, _torch()
    m, q, k = 256, 16, 1024                                             # 256 * 16 * 1152 entries * 16 B = 75 MB
    plan = das.Plan(wl.matrix_array(16), [0] * q, [[0, 0, 1]] * q, [0.0] * q, [0.0], [0.0], [5e-3],
                    c=1540.0, fc=7.8e6, fs=15.6e6, n_samples=k, storage=das.STORE_FP32, algo=das.ALGO_GENERAL)
    assert plan.converted_bytes > das.STATIC_SCRATCH_BYTES
    raw = torch.zeros((q, m, k), dtype=torch.complex64, device="cuda")
    out = torch.full((1, 1, 1), float("nan"), dtype=torch.complex64, device="cuda")
    before = das.launch_count()
    with pytest.raises(das.DasError) as ei:
        plan.beamform_static(raw.data_ptr(), out.data_ptr())
    assert das.status_string(ei.value.status) == "DAS_ERR_SIZE"
    assert "DAS_STATIC_SCRATCH_BYTES" in das.last_error()
    assert das.launch_count() == before                                 # refused before anything was enqueued
    torch.cuda.synchronize()
    assert torch.isnan(out.real).all()
    plan.destroy()
