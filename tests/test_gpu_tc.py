"""Parity of the frame-batch tensor-core path (DAS_ALGO_TC, n_frames = B) against the CPU oracle.

Every frame of a batch must equal what the oracle computes for that frame alone (the paper's
x_bn): the batch only amortises the interpolation weights.
The path stores samples AND the generated weights in FP16 and accumulates in FP32, so the gate is
the north_star's fp16-storage gate: max error <= 2e-3 of max|oracle|, relative L2 <= 1e-3, the
oracle run on the original float32 inputs.
"""
import functools

import numpy as np
import pytest

import workloads as wl
from test_gpu_parity import TOL_FP16_L2, TOL_FP16_MAX, _cfg, _sample_voxels, _subgrid, _torch, errors

pytestmark = pytest.mark.gpu


def make_batch(y, n_frames, seed, sigma=0.01):
    """B distinct frames from one seeded record: frame 0 is y; frame b > 0 is y scaled by an exact
    power of two plus an independent seeded noise realisation (total complex sigma, reading A13)."""
    rng = np.random.default_rng(seed)
    out = np.empty((n_frames,) + y.shape, np.complex64)
    out[0] = y
    sd = sigma / np.sqrt(2.0)
    for b in range(1, n_frames):
        n = (rng.normal(0.0, sd, y.shape) + 1j * rng.normal(0.0, sd, y.shape)).astype(np.complex64)
        out[b] = y * np.float32(2.0 ** (-(b % 3))) + n
    return out


def gpu_batch(das, w, yb, *, algo=None, expect_algo=None):
    torch = _torch()
    algo = das.ALGO_TC if algo is None else algo
    plan = das.Plan.from_workload(w, storage=das.STORE_FP16, algo=algo, n_frames=len(yb))
    assert plan.frames == len(yb)
    assert plan.algo == (das.ALGO_TC if expect_algo is None else expect_algo)
    assert plan.raw_bytes == yb.nbytes
    raw = torch.from_numpy(np.ascontiguousarray(yb)).cuda()
    out = torch.full((len(yb),) + tuple(w.grid_shape), 7.0 - 3.0j, dtype=torch.complex64, device="cuda")
    das.beamform_torch(plan, raw, out=out)
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    plan.destroy()
    return res


def check_frames(got, w, yb, frames=None, label=""):
    import oracle
    worst = (0.0, 0.0)
    for b in (range(len(yb)) if frames is None else frames):
        ref = oracle.das(w, y=yb[b])
        emax, el2 = errors(got[b], ref)
        assert emax <= TOL_FP16_MAX, f"{label} frame {b}: max error {emax:.3e} > {TOL_FP16_MAX}"
        assert el2 <= TOL_FP16_L2, f"{label} frame {b}: relative L2 error {el2:.3e} > {TOL_FP16_L2}"
        worst = (max(worst[0], emax), max(worst[1], el2))
    return worst


# ------------------------------------------------------------------ full-volume parity

def test_tc_config1_tiny_batch8(das_lib):
    w = _cfg(1)
    yb = make_batch(w.y, 8, 101)
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, label="config1 B=8")


def test_tc_config2_small_batch16(das_lib):
    """Config 2 full volume (64^3, 5 steered plane waves), 16 frames per call (MMA N = 32)."""
    w = _cfg(2)
    yb = make_batch(w.y, 16, 102)
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, frames=[0, 1, 7, 15], label="config2 B=16")


@pytest.mark.parametrize("sl", [(slice(5, 18), slice(10, 17), slice(3, 22)), (slice(31, 32), slice(0, 1), slice(63, 64)),
                                (slice(2, 5), slice(40, 41), slice(0, 37)), (slice(40, 59), slice(1, 18), slice(30, 35))])
def test_tc_ragged_grids(das_lib, sl):
    """Grids that are not multiples of the 16 x 8 x 3 voxel tile: 13x7x19, 1x1x1, 3x1x37, 19x17x5."""
    w = _subgrid(2, *sl)
    yb = make_batch(w.y, 8, 103)
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, frames=[0, 3, 7], label=f"sub-grid {w.grid_shape}")


def test_tc_two_chunks_of_64(das_lib):
    """B = 128 runs as two chunks of 64 frames (MMA N = 128): every frame lands in its own slot."""
    w = _subgrid(1, slice(6, 26), slice(10, 21), slice(4, 11))           # 20 x 11 x 7
    yb = make_batch(w.y, 128, 104)
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, frames=[0, 1, 63, 64, 65, 100, 127], label="B=128")


def test_tc_out_of_range_samples_dropped(das_lib):
    """t_start pushed so that part of the grid maps before sample 0 and part beyond K-2 (A6)."""
    import oracle
    base = _subgrid(2, slice(28, 34), slice(30, 35), slice(8, 56))
    y = np.ascontiguousarray(base.y[:, :, 40:160])
    w = wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs,
                  fs=base.fs, n_samples=120, t_start=5.0e-6, f_number=1.0, y=y)
    yb = make_batch(y, 8, 105)
    cnt = oracle.das(w, want_count=True)["count"]
    assert cnt.min() == 0 and cnt.max() > 0
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, frames=[0, 5], label="out-of-range")
    assert np.all(got[:, cnt == 0] == 0)


def test_tc_no_apodization(das_lib):
    base = _subgrid(1, slice(10, 18), slice(12, 18), slice(5, 15))
    w = wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs,
                  fs=base.fs, n_samples=base.n_samples, f_number=0.0, y=base.y)
    yb = make_batch(w.y, 8, 106)
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, frames=[0, 6], label="f_number=0")


def test_tc_mixed_transmits_offset_array_nonzero_tstart(das_lib):
    """Plane + diverging transmits in one plan, array plane at z != 0, t_start != 0, fc != fs/2."""
    rng = np.random.default_rng(21)
    elem = wl.matrix_array(6)
    elem[:, 2] = np.float32(-0.4e-3)
    elem[:, 0] += np.float32(0.1e-3)
    a = np.radians(7.0)
    xs, ys, zs = wl.axis(-1e-3, 1.2e-3, 23), wl.axis(-0.8e-3, 0.9e-3, 19), wl.axis(1.5e-3, 5e-3, 23)
    pos = np.stack([rng.uniform(-0.8e-3, 0.8e-3, 4), rng.uniform(-0.6e-3, 0.6e-3, 4), rng.uniform(2e-3, 4.5e-3, 4)], 1)
    w = wl.custom(elem, [wl.TX_PLANE, wl.TX_DIVERGING, wl.TX_PLANE],
                  [[np.sin(a), 0, np.cos(a)], [0.7e-3, -0.2e-3, -5e-3], [0, 0, 1]], [2e-7, -3.1e-6, 0.0],
                  xs, ys, zs, fs=20e6, fc=6.25e6, n_samples=300, t_start=1.0e-6, f_number=1.3,
                  scat_pos=pos, scat_amp=[1, 0.5, 0.8, 0.3], noise_sigma=0.01, seed=5)
    yb = make_batch(w.y, 24, 107)
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, frames=[0, 11, 23], label="mixed transmits B=24")


# ------------------------------------------------------------------ headline size, B = 64, sampled voxels

@functools.lru_cache(maxsize=None)
def _streaming_bases(n):
    return [f.y for f in wl.streaming_frames(n)]


def test_tc_headline_full_size_batch64_sampled(das_lib):
    """Config 5 shape: 64 frames of the headline layout in ONE das_execute (the launch
    configuration bench.py times).  The 64 slots hold 4 seeded config-5 frames (drifting
    scatterers over +20 dB clutter, reading A15), each repeated under an exact power-of-two scale,
    so the oracle evaluates 4 frames on a voxel sample and every one of the 64 slots is checked."""
    import oracle
    das, torch = das_lib, _torch()
    B = 64
    base = wl.config(5, generate_data=False)
    ys = _streaming_bases(4)
    vox = _sample_voxels(base, n_random=1200)
    refs = [oracle.das(base, y=y, voxels=vox) for y in ys]
    plan = das.Plan.from_workload(base, storage=das.STORE_FP16, algo=das.ALGO_AUTO, n_frames=B)
    assert plan.algo == das.ALGO_TC
    raw = torch.empty((B,) + ys[0].shape, dtype=torch.complex64, device="cuda")
    scale = [2.0 ** (-((b // 4) % 4)) for b in range(B)]
    for b in range(B):
        raw[b] = torch.from_numpy(ys[b % 4]).cuda() * scale[b]
    out, _ = das.beamform_torch(plan, raw)
    torch.cuda.synchronize()
    idx = torch.from_numpy(vox).cuda()
    got = out.reshape(B, -1)[:, idx].cpu().numpy()
    plan.destroy()
    for b in range(B):
        emax, el2 = errors(got[b], refs[b % 4] * scale[b])
        assert emax <= TOL_FP16_MAX and el2 <= TOL_FP16_L2, f"slot {b}: max {emax:.3e}, L2 {el2:.3e}"


def test_tc_headline_geometry_reduced_grid_full(das_lib):
    """Headline array, 16 diverging-wave transmits and native voxel spacing on a 40 x 24 x 9 block of
    the grid (several tiles, ragged in every axis), every voxel compared: the 8-transmits-per-stage
    sample ring and the 16-transmit generator loop at full width."""
    w = _subgrid(3, slice(30, 70), slice(50, 74), slice(60, 69))
    yb = make_batch(w.y, 8, 110)
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, frames=[0, 5], label="config3 sub-grid B=8")


def test_tc_headline_geometry_record_edges(das_lib):
    """The same with a record cut so short that the deep voxels run off its end and t_start moved so
    that the shallow ones start before sample 0: the per-tile edge path (reading A6) with 16 transmits."""
    import oracle
    base = _subgrid(3, slice(56, 72), slice(60, 68), slice(0, 128, 5))
    y = np.ascontiguousarray(base.y[:, :, 60:260])
    w = wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs,
                  fs=base.fs, n_samples=200, t_start=60.0 / base.fs, f_number=1.0, y=y)
    cnt = oracle.das(w, want_count=True)["count"]
    assert cnt.min() < cnt.max() and (cnt == 0).any()
    yb = make_batch(y, 8, 111)
    got = gpu_batch(das_lib, w, yb)
    check_frames(got, w, yb, frames=[0, 7], label="config3 record edges")


# ------------------------------------------------------------------ dispatch rules

def test_tc_refusals_and_fallback(das_lib):
    das = das_lib
    w = _subgrid(1, slice(3, 12), slice(20, 28), slice(9, 16))          # 9 x 8 x 7 at native spacing
    for kw in (dict(n_frames=12), dict(n_frames=4), dict(n_frames=72), dict(n_frames=8, storage=das.STORE_FP32)):
        args = dict(storage=das.STORE_FP16, algo=das.ALGO_TC)
        args.update(kw)
        with pytest.raises(das.DasError) as ei:
            das.Plan.from_workload(w, **args)
        assert ei.value.status == das.ERR_UNSUPPORTED
    # AUTO with a frame count the tensor-core path does not take: frame by frame, still correct
    yb = make_batch(w.y, 3, 108)
    got = gpu_batch(das, w, yb, algo=das.ALGO_AUTO, expect_algo=das.ALGO_TILED)
    check_frames(got, w, yb, label="AUTO B=3")


def test_tc_beamform_host_batch(das_lib):
    das, torch = das_lib, _torch()
    w = _cfg(1, (17, 9, 6))
    yb = make_batch(w.y, 8, 109)
    plan = das.Plan.from_workload(w, storage=das.STORE_FP16, algo=das.ALGO_TC, n_frames=8)
    h_raw = torch.from_numpy(yb).pin_memory()
    h_out = torch.empty((8,) + tuple(w.grid_shape), dtype=torch.complex64).pin_memory()
    plan.beamform_host(h_raw.data_ptr(), h_out.data_ptr())
    dev, _ = das.beamform_torch(plan, torch.from_numpy(yb).cuda())
    torch.cuda.synchronize()
    np.testing.assert_array_equal(h_out.numpy(), dev.cpu().numpy())
    check_frames(h_out.numpy(), w, yb, frames=[0, 7], label="beamform_host B=8")
    plan.destroy()


def test_tc_beamform_host_pipelined(das_lib):
    """das_beamform_host_begin / _wait (das.h): two calls in flight, three batches through two host output
    buffers; every result equals the device-resident path bit for bit, the protocol errors are reported."""
    das, torch = das_lib, _torch()
    w = _cfg(1, (17, 9, 6))
    batches = [make_batch(w.y, 8, 120 + i) for i in range(3)]
    plan = das.Plan.from_workload(w, storage=das.STORE_FP16, algo=das.ALGO_TC, n_frames=8)
    want = []
    for yb in batches:
        dev, _ = das.beamform_torch(plan, torch.from_numpy(yb).cuda())
        torch.cuda.synchronize()
        want.append(dev.cpu().numpy())
    h_raw = [torch.from_numpy(yb).pin_memory() for yb in batches]
    h_out = [torch.zeros((8,) + tuple(w.grid_shape), dtype=torch.complex64).pin_memory() for _ in range(3)]
    with pytest.raises(das.DasError):
        plan.beamform_host_wait()                                # nothing outstanding
    plan.beamform_host_begin(h_raw[0].data_ptr(), h_out[0].data_ptr())
    plan.beamform_host_begin(h_raw[1].data_ptr(), h_out[1].data_ptr())
    with pytest.raises(das.DasError):
        plan.beamform_host_begin(h_raw[2].data_ptr(), h_out[2].data_ptr())   # a third call in flight
    with pytest.raises(das.DasError):
        plan.beamform_host(h_raw[2].data_ptr(), h_out[2].data_ptr())         # the blocking call while calls are outstanding
    plan.beamform_host_wait()
    np.testing.assert_array_equal(h_out[0].numpy(), want[0])
    plan.beamform_host_begin(h_raw[2].data_ptr(), h_out[2].data_ptr())
    plan.beamform_host_wait()
    np.testing.assert_array_equal(h_out[1].numpy(), want[1])
    plan.beamform_host_wait()
    np.testing.assert_array_equal(h_out[2].numpy(), want[2])
    plan.destroy()


@pytest.mark.timeout(180)
def test_tc_repeated_launches_deterministic(das_lib):
    """Soak: the warp roles of tc_kernel hand data over through five mbarrier rings, tensor memory and (quad pacing)
    global progress words.  500 launches back to back on config 2 with 16 frames must neither hang nor change a bit
    (a voxel's terms are accumulated in a fixed order, so the kernel is deterministic)."""
    torch = _torch()
    das = das_lib
    w = wl.config(2, generate_data=False)
    plan = das.Plan.from_workload(w, storage=das.STORE_FP16, algo=das.ALGO_TC, n_frames=16)
    g = torch.Generator(device="cuda").manual_seed(5)
    raw = torch.view_as_complex(torch.randn((16, w.n_tx, w.n_elem, w.n_samples, 2), device="cuda", generator=g) * 0.1)
    conv = torch.empty(plan.converted_bytes, dtype=torch.uint8, device="cuda")
    outs = [torch.empty(plan.output_bytes // 4, dtype=torch.float32, device="cuda") for _ in range(2)]
    s = torch.cuda.current_stream().cuda_stream
    plan.convert(raw.data_ptr(), conv.data_ptr(), 1.0, s)
    plan.execute(conv.data_ptr(), outs[0].data_ptr(), s)
    for _ in range(500):
        plan.execute(conv.data_ptr(), outs[1].data_ptr(), s)
    torch.cuda.synchronize()
    assert torch.equal(outs[0], outs[1])
    plan.destroy()


def test_tc_quad_pacing_does_not_change_results(das_lib):
    """The producers' quad pacing only delays TMA copies: with it switched off (debug_tc_pace = -1 in
    the plan descriptor) the output must be bit-identical.  Config 2 geometry, ragged sub-grid (rim quads are filled up with
    empty tiles), 16 frames."""
    torch = _torch()
    das = das_lib
    w = _subgrid(2, slice(3, 56), slice(0, 37), slice(5, 60))
    g = torch.Generator(device="cuda").manual_seed(11)
    raw = torch.view_as_complex(torch.randn((16, w.n_tx, w.n_elem, w.n_samples, 2), device="cuda", generator=g) * 0.1)
    outs = []
    for pace in (-1, 0, 4):                           # off, the default lead (16), a short lead
        plan = das.Plan.from_workload(w, storage=das.STORE_FP16, algo=das.ALGO_TC, n_frames=16, debug_tc_pace=pace)
        out, _ = das.beamform_torch(plan, raw)
        torch.cuda.synchronize()
        outs.append(out.clone())
        plan.destroy()
    assert torch.equal(torch.view_as_real(outs[0]), torch.view_as_real(outs[1]))
    assert torch.equal(torch.view_as_real(outs[0]), torch.view_as_real(outs[2]))


def test_tc_pacing_gives_up_on_a_partner_that_is_not_resident(das_lib):
    """ADVICE (round 2): the quad pacing must not turn a missing partner into seconds.  A one-thread spinning kernel
    on a side stream holds one SM's registers, so one of the persistent CTAs (512 threads x 128 registers = the whole
    register file) cannot start until another CTA has finished: its three partners see a progress word that never
    moves.  Each paced receiver used to wait the full 4 000 polls (about 1 s in total on this problem); with the
    shrinking budget (das_tc.cu, pace_budget) the launch costs the serialised CTA's work plus a few ms.  The
    volume stays bit-identical, as the pacing is advisory."""
    import time
    torch = _torch()
    das = das_lib
    w = _cfg(2)                                       # 64^3 voxels: 704 tiles, one CTA on every SM
    g = torch.Generator(device="cuda").manual_seed(5)
    raw = torch.view_as_complex(torch.randn((8, w.n_tx, w.n_elem, w.n_samples, 2), device="cuda", generator=g) * 0.1)
    plan = das.Plan.from_workload(w, storage=das.STORE_FP16, algo=das.ALGO_TC, n_frames=8)
    out, conv = das.beamform_torch(plan, raw)
    torch.cuda.synchronize()
    ref = out.clone()
    main = torch.cuda.current_stream()

    def timed():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        out.fill_(0)
        e0.record(main)
        plan.execute(conv.data_ptr(), out.data_ptr(), main.cuda_stream)
        e1.record(main)
        e1.synchronize()
        return e0.elapsed_time(e1)

    t_alone = min(timed() for _ in range(3))
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        torch.cuda._sleep(int(6e8))                   # about 0.3 s on one SM, far longer than the launch
    time.sleep(0.02)                                  # let it start before the batch kernel is enqueued
    t_hog = timed()
    busy = not side.query()                           # the hog outlived the launch it was meant to disturb
    side.synchronize()
    print(f"tc_kernel alone {t_alone:.2f} ms, with one SM taken {t_hog:.2f} ms (hog still running: {busy})")
    assert torch.equal(torch.view_as_real(out), torch.view_as_real(ref))
    assert t_hog <= 3.0 * t_alone + 25.0, (t_alone, t_hog)
    plan.destroy()
