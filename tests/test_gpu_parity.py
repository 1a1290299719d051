"""Parity of the CUDA path (through the C ABI) against the CPU oracle -- run with -m gpu.

Gates (BASELINE.json north_star):
    fp32 storage:  max|GPU - oracle| / max|oracle| <= 1e-5
    fp16 storage:  the same ratio <= 2e-3  and  ||GPU - oracle||_2 / ||oracle||_2 <= 1e-3,
                   the oracle run on the ORIGINAL float32 inputs
das_convert is byte work and is checked bit-exactly against numpy's casts.
"""
import functools

import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

TOL_FP32_MAX = 1e-5
TOL_FP16_MAX = 2e-3
TOL_FP16_L2 = 1e-3


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (torch.cuda.is_available() is False)")
    return torch


def gpu_das(das, w, storage, algo, *, y=None, return_conv=False):
    torch = _torch()
    y = w.y if y is None else y
    plan = das.Plan.from_workload(w, storage=storage, algo=algo)
    raw = torch.from_numpy(np.ascontiguousarray(y)).cuda()
    out, conv = das.beamform_torch(plan, raw)
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    used = plan.algo
    conv_np = conv.cpu().numpy() if return_conv else None
    plan.destroy()
    return (res, used, conv_np) if return_conv else (res, used)


def errors(gpu, ref):
    d = gpu.astype(np.complex128 if np.iscomplexobj(ref) else np.float64) - ref
    return np.abs(d).max() / np.abs(ref).max(), np.linalg.norm(d.ravel()) / np.linalg.norm(ref.ravel())


def check(gpu, ref, storage, das, label=""):
    emax, el2 = errors(gpu, ref)
    if storage == das.STORE_FP32:
        assert emax <= TOL_FP32_MAX, f"{label}: fp32 max error {emax:.3e} > {TOL_FP32_MAX}"
    else:
        assert emax <= TOL_FP16_MAX, f"{label}: fp16 max error {emax:.3e} > {TOL_FP16_MAX}"
        assert el2 <= TOL_FP16_L2, f"{label}: fp16 relative L2 error {el2:.3e} > {TOL_FP16_L2}"
    return emax, el2


def algos(das):
    return [das.ALGO_GENERAL, das.ALGO_TILED]


@functools.lru_cache(maxsize=None)
def _cfg(number, grid=None):
    return wl.config(number, grid=grid)


@functools.lru_cache(maxsize=None)
def _oracle_full(number, grid=None):
    import oracle
    return oracle.das(_cfg(number, grid))


# ------------------------------------------------------------------ das_convert (bit-exact)

PAD_LEFT = 64      # das_internal.cuh: kPadLeft / kPadRight


def expected_table(y, kind, storage, scale=1.0):
    """The device layout das_convert must write (include/das.h, das_internal.cuh), built with
    numpy float32 arithmetic: conv[m][q][i] = (mid_k, slope_k), k = i - 64,
    mid = y_k/2 + y_k+1/2, slope = y_k+1 - y_k for 0 <= k <= K-2, zero elsewhere; then the
    round-to-nearest-even cast to the storage precision."""
    q, m, k = y.shape
    comp = 2 if kind == wl.DATA_IQ else 1
    kp = PAD_LEFT + ((k + 7) // 8) * 8 + 64
    yf = (y.view(np.float32).reshape(q, m, k, comp) * np.float32(scale)).astype(np.float32)
    a, b = yf[:, :, :-1], yf[:, :, 1:]
    with np.errstate(over="ignore", invalid="ignore"):
        mid = (a * np.float32(0.5) + b * np.float32(0.5)).astype(np.float32)
        slope = (b - a).astype(np.float32)
        dt = np.float16 if storage == 1 else np.float32
        tab = np.zeros((m, q, kp, 2, comp), dt)          # [.., (mid|slope), component]
        tab[:, :, PAD_LEFT:PAD_LEFT + k - 1, 0] = np.transpose(mid, (1, 0, 2, 3)).astype(dt)
        tab[:, :, PAD_LEFT:PAD_LEFT + k - 1, 1] = np.transpose(slope, (1, 0, 2, 3)).astype(dt)
    return tab


@pytest.mark.parametrize("kind", [wl.DATA_IQ, wl.DATA_RF])
@pytest.mark.parametrize("storage", [0, 1])
def test_convert_bit_exact(das_lib, kind, storage):
    das = das_lib
    rng = np.random.default_rng(1)
    q, m, k = 3, 5, 77                                  # ragged: K not a multiple of 4 or 8
    if kind == wl.DATA_IQ:
        y = (rng.normal(size=(q, m, k)) + 1j * rng.normal(size=(q, m, k))).astype(np.complex64)
        y[0, 0, :4] = [1e-7 + 7e4j, -65520.0 + 6e-8j, 65519.0 - 0.0j, 3.0e-5 + 1j]   # subnormal / overflow edge
    else:
        y = rng.normal(size=(q, m, k)).astype(np.float32)
        y[0, 0, :4] = [1e-7, -65520.0, 65519.0, 3.0e-5]
    w = wl.custom(wl.matrix_array(3)[:m], [0, 0, 1], [[0, 0, 1]] * 3, [0.0] * 3, [0.0], [0.0], [2e-3],
                  fs=15.6e6, n_samples=k, data_kind=kind, y=y)
    _, _, conv = gpu_das(das, w, storage, das.ALGO_GENERAL, return_conv=True)
    exp = expected_table(y, kind, storage)
    dt, it = (np.float16, np.uint16) if storage == das.STORE_FP16 else (np.float32, np.uint32)
    got = conv.view(dt).reshape(exp.shape)
    assert conv.size == exp.nbytes
    np.testing.assert_array_equal(got.view(it), exp.view(it))


def test_convert_scale(das_lib):
    das, torch = das_lib, _torch()
    w = _cfg(1, (4, 4, 4))
    plan = das.Plan.from_workload(w, storage=das.STORE_FP16, algo=das.ALGO_GENERAL)
    raw = torch.from_numpy(w.y).cuda()
    conv = torch.zeros(plan.converted_bytes, dtype=torch.uint8, device="cuda")
    plan.convert(raw.data_ptr(), conv.data_ptr(), 0.5)
    torch.cuda.synchronize()
    exp = expected_table(w.y, wl.DATA_IQ, 1, scale=0.5)
    got = conv.cpu().numpy().view(np.float16).reshape(exp.shape)
    np.testing.assert_array_equal(got.view(np.uint16), exp.view(np.uint16))
    plan.destroy()


# ------------------------------------------------------------------ full-volume parity

@pytest.mark.parametrize("storage", [0, 1])
@pytest.mark.parametrize("algo", [1, 2])
def test_config1_tiny_full(das_lib, storage, algo):
    w, ref = _cfg(1), _oracle_full(1)
    out, used = gpu_das(das_lib, w, storage, algo)
    assert used == algo and out.shape == ref.shape and out.dtype == np.complex64
    check(out, ref, storage, das_lib, f"config1 algo{algo}")


@pytest.mark.parametrize("storage", [0, 1])
@pytest.mark.parametrize("algo", [1, 2])
def test_config2_small_full(das_lib, storage, algo):
    w, ref = _cfg(2), _oracle_full(2)
    out, used = gpu_das(das_lib, w, storage, algo)
    assert used == algo
    check(out, ref, storage, das_lib, f"config2 algo{algo}")


def _subgrid(number, sx, sy, sz):
    """A sub-block of config ``number``'s native grid (native voxel spacing, ragged extents)."""
    base = _cfg(number)
    return wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs[sx], base.ys[sy], base.zs[sz],
                     fs=base.fs, n_samples=base.n_samples, data_kind=base.data_kind, fc=base.fc,
                     f_number=base.f_number, y=base.y)


@pytest.mark.parametrize("storage", [0, 1])
@pytest.mark.parametrize("algo", [1, 2])
@pytest.mark.parametrize("sl", [(slice(5, 18), slice(10, 17), slice(3, 22)), (slice(31, 32), slice(0, 1), slice(63, 64)),
                                (slice(2, 5), slice(40, 41), slice(0, 37)), (slice(50, 59), slice(1, 18), slice(30, 35))])
def test_ragged_grids(das_lib, storage, algo, sl):
    """Grids that are not multiples of the tile shape (ragged tails, degenerate axes):
    13x7x19, 1x1x1, 3x1x37, 9x17x5 voxels at config 2's native spacing."""
    import oracle
    w = _subgrid(2, *sl)
    ref = oracle.das(w)
    out, used = gpu_das(das_lib, w, storage, algo)
    assert used == algo
    check(out, ref, storage, das_lib, f"config2 sub-grid {w.grid_shape} algo{algo}")


def test_coarse_grid_falls_back_to_general(das_lib):
    """A grid so coarse that a tile's sample window exceeds the largest staged window: AUTO must
    pick the general kernel (still correct), an explicit TILED request must be refused."""
    das = das_lib
    grid = (5, 3, 7)
    w, ref = _cfg(2, grid), _oracle_full(2, grid)
    out, used = gpu_das(das, w, das.STORE_FP32, das.ALGO_AUTO)
    assert used == das.ALGO_GENERAL
    check(out, ref, das.STORE_FP32, das, "coarse grid")
    with pytest.raises(das.DasError) as ei:
        das.Plan.from_workload(w, algo=das.ALGO_TILED)
    assert ei.value.status == das.ERR_UNSUPPORTED


@pytest.mark.parametrize("storage", [0, 1])
@pytest.mark.parametrize("algo", [1, 2])
def test_config4_rf_reduced_grid(das_lib, storage, algo):
    """RF variant: real data, no rotation, real float32 output; headline array and transmits."""
    import oracle
    w = _subgrid(4, slice(40, 64), slice(50, 70), slice(20, 60))          # 24 x 20 x 40 at native spacing
    ref = _rf_ref(oracle, w)
    out, used = gpu_das(das_lib, w, storage, algo)
    assert used == algo and out.dtype == np.float32 and ref.dtype == np.float64
    check(out, ref, storage, das_lib, f"config4 algo{algo}")


_RF_REF = {}


def _rf_ref(oracle, w):
    if "ref" not in _RF_REF:
        _RF_REF["ref"] = oracle.das(w)
    return _RF_REF["ref"]


# ------------------------------------------------------------------ headline size, sampled voxels

def _sample_voxels(w, n_random=1500, seed=99):
    rng = np.random.default_rng(seed)
    nx, ny, nz = w.grid_shape
    idx = set(rng.integers(0, w.n_voxels, n_random).tolist())
    for p in w.scat_pos:                       # voxels nearest each scatterer (where max|x| lives)
        ix = int(np.argmin(np.abs(w.xs.astype(np.float64) - p[0])))
        iy = int(np.argmin(np.abs(w.ys.astype(np.float64) - p[1])))
        iz = int(np.argmin(np.abs(w.zs.astype(np.float64) - p[2])))
        for dz in (-1, 0, 1):
            idx.add((ix * ny + iy) * nz + min(max(iz + dz, 0), nz - 1))
    for c in [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (0, ny - 1, 0), (nx - 1, 0, nz - 1)]:   # grid corners
        idx.add((c[0] * ny + c[1]) * nz + c[2])
    return np.array(sorted(idx), np.int64)


@pytest.mark.parametrize("number,storage", [(3, 1), (3, 0), (4, 1), (4, 0)])
def test_headline_full_size_sampled(das_lib, number, storage):
    """Configs 3 and 4 at full size (128^3 x 1024 x 16) in the launch configuration bench.py
    times; the oracle evaluates a sample of voxels one by one (random + around every scatterer
    + the grid corners).  max|oracle| over the sample includes the strongest scatterers, so the
    ratio is (conservatively) the north_star's."""
    import oracle
    das = das_lib
    w = _cfg(number)
    vox = _sample_voxels(w)
    ref = oracle.das(w, voxels=vox)
    out, used = gpu_das(das, w, storage, das.ALGO_AUTO)
    assert used == das.ALGO_TILED
    got = out.reshape(-1)[vox]
    check(got, ref, storage, das, f"config{number} sampled")


# ------------------------------------------------------------------ edge cases

@pytest.mark.parametrize("algo", [1, 2])
@pytest.mark.parametrize("storage", [0, 1])
def test_out_of_range_samples_dropped(das_lib, algo, storage):
    """t_start pushed so that part of the grid maps before sample 0 and part beyond K-2."""
    import oracle
    base = _subgrid(2, slice(28, 34), slice(30, 35), slice(8, 56))      # 6 x 5 x 48 at native spacing
    w = wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs,
                  fs=base.fs, n_samples=120, t_start=5.0e-6, f_number=1.0,
                  y=np.ascontiguousarray(base.y[:, :, 40:160]))
    res = oracle.das(w, want_count=True)
    cnt = res["count"]
    assert cnt.min() == 0 and cnt.max() > 0 and np.count_nonzero(cnt[..., -1]) == 0
    out, _ = gpu_das(das_lib, w, storage, algo)
    check(out, res["out"], storage, das_lib, "out-of-range")
    assert np.all(out[cnt == 0] == 0)


@pytest.mark.parametrize("algo", [1, 2])
def test_no_apodization(das_lib, algo):
    import oracle
    base = _subgrid(1, slice(10, 18), slice(12, 18), slice(5, 15))      # 8 x 6 x 10 at native spacing
    w = wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs,
                  fs=base.fs, n_samples=base.n_samples, f_number=0.0, y=base.y)
    out, used = gpu_das(das_lib, w, das_lib.STORE_FP32, algo)
    assert used == algo
    check(out, oracle.das(w), das_lib.STORE_FP32, das_lib, "f_number=0")


@pytest.mark.parametrize("algo", [1, 2])
def test_mixed_transmits_offset_array_nonzero_tstart(das_lib, algo):
    """Plane + diverging transmits in one plan, array plane at z != 0, t_start != 0, fc != fs/2."""
    import oracle
    rng = np.random.default_rng(21)
    elem = wl.matrix_array(6)
    elem[:, 2] = np.float32(-0.4e-3)
    elem[:, 0] += np.float32(0.1e-3)
    tx_type = [wl.TX_PLANE, wl.TX_DIVERGING, wl.TX_PLANE]
    a = np.radians(7.0)
    tx_v = [[np.sin(a), 0, np.cos(a)], [0.7e-3, -0.2e-3, -5e-3], [0, 0, 1]]
    tx_t0 = [2e-7, -3.1e-6, 0.0]
    xs, ys, zs = wl.axis(-1e-3, 1.2e-3, 11), wl.axis(-0.8e-3, 0.9e-3, 9), wl.axis(1.5e-3, 5e-3, 23)
    pos = np.stack([rng.uniform(-0.8e-3, 0.8e-3, 4), rng.uniform(-0.6e-3, 0.6e-3, 4), rng.uniform(2e-3, 4.5e-3, 4)], 1)
    w = wl.custom(elem, tx_type, tx_v, tx_t0, xs, ys, zs, fs=20e6, fc=6.25e6, n_samples=300,
                  t_start=1.0e-6, f_number=1.3, scat_pos=pos, scat_amp=[1, 0.5, 0.8, 0.3],
                  noise_sigma=0.01, seed=5)
    out, _ = gpu_das(das_lib, w, das_lib.STORE_FP32, algo)
    check(out, oracle.das(w), das_lib.STORE_FP32, das_lib, "mixed transmits")


def test_tilted_normals(das_lib):
    """Per-element normals.  With coplanar element POSITIONS the delays are the planar array's and only the
    f-number cone turns, so the tiled kernel takes them too; a non-planar array goes to the general kernel
    (AUTO falls back, an explicit TILED request is refused)."""
    import oracle
    das = das_lib
    base = _subgrid(1, slice(2, 30), slice(4, 25), slice(3, 28))
    rng = np.random.default_rng(3)
    d = np.array([0, 0, 1.0]) + 0.2 * rng.normal(size=(64, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    w = wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs,
                  fs=base.fs, n_samples=base.n_samples, f_number=0.9, y=base.y, elem_dir=d)
    ref = oracle.das(w)
    for algo in (das.ALGO_GENERAL, das.ALGO_TILED):
        for storage in (das.STORE_FP32, das.STORE_FP16):
            out, used = gpu_das(das, w, storage, algo)
            assert used == algo
            check(out, ref, storage, das, f"tilted normals algo {algo}")
    cnt_ref = oracle.das(w, want_count=True)["count"]
    assert cnt_ref.min() < cnt_ref.max()                              # the cones do cut
    # non-planar array: general kernel only
    e2 = base.elem_pos.copy()
    e2[:, 2] = (0.05e-3 * np.sin(np.arange(64))).astype(np.float32)
    w2 = wl.custom(e2, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs,
                   fs=base.fs, n_samples=base.n_samples, f_number=0.9, y=base.y, elem_dir=d)
    out, used = gpu_das(das, w2, das.STORE_FP32, das.ALGO_AUTO)
    assert used == das.ALGO_GENERAL
    check(out, oracle.das(w2), das.STORE_FP32, das, "non-planar array")
    with pytest.raises(das.DasError) as ei:
        das.Plan.from_workload(w2, algo=das.ALGO_TILED)
    assert ei.value.status == das.ERR_UNSUPPORTED


def test_beamform_host_matches_device_path(das_lib):
    das, torch = das_lib, _torch()
    w = _cfg(1)
    plan = das.Plan.from_workload(w, storage=das.STORE_FP16)
    h_raw = torch.from_numpy(w.y).pin_memory()
    h_out = torch.empty(w.grid_shape, dtype=torch.complex64).pin_memory()
    plan.beamform_host(h_raw.data_ptr(), h_out.data_ptr())
    dev, _ = das.beamform_torch(plan, torch.from_numpy(w.y).cuda())
    torch.cuda.synchronize()
    np.testing.assert_array_equal(h_out.numpy(), dev.cpu().numpy())
    check(h_out.numpy(), _oracle_full(1), das.STORE_FP16, das, "beamform_host")
    plan.destroy()


def test_execute_overwrites_output_and_is_repeatable(das_lib):
    das, torch = das_lib, _torch()
    w = _cfg(1, (9, 9, 9))
    plan = das.Plan.from_workload(w)
    raw = torch.from_numpy(w.y).cuda()
    out = torch.full(w.grid_shape, 123.0 + 4j, dtype=torch.complex64, device="cuda")
    a, conv = das.beamform_torch(plan, raw, out=out)
    a = a.clone()
    b, _ = das.beamform_torch(plan, raw, conv=conv, out=out)
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    n0 = das.launch_count()
    plan.execute(conv.data_ptr(), out.data_ptr())
    assert das.launch_count() > n0
    plan.destroy()


# ------------------------------------------------------------------ work counter (integers: bit-exact)

@pytest.mark.parametrize("number", [1, 2])
def test_count_work_matches_oracle(das_lib, number):
    """das_plan_count_work (the bench's accounting) against the oracle's per-voxel term count
    (pin P5): integer work, so the totals must be identical.  Every sample of
    configs 1 and 2 is in range, so entered terms = Q x active pairs."""
    import oracle
    w = _cfg(number)
    cnt = oracle.das(w, want_count=True)["count"]
    plan = das_lib.Plan.from_workload(w)
    pairs, terms = plan.count_work()
    plan.destroy()
    assert terms == int(cnt.sum())
    assert pairs * w.n_tx == terms


def test_count_work_out_of_range(das_lib):
    import oracle
    base = _subgrid(2, slice(28, 34), slice(30, 35), slice(8, 56))
    w = wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs,
                  fs=base.fs, n_samples=120, t_start=5.0e-6, f_number=1.0,
                  y=np.ascontiguousarray(base.y[:, :, 40:160]))
    cnt = oracle.das(w, want_count=True)["count"]
    plan = das_lib.Plan.from_workload(w)
    pairs, terms = plan.count_work()
    plan.destroy()
    assert terms == int(cnt.sum()) and terms < pairs * w.n_tx


@pytest.mark.timeout(180)
def test_tiled_kernel_repeated_launches_do_not_hang(das_lib):
    """Regression (round 2): with 3 converter warps over 4-deep rings a converter could fall through the parity wait
    of a slot whose previous round was still in flight; about one launch in fifty of the RF fp32 headline then
    deadlocked its mbarrier rings (found with cuda-gdb: all three roles of one CTA parked in try_wait).  The rings
    are now a multiple of the converter count deep.  Few CTAs walking many tiles made the old hang certain within a
    few launches, so this runs the RF fp32 headline geometry with 74 CTAs, 40 launches back to back, and compares
    the last result with the first (the kernel is deterministic)."""
    torch = _torch()
    das = das_lib
    w = wl.config(4, generate_data=False)
    plan = das.Plan.from_workload(w, storage=das.STORE_FP32, algo=das.ALGO_TILED, debug_tiled_grid=74)
    g = torch.Generator(device="cuda").manual_seed(3)
    raw = torch.randn((w.n_tx, w.n_elem, w.n_samples), device="cuda", generator=g)
    conv = torch.empty(plan.converted_bytes, dtype=torch.uint8, device="cuda")
    outs = [torch.empty(plan.output_bytes // 4, dtype=torch.float32, device="cuda") for _ in range(2)]
    s = torch.cuda.current_stream().cuda_stream
    plan.convert(raw.data_ptr(), conv.data_ptr(), 1.0, s)
    plan.execute(conv.data_ptr(), outs[0].data_ptr(), s)
    for _ in range(40):
        plan.execute(conv.data_ptr(), outs[1].data_ptr(), s)
    torch.cuda.synchronize()
    assert torch.equal(outs[0], outs[1])
    plan.destroy()


@pytest.mark.parametrize("n_tx", [17, 33])
@pytest.mark.parametrize("kind", [wl.DATA_IQ, wl.DATA_RF])
@pytest.mark.parametrize("storage", [0, 1])
def test_more_than_16_transmits_chunked(das_lib, n_tx, kind, storage):
    """More than 16 transmits: the tiled kernel walks the receivers once per chunk of 16 transmits (n_chunks > 1:
    the producer / converter stage counters and the per-chunk phase table are reused), which no BASELINE config
    exercises (ADVICE, round 1).  Mixed plane / diverging transmits, 6 x 6 array, ragged 19 x 13 x 21 grid."""
    import oracle
    das = das_lib
    rng = np.random.default_rng(100 + n_tx)
    elem = wl.matrix_array(6)
    tx_type, tx_v, tx_t0 = [], [], []
    for q in range(n_tx):
        if q % 3 == 2:
            tx_type.append(wl.TX_DIVERGING)
            tx_v.append([rng.uniform(-1e-3, 1e-3), rng.uniform(-1e-3, 1e-3), -rng.uniform(4e-3, 8e-3)])
            tx_t0.append(-float(np.linalg.norm(tx_v[-1])) / wl.C0)
        else:
            a, b = np.radians(rng.uniform(-8, 8, 2))
            tx_type.append(wl.TX_PLANE)
            tx_v.append([np.sin(a), np.sin(b), np.sqrt(1 - np.sin(a) ** 2 - np.sin(b) ** 2)])
            tx_t0.append(rng.uniform(0, 2e-7))
    xs, ys, zs = wl.axis(-1.2e-3, 1.1e-3, 19), wl.axis(-0.9e-3, 1.0e-3, 13), wl.axis(1.5e-3, 6e-3, 21)
    pos = np.stack([rng.uniform(-1e-3, 1e-3, 5), rng.uniform(-0.8e-3, 0.8e-3, 5), rng.uniform(2e-3, 5.5e-3, 5)], 1)
    fs = 15.6e6 if kind == wl.DATA_IQ else 31.2e6
    w = wl.custom(elem, tx_type, tx_v, tx_t0, xs, ys, zs, fs=fs, n_samples=320 if kind == wl.DATA_IQ else 640,
                  data_kind=kind, scat_pos=pos, scat_amp=rng.uniform(0.3, 1, 5), noise_sigma=0.01, seed=9)
    ref = oracle.das(w)
    for algo in (das.ALGO_TILED, das.ALGO_GENERAL):
        out, used = gpu_das(das, w, storage, algo)
        assert used == algo
        check(out, ref, storage, das, f"{n_tx} transmits, algo {algo}")


@pytest.mark.parametrize("algo_name", ["tiled", "general"])
def test_record_edges_with_large_samples(das_lib, algo_name):
    """Reading A6 at the ends of the record with LARGE samples at k = 0, 1, K-2, K-1 (ADVICE, round 1: the edge rule is
    a step, and an index misrounded there would add or drop a whole |y_0| or |y_K-1| term; noise-level edge samples
    would hide it).  The grid is placed so that many (q, m, n) terms have floor(t) in {-1, 0} and {K-2, K-1}; the
    term counts must equal the oracle's exactly and the fp32 result must meet the fp32 gate."""
    import oracle
    das = das_lib
    algo = das.ALGO_TILED if algo_name == "tiled" else das.ALGO_GENERAL
    rng = np.random.default_rng(77)
    elem = wl.matrix_array(6)
    K, fs = 96, 15.6e6
    # two-way travel time to depth z is about 2 z / c: t = 0 near z = t_start c / 2, t = K - 1 near (t_start + (K-1)/fs) c / 2
    t_start = 3.0e-6
    z0, z1 = t_start * wl.C0 / 2, (t_start + (K - 1) / fs) * wl.C0 / 2
    zs = np.concatenate([np.linspace(z0 - 60e-6, z0 + 120e-6, 12), np.linspace(z1 - 120e-6, z1 + 60e-6, 12)])   # 3 + 3 depth tiles
    xs, ys = wl.axis(-0.6e-3, 0.6e-3, 9), wl.axis(-0.5e-3, 0.5e-3, 8)
    y = (rng.normal(size=(2, 36, K)) + 1j * rng.normal(size=(2, 36, K))).astype(np.complex64) * np.float32(0.01)
    for k in (0, 1, K - 2, K - 1):
        y[:, :, k] = (rng.uniform(5, 10, (2, 36)) * np.exp(2j * np.pi * rng.uniform(size=(2, 36)))).astype(np.complex64)
    w = wl.custom(elem, [wl.TX_PLANE, wl.TX_PLANE], [[0, 0, 1], [np.sin(0.05), 0, np.cos(0.05)]], [0.0, 1e-8], xs, ys, zs,
                  fs=fs, n_samples=K, t_start=t_start, f_number=0.0, y=y)
    res = oracle.das(w, want_count=True)
    ref, cnt = res["out"], res["count"]
    out, used = gpu_das(das, w, das.STORE_FP32, algo)
    assert used == algo
    k_edge = int((cnt < w.n_elem * w.n_tx).sum())
    assert k_edge > 50, "the case must have voxels that lose terms at the record ends"
    check(out, ref, das.STORE_FP32, das, "record edges")
    plan = das.Plan.from_workload(w, storage=das.STORE_FP32, algo=algo)
    pairs, terms = plan.count_work()
    plan.destroy()
    assert terms == int(cnt.sum())
