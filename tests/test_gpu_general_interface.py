"""Parity of the paper's general interface through the C ABI (run with -m gpu): transmit delay / weight
tables and per-voxel observation lists, receive
windows, voxel lists and cubic interpolation (NEXT-3), every kernel that takes the
option against the CPU oracle at the north_star tolerances."""
import numpy as np
import pytest

import workloads as wl
from test_gpu_parity import _cfg, _subgrid, _torch, check, errors, TOL_FP16_L2, TOL_FP16_MAX

pytestmark = pytest.mark.gpu


def run(das, w, storage, algo, expect=None, n_frames=0, y=None, **options):
    torch = _torch()
    plan = das.Plan.from_workload(w, storage=storage, algo=algo, n_frames=n_frames, **options)
    if expect is not None:
        assert plan.algo == expect
    raw = torch.from_numpy(np.ascontiguousarray(w.y if y is None else y)).cuda()
    out, _ = das.beamform_torch(plan, raw)
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    plan.destroy()
    return res


def tables_for(w, seed):
    """Transmit tables that differ from the delay models: the model's delay plus a smooth per-voxel offset of up to
    +-1.5 samples, weights in [0.25, 1.75] with a sign flip on one transmit, and observation lists that drop about
    a third of the (q, n) pairs (every voxel keeps at least one transmit)."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = w.grid_shape
    n, q_n = w.n_voxels, w.n_tx
    gx, gy, gz = np.meshgrid(w.xs.astype(np.float64), w.ys.astype(np.float64), w.zs.astype(np.float64), indexing="ij")
    p = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], 1)
    tau = np.empty((q_n, n), np.float64)
    for q in range(q_n):
        v = w.tx_v[q].astype(np.float64)
        base = (p @ v if w.tx_type[q] == wl.TX_PLANE else np.linalg.norm(p - v, axis=1)) / w.c + float(w.tx_t0[q])
        wob = 1.5 / w.fs * np.sin(2 * np.pi * (gx.ravel() / 3e-3 + gz.ravel() / 5e-3) + q)
        tau[q] = base + wob
    wt = rng.uniform(0.25, 1.75, (q_n, n)).astype(np.float32)
    wt[q_n // 2] *= -1.0
    mask = rng.random((q_n, n)) < 0.67
    mask[rng.integers(0, q_n, n), np.arange(n)] = True
    off = np.concatenate([[0], np.cumsum(mask.sum(0))]).astype(np.int64)
    oq = np.concatenate([np.nonzero(mask[:, i])[0] for i in range(n)]).astype(np.int32)
    return tau.astype(np.float32), wt, (off, oq)


@pytest.mark.parametrize("storage", [0, 1])
def test_general_kernel_tables_weights_lists(das_lib, storage):
    import oracle
    das = das_lib
    w = _cfg(2, (20, 18, 24))
    tau, wt, obs = tables_for(w, 31)
    ref = oracle.das(w, tau_tx=tau, w_tx=wt, obs=obs)
    got = run(das, w, storage, das.ALGO_GENERAL, das.ALGO_GENERAL, tau_tx=tau, w_tx=wt, obs=obs)
    check(got, ref, storage, das, "general: tables + weights + lists")
    # each option alone
    check(run(das, w, storage, das.ALGO_GENERAL, tau_tx=tau), oracle.das(w, tau_tx=tau), storage, das, "tau table")
    check(run(das, w, storage, das.ALGO_GENERAL, w_tx=wt), oracle.das(w, w_tx=wt), storage, das, "weights")
    check(run(das, w, storage, das.ALGO_GENERAL, obs=obs), oracle.das(w, obs=obs), storage, das, "lists")


@pytest.mark.parametrize("window,param", [("hann", 0.5), ("tukey", 0.35)])
def test_general_kernel_windows(das_lib, window, param):
    import oracle
    das = das_lib
    w = _cfg(2, (16, 16, 20))
    code = {"hann": das.WINDOW_HANN, "tukey": das.WINDOW_TUKEY}[window]
    ref = oracle.das(w, window=window, window_param=param)
    for storage in (das.STORE_FP32, das.STORE_FP16):
        got = run(das, w, storage, das.ALGO_GENERAL, window=code, window_param=param)
        check(got, ref, storage, das, f"general: {window}")
    assert np.abs(ref - oracle.das(w)).max() > 0.05 * np.abs(ref).max()          # the window does something


def test_general_kernel_voxel_list_and_cubic(das_lib):
    import oracle
    das = das_lib
    w = _cfg(1, (12, 10, 14))
    rng = np.random.default_rng(8)
    pos = np.stack([rng.uniform(-2.4e-3, 2.4e-3, 777), rng.uniform(-2.4e-3, 2.4e-3, 777), rng.uniform(3e-3, 9e-3, 777)], 1).astype(np.float32)
    ref = oracle.das(w, vox_pos=pos)
    got = run(das, w, das.STORE_FP32, das.ALGO_AUTO, das.ALGO_GENERAL, vox_pos=pos)
    assert got.shape == (777, 1, 1)
    check(got, ref, das.STORE_FP32, das, "voxel list")
    refc = oracle.das(w, interp="cubic")
    for storage in (das.STORE_FP32, das.STORE_FP16):
        gotc = run(das, w, storage, das.ALGO_AUTO, das.ALGO_GENERAL, interp=das.INTERP_CUBIC)
        check(gotc, refc, storage, das, "cubic")
    # RF data, cubic + Hann + a voxel list at once
    wr = wl.config(4, grid=(6, 6, 8))
    pr = pos[:200].copy()
    pr[:, 2] = rng.uniform(4e-3, 12e-3, 200)
    refr = oracle.das(wr, vox_pos=pr, interp="cubic", window="hann")
    gotr = run(das, wr, das.STORE_FP32, das.ALGO_AUTO, das.ALGO_GENERAL, vox_pos=pr, interp=das.INTERP_CUBIC, window=das.WINDOW_HANN)
    check(gotr, refr, das.STORE_FP32, das, "RF voxel list cubic hann")
    # the fast kernels refuse what they do not implement
    with pytest.raises(das.DasError) as ei:
        das.Plan.from_workload(w, algo=das.ALGO_TILED, interp=das.INTERP_CUBIC)
    assert ei.value.status == das.ERR_UNSUPPORTED


def test_option_validation(das_lib):
    das = das_lib
    w = _cfg(1, (4, 4, 4))
    n = w.n_voxels
    bad = [dict(window=7), dict(window=das.WINDOW_TUKEY, window_param=0.0), dict(interp=5),
           dict(obs=(np.arange(n + 1), np.full(n, 3, np.int32))),                       # transmit index out of range
           dict(obs=(2 * np.arange(n + 1), np.zeros(2 * n, np.int32))),                  # a transmit listed twice
           dict(tau_tx=np.full((1, n), np.nan, np.float32))]
    for kw in bad:
        with pytest.raises(das.DasError):
            das.Plan.from_workload(w, **kw)


# ------------------------------------------------------------------ the fast kernels

@pytest.mark.parametrize("storage", [0, 1])
def test_tiled_kernel_tables_weights_lists_windows(das_lib, storage):
    import oracle
    das = das_lib
    w = _subgrid(2, slice(6, 40), slice(10, 31), slice(5, 42))            # 34 x 21 x 37: several tiles, ragged
    tau, wt, obs = tables_for(w, 33)
    ref = oracle.das(w, tau_tx=tau, w_tx=wt, obs=obs, window="tukey", window_param=0.4)
    got = run(das, w, storage, das.ALGO_TILED, das.ALGO_TILED, tau_tx=tau, w_tx=wt, obs=obs,
              window=das.WINDOW_TUKEY, window_param=0.4)
    check(got, ref, storage, das, "tiled: tables + weights + lists + tukey")
    check(run(das, w, storage, das.ALGO_AUTO, das.ALGO_TILED, tau_tx=tau), oracle.das(w, tau_tx=tau), storage, das, "tiled: tau table")
    check(run(das, w, storage, das.ALGO_AUTO, das.ALGO_TILED, window=das.WINDOW_HANN), oracle.das(w, window="hann"), storage, das, "tiled: hann")


def test_tiled_kernel_rf_weights_and_window(das_lib):
    import oracle
    das = das_lib
    w = _subgrid(4, slice(50, 70), slice(56, 68), slice(60, 76))          # RF headline geometry, native spacing
    tau, wt, obs = tables_for(w, 34)
    ref = oracle.das(w, w_tx=wt, obs=obs, window="hann")
    for storage in (das.STORE_FP32, das.STORE_FP16):
        got = run(das, w, storage, das.ALGO_TILED, das.ALGO_TILED, w_tx=wt, obs=obs, window=das.WINDOW_HANN)
        check(got, ref, storage, das, "tiled RF: weights + lists + hann")


def test_tc_kernel_tables_weights_lists_windows(das_lib):
    """The frame-batch tensor-core kernel with the general interface: every frame against the oracle."""
    import oracle
    from test_gpu_tc import make_batch
    das = das_lib
    w = _subgrid(3, slice(40, 76), slice(52, 70), slice(70, 78))            # headline geometry, 36 x 18 x 8
    tau, wt, obs = tables_for(w, 35)
    yb = make_batch(w.y, 8, 120)
    got = run(das, w, das.STORE_FP16, das.ALGO_TC, das.ALGO_TC, n_frames=8, y=yb, tau_tx=tau, w_tx=wt, obs=obs,
              window=das.WINDOW_HANN)
    for b in (0, 3, 7):
        ref = oracle.das(w, y=yb[b], tau_tx=tau, w_tx=wt, obs=obs, window="hann")
        emax, el2 = errors(got[b], ref)
        assert emax <= TOL_FP16_MAX and el2 <= TOL_FP16_L2, (b, emax, el2)
    got2 = run(das, w, das.STORE_FP16, das.ALGO_TC, das.ALGO_TC, n_frames=8, y=yb, window=das.WINDOW_TUKEY, window_param=0.5)
    ref2 = oracle.das(w, y=yb[5], window="tukey", window_param=0.5)
    emax, el2 = errors(got2[5], ref2)
    assert emax <= TOL_FP16_MAX and el2 <= TOL_FP16_L2, (emax, el2)


def test_tc_kernel_tilted_normals(das_lib):
    """Tilted receiver normals (coplanar positions) in the frame-batch tensor-core kernel, with a Hann window."""
    import oracle
    from test_gpu_tc import make_batch
    das = das_lib
    base = _subgrid(3, slice(44, 78), slice(50, 68), slice(60, 67))
    rng = np.random.default_rng(12)
    d = np.array([0, 0, 1.0]) + 0.12 * rng.normal(size=(base.n_elem, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    w = wl.custom(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, base.xs, base.ys, base.zs, fs=base.fs,
                  n_samples=base.n_samples, f_number=1.0, y=base.y, elem_dir=d)
    yb = make_batch(w.y, 8, 121)
    got = run(das, w, das.STORE_FP16, das.ALGO_TC, das.ALGO_TC, n_frames=8, y=yb)
    goth = run(das, w, das.STORE_FP16, das.ALGO_TC, das.ALGO_TC, n_frames=8, y=yb, window=das.WINDOW_HANN)
    for b in (0, 6):
        for g_, kw in ((got, {}), (goth, {"window": "hann"})):
            ref = oracle.das(w, y=yb[b], **kw)
            emax, el2 = errors(g_[b], ref)
            assert emax <= TOL_FP16_MAX and el2 <= TOL_FP16_L2, (b, kw, emax, el2)
    assert np.abs(oracle.das(w) - oracle.das(base)).max() > 0.01 * np.abs(oracle.das(base)).max()   # the tilts matter


@pytest.mark.parametrize("algo", [1, 2])
def test_unlisted_transmit_is_never_summed(das_lib, algo):
    """Reading W5: a transmit a voxel does not list -- or lists with weight 0 --
    contributes nothing, whatever its samples hold.  Transmit 2 of config 2 is listed by no voxel and its traces
    are full of +-inf (reading A11 lets fp16 overflow to inf): the volume must equal the oracle's, finite, and the
    term count (das_plan_count_work, the roofline's unit) must equal the oracle's count with the zeros left out."""
    import oracle
    das = das_lib
    torch = _torch()
    w = _cfg(2, (20, 18, 24))
    n, q_n = w.n_voxels, w.n_tx
    rng = np.random.default_rng(8)
    mask = rng.random((q_n, n)) < 0.7
    mask[2] = False
    mask[0, ~mask.any(axis=0)] = True
    off = np.concatenate([[0], np.cumsum(mask.sum(0))]).astype(np.int64)
    oq = np.concatenate([np.nonzero(mask[:, i])[0] for i in range(n)]).astype(np.int32)
    wt = np.where(rng.random((q_n, n)) < 0.2, 0.0, rng.uniform(0.5, 1.5, (q_n, n))).astype(np.float32)   # explicit zeros too
    y = w.y.copy()
    y[2, :, ::3] = np.inf
    y[2, :, 1::3] = -np.inf
    ref = oracle.das(w, y=y, w_tx=wt, obs=(off, oq), want_count=True)
    assert np.isfinite(ref["out"]).all()
    for storage in (das.STORE_FP32, das.STORE_FP16):
        got = run(das, w, storage, algo, algo, y=y, w_tx=wt, obs=(off, oq))
        assert np.isfinite(got.view(np.float32)).all(), "an unlisted transmit leaked into the sum"
        check(got, ref["out"], storage, das, "unlisted transmit with infinite samples")
    plan = das.Plan.from_workload(w, storage=das.STORE_FP32, algo=algo, w_tx=wt, obs=(off, oq))
    assert plan.count_work()[1] == int(ref["count"].sum())
    plan.destroy()


def quadrant_lists(w):
    """A spatially selective sequence: every voxel lists the transmits whose virtual source lies in its own lateral
    quadrant (sign of x and of y): 4 of the headline's 16 sources.  Returns (obs_off, obs_q)."""
    gx, gy, _ = np.meshgrid(w.xs, w.ys, w.zs, indexing="ij")
    sx, sy = np.signbit(gx.ravel()), np.signbit(gy.ravel())
    vx, vy = np.signbit(w.tx_v[:, 0]), np.signbit(w.tx_v[:, 1])
    mask = (vx[:, None] == sx[None, :]) & (vy[:, None] == sy[None, :])                 # [Q, N]
    off = np.concatenate([[0], np.cumsum(mask.sum(0))]).astype(np.int64)
    oq = np.concatenate([np.nonzero(mask[:, i])[0] for i in range(mask.shape[1])]).astype(np.int32)
    return off, oq, mask


@pytest.mark.timeout(300)
def test_tc_kernel_skips_items_nobody_lists(das_lib):
    """the sparse list "would let the kernel skip these negligible contributions".  With quadrant lists
    most (transmit, receiver, depth group) items of a tile are listed by none of its voxels; the plan gives them no
    window, so the batch kernel stages no box and issues no MMA for them (16 transmits, so this also runs the
    run-time slot tracking instead of the compile-time phases).  Frames 0 and 5 against the oracle, on a block that
    straddles all four quadrants."""
    import oracle
    from test_gpu_tc import make_batch
    das = das_lib
    w = _subgrid(3, slice(40, 88), slice(48, 80), slice(60, 72))            # 48 x 32 x 12 around the axis
    off, oq, mask = quadrant_lists(w)
    assert mask.sum(0).min() == 4 and mask.sum(0).max() == 4 and mask.any(1).all()
    yb = make_batch(w.y, 8, 140)
    got = run(das, w, das.STORE_FP16, das.ALGO_TC, das.ALGO_TC, n_frames=8, y=yb, obs=(off, oq))
    for b in (0, 5):
        ref = oracle.das(w, y=yb[b], obs=(off, oq))
        emax, el2 = errors(got[b], ref)
        assert emax <= TOL_FP16_MAX and el2 <= TOL_FP16_L2, (b, emax, el2)
    dense = oracle.das(w, y=yb[0])
    assert np.abs(dense - oracle.das(w, y=yb[0], obs=(off, oq))).max() > 0.05 * np.abs(dense).max()   # the lists matter
