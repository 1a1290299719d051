"""Pins for the oracle's extensions (das_oracle_ex): transmit delay / weight tables, per-voxel
observation lists, voxel lists, receive windows, cubic interpolation.

SURVEY.md 8(f) NEXT-2 (PAPER.md:43, :95, :101 Alg. 1 "Require", :365) and NEXT-3 (PAPER.md:43, :50,
:101).  Nothing here touches the CUDA path.  Each option is pinned against something other than the
C loops: hand-derived values (tests/golden/ext_cases.json), the unextended oracle it must reduce to,
closed forms of the windows and of the cubic kernel, and the dense-matrix brute force."""
import json
import os

import numpy as np
import pytest

import workloads as wl
from test_oracle_pins import _ramp, _small_problem

EXT = os.path.join(os.path.dirname(__file__), "golden", "ext_cases.json")


def _ext():
    with open(EXT) as f:
        return json.load(f)


def _one_voxel(case, u, q=1, y=None, f_number=0.0, fc=None, voxel=None):
    elem = np.array(case["elem_pos_u"], np.float64) * u if "elem_pos_u" in case else np.zeros((1, 3))
    vox = np.array(case["voxel_u"] if voxel is None else voxel, np.float64) * u
    tx_type = np.full(q, wl.TX_PLANE, np.int32)
    tx_v = np.tile(np.array([0.0, 0.0, 1.0], np.float32), (q, 1))
    return wl.custom(elem, tx_type, tx_v, np.zeros(q, np.float32), [vox[0]], [vox[1]], [vox[2]],
                     fs=case["fs"], n_samples=case["K"], c=case["c"], fc=case.get("fc", 0.0) if fc is None else fc,
                     t_start=case.get("t_start", 0.0), f_number=f_number, y=y)


# ---------------------------------------------------------------- NEXT-2: tables, weights, lists

def test_table_golden(oracle):
    """Hand-derived weighted sum over two table-delayed observations (ext_cases.json table_case)."""
    g = _ext()
    case, u = g["table_case"], g["u"]
    y = _ramp(2, 1, case["K"], complex(*case["ramp_a"]), complex(*case["ramp_b"]))
    w = _one_voxel(case, u, q=2, y=y)
    tau = (np.array(case["tau_tx_units_of_2pm18"]) * 2.0 ** -18).astype(np.float32).reshape(2, 1)
    assert np.all(tau.astype(np.float64).ravel() == np.array(case["tau_tx_units_of_2pm18"]) * 2.0 ** -18)   # exact in float32
    wt = np.array(case["w_tx"], np.float32).reshape(2, 1)
    got = oracle.das(w, tau_tx=tau, w_tx=wt)[0, 0, 0]
    assert abs(got - complex(*case["expected_weighted"])) <= 1e-12 * abs(got)
    got1 = oracle.das(w, tau_tx=tau)[0, 0, 0]
    assert abs(got1 - complex(*case["expected_unit_weights"])) <= 1e-12 * abs(got1)
    got2 = oracle.das(w, tau_tx=tau, w_tx=wt, obs=([0, 1], [1]))[0, 0, 0]
    assert abs(got2 - complex(*case["expected_weighted_list_q1"])) <= 1e-12 * abs(got2)


def _dyadic_problem():
    """Plane wave along +z, c = 1024 m/s and a dyadic z axis: tau_tx = z / c is exact in float32, so a table
    that restates fn. 2 holds the very numbers the formula path computes."""
    rng = np.random.default_rng(3)
    elem = wl.matrix_array(3)
    xs, ys = wl.axis(-0.5e-3, 0.5e-3, 4), wl.axis(-0.4e-3, 0.6e-3, 3)
    zs = (np.arange(1, 6) * 2.0 ** -10).astype(np.float32)
    y = (rng.normal(size=(1, 9, 128)) + 1j * rng.normal(size=(1, 9, 128))).astype(np.complex64)
    return wl.custom(elem, [wl.TX_PLANE], [[0, 0, 1]], [0.0], xs, ys, zs, fs=2.0 ** 22, fc=2.0 ** 20, c=1024.0,
                     n_samples=128, f_number=1.0, y=y)


def test_table_restating_the_formula_is_bit_identical(oracle):
    w = _dyadic_problem()
    ref = oracle.das(w)
    zz = np.broadcast_to(w.zs.astype(np.float64)[None, None, :], w.grid_shape)
    tau = (zz / 1024.0).astype(np.float32)
    assert np.all(tau.astype(np.float64) == zz / 1024.0)
    got = oracle.das(w, tau_tx=tau.reshape(1, -1))
    assert np.array_equal(got, ref)
    assert np.abs(ref).max() > 0


def test_unit_weights_and_full_lists_reduce_to_the_plain_oracle(oracle):
    w = _small_problem(11)
    n = w.n_voxels
    ref = oracle.das(w)
    assert np.array_equal(oracle.das(w, w_tx=np.ones((2, n), np.float32)), ref)
    off = 2 * np.arange(n + 1)
    oq = np.tile([0, 1], n)
    assert np.array_equal(oracle.das(w, obs=(off, oq)), ref)
    # a list is a selection: listing only q = 1 equals the one-transmit problem
    only1 = oracle.das(w, obs=(np.arange(n + 1), np.ones(n, np.int32)))
    w1 = wl.custom(w.elem_pos, w.tx_type[1:], w.tx_v[1:], w.tx_t0[1:], w.xs, w.ys, w.zs, fs=w.fs,
                   n_samples=w.n_samples, f_number=w.f_number, y=w.y[1:])
    np.testing.assert_allclose(only1, oracle.das(w1), rtol=0, atol=1e-13 * np.abs(ref).max())
    # an empty list gives zero
    z = oracle.das(w, obs=(np.zeros(n + 1, np.int64), np.zeros(0, np.int32)))
    assert np.all(z == 0)


def test_zero_weight_equals_not_listed(oracle):
    """Reading W5: w_tx == 0 is the same as not listing the transmit.  A weight
    table with explicit zeros gives the volume AND the term count of the observation lists that leave those
    (q, n) out, bit for bit, and an infinite sample in a zero-weighted transmit is never read."""
    w = _small_problem(14)
    n = w.n_voxels
    rng = np.random.default_rng(2)
    keep = rng.random((2, n)) < 0.6                                   # which (q, n) stay
    keep[:, 0] = [False, False]                                       # one voxel with nothing left
    wt = np.where(keep, rng.uniform(0.5, 1.5, (2, n)), 0.0).astype(np.float32)
    off = np.concatenate([[0], np.cumsum(keep.sum(axis=0))])
    oq = np.concatenate([np.nonzero(keep[:, i])[0] for i in range(n)]).astype(np.int32)
    a = oracle.das(w, w_tx=wt, want_count=True)
    b = oracle.das(w, w_tx=np.where(keep, wt, 7.0).astype(np.float32), obs=(off, oq), want_count=True)
    assert np.array_equal(a["out"], b["out"]) and np.array_equal(a["count"], b["count"])
    full = oracle.das(w, want_count=True)
    assert 0 < a["count"].sum() < full["count"].sum() and a["count"].ravel()[0] == 0 and a["out"].ravel()[0] == 0
    # transmit 1 switched off everywhere: its samples may hold anything
    y = w.y.copy()
    y[1, :, ::7] = np.inf
    wt1 = np.stack([np.ones(n, np.float32), np.zeros(n, np.float32)])
    got = oracle.das(w, y=y, w_tx=wt1)
    assert np.isfinite(got).all()
    assert np.array_equal(got, oracle.das(w, obs=(np.arange(n + 1), np.zeros(n, np.int32))))


def test_weights_scale_each_transmit(oracle):
    """x = sum_q w_q x_q for weights constant over the voxels (linearity in w_tx)."""
    w = _small_problem(12)
    n = w.n_voxels
    parts = [oracle.das(w, obs=(np.arange(n + 1), np.full(n, q, np.int32))) for q in range(2)]
    wt = np.empty((2, n), np.float32)
    wt[0], wt[1] = 0.375, -1.5
    got = oracle.das(w, w_tx=wt)
    np.testing.assert_allclose(got, 0.375 * parts[0] - 1.5 * parts[1], rtol=0, atol=1e-13 * np.abs(got).max())


def test_table_delay_shift_moves_the_sample_and_the_phase(oracle):
    """Adding one sample period to tau_tx of every voxel equals shifting the data by one sample and
    rotating by exp(j 2 pi fc / fs) (the phase uses the absolute tau, reading A7)."""
    w = _dyadic_problem()
    zz = np.broadcast_to(w.zs.astype(np.float64)[None, None, :], w.grid_shape)
    tau = (zz / 1024.0).reshape(1, -1)
    shifted = (tau + 2.0 ** -22).astype(np.float32)
    y2 = np.zeros_like(w.y)
    y2[..., 1:] = w.y[..., :-1]
    a = oracle.das(w, tau_tx=shifted, y=y2)
    b = oracle.das(w, tau_tx=tau.astype(np.float32)) * np.exp(2j * np.pi * 2.0 ** 20 / 2.0 ** 22)
    cnt = oracle.das(w, tau_tx=shifted, want_count=True)["count"]
    full = cnt == cnt.max()
    np.testing.assert_allclose(a[full], b[full], rtol=0, atol=1e-12 * np.abs(b).max())


# ---------------------------------------------------------------- NEXT-3: voxel lists, windows, cubic

def test_voxel_list_equals_the_grid(oracle):
    w = _small_problem(13)
    ref = oracle.das(w)
    gx, gy, gz = np.meshgrid(w.xs, w.ys, w.zs, indexing="ij")
    pos = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], 1)
    perm = np.random.default_rng(0).permutation(len(pos))
    got = oracle.das(w, vox_pos=pos[perm])
    assert got.shape == (len(pos), 1, 1)
    assert np.array_equal(got[:, 0, 0], ref.ravel()[perm])


def test_window_golden(oracle):
    g = _ext()
    case, u = g["window_cases"], g["u"]
    y = np.ones((1, 1, case["K"]), np.complex64)
    for vox, hann, tukey in case["voxels_u_hann_tukey"]:
        w = _one_voxel(case, u, y=y, f_number=1.0, fc=0.0, voxel=vox)
        assert abs(oracle.das(w, window="hann")[0, 0, 0] - hann) <= 1e-15, vox
        assert abs(oracle.das(w, window="tukey", window_param=case["tukey_taper"])[0, 0, 0] - tukey) <= 1e-15, vox
        box = 1.0 if (hann > 0 or (vox[0] == 2 and vox[2] == 4)) else 0.0          # the cone edge is active for the boxcar
        assert oracle.das(w)[0, 0, 0] == box


def test_window_limits(oracle):
    """Tukey with taper 1 is Hann; Tukey with a vanishing taper tends to the boxcar away from the edge; every
    window is 1 without apodization; windows only ever shrink the boxcar's terms."""
    w = _small_problem(14)
    hann = oracle.das(w, window="hann")
    np.testing.assert_allclose(oracle.das(w, window="tukey", window_param=1.0), hann, rtol=0, atol=1e-13 * np.abs(hann).max())
    w0 = _small_problem(14, f_number=0.0)
    assert np.array_equal(oracle.das(w0, window="hann"), oracle.das(w0))
    ones = wl.custom(w.elem_pos, w.tx_type, w.tx_v, w.tx_t0, w.xs, w.ys, w.zs, fs=w.fs, n_samples=w.n_samples, fc=0.0,
                     f_number=1.0, y=np.ones_like(w.y))
    box, hn, tk = oracle.das(ones).real, oracle.das(ones, window="hann").real, oracle.das(ones, window="tukey", window_param=0.3).real
    assert np.all(hn <= tk + 1e-12) and np.all(tk <= box + 1e-12) and np.all(hn >= 0)


def test_cubic_golden_and_kernel(oracle):
    g = _ext()
    u = g["u"]
    with open(os.path.join(os.path.dirname(EXT), "closed_form_cases.json")) as f:
        base = json.load(f)["cases"][0]
    case = g["cubic_case"]
    kk = np.arange(base["K"], dtype=np.float64)
    row = complex(*base["ramp_a"]) + complex(*base["ramp_b"]) * kk + case["quad_c"] * kk * kk
    y = row.astype(np.complex64).reshape(1, 1, -1)
    assert np.all(y.astype(np.complex128).ravel() == row)                      # exact in float32
    w = _one_voxel(base, u, y=y)
    got = oracle.das(w, interp="cubic")[0, 0, 0]
    assert abs(got - complex(*case["expected"])) <= 1e-12 * abs(got)
    # impulse data: the kernel itself, sampled half way between two samples
    fs, c = base["fs"], base["c"]
    zv = 40.5 * c / fs                                                          # t = 40.5 samples for an element at the voxel's (x, y)
    for off, val in zip((-1, 0, 1, 2), case["kernel_half"]):
        yi = np.zeros((1, 1, 128), np.complex64)
        yi[0, 0, 40 + off] = 1.0
        wi = wl.custom(np.zeros((1, 3)), [wl.TX_PLANE], [[0, 0, 1]], [0.0], [0.0], [0.0], [zv / 2.0], fs=fs, c=c, fc=0.0,
                       n_samples=128, f_number=0.0, y=yi)
        t = (wi.zs[0].astype(np.float64) * 2.0 / c) * fs
        assert abs(t - 40.5) < 1e-4
        assert abs(oracle.das(wi, interp="cubic")[0, 0, 0].real - val) < 1e-3   # zs is float32: t is 40.5 to 1e-4 only


def test_cubic_reproduces_quadratics_and_drops_edges(oracle):
    rng = np.random.default_rng(5)
    w = _small_problem(15, f_number=0.0, k=96)
    kk = np.arange(96, dtype=np.float64)
    a, b, cq = 0.5 - 1.0j, 0.125 + 0.0625j, 2.0 ** -7
    row = (a + b * kk + cq * kk * kk).astype(np.complex64)
    y = np.broadcast_to(row, w.y.shape).copy()
    res = oracle.das(w, y=y, interp="cubic", want_count=True)
    lin = oracle.das(w, y=y, want_count=True)
    assert np.all(res["count"] <= lin["count"])
    # closed form per voxel: sum over (q, m) of (a + b t + c t^2) exp(j 2 pi fc tau)
    import oracle.brute as brute
    np.testing.assert_allclose(res["out"], brute.das(w, y=y, interp="cubic"), rtol=0, atol=1e-10 * np.abs(res["out"]).max())
    e = w.elem_pos.astype(np.float64)
    gx, gy, gz = np.meshgrid(w.xs.astype(np.float64), w.ys.astype(np.float64), w.zs.astype(np.float64), indexing="ij")
    p = np.stack([gx, gy, gz], -1)
    x = np.zeros(w.grid_shape, np.complex128)
    for q in range(2):
        v = w.tx_v[q].astype(np.float64)
        ttx = (p @ v / w.c if w.tx_type[q] == wl.TX_PLANE else np.linalg.norm(p - v, axis=-1) / w.c) + float(w.tx_t0[q])
        for m in range(len(e)):
            tau = ttx + np.linalg.norm(p - e[m], axis=-1) / w.c
            t = tau * w.fs
            ok = (np.floor(t) >= 1) & (np.floor(t) <= 96 - 3)
            x += np.where(ok, (a + b * t + cq * t * t) * np.exp(2j * np.pi * w.fc * tau), 0.0)
    np.testing.assert_allclose(res["out"], x, rtol=0, atol=2e-6 * np.abs(x).max())   # data is float32-rounded


@pytest.mark.parametrize("kind", [wl.DATA_IQ, wl.DATA_RF])
def test_bruteforce_all_options(oracle, kind):
    """Dense-matrix x = W y with tables, weights, lists, a window and both interpolations switched on."""
    import oracle.brute as brute
    rng = np.random.default_rng(21)
    w = _small_problem(16, kind=kind, n=(3, 4, 3), k=80)
    n = w.n_voxels
    tau = rng.uniform(0.9e-6, 1.6e-6, (2, n)).astype(np.float32)
    wt = rng.uniform(-1, 2, (2, n)).astype(np.float32)
    mask = rng.random((2, n)) < 0.7
    off = np.concatenate([[0], np.cumsum(mask.sum(0))])
    oq = np.concatenate([np.nonzero(mask[:, i])[0] for i in range(n)]).astype(np.int32)
    for win, par in (("hann", 0.5), ("tukey", 0.4)):
        for interp in ("linear", "cubic"):
            a = oracle.das(w, tau_tx=tau, w_tx=wt, obs=(off, oq), window=win, window_param=par, interp=interp)
            b = brute.das(w, tau_tx=tau, w_tx=wt, obs_mask=mask, window=win, window_param=par, interp=interp)
            np.testing.assert_allclose(a, b, rtol=0, atol=1e-11 * max(np.abs(b).max(), 1e-30))
            assert np.abs(b).max() > 0


def test_slack_output_counts_near_edge_terms(oracle):
    """out_slack: |term| summed over pairs within slack_rel of the cone edge (exactly on it here)."""
    g = _ext()
    case, u = g["window_cases"], g["u"]
    y = np.full((1, 1, case["K"]), 3.0 - 4.0j, np.complex64)
    w = _one_voxel(case, u, y=y, f_number=1.0, fc=0.0, voxel=[2, 0, 4])       # on the edge: margin 0
    r = oracle.das(w, want_slack=True)
    assert abs(r["slack"][0, 0, 0] - 5.0) < 1e-12
    w2 = _one_voxel(case, u, y=y, f_number=1.0, fc=0.0, voxel=[1, 0, 4])      # well inside
    assert oracle.das(w2, want_slack=True)["slack"][0, 0, 0] == 0.0


# ---------------------------------------------------------------- the interval-table evaluator (FP8 check helper)

def _exact_table(y):
    """(mid, slope) of PAPER.md:50's two-sample lerp, formed in FP64 from the float32 samples."""
    yd = np.asarray(y).astype(np.complex128)
    return 0.5 * (yd[:, :, :-1] + yd[:, :, 1:]), yd[:, :, 1:] - yd[:, :, :-1]


@pytest.mark.parametrize("kind,f_number", [(wl.DATA_IQ, 1.0), (wl.DATA_IQ, 0.0), (wl.DATA_RF, 1.0)])
def test_interval_table_equals_the_oracle_on_the_exact_table(oracle, kind, f_number):
    """mid_k + (alpha - 1/2) slope_k with mid = (y_k + y_k+1)/2, slope = y_k+1 - y_k IS (1 - alpha) y_k + alpha y_k+1
    (PAPER.md:50), so on the unquantised table oracle/brute.py::das_from_interval_table must reproduce the pinned C
    oracle: a wrong aperture rule, a transposed mid[q][m, k], a dropped 1/2 or a wrong sign in it fails here."""
    import oracle.brute as brute
    w = _small_problem(21, kind=kind, f_number=f_number, n=(5, 4, 6), k=96)
    ref = oracle.das(w)
    mid, slope = _exact_table(w.y)
    got = brute.das_from_interval_table(w, mid, slope)
    assert got.shape == ref.shape and np.iscomplexobj(got) == (kind == wl.DATA_IQ)
    assert np.abs(ref).max() > 0
    if f_number > 0:                                  # the cone really cuts pairs in this geometry
        assert oracle.das(w, want_count=True)["count"].sum() < oracle.das(
            _small_problem(21, kind=kind, f_number=0.0, n=(5, 4, 6), k=96), want_count=True)["count"].sum()
    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-12 * np.abs(ref).max())
    # a table that is NOT the lerp's must change the answer (the check above is not vacuous)
    off = brute.das_from_interval_table(w, mid, -slope)
    assert np.abs(off - ref).max() > 1e-3 * np.abs(ref).max()


def test_interval_table_hand_value():
    """closed_form_cases.json plane_345 (PAPER.md:35-37 Eq. 1, :77 fn. 2, :50): the ramp y_k = a + b k has
    mid_k = a + b (k + 1/2), slope_k = b; t = 115.2, 0.8 turn: x = -7.3799 - 64.0136j (derived by hand there)."""
    import oracle.brute as brute
    with open(os.path.join(os.path.dirname(__file__), "golden", "closed_form_cases.json")) as f:
        g = json.load(f)
    u, case = g["u"], g["cases"][0]
    assert case["name"] == "plane_345"
    a, b = complex(*case["ramp_a"]), complex(*case["ramp_b"])
    k = case["K"]
    elem, vox = np.array(case["elem_pos_u"], np.float64) * u, np.array(case["voxel_u"], np.float64) * u
    w = wl.custom(elem, [wl.TX_PLANE], [case["tx"]["v"]], [case["tx"]["t0"]], [vox[0]], [vox[1]], [vox[2]],
                  fs=case["fs"], n_samples=k, c=case["c"], fc=case["fc"], t_start=case["t_start"],
                  f_number=case["f_number"], y=_ramp(1, 1, k, a, b))
    kk = np.arange(k - 1, dtype=np.float64)
    mid = (a + b * (kk + 0.5)).reshape(1, 1, -1)
    slope = np.full((1, 1, k - 1), b)
    got = brute.das_from_interval_table(w, mid, slope)[0, 0, 0]
    exp = complex(*case["expected"])
    assert abs(got - exp) <= 1e-9 * abs(exp), (got, exp)


def test_interval_table_refuses_what_it_does_not_model():
    import oracle.brute as brute
    w = _small_problem(5, n=(2, 2, 2), k=32)
    mid, slope = _exact_table(w.y)
    with pytest.raises(TypeError):
        brute.das_from_interval_table(w, mid, slope, window="hann")
    with pytest.raises(TypeError):
        brute.das_from_interval_table(w, mid, slope, tau_tx=np.zeros((2, 8), np.float32))
    with pytest.raises(ValueError):
        brute.das_from_interval_table(w, mid[:, :, :-1], slope[:, :, :-1])
    w.elem_dir = np.tile(np.array([0.0, 0.0, 1.0], np.float32), (len(w.elem_pos), 1))
    with pytest.raises(ValueError):
        brute.das_from_interval_table(w, mid, slope)
