"""Dense-matrix brute force for tiny grids -- TEST INFRASTRUCTURE (pins oracle/das_oracle.c).

DAS is linear in the channel data (Eq. 2), so the whole method is one matrix:
x = W y with y the [Q*M*K] sample vector and W in C^{N x QMK} holding, per (n,q,m), the two
interpolation weights (1-alpha) and alpha at columns k and k+1 times the receive
weight and, for IQ, the rotation exp(+j 2 pi fc tau).  This module builds W explicitly with
numpy array operations (a formulation independent of the C loops) and reduces the sum to a
library routine, ``numpy.matmul``.  Only usable for tiny sizes: W is dense.
"""
from __future__ import annotations

import numpy as np


def _keys(x):
    """Cubic convolution kernel (Keys 1981, a = -1/2) as a function of the distance x to the sample."""
    x = np.abs(x)
    return np.where(x <= 1.0, 1.5 * x ** 3 - 2.5 * x ** 2 + 1.0,
                    np.where(x < 2.0, -0.5 * x ** 3 + 2.5 * x ** 2 - 4.0 * x + 2.0, 0.0))


def dense_matrix(w, *, tau_tx=None, w_tx=None, obs_mask=None, vox_pos=None, window="boxcar",
                 window_param=0.5, interp="linear") -> np.ndarray:
    """W [N, Q*M*K] (complex128; real-valued when the workload is RF).

    Options (das_oracle.c header): ``tau_tx`` / ``w_tx`` [Q,N] tables, ``obs_mask`` [Q,N] booleans (the
    observation lists as a mask), ``vox_pos`` [N,3], ``window`` boxcar / hann / tukey(``window_param``),
    ``interp`` linear / cubic.  Formulated apart from the C loops: the interpolation weights come from
    the kernel function h(t - k) evaluated on the whole sample axis, not from floor / fraction."""
    e = np.asarray(w.elem_pos, dtype=np.float64)                       # [M,3]
    nrm = (np.tile(np.array([0.0, 0.0, 1.0]), (len(e), 1)) if getattr(w, "elem_dir", None) is None
           else np.asarray(w.elem_dir, dtype=np.float64))
    if vox_pos is not None:
        p = np.asarray(vox_pos, dtype=np.float32).astype(np.float64).reshape(-1, 3)
    else:
        gx, gy, gz = np.meshgrid(np.asarray(w.xs, np.float64), np.asarray(w.ys, np.float64),
                                 np.asarray(w.zs, np.float64), indexing="ij")
        p = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1)      # [N,3], z fastest
    c, fc, fs = (float(np.float32(v)) for v in (w.c, w.fc, w.fs))
    t_start, fnum = float(np.float32(w.t_start)), float(np.float32(w.f_number))
    n_n, m_n, q_n, k_n = len(p), len(e), len(w.tx_type), int(w.n_samples)
    d = p[:, None, :] - e[None, :, :]                                   # [N,M,3]
    dist = np.sqrt(np.einsum("nmi,nmi->nm", d, d))
    a = np.einsum("nmi,mi->nm", d, nrm)
    if fnum > 0:
        rho2 = np.einsum("nmi,nmi->nm", d, d) - a * a
        if getattr(w, "elem_dir", None) is None:
            rho2 = d[..., 0] ** 2 + d[..., 1] ** 2
        wrx = ((a > 0) & (4.0 * fnum * fnum * rho2 <= a * a)).astype(np.float64)
        with np.errstate(divide="ignore", invalid="ignore"):
            u = np.where(wrx > 0, 2.0 * fnum * np.sqrt(np.maximum(rho2, 0.0)) / a, 0.0)
        if window == "hann":
            wrx = wrx * 0.5 * (1.0 + np.cos(np.pi * u))
        elif window == "tukey":
            b = float(np.float32(window_param))
            wrx = wrx * np.where(u <= 1.0 - b, 1.0, 0.5 * (1.0 + np.cos(np.pi * (u - 1.0 + b) / b)))
        elif window != "boxcar":
            raise ValueError(window)
    else:
        wrx = np.ones_like(a)
    mat = np.zeros((n_n, q_n, m_n, k_n), dtype=np.complex128)
    for q in range(q_n):
        v = np.asarray(w.tx_v[q], dtype=np.float64)
        t0 = float(w.tx_t0[q])
        if tau_tx is not None:
            ttx = np.asarray(tau_tx, np.float32).astype(np.float64).reshape(q_n, n_n)[q]
        elif int(w.tx_type[q]) == 0:
            ttx = p @ v / c + t0
        else:
            ttx = np.linalg.norm(p - v, axis=1) / c + t0
        tau = ttx[:, None] + dist / c                                  # [N,M]
        t = (tau - t_start) * fs
        k = np.floor(t)
        wq = wrx.copy()
        if w_tx is not None:
            wq = wq * np.asarray(w_tx, np.float32).astype(np.float64).reshape(q_n, n_n)[q][:, None]
        if obs_mask is not None:
            wq = wq * np.asarray(obs_mask, bool).reshape(q_n, n_n)[q][:, None]
        rot = np.exp(2j * np.pi * fc * tau) if int(w.data_kind) == 0 else np.ones_like(tau)
        kk = np.arange(k_n, dtype=np.float64)
        dist_k = t[:, :, None] - kk[None, None, :]                      # [N,M,K]: t - k for every sample
        if interp == "linear":
            h = np.maximum(0.0, 1.0 - np.abs(dist_k))                   # the hat function = linear interpolation
            ok = (k >= 0) & (k <= k_n - 2)
        elif interp == "cubic":
            h = _keys(dist_k)
            ok = (k >= 1) & (k <= k_n - 3)
        else:
            raise ValueError(interp)
        mat[:, q] = np.where(ok[:, :, None], h, 0.0) * (wq * rot)[:, :, None]
    return mat.reshape(n_n, q_n * m_n * k_n)


def das(w, y=None, **opts) -> np.ndarray:
    """x = W y, reshaped to [nx,ny,nz] ([N,1,1] for a voxel list)."""
    y = w.y if y is None else y
    mat = dense_matrix(w, **opts)
    x = np.matmul(mat, np.asarray(y).astype(np.complex128).ravel())
    if opts.get("vox_pos") is not None:
        x = x.reshape(-1, 1, 1)
    else:
        x = x.reshape(len(w.xs), len(w.ys), len(w.zs))
    return x if int(w.data_kind) == 0 else x.real


def das_from_interval_table(w, mid, slope, **unsupported) -> np.ndarray:
    """The definition evaluated on a given table of sample INTERVALS: y[t] = mid_k + (alpha - 1/2) slope_k for
    t = k + alpha (equal to linear interpolation, when mid_k = (y_k + y_k+1)/2 and
    slope_k = y_k+1 - y_k).  ``mid`` / ``slope``: [Q, M, K-1].  Used to check a storage format that quantises
    the interval table (fp8 storage) term by term instead of only statistically.

    Pinned by tests/test_oracle_ext_pins.py (test_interval_table_*): equal to oracle.das on the exact table of
    random data (IQ with and without the f-number cone, RF) and the hand value of closed_form_cases.json
    plane_345.  Boxcar aperture about (0, 0, 1) normals and the delay models of tx[] only: element normals,
    windows, tables, lists or cubic interpolation raise instead of being ignored."""
    if unsupported:
        raise TypeError(f"das_from_interval_table does not take {sorted(unsupported)}")
    if getattr(w, "elem_dir", None) is not None:
        raise ValueError("das_from_interval_table handles (0, 0, 1) element normals only")
    mid, slope = np.asarray(mid), np.asarray(slope)
    want = (len(w.tx_type), len(w.elem_pos), int(w.n_samples) - 1)
    if mid.shape != want or slope.shape != want:
        raise ValueError(f"mid / slope must be [Q, M, K-1] = {want}, got {mid.shape} / {slope.shape}")
    e = np.asarray(w.elem_pos, dtype=np.float64)
    gx, gy, gz = np.meshgrid(np.asarray(w.xs, np.float64), np.asarray(w.ys, np.float64),
                             np.asarray(w.zs, np.float64), indexing="ij")
    p = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1)
    c, fc, fs = (float(np.float32(v)) for v in (w.c, w.fc, w.fs))
    t_start, fnum = float(np.float32(w.t_start)), float(np.float32(w.f_number))
    k_n = int(w.n_samples)
    d = p[:, None, :] - e[None, :, :]
    dist = np.sqrt(np.einsum("nmi,nmi->nm", d, d))
    if fnum > 0:
        wrx = ((d[..., 2] > 0) & (4.0 * fnum * fnum * (d[..., 0] ** 2 + d[..., 1] ** 2) <= d[..., 2] ** 2)).astype(np.float64)
    else:
        wrx = np.ones_like(dist)
    mid = np.asarray(mid).astype(np.complex128)
    slope = np.asarray(slope).astype(np.complex128)
    x = np.zeros(len(p), np.complex128)
    mm = np.arange(len(e))[None, :]
    for q in range(len(w.tx_type)):
        v = np.asarray(w.tx_v[q], dtype=np.float64)
        ttx = (p @ v / c if int(w.tx_type[q]) == 0 else np.linalg.norm(p - v, axis=1) / c) + float(w.tx_t0[q])
        tau = ttx[:, None] + dist / c
        t = (tau - t_start) * fs
        k = np.floor(t)
        ok = (k >= 0) & (k <= k_n - 2) & (wrx > 0)
        ki = np.where(ok, k, 0).astype(np.int64)
        s = mid[q][mm, ki] + (t - k - 0.5) * slope[q][mm, ki]
        rot = np.exp(2j * np.pi * fc * tau) if int(w.data_kind) == 0 else 1.0
        x += np.where(ok, s * rot, 0.0).sum(axis=1)
    x = x.reshape(len(w.xs), len(w.ys), len(w.zs))
    return x if int(w.data_kind) == 0 else x.real
