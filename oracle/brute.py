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


def dense_matrix(w) -> np.ndarray:
    """W [N, Q*M*K] (complex128; real-valued when the workload is RF)."""
    e = np.asarray(w.elem_pos, dtype=np.float64)                       # [M,3]
    nrm = (np.tile(np.array([0.0, 0.0, 1.0]), (len(e), 1)) if getattr(w, "elem_dir", None) is None
           else np.asarray(w.elem_dir, dtype=np.float64))
    gx, gy, gz = np.meshgrid(np.asarray(w.xs, np.float64), np.asarray(w.ys, np.float64),
                             np.asarray(w.zs, np.float64), indexing="ij")
    p = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1)          # [N,3], z fastest
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
    else:
        wrx = np.ones_like(a)
    mat = np.zeros((n_n, q_n, m_n, k_n), dtype=np.complex128)
    nn, mm = np.meshgrid(np.arange(n_n), np.arange(m_n), indexing="ij")
    for q in range(q_n):
        v = np.asarray(w.tx_v[q], dtype=np.float64)
        t0 = float(w.tx_t0[q])
        if int(w.tx_type[q]) == 0:
            tau_tx = p @ v / c + t0
        else:
            tau_tx = np.linalg.norm(p - v, axis=1) / c + t0
        tau = tau_tx[:, None] + dist / c                               # [N,M]
        t = (tau - t_start) * fs
        k = np.floor(t)
        alpha = t - k
        ok = (k >= 0) & (k <= k_n - 2) & (wrx > 0)
        rot = np.exp(2j * np.pi * fc * tau) if int(w.data_kind) == 0 else np.ones_like(tau)
        ki = np.where(ok, k, 0).astype(np.int64)
        w0 = np.where(ok, (1.0 - alpha) * rot, 0.0)
        w1 = np.where(ok, alpha * rot, 0.0)
        np.add.at(mat, (nn, q, mm, ki), w0)
        np.add.at(mat, (nn, q, mm, ki + 1), w1)
    return mat.reshape(n_n, q_n * m_n * k_n)


def das(w, y=None) -> np.ndarray:
    """x = W y, reshaped to [nx,ny,nz]."""
    y = w.y if y is None else y
    mat = dense_matrix(w)
    x = np.matmul(mat, np.asarray(y).astype(np.complex128).ravel())
    x = x.reshape(len(w.xs), len(w.ys), len(w.zs))
    return x if int(w.data_kind) == 0 else x.real
