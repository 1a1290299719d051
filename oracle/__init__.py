"""CPU oracle for volumetric delay-and-sum -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It never imports paper_2606_13259_b200 and shares nothing with it.

``das(workload)`` evaluates the plain definition (oracle/das_oracle.c, double precision;
SURVEY.md 8(c.1); Eq. 1-2 + linear interpolation; Algorithm 1 loop order)
for a ``workloads.Workload``-shaped object (duck-typed: only attributes are read).
``oracle.brute`` is an independent dense-matrix formulation used to pin it on tiny grids.
"""
from __future__ import annotations

import ctypes
from typing import Optional

import numpy as np

from . import build as _build

_lib = None

WINDOWS = {"boxcar": 0, "hann": 1, "tukey": 2}
INTERPS = {"linear": 0, "cubic": 1}


class _Opts(ctypes.Structure):
    """das_oracle_opts of das_oracle.c."""
    _fields_ = [("tau_tx_tab", ctypes.POINTER(ctypes.c_float)), ("w_tx_tab", ctypes.POINTER(ctypes.c_float)),
                ("obs_off", ctypes.POINTER(ctypes.c_longlong)), ("obs_q", ctypes.POINTER(ctypes.c_int)),
                ("vox_pos", ctypes.POINTER(ctypes.c_float)), ("window", ctypes.c_int),
                ("window_param", ctypes.c_float), ("interp", ctypes.c_int)]


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        f32p = ctypes.POINTER(ctypes.c_float)
        i32p = ctypes.POINTER(ctypes.c_int)
        i64p = ctypes.POINTER(ctypes.c_longlong)
        f64p = ctypes.POINTER(ctypes.c_double)
        lib.das_oracle.restype = ctypes.c_int
        lib.das_oracle.argtypes = [
            f32p, f32p, ctypes.c_int, i32p, f32p, f32p, ctypes.c_int,
            f32p, ctypes.c_int, f32p, ctypes.c_int, f32p, ctypes.c_int,
            ctypes.c_float, ctypes.c_float, ctypes.c_float, ctypes.c_float, ctypes.c_float,
            ctypes.c_int, ctypes.c_int, f32p, i64p, ctypes.c_longlong,
            f64p, i64p, f64p, f64p, ctypes.c_double]
        lib.das_oracle_ex.restype = ctypes.c_int
        lib.das_oracle_ex.argtypes = lib.das_oracle.argtypes + [ctypes.POINTER(_Opts)]
        lib.das_oracle_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def threads() -> int:
    """Number of OpenMP threads the oracle will use."""
    return int(_load().das_oracle_threads())


def _p(a, ty):
    return a.ctypes.data_as(ctypes.POINTER(ty)) if a is not None else None


def das(w, *, y=None, voxels: Optional[np.ndarray] = None, want_count=False, want_l1=False,
        want_slack=False, slack_rel: float = 1e-6, tau_tx=None, w_tx=None, obs=None, vox_pos=None,
        window: str = "boxcar", window_param: float = 0.5, interp: str = "linear"):
    """Oracle DAS of workload ``w`` (optionally with replacement channel data ``y``).

    Returns the full volume [nx,ny,nz] (complex128 for IQ, float64 for RF), or, when
    ``voxels`` (flat indices (ix*ny+iy)*nz+iz) is given, a 1-D array over those voxels.
    With want_* flags returns a dict {"out", "count", "l1", "slack"}.

    Options of the paper's general interface (das_oracle.c header): ``tau_tx`` / ``w_tx`` tables
    [Q, N] (N = number of voxels, flat order), ``obs`` = (obs_off[N+1], obs_q[]) CSR observation
    lists, ``vox_pos`` [N,3] an arbitrary voxel list (output then has shape [N,1,1]), ``window`` in
    WINDOWS with the Tukey taper ``window_param``, ``interp`` in INTERPS."""
    lib = _load()
    y = w.y if y is None else y
    iq = int(w.data_kind) == 0
    y = np.ascontiguousarray(y, dtype=np.complex64 if iq else np.float32)
    q_n, m_n, k_n = len(w.tx_type), len(w.elem_pos), int(w.n_samples)
    if y.shape != (q_n, m_n, k_n):
        raise ValueError(f"y has shape {y.shape}, expected {(q_n, m_n, k_n)}")
    elem = np.ascontiguousarray(w.elem_pos, dtype=np.float32)
    edir = None if getattr(w, "elem_dir", None) is None else np.ascontiguousarray(w.elem_dir, dtype=np.float32)
    ttype = np.ascontiguousarray(w.tx_type, dtype=np.int32)
    tv = np.ascontiguousarray(w.tx_v, dtype=np.float32)
    t0 = np.ascontiguousarray(w.tx_t0, dtype=np.float32)
    xs, ys, zs = (np.ascontiguousarray(a, dtype=np.float32) for a in (w.xs, w.ys, w.zs))
    opts = _Opts()
    keep = []
    if vox_pos is not None:
        vp = np.ascontiguousarray(vox_pos, dtype=np.float32).reshape(-1, 3)
        xs, ys, zs = np.zeros(len(vp), np.float32), np.zeros(1, np.float32), np.zeros(1, np.float32)
        opts.vox_pos = _p(vp, ctypes.c_float)
        keep.append(vp)
    n_tot = len(xs) * len(ys) * len(zs)
    for name, tab in (("tau_tx_tab", tau_tx), ("w_tx_tab", w_tx)):
        if tab is not None:
            t = np.ascontiguousarray(tab, dtype=np.float32).reshape(q_n, n_tot)
            setattr(opts, name, _p(t, ctypes.c_float))
            keep.append(t)
    if obs is not None:
        off = np.ascontiguousarray(obs[0], dtype=np.int64).reshape(-1)
        oq = np.ascontiguousarray(obs[1], dtype=np.int32).reshape(-1)
        if len(off) != n_tot + 1 or off[0] != 0 or off[-1] != len(oq) or np.any(np.diff(off) < 0):
            raise ValueError("malformed observation lists")
        oq = oq if len(oq) else np.zeros(1, np.int32)
        opts.obs_off, opts.obs_q = _p(off, ctypes.c_longlong), _p(oq, ctypes.c_int)
        keep += [off, oq]
    opts.window, opts.window_param, opts.interp = WINDOWS[window], float(window_param), INTERPS[interp]
    if voxels is None:
        vox, n_eval = None, len(xs) * len(ys) * len(zs)
    else:
        vox = np.ascontiguousarray(voxels, dtype=np.int64).reshape(-1)
        n_eval = len(vox)
    out = np.zeros(n_eval * (2 if iq else 1), dtype=np.float64)
    cnt = np.zeros(n_eval, dtype=np.int64) if want_count else None
    l1 = np.zeros(n_eval, dtype=np.float64) if want_l1 else None
    slack = np.zeros(n_eval, dtype=np.float64) if want_slack else None
    yf = y.view(np.float32)
    rc = lib.das_oracle_ex(
        _p(elem, ctypes.c_float), _p(edir, ctypes.c_float), m_n,
        _p(ttype, ctypes.c_int), _p(tv, ctypes.c_float), _p(t0, ctypes.c_float), q_n,
        _p(xs, ctypes.c_float), len(xs), _p(ys, ctypes.c_float), len(ys), _p(zs, ctypes.c_float), len(zs),
        float(w.c), float(w.fc), float(w.fs), float(w.t_start), float(w.f_number),
        k_n, int(w.data_kind), _p(yf, ctypes.c_float),
        _p(vox, ctypes.c_longlong), n_eval,
        _p(out, ctypes.c_double), _p(cnt, ctypes.c_longlong), _p(l1, ctypes.c_double),
        _p(slack, ctypes.c_double), float(slack_rel), ctypes.byref(opts))
    if rc != 0:
        raise ValueError("das_oracle rejected its arguments")
    res = out.view(np.complex128) if iq else out
    if voxels is None:
        res = res.reshape(len(xs), len(ys), len(zs))
        shape = res.shape
    else:
        shape = (n_eval,)
    if not (want_count or want_l1 or want_slack):
        return res
    return {"out": res,
            "count": None if cnt is None else cnt.reshape(shape),
            "l1": None if l1 is None else l1.reshape(shape),
            "slack": None if slack is None else slack.reshape(shape)}
