"""Thin Python binding of libdas_b200.so (include/das.h) -- argument marshalling only.

Every step of the hot path (layout transform + cast, delays, aperture, gather, interpolation,
rotation, accumulation) runs in the CUDA kernels behind the C ABI.  PyTorch is used by callers
for device memory and streams only; this module passes raw device pointers through ctypes.

There is no CPU fallback: if the shared library cannot be built or loaded, ``load()`` raises.
This package never imports ``oracle``.

    plan = das.Plan(elem_pos, tx_type, tx_v, tx_t0, xs, ys, zs, c=..., fc=..., fs=..., ...)
    plan.convert(raw_dev_ptr, conv_dev_ptr, stream=0)        # das_convert
    plan.execute(conv_dev_ptr, out_dev_ptr, stream=0)        # das_execute
    plan.beamform_host(raw_host_ptr, out_host_ptr, stream=0) # das_beamform_host
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

from . import _build

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_ALLOC, ERR_CUDA, ERR_SIZE = range(6)
TX_PLANE, TX_DIVERGING = 0, 1
DATA_IQ, DATA_RF = 0, 1
STORE_FP32, STORE_FP16, STORE_FP8 = 0, 1, 2
ALGO_AUTO, ALGO_GENERAL, ALGO_TILED, ALGO_TC = 0, 1, 2, 3
WINDOW_BOXCAR, WINDOW_HANN, WINDOW_TUKEY = 0, 1, 2
INTERP_LINEAR, INTERP_CUBIC = 0, 1
STATIC_SCRATCH_BYTES = 16 << 20        # DAS_STATIC_SCRATCH_BYTES of include/das.h

# every symbol include/das.h declares (checked against the header by tests/test_abi.py)
EXPORTS = ("das_plan_create", "das_plan_destroy", "das_raw_bytes", "das_converted_bytes",
           "das_output_bytes", "das_plan_algo", "das_plan_frames", "das_convert", "das_execute", "das_beamform_host",
           "das_beamform_host_begin", "das_beamform_host_wait", "das_beamform_static",
           "das_plan_count_work", "das_status_string", "das_last_error", "das_launch_count")


class Transmit(ctypes.Structure):
    _fields_ = [("type", ctypes.c_int), ("v", ctypes.c_float * 3), ("t0", ctypes.c_float)]


class PlanDesc(ctypes.Structure):
    _fields_ = [
        ("elem_pos", ctypes.POINTER(ctypes.c_float)), ("n_elem", ctypes.c_int),
        ("elem_dir", ctypes.POINTER(ctypes.c_float)),
        ("tx", ctypes.POINTER(Transmit)), ("n_tx", ctypes.c_int),
        ("xs", ctypes.POINTER(ctypes.c_float)), ("nx", ctypes.c_int),
        ("ys", ctypes.POINTER(ctypes.c_float)), ("ny", ctypes.c_int),
        ("zs", ctypes.POINTER(ctypes.c_float)), ("nz", ctypes.c_int),
        ("c", ctypes.c_float), ("fc", ctypes.c_float), ("fs", ctypes.c_float),
        ("t_start", ctypes.c_float), ("f_number", ctypes.c_float),
        ("n_samples", ctypes.c_int), ("data_kind", ctypes.c_int), ("storage", ctypes.c_int),
        ("algo", ctypes.c_int), ("device", ctypes.c_int), ("n_frames", ctypes.c_int),
        ("tau_tx", ctypes.POINTER(ctypes.c_float)), ("w_tx", ctypes.POINTER(ctypes.c_float)),
        ("obs_off", ctypes.POINTER(ctypes.c_longlong)), ("obs_q", ctypes.POINTER(ctypes.c_int)),
        ("vox_pos", ctypes.POINTER(ctypes.c_float)),
        ("window", ctypes.c_int), ("window_param", ctypes.c_float), ("interp", ctypes.c_int),
        ("debug_tiled_grid", ctypes.c_int), ("debug_tc_pace", ctypes.c_int),
    ]


class DasError(RuntimeError):
    def __init__(self, status: int, detail: str):
        self.status = status
        super().__init__(f"{status_string(status)}: {detail}")


_lib = None


def library_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = True):
    """Load libdas_b200.so (building it with nvcc first if it is missing or stale).
    Raises if that is impossible: there is no other implementation to fall back to."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and _build.needs_build():
        _build.build()
    if not os.path.exists(_build.LIB):
        raise RuntimeError(f"{_build.LIB} is missing and could not be built; "
                           "the DAS beamformer has no CPU fallback")
    lib = ctypes.CDLL(_build.LIB)
    vp, sz = ctypes.c_void_p, ctypes.c_size_t
    lib.das_plan_create.restype = ctypes.c_int
    lib.das_plan_create.argtypes = [ctypes.POINTER(PlanDesc), ctypes.POINTER(vp)]
    lib.das_plan_destroy.restype = ctypes.c_int
    lib.das_plan_destroy.argtypes = [vp]
    for name in ("das_raw_bytes", "das_converted_bytes", "das_output_bytes"):
        getattr(lib, name).restype = sz
        getattr(lib, name).argtypes = [vp]
    lib.das_plan_algo.restype = ctypes.c_int
    lib.das_plan_algo.argtypes = [vp]
    lib.das_plan_frames.restype = ctypes.c_int
    lib.das_plan_frames.argtypes = [vp]
    lib.das_convert.restype = ctypes.c_int
    lib.das_convert.argtypes = [vp, vp, vp, ctypes.c_float, vp]
    lib.das_execute.restype = ctypes.c_int
    lib.das_execute.argtypes = [vp, vp, vp, vp]
    lib.das_beamform_host.restype = ctypes.c_int
    lib.das_beamform_host.argtypes = [vp, vp, vp, vp]
    lib.das_beamform_host_begin.restype = ctypes.c_int
    lib.das_beamform_host_begin.argtypes = [vp, vp, vp, vp]
    lib.das_beamform_host_wait.restype = ctypes.c_int
    lib.das_beamform_host_wait.argtypes = [vp]
    lib.das_beamform_static.restype = ctypes.c_int
    lib.das_beamform_static.argtypes = [vp, vp, vp, ctypes.c_float, vp]
    lib.das_plan_count_work.restype = ctypes.c_int
    lib.das_plan_count_work.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong), ctypes.POINTER(ctypes.c_ulonglong)]
    lib.das_status_string.restype = ctypes.c_char_p
    lib.das_status_string.argtypes = [ctypes.c_int]
    lib.das_last_error.restype = ctypes.c_char_p
    lib.das_last_error.argtypes = []
    lib.das_launch_count.restype = ctypes.c_ulonglong
    lib.das_launch_count.argtypes = []
    _lib = lib
    return lib


def status_string(status: int) -> str:
    return load().das_status_string(int(status)).decode()


def last_error() -> str:
    return load().das_last_error().decode()


def launch_count() -> int:
    return int(load().das_launch_count())


def _check(status: int):
    if status != OK:
        raise DasError(status, last_error())


def _f32(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a if shape is None else a.reshape(shape)


class Plan:
    """das_plan_t wrapper.  Arrays are host numpy arrays (copied by the library)."""

    def __init__(self, elem_pos, tx_type, tx_v, tx_t0, xs, ys, zs, *, c, fc, fs, t_start=0.0,
                 f_number=1.0, n_samples, data_kind=DATA_IQ, storage=STORE_FP32, algo=ALGO_AUTO,
                 device=0, elem_dir=None, n_frames=0, tau_tx=None, w_tx=None, obs=None, vox_pos=None,
                 window=WINDOW_BOXCAR, window_param=0.5, interp=INTERP_LINEAR, debug_tiled_grid=0, debug_tc_pace=0):
        lib = load()
        self._lib = lib
        self._h = ctypes.c_void_p()
        elem_pos = _f32(elem_pos, (-1, 3))
        tx_v = _f32(tx_v, (-1, 3))
        tx_t0 = _f32(tx_t0, (-1,))
        tx_type = np.ascontiguousarray(tx_type, dtype=np.int32).reshape(-1)
        if vox_pos is not None:
            vox_pos = _f32(vox_pos, (-1, 3))
            xs, ys, zs = np.zeros(len(vox_pos), np.float32), np.zeros(1, np.float32), np.zeros(1, np.float32)
        xs, ys, zs = _f32(xs, (-1,)), _f32(ys, (-1,)), _f32(zs, (-1,))
        edir = None if elem_dir is None else _f32(elem_dir, (-1, 3))
        txs = (Transmit * len(tx_type))()
        for q in range(len(tx_type)):
            txs[q].type = int(tx_type[q])
            txs[q].v[:] = [float(v) for v in tx_v[q]]
            txs[q].t0 = float(tx_t0[q])
        fp = ctypes.POINTER(ctypes.c_float)
        d = PlanDesc()
        d.elem_pos, d.n_elem = elem_pos.ctypes.data_as(fp), len(elem_pos)
        d.elem_dir = edir.ctypes.data_as(fp) if edir is not None else None
        d.tx, d.n_tx = txs, len(tx_type)
        d.xs, d.nx = xs.ctypes.data_as(fp), len(xs)
        d.ys, d.ny = ys.ctypes.data_as(fp), len(ys)
        d.zs, d.nz = zs.ctypes.data_as(fp), len(zs)
        d.c, d.fc, d.fs, d.t_start, d.f_number = float(c), float(fc), float(fs), float(t_start), float(f_number)
        d.n_samples, d.data_kind, d.storage = int(n_samples), int(data_kind), int(storage)
        d.algo, d.device, d.n_frames = int(algo), int(device), int(n_frames)
        n_vox = len(xs) * len(ys) * len(zs)
        keep = []
        if tau_tx is not None:
            tau_tx = _f32(tau_tx, (len(tx_type), n_vox)); d.tau_tx = tau_tx.ctypes.data_as(fp); keep.append(tau_tx)
        if w_tx is not None:
            w_tx = _f32(w_tx, (len(tx_type), n_vox)); d.w_tx = w_tx.ctypes.data_as(fp); keep.append(w_tx)
        if obs is not None:
            off = np.ascontiguousarray(obs[0], dtype=np.int64).reshape(-1)
            oq = np.ascontiguousarray(obs[1], dtype=np.int32).reshape(-1)
            if len(off) != n_vox + 1 or int(off[-1]) != len(oq):
                raise ValueError("malformed observation lists")
            oq = oq if len(oq) else np.zeros(1, np.int32)
            d.obs_off = off.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong))
            d.obs_q = oq.ctypes.data_as(ctypes.POINTER(ctypes.c_int))
            keep += [off, oq]
        if vox_pos is not None:
            d.vox_pos = vox_pos.ctypes.data_as(fp); keep.append(vox_pos)
        d.window, d.window_param, d.interp = int(window), float(window_param), int(interp)
        d.debug_tiled_grid, d.debug_tc_pace = int(debug_tiled_grid), int(debug_tc_pace)
        self.desc = d
        _check(lib.das_plan_create(ctypes.byref(d), ctypes.byref(self._h)))
        self.grid_shape = (len(xs), len(ys), len(zs))
        self.data_kind, self.storage, self.device = int(data_kind), int(storage), int(device)
        self.n_tx, self.n_elem, self.n_samples = len(tx_type), len(elem_pos), int(n_samples)

    @classmethod
    def from_workload(cls, w, *, storage=STORE_FP32, algo=ALGO_AUTO, device=0, n_frames=0, **options):
        """Plan for a ``workloads.Workload``-shaped object (duck-typed); ``options`` are the keyword
        arguments of the paper's general interface (tau_tx, w_tx, obs, vox_pos, window, window_param, interp) and
        the debugging aids of das.h (debug_tiled_grid, debug_tc_pace)."""
        return cls(w.elem_pos, w.tx_type, w.tx_v, w.tx_t0, w.xs, w.ys, w.zs, c=w.c, fc=w.fc, fs=w.fs,
                   t_start=w.t_start, f_number=w.f_number, n_samples=w.n_samples,
                   data_kind=w.data_kind, storage=storage, algo=algo, device=device,
                   elem_dir=getattr(w, "elem_dir", None), n_frames=n_frames, **options)

    # sizes -------------------------------------------------------------------------------
    @property
    def raw_bytes(self) -> int:
        return int(self._lib.das_raw_bytes(self._h))

    @property
    def converted_bytes(self) -> int:
        return int(self._lib.das_converted_bytes(self._h))

    @property
    def output_bytes(self) -> int:
        return int(self._lib.das_output_bytes(self._h))

    @property
    def algo(self) -> int:
        return int(self._lib.das_plan_algo(self._h))

    @property
    def frames(self) -> int:
        return int(self._lib.das_plan_frames(self._h))

    # calls -------------------------------------------------------------------------------
    def convert(self, d_raw: int, d_conv: int, scale: float = 1.0, stream: int = 0):
        _check(self._lib.das_convert(self._h, ctypes.c_void_p(d_raw), ctypes.c_void_p(d_conv),
                                     ctypes.c_float(scale), ctypes.c_void_p(stream)))

    def execute(self, d_conv: int, d_out: int, stream: int = 0):
        _check(self._lib.das_execute(self._h, ctypes.c_void_p(d_conv), ctypes.c_void_p(d_out),
                                     ctypes.c_void_p(stream)))

    def beamform_host(self, h_raw: int, h_out: int, stream: int = 0):
        _check(self._lib.das_beamform_host(self._h, ctypes.c_void_p(h_raw), ctypes.c_void_p(h_out),
                                           ctypes.c_void_p(stream)))

    def beamform_host_begin(self, h_raw: int, h_out: int, stream: int = 0):
        _check(self._lib.das_beamform_host_begin(self._h, ctypes.c_void_p(h_raw), ctypes.c_void_p(h_out),
                                                 ctypes.c_void_p(stream)))

    def beamform_host_wait(self):
        _check(self._lib.das_beamform_host_wait(self._h))

    def beamform_static(self, d_raw: int, d_out: int, scale: float = 1.0, stream: int = 0):
        """das_beamform_static: das_convert + das_execute through the library's built-in 16 MiB scratch array,
        for callers that cannot allocate device memory (include/das.h).  Device pointers in, nothing allocated."""
        _check(self._lib.das_beamform_static(self._h, ctypes.c_void_p(d_raw), ctypes.c_void_p(d_out),
                                             ctypes.c_float(scale), ctypes.c_void_p(stream)))

    def count_work(self):
        """(n_pairs, n_terms) of das_plan_count_work: active (m, n) pairs and entered (q, m, n) terms."""
        a, b = ctypes.c_ulonglong(), ctypes.c_ulonglong()
        _check(self._lib.das_plan_count_work(self._h, ctypes.byref(a), ctypes.byref(b)))
        return int(a.value), int(b.value)

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.das_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()


def beamform_torch(plan: Plan, raw, *, stream=None, conv=None, out=None):
    """Convenience for tests/bench: ``raw`` is a CUDA torch tensor holding [Q,M,K] (one frame) or
    [B,Q,M,K] (a plan with n_frames = B) complex64 (IQ) or float32 (RF).  Allocates (or reuses) the converted and output tensors with torch, then
    calls das_convert + das_execute with their raw pointers on torch's current stream."""
    import torch
    assert raw.is_cuda and raw.is_contiguous()
    s = torch.cuda.current_stream(raw.device) if stream is None else stream
    if conv is None:
        conv = torch.empty(plan.converted_bytes, dtype=torch.uint8, device=raw.device)
    if out is None:
        dt = torch.complex64 if plan.data_kind == DATA_IQ else torch.float32
        shape = plan.grid_shape if plan.frames == 1 else (plan.frames,) + tuple(plan.grid_shape)
        out = torch.empty(shape, dtype=dt, device=raw.device)
    plan.convert(raw.data_ptr(), conv.data_ptr(), 1.0, s.cuda_stream)
    plan.execute(conv.data_ptr(), out.data_ptr(), s.cuda_stream)
    return out, conv
