"""Seeded synthetic inputs for the five DAS workloads of BASELINE.json.

This module is shared by the oracle tests and by the CUDA path's tests and
bench.  It holds *input synthesis only*: array geometry, transmit sets, voxel
axes and a point-scatterer echo simulator.  It contains none of the
beamformer's arithmetic (no interpolation, no apodization, no summation over
elements) and imports neither ``oracle`` nor ``paper_2606_13259_b200``.

The echo model is the one BASELINE.json's configs state (SURVEY.md 8(d.1),
readings A13-A16), standing in for the paper's Green's-function simulator
(Eq. 6-7), which the paper itself says does not affect the
performance measurements:

    y[q, m, k] = sum_s A_s * exp(-(t_k - tau)^2 / (2 sigma_t^2)) * exp(-j 2 pi fc tau)   (IQ)
    y[q, m, k] = sum_s A_s * exp(-(t_k - tau)^2 / (2 sigma_t^2)) * cos(2 pi fc (t_k - tau))  (RF)
    t_k = t_start + k / fs,   tau = tau_tx(q, s) + |s - e_m| / c,   sigma_t = 0.15 us

plus Gaussian noise of total standard deviation 0.01.  Echoes are evaluated
within +-6 sigma_t of their delay (beyond that the envelope is < 1.5e-8).

Everything handed to the beamformer is float32 (positions, axes, transmit
vectors, t0, samples): the oracle and the CUDA path see bit-identical inputs.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

TX_PLANE = 0
TX_DIVERGING = 1
DATA_IQ = 0
DATA_RF = 1

BASE_SEED = 20260612          # + config number
SIGMA_T = 0.15e-6             # echo envelope standard deviation [s]
NOISE_SIGMA = 0.01            # total (complex) noise standard deviation, reading A13
C0 = 1540.0
FC = 7.8e6
PITCH = 0.3e-3


@dataclasses.dataclass
class Workload:
    """One beamforming problem: exactly the values handed to the C ABI."""
    name: str
    elem_pos: np.ndarray            # [M,3] float32, metres
    tx_type: np.ndarray             # [Q] int32 (TX_PLANE / TX_DIVERGING)
    tx_v: np.ndarray                # [Q,3] float32: unit direction (plane) or virtual source (diverging)
    tx_t0: np.ndarray               # [Q] float32, seconds added to tau_tx
    xs: np.ndarray                  # [nx] float32
    ys: np.ndarray                  # [ny] float32
    zs: np.ndarray                  # [nz] float32
    c: float
    fc: float
    fs: float
    t_start: float
    f_number: float
    n_samples: int
    data_kind: int                  # DATA_IQ / DATA_RF
    y: Optional[np.ndarray]         # [Q,M,K] complex64 (IQ) or float32 (RF); None if generate_data=False
    scat_pos: np.ndarray            # [S,3] float64 (generator's truth, for tests)
    scat_amp: np.ndarray            # [S] float64
    elem_dir: Optional[np.ndarray] = None   # [M,3] float32 or None (= +z)
    seed: int = 0

    @property
    def n_elem(self) -> int:
        return int(self.elem_pos.shape[0])

    @property
    def n_tx(self) -> int:
        return int(self.tx_type.shape[0])

    @property
    def grid_shape(self):
        return (len(self.xs), len(self.ys), len(self.zs))

    @property
    def n_voxels(self) -> int:
        return len(self.xs) * len(self.ys) * len(self.zs)

    @property
    def nominal_accumulations(self) -> int:
        """N*M*Q."""
        return self.n_voxels * self.n_elem * self.n_tx


# --------------------------------------------------------------------------
# geometry
# --------------------------------------------------------------------------

def matrix_array(n_side: int, pitch: float = PITCH) -> np.ndarray:
    """n_side x n_side matrix array centred at the origin in the plane z=0.

    Element (i, j) sits at ((i-(n-1)/2) pitch, (j-(n-1)/2) pitch, 0) and has
    index m = i*n + j."""
    idx = np.arange(n_side, dtype=np.float64) - (n_side - 1) / 2.0
    ex, ey = np.meshgrid(idx * pitch, idx * pitch, indexing="ij")
    pos = np.stack([ex.ravel(), ey.ravel(), np.zeros(n_side * n_side)], axis=1)
    return pos.astype(np.float32)


def axis(lo: float, hi: float, n: int) -> np.ndarray:
    """linspace in double, then cast to float32."""
    return np.linspace(lo, hi, n, dtype=np.float64).astype(np.float32)


def plane_wave_set(angles_deg, elem_pos: np.ndarray, c: float):
    """Steered plane waves, u = (sin a, sin b, sqrt(1 - sin^2 a - sin^2 b)).

    t0 = -min_m(e_m . u)/c so that tau_tx = (r.u)/c minus its minimum over the
    element centres (config 2, reading A2)."""
    q = len(angles_deg)
    v = np.zeros((q, 3), dtype=np.float64)
    for i, (a, b) in enumerate(angles_deg):
        sa, sb = math.sin(math.radians(a)), math.sin(math.radians(b))
        v[i] = (sa, sb, math.sqrt(1.0 - sa * sa - sb * sb))
    v32 = v.astype(np.float32)
    # the minimum is taken with the float32 direction actually handed over
    proj = elem_pos.astype(np.float64) @ v32.astype(np.float64).T      # [M,Q]
    t0 = (-proj.min(axis=0) / c).astype(np.float32)
    return np.full(q, TX_PLANE, dtype=np.int32), v32, t0


def diverging_wave_set(sources: np.ndarray, c: float):
    """Diverging waves from virtual sources; t0 = -|v|/c (config 3, reading A2)."""
    v32 = np.asarray(sources, dtype=np.float64).astype(np.float32)
    t0 = (-np.linalg.norm(v32.astype(np.float64), axis=1) / c).astype(np.float32)
    return np.full(len(v32), TX_DIVERGING, dtype=np.int32), v32, t0


def _tx_delay(tx_type, tx_v, tx_t0, pts: np.ndarray, c: float) -> np.ndarray:
    """Forward-model transmit delay of each transmit at points pts [S,3] -> [Q,S] (seconds)."""
    v = tx_v.astype(np.float64)
    t0 = tx_t0.astype(np.float64)
    out = np.empty((len(tx_type), len(pts)), dtype=np.float64)
    for q, ty in enumerate(tx_type):
        if ty == TX_PLANE:
            out[q] = pts @ v[q] / c + t0[q]
        else:
            out[q] = np.linalg.norm(pts - v[q], axis=1) / c + t0[q]
    return out


# --------------------------------------------------------------------------
# echo simulator
# --------------------------------------------------------------------------

def simulate_channel_data(elem_pos, tx_type, tx_v, tx_t0, scat_pos, scat_amp, *, c, fc, fs,
                          t_start, n_samples, data_kind, noise_sigma, rng,
                          sigma_t: float = SIGMA_T) -> np.ndarray:
    """Point-scatterer echoes (+ noise) -> [Q,M,K] complex64 (IQ) or float32 (RF).

    Every element receives every echo (no directivity, no 1/r), reading A16."""
    q_n, m_n, k_n = len(tx_type), len(elem_pos), int(n_samples)
    e = elem_pos.astype(np.float64)
    s = np.asarray(scat_pos, dtype=np.float64).reshape(-1, 3)
    amp = np.asarray(scat_amp, dtype=np.float64).reshape(-1)
    iq = data_kind == DATA_IQ
    y = np.zeros((q_n, m_n, k_n), dtype=np.complex128 if iq else np.float64)
    half = int(math.ceil(6.0 * sigma_t * fs))
    offs = np.arange(-half, half + 1)
    if len(s):
        tau_tx = _tx_delay(tx_type, tx_v, tx_t0, s, c)                       # [Q,S]
        tau_rx = np.linalg.norm(s[None, :, :] - e[:, None, :], axis=2) / c    # [M,S]
        qq, mm = np.meshgrid(np.arange(q_n), np.arange(m_n), indexing="ij")
        for si in range(len(s)):
            tau = tau_tx[:, si][:, None] + tau_rx[:, si][None, :]             # [Q,M]
            kc = np.rint((tau - t_start) * fs).astype(np.int64)
            for o in offs:
                k = kc + o
                ok = (k >= 0) & (k < k_n)
                if not ok.any():
                    continue
                t = t_start + k / fs
                env = amp[si] * np.exp(-((t - tau) ** 2) / (2.0 * sigma_t * sigma_t))
                if iq:
                    val = env * np.exp(-2j * np.pi * fc * tau)
                else:
                    val = env * np.cos(2.0 * np.pi * fc * (t - tau))
                y[qq[ok], mm[ok], k[ok]] += val[ok]
    if noise_sigma > 0:
        if iq:
            sd = noise_sigma / math.sqrt(2.0)            # total complex std = noise_sigma (A13)
            y += rng.normal(0.0, sd, size=y.shape)
            y += 1j * rng.normal(0.0, sd, size=y.shape)
        else:
            y += rng.normal(0.0, noise_sigma, size=y.shape)
    return y.astype(np.complex64 if iq else np.float32)


def _draw_scatterers(rng, n, xs, ys, zs, shrink=0.10):
    """Uniform in the grid box shrunk by 10 % per side; draw order x, y, z."""
    def span(ax):
        lo, hi = float(ax[0]), float(ax[-1])
        d = (hi - lo) * shrink
        return lo + d, hi - d
    x = rng.uniform(*span(xs), size=n)
    y = rng.uniform(*span(ys), size=n)
    z = rng.uniform(*span(zs), size=n)
    return np.stack([x, y, z], axis=1)


# --------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------

def _headline_geometry():
    elem = matrix_array(32)
    g = np.array([-3e-3, -1e-3, 1e-3, 3e-3])
    src = np.array([[xv, yv, -10e-3] for xv in g for yv in g])     # q = 4*ix_v + iy_v
    tx_type, tx_v, tx_t0 = diverging_wave_set(src, C0)
    xs, ys, zs = axis(-4.8e-3, 4.8e-3, 128), axis(-4.8e-3, 4.8e-3, 128), axis(2e-3, 14e-3, 128)
    return elem, tx_type, tx_v, tx_t0, xs, ys, zs


def config(number: int, *, generate_data: bool = True, grid: Optional[tuple] = None,
           noise: bool = True) -> Workload:
    """Build config ``number`` (1..5) of BASELINE.json.

    ``grid=(nx,ny,nz)`` overrides the voxel counts (same physical extent) for
    reduced test cases; ``noise=False`` drops the noise term."""
    seed = BASE_SEED + number
    rng = np.random.default_rng(seed)
    sig = NOISE_SIGMA if noise else 0.0
    if number == 1:
        elem = matrix_array(8)
        tx_type = np.array([TX_PLANE], dtype=np.int32)
        tx_v = np.array([[0.0, 0.0, 1.0]], dtype=np.float32)
        tx_t0 = np.zeros(1, dtype=np.float32)
        n = grid or (32, 32, 32)
        xs, ys, zs = axis(-2.4e-3, 2.4e-3, n[0]), axis(-2.4e-3, 2.4e-3, n[1]), axis(3e-3, 9e-3, n[2])
        fs, k_n, kind, n_sc = 15.6e6, 256, DATA_IQ, 3
        pos = _draw_scatterers(rng, n_sc, xs, ys, zs)
        amp = rng.uniform(0.5, 1.0, size=n_sc)
        name = "tiny"
    elif number == 2:
        elem = matrix_array(16)
        ang = [(0, 0), (5, 0), (-5, 0), (0, 5), (0, -5)]
        tx_type, tx_v, tx_t0 = plane_wave_set(ang, elem, C0)
        n = grid or (64, 64, 64)
        xs, ys, zs = axis(-2.4e-3, 2.4e-3, n[0]), axis(-2.4e-3, 2.4e-3, n[1]), axis(2e-3, 12e-3, n[2])
        fs, k_n, kind, n_sc = 15.6e6, 512, DATA_IQ, 10
        pos = _draw_scatterers(rng, n_sc, xs, ys, zs)
        amp = rng.uniform(0.5, 1.0, size=n_sc)            # reading A14
        name = "small_multi_angle"
    elif number in (3, 4, 5):
        elem, tx_type, tx_v, tx_t0, xs, ys, zs = _headline_geometry()
        if grid:
            xs, ys, zs = (axis(-4.8e-3, 4.8e-3, grid[0]), axis(-4.8e-3, 4.8e-3, grid[1]),
                          axis(2e-3, 14e-3, grid[2]))
        n_sc = 50
        # configs 3 and 4 share their scatterers ("same scatterers as 3"): seeded from config 3
        srng = np.random.default_rng(BASE_SEED + 3) if number == 4 else rng
        pos = _draw_scatterers(srng, n_sc, xs, ys, zs)
        amp = 10.0 ** (-2.0 * srng.uniform(0.0, 1.0, size=n_sc))     # 40 dB log-uniform
        if number == 4:
            fs, k_n, kind, name = 31.2e6, 2048, DATA_RF, "rf_headline"
        elif number == 3:
            fs, k_n, kind, name = 15.6e6, 1024, DATA_IQ, "headline"
        else:
            fs, k_n, kind, name = 15.6e6, 1024, DATA_IQ, "streaming_frame0"
            # reading A15: 50 movers (headline amplitude law) + 50 static clutter at +20 dB
            cpos = _draw_scatterers(rng, 50, xs, ys, zs)
            camp = 10.0 * 10.0 ** (-2.0 * rng.uniform(0.0, 1.0, size=50))
            pos = np.concatenate([pos, cpos])
            amp = np.concatenate([amp, camp])
    else:
        raise ValueError("config number must be 1..5")
    y = None
    if generate_data:
        y = simulate_channel_data(elem, tx_type, tx_v, tx_t0, pos, amp, c=C0, fc=FC, fs=fs,
                                  t_start=0.0, n_samples=k_n, data_kind=kind,
                                  noise_sigma=sig, rng=rng)
    return Workload(name=name, elem_pos=elem, tx_type=tx_type, tx_v=tx_v, tx_t0=tx_t0, xs=xs, ys=ys,
                    zs=zs, c=C0, fc=(FC if kind == DATA_IQ else 0.0), fs=fs, t_start=0.0,
                    f_number=1.0, n_samples=k_n, data_kind=kind, y=y, scat_pos=pos, scat_amp=amp,
                    seed=seed)


def streaming_frames(n_frames: int = 64, *, grid: Optional[tuple] = None, sigma_walk: float = 5e-6):
    """Config 5: generator of ``n_frames`` Workloads sharing geometry.

    The first 50 scatterers move by an N(0, (5 um)^2) random walk per axis per
    frame; the last 50 (clutter, +20 dB) are static (reading A15)."""
    base = config(5, generate_data=False, grid=grid)
    rng = np.random.default_rng(base.seed + 1000)
    pos = base.scat_pos.copy()
    for f in range(n_frames):
        if f:
            pos[:50] += rng.normal(0.0, sigma_walk, size=(50, 3))
        y = simulate_channel_data(base.elem_pos, base.tx_type, base.tx_v, base.tx_t0, pos,
                                  base.scat_amp, c=base.c, fc=FC, fs=base.fs, t_start=0.0,
                                  n_samples=base.n_samples, data_kind=DATA_IQ,
                                  noise_sigma=NOISE_SIGMA, rng=rng)
        yield dataclasses.replace(base, name=f"streaming_frame{f}", y=y, scat_pos=pos.copy())


def custom(elem_pos, tx_type, tx_v, tx_t0, xs, ys, zs, *, fs, n_samples, data_kind=DATA_IQ,
           c=C0, fc=FC, t_start=0.0, f_number=1.0, scat_pos=(), scat_amp=(), noise_sigma=0.0,
           seed=0, y=None, elem_dir=None, name="custom") -> Workload:
    """Assemble an arbitrary Workload (tests); simulates echoes unless ``y`` is given."""
    elem_pos = np.ascontiguousarray(elem_pos, dtype=np.float32).reshape(-1, 3)
    tx_type = np.ascontiguousarray(tx_type, dtype=np.int32).reshape(-1)
    tx_v = np.ascontiguousarray(tx_v, dtype=np.float32).reshape(-1, 3)
    tx_t0 = np.ascontiguousarray(tx_t0, dtype=np.float32).reshape(-1)
    xs, ys, zs = (np.ascontiguousarray(a, dtype=np.float32).reshape(-1) for a in (xs, ys, zs))
    scat_pos = np.asarray(scat_pos, dtype=np.float64).reshape(-1, 3)
    scat_amp = np.asarray(scat_amp, dtype=np.float64).reshape(-1)
    t_start32 = float(np.float32(t_start))
    if y is None:
        rng = np.random.default_rng(seed)
        y = simulate_channel_data(elem_pos, tx_type, tx_v, tx_t0, scat_pos, scat_amp, c=c,
                                  fc=fc if data_kind == DATA_IQ else FC, fs=fs, t_start=t_start32,
                                  n_samples=n_samples, data_kind=data_kind,
                                  noise_sigma=noise_sigma, rng=rng)
    if elem_dir is not None:
        elem_dir = np.ascontiguousarray(elem_dir, dtype=np.float32).reshape(-1, 3)
    return Workload(name=name, elem_pos=elem_pos, tx_type=tx_type, tx_v=tx_v, tx_t0=tx_t0, xs=xs,
                    ys=ys, zs=zs, c=float(c), fc=float(fc if data_kind == DATA_IQ else 0.0),
                    fs=float(fs), t_start=t_start32, f_number=float(f_number),
                    n_samples=int(n_samples), data_kind=int(data_kind), y=y, scat_pos=scat_pos,
                    scat_amp=scat_amp, elem_dir=elem_dir, seed=seed)
