"""Gradient waveforms, gradient amplitudes and direction sets (inputs of rms_run).

The waveform is the unit-less shape w_m[i] of the gradient at step i = 1..n_steps; the
amplitude `gamp` (rad / (ms um)) multiplies it.  These are arguments of the method
(Table 1 "Diffusion gradient g(tau)", line 195), not part of it.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


def pgse_wave(n_steps: int, n_delta: int, n_Delta: int) -> np.ndarray:
    """Pulsed-gradient spin echo shape: +1 on steps 1..n_delta, -1 on n_Delta+1..n_Delta+n_delta."""
    if n_delta < 0 or n_Delta < n_delta or n_Delta + n_delta > n_steps:
        raise ValueError("PGSE lobes do not fit: need n_delta <= n_Delta and n_Delta + n_delta <= n_steps")
    w = np.zeros(n_steps, dtype=np.float32)
    w[:n_delta] = 1.0
    w[n_Delta:n_Delta + n_delta] = -1.0
    return w


def pgse_gamp(b, delta_ms: float, Delta_ms: float) -> np.ndarray:
    """Gradient amplitude for a nominal b-value: b = g^2 delta^2 (Delta - delta/3)."""
    b = np.atleast_1d(np.asarray(b, dtype=np.float64))
    return np.sqrt(b / (delta_ms ** 2 * (Delta_ms - delta_ms / 3.0)))


def one_hot_wave(n_steps: int, at_step: int) -> np.ndarray:
    """Narrow-pulse limit: all weight on one step, so the phase is q . (x(at_step) - x(0))."""
    w = np.zeros(n_steps, dtype=np.float32)
    w[at_step - 1] = 1.0
    return w


def fibonacci_dirs(n: int) -> np.ndarray:
    """n unit vectors on a Fibonacci sphere: z_j = 1 - (2j+1)/n, phi_j = j pi (3 - sqrt 5)."""
    j = np.arange(n, dtype=np.float64)
    z = 1.0 - (2.0 * j + 1.0) / n
    phi = j * np.pi * (3.0 - np.sqrt(5.0))
    rho = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    d = np.stack([rho * np.cos(phi), rho * np.sin(phi), z], axis=1)
    return d / np.linalg.norm(d, axis=1, keepdims=True)


@dataclass
class Sequence:
    """All rms_run arguments that describe the measurement."""
    dt_ms: float
    n_steps: int
    wave: np.ndarray            # [n_wave, n_steps] float32
    gamp: np.ndarray            # [n_wave, n_g] float64, rad/(ms um)
    dirs: np.ndarray            # [n_dir, 3] float64 unit vectors
    snap_steps: np.ndarray      # [n_snap] int64, ascending, 1-based
    b_nominal: np.ndarray = field(default_factory=lambda: np.zeros(0))  # [n_g] ms/um^2, for reports
    delta_ms: float = 0.0
    Delta_ms: float = 0.0
    mix_first_step: int = 0     # stimulated echo: steps mix_first_step .. mix_first_step + mix_n_steps - 1 (1-based) are the
    mix_n_steps: int = 0        # mixing time, relaxing with T1 instead of T2 (0 steps: none)
    tensor_waves: np.ndarray | None = None   # [n_tensor, 3] int32: scalar waveform on gradient axis x, y, z (-1: off)
    tensor_gamp: np.ndarray | None = None    # [n_tensor, n_g] float64, rad/(ms um)
    rots: np.ndarray | None = None           # [n_rot, 3, 3] float64: g_lab = R g


def pgse_sequence(dt_ms: float, n_steps: int, delta_ms: float, Delta_ms: float, b, dirs, snap_steps=None) -> Sequence:
    n_delta = int(round(delta_ms / dt_ms))
    n_Delta = int(round(Delta_ms / dt_ms))
    wave = pgse_wave(n_steps, n_delta, n_Delta)[None, :]
    b = np.atleast_1d(np.asarray(b, dtype=np.float64))
    gamp = pgse_gamp(b, n_delta * dt_ms, n_Delta * dt_ms)[None, :]
    if snap_steps is None:
        snap_steps = [n_steps]
    return Sequence(dt_ms=dt_ms, n_steps=n_steps, wave=np.ascontiguousarray(wave, dtype=np.float32),
                    gamp=np.ascontiguousarray(gamp), dirs=np.ascontiguousarray(dirs, dtype=np.float64),
                    snap_steps=np.asarray(snap_steps, dtype=np.int64), b_nominal=b,
                    delta_ms=n_delta * dt_ms, Delta_ms=n_Delta * dt_ms)
