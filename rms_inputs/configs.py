"""The five workloads of BASELINE.json:configs (0-indexed cfg0..cfg4) as seeded synthetic inputs.

`scale="full"` is the size BASELINE.json names; `scale="test"` is a reduced copy with the same
structure (same radii / density / step length, smaller box, fewer walkers and steps) that the CPU
oracle finishes in seconds.  Readings of what BASELINE.json leaves open are listed in DESIGN.md.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import substrates as S
from .sequences import Sequence, fibonacci_dirs, pgse_sequence

CONFIG_NAMES = ("cfg0", "cfg1", "cfg2", "cfg3", "cfg4")

DT = 2e-4  # ms, all configs


@dataclass
class Config:
    name: str
    scale: str
    substrate: S.Substrate
    sequence: Sequence
    n_walkers: int
    seed: int


def _axes(n):
    return np.eye(3)[:n]


def make_config(name: str, scale: str = "full", **over) -> Config:
    full = scale == "full"
    if name == "cfg0":
        # single impermeable cylinder r = 1 um in 32^3, walkers inside, delta = Delta = 0.1 ms, dirs x and z
        sub = S.single_cylinder(32, 10.0, 0.1, D_extra=2.0, D_intra=2.0, place="intra")
        n_steps = 1000
        dirs = np.array([[1.0, 0.0, 0.0], [0.0, 0.0, 1.0]])
        seq = pgse_sequence(DT, n_steps, 0.1, 0.1, [0.0, 0.5, 1.0, 2.0], dirs, snap_steps=[n_steps])
        return Config(name, scale, sub, seq, over.get("n_walkers", 10_000), 1)
    if name == "cfg1":
        if full:
            sub = S.packed_cylinders(200, 200, 0.1, seed=2, place="all")
            n_steps, delta, Delta, nw = 85_000, 2.0, 15.0, 100_000
        else:
            sub = S.packed_cylinders(64, 16, 0.1, seed=2, place="all")
            n_steps, delta, Delta, nw = 2_000, 0.1, 0.3, 2_000
        seq = pgse_sequence(DT, n_steps, delta, Delta, np.arange(11.0), fibonacci_dirs(30), snap_steps=[n_steps])
        return Config(name, scale, sub, seq, over.get("n_walkers", nw), 2)
    if name in ("cfg2", "cfg3", "cfg4"):
        if full:
            geo = dict(nxy=500, nz=2000, n_axons=300)
        else:
            geo = dict(nxy=100, nz=200, n_axons=12)
        geo.update({k: v for k, v in over.items() if k in ("nxy", "nz", "n_axons")})
        if name == "cfg3":
            sub = S.axon_substrate(seed=3, D_extra=1.0, D_intra=2.0, T2_extra=40.0, T2_intra=60.0,
                                   kappa_membrane=0.02, place="all", **geo)
            if full:
                n_steps, delta, Delta, nw = 50_000, 2.0, 8.0, 1_000_000
                snaps = np.arange(5_000, 50_001, 5_000)
            else:
                n_steps, delta, Delta, nw = 5_000, 0.2, 0.8, 2_000
                snaps = np.arange(500, 5_001, 500)
            seq = pgse_sequence(DT, n_steps, delta, Delta, np.arange(11.0), fibonacci_dirs(30), snap_steps=snaps)
            return Config(name, scale, sub, seq, over.get("n_walkers", nw), 3)
        sub = S.axon_substrate(seed=3, D_extra=2.0, D_intra=2.0, place="intra", **geo)
        if name == "cfg2":
            if full:
                n_steps, delta, Delta, nw = 500_000, 10.0, 40.0, 1_000_000
                snaps = (np.array([5, 10, 20, 40, 60, 80, 100]) / DT).round().astype(np.int64)
            else:
                n_steps, delta, Delta, nw = 5_000, 0.2, 0.6, 2_000
                snaps = np.array([1000, 2000, 3000, 4000, 5000])
            seq = pgse_sequence(DT, n_steps, delta, Delta, np.linspace(0.0, 25.0, 11), fibonacci_dirs(60),
                                snap_steps=snaps)
            return Config(name, scale, sub, seq, over.get("n_walkers", nw), 3)
        # cfg4: throughput point on the cfg2 lattice, 10,000 steps
        n_steps = over.get("n_steps", 10_000 if full else 2_000)
        n_dir = over.get("n_dir", 60)
        dirs = fibonacci_dirs(n_dir) if n_dir > 1 else np.array([[0.0, 0.0, 1.0]])
        b = np.linspace(0.0, 25.0, 11) if n_dir > 1 else np.array([1.0])
        delta, Delta = 0.4 * n_steps * DT, 0.6 * n_steps * DT
        seq = pgse_sequence(DT, n_steps, delta, Delta, b, dirs, snap_steps=[n_steps])
        return Config(name, scale, sub, seq, over.get("n_walkers", 1_000_000 if full else 2_000), 3)
    raise KeyError(name)
