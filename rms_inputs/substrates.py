"""Seeded synthetic label lattices (inputs of rms_substrate_create).

Every lattice is a C-contiguous uint16 array of shape (nz, ny, nx): x is the fastest axis,
idx = (z*ny + y)*nx + x, and the box is periodic.  Label 0 is extra-cellular space.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Substrate:
    labels: np.ndarray                 # (nz, ny, nx) uint16
    voxel_um: float
    D: np.ndarray                      # [n_labels] float32, um^2/ms
    T2: np.ndarray                     # [n_labels] float32, ms (inf = no relaxation)
    kappa: np.ndarray                  # [n_labels, n_labels] float32, um/ms
    label_class: np.ndarray            # [n_labels] uint16
    n_classes: int
    label_allowed: np.ndarray          # [n_labels] uint8: 1 = walkers are placed here
    meta: dict = field(default_factory=dict)
    rho: np.ndarray | None = None      # [n_labels, n_labels] float32, um/ms: surface relaxivity (absorbing membranes), or None
    T1: np.ndarray | None = None       # [n_labels] float32, ms: relaxation during a mixing time (stimulated echo), or None
    conc: np.ndarray | None = None     # [n_labels] float32: relative spin concentration (Appendix C.2), or None = all equal

    @property
    def n_labels(self) -> int:
        return int(self.D.shape[0])

    @property
    def shape_xyz(self):
        nz, ny, nx = self.labels.shape
        return nx, ny, nz


def _tables(n_labels, D_extra, D_intra, T2_extra, T2_intra, kappa_membrane, place):
    D = np.full(n_labels, D_intra, dtype=np.float32)
    D[0] = D_extra
    T2 = np.full(n_labels, T2_intra, dtype=np.float32)
    T2[0] = T2_extra
    kappa = np.zeros((n_labels, n_labels), dtype=np.float32)
    if kappa_membrane:
        kappa[0, 1:] = kappa_membrane
        kappa[1:, 0] = kappa_membrane
    label_class = np.ones(n_labels, dtype=np.uint16)
    label_class[0] = 0
    allowed = np.ones(n_labels, dtype=np.uint8)
    if place == "intra":
        allowed[0] = 0
    elif place == "extra":
        allowed[1:] = 0
    elif place != "all":
        raise ValueError(place)
    return D, T2, kappa, label_class, allowed


def _make(labels, voxel_um, n_labels, D_extra=2.0, D_intra=2.0, T2_extra=np.inf, T2_intra=np.inf,
          kappa_membrane=0.0, place="all", meta=None) -> Substrate:
    D, T2, kappa, label_class, allowed = _tables(n_labels, D_extra, D_intra, T2_extra, T2_intra, kappa_membrane, place)
    n_classes = 2 if n_labels > 1 else 1
    if n_labels == 1:
        label_class[:] = 0
    return Substrate(labels=np.ascontiguousarray(labels, dtype=np.uint16), voxel_um=float(voxel_um), D=D, T2=T2,
                     kappa=kappa, label_class=label_class, n_classes=n_classes, label_allowed=allowed,
                     meta=dict(meta or {}))


# ----------------------------------------------------------------------------------------------
# simple geometries (pins)
# ----------------------------------------------------------------------------------------------
def uniform_lattice(n=(8, 8, 8), voxel_um=0.1, **kw) -> Substrate:
    """One compartment, no membranes: free diffusion."""
    nx, ny, nz = n
    return _make(np.zeros((nz, ny, nx), np.uint16), voxel_um, 1, **kw)


def plates(width_vox: int, wall_vox: int = 1, n_yz=(4, 4), voxel_um=0.1, **kw) -> Substrate:
    """Parallel plates normal to x: label 1 for x in [0, width), label 0 wall of `wall_vox` voxels."""
    ny, nz = n_yz
    nx = width_vox + wall_vox
    lab = np.zeros((nz, ny, nx), np.uint16)
    lab[:, :, :width_vox] = 1
    kw.setdefault("place", "intra")
    return _make(lab, voxel_um, 2, meta={"width_vox": width_vox}, **kw)


def slabs(width_a: int, width_b: int, n_yz=(4, 4), voxel_um=0.1, **kw) -> Substrate:
    """Two periodic slabs normal to x: label 0 for x in [0, width_a), label 1 for [width_a, width_a+width_b)."""
    ny, nz = n_yz
    lab = np.zeros((nz, ny, width_a + width_b), np.uint16)
    lab[:, :, width_a:] = 1
    return _make(lab, voxel_um, 2, meta={"width_a": width_a, "width_b": width_b}, **kw)


def random_lattice(n=(4, 4, 4), n_labels=3, seed=0, voxel_um=0.1, **kw) -> Substrate:
    """Independent random labels per voxel (brute-force pins; worst case for the interaction loop)."""
    nx, ny, nz = n
    rng = np.random.default_rng(seed)
    lab = rng.integers(0, n_labels, size=(nz, ny, nx)).astype(np.uint16)
    return _make(lab, voxel_um, n_labels, **kw)


# ----------------------------------------------------------------------------------------------
# cfg0: single straight cylinder
# ----------------------------------------------------------------------------------------------
def single_cylinder(n=32, radius_vox=10.0, voxel_um=0.1, nz=None, **kw) -> Substrate:
    """Label 1 iff the voxel centre lies within `radius_vox` of the box axis (along z)."""
    nz = n if nz is None else nz
    c = n / 2.0
    x = np.arange(n) + 0.5 - c
    inside = (x[None, :] ** 2 + x[:, None] ** 2) <= radius_vox ** 2
    lab = np.broadcast_to(inside[None, :, :], (nz, n, n)).astype(np.uint16)
    kw.setdefault("place", "intra")
    return _make(lab, voxel_um, 2, meta={"radius_vox": radius_vox}, **kw)


# ----------------------------------------------------------------------------------------------
# cfg1: packed parallel cylinders
# ----------------------------------------------------------------------------------------------
def packed_cylinders(n=200, nz=None, voxel_um=0.1, mean_radius_um=0.8, gamma_shape=4.0, target_fraction=0.60,
                     gap_vox=1.5, seed=2, max_fail=20000, **kw) -> Substrate:
    """Random sequential addition of z-aligned cylinders in a periodic n x n cross-section.

    Radii ~ Gamma(shape, scale = mean/shape); a large pool is drawn and sorted descending, each radius
    is tried at up to `max_fail` random centres (periodic minimum-image distance >= r_i + r_j + gap so
    that two cylinders never share a voxel face).  Placement stops at `target_fraction` of the area or
    when the pool is exhausted; count and achieved fraction go to meta.
    """
    nz = n if nz is None else nz
    rng = np.random.default_rng(seed)
    L = float(n)
    pool = np.sort(rng.gamma(gamma_shape, mean_radius_um / gamma_shape, size=4000) / voxel_um)[::-1]
    pool = pool[(pool >= 1.5) & (pool < n / 4.0)]
    # keep the gamma shape but thin the pool so that the expected covered area is ~1.3x the target
    want_area = 1.3 * target_fraction * L * L
    keep = max(1, int(round(want_area / (np.pi * np.mean(pool ** 2)))))
    pool = np.sort(rng.choice(pool, size=min(keep, pool.size), replace=False))[::-1]
    centres, radii = [], []
    area = 0.0
    for r in pool:
        if area / (L * L) >= target_fraction:
            break
        for _ in range(max_fail):
            c = rng.uniform(0.0, L, size=2)
            if centres:
                d = np.abs(np.asarray(centres) - c)
                d = np.minimum(d, L - d)
                if np.any(np.hypot(d[:, 0], d[:, 1]) < np.asarray(radii) + r + gap_vox):
                    continue
            centres.append(c)
            radii.append(r)
            area += np.pi * r * r
            break
    lab2d = np.zeros((n, n), np.uint16)
    xs = np.arange(n) + 0.5
    for j, (c, r) in enumerate(zip(centres, radii)):
        dx = np.abs(xs - c[0]); dx = np.minimum(dx, L - dx)
        dy = np.abs(xs - c[1]); dy = np.minimum(dy, L - dy)
        inside = (dx[None, :] ** 2 + dy[:, None] ** 2) <= r * r
        lab2d[inside & (lab2d == 0)] = j + 1
    lab = np.broadcast_to(lab2d[None], (nz, n, n))
    frac = float(np.count_nonzero(lab2d)) / (n * n)
    return _make(lab, voxel_um, len(radii) + 1,
                 meta={"n_cylinders": len(radii), "intra_fraction": frac,
                       "radii_um": (np.asarray(radii) * voxel_um).tolist()}, **kw)


# ----------------------------------------------------------------------------------------------
# cfg2/cfg3/cfg4: synthetic white-matter axons
# ----------------------------------------------------------------------------------------------
def _watson_tilts(rng, n, kappa):
    """cos(theta) from a Watson distribution about z, density ~ exp(kappa cos^2 theta), by rejection."""
    out = []
    while len(out) < n:
        t = rng.uniform(0.0, 1.0, size=4 * n + 16)
        acc = rng.uniform(0.0, 1.0, size=t.size) < np.exp(kappa * (t * t - 1.0))
        out.extend(t[acc].tolist())
    return np.asarray(out[:n])


def axon_substrate(nxy=500, nz=2000, n_axons=300, voxel_um=0.1, seed=3, mean_radius_um=0.5, gamma_shape=5.0,
                   watson_kappa=20.0, caliber_amp=0.3, caliber_period_um=(5.0, 15.0), undulation_amp_um=0.5,
                   undulation_wavelength_um=20.0, **kw) -> Substrate:
    """Axons near z with Watson orientation dispersion, sinusoidal caliber variation and undulation.

    Per axon a: r0 ~ Gamma(shape, mean/shape); tilt from Watson(kappa) about z with uniform azimuth;
    r(z) = r0 (1 + amp sin(2 pi z / Lambda + phi_c)), Lambda ~ U(period range);
    centre(z) = c0 + z tan(theta) (cos phi, sin phi) + A e_u sin(2 pi z / lambda_u + phi_u).
    Painted slice by slice as discs (voxel-centre rule), periodic in x and y; the first label wins on
    overlap.  The z wrap generally mismatches, which acts as an impermeable cap (R1).
    """
    rng = np.random.default_rng(seed)
    lab = np.zeros((nz, nxy, nxy), np.uint16)
    z_um = (np.arange(nz) + 0.5) * voxel_um
    r0 = rng.gamma(gamma_shape, mean_radius_um / gamma_shape, size=n_axons)
    cos_t = _watson_tilts(rng, n_axons, watson_kappa)
    tan_t = np.sqrt(np.maximum(0.0, 1.0 - cos_t ** 2)) / np.maximum(cos_t, 1e-6)
    az = rng.uniform(0.0, 2 * np.pi, n_axons)
    c0 = rng.uniform(0.0, nxy * voxel_um, size=(n_axons, 2))
    lam_c = rng.uniform(caliber_period_um[0], caliber_period_um[1], n_axons)
    ph_c = rng.uniform(0.0, 2 * np.pi, n_axons)
    az_u = rng.uniform(0.0, 2 * np.pi, n_axons)
    ph_u = rng.uniform(0.0, 2 * np.pi, n_axons)
    zi = np.arange(nz)
    for a in range(n_axons):
        r = r0[a] * (1.0 + caliber_amp * np.sin(2 * np.pi * z_um / lam_c[a] + ph_c[a])) / voxel_um
        und = undulation_amp_um * np.sin(2 * np.pi * z_um / undulation_wavelength_um + ph_u[a])
        cx = (c0[a, 0] + z_um * tan_t[a] * np.cos(az[a]) + und * np.cos(az_u[a])) / voxel_um
        cy = (c0[a, 1] + z_um * tan_t[a] * np.sin(az[a]) + und * np.sin(az_u[a])) / voxel_um
        half = int(np.ceil(r.max())) + 1
        off = np.arange(-half, half + 1)
        bx = np.floor(cx).astype(np.int64)
        by = np.floor(cy).astype(np.int64)
        X = bx[:, None] + off[None, :]                       # (nz, W) voxel x indices, unwrapped
        Y = by[:, None] + off[None, :]
        dx2 = (X + 0.5 - cx[:, None]) ** 2
        dy2 = (Y + 0.5 - cy[:, None]) ** 2
        inside = (dy2[:, :, None] + dx2[:, None, :]) <= (r * r)[:, None, None]   # (nz, Wy, Wx)
        zz, yy, xx = np.nonzero(inside)
        xi = np.mod(X[zz, xx], nxy)
        yi = np.mod(Y[zz, yy], nxy)
        free = lab[zi[zz], yi, xi] == 0
        lab[zi[zz][free], yi[free], xi[free]] = a + 1
    frac = float(np.count_nonzero(lab)) / lab.size
    kw.setdefault("place", "intra")
    return _make(lab, voxel_um, n_axons + 1,
                 meta={"n_axons": n_axons, "intra_fraction": frac, "r0_um": r0.tolist()}, **kw)
