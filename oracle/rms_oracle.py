"""ctypes wrapper of oracle/rms_oracle.c (TEST INFRASTRUCTURE, not the product).

Marshals numpy arrays into the plain-C oracle and writes out the last line of the method,
the normalisation of Eq.7 and of the narrow-pulse moments, in numpy fp64.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rms_oracle.c"
_LIB = _HERE / "librms_oracle.so"
_lib = None

_ERRORS = {-1: "bad argument", -2: "step length >= voxel size (PAPER.md lines 62, 189)",
           -3: "Eq.3 gives P > 1 for a finite kappa (PAPER.md line 624)",
           -4: "no voxel with an allowed label", -5: "out of memory"}


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"oracle error {code}: {_ERRORS.get(code, '?')}")
        self.code = code


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-fPIC", "-shared", "-o", str(_LIB), str(_SRC),
               "-lm", "-lpthread"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(str(_LIB))
        _lib.rms_oracle_run.restype = C.c_int
        _lib.rms_oracle_step.restype = C.c_int
        _lib.rms_oracle_tables.restype = C.c_int
        _lib.rms_oracle_init_walker.restype = C.c_int
        _lib.rms_oracle_philox4x32_10.restype = None
        _lib.rms_oracle_direction.restype = None
    return _lib


def _p(a, ctype):
    return None if a is None else a.ctypes.data_as(C.POINTER(ctype))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, np.uint32)
    _load().rms_oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def direction(wa: int, wb: int):
    u = np.zeros(3)
    _load().rms_oracle_direction(C.c_uint32(int(wa)), C.c_uint32(int(wb)), _p(u, C.c_double))
    return u


def tables(D, kappa, voxel_um, dt_ms, conc=None):
    """(s[n_labels], P[n_labels, n_labels]) of Eq.1 and Eq.3; with spin concentrations conc[n_labels], Eq.C.9 / C.13."""
    D = np.ascontiguousarray(D, np.float32)
    n = D.size
    kappa = None if kappa is None else np.ascontiguousarray(kappa, np.float32).reshape(n, n)
    conc = None if conc is None else np.ascontiguousarray(conc, np.float32)
    s = np.zeros(n)
    P = np.zeros((n, n))
    st = _load().rms_oracle_tables_conc(C.c_int(n), _p(D, C.c_float), _p(kappa, C.c_float), _p(conc, C.c_float),
                                        C.c_double(voxel_um), C.c_double(dt_ms), _p(s, C.c_double), _p(P, C.c_double))
    if st:
        raise OracleError(st)
    return s, P


def step(labels, s, P, vox, off, label, u, u_perm=(0.5, 0.5, 0.5)):
    """One Monte Carlo step with a given unit direction and given permeation uniforms."""
    labels = np.ascontiguousarray(labels, np.uint16)
    nz, ny, nx = labels.shape
    s = np.ascontiguousarray(s, np.float64)
    P = np.ascontiguousarray(P, np.float64)
    v = np.asarray(vox, np.int32).copy()
    f = np.asarray(off, np.float64).copy()
    L = C.c_uint16(int(label))
    uu = np.asarray(u, np.float64).copy()
    up = np.asarray(u_perm, np.float64).copy()
    cnt = np.zeros(3, np.int32)
    _load().rms_oracle_step(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(labels, C.c_uint16), C.c_int(s.size),
                            _p(s, C.c_double), _p(P, C.c_double), _p(v, C.c_int32), _p(f, C.c_double), C.byref(L),
                            _p(uu, C.c_double), _p(up, C.c_double), _p(cnt, C.c_int32))
    return v, f, int(L.value), dict(encounters=int(cnt[0]), permeations=int(cnt[1]), clamps=int(cnt[2]))


def init_walker(labels, label_allowed, seed, walker):
    labels = np.ascontiguousarray(labels, np.uint16)
    nz, ny, nx = labels.shape
    allowed = None if label_allowed is None else np.ascontiguousarray(label_allowed, np.uint8)
    v = np.zeros(3, np.int32)
    f = np.zeros(3)
    L = C.c_uint16(0)
    st = _load().rms_oracle_init_walker(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(labels, C.c_uint16),
                                        _p(allowed, C.c_uint8), C.c_uint64(seed), C.c_uint64(walker),
                                        _p(v, C.c_int32), _p(f, C.c_double), C.byref(L))
    if st:
        raise OracleError(st)
    return v, f, int(L.value)


def normalise(raw, dt_ms, snap_steps):
    """Eq.7 and the narrow-pulse D, K, pooled over classes and per class.

    K is normalised by <alpha> in both moments (R14).
    """
    out = dict(raw)
    sa = raw["sum_alpha"]
    tot = sa.sum()
    out["S"] = (raw["sig_re"].sum(-1) + 1j * raw["sig_im"].sum(-1)) / tot
    with np.errstate(divide="ignore", invalid="ignore"):
        out["S_class"] = (raw["sig_re"] + 1j * raw["sig_im"]) / sa
        t = np.asarray(snap_steps, np.float64) * dt_ms
        a_s = raw["snap_alpha"].sum(-1)                       # [n_snap]
        m2 = raw["m2"].sum(-1) / a_s[:, None]                 # [n_snap, n_dir]
        m4 = raw["m4"].sum(-1) / a_s[:, None]
        out["msd"] = m2
        out["D"] = m2 / (2.0 * t[:, None])
        out["K"] = m4 / (m2 * m2) - 3.0
    return out


def volume_weighted_signal(r, class_volume):
    """Signal of all cells from per-cell runs with any number of walkers per cell ("volume-weighted sum";
    reading R26): S = sum_c V_c S_c / sum_c V_c over the classes that hold walkers, S_c = sig_c / sum_alpha_c (Eq.7 per class)."""
    V = np.asarray(class_volume, np.float64)
    sa = r["sum_alpha"]
    use = sa > 0
    S_c = (r["sig_re"][..., use] + 1j * r["sig_im"][..., use]) / sa[use]
    return (S_c * V[use]).sum(-1) / V[use].sum()


def run(sub, seq, n_walkers, seed, first_id=0, n_threads=1, per_walker=False, interaction=0, label_weight=None):
    """Whole path on the CPU: init -> steps -> sums.  `sub`, `seq` are rms_inputs.Substrate / Sequence.
    interaction: 0 = elastic collision (the paper's method), 1 = rejection sampling (its Appendix B), 2 = equal-step-length
    random leap (its Appendix A)."""
    lib = _load()
    labels = np.ascontiguousarray(sub.labels, np.uint16)
    nz, ny, nx = labels.shape
    nL, nC = sub.n_labels, int(sub.n_classes)
    D = np.ascontiguousarray(sub.D, np.float32)
    T2 = np.ascontiguousarray(sub.T2, np.float32)
    kappa = np.ascontiguousarray(sub.kappa, np.float32)
    rho = getattr(sub, "rho", None)
    rho = None if rho is None else np.ascontiguousarray(rho, np.float32)
    T1 = getattr(sub, "T1", None)
    T1 = None if T1 is None else np.ascontiguousarray(T1, np.float32)
    mix_first, mix_steps = int(getattr(seq, "mix_first_step", 0)), int(getattr(seq, "mix_n_steps", 0))
    conc = getattr(sub, "conc", None)
    conc = None if conc is None else np.ascontiguousarray(conc, np.float32)
    label_weight = None if label_weight is None else np.ascontiguousarray(label_weight, np.float32)
    lclass = np.ascontiguousarray(sub.label_class, np.uint16)
    allowed = np.ascontiguousarray(sub.label_allowed, np.uint8)
    wave = np.ascontiguousarray(seq.wave, np.float32)
    gamp = np.ascontiguousarray(seq.gamp, np.float64)
    dirs = np.ascontiguousarray(seq.dirs, np.float64)
    snaps = np.ascontiguousarray(seq.snap_steps, np.int64)
    n_wave, n_steps = wave.shape if wave.ndim == 2 else (0, int(seq.n_steps))
    n_g = gamp.shape[1] if gamp.ndim == 2 and n_wave else 0
    n_dir, n_snap = dirs.shape[0], snaps.size
    r = dict(
        sum_alpha=np.zeros(nC), sig_re=np.zeros((n_wave, n_g, n_dir, nC)), sig_im=np.zeros((n_wave, n_g, n_dir, nC)),
        m2=np.zeros((n_snap, n_dir, nC)), m4=np.zeros((n_snap, n_dir, nC)), snap_alpha=np.zeros((n_snap, nC)),
        class_flow=np.zeros((n_snap, nC, nC), np.uint64))
    counters = np.zeros(8, np.uint64)
    pw = {}
    if per_walker:
        pw = dict(final_vox=np.zeros((n_walkers, 3), np.int32), final_off=np.zeros((n_walkers, 3)),
                  final_label=np.zeros(n_walkers, np.uint16), init_vox=np.zeros((n_walkers, 3), np.int32),
                  init_off=np.zeros((n_walkers, 3)), phi=np.zeros((n_walkers, max(n_wave, 1), 3)),
                  relax=np.zeros(n_walkers))
    st = lib.rms_oracle_run(
        C.c_int(nx), C.c_int(ny), C.c_int(nz), C.c_double(sub.voxel_um), _p(labels, C.c_uint16), C.c_int(nL),
        _p(D, C.c_float), _p(T2, C.c_float), _p(kappa, C.c_float), _p(rho, C.c_float), _p(lclass, C.c_uint16), C.c_int(nC),
        C.c_uint64(n_walkers), C.c_uint64(first_id), _p(allowed, C.c_uint8), C.c_uint64(seed),
        C.c_double(seq.dt_ms), C.c_int64(n_steps), C.c_int(n_wave), _p(wave, C.c_float), C.c_int(n_g),
        _p(gamp, C.c_double), C.c_int(n_dir), _p(dirs, C.c_double), C.c_int(n_snap), _p(snaps, C.c_int64),
        C.c_int(n_threads), C.c_int(interaction), _p(T1, C.c_float), C.c_int64(mix_first), C.c_int64(mix_steps),
        _p(conc, C.c_float), _p(label_weight, C.c_float),
        _p(r["sum_alpha"], C.c_double), _p(r["sig_re"], C.c_double), _p(r["sig_im"], C.c_double),
        _p(r["m2"], C.c_double), _p(r["m4"], C.c_double), _p(r["snap_alpha"], C.c_double),
        _p(r["class_flow"], C.c_uint64), _p(counters, C.c_uint64),
        _p(pw.get("final_vox"), C.c_int32), _p(pw.get("final_off"), C.c_double), _p(pw.get("final_label"), C.c_uint16),
        _p(pw.get("init_vox"), C.c_int32), _p(pw.get("init_off"), C.c_double),
        _p(pw.get("phi") if n_wave else None, C.c_double), _p(pw.get("relax"), C.c_double))
    if st:
        raise OracleError(st)
    r.update(pw)
    r.update(n_encounters=int(counters[0]), n_permeations=int(counters[1]), n_clamps=int(counters[2]),
             max_encounters_per_step=int(counters[3]), n_saturations=int(counters[4]))
    return normalise(r, seq.dt_ms, snaps)


def tensor_signal(sub, seq, r):
    """Eq.7 for gradient waveforms that change direction in time (B-tensor encoding; the paper's "arbitrary diffusion gradient
    waveforms"; reading R23 in DESIGN.md), from the per-walker phase vectors of run(..., per_walker=True).

    A tensor waveform t drives the gradient axes x, y, z with the scalar waveforms seq.tensor_waves[t] = (m_x, m_y, m_z)
    (-1: axis off); with the rotation R_k (seq.rots[k], g_lab = R_k g) and the amplitude seq.tensor_gamp[t, g] the phase
    of Eq.7 is phi = gamp dt l_p sum_a (R_k e_a) . Phi_{m_a}, Phi_m = sum_i w_m[i] (x_i - x_0) in voxels.
    Returns tsig_re/tsig_im [n_tensor, n_g, n_rot, n_classes] (by class of the initial label) and tS [n_tensor, n_g, n_rot]."""
    tw = np.asarray(seq.tensor_waves, np.int64).reshape(-1, 3)
    tg = np.asarray(seq.tensor_gamp, np.float64).reshape(tw.shape[0], -1)
    rots = np.asarray(seq.rots, np.float64).reshape(-1, 3, 3)
    nC = int(sub.n_classes)
    iv = r["init_vox"]
    lab0 = np.asarray(sub.labels)[iv[:, 2], iv[:, 1], iv[:, 0]]
    cls0 = np.asarray(sub.label_class)[lab0]
    alpha = np.exp(-r["relax"])
    phi = r["phi"]                                            # [n_walkers, n_wave, 3]
    re = np.zeros((tw.shape[0], tg.shape[1], rots.shape[0], nC))
    im = np.zeros_like(re)
    for t in range(tw.shape[0]):
        for k in range(rots.shape[0]):
            proj = np.zeros(phi.shape[0])
            for a in range(3):
                if tw[t, a] >= 0:
                    proj += phi[:, tw[t, a], :] @ rots[k][:, a]       # (R_k e_a) . Phi_{m_a}
            for g in range(tg.shape[1]):
                ph = tg[t, g] * seq.dt_ms * sub.voxel_um * proj
                for c in range(nC):
                    sel = cls0 == c
                    re[t, g, k, c] = np.sum(alpha[sel] * np.cos(ph[sel]))
                    im[t, g, k, c] = -np.sum(alpha[sel] * np.sin(ph[sel]))
    tS = (re.sum(-1) + 1j * im.sum(-1)) / r["sum_alpha"].sum()
    return dict(tsig_re=re, tsig_im=im, tS=tS)


def default_threads() -> int:
    return len(os.sched_getaffinity(0))
