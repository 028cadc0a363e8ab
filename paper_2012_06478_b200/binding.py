"""Thin ctypes binding of include/rms.h: argument marshalling only, every step of the path runs in the
CUDA kernels of librms_b200.so.  The function names follow the C ABI (rms_substrate_create,
rms_walkers_init, rms_run, ...).  PyTorch is used for device memory and streams only.

There is no CPU fallback: if the library has not been built (python -m paper_2012_06478_b200.build) or
there is no CUDA device, calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "librms_b200.so"
RMS_MAX_WAVES = 16

RMS_LABELS_ON_DEVICE = 1
RMS_ADOPT_DEVICE_PTR = 2
RMS_NO_BRICKS = 4
RMS_LAYOUT_X_FASTEST = 8
RMS_LAYOUT_Z_FASTEST = 16
RMS_LAYOUT_AUTO = 24
RMS_LATTICE_DICT = 32
RMS_RUN_LABEL_GATHER = 1
RMS_RUN_GENERAL_KERNEL = 2
RMS_RUN_NO_ORDERING = 4
RMS_RUN_FP64 = 8
RMS_RUN_REJECTION_SAMPLING = 16
RMS_RUN_ERL = 32
RMS_RUN_NO_SLICES = 64
RMS_STATIC_MAX_LABELS = 16384

STATUS = {0: "RMS_OK", -1: "RMS_ERR_ARG", -2: "RMS_ERR_STEP_TOO_LARGE", -3: "RMS_ERR_P_RANGE", -4: "RMS_ERR_NO_SPACE",
          -5: "RMS_ERR_OOM", -6: "RMS_ERR_CUDA", -7: "RMS_ERR_UNSUPPORTED"}

EXPORTS = ("rms_substrate_create", "rms_substrate_destroy", "rms_substrate_get_info", "rms_walkers_init",
           "rms_walkers_destroy", "rms_run", "rms_walkers_read", "rms_walkers_steps_done", "rms_tables", "rms_normalise",
           "rms_walkers_init_weighted", "rms_substrate_label_volumes", "rms_volume_weighted_signal",
           "rms_memory_trim", "rms_gather_probe", "rms_last_error", "rms_version", "rms_substrate_label_volumes_static")


class RmsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class SubstrateDesc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("voxel_um", C.c_double),
                ("labels", C.c_void_p), ("n_labels", C.c_int32), ("D", C.c_void_p), ("T2", C.c_void_p),
                ("kappa", C.c_void_p), ("rho", C.c_void_p), ("label_class", C.c_void_p), ("n_classes", C.c_int32), ("flags", C.c_uint32),
                ("T1", C.c_void_p), ("conc", C.c_void_p)]


class SubstrateInfo(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("n_labels", C.c_int32),
                ("n_classes", C.c_int32), ("n_voxels", C.c_uint64), ("n_membrane_faces", C.c_uint64),
                ("lattice_bytes", C.c_uint64), ("brick_bytes", C.c_uint64), ("has_bricks", C.c_int32),
                ("dict_entries", C.c_uint32), ("dict_escaped_voxels", C.c_uint32)]


class RunDesc(C.Structure):
    _fields_ = [("dt_ms", C.c_double), ("n_steps", C.c_int64), ("n_wave", C.c_int32), ("wave", C.c_void_p),
                ("n_g", C.c_int32), ("gamp", C.c_void_p), ("n_dir", C.c_int32), ("dirs", C.c_void_p),
                ("n_snap", C.c_int32), ("snap_steps", C.c_void_p), ("flags", C.c_uint32),
                ("mix_first_step", C.c_int64), ("mix_n_steps", C.c_int64),
                ("n_tensor", C.c_int32), ("tensor_waves", C.c_void_p), ("tensor_gamp", C.c_void_p),
                ("n_rot", C.c_int32), ("rots", C.c_void_p)]


class Result(C.Structure):
    _fields_ = [("sum_alpha", C.c_void_p), ("sig_re", C.c_void_p), ("sig_im", C.c_void_p), ("m2", C.c_void_p),
                ("m4", C.c_void_p), ("snap_alpha", C.c_void_p), ("class_flow", C.c_void_p), ("S_re", C.c_void_p),
                ("S_im", C.c_void_p), ("Dapp", C.c_void_p), ("Kapp", C.c_void_p), ("n_encounters", C.c_uint64),
                ("n_permeations", C.c_uint64), ("n_clamps", C.c_uint64), ("n_saturations", C.c_uint64), ("kernel_ms", C.c_double),
                ("total_ms", C.c_double), ("n_launches", C.c_uint32),
                ("tsig_re", C.c_void_p), ("tsig_im", C.c_void_p), ("tS_re", C.c_void_p), ("tS_im", C.c_void_p)]


class WalkerState(C.Structure):
    _fields_ = [("vox", C.c_int32 * 3), ("off", C.c_float * 3), ("vox0", C.c_int32 * 3), ("off0", C.c_float * 3),
                ("label", C.c_uint16), ("label0", C.c_uint16), ("relax", C.c_float),
                ("phi", (C.c_double * 3) * RMS_MAX_WAVES)]


WALKER_DTYPE = np.dtype([("vox", np.int32, 3), ("off", np.float32, 3), ("vox0", np.int32, 3), ("off0", np.float32, 3),
                         ("label", np.uint16), ("label0", np.uint16), ("relax", np.float32),
                         ("phi", np.float64, (RMS_MAX_WAVES, 3))], align=True)

_lib = None


def load_library():
    """dlopen librms_b200.so; raises if it is not built (the product path never falls back to the CPU)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2012_06478_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(str(LIB_PATH))
        lib.rms_last_error.restype = C.c_char_p
        lib.rms_version.restype = C.c_char_p
        for name in EXPORTS:
            getattr(lib, name)
        assert C.sizeof(WalkerState) == WALKER_DTYPE.itemsize
        _lib = lib
    return _lib


def _check(rc):
    if rc != 0:
        raise RmsError(rc, load_library().rms_last_error().decode())


def _host(a, dtype):
    return None if a is None else np.ascontiguousarray(a, dtype=dtype)


def _ptr(a):
    return None if a is None else a.ctypes.data


def _stream_ptr(stream):
    if stream is None:
        import torch
        if not torch.cuda.is_available():   # the library reports RMS_ERR_CUDA itself
            return C.c_void_p(0)
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(int(getattr(stream, "cuda_stream", stream)))


class Substrate:
    """Owner of an rms_substrate handle."""

    def __init__(self, handle, keep=None, n_labels=0, n_classes=0):
        self.handle, self._keep, self.n_labels, self.n_classes = handle, keep, n_labels, n_classes

    def info(self):
        inf = SubstrateInfo()
        _check(load_library().rms_substrate_get_info(self.handle, C.byref(inf)))
        return {k: getattr(inf, k) for k, _ in inf._fields_}

    def tables(self, dt_ms):
        s = np.zeros(self.n_labels, np.float32)
        P = np.zeros((self.n_labels, self.n_labels), np.float32)
        _check(load_library().rms_tables(self.handle, C.c_double(dt_ms), C.c_void_p(s.ctypes.data), C.c_void_p(P.ctypes.data)))
        return s, P

    def destroy(self):
        if self.handle:
            load_library().rms_substrate_destroy(self.handle)
            self.handle = None
            self._keep = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def rms_substrate_create(labels, voxel_um, D, T2=None, kappa=None, label_class=None, n_classes=1, flags=0,
                         stream=None, rho=None, T1=None, conc=None) -> Substrate:
    """labels: numpy uint16 (nz, ny, nx) on the host, or a torch.uint16/int16 CUDA tensor of that shape
    (then the lattice is adopted in place, no copy)."""
    lib = load_library()
    keep = []
    if isinstance(labels, np.ndarray):
        lab = _host(labels, np.uint16)
        nz, ny, nx = lab.shape
        lab_ptr = lab.ctypes.data
        keep.append(lab)
    else:  # torch tensor on the device
        if not labels.is_cuda or labels.element_size() != 2 or not labels.is_contiguous():
            raise ValueError("device labels must be a contiguous 16-bit CUDA tensor of shape (nz, ny, nx)")
        nz, ny, nx = labels.shape
        lab_ptr = labels.data_ptr()
        flags |= RMS_LABELS_ON_DEVICE | RMS_ADOPT_DEVICE_PTR
        keep.append(labels)
    D = _host(D, np.float32)
    T2 = _host(T2, np.float32)
    kappa = _host(kappa, np.float32)
    label_class = _host(label_class, np.uint16)
    rho = _host(rho, np.float32)
    T1 = _host(T1, np.float32)
    conc = _host(conc, np.float32)
    d = SubstrateDesc(nx, ny, nz, float(voxel_um), lab_ptr, int(D.size), _ptr(D), _ptr(T2), _ptr(kappa), _ptr(rho), _ptr(label_class),
                      int(n_classes), int(flags), _ptr(T1), _ptr(conc))
    h = C.c_void_p()
    _check(lib.rms_substrate_create(C.byref(d), _stream_ptr(stream), C.byref(h)))
    adopt = bool(flags & RMS_ADOPT_DEVICE_PTR)
    return Substrate(h, keep if adopt else None, int(D.size), int(n_classes))


class Walkers:
    def __init__(self, handle, n, substrate):
        self.handle, self.n, self.substrate = handle, n, substrate

    def read(self, first=0, count=None, stream=None):
        """Walker states as a numpy structured array (the parity hook)."""
        count = self.n - first if count is None else count
        out = np.zeros(count, WALKER_DTYPE)
        _check(load_library().rms_walkers_read(self.handle, C.c_uint64(first), C.c_uint64(count),
                                               C.c_void_p(out.ctypes.data), _stream_ptr(stream)))
        return out

    def steps_done(self):
        v = C.c_uint64()
        _check(load_library().rms_walkers_steps_done(self.handle, C.byref(v)))
        return v.value

    def destroy(self):
        if self.handle:
            load_library().rms_walkers_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def rms_walkers_init(substrate: Substrate, n_walkers, first_walker_id=0, label_allowed=None, seed=0, stream=None) -> Walkers:
    allowed = _host(label_allowed, np.uint8)
    if allowed is not None and allowed.size != substrate.n_labels:
        raise ValueError("label_allowed must have n_labels entries")
    h = C.c_void_p()
    _check(load_library().rms_walkers_init(substrate.handle, C.c_uint64(n_walkers), C.c_uint64(first_walker_id),
                                           C.c_void_p(_ptr(allowed)), C.c_uint64(seed), _stream_ptr(stream), C.byref(h)))
    return Walkers(h, int(n_walkers), substrate)


def rms_walkers_init_weighted(substrate: Substrate, n_walkers, first_walker_id=0, label_allowed=None, label_weight=None, seed=0,
                              stream=None) -> Walkers:
    allowed = _host(label_allowed, np.uint8)
    weight = _host(label_weight, np.float32)
    for a in (allowed, weight):
        if a is not None and a.size != substrate.n_labels:
            raise ValueError("label_allowed and label_weight must have n_labels entries")
    h = C.c_void_p()
    _check(load_library().rms_walkers_init_weighted(substrate.handle, C.c_uint64(n_walkers), C.c_uint64(first_walker_id),
                                                    C.c_void_p(_ptr(allowed)), C.c_void_p(_ptr(weight)), C.c_uint64(seed),
                                                    _stream_ptr(stream), C.byref(h)))
    return Walkers(h, int(n_walkers), substrate)


def rms_substrate_label_volumes(substrate: Substrate, stream=None) -> np.ndarray:
    out = np.zeros(substrate.n_labels, np.uint64)
    _check(load_library().rms_substrate_label_volumes(substrate.handle, _stream_ptr(stream), C.c_void_p(out.ctypes.data)))
    return out


def rms_substrate_label_volumes_static(substrate: Substrate, stream=None) -> np.ndarray:
    """The same count through the entry point that allocates no device memory (at most RMS_STATIC_MAX_LABELS labels)."""
    out = np.zeros(substrate.n_labels, np.uint64)
    _check(load_library().rms_substrate_label_volumes_static(substrate.handle, _stream_ptr(stream), C.c_void_p(out.ctypes.data)))
    return out


def rms_volume_weighted_signal(r: dict, class_volume) -> np.ndarray:
    """S = sum_c V_c S_c / sum_c V_c from the per-class sums of a result dict (rms_volume_weighted_signal in include/rms.h)."""
    nC = r["sum_alpha"].size
    V = _host(class_volume, np.float64)
    if V.size != nC:
        raise ValueError("class_volume must have n_classes entries")
    arrs = {k: _host(r[k], np.float64) for k in ("sum_alpha", "sig_re", "sig_im")}
    S_re, S_im = np.zeros(r["sig_re"].shape[:-1]), np.zeros(r["sig_re"].shape[:-1])
    _check(load_library().rms_volume_weighted_signal(
        C.c_int(nC), C.c_int(arrs["sig_re"].size // nC), C.c_void_p(_ptr(V)), C.c_void_p(_ptr(arrs["sum_alpha"])),
        C.c_void_p(_ptr(arrs["sig_re"])), C.c_void_p(_ptr(arrs["sig_im"])), C.c_void_p(S_re.ctypes.data), C.c_void_p(S_im.ctypes.data)))
    return S_re + 1j * S_im


def rms_run(substrate: Substrate, walkers: Walkers, dt_ms, n_steps, wave=None, gamp=None, dirs=None, snap_steps=None,
            flags=0, stream=None, mix_first_step=0, mix_n_steps=0, tensor_waves=None, tensor_gamp=None, rots=None) -> dict:
    """Returns a dict of numpy arrays named as in rms_result (include/rms.h)."""
    wave = _host(wave, np.float32)
    gamp = _host(gamp, np.float64)
    dirs = _host(dirs, np.float64)
    snaps = _host(snap_steps, np.int64)
    n_wave = 0 if wave is None or wave.size == 0 else (wave.shape[0] if wave.ndim == 2 else 1)
    if n_wave and wave.size != n_wave * n_steps:
        raise ValueError("wave must have shape [n_wave, n_steps]")
    n_g = 0 if (gamp is None or n_wave == 0) else gamp.size // n_wave
    n_dir = 0 if dirs is None else dirs.size // 3
    n_snap = 0 if snaps is None else snaps.size
    nC = substrate.n_classes
    tw = _host(tensor_waves, np.int32)
    tg = _host(tensor_gamp, np.float64)
    rots = _host(rots, np.float64)
    n_tensor = 0 if tw is None else tw.size // 3
    n_rot = 0 if rots is None else rots.size // 9
    if n_tensor and (tg is None or tg.size != n_tensor * n_g):
        raise ValueError("tensor_gamp must have shape [n_tensor, n_g]")
    r = dict(sum_alpha=np.zeros(nC), sig_re=np.zeros((n_wave, n_g, n_dir, nC)), sig_im=np.zeros((n_wave, n_g, n_dir, nC)),
             m2=np.zeros((n_snap, n_dir, nC)), m4=np.zeros((n_snap, n_dir, nC)), snap_alpha=np.zeros((n_snap, nC)),
             class_flow=np.zeros((n_snap, nC, nC), np.uint64), S_re=np.zeros((n_wave, n_g, n_dir)),
             S_im=np.zeros((n_wave, n_g, n_dir)), Dapp=np.zeros((n_snap, n_dir)), Kapp=np.zeros((n_snap, n_dir)))
    d = RunDesc(float(dt_ms), int(n_steps), n_wave, _ptr(wave), n_g, _ptr(gamp), n_dir, _ptr(dirs), n_snap, _ptr(snaps),
                int(flags), int(mix_first_step), int(mix_n_steps), n_tensor, _ptr(tw), _ptr(tg), n_rot, _ptr(rots))
    res = Result()
    keys = ["sum_alpha", "sig_re", "sig_im", "m2", "m4", "snap_alpha", "class_flow", "S_re", "S_im", "Dapp", "Kapp"]
    if n_tensor:
        r.update(tsig_re=np.zeros((n_tensor, n_g, n_rot, nC)), tsig_im=np.zeros((n_tensor, n_g, n_rot, nC)),
                 tS_re=np.zeros((n_tensor, n_g, n_rot)), tS_im=np.zeros((n_tensor, n_g, n_rot)))
        keys += ["tsig_re", "tsig_im", "tS_re", "tS_im"]
    for k in keys:
        setattr(res, k, r[k].ctypes.data)
    _check(load_library().rms_run(substrate.handle, walkers.handle, C.byref(d), _stream_ptr(stream), C.byref(res)))
    r.update(n_encounters=int(res.n_encounters), n_permeations=int(res.n_permeations), n_clamps=int(res.n_clamps),
             n_saturations=int(res.n_saturations),
             kernel_ms=float(res.kernel_ms), total_ms=float(res.total_ms), n_launches=int(res.n_launches))
    r["S"] = r["S_re"] + 1j * r["S_im"]
    if n_tensor:
        r["tS"] = r["tS_re"] + 1j * r["tS_im"]
    return r


def rms_gather_probe(table_bytes, elem_bytes=4, loads_per_thread=1024, stream=None) -> float:
    """Random gathers per second from a device table of table_bytes (include/rms.h)."""
    out = C.c_double()
    _check(load_library().rms_gather_probe(C.c_uint64(int(table_bytes)), C.c_int(int(elem_bytes)), C.c_uint32(int(loads_per_thread)),
                                           _stream_ptr(stream), C.byref(out)))
    return out.value


def rms_normalise(r: dict, t_ms) -> dict:
    """Recompute S, Dapp, Kapp of a result dict from its raw sums (rms_normalise in include/rms.h)."""
    nC = r["sum_alpha"].size
    n_q = r["sig_re"].size // nC
    n_snap, n_dir = r["m2"].shape[0], r["m2"].shape[1]
    t = _host(np.atleast_1d(t_ms), np.float64)
    S_re, S_im = np.zeros(r["sig_re"].shape[:-1]), np.zeros(r["sig_re"].shape[:-1])
    Dapp, Kapp = np.zeros((n_snap, n_dir)), np.zeros((n_snap, n_dir))
    arrs = {k: _host(r[k], np.float64) for k in ("sum_alpha", "sig_re", "sig_im", "snap_alpha", "m2", "m4")}
    _check(load_library().rms_normalise(
        C.c_int(nC), C.c_int(n_q), C.c_void_p(_ptr(arrs["sum_alpha"])), C.c_void_p(_ptr(arrs["sig_re"])),
        C.c_void_p(_ptr(arrs["sig_im"])), C.c_int(n_snap), C.c_int(n_dir), C.c_void_p(_ptr(arrs["snap_alpha"])),
        C.c_void_p(_ptr(arrs["m2"])), C.c_void_p(_ptr(arrs["m4"])), C.c_void_p(_ptr(t)), C.c_void_p(S_re.ctypes.data),
        C.c_void_p(S_im.ctypes.data), C.c_void_p(Dapp.ctypes.data), C.c_void_p(Kapp.ctypes.data)))
    out = dict(r)
    out.update(S_re=S_re, S_im=S_im, Dapp=Dapp, Kapp=Kapp, S=S_re + 1j * S_im)
    if "tsig_re" in r:       # tensor waveforms: Eq.7 once more, no moments
        tre, tim = _host(r["tsig_re"], np.float64), _host(r["tsig_im"], np.float64)
        tS_re, tS_im = np.zeros(tre.shape[:-1]), np.zeros(tre.shape[:-1])
        _check(load_library().rms_normalise(
            C.c_int(nC), C.c_int(tre.size // nC), C.c_void_p(_ptr(arrs["sum_alpha"])), C.c_void_p(_ptr(tre)), C.c_void_p(_ptr(tim)),
            C.c_int(0), C.c_int(0), None, None, None, None, C.c_void_p(tS_re.ctypes.data), C.c_void_p(tS_im.ctypes.data), None, None))
        out.update(tS_re=tS_re, tS_im=tS_im, tS=tS_re + 1j * tS_im)
    return out
