"""Convenience layer over the binding: one call for the whole hot path, and walker-id sharding.

`sub` / `seq` are duck-typed: any objects with the attributes of rms_inputs.Substrate / Sequence
(labels, voxel_um, D, T2, kappa, label_class, n_classes, label_allowed; dt_ms, n_steps, wave, gamp,
dirs, snap_steps).  Nothing here computes: it only marshals arguments into the three C-ABI calls.
"""
from __future__ import annotations

import numpy as np

from . import binding as B

RAW_SUMS = ("sum_alpha", "sig_re", "sig_im", "m2", "m4", "snap_alpha", "class_flow")
COUNTERS = ("n_encounters", "n_permeations", "n_clamps", "n_saturations")
TENSOR_SUMS = ("tsig_re", "tsig_im")          # present when the run had tensor waveforms


def shard_range(rank: int, world: int, n_walkers: int):
    """Contiguous walker-id range [first, first+count) of `rank`: walkers are independent,
    so a job shards by walker id with the substrate replicated and no collective on the data path."""
    first = n_walkers * rank // world
    return first, n_walkers * (rank + 1) // world - first


def simulate(sub, seq, n_walkers, seed, first_id=0, flags=0, substrate_flags=0, device_labels=None, read_walkers=False,
             stream=None, keep=None, label_weight=None):
    """rms_substrate_create -> rms_walkers_init -> rms_run (-> rms_walkers_read); returns the result dict.

    device_labels: optional 16-bit CUDA tensor (nz, ny, nx) already resident in HBM (adopted, not copied).
    keep: optional dict that receives the live handles ("substrate", "walkers") instead of destroying them.
    """
    labels = device_labels if device_labels is not None else sub.labels
    S = B.rms_substrate_create(labels, sub.voxel_um, sub.D, sub.T2, sub.kappa, sub.label_class, sub.n_classes,
                               flags=substrate_flags, stream=stream, rho=getattr(sub, "rho", None), T1=getattr(sub, "T1", None), conc=getattr(sub, "conc", None))
    W = None
    try:
        if label_weight is None:
            W = B.rms_walkers_init(S, n_walkers, first_id, sub.label_allowed, seed, stream=stream)
        else:
            W = B.rms_walkers_init_weighted(S, n_walkers, first_id, sub.label_allowed, label_weight, seed, stream=stream)
        r = B.rms_run(S, W, seq.dt_ms, seq.n_steps, seq.wave, seq.gamp, seq.dirs, seq.snap_steps, flags=flags, stream=stream,
                      mix_first_step=getattr(seq, "mix_first_step", 0), mix_n_steps=getattr(seq, "mix_n_steps", 0),
                      tensor_waves=getattr(seq, "tensor_waves", None), tensor_gamp=getattr(seq, "tensor_gamp", None),
                      rots=getattr(seq, "rots", None))
        if read_walkers:
            r["walkers"] = W.read(stream=stream)
        r["substrate_info"] = S.info()
        if keep is not None:
            keep["substrate"], keep["walkers"] = S, W
            S = W = None
        return r
    finally:
        if W is not None:
            W.destroy()
        if S is not None:
            S.destroy()


def merge_results(parts, t_ms):
    """Sum the raw sums of several walker-id shards and normalise again (rms_normalise, H8)."""
    out = {k: np.sum([p[k] for p in parts], axis=0) for k in RAW_SUMS + TENSOR_SUMS if k in parts[0]}
    for k in COUNTERS:
        out[k] = int(sum(p[k] for p in parts))
    return B.rms_normalise(out, t_ms)


def allreduce_result(r, t_ms, group=None):
    """Multi-process merge over torch.distributed (NCCL on GPUs, gloo in the CPU tests): the only exchange
    step of a sharded job is the sum of a few KB of accumulators."""
    import torch
    import torch.distributed as dist

    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    out = dict(r)
    for k in RAW_SUMS + TENSOR_SUMS:
        if k not in r:
            continue
        a = np.ascontiguousarray(r[k])
        t = torch.from_numpy(a.astype(np.float64 if a.dtype != np.uint64 else np.int64)).to(dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        out[k] = t.cpu().numpy().astype(a.dtype)
    cnt = torch.tensor([int(r[k]) for k in COUNTERS], dtype=torch.int64, device=dev)
    dist.all_reduce(cnt, op=dist.ReduceOp.SUM, group=group)
    for k, v in zip(COUNTERS, cnt.tolist()):
        out[k] = int(v)
    return B.rms_normalise(out, t_ms)
