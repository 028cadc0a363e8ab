"""GPU parity tests: the CUDA path (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Tolerances are north_star's: >= 99.9 % of walkers in the same final voxel, |dS| <= 1e-4 per
b-value and direction, moments within 1e-4 relative; integer work (placement) bit exact."""
import math

import numpy as np
import pytest

import rms_inputs as ri
from parity_util import compare, gpu_run, oracle_run

pytestmark = pytest.mark.gpu

LABEL_GATHER = 1   # RMS_RUN_LABEL_GATHER


@pytest.fixture(scope="module")
def rms():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2012_06478_b200 as rms
    rms.load_library()
    return rms


def _both(cfg, n_walkers=None, flags=0, first_id=0):
    # the reduced configs carry 2,000 walkers; the plain tolerances of north_star need N >= 1e5 (one lost walker is 2/N of S)
    n = (max(cfg.n_walkers, 100_000) if cfg.scale == "test" else cfg.n_walkers) if n_walkers is None else n_walkers
    g = gpu_run(cfg.substrate, cfg.sequence, n, cfg.seed, first_id=first_id, flags=flags)
    o = oracle_run(cfg.substrate, cfg.sequence, n, cfg.seed, first_id=first_id)
    return g, o, n


@pytest.mark.parametrize("flags", [0, LABEL_GATHER], ids=["facemask", "labels"])
def test_cfg0_single_cylinder(rms, flags):
    cfg = ri.make_config("cfg0")
    g, o, n = _both(cfg, flags=flags)
    rep = compare(g, o, n)
    print("cfg0", flags, rep)
    assert g["n_permeations"] == 0
    assert np.all(g["walkers"]["label"] == 1)
    # b = 0: S = 1 exactly
    assert np.allclose(g["S"][0, 0], 1.0, atol=1e-12)
    # the straight cylinder is free along z: product-of-sincs closed form for the discrete walk
    seq = cfg.sequence
    ds = math.sqrt(6 * 2.0 * seq.dt_ms)
    W = np.cumsum(seq.wave[0][::-1].astype(float))[::-1]
    for gi, gamp in enumerate(seq.gamp[0]):
        exact = np.prod(np.sinc(gamp * seq.dt_ms * ds * W / np.pi))
        assert abs(g["S"][0, gi, 1].real - exact) < 4 * math.sqrt(0.5 / n)


@pytest.mark.parametrize("flags", [0, LABEL_GATHER], ids=["facemask", "labels"])
def test_cfg1_packed_cylinders_reduced(rms, flags):
    cfg = ri.make_config("cfg1", "test")
    g, o, n = _both(cfg, flags=flags)
    print("cfg1", flags, compare(g, o, n))


@pytest.mark.parametrize("flags", [0, LABEL_GATHER], ids=["facemask", "labels"])
def test_cfg2_axons_reduced_with_snapshots(rms, flags):
    cfg = ri.make_config("cfg2", "test")
    g, o, n = _both(cfg, flags=flags)
    print("cfg2", flags, compare(g, o, n))
    assert g["m2"].shape == (5, 60, 2)


def test_cfg3_permeable_heterogeneous_reduced(rms):
    cfg = ri.make_config("cfg3", "test")
    g, o, n = _both(cfg)
    rep = compare(g, o, n)
    print("cfg3", rep)
    assert g["n_permeations"] > 0
    # T2 weights: per-walker relaxation exponent
    assert np.allclose(g["walkers"]["relax"], o["relax"], rtol=2e-6, atol=1e-7)


def test_strongly_permeable_slabs_with_D_contrast(rms):
    # P ~ 0.1-0.3 and D contrast: exercises the fine permeation draw, the rescaled remainder (R7) and Eq.C.15
    for kap in (40.0, float("inf")):
        sub = ri.slabs(6, 6, (3, 3), 0.1, D_extra=2.0, D_intra=0.5, kappa_membrane=kap, T2_extra=0.05, T2_intra=0.2)
        seq = ri.pgse_sequence(2e-4, 600, 0.04, 0.06, [0.0, 5.0, 50.0], ri.fibonacci_dirs(7), snap_steps=[101, 600])
        n = 100_000
        g = gpu_run(sub, seq, n, 7)
        o = oracle_run(sub, seq, n, 7)
        rep = compare(g, o, n)
        print("slabs", kap, rep)
        assert g["n_permeations"] > 10000


def test_weakly_permeable_runs_take_the_specialised_kernel_and_its_redo_path(rms):
    # kappa such that 512 P is ~20-45 (below the 64 that keeps the run on the specialised kernel): about one membrane
    # encounter in 15 has coarse bits that allow a permeation and is redone by the written-out loop, with D contrast
    # (hop rescaled, R7), T2 contrast (Eq.5 by compartment), heavy periodic wrapping, snapshots on odd steps, 2 waveforms
    import oracle
    sub = ri.slabs(5, 4, (3, 2), 0.1, D_extra=2.0, D_intra=1.0, kappa_membrane=4.0, T2_extra=0.05, T2_intra=0.2)
    _, P = oracle.rms_oracle.tables(sub.D, sub.kappa, sub.voxel_um, 2e-4)
    assert 15.0 < 512 * np.max(P[~np.eye(2, dtype=bool)]) < 64.0
    n_steps = 701
    wave = np.stack([ri.pgse_wave(n_steps, 201, 350), ri.pgse_wave(n_steps, 100, 500)])
    seq = ri.Sequence(dt_ms=2e-4, n_steps=n_steps, wave=wave, gamp=np.array([[0.0, 30.0], [0.0, 80.0]]),
                      dirs=ri.fibonacci_dirs(5), snap_steps=np.array([99, 350, 701]))
    n = 100_000
    o = oracle_run(sub, seq, n, 9)
    g = gpu_run(sub, seq, n, 9)
    rep = compare(g, o, n)
    print("weakly permeable, specialised kernel", rep)
    assert 1000 < g["n_permeations"] < 0.2 * g["n_encounters"]
    g2 = gpu_run(sub, seq, n, 9, flags=2)                       # RMS_RUN_GENERAL_KERNEL: same physics, other kernel
    print("weakly permeable, general kernel", compare(g2, o, n))
    assert abs(g["n_permeations"] - g2["n_permeations"]) <= 3 and np.abs(g["S"] - g2["S"]).max() < 2e-4


def test_chunked_run_continues_the_same_trajectories(rms):
    cfg = ri.make_config("cfg0")
    sub, seq = cfg.substrate, cfg.sequence
    n = 100_000
    o = oracle_run(sub, seq, n, cfg.seed)
    S = rms.rms_substrate_create(sub.labels, sub.voxel_um, sub.D, sub.T2, sub.kappa, sub.label_class, sub.n_classes)
    W = rms.rms_walkers_init(S, n, 0, sub.label_allowed, cfg.seed)
    cuts = [0, 333, 334, 1000]                                  # odd boundary: the Philox pair is split across calls
    enc = 0
    for a, b in zip(cuts[:-1], cuts[1:]):
        r = rms.rms_run(S, W, seq.dt_ms, b - a, seq.wave[:, a:b], seq.gamp, seq.dirs, [b - a])
        enc += r["n_encounters"]
    r["n_encounters"] = enc
    assert W.steps_done() == 1000
    r["walkers"] = W.read()
    rep = compare(r, o, n)
    print("chunked", rep)


def test_chunked_run_with_a_comparison_interaction_and_a_mixing_time(rms):
    """The random numbers of the retries (R25) are keyed on the absolute step and the mixing time (R22) is given per call: three
    calls -- the middle one all mixing time, its T1 weight and the ERL retries included -- equal the oracle's single run."""
    import dataclasses
    sub = dataclasses.replace(ri.single_cylinder(24, 8.5, 0.1), T2=np.array([0.3, 0.15], np.float32), T1=np.array([0.9, 0.4], np.float32))
    seq = ri.pgse_sequence(2e-4, 900, 0.06, 0.12, [0.0, 2.0], np.eye(3), snap_steps=[900])     # lobes 1..300, 601..900
    seq = dataclasses.replace(seq, mix_first_step=301, mix_n_steps=300)
    n = 100_000
    for interaction, flag in ((2, rms.binding.RMS_RUN_ERL), (1, rms.binding.RMS_RUN_REJECTION_SAMPLING)):
        o = oracle_run(sub, seq, n, 19, interaction=interaction)
        for fp in (0, 8):
            S = rms.rms_substrate_create(sub.labels, sub.voxel_um, sub.D, sub.T2, sub.kappa, sub.label_class, sub.n_classes, T1=sub.T1)
            W = rms.rms_walkers_init(S, n, 0, sub.label_allowed, 19)
            enc = 0
            for a, b, mix in ((0, 301, (301, 1)), (301, 599, (1, 298)), (599, 900, (1, 1))):     # odd cuts; window 301..600 split over all three
                r = rms.rms_run(S, W, seq.dt_ms, b - a, seq.wave[:, a:b], seq.gamp, seq.dirs, [b - a], flags=flag | fp,
                                mix_first_step=mix[0], mix_n_steps=mix[1])
                enc += r["n_encounters"]
            r["n_encounters"] = enc
            r["walkers"] = W.read()
            print("chunked, interaction", interaction, "fp64" if fp else "fp32", compare(r, o, n))
            W.destroy(); S.destroy()


def test_general_waveform_table_mode_and_two_waves(rms):
    # non-integer gradient shapes (sine, trapezoid) take the table path; two waveforms share one trajectory set
    sub = ri.single_cylinder(24, 7.5, 0.1)
    n_steps = 801
    t = (np.arange(n_steps) + 1.0) / n_steps
    wave = np.stack([np.sin(2 * np.pi * t), np.clip(4 * np.minimum(t, 1 - t), 0, 1) * np.sign(0.5 - t)]).astype(np.float32)
    seq = ri.Sequence(dt_ms=2e-4, n_steps=n_steps, wave=wave, gamp=np.array([[0.0, 40.0, 90.0], [10.0, 60.0, 120.0]]),
                      dirs=ri.fibonacci_dirs(5), snap_steps=np.array([400, 801]))
    n = 100_000
    g = gpu_run(sub, seq, n, 5)
    o = oracle_run(sub, seq, n, 5)
    print("table", compare(g, o, n))
    # integer-valued pair of waveforms (const path, NW = 2)
    wave2 = np.stack([ri.pgse_wave(n_steps, 200, 500), ri.pgse_wave(n_steps, 100, 300)])
    seq2 = ri.Sequence(dt_ms=2e-4, n_steps=n_steps, wave=wave2, gamp=np.array([[0.0, 30.0], [0.0, 80.0]]),
                       dirs=ri.fibonacci_dirs(4), snap_steps=np.array([801]))
    g = gpu_run(sub, seq2, n, 5)
    o = oracle_run(sub, seq2, n, 5)
    print("two waves", compare(g, o, n))


def test_four_integer_waveforms_odd_boundaries_and_chunks(rms):
    # specialised kernel at its widest: 4 piecewise-constant waveforms with amplitudes other than +-1, lobes that start
    # and end on odd steps (the second half of a Philox call opens a segment), snapshots on odd steps (launch boundaries
    # inside a Philox pair) and the run continued by a second call from an odd step count
    sub = ri.single_cylinder(20, 6.5, 0.1)
    n1, n2 = 333, 268
    nT = n1 + n2
    wave = np.zeros((4, nT), np.float32)
    wave[0] = ri.pgse_wave(nT, 151, 301)
    wave[1, 3:120] = 2.0; wave[1, 333:450] = -2.0
    wave[2, 0:77] = -3.0; wave[2, 77:154] = 3.0; wave[2, 401:478] = 1.0; wave[2, 478:555] = -1.0
    wave[3, 5:6] = 7.0; wave[3, 599:600] = -7.0
    gamp = np.array([[0.0, 60.0], [5.0, 45.0], [0.0, 30.0], [10.0, 400.0]])
    dirs = ri.fibonacci_dirs(7)
    n = 8000
    full = ri.Sequence(dt_ms=2e-4, n_steps=nT, wave=wave, gamp=gamp, dirs=dirs, snap_steps=np.array([1, 77, 333, 600, 601]))
    o = oracle_run(sub, full, n, 21)
    g = gpu_run(sub, full, n, 21)
    print("four waves", compare(g, o, n))
    # same run in two calls: 333 steps, then 268 more (phases keep accumulating, R11: the waveform is per call)
    keep = {}
    s1 = ri.Sequence(dt_ms=2e-4, n_steps=n1, wave=wave[:, :n1].copy(), gamp=gamp, dirs=dirs, snap_steps=np.array([n1]))
    s2 = ri.Sequence(dt_ms=2e-4, n_steps=n2, wave=wave[:, n1:].copy(), gamp=gamp, dirs=dirs, snap_steps=np.array([n2]))
    rms.simulate(sub, s1, n, 21, keep=keep)
    r2 = rms.binding.rms_run(keep["substrate"], keep["walkers"], s2.dt_ms, s2.n_steps, s2.wave, s2.gamp, s2.dirs, s2.snap_steps)
    assert np.abs(r2["S"] - g["S"]).max() < 1e-9           # identical trajectories and phases, only the summation order differs
    keep["walkers"].destroy(); keep["substrate"].destroy()


@pytest.mark.parametrize("n_wave", [6, 16])
def test_sequence_sweep_many_waveforms_on_one_set_of_trajectories(rms, n_wave):
    # S: section 8(f) N1 -- a sweep of PGSE timings (the paper's Delta = delta series) evaluated on the same
    # trajectories in one run: 6 waveforms run on the 8-waveform kernel padded with zero weights, 16 on the 16-waveform one;
    # specialised fp32 and fp64 kernels (integer and non-integer amplitudes), general kernel through RMS_RUN_GENERAL_KERNEL
    sub = ri.single_cylinder(20, 6.5, 0.1)
    nT = 640
    wave = np.zeros((n_wave, nT), np.float32)
    for m in range(n_wave):
        n_delta = 20 + 18 * m
        wave[m] = ri.pgse_wave(nT, n_delta, n_delta + (m % 3) * 7)
    gamp = np.stack([np.array([0.0, 40.0 / (1 + m)]) for m in range(n_wave)])
    seq = ri.Sequence(dt_ms=2e-4, n_steps=nT, wave=wave, gamp=gamp, dirs=ri.fibonacci_dirs(4), snap_steps=np.array([321, nT]))
    n = 100_000
    o = oracle_run(sub, seq, n, 17)
    for flags in (0, 8):
        g = gpu_run(sub, seq, n, 17, flags=flags)
        rep = compare(g, o, n)
        print("waves", n_wave, "flags", flags, rep)
        assert g["S"].shape == (n_wave, 2, 4)
        if flags == 8:
            assert rep["n_diff"] == 0
    wave2 = wave.copy()
    wave2[n_wave - 1] *= 0.37                                    # non-integer amplitudes: still piecewise constant, same kernels
    seq2 = ri.Sequence(dt_ms=2e-4, n_steps=nT, wave=wave2, gamp=gamp, dirs=ri.fibonacci_dirs(4), snap_steps=np.array([nT]))
    o2 = oracle_run(sub, seq2, n, 17)
    for flags in (0, 8):
        print("waves", n_wave, "non-integer amplitudes, flags", flags, compare(gpu_run(sub, seq2, n, 17, flags=flags), o2, n))
    print("waves", n_wave, "general kernel, table mode", compare(gpu_run(sub, seq2, n, 17, flags=2), o2, n))
    print("waves", n_wave, "general kernel, const mode", compare(gpu_run(sub, seq, n, 17, flags=2), o, n))


@pytest.mark.parametrize("dims", [(5, 7, 3), (1, 1, 9), (2, 3, 4)])
@pytest.mark.parametrize("flags", [0, LABEL_GATHER], ids=["facemask", "labels"])
def test_ragged_tiny_lattices_with_heavy_wrapping(rms, dims, flags):
    # random labels per voxel, impermeable: almost every face is a membrane or a periodic wrap
    sub = ri.random_lattice(dims, n_labels=2, seed=3)
    seq = ri.pgse_sequence(2e-4, 400, 0.02, 0.04, [0.0, 20.0], np.eye(3), snap_steps=[399, 400])
    n = 100_000
    g = gpu_run(sub, seq, n, 11, flags=flags)
    o = oracle_run(sub, seq, n, 11)
    print("tiny", dims, compare(g, o, n))


@pytest.mark.parametrize("layout", [8, 16, 24], ids=["x_fastest", "z_fastest", "auto"])
def test_both_memory_orders_of_the_neighbourhood_lattice(rms, layout):
    # RMS_LAYOUT_X_FASTEST (the default) / RMS_LAYOUT_Z_FASTEST / RMS_LAYOUT_AUTO (picked from a sample of the lattice):
    # ragged box with heavy wrapping through both step kernels, and the reduced axon substrate
    sub = ri.random_lattice((37, 5, 70), n_labels=2, seed=4)
    seq = ri.pgse_sequence(2e-4, 300, 0.02, 0.03, [0.0, 20.0], np.eye(3), snap_steps=[299, 300])
    n = 100_000
    o = oracle_run(sub, seq, n, 12)
    for flags in (0, 2):                       # specialised and general kernel
        g = rms.simulate(sub, seq, n, 12, flags=flags, substrate_flags=layout, read_walkers=True)
        print("layout", layout, flags, compare(g, o, n))
    cfg = ri.make_config("cfg2", "test")
    g = rms.simulate(cfg.substrate, cfg.sequence, cfg.n_walkers, cfg.seed, substrate_flags=layout, read_walkers=True)
    o = oracle_run(cfg.substrate, cfg.sequence, cfg.n_walkers, cfg.seed)
    print("layout cfg2", layout, compare(g, o, cfg.n_walkers))
    assert g["substrate_info"]["n_membrane_faces"] == sum(
        int(np.count_nonzero(cfg.substrate.labels != np.roll(cfg.substrate.labels, 1, axis=ax))) for ax in range(3))


def test_free_box_wraps_many_times(rms):
    # no membranes at all, small periodic box: every walker wraps the box repeatedly (ghost-shell folding)
    sub = ri.uniform_lattice((4, 3, 5))
    seq = ri.pgse_sequence(2e-4, 2000, 0.1, 0.2, [0.0, 1.0, 3.0], ri.fibonacci_dirs(6), snap_steps=[2000])
    n = 5000
    g = gpu_run(sub, seq, n, 13)
    o = oracle_run(sub, seq, n, 13)
    rep = compare(g, o, n)
    print("free", rep)
    assert g["n_encounters"] == 0
    assert np.abs(g["walkers"]["vox"]).max() > 8               # really left the box


def test_one_voxel_wide_lattice_over_200k_steps_wrap_counters(rms):
    """A (1, 1, 9) lattice without membranes, 200,000 steps: a walker wraps the 1-voxel axes ~+-250 times (sigma) and more than
    +-511 times for ~4 % of the walkers; the general kernels count wraps per launch in 10-bit fields, so rms_run must split
    the run.  Default path (specialised kernel) and the general fp32 / fp64 kernels against the oracle."""
    sub = ri.uniform_lattice((1, 1, 9), 0.1, D_extra=8.0)           # hop of 0.98 voxel: sigma = 253 voxels after 200,000 steps
    n, n_steps = 5_000, 200_000
    seq = ri.pgse_sequence(2e-4, n_steps, 10.0, 20.0, [0.0, 0.05], np.eye(3), snap_steps=[n_steps])
    o = oracle_run(sub, seq, n, 13)
    assert np.abs(o["final_vox"][:, 0]).max() > 511
    for flags in (0, 2, 8 | 2):
        g = gpu_run(sub, seq, n, 13, flags=flags)
        # free diffusion: no membrane, no discontinuity -- every walker stays with its twin; fp32 offsets drift by ~1e-5
        same = np.all(g["walkers"]["vox"] == o["final_vox"], axis=1)
        print("1x1x9, flags", flags, "same voxel", same.mean(), "max |dS|", np.abs(g["S"] - o["S"]).max(), "launches", g["n_launches"])
        assert same.mean() >= 0.999
        assert np.abs(g["S"] - o["S"]).max() <= 1e-4 + 2.0 * (1 - same.mean())
        assert np.allclose(g["m2"], o["m2"], rtol=1e-4 + 8 * (1 - same.mean()))


def test_walker_subrange_and_placement_only(rms):
    cfg = ri.make_config("cfg1", "test")
    g, o, n = _both(cfg, n_walkers=257, first_id=1000)          # ragged: 2 blocks + 1 walker
    print("subrange", compare(g, o, n))
    # zero steps: placement only
    seq0 = ri.Sequence(dt_ms=2e-4, n_steps=0, wave=np.zeros((1, 0), np.float32), gamp=np.array([[0.0, 1.0]]),
                       dirs=np.eye(3), snap_steps=np.zeros(0, np.int64))
    g0 = gpu_run(cfg.substrate, seq0, 1, cfg.seed)
    assert np.allclose(g0["S"], 1.0) and g0["sum_alpha"].sum() == 1.0


def test_error_codes(rms):
    cfg = ri.make_config("cfg0")
    sub, seq = cfg.substrate, cfg.sequence
    with pytest.raises(rms.RmsError) as e:      # label >= n_labels
        rms.rms_substrate_create(sub.labels, 0.1, sub.D[:1], None, None, None, 1)
    assert e.value.code == -1
    S = rms.rms_substrate_create(sub.labels, 0.1, sub.D, sub.T2, sub.kappa, sub.label_class, 2)
    with pytest.raises(rms.RmsError) as e:
        rms.rms_walkers_init(S, 10, 0, np.zeros(2, np.uint8), 1)
    assert e.value.code == -4
    W = rms.rms_walkers_init(S, 10, 0, sub.label_allowed, 1)
    with pytest.raises(rms.RmsError) as e:      # hop longer than a voxel
        rms.rms_run(S, W, 1e-3, 10, seq.wave[:, :10], seq.gamp, seq.dirs, [10])
    assert e.value.code == -2
    with pytest.raises(rms.RmsError) as e:      # non-unit direction
        rms.rms_run(S, W, 2e-4, 10, seq.wave[:, :10], seq.gamp, seq.dirs * 2, [10])
    assert e.value.code == -1
    with pytest.raises(rms.RmsError) as e:      # unsorted snapshots
        rms.rms_run(S, W, 2e-4, 10, seq.wave[:, :10], seq.gamp, seq.dirs, [5, 4])
    assert e.value.code == -1
    assert W.steps_done() == 0
    S2 = rms.rms_substrate_create(sub.labels, 0.1, [2.0, 0.01], None, [[0, 5000.0], [5000.0, 0]], sub.label_class, 2)
    W2 = rms.rms_walkers_init(S2, 10, 0, None, 1)
    with pytest.raises(rms.RmsError) as e:      # Eq.3 above 1
        rms.rms_run(S2, W2, 2e-4, 10, seq.wave[:, :10], seq.gamp, seq.dirs, [10])
    assert e.value.code == -3


def test_full_size_bench_workload_against_the_oracle(rms):
    """The workload bench.py times, whole: cfg4 point on the full 500x500x2000 axon lattice, 1e6 walkers x 10,000
    steps, 60 directions x 11 b-values, in bench.py's launch configuration (device-resident labels, specialised
    kernel, spatial ordering, RMS_LAYOUT_AUTO | RMS_LATTICE_DICT as bench.py's defaults), against the oracle run on every one of
    those walkers (about a minute of host time).
    Plain north_star tolerances: >= 99.9 % same final voxel, |dS| <= 1e-4 for all 660 (b, direction), moments 1e-4."""
    import torch
    cfg = ri.make_config("cfg4", "full")
    n = cfg.n_walkers
    labels_dev = torch.from_numpy(cfg.substrate.labels.view(np.int16)).cuda()
    g = rms.simulate(cfg.substrate, cfg.sequence, n, cfg.seed, device_labels=labels_dev, read_walkers=True,
                     substrate_flags=rms.binding.RMS_LAYOUT_AUTO | rms.binding.RMS_LATTICE_DICT)
    assert g["substrate_info"]["dict_entries"] > 60_000
    o = oracle_run(cfg.substrate, cfg.sequence, n, cfg.seed)
    rep = compare(g, o, n)
    print("full-size cfg4", rep)
    assert g["n_launches"] >= 5 and g["kernel_ms"] > 0


def _same_trajectories(a, b, tag, exact_relax=True):
    """Two runs of the CUDA path that must have walked the same trajectories: positions, labels and counts bit for bit; the
    phase and signal sums may differ by the order of their fp64 additions only."""
    wa, wb = a["walkers"], b["walkers"]
    for k in ("vox", "off", "label") + (("relax",) if exact_relax else ()):
        assert np.array_equal(wa[k], wb[k]), (tag, k)
    assert np.allclose(wa["relax"], wb["relax"], rtol=0, atol=2e-8), tag
    assert a["n_encounters"] == b["n_encounters"] and a["n_permeations"] == b["n_permeations"], tag
    scale = max(1e-30, float(np.abs(wa["phi"]).max()))
    assert float(np.abs(wa["phi"] - wb["phi"]).max()) <= 1e-11 * scale, tag
    # (relaxation sums that differ in their last fp32 bit move the weights alpha = exp(-relax) by 1e-8)
    assert float(np.abs(a["S"] - b["S"]).max()) <= (1e-10 if exact_relax else 1e-7), tag
    rtol = 1e-12 if exact_relax else 1e-7
    assert np.allclose(a["m2"], b["m2"], rtol=rtol) and np.allclose(a["m4"], b["m4"], rtol=rtol), tag


def test_time_slices_of_the_specialised_kernel_leave_the_trajectories_alone(rms):
    """rms_step_fast.cu cuts the last one to two waves of blocks of a launch into time slices dealt from a queue.  Enough
    walkers for a whole-range wave and a sliced part (782 groups of 512), a launch long enough to be sliced (3 slices, the
    last one ragged, odd step count): the same run with RMS_RUN_NO_SLICES must end in the same place, fp32 and fp64,
    impermeable and permeable (whose relaxation sums are added slice by slice: fp32 rounding), octant and dictionary
    lattice; and the sliced permeable run holds north_star's tolerances against the oracle."""
    NO_SLICES, DICT = rms.binding.RMS_RUN_NO_SLICES, rms.binding.RMS_LATTICE_DICT
    n = 400_001
    c2, c3 = ri.make_config("cfg2", "test"), ri.make_config("cfg3", "test")
    seq = ri.pgse_sequence(2e-4, 6301, 0.3, 0.8, np.linspace(0.0, 4.0, 4), ri.fibonacci_dirs(6), snap_steps=[6301])
    for name, sub in (("cfg2", c2.substrate), ("cfg3", c3.substrate)):
        for flags in (0, 8):
            for sf in (0, DICT):
                whole = gpu_run(sub, seq, n, 11, flags=flags | NO_SLICES, substrate_flags=sf)
                sliced = gpu_run(sub, seq, n, 11, flags=flags, substrate_flags=sf)
                _same_trajectories(whole, sliced, (name, flags, sf), exact_relax=(name == "cfg2"))
                if name == "cfg3" and flags == 0 and sf == 0:
                    print("sliced cfg3 against the oracle", compare(sliced, oracle_run(sub, seq, n, 11), n))
    # two launches (a snapshot in the middle), both long enough to be sliced: the schedule is set up again for each; and
    # the kernel variants that can cancel a step (rejection sampling, ERL), which carry more state over a slice boundary
    seq2 = ri.pgse_sequence(2e-4, 9000, 0.4, 1.0, np.linspace(0.0, 4.0, 3), ri.fibonacci_dirs(3), snap_steps=[4500, 9000])
    RS, ERL = rms.binding.RMS_RUN_REJECTION_SAMPLING, rms.binding.RMS_RUN_ERL
    for flags in (0, 8, RS, ERL | 8):
        whole = gpu_run(c2.substrate, seq2, n, 12, flags=flags | NO_SLICES)
        sliced = gpu_run(c2.substrate, seq2, n, 12, flags=flags)
        assert sliced["n_launches"] == whole["n_launches"]
        _same_trajectories(whole, sliced, ("two launches", flags))


@pytest.mark.parametrize("dict_cap", [None, "40", "3"], ids=["full_dictionary", "escapes", "gives_up"])
def test_dictionary_lattice_walks_the_trajectories_of_the_octant_lattice(rms, monkeypatch, dict_cap):
    """RMS_LATTICE_DICT stores a 16-bit code per voxel and the octant words of the distinct neighbourhoods once; the words a
    walker reads are the same, so the trajectories are those of the octant lattice bit for bit: axons (impermeable,
    permeable), a cylinder, independent random labels, a one-voxel-wide box, both memory orders, fp32 and fp64 directions.
    RMS_DICT_CAP (a test hook of rms_substrate_create) shrinks the dictionary: 40 codes push most boundary voxels into the
    escape table; with 3 codes that table overflows too on some of the lattices and the build falls back to the octant lattice."""
    DICT = rms.binding.RMS_LATTICE_DICT
    if dict_cap:
        monkeypatch.setenv("RMS_DICT_CAP", dict_cap)
    c2, c3, c0 = ri.make_config("cfg2", "test"), ri.make_config("cfg3", "test"), ri.make_config("cfg0")
    seq_r = ri.pgse_sequence(2e-4, 400, 0.02, 0.04, [0.0, 20.0], np.eye(3), snap_steps=[400])
    cases = [("cfg2", c2.substrate, c2.sequence, 20_000), ("cfg3", c3.substrate, c3.sequence, 20_000),
             ("cfg0", c0.substrate, c0.sequence, 5_000),
             ("random", ri.random_lattice((12, 11, 10), n_labels=3, seed=9, place="all"), seq_r, 5_000),
             ("1x1x9", ri.random_lattice((1, 1, 9), n_labels=2, seed=2, place="all"), seq_r, 2_000)]
    seen = set()
    for name, sub, seq, n in cases:
        for layout in (rms.binding.RMS_LAYOUT_X_FASTEST, rms.binding.RMS_LAYOUT_Z_FASTEST):
            for flags in (0, 8):
                a = gpu_run(sub, seq, n, 5, flags=flags, substrate_flags=layout)
                b = gpu_run(sub, seq, n, 5, flags=flags, substrate_flags=layout | DICT)
                _same_trajectories(a, b, (name, layout, flags))
                info = b["substrate_info"]
                assert a["substrate_info"]["dict_entries"] == 0 and info["has_bricks"] == 1
                seen.add("octant" if info["dict_entries"] == 0 else ("escapes" if info["dict_escaped_voxels"] else "dictionary"))
                if dict_cap is None:
                    assert info["dict_entries"] > 1 and info["dict_escaped_voxels"] == 0
                    assert info["brick_bytes"] < a["substrate_info"]["brick_bytes"] or info["n_voxels"] < 100_000
    print("lattices in use", sorted(seen))
    assert {None: seen == {"dictionary"}, "40": "escapes" in seen, "3": "octant" in seen}[dict_cap]


def test_host_labels_uploaded_in_slabs_give_the_lattice_of_device_labels(rms):
    """rms_substrate_create uploads the host labels of a large lattice in slabs of z-planes on a stream of its own and builds
    the octant lattice chunk by chunk behind them.  The full axon lattice from host memory (pageable and pinned), in both
    memory orders and with RMS_LAYOUT_AUTO (decided on the first slab then), against the same lattice adopted from device
    memory: same membrane count, same trajectories (walkers over the whole box, enough steps to cross faces everywhere)."""
    import torch
    cfg = ri.make_config("cfg4", "full")
    sub = cfg.substrate
    seq = ri.pgse_sequence(2e-4, 300, 0.01, 0.03, [0.0, 1.0], np.eye(3), snap_steps=[300])
    n = 200_000
    labels_dev = torch.from_numpy(sub.labels.view(np.int16)).cuda()
    pinned = torch.from_numpy(sub.labels.view(np.int16)).pin_memory()
    import dataclasses
    sub_pinned = dataclasses.replace(sub, labels=pinned.numpy().view(np.uint16))
    for layout in (rms.binding.RMS_LAYOUT_X_FASTEST, rms.binding.RMS_LAYOUT_Z_FASTEST, rms.binding.RMS_LAYOUT_AUTO):
        ref = rms.simulate(sub, seq, n, 3, device_labels=labels_dev, read_walkers=True, substrate_flags=layout)
        for name, s_host in (("pageable", sub), ("pinned", sub_pinned)):
            g = rms.simulate(s_host, seq, n, 3, read_walkers=True, substrate_flags=layout)
            assert g["substrate_info"]["n_membrane_faces"] == ref["substrate_info"]["n_membrane_faces"], (layout, name)
            _same_trajectories(ref, g, (layout, name))
        # the dictionary lattice is built behind the slabs in the same way
        g = rms.simulate(sub_pinned, seq, n, 3, read_walkers=True, substrate_flags=layout | rms.binding.RMS_LATTICE_DICT)
        assert g["substrate_info"]["dict_entries"] > 60_000 and g["substrate_info"]["n_membrane_faces"] == ref["substrate_info"]["n_membrane_faces"]
        _same_trajectories(ref, g, (layout, "dictionary lattice, pinned"))
    assert ref["n_encounters"] > 100_000
    # a narrow box whose plane count is no multiple of the slab or chunk sizes (one block per row, ragged last chunk and slab)
    small = ri.random_lattice((40, 30, 1100 + 37), n_labels=3, seed=21, place="all")
    dev = torch.from_numpy(small.labels.view(np.int16)).cuda()
    for layout in (rms.binding.RMS_LAYOUT_X_FASTEST, rms.binding.RMS_LAYOUT_Z_FASTEST, rms.binding.RMS_LAYOUT_AUTO):
        ref = rms.simulate(small, seq, 50_000, 4, device_labels=dev, read_walkers=True, substrate_flags=layout)
        g = rms.simulate(small, seq, 50_000, 4, read_walkers=True, substrate_flags=layout)
        assert g["substrate_info"]["n_membrane_faces"] == ref["substrate_info"]["n_membrane_faces"]
        _same_trajectories(ref, g, ("narrow box", layout))


def test_general_kernel_and_id_order_agree_with_the_specialised_path(rms):
    # same inputs through the general step kernel and without spatial ordering: identical physics, so the results
    # agree with the oracle under the same tolerances, and with each other to rounding
    cfg = ri.make_config("cfg2", "test")
    n = cfg.n_walkers
    o = oracle_run(cfg.substrate, cfg.sequence, n, cfg.seed)
    for flags in (2, 4, 6):      # RMS_RUN_GENERAL_KERNEL, RMS_RUN_NO_ORDERING, both
        g = gpu_run(cfg.substrate, cfg.sequence, n, cfg.seed, flags=flags)
        print("flags", flags, compare(g, o, n))


def test_fp64_mode_stays_on_the_oracle_trajectories_over_a_long_run(rms):
    """RMS_RUN_FP64 on the reduced axon substrate for 200,000 steps (40 ms of diffusion, the length scale of
    BASELINE.json's configs 1-3): fp32 positions lose walkers at every convex membrane corner they pass within
    ~1e-6 voxel of and fall below 99.9 % same-voxel long before this; fp64 positions differ
    from the oracle's by ~1e-13 and must hold the plain tolerances."""
    cfg = ri.make_config("cfg2", "test")
    n, n_steps = 20_000, 200_000
    seq = ri.pgse_sequence(cfg.sequence.dt_ms, n_steps, 10.0, 25.0, np.linspace(0.0, 10.0, 5), ri.fibonacci_dirs(12),
                           snap_steps=[50_001, 100_000, n_steps])
    o = oracle_run(cfg.substrate, seq, n, cfg.seed)
    g64 = gpu_run(cfg.substrate, seq, n, cfg.seed, flags=8)
    rep = compare(g64, o, n)
    print("fp64 200k steps", rep)
    assert rep["n_diff"] <= 2 and rep["max_offset_diff"] < 1e-6          # offsets are read back as fp32
    g32 = gpu_run(cfg.substrate, seq, n, cfg.seed)
    same32 = float(np.all(g32["walkers"]["vox"] == o["final_vox"], axis=1).mean())
    print("fp32 same-voxel fraction at 200k steps:", same32)
    assert rep["same_voxel"] >= same32


def test_fp32_accuracy_envelope_on_the_axon_substrate(rms):
    """The fp32 path (fp32 direction arithmetic, exact fixed-point positions) parts company with the oracle only where a hop
    passes a convex membrane corner within its position error; the share of walkers that have done
    so grows like steps^1.5.  The measured curve on the reduced axon substrate, less a margin, so that a change that
    costs accuracy (a cheaper square root, sine or conversion) is caught even where it still passes 99.9 % on one case."""
    cfg = ri.make_config("cfg2", "test")
    n = 50_000
    for n_steps, floor in ((10_000, 0.9999), (40_000, 0.9985)):
        seq = ri.pgse_sequence(cfg.sequence.dt_ms, n_steps, 0.2 * n_steps * cfg.sequence.dt_ms, 0.5 * n_steps * cfg.sequence.dt_ms,
                               [0.0, 4.0], np.eye(3), snap_steps=[n_steps])
        o = oracle_run(cfg.substrate, seq, n, cfg.seed)
        g = gpu_run(cfg.substrate, seq, n, cfg.seed)
        same = float(np.all(g["walkers"]["vox"] == o["final_vox"], axis=1).mean())
        print("fp32 same-voxel fraction at", n_steps, "steps:", same)
        assert same >= floor, (n_steps, same)


def test_fp64_mode_general_kernel_permeable_and_table_waveforms(rms):
    # RMS_RUN_FP64 outside the specialised case: permeable + D contrast + T2 (cfg3 reduced), and a non-integer waveform
    c3 = ri.make_config("cfg3", "test")
    n3 = 100_000
    o = oracle_run(c3.substrate, c3.sequence, n3, c3.seed)
    for flags in (8, 8 | 2):       # the specialised kernel with fp64 directions (redo path for permeations); the general fp64 kernel
        g = gpu_run(c3.substrate, c3.sequence, n3, c3.seed, flags=flags)
        rep = compare(g, o, n3)
        print("fp64 cfg3 reduced, flags", flags, rep)
        assert rep["n_diff"] <= 2 and rep["perm_diff"] <= 2 and g["n_permeations"] > 0
    sub = ri.single_cylinder(24, 7.5, 0.1)
    n_steps = 801
    t = (np.arange(n_steps) + 1.0) / n_steps
    wave = np.stack([np.sin(2 * np.pi * t), np.clip(4 * np.minimum(t, 1 - t), 0, 1) * np.sign(0.5 - t)]).astype(np.float32)
    seq = ri.Sequence(dt_ms=2e-4, n_steps=n_steps, wave=wave, gamp=np.array([[0.0, 40.0, 90.0], [10.0, 60.0, 120.0]]),
                      dirs=ri.fibonacci_dirs(5), snap_steps=np.array([400, 801]))
    g = gpu_run(sub, seq, 100_000, 5, flags=8)
    o = oracle_run(sub, seq, 100_000, 5)
    rep = compare(g, o, 100_000)
    print("fp64 table waveforms", rep)
    assert rep["n_diff"] == 0


@pytest.mark.parametrize("name,n_ids", [("cfg1", 100_000), ("cfg2", 10_000), ("cfg3", 100_000)])
def test_full_length_configs_in_fp64_on_a_sample_of_walker_ids(rms, name, n_ids):
    """BASELINE.json configs 1-3 at their full lattice size and full number of steps (85,000 / 500,000 / 50,000), on
    the first n_ids walker ids -- cfg1 whole (all of its 1e5 walkers), cfg3 and cfg2 on 10 % and 1 % of theirs (what the
    oracle finishes in under a minute; trajectories depend on (seed, id) only, so the sample is exactly the corresponding
    slice of the full job) -- in RMS_RUN_FP64: plain tolerances."""
    import torch
    cfg = ri.make_config(name, "full")
    labels_dev = torch.from_numpy(cfg.substrate.labels.view(np.int16)).cuda()
    g = rms.simulate(cfg.substrate, cfg.sequence, n_ids, cfg.seed, flags=8, device_labels=labels_dev, read_walkers=True)
    g["_sub"], g["_seq"] = cfg.substrate, cfg.sequence
    o = oracle_run(cfg.substrate, cfg.sequence, n_ids, cfg.seed)
    rep = compare(g, o, n_ids)
    print("full length", name, cfg.sequence.n_steps, "steps", rep, "kernel_ms", g["kernel_ms"])
    assert rep["n_diff"] <= max(1, n_ids // 5000)


def test_per_cell_outputs_class_equals_label(rms):
    """S: section 8(f) N2 -- the paper reports its results per axon: class = label, so that signals and moments
    come out per cell.  13 classes on the reduced axon substrate, 300 on a lattice of random labels; more than 8
    classes take the class-ordered signal reduction."""
    import dataclasses
    cfg = ri.make_config("cfg2", "test")
    sub = cfg.substrate
    nL = len(sub.D)
    per_cell = dataclasses.replace(sub, label_class=np.arange(nL, dtype=np.uint16), n_classes=nL)
    n = cfg.n_walkers
    g = gpu_run(per_cell, cfg.sequence, n, cfg.seed)
    o = oracle_run(per_cell, cfg.sequence, n, cfg.seed)
    rep = compare(g, o, n)
    print("per-axon classes", nL, rep)
    assert g["sig_re"].shape[-1] == nL and g["sum_alpha"][0] == 0 and np.count_nonzero(g["sum_alpha"]) >= nL - 2
    # pooled over the classes it is the two-class run
    g2 = gpu_run(sub, cfg.sequence, n, cfg.seed)
    assert np.abs(g["S"] - g2["S"]).max() < 1e-9 and np.allclose(g["sig_re"].sum(-1), g2["sig_re"].sum(-1), atol=1e-6)
    # 300 classes, walkers everywhere, two waveforms, a snapshot on the way
    sub3 = ri.random_lattice((12, 11, 10), n_labels=300, seed=8)
    sub3 = dataclasses.replace(sub3, label_class=np.arange(300, dtype=np.uint16), n_classes=300)
    wave = np.stack([ri.pgse_wave(300, 100, 150), ri.pgse_wave(300, 40, 200)])
    seq = ri.Sequence(dt_ms=2e-4, n_steps=300, wave=wave, gamp=np.array([[0.0, 25.0], [5.0, 60.0]]), dirs=ri.fibonacci_dirs(3),
                      snap_steps=np.array([150, 300]))
    g = gpu_run(sub3, seq, 20000, 3)
    o = oracle_run(sub3, seq, 20000, 3)
    print("300 classes", compare(g, o, 20000))
    assert g["class_flow"].shape == (2, 300, 300) and g["class_flow"].sum() == 2 * 20000


def test_absorbing_membranes_magnetisation_transfer(rms):
    """S: section 8(f) N3 -- Eq.4: an encounter saturates the walker with P_MT = rho ds / D C_d; its weight is 0
    from then on.  Absorbing cylinder wall (impermeable), and permeable + absorbing slabs with D and T2 contrast; fp32 and
    fp64; saturation counts against the oracle, exactly where the trajectories agree."""
    import dataclasses
    cyl = ri.single_cylinder(24, 8.5, 0.1)
    rho = np.zeros((2, 2), np.float32); rho[1, 0] = 3.0
    cyl = dataclasses.replace(cyl, rho=rho)
    seq = ri.pgse_sequence(2e-4, 1500, 0.1, 0.15, [0.0, 2.0], np.eye(3), snap_steps=[500, 1500])
    n = 100_000
    o = oracle_run(cyl, seq, n, 23)
    for flags in (0, 2, 8):
        g = gpu_run(cyl, seq, n, 23, flags=flags)
        rep = compare(g, o, n)
        print("absorbing cylinder, flags", flags, rep, "saturated", g["n_saturations"], o["n_saturations"])
        assert abs(g["n_saturations"] - o["n_saturations"]) <= 2 * rep["n_diff"] + (0 if flags == 8 else 2)
        assert 0.2 * n < g["n_saturations"] < 0.9 * n and abs(g["sum_alpha"].sum() - (n - g["n_saturations"])) < 1e-6
    sl = ri.slabs(6, 5, (3, 2), 0.1, D_extra=2.0, D_intra=1.0, kappa_membrane=4.0, T2_extra=0.3, T2_intra=0.6)
    rho = np.array([[0.0, 1.5], [0.7, 0.0]], np.float32)
    sl = dataclasses.replace(sl, rho=rho)
    seq = ri.pgse_sequence(2e-4, 800, 0.05, 0.08, [0.0, 5.0], ri.fibonacci_dirs(4), snap_steps=[399, 800])
    o = oracle_run(sl, seq, n, 29)
    for flags in (0, 2, 8):
        g = gpu_run(sl, seq, n, 29, flags=flags)
        rep = compare(g, o, n)
        print("absorbing + permeable slabs, flags", flags, rep, "saturated", g["n_saturations"], o["n_saturations"])
        assert abs(g["n_saturations"] - o["n_saturations"]) <= 2 * rep["n_diff"] + (0 if flags == 8 else 2) and g["n_permeations"] > 1000
    bad = dataclasses.replace(sl, rho=np.array([[0.0, 200.0], [0.0, 0.0]], np.float32))
    with pytest.raises(rms.RmsError) as e:
        gpu_run(bad, seq, 10, 1)
    assert e.value.code == -3          # RMS_ERR_P_RANGE: P_MT > 1


def test_rejection_sampling_interaction(rms):
    """S: section 8(f) N4 -- the paper's other membrane interaction (Appendix B; R21): a step that meets a membrane it
    does not cross is cancelled.  Impermeable cylinder (integer and non-integer waveforms: both modes of the fp32 general
    kernel), equal-D permeable slabs with T2 contrast (P_T = A / (1 + A)), and an absorbing wall on top; fp32 and fp64,
    against the oracle run with interaction = 1.  The elastic-collision result must differ (the flag is not a no-op)."""
    import dataclasses
    RS = rms.binding.RMS_RUN_REJECTION_SAMPLING
    n = 100_000
    cyl = ri.single_cylinder(24, 8.5, 0.1)
    seq = ri.pgse_sequence(2e-4, 1500, 0.1, 0.15, [0.0, 2.0], np.eye(3), snap_steps=[500, 1500])
    o = oracle_run(cyl, seq, n, 31, interaction=1)
    o_ecs = oracle_run(cyl, seq, n, 31)
    assert np.abs(o["S"] - o_ecs["S"]).max() > 1e-3
    for flags in (RS, RS | 8, RS | 2, RS | 2 | 8):      # specialised kernel (fp32 / fp64 directions), general kernels (fp32 / fp64)
        g = gpu_run(cyl, seq, n, 31, flags=flags)
        print("rejection sampling, cylinder, flags", flags, compare(g, o, n))
        assert g["n_encounters"] > n and g["n_permeations"] == 0
    seq_f = dataclasses.replace(seq, wave=(seq.wave * 0.37).astype(np.float32))            # table-driven waveform
    o = oracle_run(cyl, seq_f, n, 32, interaction=1)
    for flags in (RS, RS | 8):
        print("rejection sampling, non-integer waveform, flags", flags, compare(gpu_run(cyl, seq_f, n, 32, flags=flags), o, n))
    sl = ri.slabs(6, 5, (3, 2), 0.1, D_extra=2.0, D_intra=2.0, kappa_membrane=4.0, T2_extra=0.3, T2_intra=0.6)
    sl = dataclasses.replace(sl, rho=np.array([[0.0, 0.4], [0.2, 0.0]], np.float32))
    seq = ri.pgse_sequence(2e-4, 800, 0.05, 0.08, [0.0, 5.0], ri.fibonacci_dirs(4), snap_steps=[399, 800])
    o = oracle_run(sl, seq, n, 33, interaction=1)
    for flags in (RS, RS | 8):
        g = gpu_run(sl, seq, n, 33, flags=flags)
        rep = compare(g, o, n)
        print("rejection sampling, permeable + absorbing slabs, flags", flags, rep, "permeations", g["n_permeations"], o["n_permeations"])
        assert g["n_permeations"] > 1000 and abs(g["n_permeations"] - o["n_permeations"]) <= 4 * rep["n_diff"] + 2
        assert abs(g["n_saturations"] - o["n_saturations"]) <= 2 * rep["n_diff"] + 2
    bad = ri.slabs(6, 5, (3, 2), 0.1, D_extra=2.0, D_intra=1.0, kappa_membrane=4.0)
    with pytest.raises(rms.RmsError) as e:
        gpu_run(bad, seq, 10, 1, flags=RS)
    assert e.value.code == -7          # RMS_ERR_UNSUPPORTED: Appendix B.1 gives P_T for equal D only


def test_t1_weighting_in_the_mixing_time_of_a_stimulated_echo(rms):
    """S: section 8(f) N3, second half -- P:135 (R22): the steps of the mixing time relax with T1 of the walker's compartment.
    Impermeable cylinder (specialised kernels), permeable slabs with D, T2 and T1 contrast (general kernels) and weakly
    permeable ones (the redo path of the specialised kernel); snapshots inside the window; windows touching step 1 and
    the last step; fp32 and fp64."""
    import dataclasses
    n = 100_000
    cyl = dataclasses.replace(ri.single_cylinder(24, 8.5, 0.1), T1=np.array([0.9, 0.4], np.float32))
    cyl = dataclasses.replace(cyl, T2=np.array([0.3, 0.15], np.float32))
    base = ri.pgse_sequence(2e-4, 1500, 0.06, 0.24, [0.0, 2.0], np.eye(3), snap_steps=[500, 900, 1500])   # lobes 1..300, 1201..1500
    for first, cnt in ((301, 900), (1, 1500), (1500, 1), (700, 1)):
        seq = dataclasses.replace(base, mix_first_step=first, mix_n_steps=cnt)
        if cnt == 1500:
            seq = dataclasses.replace(seq, wave=np.zeros_like(base.wave))
        o = oracle_run(cyl, seq, n, 41)
        for flags in (0, 2, 8):
            g = gpu_run(cyl, seq, n, 41, flags=flags)
            print("stimulated echo, cylinder, window", first, cnt, "flags", flags, compare(g, o, n))
    o_t2 = oracle_run(cyl, base, n, 41)
    assert abs(o["sum_alpha"].sum() / o_t2["sum_alpha"].sum() - 1) > 1e-4                     # the window is not a no-op
    for kappa, name in ((4.0, "permeable"), (0.05, "weakly permeable")):
        sl = ri.slabs(6, 5, (3, 2), 0.1, D_extra=2.0, D_intra=1.0, kappa_membrane=kappa, T2_extra=0.3, T2_intra=0.6)
        sl = dataclasses.replace(sl, T1=np.array([1.5, 0.2], np.float32))
        seq = ri.pgse_sequence(2e-4, 800, 0.03, 0.13, [0.0, 5.0], ri.fibonacci_dirs(4), snap_steps=[399, 800])  # lobes 1..150, 651..800
        seq = dataclasses.replace(seq, mix_first_step=151, mix_n_steps=500)
        o = oracle_run(sl, seq, n, 43)
        for flags in (0, 2, 8):
            g = gpu_run(sl, seq, n, 43, flags=flags)
            print("stimulated echo,", name, "slabs, flags", flags, compare(g, o, n), "permeations", g["n_permeations"])
            assert g["n_permeations"] > 100
    with pytest.raises(rms.RmsError) as e:
        gpu_run(cyl, dataclasses.replace(base, mix_first_step=1400, mix_n_steps=200), 10, 1)
    assert e.value.code == -1          # RMS_ERR_ARG: the window leaves 1 .. n_steps


def _rotations(k, seed):
    q, _ = np.linalg.qr(np.random.default_rng(seed).normal(size=(k, 3, 3)))
    return q * np.sign(np.linalg.det(q))[:, None, None]


def test_tensor_waveforms_b_tensor_encoding(rms):
    """S: section 8(f) N1, "arbitrary g(tau) shapes (B-tensor encoding)" -- P:336 (R23): gradient waveforms that change
    direction, phi = gamp dt l_p sum_a (R e_a) . Phi_{m_a}, evaluated in the signal reduction from the phase vectors of
    the run's scalar waveforms.  Against oracle.tensor_signal on the same walkers: two classes (per-block sums), 13 classes
    (class-ordered reduction), fp32 and fp64 walks, a permeable substrate with T2 contrast; the scalar signals of the same
    run must not change; sharded runs merge."""
    import dataclasses
    import oracle
    n_steps = 600
    lobes = np.zeros((4, n_steps), np.float32)
    for a in range(3):                       # three lobe pairs, one after the other (spherical encoding) ...
        lobes[a, 200 * a:200 * a + 80] = 1.0
        lobes[a, 200 * a + 110:200 * a + 190] = -1.0
    lobes[3] = ri.pgse_wave(n_steps, 150, 400) * 0.5                        # ... and a plain pulsed gradient of half amplitude
    tw = np.array([[0, 1, 2], [3, -1, 0], [-1, -1, -1], [1, 1, 1]], np.int32)
    tg = np.array([[0.0, 900.0, 2500.0], [300.0, 1200.0, 2000.0], [1.0, 2.0, 3.0], [100.0, 700.0, 1500.0]])
    rots = np.concatenate([np.eye(3)[None], _rotations(4, 3)])
    seq = ri.Sequence(dt_ms=2e-4, n_steps=n_steps, wave=lobes, gamp=np.array([[0.0, 500.0, 1500.0]] * 4), dirs=ri.fibonacci_dirs(3),
                      snap_steps=np.array([300, n_steps]), tensor_waves=tw, tensor_gamp=tg, rots=rots)
    cfg = ri.make_config("cfg2", "test")
    axons = cfg.substrate
    nL = len(axons.D)
    per_cell = dataclasses.replace(axons, label_class=np.arange(nL, dtype=np.uint16), n_classes=nL)
    sl = ri.slabs(6, 5, (3, 2), 0.1, D_extra=2.0, D_intra=1.0, kappa_membrane=4.0, T2_extra=0.3, T2_intra=0.6)
    n = 100_000
    for name, sub in (("cylinder", ri.single_cylinder(24, 8.5, 0.1)), ("axons, per-cell classes", per_cell), ("permeable slabs", sl)):
        o = oracle_run(sub, seq, n, 71)
        ot = oracle.tensor_signal(sub, seq, o)
        assert np.abs(ot["tS"][0]).min() < 0.9                              # real attenuations
        for flags in (0, 8):
            g = gpu_run(sub, seq, n, 71, flags=flags)
            rep = compare(g, o, n)
            tol = 1e-4 + 2.0 * rep["n_diff"] / n
            d = np.abs(g["tS"] - ot["tS"])
            scale = float(o["sum_alpha"].sum())
            d_cls = max(np.abs(g["tsig_re"] - ot["tsig_re"]).max(), np.abs(g["tsig_im"] - ot["tsig_im"]).max()) / scale
            print("tensor waveforms,", name, "flags", flags, rep, "max |d tS|", d.max(), "per class", d_cls)
            assert g["tS"].shape == (4, 3, 5) and g["tsig_re"].shape == (4, 3, 5, sub.n_classes)
            assert d.max() <= tol and d_cls <= tol
            assert np.abs(g["tS"][2] - 1.0).max() < 1e-12                   # all axes off: no phase
    # the scalar outputs do not depend on the tensor ones riding along
    plain = dataclasses.replace(seq, tensor_waves=None, tensor_gamp=None, rots=None)
    g0 = gpu_run(sl, plain, n, 71)
    g1 = gpu_run(sl, seq, n, 71)
    assert np.abs(g0["S"] - g1["S"]).max() < 1e-12 and "tS" not in g0
    # two shards of walker ids merge into the whole job
    parts = [gpu_run(sl, seq, n // 2, 71, first_id=f) for f in (0, n // 2)]
    m = rms.api.merge_results(parts, np.array([300, n_steps]) * 2e-4)
    assert np.abs(m["tS"] - g1["tS"]).max() < 1e-12 and np.abs(m["S"] - g1["S"]).max() < 1e-12
    with pytest.raises(rms.RmsError) as e:
        gpu_run(sl, dataclasses.replace(seq, tensor_waves=np.array([[0, 4, 1]], np.int32), tensor_gamp=tg[:1]), 10, 1)
    assert e.value.code == -1          # RMS_ERR_ARG: waveform 4 does not exist


def test_spin_concentrations_permeation_and_placement(rms):
    """S: section 8(f) N4, "concentration-dependent (Eq.C.9)" and Baxter-Frank (Eq.C.15) -- Appendix C.2-C.3 (R24): per-label spin
    concentrations change the permeation table and the initial density.  Tables against the oracle's (fp32-rounded on
    both sides: identical), placement bit exact, the walk on slabs with D, T2 and concentration contrast (general and
    specialised-with-redo kernels, fp64), on a lattice of random labels with kappa = inf pairs, and a label without
    spins that is allowed but never populated."""
    import dataclasses
    import oracle
    n = 100_000
    seq = ri.pgse_sequence(2e-4, 800, 0.05, 0.08, [0.0, 5.0], ri.fibonacci_dirs(4), snap_steps=[399, 800])
    for kappa, name in ((4.0, "permeable"), (0.05, "weakly permeable")):
        sl = ri.slabs(6, 5, (3, 2), 0.1, D_extra=2.0, D_intra=1.0, kappa_membrane=kappa, T2_extra=0.3, T2_intra=0.6, place="all")
        sl = dataclasses.replace(sl, conc=np.array([1.0, 0.4], np.float32))
        o = oracle_run(sl, seq, n, 81)
        _, P = oracle.tables(sl.D, sl.kappa, sl.voxel_um, seq.dt_ms, conc=sl.conc)
        S = rms.binding.rms_substrate_create(sl.labels, sl.voxel_um, sl.D, sl.T2, sl.kappa, sl.label_class, sl.n_classes, conc=sl.conc)
        _, Pg = S.tables(seq.dt_ms)
        S.destroy()
        assert np.array_equal(Pg.astype(np.float64), P) and P[0, 1] != P[1, 0]
        n_intra = int((o["init_vox"][:, 0] % 11 >= 6).sum())
        assert abs(n_intra / n - 0.4 * 5 / (6 + 0.4 * 5)) < 0.015                    # density ~ c
        for flags in (0, 2, 8):
            g = gpu_run(sl, seq, n, 81, flags=flags)
            print("spin concentrations,", name, "slabs, flags", flags, compare(g, o, n), "permeations", g["n_permeations"])
            assert g["n_permeations"] == o["n_permeations"] or flags != 8
    rl = ri.random_lattice((12, 11, 10), n_labels=5, seed=9, D_extra=2.0, D_intra=1.2, place="all")
    kap = np.full((5, 5), 3.0, np.float32); kap[0, 1] = kap[1, 0] = np.inf; kap[2, 3] = kap[3, 2] = np.inf
    rl = dataclasses.replace(rl, kappa=kap, conc=np.array([1.0, 0.7, 0.5, 0.5, 0.0], np.float32))
    o = oracle_run(rl, seq, n, 82)
    assert not np.any(o["final_label"] == 4) and o["n_permeations"] > 10000
    for flags in (0, 8):
        print("spin concentrations, random labels, flags", flags, compare(gpu_run(rl, seq, n, 82, flags=flags), o, n))
    with pytest.raises(rms.RmsError) as e:
        gpu_run(dataclasses.replace(rl, conc=np.array([1.0, -1.0, 1, 1, 1], np.float32)), seq, 10, 1)
    assert e.value.code == -1          # RMS_ERR_ARG


def test_equal_step_length_random_leap_interaction(rms):
    """S: section 8(f) N4 -- ERL, the paper's third interaction (Appendix A; R25): a step that meets a membrane is
    cancelled and retried in a new direction.  Impermeable cylinder (integer and non-integer waveforms), the reduced axon
    substrate, a lattice of random labels with kappa = inf pairs (passages before the cancelling face are undone) and a
    hop of 0.9 voxel (many retries); fp32 and fp64, against the oracle's interaction = 2."""
    import dataclasses
    ERL = rms.binding.RMS_RUN_ERL
    n = 100_000
    cyl = ri.single_cylinder(24, 8.5, 0.1)
    seq = ri.pgse_sequence(2e-4, 1500, 0.1, 0.15, [0.0, 2.0], np.eye(3), snap_steps=[500, 1500])
    o = oracle_run(cyl, seq, n, 95, interaction=2)
    assert np.abs(o["S"] - oracle_run(cyl, seq, n, 95, interaction=1)["S"]).max() > 1e-3       # not rejection sampling
    # the specialised kernel (fp32, fp64 directions) and, with RMS_RUN_GENERAL_KERNEL = 2, the general ones
    ALL = (ERL, ERL | 8, ERL | 2, ERL | 2 | 8)
    for flags in ALL:
        g = gpu_run(cyl, seq, n, 95, flags=flags)
        print("ERL, cylinder, flags", flags, compare(g, o, n))
        assert g["n_encounters"] == o["n_encounters"] or not (flags & 8)
    seq_f = dataclasses.replace(seq, wave=(seq.wave * 0.37).astype(np.float32))
    o = oracle_run(cyl, seq_f, n, 96, interaction=2)
    for flags in ALL:
        print("ERL, non-integer waveform, flags", flags, compare(gpu_run(cyl, seq_f, n, 96, flags=flags), o, n))
    cfg = ri.make_config("cfg2", "test")
    seq_a = dataclasses.replace(cfg.sequence)
    o = oracle_run(cfg.substrate, seq_a, 100_000, 97, interaction=2)
    for flags in ALL:
        print("ERL, axons, flags", flags, compare(gpu_run(cfg.substrate, seq_a, 100_000, 97, flags=flags), o, 100_000))
    print("ERL, axons, dictionary lattice", compare(gpu_run(cfg.substrate, seq_a, 100_000, 97, flags=ERL, substrate_flags=rms.binding.RMS_LATTICE_DICT), o, 100_000))
    hop = 0.9 ** 2 * 0.01 / (6 * 2e-4)
    rl = ri.random_lattice((12, 11, 10), n_labels=4, seed=9, D_extra=hop, D_intra=hop, place="all")
    kap = np.zeros((4, 4), np.float32); kap[0, 1] = kap[1, 0] = np.inf; kap[2, 3] = kap[3, 2] = np.inf
    rl = dataclasses.replace(rl, kappa=kap)
    seq_r = ri.pgse_sequence(2e-4, 400, 0.02, 0.04, [0.0, 20.0], np.eye(3), snap_steps=[400])
    o = oracle_run(rl, seq_r, n, 98, interaction=2)
    assert o["n_permeations"] > 1000 and o["n_encounters"] > 5 * n * 400 // 10
    # (with kappa = inf pairs ERL stays on the general kernels: the specialised one would redo every step in its fp32 side path)
    for flags in (ERL, ERL | 8):
        g = gpu_run(rl, seq_r, n, 98, flags=flags)
        rep = compare(g, o, n)
        print("ERL, random labels, hop 0.9 voxel, flags", flags, rep, "permeations", g["n_permeations"], o["n_permeations"])
        assert abs(g["n_permeations"] - o["n_permeations"]) <= 8 * rep["n_diff"] + 2
    perm = ri.slabs(6, 5, (3, 2), 0.1, D_extra=2.0, D_intra=2.0, kappa_membrane=4.0)
    with pytest.raises(rms.RmsError) as e:
        gpu_run(perm, seq, 10, 1, flags=ERL)
    assert e.value.code == -7          # RMS_ERR_UNSUPPORTED: the paper rules ERL out for exchange


def test_walkers_per_axon_placement_and_volume_weighted_sum(rms):
    """S: section 8(f) N2, "volume-weighted sums; walkers-per-axon placement" -- P:258-266 (R26): placement weights per label
    (bit exact against the oracle), the voxel count per label on the device, and the volume-weighted sum of the per-cell
    signals; with w_L = 1 / V_L every axon gets the same expected number of walkers."""
    import dataclasses
    import oracle
    cfg = ri.make_config("cfg2", "test")
    sub = cfg.substrate
    nL = sub.n_labels
    vol = np.bincount(sub.labels.ravel(), minlength=nL)
    intra = np.nonzero(np.asarray(sub.label_allowed) != 0)[0]
    per_cell = dataclasses.replace(sub, label_class=np.arange(nL, dtype=np.uint16), n_classes=nL)
    S = rms.rms_substrate_create(per_cell.labels, per_cell.voxel_um, per_cell.D, per_cell.T2, per_cell.kappa, per_cell.label_class, nL)
    assert np.array_equal(rms.rms_substrate_label_volumes(S), vol.astype(np.uint64))
    S.destroy()
    big = ri.random_lattice((70, 33, 41), n_labels=9000, seed=4)            # more labels than the shared-memory histogram holds
    S = rms.rms_substrate_create(big.labels, big.voxel_um, big.D, big.T2, big.kappa, big.label_class, big.n_classes)
    assert np.array_equal(rms.rms_substrate_label_volumes(S), np.bincount(big.labels.ravel(), minlength=9000).astype(np.uint64))
    S.destroy()
    w = np.zeros(nL, np.float32); w[intra] = (1.0 / vol[intra]).astype(np.float32)
    seq = ri.pgse_sequence(2e-4, 1500, 0.1, 0.15, [0.0, 1.0, 3.0], np.eye(3)[:2], snap_steps=[1500])
    n = 30000
    o = oracle.run(per_cell, seq, n, 37, n_threads=oracle.rms_oracle.default_threads(), per_walker=True, label_weight=w)
    for flags in (0, 8):
        g = rms.simulate(per_cell, seq, n, 37, flags=flags, read_walkers=True, label_weight=w)
        rep = compare(g, o, n)                                               # includes the bit-exact placement
        got = rms.rms_volume_weighted_signal(g, vol.astype(float))
        want = oracle.volume_weighted_signal(o, vol.astype(float))
        print("walkers per axon, flags", flags, rep, "max |d S_vw|", np.abs(got - want).max())
        assert np.abs(got - want).max() <= 1e-4 + 2.0 * rep["n_diff"] / n
    counts = np.bincount(g["walkers"]["label"], minlength=nL)[intra]
    assert counts.sum() == n and counts.min() > 0.8 * n / intra.size and counts.max() < 1.2 * n / intra.size
    with pytest.raises(rms.RmsError) as e:
        rms.simulate(per_cell, seq, 10, 1, label_weight=np.zeros(nL, np.float32))
    assert e.value.code == -4          # RMS_ERR_NO_SPACE


def test_degenerate_and_ragged_cases(rms):
    # one walker; 1, 2, 3 steps with a snapshot on every step; no waveform / no directions; hop of 0.99 voxel (three
    # interactions in most steps); a single-voxel pore (every face a membrane: the corner reflector of Fig.2)
    sub = ri.single_cylinder(16, 5.5, 0.1)
    for n_steps in (1, 2, 3):
        seq = ri.Sequence(dt_ms=2e-4, n_steps=n_steps, wave=np.ones((1, n_steps), np.float32), gamp=np.array([[0.0, 300.0]]),
                          dirs=np.eye(3), snap_steps=np.arange(1, n_steps + 1))
        for n in (1, 129):
            print("steps", n_steps, "walkers", n, compare(gpu_run(sub, seq, n, 3), oracle_run(sub, seq, n, 3), n,
                                                              few_walkers=True))   # about 1 and 129 walkers: ragged launch shapes
    seq0 = ri.Sequence(dt_ms=2e-4, n_steps=200, wave=np.zeros((0, 200), np.float32), gamp=np.zeros((0, 0)), dirs=np.eye(3),
                       snap_steps=np.array([100, 200]))
    g, o = gpu_run(sub, seq0, 100_000, 4), oracle_run(sub, seq0, 100_000, 4)
    print("no waveform", compare(g, o, 100_000))
    assert g["S"].size == 0 and g["m2"].shape == (2, 3, 2)
    seq1 = ri.Sequence(dt_ms=2e-4, n_steps=200, wave=ri.pgse_wave(200, 50, 100)[None], gamp=np.array([[0.0, 50.0]]),
                       dirs=np.zeros((0, 3)), snap_steps=np.zeros(0, np.int64))
    g, o = gpu_run(sub, seq1, 100_000, 4), oracle_run(sub, seq1, 100_000, 4)
    print("no directions", compare(g, o, 100_000))
    # hop length 0.99 voxel: D = 0.99^2 l_p^2 / (6 dt)
    big = ri.random_lattice((6, 5, 7), n_labels=2, seed=5, D_extra=0.99 ** 2 * 0.01 / (6 * 2e-4), D_intra=0.99 ** 2 * 0.01 / (6 * 2e-4))
    seq = ri.pgse_sequence(2e-4, 300, 0.02, 0.03, [0.0, 20.0], np.eye(3), snap_steps=[300])
    for flags in (0, 2, 8):
        print("hop 0.99 voxel, flags", flags, compare(gpu_run(big, seq, 100_000, 6, flags=flags), oracle_run(big, seq, 100_000, 6), 100_000))
    lab = np.zeros((3, 3, 3), np.uint16); lab[1, 1, 1] = 1
    pore = ri.Substrate(labels=lab, voxel_um=0.1, D=np.array([2.0, 2.0], np.float32), T2=np.array([np.inf, np.inf], np.float32),
                        kappa=np.zeros((2, 2), np.float32), label_class=np.array([0, 1], np.uint16), n_classes=2,
                        label_allowed=np.array([0, 1], np.uint8))
    g, o = gpu_run(pore, seq, 100_000, 8), oracle_run(pore, seq, 100_000, 8)
    print("single-voxel pore", compare(g, o, 100_000))
    assert np.all(g["walkers"]["vox"] == 1) and g["n_encounters"] > 100_000 * 300 * 0.5


def test_gather_probe_reports_sane_ceilings(rms):
    l2 = rms.binding.rms_gather_probe(32 << 20, 4, 256)
    hbm = rms.binding.rms_gather_probe(1 << 30, 2, 128)
    print("gather ceilings: L2-resident %.3g /s, HBM %.3g /s" % (l2, hbm))
    assert l2 > hbm > 1e9
    with pytest.raises(rms.RmsError):
        rms.binding.rms_gather_probe(1 << 20, 3, 128)


def test_tables_match_oracle(rms):
    import oracle
    D = np.array([2.0, 1.0, 0.5], np.float32)
    kap = np.array([[0, 0.02, 0.4], [0.02, 0, np.inf], [0.4, np.inf, 0]], np.float32)
    lab = np.zeros((2, 2, 3), np.uint16)
    S = rms.rms_substrate_create(lab, 0.1, D, None, kap, None, 1)
    s_g, P_g = S.tables(2e-4)
    s_o, P_o = oracle.tables(D, kap, 0.1, 2e-4)
    assert np.array_equal(s_g.astype(np.float64), s_o) and np.array_equal(P_g.astype(np.float64), P_o)
    info = S.info()
    assert info["n_membrane_faces"] == 0 and info["has_bricks"] == 1


def test_philox_of_the_cuda_path_matches_curand_and_the_oracle(rms, tmp_path):
    """K1 (S: section 8(c)): the product's Philox4x32-10 against cuRAND's Philox4_32_10 generator (a third implementation, NVIDIA's)
    and against the oracle's, on 4096 (key, counter) pairs spread over all four counter words."""
    import pathlib
    import subprocess
    import oracle
    src = pathlib.Path(__file__).resolve().parent / "cuda" / "philox_vs_curand.cu"
    exe = tmp_path / "philox_vs_curand"
    subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-std=c++17", "-o", str(exe), str(src)], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()
    v = np.array([int(x, 16) for x in out], np.uint64).reshape(-1, 8)
    assert v.shape[0] == 4096 and np.array_equal(v[:, :4], v[:, 4:])
    seed = 0x123456789ABCDEF1
    for t in (0, 1, 77, 4095):
        c01, c23 = (7919 * t * 1000003 + 1) & (2 ** 64 - 1), ((104729 * t << 20) + 3) & (2 ** 64 - 1)
        ctr = [c01 & 0xFFFFFFFF, c01 >> 32, c23 & 0xFFFFFFFF, c23 >> 32]
        ref = oracle.rms_oracle.philox4x32_10(ctr, [seed & 0xFFFFFFFF, seed >> 32])
        assert np.array_equal(ref.astype(np.uint64), v[t, :4])
