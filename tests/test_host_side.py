"""CPU-side tests of the product: the C-ABI library loads and exports every symbol include/rms.h declares, fails
loudly without a GPU (no CPU fallback), its pure-host entry point rms_normalise computes Eq.7 / P:174, and the
walker-id sharding + the one exchange step of a multi-process job (sum of the accumulators) work over gloo with
world_size 2.  No kernel is launched here."""
import os
import re
import socket
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def rms():
    import paper_2012_06478_b200 as rms
    from paper_2012_06478_b200 import build
    build.build()
    rms.load_library()
    return rms


def _declared_functions():
    text = (ROOT / "include" / "rms.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rms_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(rms):
    import ctypes
    names = _declared_functions()
    assert {"rms_substrate_create", "rms_walkers_init", "rms_run"} <= set(names)      # the three calls north_star names
    lib = ctypes.CDLL(str(rms.binding.LIB_PATH))
    for nm in names:
        assert hasattr(lib, nm), nm
    assert set(rms.binding.EXPORTS) == set(names)
    lib.rms_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.rms_version()


def test_no_cpu_fallback_without_a_gpu(rms):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    lab = np.zeros((4, 4, 4), np.uint16)
    with pytest.raises(rms.RmsError) as e:
        rms.rms_substrate_create(lab, 0.1, np.array([2.0], np.float32))
    assert e.value.code == -6 and "no CPU fallback" in str(e.value)      # RMS_ERR_CUDA


def test_product_does_not_import_the_oracle():
    pat = re.compile(r"^\s*(from|import)\s+oracle\b|import_module\(.oracle|#\s*include.*oracle|oracle[/.]rms_oracle", re.M)
    files = [p for p in (ROOT / "paper_2012_06478_b200").rglob("*") if p.suffix in (".py", ".cu", ".cuh", ".h")]
    files += [ROOT / "include" / "rms.h"]
    assert len(files) > 8
    for p in files:
        assert not pat.search(p.read_text()), p


def test_rms_normalise_is_eq7_and_the_narrow_pulse_moments(rms):
    rng = np.random.default_rng(5)
    nC, nW, nG, nD, nS = 3, 2, 4, 5, 2
    r = dict(sum_alpha=rng.uniform(10, 20, nC), sig_re=rng.normal(size=(nW, nG, nD, nC)), sig_im=rng.normal(size=(nW, nG, nD, nC)),
             m2=rng.uniform(1, 2, (nS, nD, nC)), m4=rng.uniform(3, 9, (nS, nD, nC)), snap_alpha=rng.uniform(10, 20, (nS, nC)))
    t = np.array([3.0, 7.5])
    out = rms.binding.rms_normalise(r, t)
    S = (r["sig_re"].sum(-1) + 1j * r["sig_im"].sum(-1)) / r["sum_alpha"].sum()          # Eq.7, classes pooled
    assert np.allclose(out["S"], S, rtol=1e-14)
    a = r["snap_alpha"].sum(-1)[:, None]
    x2, x4 = r["m2"].sum(-1) / a, r["m4"].sum(-1) / a
    assert np.allclose(out["Dapp"], x2 / (2 * t[:, None]), rtol=1e-14)                     # D = <a X^2> / (2 t <a>)
    assert np.allclose(out["Kapp"], x4 / x2 ** 2 - 3.0, rtol=1e-13)                        # K, both moments over <a> (R14)


def test_rms_volume_weighted_signal_is_the_volume_weighted_sum_of_per_class_signals(rms):
    rng = np.random.default_rng(6)
    nC, nW, nG, nD = 5, 2, 3, 4
    r = dict(sum_alpha=np.array([7.0, 0.0, 3.0, 11.0, 2.0]), sig_re=rng.normal(size=(nW, nG, nD, nC)), sig_im=rng.normal(size=(nW, nG, nD, nC)))
    V = np.array([10.0, 99.0, 1.0, 4.0, 6.0])
    use = r["sum_alpha"] > 0                                                              # class 1 holds no walkers: left out
    want = (((r["sig_re"] + 1j * r["sig_im"])[..., use] / r["sum_alpha"][use]) * V[use]).sum(-1) / V[use].sum()   # P:266, R26
    got = rms.binding.rms_volume_weighted_signal(r, V)
    assert got.shape == (nW, nG, nD) and np.allclose(got, want, rtol=1e-14)
    with pytest.raises(rms.RmsError):
        rms.binding.rms_volume_weighted_signal(dict(r, sum_alpha=np.zeros(nC)), V)


def test_shard_range_partitions_the_walker_ids(rms):
    for n, world in ((10, 3), (1_000_000, 8), (7, 8), (0, 2)):
        got = [rms.api.shard_range(r, world, n) for r in range(world)]
        assert got[0][0] == 0 and sum(c for _, c in got) == n
        for (f0, c0), (f1, _) in zip(got, got[1:]):
            assert f0 + c0 == f1
        assert max(c for _, c in got) - min(c for _, c in got) <= 1


def _fake_result(rank, nC=2, nW=1, nG=3, nD=4, nS=2):
    rng = np.random.default_rng(100 + rank)
    return dict(sum_alpha=rng.uniform(5, 6, nC), sig_re=rng.normal(size=(nW, nG, nD, nC)), sig_im=rng.normal(size=(nW, nG, nD, nC)),
                m2=rng.uniform(1, 2, (nS, nD, nC)), m4=rng.uniform(3, 9, (nS, nD, nC)), snap_alpha=rng.uniform(5, 6, (nS, nC)),
                class_flow=rng.integers(0, 1000, (nS, nC, nC)).astype(np.uint64), n_encounters=10 + rank, n_permeations=rank,
                n_clamps=0, n_saturations=3 * rank)


def _worker(rank, world, port, out_dir):
    import sys
    sys.path.insert(0, str(ROOT))
    import torch.distributed as dist
    import paper_2012_06478_b200 as rms
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        out = rms.api.allreduce_result(_fake_result(rank), np.array([1.0, 2.0]))
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), **{k: np.asarray(v) for k, v in out.items()})
    finally:
        dist.destroy_process_group()


def test_allreduce_of_two_shards_over_gloo_equals_the_merged_job(rms, tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    ref = rms.api.merge_results([_fake_result(0), _fake_result(1)], np.array([1.0, 2.0]))
    for rank in range(2):
        got = np.load(tmp_path / f"r{rank}.npz")
        for k in ("sum_alpha", "sig_re", "sig_im", "m2", "m4", "snap_alpha", "S", "Dapp", "Kapp"):
            assert np.allclose(got[k], ref[k], rtol=1e-13), k
        assert np.array_equal(got["class_flow"], ref["class_flow"])
        assert int(got["n_encounters"]) == 21 and int(got["n_permeations"]) == 1 and int(got["n_saturations"]) == 3


def test_fixed_codes_of_the_dictionary_lattice(tmp_path):
    """RMS_LATTICE_DICT gives interior and prismatic neighbourhoods (and their ghost variants) codes that need no search
    (csrc/rms_internal.cuh: rms_fixed_code / rms_fixed_word).  The host-only program tests/cuda/fixed_codes_host.cu checks that
    every fixed code and its 27-bit word map onto each other, that a word gets a code exactly when it does not change along a
    lattice axis (4e6 pseudo-random words, every z-invariant word), and the two interior codes."""
    import shutil
    import subprocess
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not on PATH")
    exe = tmp_path / "fixed_codes_host"
    subprocess.run(["nvcc", "-std=c++17", "-O1", "-Wno-deprecated-gpu-targets", "-o", str(exe), str(ROOT / "tests" / "cuda" / "fixed_codes_host.cu")], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0 and out.stdout.split()[:4] == ["bad", "0", "fixed", "1538"], out.stdout
