"""rms_substrate_label_volumes_static (include/rms.h): the per-label voxel count through the entry point that allocates
no device memory -- its counters are a static device array -- against the existing rms_substrate_label_volumes and against
numpy's bincount of the same lattice.  Integer work: bit exact.  The file is named to be collected last (the suite runs
with pytest -x); it passes alone in a fresh process and after the other tests (it shares nothing with them but the
library, and the static array is cleared at the start of every call)."""
import numpy as np
import pytest

import rms_inputs as ri

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rms():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2012_06478_b200 as rms
    rms.load_library()
    return rms


def _substrate(rms, sub):
    return rms.rms_substrate_create(sub.labels, sub.voxel_um, sub.D, sub.T2, sub.kappa, sub.label_class, sub.n_classes)


def test_static_label_volumes_match_the_allocating_path_on_calls_in_a_row(rms):
    # three lattices with different label counts, visited a, b, a, c: a later call must not see an earlier call's counts
    # (b has more labels than the kernel's shared-memory histogram holds, so its blocks add into the static array directly)
    a = ri.make_config("cfg2", "test").substrate
    b = ri.random_lattice((70, 33, 41), n_labels=9000, seed=4)
    c = ri.random_lattice((37, 29, 23), n_labels=5, seed=6)
    subs = {k: _substrate(rms, v) for k, v in (("a", a), ("b", b), ("c", c))}
    want = {k: np.bincount(v.labels.ravel(), minlength=v.n_labels).astype(np.uint64) for k, v in (("a", a), ("b", b), ("c", c))}
    try:
        for k in ("a", "a", "b", "a", "c", "b"):
            got = rms.rms_substrate_label_volumes_static(subs[k])
            ref = rms.rms_substrate_label_volumes(subs[k])
            assert got.dtype == np.uint64 and got.shape == ref.shape
            assert np.array_equal(got, ref), k
            assert np.array_equal(got, want[k]), k
            assert int(got.sum()) == subs[k].info()["n_voxels"]
    finally:
        for s in subs.values():
            s.destroy()


def test_static_label_volumes_on_a_side_stream(rms):
    import torch
    sub = ri.random_lattice((64, 48, 40), n_labels=300, seed=8)
    S = _substrate(rms, sub)
    try:
        st = torch.cuda.Stream()
        got = [rms.rms_substrate_label_volumes_static(S, stream=st) for _ in range(2)]
        want = np.bincount(sub.labels.ravel(), minlength=sub.n_labels).astype(np.uint64)
        assert np.array_equal(got[0], want) and np.array_equal(got[1], want)
    finally:
        S.destroy()


def _many_labels(rms, n_labels, seed):
    # no kappa table (NULL = impermeable): n_labels^2 floats would be a gigabyte here
    labels = np.random.default_rng(seed).integers(0, n_labels, size=(16, 20, 24)).astype(np.uint16)
    labels.ravel()[:2] = (0, n_labels - 1)          # both ends of the counter array are used
    return labels, rms.rms_substrate_create(labels, 0.1, np.full(n_labels, 2.0, np.float32), n_classes=1)


def test_static_label_volumes_reject_more_labels_than_the_static_array_holds(rms):
    from paper_2012_06478_b200 import binding
    n_max = binding.RMS_STATIC_MAX_LABELS
    labels, S = _many_labels(rms, n_max + 1, 3)
    try:
        with pytest.raises(rms.RmsError) as e:
            rms.rms_substrate_label_volumes_static(S)
        assert e.value.code == -7 and "RMS_STATIC_MAX_LABELS" in str(e.value)      # RMS_ERR_UNSUPPORTED, and says why
        # the allocating path serves that substrate
        assert np.array_equal(rms.rms_substrate_label_volumes(S), np.bincount(labels.ravel(), minlength=n_max + 1).astype(np.uint64))
    finally:
        S.destroy()
    labels, S = _many_labels(rms, n_max, 5)             # the largest size the static path takes
    try:
        got = rms.rms_substrate_label_volumes_static(S)
        assert np.array_equal(got, np.bincount(labels.ravel(), minlength=n_max).astype(np.uint64)) and got[-1] >= 1
    finally:
        S.destroy()
