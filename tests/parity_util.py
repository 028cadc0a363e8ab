"""Shared helpers of the GPU parity tests: run the CUDA path and the oracle on the same seeded inputs and
compare element by element with the tolerances BASELINE.json:north_star states."""
import numpy as np

TOL_SAME_VOXEL = 0.999     # >= 99.9 % of walkers in the same final voxel
TOL_S = 1e-4               # |dS| absolute per b-value and direction (real and imaginary part)
TOL_MOMENT = 1e-4          # cumulants / moments, relative


def gpu_run(cfg_sub, cfg_seq, n_walkers, seed, first_id=0, flags=0, read_walkers=True):
    import paper_2012_06478_b200 as rms
    return rms.simulate(cfg_sub, cfg_seq, n_walkers, seed, first_id=first_id, flags=flags, read_walkers=read_walkers)


def oracle_run(cfg_sub, cfg_seq, n_walkers, seed, first_id=0, interaction=0):
    import oracle
    return oracle.run(cfg_sub, cfg_seq, n_walkers, seed, first_id=first_id, n_threads=oracle.rms_oracle.default_threads(),
                      per_walker=True, interaction=interaction)


def compare(g, o, n_walkers, tol_s=TOL_S, tol_m=TOL_MOMENT, same_voxel=TOL_SAME_VOXEL, check_init=True, strict_s=False):
    """g: dict from the CUDA path (with "walkers"); o: dict from the oracle (per_walker=True).

    A trajectory is discontinuous where a hop passes the edge of a convex membrane corner (one way round it
    misses the corner, the other way it is reflected), so an fp32 and an fp64 walker that differ by 1e-6 voxel
    part company there for good; north_star allows 0.1 % of the walkers to do so.  Each such walker can move
    S by at most 2/N, which at the small N of most cases here is above 1e-4 by itself: those cases bound
    |dS| by 1e-4 + 2 n_diff / N (the agreeing walkers must agree to 1e-4) and widen the moment tolerances in
    the same way (under rejection sampling every membrane met is such a discontinuity: a grazing step is cancelled
    whole or not at all); strict_s=True, used at full size where N is large, applies the plain tolerances
    (DESIGN.md "Tolerances")."""
    rep = {}
    w = g["walkers"]
    if check_init:   # placement is integer work: bit exact
        assert np.array_equal(w["vox0"], o["init_vox"])
        assert np.array_equal(w["off0"].astype(np.float64), o["init_off"])
    same = np.all(w["vox"] == o["final_vox"], axis=1)
    # a walker that parted company may by chance end in the voxel of its twin (likely on the few-voxel periodic lattices
    # of the small cases): offsets 0.01 voxel apart are no rounding difference, so it counts as diverged all the same
    same &= np.abs(w["off"].astype(np.float64) - o["final_off"]).max(axis=1) < 0.01
    rep["same_voxel"] = float(same.mean())
    rep["n_diff"] = int((~same).sum())
    assert rep["same_voxel"] >= same_voxel, rep
    slack = 0.0 if strict_s else rep["n_diff"] / n_walkers
    tol_s = tol_s + 2.0 * slack
    # positions agree to rounding for the walkers in the same voxel
    d_off = np.abs(w["off"][same].astype(np.float64) - o["final_off"][same])
    rep["max_offset_diff"] = float(d_off.max()) if d_off.size else 0.0
    rep["label_mismatch"] = int(np.count_nonzero(w["label"] != o["final_label"]))
    assert rep["label_mismatch"] <= (1 - same_voxel) * n_walkers + 1
    if o["S"].size:
        dS = g["S"] - o["S"]
        rep["max_dS"] = float(max(np.abs(dS.real).max(), np.abs(dS.imag).max()))
        assert rep["max_dS"] <= tol_s, rep
        # raw per-class sums too
        scale = max(1.0, float(o["sum_alpha"].sum()))
        assert np.abs(g["sig_re"] - o["sig_re"]).max() / scale <= tol_s
        assert np.abs(g["sig_im"] - o["sig_im"]).max() / scale <= tol_s
    assert np.allclose(g["sum_alpha"], o["sum_alpha"], rtol=1e-6, atol=1e-9)
    if o["m2"].size:
        for k in ("m2", "m4", "snap_alpha"):
            ref = o[k]
            err = np.abs(g[k] - ref) / np.maximum(np.abs(ref), 1e-300)
            err = np.where(ref == 0, np.abs(g[k]), err)
            rep["rel_" + k] = float(err.max())
            # a walker that parted company moves sum X^2 (X^4) by a few mean squares (fourth powers) of one walker
            assert rep["rel_" + k] <= tol_m + {"m2": 8.0, "m4": 32.0, "snap_alpha": 0.0}[k] * slack, (k, rep)
        assert np.allclose(g["Dapp"], o["D"], rtol=tol_m + 8.0 * slack, atol=0)
        assert np.allclose(g["Kapp"], o["K"], rtol=0, atol=2e-4 + tol_m * np.abs(o["K"]).max() + 64.0 * slack)
        flow_diff = np.abs(g["class_flow"].astype(np.int64) - o["class_flow"].astype(np.int64)).sum()
        rep["class_flow_diff"] = int(flow_diff)
        assert flow_diff <= 2 * (1 - same_voxel) * n_walkers * max(1, o["class_flow"].shape[0])
    enc = max(1, o["n_encounters"])
    rep["rel_encounters"] = abs(g["n_encounters"] - o["n_encounters"]) / enc
    assert rep["rel_encounters"] <= 1e-3, rep
    rep["perm_diff"] = abs(g["n_permeations"] - o["n_permeations"])
    assert rep["perm_diff"] <= max(3, 1e-3 * o["n_permeations"]), rep
    return rep
