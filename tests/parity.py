"""Parity rule between the CUDA path and the oracle (BASELINE.json north_star).

* charge maps: bit-exact, except pixels where the ORACLE's best and second-best fp64 energies differ by less than
  1e-9 * E_C (E_C = 1/2 min_i M_ii, "the charging energy") -- these near-tie pixels are counted and reported;
* sensor-dot columns (reading R8): bit-exact, except pixels where the margin of the sensor's two-way choice
  |e(c0+1) - e(c0)| (oracle, `sgap`) is below 1e-9 * E_C of the full model -- counted and reported;
* energies: |E_gpu - E_oracle| <= 1e-9 * max(|E_oracle|, E_C);
* continuous minima: |x_gpu - x_oracle| <= 1e-9 * max(1, |x_oracle|) (bit-exact where no QP ran).

`full_size_report` runs the five BASELINE.json configs at their full sizes through the C ABI binding and compares EVERY
pixel with the oracle (OpenMP over pixels); bench.py prints its result as the "parity" object of the JSON line and
tests/test_gpu_parity.py asserts on it.  This module is test infrastructure (it imports the oracle).
"""
import os
import time

import numpy as np

TOL = 1e-9


def compare(gpu_N, gpu_E, orc, EC, gpu_x=None, cols=None, strict=True):
    """gpu_N [P,n] int32, gpu_E [P]; orc = oracle dict (N, E, E2[, x, flags]); cols = columns of gpu_N compared with
    orc['N'].  Returns a report dict; with strict=True raises AssertionError on a non-excused mismatch or an energy /
    continuous-minimum error above tolerance (strict=False only counts them: bench.py's report)."""
    gN = np.asarray(gpu_N)
    gE = np.asarray(gpu_E)
    oN, oE, oE2 = orc["N"], orc["E"], orc["E2"]
    if cols is not None:
        gN = gN[:, cols]
    mism = (gN != oN).any(axis=1)
    near_tie = (oE2 - oE) < TOL * EC
    bad = mism & ~near_tie
    rep = {"pixels": int(len(oE)), "mismatch": int(mism.sum()), "excused_near_tie": int((mism & near_tie).sum()),
           "near_tie_pixels": int(near_tie.sum()), "unexcused": int(bad.sum())}
    if strict:
        assert rep["unexcused"] == 0, (rep, np.nonzero(bad)[0][:10], gN[bad][:5], oN[bad][:5])
    same = ~mism
    err = np.abs(gE[same] - oE[same])
    den = np.maximum(np.abs(oE[same]), EC)
    rep["max_rel_E_err"] = float((err / den).max()) if same.any() else 0.0
    rep["E_out_of_tolerance"] = int((err > TOL * den).sum())
    if strict:
        assert rep["E_out_of_tolerance"] == 0, rep
    if gpu_x is not None and "x" in orc:
        gx = np.asarray(gpu_x)
        ex = np.abs(gx - orc["x"]) / np.maximum(1.0, np.abs(orc["x"]))
        rep["max_rel_x_err"] = float(ex.max()) if ex.size else 0.0
        rep["x_out_of_tolerance"] = int((ex > TOL).sum())
        if strict:
            assert rep["x_out_of_tolerance"] == 0, rep
        if "flags" in orc:
            noqp = (orc["flags"] & 1) == 0
            rep["qp_pixels"] = int((~noqp).sum())
            rep["x_not_bit_identical_without_qp"] = int((gx[noqp] != orc["x"][noqp]).any(axis=1).sum())
            if strict:
                assert rep["x_not_bit_identical_without_qp"] == 0, "analytic minimum must be bit-identical (R1)"
            # residual class of SURVEY 8(c): QP pixels whose x sits within 1e-9 of an integer (floor may differ by a last bit)
            xq = orc["x"][~noqp]
            rep["qp_pixels_x_near_integer"] = int(((np.abs(xq - np.round(xq)) < TOL) & (xq != 0.0)).any(axis=1).sum())
    return rep


def compare_sensor(gpu_N, gpu_E, gpu_Vs, orc, sens, EC_sub, EC_full, strict=True):
    """Models with sensor dots (reading R8).  orc = oracle.sensor_ground_state(...) (N [P,n_full], E, E2, Vs, sgap).
    Array columns follow `compare`; a sensor column may differ only where that sensor's margin sgap < 1e-9 E_C(full)
    (counted).  V_s is compared on EVERY pixel whose full charge row agrees (i.e. every non-excused pixel)."""
    gN, gVs = np.asarray(gpu_N), np.asarray(gpu_Vs)
    n = gN.shape[1]
    sens = list(sens)
    D = [i for i in range(n) if i not in sens]
    rep = compare(gN, gpu_E, dict(orc, N=orc["N"][:, D]), EC_sub, cols=D, strict=strict)
    arr_same = (gN[:, D] == orc["N"][:, D]).all(axis=1)
    smis = gN[:, sens] != orc["N"][:, sens]                  # [P, ns]
    near = orc["sgap"] < TOL * EC_full
    # a sensor's choice depends on the array charges: only pixels whose array columns agree are judged here
    bad = (smis & ~near).any(axis=1) & arr_same
    rep["sensor_mismatch"] = int((smis.any(axis=1) & arr_same).sum())
    rep["sensor_excused_near_tie"] = int(((smis & near).any(axis=1) & ~(smis & ~near).any(axis=1) & arr_same).sum())
    rep["sensor_unexcused"] = int(bad.sum())
    rep["sensor_values_seen"] = int(len(np.unique(orc["N"][:, sens])))
    same = (gN == orc["N"]).all(axis=1)
    errv = np.abs(gVs[same] - orc["Vs"][same])
    den = np.maximum(np.abs(orc["Vs"][same]), EC_full)      # V_s is an energy per unit charge: floored at E_C (|e| = 1)
    rep["max_rel_Vs_err"] = float((errv / den).max()) if same.any() else 0.0
    rep["Vs_out_of_tolerance"] = int((errv > TOL * den).sum())
    rep["Vs_compared_pixels"] = int(same.sum())
    if strict:
        assert rep["sensor_unexcused"] == 0, (rep, np.nonzero(bad)[0][:10])
        assert rep["Vs_out_of_tolerance"] == 0, rep
        assert rep["Vs_compared_pixels"] >= len(same) - rep["mismatch"] - rep["sensor_mismatch"]
    return rep


# ---------------------------------------------------------------------------------------------------------------------
def _gpu(api, torch, w, variant=None, **kw):
    m = api.Model(w.C_dd, w.C_gd, sensor_dots=w.sensor_dots, walk_variant=variant)
    r = m.ground_state(torch.from_numpy(w.Vg).cuda(), regime=w.regime, N_hat=w.N_hat, want_xcont=True, want_stats=True, **kw)
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in r.items() if k != "stats"}
    out["stats"] = api.stats_dict(r["stats"])
    return out


def _merge(reps):
    """Sum the counters / take the max of the errors of several reports."""
    out = {}
    for r in reps:
        for k, v in r.items():
            if k.startswith("max_"):
                out[k] = max(out.get(k, 0.0), v)
            elif isinstance(v, (int, float)):
                out[k] = out.get(k, 0) + v
    return out


def full_size_report(api, oracle, wl, torch, strict=False, config5_members=256, configs=(1, 2, 3, 4, 5), n_threads=None):
    """Every pixel of the five BASELINE.json configs at full size, CUDA path (through the binding) vs oracle (OpenMP over
    pixels).  Returns {config: report}; report fields as `compare` plus the algorithms / variants covered, the R7
    exclusion count of config 1 and the wall time of the oracle."""
    nt = n_threads or os.cpu_count() or 1
    rep = {}
    if 1 in configs:
        t0 = time.perf_counter()
        w = wl.config1(100, 100)
        om = oracle.Model(w.C_dd, w.C_gd)
        od = om.ground_state(w.Vg, n_threads=nt)
        ob = om.ground_state(w.Vg, algorithm="brute", n_max=5, n_threads=nt)
        gd, gb = _gpu(api, torch, w), _gpu(api, torch, w, algorithm="brute", n_max=5)
        r = _merge([compare(gd["N"], gd["E"], od, om.EC, gd["xcont"], strict=strict),
                    compare(gb["N"], gb["E"], ob, om.EC, gb["xcont"], strict=strict)])
        # default vs brute force on the GPU maps (P2 / L472 "identical plots"), R7: pixels where default reaches n_max excluded
        excl = (gd["N"] >= 5).any(axis=1)
        r["default_vs_brute_R7_excluded"] = int(excl.sum())
        r["default_vs_brute_mismatch"] = int(((gd["N"] != gb["N"]).any(axis=1) & ~excl).sum())
        r.update(algorithms="default + brute force n_max=5", oracle_s=round(time.perf_counter() - t0, 2))
        rep["config1"] = r
    if 2 in configs:
        t0 = time.perf_counter()
        w = wl.config2(100, 100)
        om = oracle.Model(w.C_dd, w.C_gd)
        rs = []
        for kw in (dict(algorithm="default"), dict(algorithm="brute", n_max=5), dict(algorithm="thresholded", t=0.3)):
            o = om.ground_state(w.Vg, regime="closed", N_hat=5, n_threads=nt, **kw)
            g = _gpu(api, torch, w, **kw)
            rs.append(compare(g["N"], g["E"], o, om.EC, g["xcont"], strict=strict))
        r = _merge(rs)
        r.update(algorithms="default + brute force n_max=5 + thresholded t=0.3 (closed, N_hat=5)",
                 oracle_s=round(time.perf_counter() - t0, 2))
        rep["config2"] = r
    if 3 in configs:
        t0 = time.perf_counter()
        w = wl.config3(200, 200)
        o = oracle.sensor_ground_state(w.C_dd, w.C_gd, w.sensor_dots, w.Vg)
        D = [i for i in range(w.n_dot) if i not in w.sensor_dots]
        ec_sub = oracle.Model(w.C_dd[np.ix_(D, D)], w.C_gd[D, :]).EC
        ec_full = oracle.Model(w.C_dd, w.C_gd).EC
        g = _gpu(api, torch, w)
        r = compare_sensor(g["N"], g["E"], g["Vsensor"], o, w.sensor_dots, ec_sub, ec_full, strict=strict)
        r.update(algorithms="default, sensor column and V_s included", oracle_s=round(time.perf_counter() - t0, 2))
        rep["config3"] = r
    if 4 in configs:
        t0 = time.perf_counter()
        w = wl.config4(100, 100)
        om = oracle.Model(w.C_dd, w.C_gd)
        o = om.ground_state(w.Vg, n_threads=nt)
        rs = []
        for variant in (1, 2, 0, 3, 4):
            g = _gpu(api, torch, w, variant=variant)
            rs.append(compare(g["N"], g["E"], o, om.EC, g["xcont"], strict=strict))
            if variant == 1:
                g1 = g
            if variant == 3:
                g3 = g
        r_mixed_equal = bool(np.array_equal(g3["N"], g1["N"]) and np.array_equal(g3["E"], g1["E"]))
        r_fused_equal = bool(np.array_equal(g["N"], g1["N"]) and np.array_equal(g["E"], g1["E"]))
        r = dict(rs[0])
        for k in ("mismatch", "excused_near_tie", "unexcused", "E_out_of_tolerance"):
            r[k + "_all_variants"] = int(sum(x[k] for x in rs))
        r["mixed_precision_walk_bit_identical_to_fp64_walk"] = r_mixed_equal
        r["one_kernel_path_bit_identical_to_fp64_walk"] = r_fused_equal
        r.update(algorithms="default; walk variants 1 (min-plus), 2 (pruned), 0 (exact-compare walk), 3 (fp32 lower-bound pass + "
                            "fp64 re-score), 4 (S1-S7 in one persistent kernel), each vs the oracle",
                 oracle_s=round(time.perf_counter() - t0, 2))
        rep["config4"] = r
    if 5 in configs:
        t0 = time.perf_counter()
        B = config5_members
        wls = [wl.config5_array(j) for j in range(B)]
        algs = (("default", dict(algorithm="default")), ("t0.2", dict(algorithm="thresholded", t=0.2)),
                ("t0.5", dict(algorithm="thresholded", t=0.5)))
        rs = []
        CH = 64
        for c0 in range(0, B, CH):
            chunk = wls[c0:c0 + CH]
            batch = api.Batch([api.Model(w.C_dd, w.C_gd) for w in chunk])
            Vg = torch.from_numpy(np.stack([w.Vg for w in chunk])).cuda()
            res = {}
            for name, kw in algs:
                rr = batch.ground_state(Vg, want_xcont=True, **kw)
                torch.cuda.synchronize()
                res[name] = (rr["N"].cpu().numpy(), rr["E"].cpu().numpy(), rr["xcont"].cpu().numpy())
            for j, w in enumerate(chunk):
                om = oracle.Model(w.C_dd, w.C_gd)
                for name, kw in algs:
                    o = om.ground_state(w.Vg, n_threads=nt, **kw)
                    N, E, x = res[name]
                    rs.append(compare(N[j], E[j], o, om.EC, x[j], strict=strict))
        r = _merge(rs)
        r.update(algorithms="default + thresholded t=0.2 + t=0.5 through qa_ground_state_batch", members=B,
                 oracle_s=round(time.perf_counter() - t0, 2))
        rep["config5"] = r
    return rep
