"""Parity rule between the CUDA path and the oracle (BASELINE.json north_star).

* charge maps: bit-exact, except pixels where the ORACLE's best and second-best fp64 energies differ by less than
  1e-9 * E_C (E_C = 1/2 min_i M_ii, "the charging energy") -- these near-tie pixels are counted and reported;
* energies: |E_gpu - E_oracle| <= 1e-9 * max(|E_oracle|, E_C);
* continuous minima: |x_gpu - x_oracle| <= 1e-9 * max(1, |x_oracle|) (bit-exact where no QP ran).
"""
import numpy as np

TOL = 1e-9


def compare(gpu_N, gpu_E, orc, EC, gpu_x=None, cols=None):
    """gpu_N [P,n] int32, gpu_E [P]; orc = oracle dict (N, E, E2[, x]); cols = columns of N compared with orc['N'].
    Returns a report dict; raises AssertionError on a non-excused mismatch."""
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
    assert rep["unexcused"] == 0, (rep, np.nonzero(bad)[0][:10], gN[bad][:5], oN[bad][:5])
    same = ~mism
    err = np.abs(gE[same] - oE[same])
    lim = TOL * np.maximum(np.abs(oE[same]), EC)
    rep["max_rel_E_err"] = float((err / np.maximum(np.abs(oE[same]), EC)).max()) if same.any() else 0.0
    assert (err <= lim).all(), rep
    if gpu_x is not None and "x" in orc:
        gx = np.asarray(gpu_x)
        ex = np.abs(gx - orc["x"]) / np.maximum(1.0, np.abs(orc["x"]))
        rep["max_rel_x_err"] = float(ex.max())
        assert ex.max() <= TOL, rep
        if "flags" in orc:
            noqp = (orc["flags"] & 1) == 0
            assert np.array_equal(gx[noqp], orc["x"][noqp]), "analytic minimum must be bit-identical (R1)"
    return rep
