"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI binding, against the oracle, element by element on
the same seeded inputs; plus edge cases and full-size sampled checks in the launch configuration bench.py times."""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2404_04994_b200 import workloads as wl
from parity import compare, compare_sensor, full_size_report

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2404_04994_b200 import api as _api
    assert torch.cuda.is_available()
    return _api


def run_gpu(api, w, variant=None, **kw):
    m = api.Model(w.C_dd, w.C_gd, sensor_dots=w.sensor_dots, walk_variant=variant)
    Vg = torch.from_numpy(w.Vg).cuda()
    r = m.ground_state(Vg, regime=w.regime, N_hat=w.N_hat, want_xcont=True, want_stats=True, **kw)
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in r.items() if k != "stats"}
    out["stats"] = api.stats_dict(r["stats"])
    out["plan"] = api.last_launch_plan()
    M, EC = m.inverse()
    out["EC"] = EC
    return out


def run_oracle(w, **kw):
    m = oracle.Model(w.C_dd, w.C_gd)
    kw = dict(kw)
    if "algorithm" in kw and kw["algorithm"] == "brute_force":
        kw["algorithm"] = "brute"
    return m, m.ground_state(w.Vg, regime=w.regime, N_hat=w.N_hat, **kw)


def check(api, w, variant=None, **kw):
    g = run_gpu(api, w, variant=variant, **kw)
    m, o = run_oracle(w, **kw)
    rep = compare(g["N"], g["E"], o, m.EC, gpu_x=g["xcont"])
    st = g["stats"]
    assert st["n_pixels"] == w.P and st["n_qp_failed"] == 0
    assert st["n_qp_pixels"] == int(((o["flags"] & oracle.FLAG_QP) != 0).sum())
    assert st["n_candidates_enumerated"] == int(o["n_enum"].sum())
    assert st["n_candidates_scored"] == int(o["n_scored"].sum())
    assert st["n_threshold_doublings"] == int(o["doublings"].sum())
    assert st["n_widened_pixels"] == 0 and int(((o["flags"] & oracle.FLAG_WIDENED) != 0).sum()) == 0
    assert abs(g["EC"] - m.EC) <= 1e-12 * m.EC
    return rep, g, o


# ---- the five BASELINE.json configs at sizes the oracle finishes in seconds (several tiles + ragged tails) ----------
def test_config1_open_double_dot_default_and_brute(api):
    w = wl.config1(100, 100)
    rep, g, o = check(api, w, algorithm="default")
    assert g["plan"][0] == ["qa_fused_open_kernel"]
    assert st_zero_qp(g)
    rep, g, o = check(api, w, algorithm="brute", n_max=5)
    assert g["plan"][0] == ["qa_fused_small_kernel"]


def st_zero_qp(g):
    return g["stats"]["n_qp_pixels"] == 0


def test_config2_closed_chain_default_and_brute(api):
    w = wl.config2(100, 100)
    rep, g, o = check(api, w, algorithm="default")
    assert g["stats"]["n_qp_pixels"] > 0
    assert (g["N"].sum(1) == 5).all()
    check(api, w, algorithm="brute", n_max=5)          # full 100x100: 7776 enumerated, 126 valid per pixel
    check(api, w, algorithm="thresholded", t=0.3)
    check(api, w, algorithm="thresholded", t=0.0)
    w2 = wl.config2(37, 23)                            # ragged sizes
    check(api, w2, algorithm="brute", n_max=5)
    check(api, w2, algorithm="thresholded", t=0.3)


def sensor_check(api, w, variant=None):
    g = run_gpu(api, w, variant=variant, algorithm="default")
    o = oracle.sensor_ground_state(w.C_dd, w.C_gd, w.sensor_dots, w.Vg)
    D = [i for i in range(w.n_dot) if i not in w.sensor_dots]
    sub = oracle.Model(w.C_dd[np.ix_(D, D)], w.C_gd[D, :])
    full = oracle.Model(w.C_dd, w.C_gd)
    rep = compare_sensor(g["N"], g["E"], g["Vsensor"], o, w.sensor_dots, sub.EC, full.EC)
    assert g["xcont"].shape == (w.P, len(D))
    assert np.array_equal(g["xcont"][(o["flags"] & 1) == 0], sub.ground_state(w.Vg)["x"][(o["flags"] & 1) == 0])
    return rep


def test_config3_sensor_full_size(api):
    """Config 3 at its full 200x200: array columns by the near-tie rule, the sensor column bit-exact except where the
    sensor's own two-way margin is below 1e-9 E_C (counted), V_s on every pixel whose charge row agrees."""
    w = wl.config3(200, 200)
    rep = sensor_check(api, w)
    assert rep["Vs_compared_pixels"] >= w.P - rep["excused_near_tie"] - rep["sensor_excused_near_tie"]
    # config 3 keeps the sensor gate fixed (its carrier number never changes on the sweep); ramp it so the sensor's
    # two-way choice flips many times, on both kernel paths
    w2 = wl.config3(64, 45)
    w2.Vg[:, 4] = np.linspace(0.0, 3.5, w2.P) / w2.C_gd[4, 4]
    for variant in (1, 0):
        rep = sensor_check(api, w2, variant=variant)
        assert rep["sensor_values_seen"] >= 3


@pytest.mark.parametrize("n,sens,P", [(6, (2, 5), 1203), (5, (0,), 700), (11, (3, 7, 10), 150), (16, (0, 9), 60)])
def test_multi_sensor_models(api, n, sens, P):
    """ns > 1 and sensors at non-trailing indices, through the one-kernel path (n_search <= 8), the three-kernel path and
    the min-plus path (n_search = 14) with the finalize kernel's sensor step."""
    w = wl.random_open(n, n + 1, P, seed=700 + n, lo=-0.3, hi=2.7)
    w.sensor_dots = tuple(sens)
    for variant in (1, 0):
        rep = sensor_check(api, w, variant=variant)
        assert rep["sensor_values_seen"] >= 2


@pytest.mark.parametrize("W,H", [(9, 7), (33, 3)])
def test_config4_open_grid16_default(api, W, H):
    """n = 16, 2^16 candidates per pixel: the hot kernel (NL = 8, NH = 8), QP pixels included."""
    w = wl.config4(W, H)
    rep, g, o = check(api, w, algorithm="default")
    assert g["plan"][0] == ["qa_prologue_lanes_kernel", "qa_minplus_walk_kernel", "qa_minplus_finish_kernel"]
    assert g["stats"]["n_candidates_scored"] == w.P * 65536


@pytest.mark.parametrize("n,P", [(13, 45), (14, 46), (15, 33), (16, 45), (16, 1)])
def test_walk_variants_agree(api, n, P):
    """The exact-compare walk (variant 0), the min-plus walk + finish kernel (variant 1, the default for n >= 13)
    and the min-plus walk with exact pruning of the high patterns (variant 2) give the same charge map and the same
    energies up to the summation order of E(N*); each is also checked against the oracle.  P odd / P = 1: the ragged
    last pixel pair of the min-plus walks."""
    w = wl.random_open(n, n, P, seed=200 + n)
    ref = None
    plans = {0: ["qa_prologue_kernel", "qa_walk_kernel", "qa_finalize_kernel"],
             1: ["qa_prologue_lanes_kernel", "qa_minplus_walk_kernel", "qa_minplus_finish_kernel"],
             2: ["qa_prologue_lanes_kernel", "qa_minplus_pruned_kernel", "qa_minplus_finish_kernel"],
             3: ["qa_prologue_lanes_kernel", "qa_minplus_walk32_kernel", "qa_minplus_finish_kernel"],
             # variant 4: S1-S7 in one persistent kernel (16 dots only; other sizes run as variant 1)
             4: ["qa_minplus_fused_kernel"] if n == 16 else
                ["qa_prologue_lanes_kernel", "qa_minplus_walk_kernel", "qa_minplus_finish_kernel"]}
    for variant in (0, 1, 2, 3, 4):
        rep, g, o = check(api, w, variant=variant, algorithm="default")
        assert g["plan"][0] == plans[variant]
        if ref is None:
            ref = g
        else:
            assert np.array_equal(ref["N"], g["N"])
            assert np.allclose(ref["E"], g["E"], rtol=1e-13, atol=1e-13 * g["EC"])


@pytest.mark.parametrize("n,P", [(13, 20001), (16, 2501)])
def test_minplus_walk_many_groups_per_worker(api, n, P):
    """The persistent min-plus walk's multi-iteration path (grp += workers with the one-ahead prefetch) and several
    hand-outs per warp of the pruned walk's work counter: n = 13 has 8 pixel slots per CTA and 296 CTAs, so P = 20001 gives
    every worker 4-5 pixel pairs (n = 16: one slot per CTA, 1251 pairs over 296 workers); element by element against the
    oracle (OpenMP over pixels), all three variants, odd P (ragged last pair)."""
    w = wl.random_open(n, n, P, seed=310 + n, lo=-0.7, hi=3.3)
    om = oracle.Model(w.C_dd, w.C_gd)
    o = om.ground_state(w.Vg, n_threads=os.cpu_count() or 1)
    ref = None
    for variant in (0, 1, 2, 3, 4):
        g = run_gpu(api, w, variant=variant)
        compare(g["N"], g["E"], o, om.EC, gpu_x=g["xcont"])
        assert g["stats"]["n_qp_pixels"] == int(((o["flags"] & oracle.FLAG_QP) != 0).sum()) and g["stats"]["n_qp_failed"] == 0
        if ref is None:
            ref = g
        else:
            diff = (ref["N"] != g["N"]).any(1)
            assert np.abs(ref["E"] - g["E"])[diff].max(initial=0.0) <= 1e-9 * om.EC


@pytest.mark.parametrize("n", [13, 16])
def test_minplus_walks_against_exact_walk_many_models(api, n):
    """Many seeded models and pixels, GPU against GPU: the min-plus walks (lower-bound filter, and with pruning) must
    return the charge state of the exact-compare walk; a differing pixel is accepted only as a near tie (energies equal
    to 1e-9 E_C), and there must be next to none."""
    bad = 0
    for seed in range(10):
        w = wl.random_open(n, n, 301, seed=900 + 17 * seed + n, lo=-0.7, hi=3.4)
        m = api.Model(w.C_dd, w.C_gd)
        _, EC = m.inverse()
        Vg = torch.from_numpy(w.Vg).cuda()
        outs = {}
        for variant in (0, 1, 2, 3, 4):
            m.set_walk_variant(variant)
            r = m.ground_state(Vg)
            torch.cuda.synchronize()
            outs[variant] = (r["N"].cpu().numpy(), r["E"].cpu().numpy())
        # the mixed-precision walk (fp32 lower bound, fp64 exact re-score) must reproduce the fp64 walk bit for bit, and so
        # must the one-kernel path (same arithmetic, inputs through shared memory instead of the workspace)
        for variant in (3, 4):
            assert np.array_equal(outs[variant][0], outs[1][0]) and np.array_equal(outs[variant][1], outs[1][1])
        for variant in (1, 2):
            diff = (outs[variant][0] != outs[0][0]).any(1)
            assert np.abs(outs[variant][1] - outs[0][1])[diff].max(initial=0.0) <= 1e-9 * EC
            assert np.allclose(outs[variant][1], outs[0][1], rtol=1e-12, atol=1e-12 * EC)
            bad += int(diff.sum())
    assert bad <= 2


def test_minplus_walk_extreme_inputs(api):
    """Pixels far outside the operating range: every dot clamped (N_c << 0, huge positive h) and large occupations."""
    w = wl.config4(6, 5)
    rng = np.random.default_rng(7)
    # (the last two blocks stress the per-pixel fixed-point scale of the walk's keys: energies of 1e12 and of 1e-18 E_C)
    Vg = np.concatenate([w.Vg, -50.0 * np.abs(rng.standard_normal((7, 16))), w.Vg[:9] * 40.0, np.zeros((3, 16)),
                         w.Vg[:6] * 1.0e6, w.Vg[:6] * 1.0e-9])
    w.Vg, w.W, w.H = np.ascontiguousarray(Vg), Vg.shape[0], 1
    for variant in (0, 1, 2, 3, 4):
        check(api, w, variant=variant, algorithm="default")


def test_config5_open_grid8_default_and_thresholded(api):
    for j in (0, 7):
        w = wl.config5_array(j, 48, 41)
        check(api, w, algorithm="default")
        for t in (0.2, 0.5, 0.7, 1.0):   # (t <= 0.6: every thread walks its own pixel; above: bucket sort by free dots)
            check(api, w, algorithm="thresholded", t=t)


# ---- every n_dot through the static walk and the generic enumeration ----------------------------------------------
@pytest.mark.parametrize("n", list(range(1, 17)))
def test_all_sizes_default_open(api, n):
    w = wl.random_open(n, n + (n % 3), 301 if n <= 10 else (67 if n <= 13 else 37), seed=50 + n)
    rep, g, o = check(api, w, algorithm="default")
    if n <= 12:   # the one-kernel paths above; the three-kernel path (static walk) below
        assert g["plan"][0] == (["qa_fused_open_kernel"] if n <= 8 else ["qa_fused_mid_kernel"])
        rep, g0, o = check(api, w, variant=0, algorithm="default")
        assert g0["plan"][0] == ["qa_prologue_kernel", "qa_walk_kernel", "qa_finalize_kernel"]
        assert np.array_equal(g["N"], g0["N"])


@pytest.mark.parametrize("n,g,P", [(9, 9, 1003), (10, 13, 517), (11, 11, 259), (12, 12, 130), (12, 64, 33), (9, 2, 17)])
def test_fused_mid_kernel(api, n, g, P):
    """Open default search of 9..12 dots in one kernel (a warp per two pixels): sizes that are not multiples of the 16 pixels
    of a CTA (a ragged last CTA, an odd last pixel of a warp), more gates than dots up to the 64-gate limit and fewer, QP
    pixels with one to three and with more clamped dots (the serial solver), a general SPD c_dd, extreme gate voltages;
    element by element against the oracle, counters included, and bit-identical N to the three-kernel path."""
    w = wl.random_open(n, g, P, seed=820 + n + g, lo=-0.9, hi=3.1)
    rep, gg, o = check(api, w, algorithm="default")
    assert gg["plan"][0] == ["qa_fused_mid_kernel"] and gg["stats"]["n_qp_pixels"] > 0
    assert gg["stats"]["n_candidates_scored"] == P * 2 ** n
    rep0, g0, _ = check(api, w, variant=0, algorithm="default")
    assert np.array_equal(gg["N"], g0["N"])
    if g == n:
        wg = wl.random_general(n, n, 77, seed=860 + n)
        rep, gg, o = check(api, wg, algorithm="default")
        assert gg["plan"][0] == ["qa_fused_mid_kernel"] and gg["stats"]["n_qp_pixels"] > 0
        rng = np.random.default_rng(n)
        w.Vg = np.ascontiguousarray(np.concatenate([w.Vg[:20], -40.0 * np.abs(rng.standard_normal((9, g))), w.Vg[:5] * 30.0,
                                                    np.zeros((2, g))]))
        w.W, w.H = w.Vg.shape[0], 1
        check(api, w, algorithm="default")


@pytest.mark.parametrize("n", [1, 2, 3, 6, 9, 11])
@pytest.mark.parametrize("variant", [1, 0])
def test_all_sizes_closed_and_thresholded(api, n, variant):
    w = wl.random_open(n, n, 203, seed=80 + n, lo=-0.4, hi=2.5)
    w.regime, w.N_hat = "closed", max(1, n)
    check(api, w, variant=variant, algorithm="default")
    check(api, w, variant=variant, algorithm="thresholded", t=0.25)
    w.regime = "open"
    check(api, w, variant=variant, algorithm="thresholded", t=0.4)
    if n <= 6:
        check(api, w, variant=variant, algorithm="brute", n_max=3)
        w.regime = "closed"
        check(api, w, variant=variant, algorithm="brute", n_max=3)


# ---- closed arrays at scale: only the C(n, k) states with the right total are visited ------------
@pytest.mark.parametrize("n", list(range(9, 17)))
def test_closed_default_large_arrays(api, n):
    """Closed default search for n = 9..16 through qa_closed_walk_kernel (popcount classes of the min-plus split), N_hat = n
     and a second total, QP pixels included, element by element against the oracle; the scored-candidate
    counter must equal the oracle's sum of C(n, N_hat - sum lo).  Variant 0 (the generic odometer over all 2^n states,
    filtered) must give the same maps.  Also a general SPD c_dd (no Maxwell structure is used by the kernel)."""
    P = 301 if n <= 12 else (131 if n <= 14 else 67)
    for N_hat in (n, max(1, n // 3)):
        w = wl.random_open(n, n, P, seed=700 + n, lo=-0.5, hi=2.4)
        w.regime, w.N_hat = "closed", N_hat
        rep, g, o = check(api, w, algorithm="default")
        pro = "qa_prologue_lanes_kernel" if 12 <= n <= 15 else "qa_prologue_kernel"
        assert g["plan"][0] == [pro, "qa_closed_walk_kernel", "qa_finalize_lanes_kernel"]
        assert g["stats"]["n_qp_pixels"] > 0
        rep0, g0, _ = check(api, w, variant=0, algorithm="default")
        assert g0["plan"][0][1].startswith("qa_enumerate_kernel")
        assert np.array_equal(g["N"], g0["N"])
    w = wl.random_general(n, n, 61, seed=740 + n)
    w.regime, w.N_hat = "closed", n
    rep, g, o = check(api, w, algorithm="default")
    assert g["plan"][0][1] == "qa_closed_walk_kernel"


def test_closed16_full_size_every_pixel(api):
    """bench.py's closed16 workload in its launch configuration: the config-4 model and sweep as a CLOSED array with N_hat = 16
    (PAPER.md L496), all 10^4 pixels against the oracle (OpenMP), counters included."""
    w = wl.config4(100, 100)
    w.regime, w.N_hat = "closed", 16
    g = run_gpu(api, w)
    om = oracle.Model(w.C_dd, w.C_gd)
    o = om.ground_state(w.Vg, regime="closed", N_hat=16, n_threads=os.cpu_count() or 1)
    rep = compare(g["N"], g["E"], o, om.EC, gpu_x=g["xcont"])
    assert rep["unexcused"] == 0 and rep["qp_pixels"] > 5000
    assert g["plan"][0] == ["qa_prologue_kernel", "qa_closed_walk_kernel", "qa_finalize_lanes_kernel"]
    assert g["stats"]["n_candidates_scored"] == int(o["n_scored"].sum()) and g["stats"]["n_qp_failed"] == 0
    assert (g["N"].sum(1) == 16).all()


def test_closed_default_edge_totals(api):
    """N_hat = 0 (only the all-zero state), N_hat far above what the gates ask for, and P not a multiple of the pixels per
    CTA, on a 10-dot and a 16-dot array."""
    for n, P in ((10, 97), (16, 13)):
        for N_hat in (0, 1, 3 * n):
            w = wl.random_open(n, n, P, seed=760 + n, lo=-0.5, hi=2.4)
            w.regime, w.N_hat = "closed", N_hat
            check(api, w, algorithm="default")


# ---- c_dd with positive off-diagonals (SPD, not Maxwell): general active-set phase of the QP (reading R3) -------------
@pytest.mark.parametrize("n", [2, 3, 5, 8, 11, 13, 16])
def test_general_spd_matrices(api, n):
    w = wl.random_general(n, n, 257 if n <= 11 else 41, seed=400 + n)
    assert (w.C_dd - np.diag(np.diag(w.C_dd)) > 0).any()
    rep, g, o = check(api, w, algorithm="default")
    assert g["stats"]["n_qp_pixels"] > 0
    if n >= 13:
        assert g["plan"][0][1] == "qa_walk_kernel"      # the min-plus walk needs M >= 0 (Maxwell); exact walk here
    if n <= 11:
        check(api, w, algorithm="thresholded", t=0.3)
        w.regime, w.N_hat = "closed", n
        check(api, w, algorithm="default")
        check(api, w, algorithm="thresholded", t=0.3)
        if n <= 5:
            check(api, w, algorithm="brute", n_max=3)


# ---- thermal broadening, Eq. (10): mean occupation vs the oracle ----------------------------
def check_thermal(api, w, kT_over_EC, **kw):
    m = api.Model(w.C_dd, w.C_gd)
    om = oracle.Model(w.C_dd, w.C_gd)
    kT = kT_over_EC * om.EC
    r = m.thermal(torch.from_numpy(w.Vg).cuda(), kT, regime=w.regime, N_hat=w.N_hat, want_stats=True, **kw)
    torch.cuda.synchronize()
    okw = dict(kw)
    if okw.get("algorithm") == "brute_force":
        okw["algorithm"] = "brute"
    o = om.thermal(w.Vg, kT, regime=w.regime, N_hat=w.N_hat, **okw)
    Nm, Em = r["Nmean"].cpu().numpy(), r["Emin"].cpu().numpy()
    # tolerance: the incremental energies drift by <~ 1e-13 E_C over a walk, i.e. 1e-13 E_C / kT in a weight
    tol = 1e-9 * max(1.0, 0.02 / kT_over_EC)
    assert np.abs(Nm - o["Nmean"]).max() <= tol * max(1.0, np.abs(o["Nmean"]).max())
    fin = np.isfinite(o["Emin"])
    assert np.abs(Em[fin] - o["Emin"][fin]).max() <= 1e-9 * max(om.EC, np.abs(o["Emin"][fin]).max())
    assert api.stats_dict(r["stats"])["n_candidates_scored"] == int(o["n_scored"].sum())
    return Nm, o


def test_thermal_small_configs(api):
    w = wl.config1(60, 50)
    Nm, o = check_thermal(api, w, 0.05, algorithm="default")
    assert api.last_launch_plan()[0] == ["qa_prologue_kernel", "qa_thermal_gray_kernel<G=1>"]
    assert ((Nm > 0.01) & (Nm < 0.99)).any()          # transitions are actually broadened
    check_thermal(api, w, 0.3, algorithm="brute", n_max=5)
    w2 = wl.config2(40, 30)
    Nm, o = check_thermal(api, w2, 0.05, algorithm="default")
    assert np.allclose(Nm.sum(1), 5.0, atol=1e-9)     # closed array: the total charge survives the average
    check_thermal(api, w2, 0.2, algorithm="thresholded", t=0.3)
    check_thermal(api, w2, 0.1, algorithm="brute", n_max=5)
    assert api.last_launch_plan()[0][1] == "qa_thermal_kernel<G=256>"


@pytest.mark.parametrize("n,P", [(1, 300), (4, 300), (8, 257), (11, 65), (13, 9), (16, 5)])
def test_thermal_all_sizes(api, n, P):
    w = wl.random_open(n, n, P, seed=600 + n, lo=-0.4, hi=2.6)
    check_thermal(api, w, 0.08, algorithm="default")
    check_thermal(api, w, 0.5, algorithm="thresholded", t=0.4)
    if n <= 11:
        w.regime, w.N_hat = "closed", max(1, n)
        check_thermal(api, w, 0.08, algorithm="default")


@pytest.mark.parametrize("n,P", [(9, 515), (10, 300), (12, 131), (13, 77), (14, 40), (15, 21), (16, 33)])
def test_thermal_sum_product_kernel(api, n, P):
    """Open default set of 9..16 dots: the sum-product kernel (qa_thermal_sp_kernel, factorised Boltzmann weights over the
    min-plus split) against the oracle at a warm and a cool temperature, and against the two-pass Gray kernel (variant 0 of
    the model) on the same pixels; at a temperature so low that the factorised weights could underflow the launcher must
    fall back to the Gray kernel by itself."""
    w = wl.random_open(n, n, P, seed=650 + n, lo=-0.4, hi=2.6)
    M = np.linalg.inv(w.C_dd)
    gsum = np.abs(np.triu(M, 1)).sum()
    EC = 0.5 * np.diag(M).min()
    for kT_over_EC in (0.3, max(0.05, 1.05 * gsum / 600.0 / EC)):
        Nm, o = check_thermal(api, w, kT_over_EC, algorithm="default")
        assert api.last_launch_plan()[0] == ["qa_prologue_lanes_kernel", "qa_thermal_sp_kernel"]
        m0 = api.Model(w.C_dd, w.C_gd, walk_variant=0)
        r0 = m0.thermal(torch.from_numpy(w.Vg).cuda(), kT_over_EC * EC)
        assert api.last_launch_plan()[0][1].startswith("qa_thermal_gray_kernel")
        assert np.abs(r0["Nmean"].cpu().numpy() - Nm).max() <= 1e-9 * max(1.0, 0.02 / kT_over_EC) * max(1.0, np.abs(Nm).max())
    check_thermal(api, w, 0.9 * gsum / 600.0 / EC, algorithm="default")
    assert api.last_launch_plan()[0][1].startswith("qa_thermal_gray_kernel")


def test_thermal_sum_product_full_size_sample(api):
    """bench.py's thermal workload (config 4, 100x100, kT = 0.05 E_C) in its launch configuration: 300 seeded pixels of the
    full diagram against the oracle."""
    w = wl.config4(100, 100)
    m = api.Model(w.C_dd, w.C_gd)
    om = oracle.Model(w.C_dd, w.C_gd)
    kT = 0.05 * om.EC
    r = m.thermal(torch.from_numpy(w.Vg).cuda(), kT)
    assert api.last_launch_plan()[0] == ["qa_prologue_lanes_kernel", "qa_thermal_sp_kernel"]
    sel = np.sort(np.random.default_rng(1).choice(w.P, size=300, replace=False))
    o = om.thermal(w.Vg[sel], kT)
    assert np.abs(r["Nmean"].cpu().numpy()[sel] - o["Nmean"]).max() <= 1e-9 * max(1.0, np.abs(o["Nmean"]).max())
    assert np.abs(r["Emin"].cpu().numpy()[sel] - o["Emin"]).max() <= 1e-9 * max(om.EC, np.abs(o["Emin"]).max())


def test_thermal_cold_limit_is_the_ground_state_and_errors(api):
    w = wl.config5_array(1, 40, 40)
    m = api.Model(w.C_dd, w.C_gd)
    Vg = torch.from_numpy(w.Vg).cuda()
    g = m.ground_state(Vg)
    _, EC = m.inverse()
    c = m.thermal(Vg, 1e-5 * EC)
    om = oracle.Model(w.C_dd, w.C_gd)
    o = om.ground_state(w.Vg)
    clear = torch.from_numpy(o["E2"] - o["E"] > 1e-2 * EC).cuda()
    assert clear.sum() > 1000
    assert torch.allclose(c["Nmean"][clear], g["N"][clear].double(), atol=1e-9)
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(api.QaError) as e:
            m.thermal(Vg, bad)
        assert e.value.status == 1


# ---- dataset batch: one launch over several models == a loop over the single-model call ------------------------------
def test_batch_equals_loop_and_oracle(api):
    wls = [wl.config5_array(j, 40, 33) for j in range(5)]
    models = [api.Model(w.C_dd, w.C_gd) for w in wls]
    batch = api.Batch(models)
    assert len(batch) == 5
    Vg = torch.from_numpy(np.stack([w.Vg for w in wls])).cuda()
    for kw in (dict(algorithm="default"), dict(algorithm="thresholded", t=0.2), dict(algorithm="thresholded", t=0.5),
               dict(algorithm="default", regime="closed", N_hat=8)):
        rb = batch.ground_state(Vg, want_xcont=True, want_stats=True, **kw)
        torch.cuda.synchronize()
        assert api.last_launch_plan()[0] == ["qa_fused_small_kernel" if kw.get("regime") == "closed" else "qa_fused_open_kernel"]
        tot = 0
        for j, (w, m) in enumerate(zip(wls, models)):
            r1 = m.ground_state(Vg[j], **kw)
            assert torch.equal(rb["N"][j], r1["N"]) and torch.equal(rb["E"][j], r1["E"])
            om = oracle.Model(w.C_dd, w.C_gd)
            okw = {k: v for k, v in kw.items() if k not in ("regime", "N_hat")}
            o = om.ground_state(w.Vg, regime=kw.get("regime", "open"), N_hat=kw.get("N_hat", 0), **okw)
            compare(rb["N"][j].cpu().numpy(), rb["E"][j].cpu().numpy(), o, om.EC, gpu_x=rb["xcont"][j].cpu().numpy())
            tot += int(o["n_scored"].sum())
        st = api.stats_dict(rb["stats"])
        assert st["n_pixels"] == 5 * wls[0].P and st["n_candidates_scored"] == tot
    with pytest.raises(api.QaError) as e:
        api.Batch([models[0], api.Model(wl.config1(4, 4).C_dd, wl.config1(4, 4).C_gd)])
    assert e.value.status == 1
    w16 = wl.config4(2, 2)
    with pytest.raises(api.QaError) as e:
        api.Batch([api.Model(w16.C_dd, w16.C_gd)])
    assert e.value.status == 4


@pytest.mark.parametrize("n", [2, 4, 5, 7, 8])
def test_batch_multi_equals_separate_calls(api, n):
    """qa_ground_state_batch_multi (several algorithms on one sweep in one launch: S1-S3 once per pixel) is a loop over
    qa_ground_state_batch: N, E, x bit-identical, statistics summed; ragged P; a pass order with the default algorithm in
    the middle; QP pixels present (negative N_c)."""
    B, P = 3, 333
    wls = [wl.random_open(n, n + 1, P, seed=4000 + 10 * n + j, lo=-0.8, hi=2.6) for j in range(B)]
    models = [api.Model(w.C_dd, w.C_gd) for w in wls]
    batch = api.Batch(models)
    Vg = torch.from_numpy(np.stack([w.Vg for w in wls])).cuda()
    algs = [("thresholded", 0.2), ("default", None), ("thresholded", 0.5), ("thresholded", 0.0)]
    rm = batch.ground_state_multi(Vg, algs, want_xcont=True, want_stats=True)
    torch.cuda.synchronize()
    assert api.last_launch_plan()[0] == ["qa_fused_open_multi_kernel"]
    tot = {}
    for k, (name, t) in enumerate(algs):
        kw = dict(algorithm=name) if t is None else dict(algorithm=name, t=t)
        r1 = batch.ground_state(Vg, want_xcont=True, want_stats=True, **kw)
        assert torch.equal(rm[k]["N"], r1["N"]) and torch.equal(rm[k]["E"], r1["E"])
        assert torch.equal(rm[0]["xcont"], r1["xcont"])
        for key, v in api.stats_dict(r1["stats"]).items():
            tot[key] = tot.get(key, 0) + v
    assert api.stats_dict(rm[0]["stats"]) == tot and tot["n_qp_pixels"] > 0
    # against the oracle, one member
    om = oracle.Model(wls[1].C_dd, wls[1].C_gd)
    for k, (name, t) in enumerate(algs):
        okw = dict(algorithm=name) if t is None else dict(algorithm=name, t=t)
        o = om.ground_state(wls[1].Vg, **okw)
        compare(rm[k]["N"][1].cpu().numpy(), rm[k]["E"][1].cpu().numpy(), o, om.EC, gpu_x=rm[0]["xcont"][1].cpu().numpy())
    # a threshold above 0.6 among them: the call falls back to one launch per algorithm, same results
    rf = batch.ground_state_multi(Vg, [("thresholded", 0.8), ("default", None)])
    assert api.last_launch_plan()[0] == ["qa_fused_open_kernel", "qa_fused_open_kernel"]
    r8 = batch.ground_state(Vg, algorithm="thresholded", t=0.8)
    assert torch.equal(rf[0]["N"], r8["N"]) and torch.equal(rf[0]["E"], r8["E"]) and torch.equal(rf[1]["N"], rm[1]["N"])
    with pytest.raises(api.QaError):
        batch.ground_state_multi(Vg, [("brute", None)])
    with pytest.raises(api.QaError):
        batch.ground_state_multi(Vg, [0.2] * 5)


def test_batch_multi_general_cdd(api):
    """A c_dd with positive off-diagonals (every pixel takes the general QP solver's slow path) through the multi call."""
    wls = [wl.random_general(6, 6, 97, seed=4200 + j) for j in range(2)] if hasattr(wl, "random_general") else None
    if wls is None:
        pytest.skip("no general-c_dd generator")
    models = [api.Model(w.C_dd, w.C_gd) for w in wls]
    batch = api.Batch(models)
    Vg = torch.from_numpy(np.stack([w.Vg for w in wls])).cuda()
    rm = batch.ground_state_multi(Vg, ["default", 0.3])
    for k, kw in enumerate((dict(algorithm="default"), dict(algorithm="thresholded", t=0.3))):
        r1 = batch.ground_state(Vg, **kw)
        assert torch.equal(rm[k]["N"], r1["N"]) and torch.equal(rm[k]["E"], r1["E"])


# ---- edge cases -----------------------------------------------------------------------------------------------------
def test_edge_cases(api):
    w = wl.config1(4, 4)
    m = api.Model(w.C_dd, w.C_gd)
    # empty input
    r = m.ground_state(torch.empty((0, 2), dtype=torch.float64, device="cuda"))
    assert r["N"].shape == (0, 2)
    # single pixel, all-negative N_c (everything clamped -> N = 0)
    r = m.ground_state(torch.tensor([[-3.0, -2.0]], dtype=torch.float64, device="cuda"), want_xcont=True)
    assert r["N"].cpu().tolist() == [[0, 0]] and r["xcont"].cpu().tolist() == [[0.0, 0.0]]
    # closed with N_hat = 0
    r = m.ground_state(torch.from_numpy(w.Vg).cuda(), regime="closed", N_hat=0)
    assert int(r["N"].abs().sum()) == 0
    # argument errors
    with pytest.raises(api.QaError) as e:
        m.ground_state(torch.from_numpy(w.Vg).cuda(), algorithm="thresholded", t=1.5)
    assert e.value.status == 1
    with pytest.raises(api.QaError) as e:
        m.ground_state(torch.from_numpy(w.Vg).cuda(), regime="closed", N_hat=-1)
    assert e.value.status == 5
    with pytest.raises(api.QaError) as e:
        m.ground_state(torch.from_numpy(w.Vg).cuda(), regime="closed", N_hat=30, algorithm="brute", n_max=3)
    assert e.value.status == 5
    w16 = wl.config4(2, 2)
    m16 = api.Model(w16.C_dd, w16.C_gd)
    with pytest.raises(api.QaError) as e:
        m16.ground_state(torch.from_numpy(w16.Vg).cuda(), algorithm="brute", n_max=20)
    assert e.value.status == 6
    with pytest.raises(api.QaError) as e:
        api.Model(np.array([[1.0, 0.3], [0.1, 1.0]]), np.eye(2))
    assert e.value.status == 2
    with pytest.raises(api.QaError) as e:
        api.Model(np.array([[1.0, -3.0], [-3.0, 1.0]]), np.eye(2))
    assert e.value.status == 3
    with pytest.raises(api.QaError) as e:
        api.Model(np.eye(17), np.eye(17))
    assert e.value.status == 4
    mp = api.Model(np.array([[1.0, 0.1], [0.1, 1.0]]), np.eye(2))   # positive off-diagonal: legal (general QP phase)
    r = mp.ground_state(torch.from_numpy(w.Vg).cuda())
    assert (r["N"] >= 0).all()
    with pytest.raises(TypeError):
        m.ground_state(torch.from_numpy(w.Vg))          # no CPU path


def test_host_entry_point_matches_device_entry_point(api):
    w = wl.config2(40, 30)
    m = api.Model(w.C_dd, w.C_gd)
    a = m.ground_state(torch.from_numpy(w.Vg).cuda(), regime="closed", N_hat=5)
    b = m.ground_state_host(torch.from_numpy(w.Vg).pin_memory(), regime="closed", N_hat=5, want_stats=True)
    assert torch.equal(a["N"].cpu(), b["N"]) and torch.equal(a["E"].cpu(), b["E"])
    assert b["stats"]["n_pixels"] == w.P


def test_deterministic_across_runs_and_streams(api):
    w = wl.config4(8, 8)
    m = api.Model(w.C_dd, w.C_gd)
    Vg = torch.from_numpy(w.Vg).cuda()
    a = m.ground_state(Vg)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        m2 = api.Model(w.C_dd, w.C_gd)
        b = m2.ground_state(Vg)
    torch.cuda.synchronize()
    assert torch.equal(a["N"], b["N"]) and torch.equal(a["E"], b["E"])


# ---- exact ties (reading R6): the lexicographically smallest N among bitwise-equal energies ------------------------
@pytest.mark.parametrize("n,regime", [(5, "open"), (8, "open"), (10, "open"), (13, "open"), (16, "open"), (13, "closed"), (16, "closed")])
def test_pixels_are_independent_of_their_neighbours(api, n, regime):
    """Pixel-range sharding relies on it: the result of a pixel must not depend on which pixels share its
    thread, warp, CTA or call.  The same gate vectors in a shuffled order, and a sub-range of them, must give bit-identical
    N, E and x (two pixels per thread / warp, the CTA bucket sort, pixel pairs of the min-plus walk, the per-pixel choice of
    the QP solver in the sixteen-lanes prologue)."""
    w = wl.random_open(n, n, 419, seed=930 + n, lo=-0.8, hi=3.0)
    w.regime, w.N_hat = regime, n
    ref = run_gpu(api, w)
    perm = np.random.default_rng(n).permutation(w.P)
    w2 = wl.random_open(n, n, 419, seed=930 + n, lo=-0.8, hi=3.0)
    w2.regime, w2.N_hat = regime, n
    w2.Vg = np.ascontiguousarray(w.Vg[perm])
    g2 = run_gpu(api, w2)
    for key in ("N", "E", "xcont"):
        assert np.array_equal(ref[key][perm], g2[key]), key
    w3 = wl.random_open(n, n, 419, seed=930 + n, lo=-0.8, hi=3.0)
    w3.regime, w3.N_hat = regime, n
    w3.Vg = np.ascontiguousarray(w.Vg[37:230])
    w3.W = 193
    g3 = run_gpu(api, w3)
    for key in ("N", "E", "xcont"):
        assert np.array_equal(ref[key][37:230], g3[key]), key
    for algkw in (dict(algorithm="thresholded", t=0.4),):
        a = run_gpu(api, w, **algkw)
        b = run_gpu(api, w2, **algkw)
        assert np.array_equal(a["N"][perm], b["N"]) and np.array_equal(a["E"][perm], b["E"])


@pytest.mark.parametrize("n", [2, 5, 8, 10, 12, 13, 16])
def test_exact_ties_fall_to_the_lexicographically_smallest_state(api, n):
    """Diagonal c_dd with entries in {1/4, 1, 4} (so M = c_dd^-1 is exact), C_gd = I and N_c on quarter-integers: every
    energy term is a dyadic rational, all partial sums are exact in fp64 in ANY summation order, so the oracle's bitwise
    ties are bitwise ties on the GPU too and the result must equal the oracle's N exactly -- no near-tie excuse is used.
    First 64 pixels: N_c = k + 1/2 on every dot (all 2^n states tie -> N = floor N_c); last 64: a random subset of the
    dots at k + 1/2, the others at k + 1/4 or k + 3/4 (ties inside a sub-lattice)."""
    rng = np.random.default_rng(n)
    C_dd = np.diag(rng.choice([0.25, 1.0, 4.0], size=n))
    C_gd = np.eye(n)
    k = rng.integers(0, 3, size=(64, n)).astype(np.float64)
    Vg = k + 0.5
    half = rng.random((64, n)) < 0.5
    Vg2 = np.where(half, k + 0.5, k + rng.choice([0.25, 0.75], size=(64, n)))
    w = wl.Workload("ties", C_dd, C_gd, np.ascontiguousarray(np.concatenate([Vg, Vg2])), 128, 1)
    om = oracle.Model(C_dd, C_gd)
    assert np.array_equal(om.M, np.diag(1.0 / np.diag(C_dd)))
    o = om.ground_state(w.Vg)
    assert np.array_equal(o["N"][:64], k.astype(np.int32)) and (o["E2"] == o["E"])[:64].all()
    assert (o["E2"] == o["E"])[64:].sum() >= 32
    for variant in (1, 0, 2):
        g = run_gpu(api, w, variant=variant)
        assert np.array_equal(g["N"], o["N"]), (variant, np.nonzero((g["N"] != o["N"]).any(1))[0][:5])
        assert np.array_equal(g["E"], o["E"])
    if n <= 8:
        g = run_gpu(api, w, algorithm="thresholded", t=1.0)
        assert np.array_equal(g["N"], o["N"])


def test_device_affinity_and_batch_membership(api):
    w = wl.config1(4, 4)
    m = api.Model(w.C_dd, w.C_gd)
    b = api.Batch([m])
    with pytest.raises(api.QaError) as e:
        m.set_sensor_dots([1])                      # a batch holds the model's device constants
    assert e.value.status == 1
    b.close()
    m.set_sensor_dots([1])
    assert m.n_sensor == 1
    if torch.cuda.device_count() > 1:
        with pytest.raises(ValueError):
            m.ground_state(torch.from_numpy(w.Vg).to("cuda:1"))


# ---- full BASELINE.json sizes, EVERY pixel against the oracle (OpenMP over pixels), in bench.py's launch configuration ----
def test_full_size_every_pixel_configs_1_to_4(api):
    """The report bench.py prints as "parity": configs 1-4 at full size, every pixel, strict (any unexcused mismatch or an
    energy / continuous-minimum error above tolerance raises).  Config 4: the min-plus walk, the pruned walk and the
    exact-compare walk, each against the oracle (10^4 pixels x 2^16 candidates)."""
    rep = full_size_report(api, oracle, wl, torch, strict=True, configs=(1, 2, 3, 4))
    assert rep["config1"]["pixels"] == 20000 and rep["config1"]["default_vs_brute_mismatch"] == 0
    assert rep["config2"]["pixels"] == 30000 and rep["config2"]["qp_pixels"] > 0
    assert rep["config3"]["pixels"] == 40000 and rep["config3"]["sensor_unexcused"] == 0
    assert rep["config4"]["pixels"] == 10000 and rep["config4"]["unexcused_all_variants"] == 0
    assert rep["config4"]["qp_pixels"] > 1000


def test_full_size_config4_properties(api):
    """Properties that hold at any size, on the full 100x100 diagram in bench.py's launch configuration."""
    w = wl.config4(100, 100)
    m = api.Model(w.C_dd, w.C_gd)
    r = m.ground_state(torch.from_numpy(w.Vg).cuda(), want_xcont=True)
    torch.cuda.synchronize()
    N, E, x = r["N"].cpu().numpy(), r["E"].cpu().numpy(), r["xcont"].cpu().numpy()
    assert (N >= 0).all() and (N - np.floor(x) >= 0).all() and (N - np.floor(x) <= 1).all()
    # E(N*) equals the definition, and no single-dot move inside the candidate box lowers it
    Minv = np.linalg.inv(w.C_dd)
    nc = w.Vg @ w.C_gd.T
    d = N - nc
    assert np.allclose(E, 0.5 * np.einsum("pi,ij,pj->p", d, Minv, d), rtol=1e-9)
    grad = d @ Minv
    lo = np.maximum(np.floor(x), 0)
    up_ok = (N - lo) < 1
    dn_ok = (N - lo) > 0
    half = 0.5 * np.diag(Minv)
    assert (np.where(up_ok, grad + half, 1.0) >= -1e-9).all()
    assert (np.where(dn_ok, -grad + half, 1.0) >= -1e-9).all()


def test_full_size_config5_every_member_every_pixel(api):
    """The launch configuration bench.py times for the dataset batch (qa_ground_state_batch over full 128x128 members): all
    256 members x 3 algorithms, every pixel against the oracle (3 x 4.19 M pixel searches)."""
    rep = full_size_report(api, oracle, wl, torch, strict=True, configs=(5,))["config5"]
    assert rep["pixels"] == 3 * 256 * 128 * 128 and rep["unexcused"] == 0 and rep["qp_pixels"] > 0


# ---- charge-sensor response, noise and gradient (reading R14) ------------------------------------
@pytest.mark.parametrize("W,H", [(200, 200), (37, 29), (1, 5), (4099, 3)])
def test_sensor_response_config3_profiles_noise_gradient(api, W, H):
    """qa_sensor_response on the sensor potential of config 3 (computed by the CUDA path) against qo_sensor_response on the
    same potentials: every profile, each noise term alone and all together, gradient included.  Tolerance: 1e-9 of the
    signal scale (the draws are the same counter-based numbers; log / cos / the order of the jump prefix sum differ in the
    last bits).  Sizes span several 1024-pixel chunks, ragged tails and rows longer than a chunk."""
    w = wl.config3(W, H)
    m = api.Model(w.C_dd, w.C_gd, sensor_dots=w.sensor_dots)
    r = m.ground_state(torch.from_numpy(w.Vg).cuda())
    Vs = r["Vsensor"]
    vs = Vs.cpu().numpy()
    v0, wd = float(np.median(vs)), float(max(1e-3, 0.3 * (vs.max() - vs.min() + 1e-3)))
    cases = [dict(profile="lorentzian", v0=v0, width=wd, amplitude=1.5),
             dict(profile="gaussian", v0=v0, width=wd, amplitude=0.7),
             dict(profile="linear", v0=v0, width=wd, amplitude=-2.0),
             dict(profile="lorentzian", v0=v0, width=wd, amplitude=1.0, white_sigma=0.05, seed=5),
             dict(profile="lorentzian", v0=v0, width=wd, amplitude=1.0, pink_sigma=0.08, pink_octaves=14, seed=6),
             dict(profile="gaussian", v0=v0, width=wd, amplitude=1.0, jump_rate=0.004, jump_sigma=0.2, seed=7),
             dict(profile="lorentzian", v0=v0, width=wd, amplitude=1.0, white_sigma=0.02, pink_sigma=0.05, pink_octaves=30,
                  jump_rate=0.01, jump_sigma=0.1, seed=2 ** 63 + 11)]
    for kw in cases:
        g = api.sensor_response(Vs, W, [api.sensor_params(**kw)])
        torch.cuda.synchronize()
        o = oracle.sensor_response(vs, W, [oracle.sensor_params(**kw)])
        scale = abs(kw["amplitude"]) + kw.get("white_sigma", 0) + kw.get("pink_sigma", 0) + np.abs(o["S"]).max()
        assert np.abs(g["S"].cpu().numpy() - o["S"]).max() <= 1e-9 * scale, kw
        assert np.abs(g["G"].cpu().numpy() - o["G"]).max() <= 1e-9 * scale, kw
    if W == 200:
        assert api.last_launch_plan()[0] == ["qa_sensor_jump_partials_kernel", "qa_sensor_jump_scan_kernel",
                                             "qa_sensor_signal_kernel", "qa_sensor_gradient_kernel"]


def test_sensor_response_two_sensors_long_trace_and_errors(api):
    """Two sensors with different parameters (independent streams), a trace of 3 * 2^18 pixels (768 chunks: the scan of the
    chunk sums runs three rounds), no gradient requested; argument errors."""
    P, W = 3 << 18, 1 << 10
    rng = np.random.default_rng(3)
    vs = np.ascontiguousarray(rng.uniform(-0.1, 0.1, size=(P, 2)))
    Vs = torch.from_numpy(vs).cuda()
    kws = [dict(profile="lorentzian", v0=0.01, width=0.03, amplitude=1.0, white_sigma=0.01, pink_sigma=0.02, pink_octaves=18,
                jump_rate=0.0005, jump_sigma=0.3, seed=21),
           dict(profile="gaussian", v0=-0.02, width=0.05, amplitude=2.0, jump_rate=0.002, jump_sigma=0.1, seed=21)]
    g = api.sensor_response(Vs, W, [api.sensor_params(**k) for k in kws], want_gradient=False)
    torch.cuda.synchronize()
    o = oracle.sensor_response(vs, W, [oracle.sensor_params(**k) for k in kws], want_gradient=False)
    scale = 2.0 + np.abs(o["S"]).max()
    assert np.abs(g["S"].cpu().numpy() - o["S"]).max() <= 1e-9 * scale
    assert "G" not in g
    for bad in (dict(width=0.0), dict(pink_octaves=31), dict(jump_rate=1.5), dict(white_sigma=-1.0), dict(profile=3)):
        with pytest.raises(api.QaError):
            api.sensor_response(Vs, W, [api.sensor_params(**bad)] * 2)
    with pytest.raises(api.QaError):
        api.sensor_response(Vs, W + 1, [api.sensor_params()] * 2)
