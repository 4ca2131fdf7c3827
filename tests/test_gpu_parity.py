"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI binding, against the oracle, element by element on
the same seeded inputs; plus edge cases and full-size sampled checks in the launch configuration bench.py times."""
import numpy as np
import pytest
import torch

import oracle
from paper_2404_04994_b200 import workloads as wl
from parity import compare

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2404_04994_b200 import api as _api
    assert torch.cuda.is_available()
    return _api


def run_gpu(api, w, **kw):
    m = api.Model(w.C_dd, w.C_gd, sensor_dots=w.sensor_dots)
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


def check(api, w, **kw):
    g = run_gpu(api, w, **kw)
    m, o = run_oracle(w, **kw)
    rep = compare(g["N"], g["E"], o, m.EC, gpu_x=g["xcont"])
    st = g["stats"]
    assert st["n_pixels"] == w.P and st["n_qp_failed"] == 0
    assert st["n_qp_pixels"] == int(((o["flags"] & oracle.FLAG_QP) != 0).sum())
    assert st["n_candidates_enumerated"] == int(o["n_enum"].sum())
    assert st["n_candidates_scored"] == int(o["n_scored"].sum())
    assert st["n_threshold_doublings"] == int(o["doublings"].sum())
    assert st["n_widened_pixels"] == int(((o["flags"] & oracle.FLAG_WIDENED) != 0).sum())
    assert abs(g["EC"] - m.EC) <= 1e-12 * m.EC
    return rep, g, o


# ---- the five BASELINE.json configs at sizes the oracle finishes in seconds (several tiles + ragged tails) ----------
def test_config1_open_double_dot_default_and_brute(api):
    w = wl.config1(100, 100)
    rep, g, o = check(api, w, algorithm="default")
    assert g["plan"][0] == ["qa_fused_small_kernel"]
    assert st_zero_qp(g)
    check(api, w, algorithm="brute", n_max=5)


def st_zero_qp(g):
    return g["stats"]["n_qp_pixels"] == 0


def test_config2_closed_chain_default_and_brute(api):
    w = wl.config2(100, 100)
    rep, g, o = check(api, w, algorithm="default")
    assert g["stats"]["n_qp_pixels"] > 0
    assert (g["N"].sum(1) == 5).all()
    w2 = wl.config2(37, 23)
    check(api, w2, algorithm="brute", n_max=5)
    check(api, w2, algorithm="thresholded", t=0.3)
    check(api, w2, algorithm="thresholded", t=0.0)


def test_config3_sensor(api):
    w = wl.config3(64, 45)
    g = run_gpu(api, w, algorithm="default")
    o = oracle.sensor_ground_state(w.C_dd, w.C_gd, w.sensor_dots, w.Vg)
    full = oracle.Model(w.C_dd, w.C_gd)
    D = [0, 1, 2, 3]
    sub = oracle.Model(w.C_dd[np.ix_(D, D)], w.C_gd[D, :])
    rep = compare(g["N"], g["E"], dict(o, N=o["N"][:, D]), sub.EC, cols=D)
    same = (g["N"] == o["N"]).all(1)
    assert same.mean() > 0.999
    assert np.allclose(g["Vsensor"][same], o["Vs"][same], rtol=1e-9, atol=1e-9 * full.EC)
    assert g["xcont"].shape == (w.P, 4)


@pytest.mark.parametrize("W,H", [(9, 7), (33, 3)])
def test_config4_open_grid16_default(api, W, H):
    """n = 16, 2^16 candidates per pixel: the hot kernel (NL = 8, NH = 8), QP pixels included."""
    w = wl.config4(W, H)
    rep, g, o = check(api, w, algorithm="default")
    assert g["plan"][0] == ["qa_prologue_kernel", "qa_minplus_walk_kernel", "qa_minplus_finish_kernel"]
    assert g["stats"]["n_candidates_scored"] == w.P * 65536


@pytest.mark.parametrize("n,P", [(13, 45), (14, 46), (15, 33), (16, 45), (16, 1)])
def test_walk_variants_agree(api, n, P):
    """The exact-compare Gray walk (variant 0), the min-plus walk + finish kernel (variant 1, the default for n >= 13)
    and the min-plus walk with exact pruning of the high patterns (variant 2) give the same charge map and the same
    energies up to the summation order of E(N*); each is also checked against the oracle.  P odd / P = 1: the ragged
    last pixel pair of the min-plus walks."""
    w = wl.random_open(n, n, P, seed=200 + n)
    ref = None
    plans = {0: ["qa_prologue_kernel", "qa_walk_kernel", "qa_finalize_kernel"],
             1: ["qa_prologue_kernel", "qa_minplus_walk_kernel", "qa_minplus_finish_kernel"],
             2: ["qa_prologue_kernel", "qa_minplus_pruned_kernel", "qa_minplus_finish_kernel"]}
    try:
        for variant in (0, 1, 2):
            api.set_walk_variant(variant)
            rep, g, o = check(api, w, algorithm="default")
            assert g["plan"][0] == plans[variant]
            if ref is None:
                ref = g
            else:
                assert np.array_equal(ref["N"], g["N"])
                assert np.allclose(ref["E"], g["E"], rtol=1e-13, atol=1e-13 * g["EC"])
    finally:
        api.set_walk_variant(1)


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
        try:
            for variant in (0, 1, 2):
                api.set_walk_variant(variant)
                r = m.ground_state(Vg)
                torch.cuda.synchronize()
                outs[variant] = (r["N"].cpu().numpy(), r["E"].cpu().numpy())
        finally:
            api.set_walk_variant(1)
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
    Vg = np.concatenate([w.Vg, -50.0 * np.abs(rng.standard_normal((7, 16))), w.Vg[:9] * 40.0, np.zeros((3, 16))])
    w.Vg, w.W, w.H = np.ascontiguousarray(Vg), Vg.shape[0], 1
    try:
        for variant in (0, 1, 2):
            api.set_walk_variant(variant)
            check(api, w, algorithm="default")
    finally:
        api.set_walk_variant(1)


def test_config5_open_grid8_default_and_thresholded(api):
    for j in (0, 7):
        w = wl.config5_array(j, 48, 41)
        check(api, w, algorithm="default")
        for t in (0.2, 0.5, 1.0):
            check(api, w, algorithm="thresholded", t=t)


# ---- every n_dot through the static walk and the generic enumeration ----------------------------------------------
@pytest.mark.parametrize("n", list(range(1, 17)))
def test_all_sizes_default_open(api, n):
    w = wl.random_open(n, n + (n % 3), 301 if n <= 10 else (67 if n <= 13 else 37), seed=50 + n)
    rep, g, o = check(api, w, algorithm="default")
    if n <= 8:   # the one-kernel path above; the three-kernel path (static Gray walk) below
        assert g["plan"][0] == ["qa_fused_small_kernel"]
        try:
            api.set_walk_variant(0)
            rep, g0, o = check(api, w, algorithm="default")
            assert g0["plan"][0] == ["qa_prologue_kernel", "qa_walk_kernel", "qa_finalize_kernel"]
            assert np.array_equal(g["N"], g0["N"])
        finally:
            api.set_walk_variant(1)


@pytest.mark.parametrize("n", [1, 2, 3, 6, 9, 11])
@pytest.mark.parametrize("variant", [1, 0])
def test_all_sizes_closed_and_thresholded(api, n, variant):
    api.set_walk_variant(variant)
    try:
        _closed_and_thresholded(api, n)
    finally:
        api.set_walk_variant(1)


def _closed_and_thresholded(api, n):
    w = wl.random_open(n, n, 203, seed=80 + n, lo=-0.4, hi=2.5)
    w.regime, w.N_hat = "closed", max(1, n)
    check(api, w, algorithm="default")
    check(api, w, algorithm="thresholded", t=0.25)
    w.regime = "open"
    check(api, w, algorithm="thresholded", t=0.4)
    if n <= 6:
        check(api, w, algorithm="brute", n_max=3)
        w.regime = "closed"
        check(api, w, algorithm="brute", n_max=3)


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
        assert api.last_launch_plan()[0] == ["qa_fused_small_kernel"]
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


# ---- full BASELINE.json sizes in bench.py's launch configuration: sampled outputs + properties ---------------------
@pytest.mark.parametrize("variant", [1, 2])
def test_full_size_config4_sampled(api, variant):
    w = wl.config4(100, 100)
    m = api.Model(w.C_dd, w.C_gd)
    api.set_walk_variant(variant)
    try:
        r = m.ground_state(torch.from_numpy(w.Vg).cuda(), want_xcont=True)
        torch.cuda.synchronize()
    finally:
        api.set_walk_variant(1)
    N, E, x = r["N"].cpu().numpy(), r["E"].cpu().numpy(), r["xcont"].cpu().numpy()
    assert (N >= 0).all() and (N - np.floor(x) >= 0).all() and (N - np.floor(x) <= 1).all()
    rng = np.random.default_rng(0)
    sel = np.sort(rng.choice(w.P, size=24, replace=False))
    om = oracle.Model(w.C_dd, w.C_gd)
    o = om.ground_state(w.Vg[sel])
    compare(N[sel], E[sel], o, om.EC, gpu_x=x[sel])
    # property at any size: E(N*) equals the definition, and no single-dot move inside the candidate box lowers it
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


def test_full_size_config5_batch_call_sampled(api):
    """The launch configuration bench.py --workload config5 times (qa_ground_state_batch over full 128x128 members),
    on 16 members: sampled pixels of every member against the oracle, all three algorithms."""
    B = 16
    wls = [wl.config5_array(j) for j in range(B)]
    batch = api.Batch([api.Model(w.C_dd, w.C_gd) for w in wls])
    Vg = torch.from_numpy(np.stack([w.Vg for w in wls])).cuda()
    rng = np.random.default_rng(3)
    for kw in (dict(algorithm="default"), dict(algorithm="thresholded", t=0.2), dict(algorithm="thresholded", t=0.5)):
        r = batch.ground_state(Vg, **kw)
        N, E = r["N"].cpu().numpy(), r["E"].cpu().numpy()
        assert (N >= 0).all()
        for j, w in enumerate(wls):
            sel = np.sort(rng.choice(w.P, size=250, replace=False))
            om = oracle.Model(w.C_dd, w.C_gd)
            compare(N[j][sel], E[j][sel], om.ground_state(w.Vg[sel], **kw), om.EC)


def test_full_size_config5_batch_member_sampled(api):
    w = wl.config5_array(3)
    m = api.Model(w.C_dd, w.C_gd)
    om = oracle.Model(w.C_dd, w.C_gd)
    rng = np.random.default_rng(1)
    sel = np.sort(rng.choice(w.P, size=3000, replace=False))
    Vg = torch.from_numpy(w.Vg).cuda()
    for kw in (dict(algorithm="default"), dict(algorithm="thresholded", t=0.2), dict(algorithm="thresholded", t=0.5)):
        r = m.ground_state(Vg, **kw)
        o = om.ground_state(w.Vg[sel], **kw)
        compare(r["N"].cpu().numpy()[sel], r["E"].cpu().numpy()[sel], o, om.EC)
