"""Pins P0..P12 of DESIGN.md: the C oracle (oracle/qarray_oracle.c) checked against what the paper and the mathematics
fix -- values the paper prints, closed forms, invariants, special cases, brute force on tiny inputs, and independent
numpy / exact-rational routes.  No GPU, no CUDA path.  "L" = /root/reference/PAPER.md line."""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2404_04994_b200 import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    vals = {}
    with open(os.path.join(HERE, "golden", "paper_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                vals[k.strip()] = float(v)
    return vals


G = golden()
J1 = np.array([[G["j1_cdd_diag"], G["j1_cdd_off"]], [G["j1_cdd_off"], G["j1_cdd_diag"]]])
EX_CDD = np.array([[G["example_cdd_00"], G["example_cdd_01"]], [G["example_cdd_01"], G["example_cdd_00"]]])
EX_CGD = np.array([[G["example_cgd_00"], G["example_cgd_01"]], [G["example_cgd_01"], G["example_cgd_00"]]])


def chain(n, seed, coupling=(0.1, 0.3)):
    """config-2-shaped weakly coupled chain (kappa(M) well under Theorem E.3's bound for n <= 5)."""
    rng = np.random.default_rng(seed)
    C_m = np.zeros((n, n))
    for i in range(n - 1):
        C_m[i, i + 1] = C_m[i + 1, i] = rng.uniform(*coupling)
    lever = rng.uniform(0.8, 1.2, size=n)
    C_gd = np.array([[lever[i] * 0.3 ** abs(i - k) for k in range(n)] for i in range(n)])
    return wl.maxwell(C_m, C_gd), C_gd


# ---------------------------------------------------------------------------------------------------------- P0
def test_P0_maxwell_convention_paper_example():
    """L186-L192: cdd diagonal 1.3 = gate couplings 1.0 + 0.2 plus dot-dot coupling 0.1; offdiag = -0.1 (L35)."""
    C_m = np.array([[0.0, 0.1], [0.1, 0.0]])
    got = wl.maxwell(C_m, EX_CGD, self_cap=0.0)
    assert np.allclose(got, EX_CDD, atol=1e-15)
    m = oracle.Model(EX_CDD, EX_CGD)
    assert np.allclose(m.M @ EX_CDD, np.eye(2), atol=1e-14)


def test_model_inverse_and_validation():
    """M = c_dd^-1 (L41) against numpy; L204: symmetric + positive definite are validated."""
    for seed in range(5):
        w = wl.random_open(7, 9, 1, seed)
        m = oracle.Model(w.C_dd, w.C_gd)
        assert np.allclose(m.M, np.linalg.inv(w.C_dd), rtol=1e-12, atol=1e-14)
        assert np.allclose(m.C1, w.C_dd.sum(1)) and np.isclose(m.oneC1, w.C_dd.sum())
        assert np.isclose(m.EC, 0.5 * np.min(np.diag(np.linalg.inv(w.C_dd))))
    with pytest.raises(oracle.ModelError) as e:
        oracle.Model(np.array([[1.0, 0.2], [0.1, 1.0]]), np.eye(2))
    assert e.value.code == 2
    with pytest.raises(oracle.ModelError) as e:
        oracle.Model(np.array([[1.0, -2.0], [-2.0, 1.0]]), np.eye(2))
    assert e.value.code == 3


def test_R1_nc_is_the_fixed_order_fma_chain_bit_exact():
    """Reading R1: N_c,i = fma(C_gd[i,g-1], V[g-1], ... fma(C_gd[i,0], V[0], 0)).  Emulated in exact rational
    arithmetic (one rounding per fma) -- must agree to the last bit, and a reversed order must not always agree."""
    w = wl.random_open(5, 7, 40, seed=11)
    m = oracle.Model(w.C_dd, w.C_gd)
    differs_reversed = 0
    for p in range(w.P):
        got = m.nc(w.Vg[p])
        for i in range(5):
            acc, rev = 0.0, 0.0
            for k in range(7):
                acc = float(Fraction(w.C_gd[i, k]) * Fraction(w.Vg[p, k]) + Fraction(acc))
            for k in reversed(range(7)):
                rev = float(Fraction(w.C_gd[i, k]) * Fraction(w.Vg[p, k]) + Fraction(rev))
            assert got[i] == acc
            differs_reversed += got[i] != rev
    assert differs_reversed > 0
    assert np.allclose(m.nc(w.Vg[0]), w.C_gd @ w.Vg[0], rtol=1e-14)


# ---------------------------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("alg,kw", [("default", {}), ("thresholded", {"t": 0.3}), ("brute", {"n_max": 4})])
def test_P1_constraints(alg, kw):
    """(ii) N_i >= 0 (L52); (iii) closed sum N = N_hat (L56); Eq. (7): sum x = N_hat (L102)."""
    C_dd, C_gd = chain(4, 5)
    m = oracle.Model(C_dd, C_gd)
    rng = np.random.default_rng(0)
    Vg = rng.uniform(-1.0, 3.0, size=(300, 4))
    ro = m.ground_state(Vg, algorithm=alg, **kw)
    assert (ro["N"] >= 0).all() and (ro["flags"] & oracle.FLAG_QP_FAIL).max() == 0
    assert (ro["x"] >= 0).all()
    for N_hat in (0, 1, 3, 4):
        if alg == "brute" and N_hat > 4 * kw["n_max"]:
            continue
        rc = m.ground_state(Vg, regime="closed", N_hat=N_hat, algorithm=alg, **kw)
        assert (rc["N"] >= 0).all() and (rc["N"].sum(1) == N_hat).all()
        assert (rc["flags"] & (oracle.FLAG_QP_FAIL | oracle.FLAG_EMPTY | oracle.FLAG_WIDENED)).max() == 0
        assert (rc["x"] >= 0).all() and np.allclose(rc["x"].sum(1), N_hat, atol=1e-12)


def test_closed_analytic_minimum_solves_the_lagrangian_system():
    """Eq. (7) / (D1)-(D7) L630-L663: x, lambda solve [[M, -1], [1^T, 0]] [x; lambda] = [M N_c; N_hat] (independent
    numpy route through the stationarity conditions (D3), (D4))."""
    C_dd, C_gd = chain(5, 3)
    m = oracle.Model(C_dd, C_gd)
    M = np.linalg.inv(C_dd)
    rng = np.random.default_rng(3)
    for _ in range(50):
        nc = rng.uniform(0.5, 2.0, size=5)          # stays positive: no QP
        x, flags = m.continuous_min(nc, closed=True, N_hat=6)
        assert flags == 0
        K = np.block([[M, -np.ones((5, 1))], [np.ones((1, 5)), np.zeros((1, 1))]])
        sol = np.linalg.solve(K, np.concatenate([M @ nc, [6.0]]))
        assert np.allclose(x, sol[:5], rtol=1e-11, atol=1e-12)
    x, flags = m.continuous_min(np.array([0.3, 0.6, 1.2, 0.2, 0.9]), closed=False)
    assert flags == 0 and np.array_equal(x, [0.3, 0.6, 1.2, 0.2, 0.9])      # Eq. (6): x = N_c


# ---------------------------------------------------------------------------------------------------------- P2
@pytest.mark.parametrize("n,regime,N_hat", [(2, "open", 0), (4, "open", 0), (5, "closed", 5), (3, "closed", 2)])
def test_P2_default_equals_brute_force_on_weakly_coupled_arrays(n, regime, N_hat):
    """L472 "all implementations of all algorithms produce identical plots"; guaranteed when kappa(M) <= 1 + 4/n
    (Theorem E.3)."""
    C_dd, C_gd = chain(n, 100 + n, coupling=(0.02, 0.08))
    M = np.linalg.inv(C_dd)
    ev = np.linalg.eigvalsh(M)
    assert ev[-1] / ev[0] <= 1 + G["kappa_bound_numerator"] / n
    m = oracle.Model(C_dd, C_gd)
    rng = np.random.default_rng(n)
    target = rng.uniform(-0.5, 2.6, size=(400, n))
    Vg = target @ np.linalg.inv(C_gd).T
    rd = m.ground_state(Vg, regime=regime, N_hat=N_hat, algorithm="default")
    rb = m.ground_state(Vg, regime=regime, N_hat=N_hat, algorithm="brute", n_max=5)
    assert rd["N"].max() < 5
    assert np.array_equal(rd["N"], rb["N"])
    assert np.allclose(rd["E"], rb["E"], rtol=0, atol=0)


# ---------------------------------------------------------------------------------------------------------- P3
def test_P3_diagonal_cdd_rounds_to_nearest():
    """Theorem E.1 (L681-L683): diagonal M => N* = round-to-nearest of max(N_c, 0), open array."""
    rng = np.random.default_rng(7)
    n = 6
    C_dd = np.diag(rng.uniform(1.0, 3.0, size=n))
    C_gd = rng.uniform(0.0, 0.2, size=(n, n)) + np.diag(rng.uniform(0.8, 1.2, size=n))
    m = oracle.Model(C_dd, C_gd)
    target = rng.uniform(-1.0, 3.5, size=(500, n))
    Vg = target @ np.linalg.inv(C_gd).T
    nc = Vg @ C_gd.T
    keep = np.abs(nc - np.floor(nc) - 0.5).min(1) > 1e-9
    want = np.floor(np.maximum(nc, 0.0) + 0.5).astype(np.int32)
    for alg, kw in (("default", {}), ("brute", {"n_max": 5}), ("thresholded", {"t": 0.0}), ("thresholded", {"t": 0.4})):
        got = m.ground_state(Vg, algorithm=alg, **kw)["N"]
        assert np.array_equal(got[keep], want[keep]), alg


# ---------------------------------------------------------------------------------------------------------- P4
def test_P4_energy_definition_offset_and_local_minimum():
    """E = 1/2 d^T M d >= 0 (C1 L607); Eq. (4) L45 = E - 1/2 N_c^T M N_c; E via an independent route (solve c_dd y = d,
    E = 1/2 d.y, no inverse); brute-force winner is a discrete local minimum inside the box."""
    w = wl.random_open(6, 6, 200, seed=21)
    m = oracle.Model(w.C_dd, w.C_gd)
    rng = np.random.default_rng(1)
    Minv = np.linalg.inv(w.C_dd)
    for p in range(60):
        nc = m.nc(w.Vg[p])
        N = rng.integers(0, 4, size=6).astype(np.int32)
        d = N - nc
        e = m.energy(nc, N)
        assert e >= 0
        assert np.isclose(e, 0.5 * d @ np.linalg.solve(w.C_dd, d), rtol=1e-12)
        assert np.isclose(m.free_energy_eq4(nc, N), e - 0.5 * nc @ Minv @ nc, rtol=1e-11, atol=1e-12)
        # an asymmetric probe catches a transposed / half-summed M: E(N + e_i) - E(N) = (M d)_i + 1/2 M_ii, one dot only
        i = int(rng.integers(0, 6))
        N2 = N.copy()
        N2[i] += 1
        assert np.isclose(m.energy(nc, N2) - e, (Minv @ d)[i] + 0.5 * Minv[i, i], rtol=1e-10, atol=1e-12)
    assert m.energy(np.array([1.0, 2, 0, 3, 1, 1]), np.array([1, 2, 0, 3, 1, 1], dtype=np.int32)) == 0.0
    rb = m.ground_state(w.Vg, algorithm="brute", n_max=4)
    for p in range(w.P):
        nc = m.nc(w.Vg[p])
        N = rb["N"][p]
        assert np.isclose(rb["E"][p], m.energy(nc, N))
        for i in range(6):
            for s in (-1, 1):
                N2 = N.copy()
                N2[i] += s
                if 0 <= N2[i] <= 4:
                    assert m.energy(nc, N2) >= rb["E"][p]
        assert rb["E2"][p] >= rb["E"][p]


# ---------------------------------------------------------------------------------------------------------- P5
def test_P5_single_dot_transition_lines_closed_form():
    """From Eq. (4): E(N + e_i) - E(N) = 1/2 M_ii + [M (N - N_c)]_i.  So N* is a ground state only if, for every dot,
    [M (N* - N_c)]_i >= -1/2 M_ii and (where N*_i > 0) <= +1/2 M_ii -- i.e. every pixel lies on the correct side of
    the i-th addition lines (M C_gd V_g)_i = (M N)_i +- 1/2 M_ii.  Evaluated with numpy's inverse on config 1 and on the
    n = 5 chain; also locates the dot-1 line of the double dot to within one pixel and checks its slope -c/a."""
    for w, kw in ((wl.config1(60, 60), {}), (wl.config2(24, 24), {})):
        m = oracle.Model(w.C_dd, w.C_gd)
        M = np.linalg.inv(w.C_dd)
        if w.regime == "closed":
            continue
        r = m.ground_state(w.Vg)
        nc = w.Vg @ w.C_gd.T
        grad = (r["N"] - nc) @ M.T
        half = 0.5 * np.diag(M)
        assert (grad >= -half - 1e-12).all()
        assert (np.where(r["N"] > 0, grad, 0.0) <= half + 1e-12).all()
    # line location + slope in u = N_c coordinates: C_gd = I so that V = u
    C_dd = np.array([[1.5, -0.3], [-0.3, 1.2]])
    m = oracle.Model(C_dd, np.eye(2))
    M = np.linalg.inv(C_dd)
    a, c = M[0, 0], M[0, 1]
    u2s = np.array([0.1, 0.2, 0.3])             # dot 2 stays at 0 on this stretch
    xs = np.linspace(0.3, 0.7, 4001)
    cross = []
    for u2 in u2s:
        Vg = np.stack([xs, np.full_like(xs, u2)], 1)
        N = m.ground_state(Vg)["N"]
        assert (N[:, 1] == 0).all()
        k = int(np.argmax(N[:, 0] == 1))
        cross.append(xs[k])
        # closed form: a*(0 - u1) + c*(0 - u2) = -a/2  ->  u1 = 1/2 - (c/a) u2
        assert abs(xs[k] - (0.5 - c / a * u2)) <= 2e-4
    slope = np.polyfit(u2s, cross, 1)[0]
    assert abs(slope - (-c / a)) < 5e-3


# ---------------------------------------------------------------------------------------------------------- P6
def test_P6_honeycomb_triple_points_symmetric_double_dot():
    """Symmetric double dot M = [[a, c], [c, a]], C_gd = I.  Along the diagonal u1 = u2 = k + f:
    E(k,k) = E(k+1,k) at f = a / (2 (a + c)) and E(k+1,k) = E(k+1,k+1) at f = (a + 2c) / (2 (a + c)).
    For (J1) (L772): 0.4375 and 0.5625, spacing c/(a+c) = 0.125."""
    m = oracle.Model(J1, np.eye(2))
    M = np.linalg.inv(J1)
    a, c = M[0, 0], M[0, 1]
    f1, f2 = a / (2 * (a + c)), (a + 2 * c) / (2 * (a + c))
    assert np.isclose(f1, 0.4375) and np.isclose(f2, 0.5625)
    for k in (0, 1, 2):
        fs = np.linspace(0.0, 1.0, 2001)[:-1]
        u = k + fs
        # slightly off-diagonal (u1 > u2) so the middle state is (k+1, k) without a tie
        N = m.ground_state(np.stack([u + 1e-7, u], 1))["N"]
        lo = fs < f1 - 1e-3
        mid = (fs > f1 + 1e-3) & (fs < f2 - 1e-3)
        hi = fs > f2 + 1e-3
        assert (N[lo] == [k, k]).all() and (N[mid] == [k + 1, k]).all() and (N[hi] == [k + 1, k + 1]).all()
        # exactly on the diagonal the two middle states tie (up to rounding of M): either one, gap ~ 0
        rd = m.ground_state(np.stack([u, u], 1))
        assert (rd["N"][mid].sum(1) == 2 * k + 1).all() and (rd["E2"][mid] - rd["E"][mid] < 1e-12).all()


# ---------------------------------------------------------------------------------------------------------- P7
def test_P7_translation_invariance():
    """N*(V + C_gd^-1 k) = N*(V) + k for integer k when all N_c >= 1 (open; lattice periodicity of Eq. (4))."""
    C_dd, C_gd = chain(4, 9)
    m = oracle.Model(C_dd, C_gd)
    rng = np.random.default_rng(4)
    target = rng.uniform(1.0, 3.0, size=(200, 4))
    Vg = target @ np.linalg.inv(C_gd).T
    k = np.array([2, 0, 1, 3])
    r0 = m.ground_state(Vg)
    r1 = m.ground_state(Vg + np.linalg.solve(C_gd, k.astype(float))[None, :])
    assert np.array_equal(r1["N"], r0["N"] + k)
    assert np.allclose(r1["E"], r0["E"], rtol=1e-9, atol=1e-12)


# ---------------------------------------------------------------------------------------------------------- P8
def test_P8_thresholded_enumeration():
    """t = 1 == default on every pixel (L786); #candidates is a power of two <= 2^n; its mean over uniform fracs is
    (1 + t)^n within sampling error (Theorem G.1)."""
    n = 6
    C_dd, C_gd = chain(n, 12)
    m = oracle.Model(C_dd, C_gd)
    rng = np.random.default_rng(8)
    target = rng.uniform(0.0, 3.0, size=(4000, n))
    Vg = target @ np.linalg.inv(C_gd).T
    rd = m.ground_state(Vg)
    r1 = m.ground_state(Vg, algorithm="thresholded", t=1.0)
    assert np.array_equal(rd["N"], r1["N"]) and np.array_equal(rd["E"], r1["E"])
    assert (rd["n_scored"] == 2 ** n).all()
    for t in (0.2, 0.5):
        rt = m.ground_state(Vg, algorithm="thresholded", t=t)
        cnt = rt["n_scored"]
        assert ((cnt & (cnt - 1)) == 0).all() and (cnt <= 2 ** n).all() and (cnt >= 1).all()
        # exact per-pixel count from Eq. (9) applied to x = N_c (no QP here)
        frac = rt["x"] - np.floor(rt["x"])
        free = np.abs(frac - 0.5) <= t / 2
        assert np.array_equal(cnt, 2 ** free.sum(1))
        mean, want = cnt.mean(), (1 + t) ** n
        sem = cnt.std() / np.sqrt(len(cnt))
        assert abs(mean - want) < 5 * sem, (mean, want, sem)
        # fixed dots are rounded to the closest integer (L133)
        fixed_val = np.where(frac < 0.5, np.floor(rt["x"]), np.floor(rt["x"]) + 1)
        assert (np.where(free, rt["N"], fixed_val) == rt["N"]).all()


# ---------------------------------------------------------------------------------------------------------- P9
def test_P9_threshold_worked_example_J1():
    """App. J (L770-L774): for c_dd (J1) the thresholded diagram equals the default one for every t >= t_min, with the
    paper's empirical t_min = 1/7; the exact bound is c/(a+c) = 0.125 (P6 spacing).  Below it mismatches appear and grow;
    at t = 0 all interdot transitions are lost (the map is plain rounding of N_c)."""
    m = oracle.Model(J1, EX_CGD)
    g = np.linspace(0.0, 3.0, 161)
    u = np.stack(np.meshgrid(g, g), -1).reshape(-1, 2)
    Vg = u @ np.linalg.inv(EX_CGD).T
    ref = m.ground_state(Vg)["N"]
    mism = {}
    for t in (0.0, 0.05, 0.10, 0.125 + 1e-9, G["j1_tmin_empirical"], 0.5, 1.0):
        N = m.ground_state(Vg, algorithm="thresholded", t=t)["N"]
        mism[t] = int((N != ref).any(1).sum())
    assert mism[1.0] == 0 and mism[0.5] == 0 and mism[G["j1_tmin_empirical"]] == 0 and mism[0.125 + 1e-9] == 0
    assert mism[0.0] > mism[0.05] > mism[0.10] > 0
    N0 = m.ground_state(Vg, algorithm="thresholded", t=0.0)["N"]
    nc = Vg @ EX_CGD.T
    frac = nc - np.floor(nc)
    keep = np.abs(frac - 0.5).min(1) > 1e-9
    assert np.array_equal(N0[keep], np.floor(nc + 0.5).astype(np.int32)[keep])


# ---------------------------------------------------------------------------------------------------------- P10
def test_P10_candidate_counts():
    """2^n default (L127); 6^5 / 2^5 = 243 (L17); closed brute n=5, N_hat=5, n_max=5: C(9,4) = 126 valid of 7776."""
    C_dd, C_gd = chain(5, 2)
    m = oracle.Model(C_dd, C_gd)
    Vg = np.random.default_rng(0).uniform(0.2, 2.0, size=(20, 5))
    rd = m.ground_state(Vg)
    rb = m.ground_state(Vg, algorithm="brute", n_max=5)
    assert (rd["n_enum"] == 32).all() and (rb["n_enum"] == 7776).all() and (rb["n_scored"] == 7776).all()
    assert rb["n_enum"][0] // rd["n_enum"][0] == int(G["reduction_5dots_5charges"])
    rc = m.ground_state(Vg, regime="closed", N_hat=5, algorithm="brute", n_max=5)
    assert (rc["n_enum"] == 7776).all() and (rc["n_scored"] == 126).all()
    rcd = m.ground_state(Vg, regime="closed", N_hat=5, algorithm="default")
    assert (rcd["n_enum"] == 32).all()
    from math import comb
    k = 5 - np.floor(rcd["x"]).astype(int).sum(1)
    assert np.array_equal(rcd["n_scored"], [comb(5, int(v)) for v in k])


def test_P10_closed_default_scores_C_n_k_states_at_16_dots():
    """Closed default set at n = 16, N_hat = 16 (Fig. 4(b) shape, L496): 2^16 enumerated, exactly C(16, N_hat - sum lo) scored
    (L127: candidates with the wrong total are eliminated) -- 12 870 when k = 8 -- and the winner carries the total."""
    from math import comb
    from paper_2404_04994_b200 import workloads as wl
    w = wl.config4(5, 4)
    m = oracle.Model(w.C_dd, w.C_gd)
    r = m.ground_state(w.Vg, regime="closed", N_hat=16)
    lo = np.maximum(np.floor(r["x"]), 0).astype(int)
    k = 16 - lo.sum(1)
    assert (r["n_enum"] == 65536).all() and (k >= 0).all() and (k <= 16).all()
    assert np.array_equal(r["n_scored"], [comb(16, int(v)) for v in k])
    assert (r["N"].sum(1) == 16).all() and ((r["N"] - lo) >= 0).all() and ((r["N"] - lo) <= 1).all()


# ---------------------------------------------------------------------------------------------------------- P11
def _qp_by_active_set_enumeration(M, c, closed, N_hat):
    """All 2^n active sets with numpy; returns the unique KKT point (strict convexity, App. B)."""
    n = len(c)
    best = None
    for bits in range(2 ** n):
        A = [i for i in range(n) if bits >> i & 1]
        F = [i for i in range(n) if not bits >> i & 1]
        x = np.zeros(n)
        lam = 0.0
        if F:
            MFF = M[np.ix_(F, F)]
            rhs = (M @ c)[F]
            if closed:
                K = np.block([[MFF, -np.ones((len(F), 1))], [np.ones((1, len(F))), np.zeros((1, 1))]])
                sol = np.linalg.solve(K, np.concatenate([rhs, [N_hat]]))
                x[F], lam = sol[:-1], sol[-1]
            else:
                x[F] = np.linalg.solve(MFF, rhs)
        elif closed and N_hat != 0:
            continue
        r = M @ (x - c) - lam
        if (x >= -1e-11).all() and (r[A] >= -1e-11).all():
            obj = 0.5 * (x - c) @ M @ (x - c)
            if best is None or obj < best[1]:
                best = (x, obj)
    return best[0]


@pytest.mark.parametrize("closed", [False, True])
def test_P11_qp_exact(closed):
    """Eq. (8) L110-L119 solved exactly: agrees with exhaustive enumeration of active sets (n <= 7), KKT violation ~ 0,
    reduces to Eq. (6)/(7) when no bound is active, n = 1 closed => x = N_hat."""
    rng = np.random.default_rng(5 + closed)
    for trial in range(60):
        n = int(rng.integers(2, 8))
        w = wl.random_open(n, n, 1, seed=1000 + trial)
        m = oracle.Model(w.C_dd, w.C_gd)
        M = np.linalg.inv(w.C_dd)
        c = rng.uniform(-1.5, 2.0, size=n)
        N_hat = float(rng.integers(1, n + 2))
        x, it, kkt = m.qp(c, closed=closed, N_hat=N_hat)
        assert it > 0 and kkt < 1e-11
        want = _qp_by_active_set_enumeration(M, c, closed, N_hat)
        assert np.allclose(x, want, rtol=1e-9, atol=1e-10), (trial, x, want)
        assert (x >= 0).all()
        if closed:
            assert np.isclose(x.sum(), N_hat, atol=1e-12)
    # general SPD (non-Maxwell, positive off-diagonals) is handled too
    for trial in range(30):
        n = int(rng.integers(2, 7))
        A = rng.normal(size=(n, n))
        C_dd = A @ A.T + n * np.eye(n) * 0.3
        m = oracle.Model(C_dd, np.eye(n))
        c = rng.uniform(-1.5, 2.0, size=n)
        x, it, kkt = m.qp(c, closed=closed, N_hat=2.0)
        want = _qp_by_active_set_enumeration(np.linalg.inv(C_dd), c, closed, 2.0)
        assert it > 0 and np.allclose(x, want, rtol=1e-8, atol=1e-9)
    # inactive bounds: Eq. (6) / Eq. (7)
    w = wl.random_open(4, 4, 1, seed=3)
    m = oracle.Model(w.C_dd, w.C_gd)
    c = np.array([0.4, 1.2, 2.2, 0.7])
    x, it, _ = m.qp(c, closed=closed, N_hat=5.0)
    if closed:
        want = c + (5.0 - c.sum()) * w.C_dd.sum(1) / w.C_dd.sum()
        assert np.allclose(x, want, rtol=1e-12)
    else:
        assert np.allclose(x, c, rtol=1e-13)
    m1 = oracle.Model(np.array([[1.7]]), np.array([[1.0]]))
    x, it, _ = m1.qp(np.array([-0.3]), closed=True, N_hat=3.0)
    if closed:
        assert x[0] == 3.0


def test_qp_used_only_when_needed_and_flagged():
    """L82-L84, L106: the analytic solution is accepted iff it has no negative component."""
    w = wl.config2(20, 20)
    m = oracle.Model(w.C_dd, w.C_gd)
    r = m.ground_state(w.Vg, regime="closed", N_hat=5)
    nc = w.Vg @ w.C_gd.T
    x7 = nc + (5 - nc.sum(1))[:, None] * w.C_dd.sum(1)[None, :] / w.C_dd.sum()
    need = (x7 < 0).any(1)
    assert np.array_equal((r["flags"] & oracle.FLAG_QP) != 0, need)
    assert 0 < need.sum() < len(need)
    assert np.allclose(r["x"][~need], x7[~need], rtol=1e-12, atol=1e-13)
    assert (r["x"][need].min(1) == 0.0).all()       # clamped components are exactly 0 (R3)


def test_closed_qp_single_free_dot_is_bitwise_N_hat():
    """Reading R3: when all dots but one clamp, 1^T x = N_hat fixes the free component: exactly N_hat, bitwise (n >= 2);
    the clamped components are exactly 0, and the point is the KKT point of the exhaustive enumeration."""
    rng = np.random.default_rng(41)
    hits = 0
    for trial in range(40):
        n = int(rng.integers(2, 8))
        w = wl.random_open(n, n, 1, seed=2000 + trial)
        m = oracle.Model(w.C_dd, w.C_gd)
        M = np.linalg.inv(w.C_dd)
        f = int(rng.integers(0, n))
        c = rng.uniform(-6.0, -3.0, size=n)          # everything strongly repelled ...
        c[f] = rng.uniform(0.5, 3.0)                 # ... except one dot
        N_hat = float(rng.integers(1, 5))
        x, it, kkt = m.qp(c, closed=True, N_hat=N_hat)
        want = _qp_by_active_set_enumeration(M, c, True, N_hat)
        assert it > 0 and kkt < 1e-11 and np.allclose(x, want, atol=1e-10)
        if (want > 1e-9).sum() == 1:
            hits += 1
            assert x[f] == N_hat                      # bitwise
            assert (np.delete(x, f) == 0.0).all()
    assert hits >= 30
    # the same through the whole pixel pipeline: closed chain, one gate far positive, the others far negative
    C_dd, C_gd = chain(4, 3)
    m = oracle.Model(C_dd, C_gd)
    target = np.array([[-5.0, 2.0, -5.0, -5.0], [-4.0, -4.0, -4.0, 1.5]])
    r = m.ground_state(target @ np.linalg.inv(C_gd).T, regime="closed", N_hat=3)
    assert r["x"].tolist() == [[0.0, 3.0, 0.0, 0.0], [0.0, 0.0, 0.0, 3.0]]
    assert r["N"].tolist() == [[0, 3, 0, 0], [0, 0, 0, 3]]


def test_R5_closed_default_set_is_never_empty():
    """Reading R5: at t = 1 the kept set is the closed default set; for a feasible continuous minimum (x >= 0, sum x =
    N_hat up to rounding) sum floor(x) <= N_hat <= sum floor(x) + n, so it is never empty and no wider set is needed.
    Checked on the oracle's own x over analytic and QP pixels, Maxwell and general SPD c_dd, and through the flags."""
    for seed, gen in ((1, wl.random_open), (2, wl.random_open), (3, wl.random_general)):
        for n in (1, 2, 5, 8):
            if n == 1 and gen is wl.random_general:
                continue
            w = gen(n, n, 800, seed=300 + 10 * seed + n, lo=-1.5, hi=3.0)
            m = oracle.Model(w.C_dd, w.C_gd)
            for N_hat in (0, 1, n, 2 * n + 1):
                r = m.ground_state(w.Vg, regime="closed", N_hat=N_hat)
                x = r["x"]
                assert (x >= 0).all() and np.allclose(x.sum(1), N_hat, atol=1e-9)
                lo = np.floor(x).sum(1)
                assert ((lo <= N_hat) & (N_hat <= lo + n)).all()
                assert (r["flags"] & (oracle.FLAG_EMPTY | oracle.FLAG_WIDENED | oracle.FLAG_QP_FAIL)).max() == 0
                assert (r["N"].sum(1) == N_hat).all() and (r["n_scored"] >= 1).all()
                rt = m.ground_state(w.Vg, regime="closed", N_hat=N_hat, algorithm="thresholded", t=0.0)
                assert (rt["flags"] & oracle.FLAG_EMPTY).max() == 0 and (rt["N"].sum(1) == N_hat).all()


# ---------------------------------------------------------------------------------------------------------- P12
def test_P12_closed_two_dot_detuning_axis():
    """Closed double dot, N_hat = 1, M = [[a,c],[c,a']]: E(1,0) = E(0,1) <=> (a-c) u1 - (a'-c) u2 = (a-a')/2.  For
    a = a' the state switches exactly on u1 = u2, (1,0) where u1 > u2; the paper's own closed example keeps the total
    at 2 on every pixel (L454-L459)."""
    m = oracle.Model(J1, np.eye(2))
    rng = np.random.default_rng(2)
    u = rng.uniform(0.0, 1.5, size=(2000, 2))
    N = m.ground_state(u, regime="closed", N_hat=1)["N"]
    big = np.abs(u[:, 0] - u[:, 1]) > 1e-9
    assert (N[big & (u[:, 0] > u[:, 1])] == [1, 0]).all() and (N[big & (u[:, 0] < u[:, 1])] == [0, 1]).all()
    C_dd = np.array([[1.6, -0.25], [-0.25, 1.1]])
    m2 = oracle.Model(C_dd, np.eye(2))
    M = np.linalg.inv(C_dd)
    a, c, a2 = M[0, 0], M[0, 1], M[1, 1]
    s = (a - c) * u[:, 0] - (a2 - c) * u[:, 1] - (a - a2) / 2
    N2 = m2.ground_state(u, regime="closed", N_hat=1)["N"]
    far = np.abs(s) > 1e-9
    assert (N2[far & (s > 0)] == [1, 0]).all() and (N2[far & (s < 0)] == [0, 1]).all()
    mex = oracle.Model(EX_CDD, EX_CGD)
    g = np.linspace(-0.5, 3.0, 40)
    Vg = np.stack(np.meshgrid(g, g), -1).reshape(-1, 2)
    Nc = mex.ground_state(Vg, regime="closed", N_hat=int(G["closed_example_total"]))["N"]
    assert (Nc.sum(1) == G["closed_example_total"]).all() and (Nc >= 0).all()


# ---------------------------------------------------------------------------------------------------------- R5
def test_R5_closed_threshold_doubling():
    """L141: closed + thresholded with no admissible state -> double t (t = 0 -> 1) per pixel until non-empty."""
    C_dd, C_gd = chain(5, 6)
    m = oracle.Model(C_dd, C_gd)
    rng = np.random.default_rng(9)
    target = rng.uniform(0.0, 2.0, size=(1500, 5))
    Vg = target @ np.linalg.inv(C_gd).T
    rd = m.ground_state(Vg, regime="closed", N_hat=5)
    for t in (0.0, 0.1, 0.3):
        rt = m.ground_state(Vg, regime="closed", N_hat=5, algorithm="thresholded", t=t)
        assert (rt["N"].sum(1) == 5).all() and (rt["n_scored"] >= 1).all()
        assert rt["doublings"].max() >= 1 and (rt["flags"] & oracle.FLAG_WIDENED).max() == 0
        # replay the rule in numpy: smallest t_k in {t, 2t, 4t, .., 1} whose kept set can reach N_hat
        x = rt["x"]
        fl = np.floor(x)
        frac = x - fl
        for p in range(0, 1500, 7):
            tt, k = t, 0
            while True:
                free = np.abs(frac[p] - 0.5) <= tt / 2
                fixed = np.where(frac[p] < 0.5, fl[p], fl[p] + 1)
                smin = np.where(free, fl[p], fixed).sum()
                if smin <= 5 <= smin + free.sum() or tt >= 1.0:
                    break
                tt = min(1.0, 2 * tt) if tt > 0 else 1.0
                k += 1
            assert rt["doublings"][p] == k
        same = (rt["N"] == rd["N"]).all(1).mean()
        assert same > 0.5


# ---------------------------------------------------------------------------------------------------------- R6
def test_R6_tie_break_is_lexicographic():
    """Exact ties: symmetric double dot at N_c = (1/2, 1/2) + symmetric point: (0,1) and (1,0) tie -> (0,1); with a
    diagonal M at N_c = (0.5, 0.5) all four states tie -> (0,0)."""
    m = oracle.Model(np.diag([2.0, 2.0]), np.eye(2))
    r = m.ground_state(np.array([[0.5, 0.5]]))
    assert r["N"].tolist() == [[0, 0]] and r["E2"][0] == r["E"][0]
    rb = m.ground_state(np.array([[0.5, 0.5]]), algorithm="brute", n_max=3)
    assert rb["N"].tolist() == [[0, 0]]


# ---------------------------------------------------------------------------------------------------------- R8
def test_R8_sensor_closed_forms():
    """L149 + Eq. (3): array dots solved on the sub-blocks; sensor carrier number = integer nearest to the 1-D
    parabola's vertex s* (Theorem E.1 in one dimension), clamped at 0; V_s = [M (N - N_c)]_s.  numpy route."""
    w = wl.config3(30, 30)
    # config 3 keeps its sensor gate fixed (the sensor's carrier number is 1 on the whole sweep); ramp it here so that
    # the two-way choice of the sensor step is exercised across several transitions
    w.Vg[:, 4] = np.linspace(0.0, 3.0, w.P) / w.C_gd[4, 4]
    out = oracle.sensor_ground_state(w.C_dd, w.C_gd, w.sensor_dots, w.Vg)
    D = [0, 1, 2, 3]
    sub = oracle.Model(w.C_dd[np.ix_(D, D)], w.C_gd[D, :])
    rs = sub.ground_state(w.Vg)
    assert np.array_equal(out["N"][:, D], rs["N"]) and np.array_equal(out["E"], rs["E"])
    M = np.linalg.inv(w.C_dd)
    nc = w.Vg @ w.C_gd.T
    dD = out["N"][:, D] - nc[:, D]
    sstar = nc[:, 4] - (dD @ M[4, D]) / M[4, 4]
    keep = np.abs(sstar - np.floor(sstar) - 0.5) > 1e-9
    want = np.floor(np.maximum(sstar, 0.0) + 0.5).astype(np.int32)
    assert np.array_equal(out["N"][keep, 4], want[keep])
    d = out["N"] - nc
    assert np.allclose(out["Vs"][:, 0], d @ M[4, :], rtol=1e-11, atol=1e-13)
    assert len(np.unique(out["N"][:, 4])) >= 2 and out["Vs"].std() > 0
    # margin of the two-way choice: |e(c0+1) - e(c0)| with e(c) = (c - u) y + 1/2 M_ss (c - u)^2, i.e. M_ss |c0 + 1/2 - s*|
    c0 = np.floor(np.maximum(sstar, 0.0))
    assert np.allclose(out["sgap"][:, 0], M[4, 4] * np.abs(c0 + 0.5 - sstar), rtol=1e-9, atol=1e-12)


def test_R8_two_sensors_at_non_trailing_indices():
    """Reading R8 with several sensors: 6 dots, sensors {2, 5} (ns > 1, sensor indices between array dots).  Each sensor is
    rounded independently with the OTHER sensor at its continuous value (d = 0); V_s uses every final N.  numpy route."""
    w = wl.random_open(6, 7, 400, seed=77, lo=-0.3, hi=2.6)
    sens = (2, 5)
    D = [0, 1, 3, 4]
    out = oracle.sensor_ground_state(w.C_dd, w.C_gd, sens, w.Vg)
    sub = oracle.Model(w.C_dd[np.ix_(D, D)], w.C_gd[D, :])
    rs = sub.ground_state(w.Vg)
    assert np.array_equal(out["N"][:, D], rs["N"]) and np.array_equal(out["E"], rs["E"])
    M = np.linalg.inv(w.C_dd)
    nc = w.Vg @ w.C_gd.T
    dD = out["N"][:, D] - nc[:, D]
    for a, s_ in enumerate(sens):
        sstar = nc[:, s_] - (dD @ M[s_, D]) / M[s_, s_]
        keep = np.abs(sstar - np.floor(sstar) - 0.5) > 1e-9
        want = np.floor(np.maximum(sstar, 0.0) + 0.5).astype(np.int32)
        assert np.array_equal(out["N"][keep, s_], want[keep])
        assert len(np.unique(out["N"][:, s_])) >= 2
        c0 = np.floor(np.maximum(sstar, 0.0))
        assert np.allclose(out["sgap"][:, a], M[s_, s_] * np.abs(c0 + 0.5 - sstar), rtol=1e-9, atol=1e-12)
    d = out["N"] - nc
    assert np.allclose(out["Vs"], d @ M[list(sens), :].T, rtol=1e-11, atol=1e-13)


def test_brute_force_is_the_definition_on_the_box():
    """Eq. (5) L60 restricted to {0..n_max}^n: compare with itertools.product + numpy energies on a tiny array."""
    C_dd, C_gd = chain(3, 1, coupling=(0.2, 0.4))
    m = oracle.Model(C_dd, C_gd)
    M = np.linalg.inv(C_dd)
    rng = np.random.default_rng(3)
    Vg = rng.uniform(-0.5, 2.5, size=(40, 3))
    states = np.array(list(itertools.product(range(4), repeat=3)))
    for regime, N_hat in (("open", 0), ("closed", 4)):
        rb = m.ground_state(Vg, regime=regime, N_hat=N_hat, algorithm="brute", n_max=3)
        for p in range(40):
            nc = C_gd @ Vg[p]
            d = states - nc
            e = 0.5 * np.einsum("si,ij,sj->s", d, M, d)
            if regime == "closed":
                e = np.where(states.sum(1) == N_hat, e, np.inf)
            srt = np.sort(e)
            assert np.array_equal(rb["N"][p], states[int(np.argmin(e))])
            assert np.isclose(rb["E"][p], srt[0], rtol=1e-12) and np.isclose(rb["E2"][p], srt[1], rtol=1e-12)


def test_openmp_variant_is_the_same_function():
    if not oracle.has_openmp():
        pytest.skip("no OpenMP")
    w = wl.config2(16, 16)
    m = oracle.Model(w.C_dd, w.C_gd)
    a = m.ground_state(w.Vg, regime="closed", N_hat=5)
    b = m.ground_state(w.Vg, regime="closed", N_hat=5, n_threads=4)
    assert np.array_equal(a["N"], b["N"]) and np.array_equal(a["E"], b["E"])


# ---- P13: thermal broadening, Eq. (10) (L153-L159) -------------------------------------------------------------------
def _softargmin_numpy(C_dd, C_gd, vg, cands, kT):
    """Independent route: Eq. (4) free energy (NOT the completed square the oracle uses) and plain numpy sums."""
    M = np.linalg.inv(C_dd)
    q = np.asarray(cands, float)                                   # [K, n]
    nc = C_gd @ vg
    F = 0.5 * np.einsum("ki,ij,kj->k", q, M, q) - q @ (M @ nc)      # Eq. (4) L45 (positive-C_gd convention, R0b)
    w = np.exp(-(F - F.min()) / kT)
    return (w[:, None] * q).sum(0) / w.sum()


def test_P13_single_dot_is_a_fermi_function():
    """n = 1, default: candidates lo, lo+1 with E(N) = 1/2 M (N - N_c)^2, so <N> = lo + 1 / (1 + exp(dE / kT)),
    dE = E(lo+1) - E(lo) = M (lo - N_c) + M / 2: a Fermi function centred on the half-integer."""
    C = np.array([[1.7]])
    m = oracle.Model(C, np.array([[0.9]]))
    M = 1.0 / 1.7
    vg = np.linspace(0.05, 4.0, 173)[:, None]
    for kT in (0.004, 0.03, 0.4):
        o = m.thermal(vg, kT)
        nc = 0.9 * vg[:, 0]
        lo = np.floor(nc)
        dE = M * (lo - nc) + 0.5 * M
        assert np.allclose(o["Nmean"][:, 0], lo + 1.0 / (1.0 + np.exp(dE / kT)), rtol=0, atol=1e-13)
        assert np.allclose(o["Emin"], 0.5 * M * np.minimum(nc - lo, lo + 1 - nc) ** 2, atol=1e-15)


@pytest.mark.parametrize("regime,N_hat", [("open", 0), ("closed", 3)])
def test_P13_limits_and_independent_sum(regime, N_hat):
    n = 4
    C_dd, C_gd = chain(n, 21)
    m = oracle.Model(C_dd, C_gd)
    rng = np.random.default_rng(5)
    Vg = rng.uniform(0.1, 2.2, size=(60, n)) @ np.linalg.inv(C_gd).T
    g = m.ground_state(Vg, regime=regime, N_hat=N_hat)
    EC = m.EC
    # kT -> 0: the arg min of Eq. (5), wherever the runner-up is not within reach
    cold = m.thermal(Vg, 1e-4 * EC, regime=regime, N_hat=N_hat)
    clear = g["E2"] - g["E"] > 1e-2 * EC
    assert clear.sum() > 40 and np.allclose(cold["Nmean"][clear], g["N"][clear], atol=1e-12)
    assert np.array_equal(cold["Emin"], g["E"])
    # kT -> infinity: the plain mean of the candidate set
    hot = m.thermal(Vg, 1e12 * EC, regime=regime, N_hat=N_hat)
    lo = np.maximum(np.floor(g["x"]), 0)
    for p in range(len(Vg)):
        cands = [lo[p] + np.array(b) for b in itertools.product((0, 1), repeat=n)]
        if regime == "closed":
            cands = [c for c in cands if c.sum() == N_hat]
        assert np.allclose(hot["Nmean"][p], np.mean(cands, axis=0), atol=1e-9)
        # in between: Eq. (10) written out with Eq. (4) energies (per-pixel constants cancel)
        for kT in (0.02 * EC, 0.5 * EC):
            o = m.thermal(Vg[p:p + 1], kT, regime=regime, N_hat=N_hat)
            assert np.allclose(o["Nmean"][0], _softargmin_numpy(C_dd, C_gd, Vg[p], cands, kT), rtol=1e-10, atol=1e-12)
    if regime == "closed":   # constraint (iii) survives the average
        warm = m.thermal(Vg, 0.1 * EC, regime=regime, N_hat=N_hat)
        assert np.allclose(warm["Nmean"].sum(1), N_hat, atol=1e-12)


def test_P13_brute_force_box_and_bounds():
    C_dd, C_gd = chain(3, 8)
    m = oracle.Model(C_dd, C_gd)
    rng = np.random.default_rng(2)
    Vg = rng.uniform(0.0, 2.5, size=(25, 3)) @ np.linalg.inv(C_gd).T
    o = m.thermal(Vg, 0.07 * m.EC, algorithm="brute", n_max=3)
    box = [np.array(c, float) for c in itertools.product(range(4), repeat=3)]
    for p in range(len(Vg)):
        assert np.allclose(o["Nmean"][p], _softargmin_numpy(C_dd, C_gd, Vg[p], box, 0.07 * m.EC), rtol=1e-10, atol=1e-12)
    assert (o["Nmean"] >= 0).all() and (o["Nmean"] <= 3).all()
    with pytest.raises(ValueError):
        m.thermal(Vg, 0.0)


# ---------------------------------------------------------------------------------------------------------- P14
# Sensor response, noise and gradient (L149, L464; reading R14).  The paper prints no formula: what is pinned is what R14 fixes.
def test_P14_response_profiles_closed_forms():
    """Lorentzian: S(v0) = A, S(v0 +- w) = A/2 (w = HWHM), symmetric, S(v0 + 3w) = A/10; Gaussian: S(v0 +- w) = A e^-1/2,
    inflection at +-w; linear: A (V - v0)/w; Lorentzian and Gaussian agree to second order at the peak after matching
    curvature (w_G = w_L / sqrt 2)."""
    A, v0, w = 2.5, 0.3, 0.07
    V = np.array([v0, v0 + w, v0 - w, v0 + 3 * w, v0 - 3 * w, v0 + 1e-4, v0 - 1e-4])[:, None]
    L = oracle.sensor_response(V, 1, [oracle.sensor_params("lorentzian", v0, w, A)])["S"][:, 0]
    assert L[0] == A and abs(L[1] - A / 2) < 1e-15 and abs(L[2] - A / 2) < 1e-15
    assert abs(L[3] - A / 10) < 1e-15 and abs(L[4] - A / 10) < 1e-15
    Gs = oracle.sensor_response(V, 1, [oracle.sensor_params("gaussian", v0, w, A)])["S"][:, 0]
    assert Gs[0] == A and abs(Gs[1] - A * np.exp(-0.5)) < 1e-15 and abs(Gs[1] - Gs[2]) < 1e-15
    assert abs(Gs[3] - A * np.exp(-4.5)) < 1e-15
    lin = oracle.sensor_response(V, 1, [oracle.sensor_params("linear", v0, w, A)])["S"][:, 0]
    assert np.allclose(lin, A * (V[:, 0] - v0) / w, rtol=0, atol=1e-12)
    # curvature at the peak: Lorentzian -2A/w^2, Gaussian -A/w^2
    h = 1e-4
    assert abs((L[5] + L[6] - 2 * L[0]) / h ** 2 - (-2 * A / w ** 2)) < 1e-2 * A / w ** 2
    assert abs((Gs[5] + Gs[6] - 2 * Gs[0]) / h ** 2 - (-A / w ** 2)) < 1e-2 * A / w ** 2


def test_P14_counter_based_generator():
    """SplitMix64: the first output of the generator seeded with 0 is 0xE220A8397B1DCDAF (published test vector) -- the inner
    stage of r(seed=0, stream=0, .).  The composition, the (0,1) mapping and Box-Muller are re-derived here with Python
    integers / math (exact integer arithmetic modulo 2^64)."""
    import math
    MASK, GOLD = (1 << 64) - 1, 0x9E3779B97F4A7C15

    def mix(z):
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK
        return z ^ (z >> 31)

    assert mix(GOLD) == 0xE220A8397B1DCDAF
    for seed, stream, idx in ((0, 0, 0), (12345, 7, 99), (2 ** 63 + 5, 200, 2 ** 40 + 3)):
        r = mix((mix((seed + GOLD * (stream + 1)) & MASK) + GOLD * (idx + 1)) & MASK)
        assert oracle.rng_u64(seed, stream, idx) == r
        assert oracle.rng_uniform(seed, stream, idx) == ((r >> 11) + 0.5) * 2.0 ** -53
    u1, u2 = oracle.rng_uniform(5, 6, 11), oracle.rng_uniform(5, 7, 11)
    assert abs(oracle.rng_normal(5, 3, 11) - math.sqrt(-2 * math.log(u1)) * math.cos(2 * math.pi * u2)) < 1e-14
    # different (stream, idx) give different numbers; uniforms fill (0,1) evenly
    u = np.array([oracle.rng_uniform(1, 0, i) for i in range(20000)])
    assert 0 < u.min() and u.max() < 1 and abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1 / 12) < 0.005
    assert len({oracle.rng_u64(1, s, i) for s in range(8) for i in range(100)}) == 800


def test_P14_noise_statistics():
    """White: zero mean, variance sigma^2, flat spectrum.  1/f (Voss-McCartney, K octaves): variance sigma_p^2, octave j is
    constant over blocks of 2^j pixels, power spectral density falls with frequency (log-log slope about -1).  Jumps: the
    baseline is piecewise constant, the number of steps is Binomial(P, rate), step sizes have standard deviation sigma_j."""
    P = 1 << 16
    V = np.zeros((P, 1))
    base = dict(profile="linear", v0=0.0, width=1.0, amplitude=0.0)
    w = oracle.sensor_response(V, P, [oracle.sensor_params(white_sigma=0.3, seed=11, **base)], False)["S"][:, 0]
    assert abs(w.mean()) < 4 * 0.3 / np.sqrt(P) and abs(w.var() / 0.09 - 1) < 0.03
    psd = np.abs(np.fft.rfft(w)) ** 2
    lo, hi = psd[1:P // 8].mean(), psd[3 * P // 8:].mean()
    assert abs(lo / hi - 1) < 0.1                                    # flat
    K = 12
    pk = oracle.sensor_response(V, P, [oracle.sensor_params(pink_sigma=0.5, pink_octaves=K, seed=12, **base)], False)["S"][:, 0]
    assert abs(pk.var() / 0.25 - 1) < 0.25 and abs(pk.mean()) < 0.2
    f = np.fft.rfftfreq(P)[1:]
    psd = np.abs(np.fft.rfft(pk))[1:] ** 2
    sel = (f > 2.0 ** -(K - 1)) & (f < 0.25)
    edges = np.logspace(np.log10(f[sel][0]), np.log10(f[sel][-1]), 12)
    fc, pc = [], []
    for a, b in zip(edges[:-1], edges[1:]):
        m = (f >= a) & (f < b)
        fc.append(np.sqrt(a * b))
        pc.append(psd[m].mean())
    slope = np.polyfit(np.log(fc), np.log(pc), 1)[0]
    assert -1.4 < slope < -0.6, slope
    # a single octave j is constant over aligned blocks of 2^j pixels: with K = 1 the noise is white; the difference between
    # K = 4 and K = 3 signals (rescaled) is the j = 3 source alone
    s4 = oracle.sensor_response(V, P, [oracle.sensor_params(pink_sigma=2.0, pink_octaves=4, seed=13, **base)], False)["S"][:, 0] * 2.0 / 2.0
    s3 = oracle.sensor_response(V, P, [oracle.sensor_params(pink_sigma=np.sqrt(3.0), pink_octaves=3, seed=13, **base)], False)["S"][:, 0]
    src3 = (s4 - s3).reshape(-1, 8)                                  # sigma/sqrt(K) = 1 in both
    assert np.abs(src3 - src3[:, :1]).max() < 1e-12 and abs(src3[:, 0].var() - 1) < 0.1
    rate, sj = 0.002, 0.7
    j = oracle.sensor_response(V, P, [oracle.sensor_params(jump_rate=rate, jump_sigma=sj, seed=14, **base)], False)["S"][:, 0]
    steps = np.diff(np.concatenate([[0.0], j]))
    nj = int((steps != 0).sum())
    assert abs(nj - rate * P) < 5 * np.sqrt(rate * P)
    assert abs(steps[steps != 0].std() / sj - 1) < 0.25
    # determinism and independence of the sensors
    V2 = np.zeros((1000, 2))
    q = [oracle.sensor_params(white_sigma=1.0, seed=3, **base)] * 2
    r1, r2 = oracle.sensor_response(V2, 1000, q, False)["S"], oracle.sensor_response(V2, 1000, q, False)["S"]
    assert np.array_equal(r1, r2) and abs(np.corrcoef(r1[:, 0], r1[:, 1])[0, 1]) < 0.15


def test_P14_gradient_is_numpy_gradient_along_the_fast_axis():
    rng = np.random.default_rng(5)
    W, H = 37, 11
    V = rng.uniform(-0.2, 0.2, size=(W * H, 2))
    q = [oracle.sensor_params("lorentzian", 0.05, 0.03, 1.0, white_sigma=0.01, seed=1),
         oracle.sensor_params("gaussian", -0.02, 0.05, 2.0, jump_rate=0.01, jump_sigma=0.1, seed=2)]
    r = oracle.sensor_response(V, W, q)
    for a in range(2):
        assert np.allclose(r["G"][:, a].reshape(H, W), np.gradient(r["S"][:, a].reshape(H, W), axis=1), rtol=0, atol=1e-15)
    assert np.array_equal(oracle.sensor_response(V[:W], 1, q)["G"], np.zeros((W, 2)))
    with pytest.raises(ValueError):
        oracle.sensor_response(V, W + 1, q)
    with pytest.raises(ValueError):
        oracle.sensor_response(V, W, [oracle.sensor_params(width=0.0)] * 2)
