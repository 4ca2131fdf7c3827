"""Seeded synthetic workloads (the five BASELINE.json configs) shared by the oracle tests and the CUDA path.

This module only *builds inputs*: capacitance matrices in Maxwell format (Eq. (2), L593 Eq. (B1)) and
dense gate-voltage arrays ``Vg[P, n_gate]``.  It holds none of the method's arithmetic (no N_c, no energy,
no candidate logic) and imports neither ``oracle/`` nor the CUDA binding.  The recipes are the ones fixed in
SURVEY.md section 8(d) / DESIGN.md "Input recipe"; choices BASELINE.json leaves open are marked (+) there.

Pixel index p = iy * W + ix (ix the fast axis).  All arrays are float64, C-contiguous.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Workload:
    name: str
    C_dd: np.ndarray            # [n, n] Maxwell dot-dot matrix (SPD, offdiag <= 0)
    C_gd: np.ndarray            # [n, g] positive gate->dot couplings
    Vg: np.ndarray              # [P, g] gate voltages, pixel p = iy*W + ix
    W: int
    H: int
    regime: str = "open"        # "open" | "closed"
    N_hat: int = 0              # closed arrays only
    sensor_dots: tuple = ()     # indices of charge-sensor dots (config 3)
    meta: dict = field(default_factory=dict)

    @property
    def n_dot(self) -> int:
        return self.C_dd.shape[0]

    @property
    def n_gate(self) -> int:
        return self.C_gd.shape[1]

    @property
    def P(self) -> int:
        return self.Vg.shape[0]


def maxwell(C_m: np.ndarray, C_gd: np.ndarray, self_cap: float = 1.0) -> np.ndarray:
    """C_dd = diag(self + sum_k C_gd[i,k] + sum_j C_m[i,j]) - C_m  (Eq. (B1); BASELINE.json config 1)."""
    C_m = np.asarray(C_m, dtype=np.float64)
    C_gd = np.asarray(C_gd, dtype=np.float64)
    diag = self_cap + C_gd.sum(axis=1) + C_m.sum(axis=1)
    return np.ascontiguousarray(np.diag(diag) - C_m)


def _grid2(W: int, H: int):
    """ix, iy index arrays for p = iy*W + ix."""
    p = np.arange(W * H)
    return p % W, p // W


def _unit(i: np.ndarray, count: int) -> np.ndarray:
    return i / (count - 1) if count > 1 else np.zeros_like(i, dtype=np.float64)


def config1(W: int = 100, H: int = 100, seed: int = 0) -> Workload:
    """Open double dot (BASELINE.json configs[0])."""
    rng = np.random.default_rng(seed)
    C_m = np.zeros((2, 2))
    C_m[0, 1] = C_m[1, 0] = 0.1
    C_gd = np.zeros((2, 2))
    C_gd[0, 0], C_gd[1, 1] = rng.uniform(0.8, 1.2, size=2)
    C_gd[0, 1], C_gd[1, 0] = rng.uniform(0.05, 0.2, size=2)
    C_dd = maxwell(C_m, C_gd)
    ix, iy = _grid2(W, H)
    Vg = np.empty((W * H, 2))
    Vg[:, 0] = _unit(ix, W) * 5.0 / C_gd[0, 0]
    Vg[:, 1] = _unit(iy, H) * 5.0 / C_gd[1, 1]
    return Workload("config1_open_double_dot", C_dd, C_gd, np.ascontiguousarray(Vg), W, H)


def config2(W: int = 100, H: int = 100, seed: int = 1) -> Workload:
    """Closed linear 5-dot chain, N_hat = 5 (BASELINE.json configs[1])."""
    n = 5
    rng = np.random.default_rng(seed)
    C_m = np.zeros((n, n))
    nn = rng.uniform(0.1, 0.3, size=n - 1)
    nnn = 0.3 * rng.uniform(0.1, 0.3, size=n - 2)
    for i in range(n - 1):
        C_m[i, i + 1] = C_m[i + 1, i] = nn[i]
    for i in range(n - 2):
        C_m[i, i + 2] = C_m[i + 2, i] = nnn[i]
    lever = rng.uniform(0.8, 1.2, size=n)
    C_gd = np.array([[lever[i] * 0.3 ** abs(i - k) for k in range(n)] for i in range(n)])
    C_dd = maxwell(C_m, C_gd)
    fixed = rng.uniform(0.0, 2.0, size=3)
    ix, iy = _grid2(W, H)
    Vg = np.empty((W * H, n))
    for j, k in enumerate((1, 2, 3)):
        Vg[:, k] = fixed[j] / C_gd[k, k]
    Vg[:, 0] = (-1.0 + 5.0 * _unit(ix, W)) / C_gd[0, 0]
    Vg[:, 4] = (-1.0 + 5.0 * _unit(iy, H)) / C_gd[4, 4]
    return Workload("config2_closed_chain5", C_dd, C_gd, np.ascontiguousarray(Vg), W, H, regime="closed", N_hat=5)


def config3(W: int = 200, H: int = 200, seed: int = 2) -> Workload:
    """Open 2x2 quadruple dot + one charge-sensor dot (5 dots, 6 gates) (BASELINE.json configs[2])."""
    n, g = 5, 6
    rng = np.random.default_rng(seed)
    C_m = np.zeros((n, n))
    ring = [(0, 1), (1, 3), (3, 2), (2, 0)]
    e = rng.uniform(0.1, 0.3, size=4)
    for (a, b), v in zip(ring, e):
        C_m[a, b] = C_m[b, a] = v
    dg = 0.3 * rng.uniform(0.1, 0.3, size=2)
    for (a, b), v in zip([(0, 3), (1, 2)], dg):
        C_m[a, b] = C_m[b, a] = v
    for a in range(4):
        C_m[a, 4] = C_m[4, a] = 0.05
    lever = rng.uniform(0.8, 1.2, size=4)
    ring_nb = {0: (1, 2), 1: (0, 3), 2: (0, 3), 3: (1, 2)}
    diag_nb = {0: 3, 1: 2, 2: 1, 3: 0}
    C_gd = np.zeros((n, g))
    for k in range(4):                       # plunger k sits on dot k
        C_gd[k, k] = lever[k]
        for a in ring_nb[k]:
            C_gd[a, k] = 0.3 * lever[k]
        C_gd[diag_nb[k], k] = 0.09 * lever[k]
        C_gd[4, k] = 0.05                    # (+) plunger -> sensor-dot cross-talk
    C_gd[4, 4] = rng.uniform(0.8, 1.2)
    C_gd[0:4, 4] = 0.05
    C_gd[:, 5] = rng.uniform(0.05, 0.15, size=n)
    C_dd = maxwell(C_m, C_gd)
    others = rng.uniform(0.0, 2.0, size=2)
    vs = rng.uniform(0.0, 1.0)
    ix, iy = _grid2(W, H)
    Vg = np.zeros((W * H, g))
    Vg[:, 0] = 4.0 * _unit(ix, W) / C_gd[0, 0]
    Vg[:, 3] = 4.0 * _unit(iy, H) / C_gd[3, 3]
    Vg[:, 1] = others[0] / C_gd[1, 1]
    Vg[:, 2] = others[1] / C_gd[2, 2]
    Vg[:, 4] = vs / C_gd[4, 4]
    return Workload("config3_open_quad_sensor", C_dd, C_gd, np.ascontiguousarray(Vg), W, H, sensor_dots=(4,))


def _grid_array(rows: int, cols: int, rng: np.random.Generator):
    """Random rows x cols dot grid: NN couplings U[0.1,0.3], diagonal neighbours x0.3, levers U[0.8,1.2], cross-lever
    U[0,0.15] onto nearest neighbours (BASELINE.json configs[3], configs[4])."""
    n = rows * cols
    idx = lambda r, c: r * cols + c
    C_m = np.zeros((n, n))
    for r in range(rows):                    # NN edges, row-major, right then down
        for c in range(cols):
            if c + 1 < cols:
                C_m[idx(r, c), idx(r, c + 1)] = C_m[idx(r, c + 1), idx(r, c)] = rng.uniform(0.1, 0.3)
            if r + 1 < rows:
                C_m[idx(r, c), idx(r + 1, c)] = C_m[idx(r + 1, c), idx(r, c)] = rng.uniform(0.1, 0.3)
    for r in range(rows - 1):                # diagonal neighbours, down-right then down-left
        for c in range(cols):
            if c + 1 < cols:
                C_m[idx(r, c), idx(r + 1, c + 1)] = C_m[idx(r + 1, c + 1), idx(r, c)] = 0.3 * rng.uniform(0.1, 0.3)
            if c - 1 >= 0:
                C_m[idx(r, c), idx(r + 1, c - 1)] = C_m[idx(r + 1, c - 1), idx(r, c)] = 0.3 * rng.uniform(0.1, 0.3)
    C_gd = np.zeros((n, n))
    for i in range(n):
        C_gd[i, i] = rng.uniform(0.8, 1.2)
    for i in range(n):
        ri, ci = divmod(i, cols)
        for k in range(n):
            rk, ck = divmod(k, cols)
            if abs(ri - rk) + abs(ci - ck) == 1:
                C_gd[i, k] = rng.uniform(0.0, 0.15)
    return C_m, C_gd


def _plane_sweep(C_gd: np.ndarray, rng: np.random.Generator, W: int, H: int) -> np.ndarray:
    """V = V0 + alpha*u1 + beta*u2: two seeded random directions around a seeded operating point (configs 4, 5)."""
    n = C_gd.shape[0]
    n0 = rng.uniform(0.75, 2.25, size=n)
    w = rng.standard_normal(size=(2, n))
    w /= np.abs(w).max(axis=1, keepdims=True)
    V0 = np.linalg.solve(C_gd, n0)
    u = np.linalg.solve(C_gd, w.T).T
    ix, iy = _grid2(W, H)
    alpha = -1.5 + 3.0 * _unit(ix, W)
    beta = -1.5 + 3.0 * _unit(iy, H)
    return np.ascontiguousarray(V0[None, :] + alpha[:, None] * u[0][None, :] + beta[:, None] * u[1][None, :])


def config4(W: int = 100, H: int = 100, seed: int = 3) -> Workload:
    """Open 4x4 grid of 16 dots, the headline workload (BASELINE.json configs[3])."""
    rng = np.random.default_rng(seed)
    C_m, C_gd = _grid_array(4, 4, rng)
    C_dd = maxwell(C_m, C_gd)
    Vg = _plane_sweep(C_gd, rng, W, H)
    return Workload("config4_open_grid16", C_dd, C_gd, Vg, W, H)


def config5_array(j: int, W: int = 128, H: int = 128) -> Workload:
    """Array j of the dataset batch: open 8-dot 2x4 grid, seed 1000 + j (BASELINE.json configs[4])."""
    rng = np.random.default_rng(1000 + j)
    C_m, C_gd = _grid_array(2, 4, rng)
    C_dd = maxwell(C_m, C_gd)
    Vg = _plane_sweep(C_gd, rng, W, H)
    return Workload(f"config5_open_grid8_{j:03d}", C_dd, C_gd, Vg, W, H)


def config5(B: int = 256, W: int = 128, H: int = 128):
    return [config5_array(j, W, H) for j in range(B)]


def random_open(n: int, g: int, P: int, seed: int, lo: float = -0.6, hi: float = 3.2) -> Workload:
    """Generic test array: random dense Maxwell matrix (elements drawn uniformly, converted to Maxwell
    format) and P random gate vectors chosen so that C_gd.Vg spans [lo, hi] per dot (negative part exercises the QP)."""
    rng = np.random.default_rng(seed)
    C_m = np.triu(rng.uniform(0.0, 0.25, size=(n, n)), 1)
    C_m = C_m + C_m.T
    C_gd = rng.uniform(0.0, 0.15, size=(n, g))
    for i in range(min(n, g)):
        C_gd[i, i] = rng.uniform(0.8, 1.2)
    C_dd = maxwell(C_m, C_gd)
    target = rng.uniform(lo, hi, size=(P, n))
    Vg = target @ np.linalg.pinv(C_gd).T
    return Workload(f"random_open_n{n}_g{g}_s{seed}", C_dd, C_gd, np.ascontiguousarray(Vg), P, 1)


def random_general(n: int, g: int, P: int, seed: int, lo: float = -0.8, hi: float = 3.2) -> Workload:
    """Test array whose c_dd is symmetric positive definite but NOT a Maxwell matrix: mutual terms of both signs, so some
    off-diagonals of c_dd are positive (legal input, PAPER.md L204 asks only for SPD); diagonally dominant by
    construction.  Exercises the general active-set phase of the continuous QP."""
    rng = np.random.default_rng(seed)
    C_m = np.triu(rng.uniform(-0.15, 0.25, size=(n, n)), 1)
    C_m[0, 1] = -0.12                        # at least one positive off-diagonal in c_dd
    C_m = C_m + C_m.T
    C_gd = rng.uniform(0.0, 0.15, size=(n, g))
    for i in range(min(n, g)):
        C_gd[i, i] = rng.uniform(0.8, 1.2)
    C_dd = np.diag(1.0 + C_gd.sum(1) + np.abs(C_m).sum(1)) - C_m
    target = rng.uniform(lo, hi, size=(P, n))
    Vg = target @ np.linalg.pinv(C_gd).T
    return Workload(f"random_general_n{n}_g{g}_s{seed}", C_dd, C_gd, np.ascontiguousarray(Vg), P, 1)


def shard_range(P: int, rank: int, world: int):
    """Contiguous pixel range [p0, p1) of rank `rank` of `world` (pixels are independent: SURVEY.md section 8(e))."""
    base, rem = divmod(P, world)
    p0 = rank * base + min(rank, rem)
    return p0, p0 + base + (1 if rank < rem else 0)
