"""ctypes front-end of the C oracle (oracle/qarray_oracle.c).  TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this package.  It imports nothing from the CUDA path."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

ALG = {"default": 0, "thresholded": 1, "brute": 2, "brute_force": 2}
FLAG_QP, FLAG_WIDENED, FLAG_QP_FAIL, FLAG_EMPTY = 1, 2, 4, 8

_HERE = os.path.dirname(os.path.abspath(__file__))
_libs = {}


def _lib(omp: bool = False):
    key = "omp" if omp else "st"
    if key not in _libs:
        _build.build()
        path = os.path.join(_HERE, "libqarray_oracle_omp.so" if omp else "libqarray_oracle.so")
        if not os.path.exists(path):
            raise RuntimeError(f"oracle library {path} not built")
        lib = C.CDLL(path)
        dp, ip, lp, vp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.c_void_p
        lib.qo_model_init.argtypes = [vp, dp, dp, C.c_int, C.c_int]
        lib.qo_nc.argtypes = [vp, dp, dp]
        lib.qo_energy.argtypes = [vp, dp, ip]
        lib.qo_energy.restype = C.c_double
        lib.qo_free_energy_eq4.argtypes = [vp, dp, ip]
        lib.qo_free_energy_eq4.restype = C.c_double
        lib.qo_qp.argtypes = [vp, dp, C.c_int, C.c_double, dp, dp]
        lib.qo_continuous_min.argtypes = [vp, dp, C.c_int, C.c_int, dp]
        lib.qo_ground_state.argtypes = [vp, dp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, ip, dp, dp, dp,
                                        lp, lp, ip, ip, C.c_int]
        lib.qo_thermal.argtypes = [vp, dp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.c_double, dp, dp,
                                   lp, ip]
        lib.qo_sensor.argtypes = [vp, vp, ip, C.c_int, dp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, ip,
                                  dp, dp, dp, dp, ip]
        lib.qo_rng_u64.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
        lib.qo_rng_u64.restype = C.c_uint64
        for f in ("qo_rng_uniform", "qo_rng_normal"):
            getattr(lib, f).argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
            getattr(lib, f).restype = C.c_double
        lib.qo_sensor_response.argtypes = [dp, C.c_int64, C.c_int, C.c_int64, vp, dp, dp]
        _libs[key] = lib
    return _libs[key]


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32)) if a is not None else None


def _lp(a):
    return a.ctypes.data_as(C.POINTER(C.c_int64)) if a is not None else None


class ModelError(ValueError):
    def __init__(self, code):
        self.code = code
        super().__init__({1: "invalid argument", 2: "c_dd not symmetric", 3: "c_dd not positive definite"}.get(code, str(code)))


class Model:
    """Validated model: c_dd (Maxwell, SPD), c_gd, M = c_dd^-1."""

    def __init__(self, C_dd, C_gd):
        C_dd = np.ascontiguousarray(C_dd, dtype=np.float64)
        C_gd = np.ascontiguousarray(C_gd, dtype=np.float64)
        if C_dd.ndim != 2 or C_dd.shape[0] != C_dd.shape[1] or C_gd.ndim != 2 or C_gd.shape[0] != C_dd.shape[0]:
            raise ModelError(1)
        self.n, self.g = C_dd.shape[0], C_gd.shape[1]
        lib = _lib()
        self._buf = C.create_string_buffer(lib.qo_sizeof_model())
        rc = lib.qo_model_init(self._buf, _dp(C_dd), _dp(C_gd), self.n, self.g)
        if rc:
            raise ModelError(rc)
        self.C_dd, self.C_gd = C_dd, C_gd

    # -- views into the C struct (layout: int n, g; double C[256], Cgd[1024], M[256], C1[16], oneC1, EC) --
    def _field(self, off, count):
        return np.frombuffer(self._buf, dtype=np.float64, count=count, offset=8 + 8 * off).copy()

    @property
    def M(self):
        return self._field(256 + 1024, 256)[: self.n * self.n].reshape(self.n, self.n)

    @property
    def C1(self):
        return self._field(256 + 1024 + 256, 16)[: self.n]

    @property
    def oneC1(self):
        return float(self._field(256 + 1024 + 256 + 16, 1)[0])

    @property
    def EC(self):
        return float(self._field(256 + 1024 + 256 + 17, 1)[0])

    def nc(self, vg):
        vg = np.ascontiguousarray(vg, dtype=np.float64)
        out = np.empty(self.n)
        _lib().qo_nc(self._buf, _dp(vg), _dp(out))
        return out

    def energy(self, nc, N):
        nc = np.ascontiguousarray(nc, dtype=np.float64)
        N = np.ascontiguousarray(N, dtype=np.int32)
        return _lib().qo_energy(self._buf, _dp(nc), _ip(N))

    def free_energy_eq4(self, nc, N):
        nc = np.ascontiguousarray(nc, dtype=np.float64)
        N = np.ascontiguousarray(N, dtype=np.int32)
        return _lib().qo_free_energy_eq4(self._buf, _dp(nc), _ip(N))

    def qp(self, c, closed=False, N_hat=0.0):
        """Exact QP of Eq. (8): returns (x, iterations or -1, scaled KKT violation)."""
        c = np.ascontiguousarray(c, dtype=np.float64)
        x = np.empty(self.n)
        kkt = C.c_double()
        it = _lib().qo_qp(self._buf, _dp(c), int(closed), float(N_hat), _dp(x), C.byref(kkt))
        return x, it, kkt.value

    def continuous_min(self, nc, closed=False, N_hat=0):
        nc = np.ascontiguousarray(nc, dtype=np.float64)
        x = np.empty(self.n)
        flags = _lib().qo_continuous_min(self._buf, _dp(nc), int(closed), int(N_hat), _dp(x))
        return x, flags

    def ground_state(self, Vg, regime="open", N_hat=0, algorithm="default", t=1.0, n_max=0, n_threads=1):
        """Whole sweep.  Returns dict(N[P,n] int32, E[P], E2[P], x[P,n], n_scored[P], n_enum[P], flags[P], doublings[P])."""
        Vg = np.ascontiguousarray(Vg, dtype=np.float64).reshape(-1, self.g)
        P = Vg.shape[0]
        out = dict(N=np.empty((P, self.n), np.int32), E=np.empty(P), E2=np.empty(P), x=np.empty((P, self.n)),
                   n_scored=np.empty(P, np.int64), n_enum=np.empty(P, np.int64), flags=np.empty(P, np.int32),
                   doublings=np.empty(P, np.int32))
        lib = _lib(omp=n_threads > 1)
        rc = lib.qo_ground_state(self._buf, _dp(Vg), P, int(regime == "closed"), int(N_hat), ALG[algorithm], float(t),
                                 int(n_max), _ip(out["N"]), _dp(out["E"]), _dp(out["E2"]), _dp(out["x"]),
                                 _lp(out["n_scored"]), _lp(out["n_enum"]), _ip(out["flags"]), _ip(out["doublings"]),
                                 int(n_threads))
        if rc:
            raise ValueError(f"qo_ground_state: invalid argument ({rc})")
        return out


def _thermal(self, Vg, kT, regime="open", N_hat=0, algorithm="default", t=1.0, n_max=0):
    """Eq. (10): Boltzmann-weighted mean occupation over the candidate set.  Returns dict(Nmean[P,n], Emin[P], n_scored, flags)."""
    Vg = np.ascontiguousarray(Vg, dtype=np.float64).reshape(-1, self.g)
    P = Vg.shape[0]
    out = dict(Nmean=np.empty((P, self.n)), Emin=np.empty(P), n_scored=np.empty(P, np.int64), flags=np.empty(P, np.int32))
    rc = _lib().qo_thermal(self._buf, _dp(Vg), P, int(regime == "closed"), int(N_hat), ALG[algorithm], float(t), int(n_max),
                           float(kT), _dp(out["Nmean"]), _dp(out["Emin"]), _lp(out["n_scored"]), _ip(out["flags"]))
    if rc:
        raise ValueError(f"qo_thermal: invalid argument ({rc})")
    return out


Model.thermal = _thermal


def sensor_ground_state(C_dd, C_gd, sensor_dots, Vg, regime="open", N_hat=0, algorithm="default", t=1.0, n_max=0):
    """Reading R8: array sub-problem on the sub-blocks, then the sensor dots.  Returns dict(N[P,n_full], E, E2, Vs[P,ns],
    sgap[P,ns] = margin |e(c0+1) - e(c0)| of every sensor's two-way choice, flags)."""
    C_dd = np.ascontiguousarray(C_dd, dtype=np.float64)
    C_gd = np.ascontiguousarray(C_gd, dtype=np.float64)
    n = C_dd.shape[0]
    sens = np.ascontiguousarray(sensor_dots, dtype=np.int32)
    D = [i for i in range(n) if i not in set(sens.tolist())]
    full = Model(C_dd, C_gd)
    sub = Model(C_dd[np.ix_(D, D)], C_gd[D, :])
    Vg = np.ascontiguousarray(Vg, dtype=np.float64).reshape(-1, full.g)
    P = Vg.shape[0]
    out = dict(N=np.empty((P, n), np.int32), E=np.empty(P), E2=np.empty(P), Vs=np.empty((P, len(sens))),
               sgap=np.empty((P, len(sens))), flags=np.empty(P, np.int32))
    rc = _lib().qo_sensor(full._buf, sub._buf, _ip(sens), len(sens), _dp(Vg), P, int(regime == "closed"), int(N_hat),
                          ALG[algorithm], float(t), int(n_max), _ip(out["N"]), _dp(out["E"]), _dp(out["E2"]),
                          _dp(out["Vs"]), _dp(out["sgap"]), _ip(out["flags"]))
    if rc:
        raise ValueError(f"qo_sensor: invalid argument ({rc})")
    return out


class SensorParams(C.Structure):
    """Parameters of one sensor's response (reading R14; mirrors qo_sensor_params)."""
    _fields_ = [("profile", C.c_int32), ("pink_octaves", C.c_int32), ("v0", C.c_double), ("width", C.c_double),
                ("amplitude", C.c_double), ("white_sigma", C.c_double), ("pink_sigma", C.c_double),
                ("jump_rate", C.c_double), ("jump_sigma", C.c_double), ("seed", C.c_uint64)]


PROFILE = {"lorentzian": 0, "gaussian": 1, "linear": 2}


def sensor_params(profile="lorentzian", v0=0.0, width=1.0, amplitude=1.0, white_sigma=0.0, pink_sigma=0.0, pink_octaves=0,
                  jump_rate=0.0, jump_sigma=0.0, seed=0):
    return SensorParams(PROFILE[profile] if isinstance(profile, str) else int(profile), int(pink_octaves), float(v0),
                        float(width), float(amplitude), float(white_sigma), float(pink_sigma), float(jump_rate),
                        float(jump_sigma), int(seed))


def sensor_response(Vs, W, params, want_gradient=True):
    """Reading R14 (L149, L464): response profile + white / 1/f / jump noise of every sensor column of Vs[P, ns], and its
    gradient along the fast axis (row length W).  params: one SensorParams per sensor.  Returns dict(S[, G])."""
    Vs = np.ascontiguousarray(Vs, dtype=np.float64)
    Vs = Vs.reshape(Vs.shape[0], -1)
    P, ns = Vs.shape
    arr = (SensorParams * ns)(*params)
    S = np.empty((P, ns))
    G = np.empty((P, ns)) if want_gradient else None
    rc = _lib().qo_sensor_response(_dp(Vs), P, ns, int(W), C.byref(arr), _dp(S), _dp(G))
    if rc:
        raise ValueError(f"qo_sensor_response: invalid argument ({rc})")
    return dict(S=S, G=G) if want_gradient else dict(S=S)


def rng_u64(seed, stream, idx):
    return int(_lib().qo_rng_u64(seed, stream, idx))


def rng_uniform(seed, stream, idx):
    return float(_lib().qo_rng_uniform(seed, stream, idx))


def rng_normal(seed, stream, idx):
    return float(_lib().qo_rng_normal(seed, stream, idx))


def has_openmp() -> bool:
    try:
        return bool(_lib(omp=True).qo_has_openmp())
    except Exception:
        return False
