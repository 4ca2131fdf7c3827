"""Thin Python binding over the C ABI of libqarray_b200.so (include/qarray_b200.h): same names, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device memory, streams and nothing
else.  There is no CPU fallback: importing this module fails if the library is not built, and every ground-state call
fails if there is no CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqarray_b200.so")

QA_OK = 0
QA_ALG_DEFAULT, QA_ALG_THRESHOLDED, QA_ALG_BRUTE_FORCE = 0, 1, 2
ALG = {"default": 0, "thresholded": 1, "brute": 2, "brute_force": 2}
STATUS_NAMES = ["QA_OK", "QA_ERR_INVALID_ARG", "QA_ERR_NOT_SYMMETRIC", "QA_ERR_NOT_POSDEF", "QA_ERR_UNSUPPORTED_SIZE",
                "QA_ERR_INFEASIBLE", "QA_ERR_OVERFLOW", "QA_ERR_CUDA", "QA_ERR_UNSUPPORTED", "QA_ERR_STATIC_WORKSPACE"]
EXPORTS = ["qa_model_create", "qa_model_set_sensor_dots", "qa_model_destroy", "qa_model_n_dot", "qa_model_n_gate",
           "qa_model_n_sensor", "qa_model_n_search", "qa_model_get_inverse", "qa_workspace_bytes", "qa_ground_state_open",
           "qa_ground_state_closed", "qa_ground_state_host", "qa_measure_fp64_rate", "qa_set_kernel_timing",
           "qa_get_kernel_timings", "qa_model_set_walk_variant", "qa_batch_create", "qa_batch_destroy", "qa_batch_size",
           "qa_ground_state_batch", "qa_thermal_open", "qa_thermal_closed", "qa_sensor_response",
           "qa_sensor_response_workspace_bytes", "qa_last_launch_plan",
           "qa_last_launch_count", "qa_status_string", "qa_last_cuda_error", "qa_version", "qa_static_workspace_bytes",
           "qa_static_workspace_init", "qa_static_workspace_last_error", "qa_ground_state_open_static",
           "qa_ground_state_batch_multi"]


class qa_stats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("n_pixels", "n_qp_pixels", "n_qp_rounds", "n_candidates_enumerated",
                                         "n_candidates_scored", "n_threshold_doublings", "n_widened_pixels",
                                         "n_qp_failed")]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


class qa_sensor_params(C.Structure):
    """include/qarray_b200.h qa_sensor_params (reading R14)."""
    _fields_ = [("profile", C.c_int32), ("pink_octaves", C.c_int32), ("v0", C.c_double), ("width", C.c_double),
                ("amplitude", C.c_double), ("white_sigma", C.c_double), ("pink_sigma", C.c_double),
                ("jump_rate", C.c_double), ("jump_sigma", C.c_double), ("seed", C.c_uint64)]


PROFILE = {"lorentzian": 0, "gaussian": 1, "linear": 2}


def sensor_params(profile="lorentzian", v0=0.0, width=1.0, amplitude=1.0, white_sigma=0.0, pink_sigma=0.0, pink_octaves=0,
                  jump_rate=0.0, jump_sigma=0.0, seed=0) -> qa_sensor_params:
    return qa_sensor_params(PROFILE[profile] if isinstance(profile, str) else int(profile), int(pink_octaves), float(v0),
                            float(width), float(amplitude), float(white_sigma), float(pink_sigma), float(jump_rate),
                            float(jump_sigma), int(seed))


class QaError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        msg = lib().qa_status_string(status).decode()
        extra = lib().qa_last_cuda_error().decode() if status == 7 else ""
        if status == 9 or "static" in where:
            extra = (extra + " " + lib().qa_static_workspace_last_error().decode()).strip()
        super().__init__(f"{where}: {name} ({msg}) {extra}".strip())


_lib = None


def lib() -> C.CDLL:
    """The loaded library; raises if it has not been built (python -m paper_2404_04994_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2404_04994_b200.build` "
                              "(there is no CPU fallback)")
        l = C.CDLL(LIB_PATH)
        vp, dp, ip = C.c_void_p, C.c_void_p, C.c_void_p
        l.qa_model_create.argtypes = [vp, vp, C.c_int, C.c_int, C.POINTER(vp)]
        l.qa_model_set_sensor_dots.argtypes = [vp, vp, C.c_int]
        l.qa_model_destroy.argtypes = [vp]
        for f in ("qa_model_n_dot", "qa_model_n_gate", "qa_model_n_sensor", "qa_model_n_search"):
            getattr(l, f).argtypes = [vp]
        l.qa_model_get_inverse.argtypes = [vp, vp, C.POINTER(C.c_double)]
        l.qa_workspace_bytes.argtypes = [vp, C.c_int64]
        l.qa_workspace_bytes.restype = C.c_size_t
        l.qa_ground_state_open.argtypes = [vp, dp, C.c_int64, C.c_int, C.c_double, C.c_int, ip, dp, dp, dp, vp, vp,
                                           C.c_size_t, vp]
        l.qa_ground_state_open_static.argtypes = [vp, dp, C.c_int64, C.c_int, C.c_double, C.c_int, ip, dp, dp, dp, vp, vp]
        l.qa_static_workspace_bytes.restype = C.c_size_t
        l.qa_static_workspace_last_error.restype = C.c_char_p
        l.qa_ground_state_closed.argtypes = [vp, dp, C.c_int64, C.c_int, C.c_int, C.c_double, C.c_int, ip, dp, dp, dp, vp,
                                             vp, C.c_size_t, vp]
        l.qa_ground_state_host.argtypes = [vp, vp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, vp, vp, vp,
                                           vp, vp]
        l.qa_batch_create.argtypes = [vp, C.c_int, C.POINTER(vp)]
        l.qa_batch_destroy.argtypes = [vp]
        l.qa_batch_size.argtypes = [vp]
        l.qa_ground_state_batch.argtypes = [vp, dp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, ip, dp, dp, vp, vp]
        l.qa_ground_state_batch_multi.argtypes = [vp, dp, C.c_int64, C.c_int, vp, vp, vp, vp, dp, vp, vp]
        l.qa_thermal_open.argtypes = [vp, dp, C.c_int64, C.c_int, C.c_double, C.c_int, C.c_double, dp, dp, vp, vp, C.c_size_t, vp]
        l.qa_thermal_closed.argtypes = [vp, dp, C.c_int64, C.c_int, C.c_int, C.c_double, C.c_int, C.c_double, dp, dp, vp, vp,
                                        C.c_size_t, vp]
        l.qa_sensor_response_workspace_bytes.argtypes = [C.c_int64, C.c_int]
        l.qa_sensor_response_workspace_bytes.restype = C.c_size_t
        l.qa_sensor_response.argtypes = [dp, C.c_int64, C.c_int, C.c_int64, vp, dp, dp, vp, C.c_size_t, vp]
        l.qa_measure_fp64_rate.argtypes = [C.c_double, C.POINTER(C.c_double), vp]
        l.qa_set_kernel_timing.argtypes = [C.c_int]
        l.qa_model_set_walk_variant.argtypes = [vp, C.c_int]
        l.qa_get_kernel_timings.argtypes = [C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_int)]
        l.qa_last_launch_plan.restype = C.c_char_p
        l.qa_status_string.restype = C.c_char_p
        l.qa_status_string.argtypes = [C.c_int]
        l.qa_last_cuda_error.restype = C.c_char_p
        l.qa_version.restype = C.c_char_p
        _lib = l
    return _lib


def _check(status: int, where: str):
    if status != QA_OK:
        raise QaError(status, where)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class Model:
    """qa_model_create(C_dd, C_gd).  Owns the opaque handle."""

    def __init__(self, C_dd, C_gd, sensor_dots=(), walk_variant=None):
        C_dd = np.ascontiguousarray(C_dd, dtype=np.float64)
        C_gd = np.ascontiguousarray(C_gd, dtype=np.float64)
        if C_dd.ndim != 2 or C_dd.shape[0] != C_dd.shape[1] or C_gd.ndim != 2 or C_gd.shape[0] != C_dd.shape[0]:
            raise QaError(1, "qa_model_create")
        self._h = C.c_void_p()
        _check(lib().qa_model_create(C_dd.ctypes.data, C_gd.ctypes.data, C_dd.shape[0], C_gd.shape[1],
                                     C.byref(self._h)), "qa_model_create")
        self.device = torch.device("cuda", torch.cuda.current_device()) if torch.cuda.is_available() else None
        if len(sensor_dots):
            self.set_sensor_dots(sensor_dots)
        if walk_variant is not None:
            self.set_walk_variant(walk_variant)
        self._ws = None
        self._stats = None

    def set_walk_variant(self, variant: int):
        """qa_model_set_walk_variant (cross-check aid, qarray_b200_aids.h): 0 = three-kernel path with the exact-compare walk /
        generic enumeration everywhere, 1 = production dispatch, 2 = as 1 with exact pruning in the 13..16-dot min-plus walk,
        3 = as 1 with the mixed-precision pass 1 (fp32 bound, fp64 re-score; bit-identical results), 4 = as 1 with the open
        default search of 16 dots in one persistent kernel (no workspace traffic; bit-identical results)."""
        _check(lib().qa_model_set_walk_variant(self._h, int(variant)), "qa_model_set_walk_variant")

    def _check_device(self, Vg):
        if Vg.device != self.device:
            raise ValueError(f"Vg is on {Vg.device}, the model lives on {self.device}")

    def set_sensor_dots(self, dots):
        idx = np.ascontiguousarray(dots, dtype=np.int32)
        _check(lib().qa_model_set_sensor_dots(self._h, idx.ctypes.data, len(idx)), "qa_model_set_sensor_dots")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().qa_model_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    n_dot = property(lambda self: lib().qa_model_n_dot(self._h))
    n_gate = property(lambda self: lib().qa_model_n_gate(self._h))
    n_sensor = property(lambda self: lib().qa_model_n_sensor(self._h))
    n_search = property(lambda self: lib().qa_model_n_search(self._h))

    def inverse(self):
        M = np.empty((self.n_dot, self.n_dot))
        ec = C.c_double()
        _check(lib().qa_model_get_inverse(self._h, M.ctypes.data, C.byref(ec)), "qa_model_get_inverse")
        return M, ec.value

    def workspace_bytes(self, P: int) -> int:
        return int(lib().qa_workspace_bytes(self._h, int(P)))

    def _workspace(self, P, device):
        need = self.workspace_bytes(P)
        if self._ws is None or self._ws.numel() < need or self._ws.device != device:
            self._ws = torch.empty(need, dtype=torch.uint8, device=device)
        return self._ws

    # -- device-resident call: the C-ABI entry points proper -----------------------------------------------------
    def ground_state(self, Vg: torch.Tensor, regime="open", N_hat=0, algorithm="default", t=1.0, n_max=0,
                     want_xcont=False, want_stats=False, out=None, stream=None):
        """qa_ground_state_open / qa_ground_state_closed on a CUDA tensor Vg[P, n_gate] (float64).  Asynchronous on the
        current torch stream.  Returns dict(N, E[, xcont][, Vsensor][, stats (a device tensor of 8 int64)])."""
        if not (isinstance(Vg, torch.Tensor) and Vg.is_cuda and Vg.dtype == torch.float64):
            raise TypeError("Vg must be a CUDA float64 tensor (there is no CPU path)")
        self._check_device(Vg)
        Vg = Vg.contiguous().view(-1, self.n_gate)
        P, dev = Vg.shape[0], Vg.device
        out = out or {}
        N = out.get("N")
        if N is None:
            N = torch.empty((P, self.n_dot), dtype=torch.int32, device=dev)
        E = out.get("E")
        if E is None:
            E = torch.empty(P, dtype=torch.float64, device=dev)
        xc = (out.get("xcont") if out.get("xcont") is not None
              else torch.empty((P, self.n_search), dtype=torch.float64, device=dev)) if want_xcont else None
        Vs = (out.get("Vsensor") if out.get("Vsensor") is not None
              else torch.empty((P, self.n_sensor), dtype=torch.float64, device=dev)) if self.n_sensor else None
        st = torch.zeros(8, dtype=torch.int64, device=dev) if want_stats else None
        ws = self._workspace(P, dev)
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        sp = C.c_void_p(s.cuda_stream)
        alg = ALG[algorithm] if isinstance(algorithm, str) else int(algorithm)
        if torch.cuda.current_device() != dev.index:      # the C call checks the current device against the model's
            with torch.cuda.device(dev):
                rc = self._call_ground_state(regime, Vg, P, N_hat, alg, t, n_max, N, E, xc, Vs, st, ws, sp)
        else:
            rc = self._call_ground_state(regime, Vg, P, N_hat, alg, t, n_max, N, E, xc, Vs, st, ws, sp)
        _check(rc, f"qa_ground_state_{regime}")
        res = {"N": N, "E": E}
        if xc is not None:
            res["xcont"] = xc
        if Vs is not None:
            res["Vsensor"] = Vs
        if st is not None:
            res["stats"] = st
        return res

    def ground_state_static(self, Vg: torch.Tensor, algorithm="default", t=1.0, n_max=0, out=None, stream=None):
        """qa_ground_state_open_static: the open-array search with the library's own static 16 MiB device workspace -- the C
        call allocates nothing (for callers that cannot call cudaMalloc; limit: qa_workspace_bytes(P) <= 16 MiB, calls that
        overlap on the GPU race on the array).  With `out` = dict(N, E) given, this binding allocates nothing either;
        otherwise N and E are torch tensors it creates.  Returns dict(N, E)."""
        if not (isinstance(Vg, torch.Tensor) and Vg.is_cuda and Vg.dtype == torch.float64):
            raise TypeError("Vg must be a CUDA float64 tensor (there is no CPU path)")
        self._check_device(Vg)
        Vg = Vg.contiguous().view(-1, self.n_gate)
        P, dev = Vg.shape[0], Vg.device
        out = out or {}
        N = out.get("N") if out.get("N") is not None else torch.empty((P, self.n_dot), dtype=torch.int32, device=dev)
        E = out.get("E") if out.get("E") is not None else torch.empty(P, dtype=torch.float64, device=dev)
        Vs = torch.empty((P, self.n_sensor), dtype=torch.float64, device=dev) if self.n_sensor else None
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        alg = ALG[algorithm] if isinstance(algorithm, str) else int(algorithm)
        with torch.cuda.device(dev):
            rc = lib().qa_ground_state_open_static(self._h, _ptr(Vg), P, alg, float(t), int(n_max), _ptr(N), _ptr(E), None,
                                                   _ptr(Vs), None, C.c_void_p(s.cuda_stream))
        _check(rc, "qa_ground_state_open_static")
        res = {"N": N, "E": E}
        if Vs is not None:
            res["Vsensor"] = Vs
        return res

    def _call_ground_state(self, regime, Vg, P, N_hat, alg, t, n_max, N, E, xc, Vs, st, ws, sp):
        if regime == "open":
            rc = lib().qa_ground_state_open(self._h, _ptr(Vg), P, alg, float(t), int(n_max), _ptr(N), _ptr(E), _ptr(xc),
                                            _ptr(Vs), _ptr(st), _ptr(ws), ws.numel(), sp)
        elif regime == "closed":
            rc = lib().qa_ground_state_closed(self._h, _ptr(Vg), P, int(N_hat), alg, float(t), int(n_max), _ptr(N),
                                              _ptr(E), _ptr(xc), _ptr(Vs), _ptr(st), _ptr(ws), ws.numel(), sp)
        else:
            raise ValueError("regime must be 'open' or 'closed'")
        return rc

    def thermal(self, Vg: torch.Tensor, kT: float, regime="open", N_hat=0, algorithm="default", t=1.0, n_max=0,
                want_stats=False, stream=None):
        """qa_thermal_open / qa_thermal_closed: Eq. (10) mean occupation on a CUDA tensor Vg[P, n_gate].  Returns
        dict(Nmean[P, n_search] float64, Emin[P][, stats])."""
        if not (isinstance(Vg, torch.Tensor) and Vg.is_cuda and Vg.dtype == torch.float64):
            raise TypeError("Vg must be a CUDA float64 tensor (there is no CPU path)")
        self._check_device(Vg)
        Vg = Vg.contiguous().view(-1, self.n_gate)
        P, dev = Vg.shape[0], Vg.device
        Nm = torch.empty((P, self.n_search), dtype=torch.float64, device=dev)
        Em = torch.empty(P, dtype=torch.float64, device=dev)
        st = torch.zeros(8, dtype=torch.int64, device=dev) if want_stats else None
        ws = self._workspace(P, dev)
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        sp = C.c_void_p(s.cuda_stream)
        alg = ALG[algorithm] if isinstance(algorithm, str) else int(algorithm)
        if regime == "open":
            rc = lib().qa_thermal_open(self._h, _ptr(Vg), P, alg, float(t), int(n_max), float(kT), _ptr(Nm), _ptr(Em),
                                       _ptr(st), _ptr(ws), ws.numel(), sp)
        elif regime == "closed":
            rc = lib().qa_thermal_closed(self._h, _ptr(Vg), P, int(N_hat), alg, float(t), int(n_max), float(kT), _ptr(Nm),
                                         _ptr(Em), _ptr(st), _ptr(ws), ws.numel(), sp)
        else:
            raise ValueError("regime must be 'open' or 'closed'")
        _check(rc, f"qa_thermal_{regime}")
        res = {"Nmean": Nm, "Emin": Em}
        if st is not None:
            res["stats"] = st
        return res

    # -- host-buffer call (end-to-end path) -------------------------------------------------------------------------
    def ground_state_host(self, Vg, regime="open", N_hat=0, algorithm="default", t=1.0, n_max=0, want_xcont=False,
                          want_stats=False, out=None):
        """qa_ground_state_host on HOST buffers (numpy arrays or CPU torch tensors, ideally pinned): H2D copy, search,
        D2H copy and synchronisation all happen inside the C call."""
        tv = Vg if isinstance(Vg, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(Vg, dtype=np.float64))
        tv = tv.contiguous().view(-1, self.n_gate)
        assert tv.dtype == torch.float64 and not tv.is_cuda
        P = tv.shape[0]
        out = out or {}
        N = out.get("N") if out.get("N") is not None else torch.empty((P, self.n_dot), dtype=torch.int32)
        E = out.get("E") if out.get("E") is not None else torch.empty(P, dtype=torch.float64)
        xc = torch.empty((P, self.n_search), dtype=torch.float64) if want_xcont else None
        Vs = torch.empty((P, self.n_sensor), dtype=torch.float64) if self.n_sensor else None
        st = qa_stats() if want_stats else None
        alg = ALG[algorithm] if isinstance(algorithm, str) else int(algorithm)
        rc = lib().qa_ground_state_host(self._h, _ptr(tv), P, int(regime == "closed"), int(N_hat), alg, float(t),
                                        int(n_max), _ptr(N), _ptr(E), _ptr(xc), _ptr(Vs),
                                        C.byref(st) if st is not None else None)
        _check(rc, "qa_ground_state_host")
        res = {"N": N, "E": E}
        if xc is not None:
            res["xcont"] = xc
        if Vs is not None:
            res["Vsensor"] = Vs
        if st is not None:
            res["stats"] = st.as_dict()
        return res


class Batch:
    """qa_batch_create over a list of Model objects with the same n_dot (<= 8) and n_gate: one launch for the whole list."""

    def __init__(self, models):
        self.models = list(models)          # keep them alive
        arr = (C.c_void_p * len(self.models))(*[m._h.value for m in self.models])
        self._h = C.c_void_p()
        _check(lib().qa_batch_create(arr, len(self.models), C.byref(self._h)), "qa_batch_create")
        self.n_dot, self.n_gate = self.models[0].n_dot, self.models[0].n_gate
        self.device = self.models[0].device

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().qa_batch_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __len__(self):
        return int(lib().qa_batch_size(self._h))

    def ground_state(self, Vg: torch.Tensor, regime="open", N_hat=0, algorithm="default", t=1.0, n_max=0,
                     want_xcont=False, want_stats=False, out=None, stream=None):
        """qa_ground_state_batch on a CUDA tensor Vg[B, P, n_gate] (float64).  Returns dict(N[B,P,n], E[B,P], ...)."""
        if not (isinstance(Vg, torch.Tensor) and Vg.is_cuda and Vg.dtype == torch.float64):
            raise TypeError("Vg must be a CUDA float64 tensor (there is no CPU path)")
        if Vg.device != self.device:
            raise ValueError(f"Vg is on {Vg.device}, the batch lives on {self.device}")
        B = len(self)
        Vg = Vg.contiguous().view(B, -1, self.n_gate)
        P, dev = Vg.shape[1], Vg.device
        out = out or {}
        N = out.get("N") if out.get("N") is not None else torch.empty((B, P, self.n_dot), dtype=torch.int32, device=dev)
        E = out.get("E") if out.get("E") is not None else torch.empty((B, P), dtype=torch.float64, device=dev)
        xc = torch.empty((B, P, self.n_dot), dtype=torch.float64, device=dev) if want_xcont else None
        st = torch.zeros(8, dtype=torch.int64, device=dev) if want_stats else None
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        alg = ALG[algorithm] if isinstance(algorithm, str) else int(algorithm)
        _check(lib().qa_ground_state_batch(self._h, _ptr(Vg), P, int(regime == "closed"), int(N_hat), alg, float(t),
                                           int(n_max), _ptr(N), _ptr(E), _ptr(xc), _ptr(st), C.c_void_p(s.cuda_stream)),
               "qa_ground_state_batch")
        res = {"N": N, "E": E}
        if xc is not None:
            res["xcont"] = xc
        if st is not None:
            res["stats"] = st
        return res

    def ground_state_multi(self, Vg: torch.Tensor, algorithms, want_xcont=False, want_stats=False, out=None, stream=None):
        """qa_ground_state_batch_multi: several algorithms on the same sweep in one launch (V_g read once, N_c and the QP
        once per pixel).  algorithms: list of ("default", None) / ("thresholded", t) pairs (or the strings "default" /
        floats t).  out: optional list of dict(N, E), one per algorithm.  Returns a list of dict(N[B,P,n], E[B,P]) (the
        first one also carries xcont / stats when asked for)."""
        if not (isinstance(Vg, torch.Tensor) and Vg.is_cuda and Vg.dtype == torch.float64):
            raise TypeError("Vg must be a CUDA float64 tensor (there is no CPU path)")
        if Vg.device != self.device:
            raise ValueError(f"Vg is on {Vg.device}, the batch lives on {self.device}")
        B = len(self)
        Vg = Vg.contiguous().view(B, -1, self.n_gate)
        P, dev = Vg.shape[1], Vg.device
        spec = []
        for a in algorithms:
            if isinstance(a, str):
                a = (a, None)
            elif isinstance(a, (int, float)):
                a = ("thresholded", float(a))
            spec.append((ALG[a[0]], 1.0 if a[1] is None else float(a[1])))
        n_alg = len(spec)
        res = []
        for k in range(n_alg):
            o = (out[k] if out is not None else None) or {}
            N = o.get("N") if o.get("N") is not None else torch.empty((B, P, self.n_dot), dtype=torch.int32, device=dev)
            E = o.get("E") if o.get("E") is not None else torch.empty((B, P), dtype=torch.float64, device=dev)
            res.append({"N": N, "E": E})
        xc = torch.empty((B, P, self.n_dot), dtype=torch.float64, device=dev) if want_xcont else None
        st = torch.zeros(8, dtype=torch.int64, device=dev) if want_stats else None
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        algs = (C.c_int * n_alg)(*[a for a, _ in spec])
        ts = (C.c_double * n_alg)(*[t for _, t in spec])
        pN = (C.c_void_p * n_alg)(*[r["N"].data_ptr() for r in res])
        pE = (C.c_void_p * n_alg)(*[r["E"].data_ptr() for r in res])
        _check(lib().qa_ground_state_batch_multi(self._h, _ptr(Vg), P, n_alg, algs, ts, pN, pE, _ptr(xc), _ptr(st),
                                                 C.c_void_p(s.cuda_stream)), "qa_ground_state_batch_multi")
        if xc is not None:
            res[0]["xcont"] = xc
        if st is not None:
            res[0]["stats"] = st
        return res


def sensor_response(Vs: torch.Tensor, W: int, params, want_gradient=True, stream=None) -> dict:
    """qa_sensor_response on a CUDA tensor Vs[P, n_sensor] (float64; the Vsensor output of a ground-state call): response
    profile + noise of every sensor (params: one qa_sensor_params per sensor) and the gradient along the fast axis (row
    length W).  Returns dict(S[P, n_sensor][, G[P, n_sensor]])."""
    if not (isinstance(Vs, torch.Tensor) and Vs.is_cuda and Vs.dtype == torch.float64):
        raise TypeError("Vs must be a CUDA float64 tensor (there is no CPU path)")
    Vs = Vs.contiguous()
    Vs = Vs.view(Vs.shape[0], -1)
    P, ns = Vs.shape
    dev = Vs.device
    arr = (qa_sensor_params * ns)(*params)
    S = torch.empty((P, ns), dtype=torch.float64, device=dev)
    G = torch.empty((P, ns), dtype=torch.float64, device=dev) if want_gradient else None
    ws = torch.empty(max(256, int(lib().qa_sensor_response_workspace_bytes(P, ns))), dtype=torch.uint8, device=dev)
    s = stream if stream is not None else torch.cuda.current_stream(dev)
    with torch.cuda.device(dev):
        _check(lib().qa_sensor_response(_ptr(Vs), P, ns, int(W), C.byref(arr), _ptr(S), _ptr(G), _ptr(ws), ws.numel(),
                                        C.c_void_p(s.cuda_stream)), "qa_sensor_response")
    return {"S": S, "G": G} if want_gradient else {"S": S}


def stats_dict(t: torch.Tensor) -> dict:
    v = t.cpu().tolist()
    return {k: int(v[i]) for i, (k, _) in enumerate(qa_stats._fields_)}


def measure_fp64_rate(seconds: float = 1.0) -> float:
    """qa_measure_fp64_rate: sustained FP64 thread-instructions/s of the current device."""
    r = C.c_double()
    _check(lib().qa_measure_fp64_rate(float(seconds), C.byref(r), C.c_void_p(torch.cuda.current_stream().cuda_stream)),
           "qa_measure_fp64_rate")
    return r.value


def kernel_times(model: "Model", Vg: torch.Tensor, steps: int = 10, flush: torch.Tensor | None = None, call: str = "ground_state",
                 **kw) -> dict:
    """Average device time (ms) of each kernel of model.ground_state(Vg, **kw) (or model.thermal with call="thermal"), from
    CUDA events recorded by the library between its kernels on the launching stream (qa_set_kernel_timing /
    qa_get_kernel_timings)."""
    acc: dict = {}
    lib().qa_set_kernel_timing(1)
    try:
        for k in range(steps):
            if flush is not None:
                flush.fill_(k & 0xff)
            getattr(model, call)(Vg, **kw)
            ms = (C.c_float * 8)()
            n = C.c_int()
            _check(lib().qa_get_kernel_timings(8, ms, C.byref(n)), "qa_get_kernel_timings")
            names = last_launch_plan()[0]
            for i in range(n.value):
                key = names[i].split("<")[0]
                acc[key] = acc.get(key, 0.0) + ms[i] / steps
    finally:
        lib().qa_set_kernel_timing(0)
    return acc


def last_launch_plan():
    return lib().qa_last_launch_plan().decode().split(","), int(lib().qa_last_launch_count())


def version() -> str:
    return lib().qa_version().decode()
