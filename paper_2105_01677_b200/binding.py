"""Thin ctypes binding of libmps_b200.so (include/mps_b200.h), same names.

Argument marshalling only: every step of the path runs in the library's CUDA
kernels.  torch is used for device memory and streams.  There is no CPU
fallback: importing this module raises if the library has not been built, and
every call raises `MpsError` on a non-zero return code.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmps_b200.so")

MPS_OK, MPS_ERR_ARG, MPS_ERR_CUDA, MPS_ERR_NEIGHBOUR_OVERFLOW = 0, -1, -2, -3
MPS_ERR_NOCONV, MPS_ERR_NONFINITE, MPS_ERR_ORDER = -4, -5, -6
ORDER_ORIGINAL, ORDER_SORTED = 0, 1
ROUTE_EXPLICIT, ROUTE_PPE = 0, 1
RADIUS_N, RADIUS_LAP = 0, 1

FIELDS = {"x": 0, "y": 1, "z": 2, "u": 3, "v": 4, "w": 5, "n": 6, "p": 7, "ax": 8, "ay": 9,
          "az": 10, "nut": 11, "b": 12, "phat": 13, "gx": 14, "gy": 15, "gz": 16, "xcg": 17,
          "dndt": 18, "nk": 19, "dndtk": 20, "rhos": 21,
          "type": 32, "phase": 33, "bc": 34, "key": 35}
TIMERS = ["bin_sort", "bin_list", "viscosity", "predict", "density", "pressure_explicit",
          "ppe_setup", "cg_spmv", "cg_update", "gradient", "correct"]

# Names the header declares (checked by tests/test_abi.py against include/mps_b200.h).
SYMBOLS = ["mps_init", "mps_init_host", "mps_destroy", "mps_bin", "mps_density", "mps_dndt", "mps_smooth_density", "mps_viscosity",
           "mps_predict", "mps_pressure_explicit", "mps_pressure_ppe", "mps_gradient",
           "mps_correct", "mps_step", "mps_step_host", "mps_upload_host", "mps_download_host",
           "mps_get_field", "mps_set_field",
           "mps_get_perm", "mps_get_grid", "mps_get_cell_start", "mps_get_neighbours",
           "mps_ppe_apply", "mps_get_constants", "mps_get_stats", "mps_sync",
           "mps_timers_enable", "mps_timers_read", "mps_launch_count", "mps_last_error",
           "mps_version", "mps_cell_start_noalloc", "mps_cell_start_noalloc_max_cells",
           "mps_cell_start_noalloc_error"]


class MpsParams(C.Structure):
    _fields_ = [
        ("dim", C.c_int32), ("n_phases", C.c_int32), ("cg_maxit", C.c_int32),
        ("grad_variant", C.c_int32), ("clamp_negative_p", C.c_int32),
        ("rho_pair_mean", C.c_int32), ("nu_pair_mean", C.c_int32), ("key_mode", C.c_int32),
        ("cell_div", C.c_int32), ("max_neighbours", C.c_int32), ("ppe_source", C.c_int32),
        ("ppe_laplacian", C.c_int32), ("kernel", C.c_int32), ("rebin_every", C.c_int32),
        ("ppe_operator", C.c_int32), ("cg_warm_start", C.c_int32),
        ("l0", C.c_double), ("re_n", C.c_double), ("re_grad", C.c_double),
        ("re_lap", C.c_double), ("dt", C.c_double), ("g", C.c_double * 3),
        ("rho", C.c_double * 2), ("nu", C.c_double * 2), ("c0", C.c_double),
        ("gamma", C.c_double), ("beta", C.c_double), ("compress", C.c_double),
        ("ppe_relax", C.c_double), ("cg_rtol", C.c_double), ("cs", C.c_double),
        ("domain_min", C.c_double * 3), ("domain_max", C.c_double * 3),
        ("n0_n", C.c_double), ("n0_lap", C.c_double), ("lambda_", C.c_double),
        ("row_skin", C.c_double),
    ]


class MpsStats(C.Structure):
    _fields_ = [
        ("cg_iters", C.c_int32), ("cg_converged", C.c_int32), ("cg_relres", C.c_double),
        ("max_neighbours", C.c_int32), ("n_surface", C.c_int32), ("n_ghost", C.c_int32),
        ("n_rows", C.c_int32), ("cg_iters_total", C.c_int64), ("steps_total", C.c_int64),
        ("device_error", C.c_int32), ("cg_noconv_total", C.c_int32),
        ("cg_setup_ms", C.c_double), ("cg_loop_ms", C.c_double), ("cg_loop_ms_total", C.c_double),
        ("cg_nnz", C.c_int64), ("bins_total", C.c_int64), ("row_skin_now", C.c_double),
    ]

    def as_dict(self) -> Dict[str, float]:
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class MpsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libmps_b200 error {code}: {msg}")
        self.code = code


def make_params(p: Dict[str, object]) -> MpsParams:
    """Scene/param dict (paper_2105_01677_b200.scenes.default_params keys) -> struct."""
    s = MpsParams()
    for k in ("dim", "n_phases", "cg_maxit", "grad_variant", "clamp_negative_p", "rho_pair_mean",
              "nu_pair_mean", "cell_div", "max_neighbours"):
        setattr(s, k, int(p[k]))
    s.key_mode = int(p.get("key_mode", 0))
    s.ppe_source = int(p.get("ppe_source", 0))
    s.ppe_laplacian = int(p.get("ppe_laplacian", 0))
    s.kernel = int(p.get("kernel", 0))
    s.rebin_every = int(p.get("rebin_every", 1))
    s.ppe_operator = int(p.get("ppe_operator", 1))
    s.cg_warm_start = int(p.get("cg_warm_start", 0))
    for k in ("l0", "re_n", "re_lap", "dt", "c0", "gamma", "beta", "compress", "ppe_relax",
              "cg_rtol", "cs", "n0_n", "n0_lap"):
        setattr(s, k, float(p[k]))
    s.re_grad = float(p.get("re_grad", p["re_n"]))
    s.lambda_ = float(p["lam"])
    s.row_skin = float(p.get("row_skin", 0.0))
    for k, m in (("g", 3), ("rho", 2), ("nu", 2), ("domain_min", 3), ("domain_max", 3)):
        arr = getattr(s, k)
        for i in range(m):
            arr[i] = float(p[k][i])
    return s


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2105_01677_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.mps_init.argtypes = [C.POINTER(vp), C.POINTER(MpsParams), i64] + [vp] * 8 + [vp]
    L.mps_init_host.argtypes = L.mps_init.argtypes
    L.mps_destroy.argtypes = [vp]
    for nm in ("mps_smooth_density", "mps_bin", "mps_density", "mps_viscosity", "mps_predict", "mps_pressure_explicit",
               "mps_gradient", "mps_correct", "mps_sync"):
        getattr(L, nm).argtypes = [vp]
    L.mps_dndt.argtypes = [vp, i32]
    L.mps_pressure_ppe.argtypes = [vp, C.POINTER(i32), C.POINTER(dbl)]
    L.mps_step.argtypes = [vp, i32, i32]
    L.mps_step_host.argtypes = [C.POINTER(MpsParams), i64] + [vp] * 6 + [vp, vp, vp, i32, i32,
                                                                      C.POINTER(MpsStats), vp]
    L.mps_upload_host.argtypes = [vp] + [vp] * 8
    L.mps_download_host.argtypes = [vp] + [vp] * 7
    L.mps_get_field.argtypes = [vp, i32, vp, i32]
    L.mps_set_field.argtypes = [vp, i32, vp, i32]
    L.mps_get_perm.argtypes = [vp, vp]
    L.mps_get_grid.argtypes = [vp, C.POINTER(i32)]
    L.mps_get_cell_start.argtypes = [vp, vp]
    L.mps_get_neighbours.argtypes = [vp, i32, vp, vp, i64, C.POINTER(i64)]
    L.mps_ppe_apply.argtypes = [vp, vp, vp, i32]
    L.mps_get_constants.argtypes = [vp, C.POINTER(dbl)]
    L.mps_get_stats.argtypes = [vp, C.POINTER(MpsStats)]
    L.mps_timers_enable.argtypes = [vp, i32]
    L.mps_timers_read.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
    L.mps_launch_count.argtypes = [vp]
    L.mps_launch_count.restype = i64
    L.mps_last_error.argtypes = [vp]
    L.mps_last_error.restype = C.c_char_p
    L.mps_version.restype = C.c_char_p
    L.mps_cell_start_noalloc.argtypes = [vp, i64, i32, vp, vp]
    L.mps_cell_start_noalloc_max_cells.restype = i32
    L.mps_cell_start_noalloc_error.restype = C.c_char_p
    return L


lib = _load()


def version() -> str:
    return lib.mps_version().decode()


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libmps_b200 needs a CUDA device (B200); there is no CPU fallback")
    return torch


def cell_start_noalloc(key, n_cells: int, cell_start, stream=None) -> None:
    """mps_cell_start_noalloc: key and cell_start are CUDA tensors (int32 / uint32 words; cell_start has
    n_cells + 1 entries and is written asynchronously on `stream`, default torch's current stream)."""
    torch = _torch()
    st = stream if stream is not None else torch.cuda.current_stream(key.device)
    rc = lib.mps_cell_start_noalloc(key.data_ptr(), int(key.numel()), int(n_cells), cell_start.data_ptr(),
                                    st.cuda_stream)
    if rc != 0:
        raise MpsError(rc, lib.mps_cell_start_noalloc_error().decode())


def cell_start_noalloc_max_cells() -> int:
    return int(lib.mps_cell_start_noalloc_max_cells())


class Mps:
    """One simulation context.  Methods mirror the C entry points one to one."""

    def __init__(self, scene=None, *, params: Optional[Dict[str, object]] = None, arrays=None,
                 stream=None, device="cuda:0", **override):
        torch = _torch()
        self.torch = torch
        self.device = torch.device(device)
        if scene is not None:
            p = dict(scene.params)
            arrays = {k: getattr(scene, k) for k in ("x", "y", "z", "u", "v", "w", "type", "phase")}
        else:
            p = dict(params)
        p.update(override)
        self.params = p
        self._prm = make_params(p)
        self.n = int(arrays["x"].shape[0])
        # a stream of the ctx's own by default: the legacy default stream cannot be captured, and
        # mps_step replays its launch sequence from CUDA graphs.  Every method below orders the ctx
        # stream against torch's current stream where data changes hands.
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        with torch.cuda.device(self.device):
            dev = {}
            for k in ("x", "y", "z", "u", "v", "w"):
                dev[k] = torch.as_tensor(np.ascontiguousarray(arrays[k], np.float64)).to(self.device)
            for k in ("type", "phase"):
                dev[k] = torch.as_tensor(np.ascontiguousarray(arrays[k], np.int32)).to(self.device)
            self.h = C.c_void_p()
            torch.cuda.current_stream(self.device).synchronize()
            rc = lib.mps_init(C.byref(self.h), C.byref(self._prm), self.n,
                              *[dev[k].data_ptr() for k in ("x", "y", "z", "u", "v", "w", "type", "phase")],
                              self.stream.cuda_stream)
            if rc != 0:
                raise MpsError(rc, lib.mps_last_error(None).decode())
            self.stream.synchronize()

    # ---- plumbing ------------------------------------------------------------
    def _ck(self, rc: int, allow=()):
        if rc != 0 and rc not in allow:
            raise MpsError(rc, lib.mps_last_error(self.h).decode())
        return rc

    def close(self):
        if getattr(self, "h", None):
            lib.mps_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the path --------------------------------------------------------------
    def bin(self): self._ck(lib.mps_bin(self.h))
    def density(self): self._ck(lib.mps_density(self.h))
    def smooth_density(self): self._ck(lib.mps_smooth_density(self.h))
    def dndt(self, keep: bool = False): self._ck(lib.mps_dndt(self.h, 1 if keep else 0))
    def viscosity(self): self._ck(lib.mps_viscosity(self.h))
    def predict(self): self._ck(lib.mps_predict(self.h))
    def pressure_explicit(self): self._ck(lib.mps_pressure_explicit(self.h))
    def gradient(self): self._ck(lib.mps_gradient(self.h))
    def correct(self): self._ck(lib.mps_correct(self.h))

    def pressure_ppe(self, allow_noconv: bool = False) -> Tuple[int, float]:
        it, rr = C.c_int32(0), C.c_double(0.0)
        self._ck(lib.mps_pressure_ppe(self.h, C.byref(it), C.byref(rr)),
                 allow=(MPS_ERR_NOCONV,) if allow_noconv else ())
        return int(it.value), float(rr.value)

    def step(self, nsteps: int = 1, route: int = 0) -> int:
        return self._ck(lib.mps_step(self.h, nsteps, route))

    def sync(self): self._ck(lib.mps_sync(self.h))

    def upload_host(self, ptrs) -> None:
        """ptrs: 8 host addresses (x, y, z, u, v, w, type, phase), n elements each."""
        self._ck(lib.mps_upload_host(self.h, *ptrs))

    def download_host(self, ptrs) -> None:
        """ptrs: 7 host addresses (x, y, z, u, v, w, p) or None; synchronises."""
        self._ck(lib.mps_download_host(self.h, *ptrs))

    # ---- fields -------------------------------------------------------------------
    def get_dev(self, name: str, order: int = ORDER_ORIGINAL):
        fid = FIELDS[name]
        t = self.torch.empty(self.n, dtype=self.torch.float64 if fid < 32 else self.torch.int32,
                             device=self.device)
        self._ck(lib.mps_get_field(self.h, fid, t.data_ptr(), order))
        self.stream.synchronize()
        return t

    def get(self, name: str, order: int = ORDER_ORIGINAL) -> np.ndarray:
        return self.get_dev(name, order).cpu().numpy()

    def set(self, name: str, a, order: int = ORDER_ORIGINAL) -> None:
        fid = FIELDS[name]
        dt = np.float64 if fid < 32 else np.int32
        t = self.torch.as_tensor(np.ascontiguousarray(a, dt)).to(self.device)
        assert t.numel() == self.n
        self.torch.cuda.current_stream(self.device).synchronize()
        self._ck(lib.mps_set_field(self.h, fid, t.data_ptr(), order))
        self.stream.synchronize()

    def perm(self) -> np.ndarray:
        t = self.torch.empty(self.n, dtype=self.torch.int32, device=self.device)
        self._ck(lib.mps_get_perm(self.h, t.data_ptr()))
        self.stream.synchronize()
        return t.cpu().numpy()

    def grid(self) -> Tuple[int, int, int, int]:
        g = (C.c_int32 * 4)()
        self._ck(lib.mps_get_grid(self.h, g))
        return tuple(int(v) for v in g)

    def cell_start(self) -> np.ndarray:
        nc = self.grid()[3]
        t = self.torch.empty(nc + 1, dtype=self.torch.int32, device=self.device)
        self._ck(lib.mps_get_cell_start(self.h, t.data_ptr()))
        self.stream.synchronize()
        return t.cpu().numpy()

    def neighbours(self, radius_id: int) -> Tuple[np.ndarray, np.ndarray]:
        counts = self.torch.empty(self.n, dtype=self.torch.int32, device=self.device)
        tot = C.c_int64(0)
        self._ck(lib.mps_get_neighbours(self.h, radius_id, counts.data_ptr(), None, 0, C.byref(tot)))
        idx = self.torch.empty(max(tot.value, 1), dtype=self.torch.int32, device=self.device)
        self._ck(lib.mps_get_neighbours(self.h, radius_id, counts.data_ptr(), idx.data_ptr(),
                                        tot.value, C.byref(tot)))
        self.stream.synchronize()
        return counts.cpu().numpy(), idx.cpu().numpy()[: tot.value]

    def neighbour_counts(self, radius_id: int) -> np.ndarray:
        counts = self.torch.empty(self.n, dtype=self.torch.int32, device=self.device)
        tot = C.c_int64(0)
        self._ck(lib.mps_get_neighbours(self.h, radius_id, counts.data_ptr(), None, 0, C.byref(tot)))
        self.stream.synchronize()
        return counts.cpu().numpy()

    def ppe_apply(self, x, order: int = ORDER_ORIGINAL) -> np.ndarray:
        xt = self.torch.as_tensor(np.ascontiguousarray(x, np.float64)).to(self.device)
        yt = self.torch.empty_like(xt)
        self.torch.cuda.current_stream(self.device).synchronize()
        self._ck(lib.mps_ppe_apply(self.h, xt.data_ptr(), yt.data_ptr(), order))
        self.stream.synchronize()
        return yt.cpu().numpy()

    def constants(self) -> Dict[str, float]:
        out = (C.c_double * 6)()
        self._ck(lib.mps_get_constants(self.h, out))
        return dict(n0_n=out[0], n0_lap=out[1], lam=out[2], A_lap=out[3], h=out[4], inv_h=out[5])

    def stats(self) -> Dict[str, float]:
        s = MpsStats()
        self._ck(lib.mps_get_stats(self.h, C.byref(s)))
        return s.as_dict()

    def timers_enable(self, mask: int) -> None:
        self._ck(lib.mps_timers_enable(self.h, mask))

    def timers_read(self) -> Dict[str, Tuple[float, int]]:
        ms = (C.c_double * len(TIMERS))()
        ln = (C.c_int64 * len(TIMERS))()
        self._ck(lib.mps_timers_read(self.h, ms, ln))
        return {k: (float(ms[i]), int(ln[i])) for i, k in enumerate(TIMERS)}

    def launch_count(self) -> int:
        return int(lib.mps_launch_count(self.h))


def step_host(scene_or_params, arrays: Dict[str, np.ndarray], nsteps: int, route: int,
              want_p: bool = True, stream_ptr: int = 0):
    """mps_step_host on HOST numpy buffers (in place); returns (rc, stats dict, p)."""
    p = scene_or_params if isinstance(scene_or_params, dict) else scene_or_params.params
    prm = make_params(p)
    n = int(arrays["x"].shape[0])
    ptr = lambda a: a.ctypes.data_as(C.c_void_p)
    pout = np.empty(n, np.float64) if want_p else None
    st = MpsStats()
    rc = lib.mps_step_host(C.byref(prm), n, *[ptr(arrays[k]) for k in ("x", "y", "z", "u", "v", "w")],
                           ptr(arrays["type"]), ptr(arrays["phase"]),
                           ptr(pout) if want_p else None, nsteps, route, C.byref(st), stream_ptr)
    if rc not in (0, MPS_ERR_NOCONV):
        raise MpsError(rc, lib.mps_last_error(None).decode())
    return rc, st.as_dict(), pout
