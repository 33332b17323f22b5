"""ctypes front end of the C++ oracle (oracle/mps_oracle.cpp).

TEST INFRASTRUCTURE.  Argument marshalling only; every number is computed by
the single-threaded C++ code.  Imports nothing from the CUDA path.
"""
from __future__ import annotations

import ctypes as C
from typing import Dict, Tuple

import numpy as np

from . import build as _build

_lib = None

F64 = {"x": 0, "y": 1, "z": 2, "u": 3, "v": 4, "w": 5, "n": 6, "p": 7, "ax": 8, "ay": 9,
       "az": 10, "nut": 11, "b": 12, "phat": 13, "gx": 14, "gy": 15, "gz": 16, "xcg": 17,
       "dndt": 18, "n_k": 19, "dndt_k": 20, "rho_s": 21}
I32 = {"type": 0, "phase": 1, "bc": 2, "key": 3, "perm": 4}

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [_dp, _ip, C.c_int] + [_dp] * 6 + [_ip] * 2
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_brute.argtypes = [C.c_void_p, C.c_int]
        for nm in ("orc_set_f64", "orc_get_f64"):
            getattr(L, nm).argtypes = [C.c_void_p, C.c_int, _dp]
        for nm in ("orc_set_i32", "orc_get_i32"):
            getattr(L, nm).argtypes = [C.c_void_p, C.c_int, _ip]
        L.orc_constants.argtypes = [C.c_void_p, _dp]
        L.orc_stats.argtypes = [C.c_void_p, _dp]
        L.orc_grid.argtypes = [C.c_void_p, _ip]
        L.orc_get_cell_start.argtypes = [C.c_void_p, _ip]
        L.orc_neighbours.restype = C.c_longlong
        L.orc_neighbours.argtypes = [C.c_void_p, C.c_double, _ip, _ip, C.c_longlong]
        for nm in ("orc_smooth_density", "orc_bin", "orc_density", "orc_viscosity", "orc_predict",
                   "orc_pressure_explicit", "orc_ppe_flags", "orc_ppe_rhs", "orc_pressure_ppe",
                   "orc_phat", "orc_gradient", "orc_correct"):
            getattr(L, nm).argtypes = [C.c_void_p]
        L.orc_dndt.argtypes = [C.c_void_p, C.c_int]
        L.orc_freeze_lists.argtypes = [C.c_void_p, C.c_int]
        L.orc_ppe_apply.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_ppe_solve.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.orc_step.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_morton3.argtypes = [C.c_int, C.c_int, C.c_int]
        L.orc_ppe_solve_pcg.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_int, C.c_double]
        L.orc_lattice_constants.argtypes = [C.c_int, C.c_double, C.c_double, _dp]
        L.orc_lattice_constants_k.argtypes = [C.c_int, C.c_double, C.c_double, C.c_int, _dp]
        L.orc_eos.restype = C.c_double
        L.orc_eos.argtypes = [C.c_double] * 5
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def lattice_constants(dim: int, l0: float, re: float, kernel: int = 0) -> Tuple[float, float, int]:
    out = np.zeros(3)
    lib().orc_lattice_constants_k(dim, l0, re, kernel, _d(out))
    return float(out[0]), float(out[1]), int(out[2])


def morton3(cx: int, cy: int, cz: int) -> int:
    return int(lib().orc_morton3(cx, cy, cz))


def eos(rho, c0, gamma, n, n0) -> float:
    return float(lib().orc_eos(rho, c0, gamma, n, n0))


def pack_params(p: Dict[str, object]):
    dp = np.array([p["l0"], p["re_n"], p["re_lap"], p["dt"], *p["g"], *p["rho"], *p["nu"],
                   p["c0"], p["gamma"], p["beta"], p["compress"], p["ppe_relax"], p["cg_rtol"],
                   p["cs"], *p["domain_min"], *p["domain_max"], p["n0_n"], p["n0_lap"],
                   p["lam"]], dtype=np.float64)
    ip = np.array([p["dim"], p["n_phases"], p["cg_maxit"], p["grad_variant"],
                   p["clamp_negative_p"], p["rho_pair_mean"], p["nu_pair_mean"], p["cell_div"],
                   p["max_neighbours"], p.get("ppe_source", 0), p.get("ppe_laplacian", 0),
                   p.get("kernel", 0), p.get("rebin_every", 1), p.get("key_mode", 0),
                   p.get("cg_warm_start", 0)], dtype=np.int32)
    assert dp.size == 27 and ip.size == 15
    return dp, ip


class Oracle:
    """One MPS state in the caller's original particle order."""

    def __init__(self, scene, brute: bool = False, **override):
        self.L = lib()
        p = dict(scene.params)
        p.update(override)
        self.params = p
        dp, ip = pack_params(p)
        self.n = scene.n
        arrs = [np.ascontiguousarray(getattr(scene, k), dtype=np.float64) for k in "xyzuvw"]
        ty = np.ascontiguousarray(scene.type, dtype=np.int32)
        ph = np.ascontiguousarray(scene.phase, dtype=np.int32)
        self.h = C.c_void_p(self.L.orc_create(_d(dp), _i(ip), self.n, *[_d(a) for a in arrs],
                                              _i(ty), _i(ph)))
        if brute:
            self.L.orc_set_brute(self.h, 1)

    def __del__(self):
        try:
            if self.h:
                self.L.orc_destroy(self.h)
                self.h = None
        except Exception:
            pass

    # ---- fields -----------------------------------------------------------
    def get(self, name: str) -> np.ndarray:
        if name in F64:
            out = np.empty(self.n, np.float64)
            assert self.L.orc_get_f64(self.h, F64[name], _d(out)) == 0
        else:
            out = np.empty(self.n, np.int32)
            assert self.L.orc_get_i32(self.h, I32[name], _i(out)) == 0, name
        return out

    def set(self, name: str, a) -> None:
        if name in F64:
            a = np.ascontiguousarray(a, np.float64)
            assert a.size == self.n
            assert self.L.orc_set_f64(self.h, F64[name], _d(a)) == 0
        else:
            a = np.ascontiguousarray(a, np.int32)
            assert a.size == self.n
            assert self.L.orc_set_i32(self.h, I32[name], _i(a)) == 0

    def constants(self) -> Dict[str, float]:
        out = np.zeros(6)
        self.L.orc_constants(self.h, _d(out))
        return dict(n0_n=out[0], n0_lap=out[1], lam=out[2], A_lap=out[3], h=out[4], inv_h=out[5])

    def stats(self) -> Dict[str, float]:
        out = np.zeros(5)
        self.L.orc_stats(self.h, _d(out))
        return dict(cg_iters=int(out[0]), cg_relres=out[1], n_ghost=int(out[2]),
                    n_surface=int(out[3]), max_nb=int(out[4]))

    def grid(self):
        out = np.zeros(4, np.int32)
        self.L.orc_grid(self.h, _i(out))
        return tuple(int(v) for v in out)

    # ---- stages -----------------------------------------------------------
    def bin(self):
        self.L.orc_bin(self.h)
        ncells = self.grid()[3]
        cs = np.empty(ncells + 1, np.int32)
        self.L.orc_get_cell_start(self.h, _i(cs))
        return self.get("key"), self.get("perm"), cs

    def neighbours(self, re: float):
        counts = np.zeros(self.n, np.int32)
        tot = self.L.orc_neighbours(self.h, re, _i(counts), None, 0)
        idx = np.zeros(max(int(tot), 1), np.int32)
        tot2 = self.L.orc_neighbours(self.h, re, _i(counts), _i(idx), int(tot))
        assert tot2 == tot
        return counts, idx[:tot]

    def density(self): self.L.orc_density(self.h)
    def viscosity(self): self.L.orc_viscosity(self.h)
    def predict(self): self.L.orc_predict(self.h)
    def pressure_explicit(self): self.L.orc_pressure_explicit(self.h)
    def smooth_density(self): self.L.orc_smooth_density(self.h)
    def freeze_lists(self, on: bool = True): self.L.orc_freeze_lists(self.h, 1 if on else 0)
    def dndt(self, keep: bool = False): self.L.orc_dndt(self.h, 20 if keep else 18)
    def ppe_flags(self): self.L.orc_ppe_flags(self.h)
    def ppe_rhs(self): self.L.orc_ppe_rhs(self.h)
    def pressure_ppe(self) -> int: return int(self.L.orc_pressure_ppe(self.h))
    def phat(self): self.L.orc_phat(self.h)
    def gradient(self): self.L.orc_gradient(self.h)
    def correct(self): self.L.orc_correct(self.h)

    def ppe_apply(self, x) -> np.ndarray:
        x = np.ascontiguousarray(x, np.float64)
        y = np.empty(self.n, np.float64)
        self.L.orc_ppe_apply(self.h, _d(x), _d(y))
        return y

    def ppe_solve(self, rtol: float, maxit: int) -> int:
        return int(self.L.orc_ppe_solve(self.h, rtol, maxit))

    def ppe_solve_pcg(self, rtol: float, maxit: int, precond: int, degree: int = 0, ratio: float = 30.0) -> int:
        """Preconditioned CG on the assembled rows (needs ppe_flags + ppe_rhs): precond 0 none, 1 Jacobi,
        2 cell-block Jacobi, 3 IC(0), 4 Chebyshev polynomial (degree, lmax/lmin ratio).  Returns iterations."""
        return int(self.L.orc_ppe_solve_pcg(self.h, rtol, maxit, precond, degree, ratio))

    def step(self, nsteps: int = 1, route: int = 0) -> int:
        return int(self.L.orc_step(self.h, nsteps, route))
