"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front-end of ``oracle/dualip_oracle.c``: the plain fp64 CPU restatement of the paper's dual
function, gradient, projections and AGD / gamma-continuation loop (arxiv/paper_2606_07777, Eq. 1-4,
P:55-75).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports nothing from
``paper_2606_07777_b200`` and shares no code with it.

Everything here is argument marshalling (numpy arrays -> C pointers); the arithmetic is in the C file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dualip_oracle.c")
_LIB = os.path.join(_HERE, "libdualip_oracle.so")

PROJ_SIMPLEX_INEQ, PROJ_BOX, PROJ_BOXCUT, PROJ_SIMPLEX_EQ = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c11", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        d, i64, i32, vp = ctypes.c_double, ctypes.c_int64, ctypes.c_int32, ctypes.c_void_p
        lib.dualip_oracle_project_simplex.argtypes = [vp, i64, d, vp]
        lib.dualip_oracle_project_simplex_eq.argtypes = [vp, i64, d, vp]
        lib.dualip_oracle_project_box.argtypes = [vp, i64, d, d, vp]
        lib.dualip_oracle_project_boxcut.argtypes = [vp, i64, d, d, vp]
        for f in (lib.dualip_oracle_project_simplex, lib.dualip_oracle_project_simplex_eq,
                  lib.dualip_oracle_project_box, lib.dualip_oracle_project_boxcut):
            f.restype = None
        lib.dualip_oracle_grad.argtypes = [i64, i32, i32, vp, vp, vp, vp, vp, vp, d, ctypes.c_int, d, d, vp, i32, d, vp, vp, vp]
        lib.dualip_oracle_grad.restype = ctypes.c_int
        lib.dualip_oracle_lipschitz.argtypes = [i64, i32, i32, vp, vp, vp, i32]
        lib.dualip_oracle_lipschitz.restype = d
        lib.dualip_oracle_jacobi_scaling.argtypes = [i64, i32, i32, vp, vp, vp, vp]
        lib.dualip_oracle_jacobi_scaling.restype = None
        lib.dualip_oracle_solve.argtypes = [i64, i32, i32, vp, vp, vp, vp, vp, ctypes.c_int, d, d,
                                            vp, i32, vp, i32, i32, vp, i32, d, d, i32, d,
                                            vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        lib.dualip_oracle_solve.restype = ctypes.c_int
        _lib = lib
    return _lib


def _ptr(arr):
    return None if arr is None else arr.ctypes.data_as(ctypes.c_void_p)


def _f64(v):
    return np.ascontiguousarray(np.asarray(v, dtype=np.float64))


def project_simplex(v, z: float = 1.0):
    """{x >= 0, sum x <= z}."""
    v = _f64(v); x = np.empty_like(v)
    _load().dualip_oracle_project_simplex(_ptr(v), v.size, z, _ptr(x))
    return x


def project_simplex_eq(v, z: float = 1.0):
    """{x >= 0, sum x = z} (Duchi et al.)."""
    v = _f64(v); x = np.empty_like(v)
    _load().dualip_oracle_project_simplex_eq(_ptr(v), v.size, z, _ptr(x))
    return x


def project_box(v, lo: float = 0.0, hi: float = 1.0):
    v = _f64(v); x = np.empty_like(v)
    _load().dualip_oracle_project_box(_ptr(v), v.size, lo, hi, _ptr(x))
    return x


def project_boxcut(v, ub: float = 1.0, z: float = 1.0):
    """{0 <= x <= ub, sum x <= z}."""
    v = _f64(v); x = np.empty_like(v)
    _load().dualip_oracle_project_boxcut(_ptr(v), v.size, ub, z, _ptr(x))
    return x


@dataclass
class Problem:
    """Per-user CSR rows of (item_idx:int32, c:fp32, a:fp32[m]) plus b:fp32[J*m]."""
    I: int
    J: int
    m: int
    row_ptr: np.ndarray
    item_idx: np.ndarray
    c: np.ndarray
    a: np.ndarray
    b: np.ndarray
    proj_kind: int = PROJ_SIMPLEX_INEQ
    p0: float = 1.0
    p1: float = 0.0
    count_M: float | None = None      # global-count row  sum_{(i,j)} x_ij <= count_M  (reading R21); None = absent

    @property
    def rows(self) -> int:
        """coupling rows = duals: J*m, plus one for the global-count row"""
        return self.J * self.m + (1 if self.count_M is not None else 0)

    def __post_init__(self):
        self.row_ptr = np.ascontiguousarray(self.row_ptr, dtype=np.int64)
        self.item_idx = np.ascontiguousarray(self.item_idx, dtype=np.int32)
        self.c = np.ascontiguousarray(self.c, dtype=np.float32)
        self.a = np.ascontiguousarray(self.a, dtype=np.float32).reshape(-1)
        self.b = np.ascontiguousarray(self.b, dtype=np.float32).reshape(-1)
        assert self.row_ptr.size == self.I + 1
        nnz = int(self.row_ptr[-1])
        assert self.item_idx.size == nnz and self.c.size == nnz and self.a.size == nnz * self.m
        assert self.b.size == self.J * self.m

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])


@dataclass
class GradResult:
    g: float
    obj: float
    reg: float
    r_inf: float
    r_2: float
    grad: np.ndarray
    x: np.ndarray | None
    gap: float = 0.0


def _eq_mask(p: Problem, is_eq):
    if is_eq is None:
        return None
    eq = np.ascontiguousarray(np.asarray(is_eq, dtype=np.uint8)).reshape(-1)
    assert eq.size == p.rows
    return eq


def grad(p: Problem, lam, gamma: float, want_x: bool = True, is_eq=None) -> GradResult:
    """(g, grad g, x*) at lambda -- Eq. 2-4.  lambda / grad have p.rows entries (the last one belongs to the
    global-count row when the problem has one); is_eq: uint8 mask of equality rows (residuals count |grad| there, R19)."""
    lam = _f64(lam).reshape(-1)
    assert lam.size == p.rows
    g = np.empty(p.rows, dtype=np.float64)
    sc = np.empty(6, dtype=np.float64)
    x = np.empty(p.nnz, dtype=np.float64) if want_x else None
    eq = _eq_mask(p, is_eq)
    rc = _load().dualip_oracle_grad(p.I, p.J, p.m, _ptr(p.row_ptr), _ptr(p.item_idx), _ptr(p.c), _ptr(p.a),
                                    _ptr(p.b), _ptr(lam), gamma, p.proj_kind, p.p0, p.p1, _ptr(eq),
                                    0 if p.count_M is None else 1, 0.0 if p.count_M is None else float(p.count_M),
                                    _ptr(g), _ptr(sc), _ptr(x))
    if rc != 0:
        raise MemoryError("oracle grad failed")
    return GradResult(sc[0], sc[1], sc[2], sc[3], sc[4], g, x, sc[5])


def lipschitz(p: Problem) -> float:
    """L = max_j sum_k sum_i (a^k_ij)^2 (reading R2), + nnz with the global-count row (R21)."""
    return float(_load().dualip_oracle_lipschitz(p.I, p.J, p.m, _ptr(p.row_ptr), _ptr(p.item_idx), _ptr(p.a),
                                                 0 if p.count_M is None else 1))


def jacobi_scaling(p: Problem) -> np.ndarray:
    """diag(D), D_rr = 1/|A_r*|_2 per coupling row r = (j,k), 1 for rows of zero norm."""
    d = np.empty(p.J * p.m, dtype=np.float64)
    _load().dualip_oracle_jacobi_scaling(p.I, p.J, p.m, _ptr(p.row_ptr), _ptr(p.item_idx), _ptr(p.a), _ptr(d))
    return d


@dataclass
class SolveResult:
    lam: np.ndarray
    x: np.ndarray | None
    final: GradResult
    trace_g: np.ndarray
    trace_rinf: np.ndarray
    trace_r2: np.ndarray
    trace_grad: np.ndarray | None
    trace_lambda: np.ndarray | None
    stage_x: np.ndarray | None
    trace_eta: np.ndarray | None = None


def solve(p: Problem, gammas, iters, lam0=None, momentum: bool = True, want_x: bool = True,
          trace_grad: bool = False, trace_lambda: bool = False, stage_x: bool = False, jacobi: bool = False,
          is_eq=None, adaptive: bool = False, eta_min: float = 1e-5, eta_max: float = 1e-1) -> SolveResult:
    """gamma-continuation + projected Nesterov ascent (readings R1-R4); jacobi: on the row-scaled
    system A' = D A, b' = D b, results reported in the original units (R18); is_eq: uint8 mask
    over the coupling rows, nonzero = equality row whose dual is not projected (R19); adaptive: the range-clipped
    secant step (R20) with the range [eta_min, eta_max * gamma_s / gamma_1]."""
    gammas = _f64(gammas).reshape(-1)
    iters = np.ascontiguousarray(np.asarray(iters, dtype=np.int32)).reshape(-1)
    assert gammas.size == iters.size
    R, T = p.rows, int(iters.sum())
    lam = np.zeros(R) if lam0 is None else _f64(lam0).reshape(-1).copy()
    assert lam.size == R
    x = np.empty(p.nnz) if want_x else None
    sc, fg = np.empty(6), np.empty(R)
    tg, ti, t2, te = np.empty(T), np.empty(T), np.empty(T), np.empty(T)
    tgrad = np.empty((T, R)) if trace_grad else None
    tlam = np.empty((T, R)) if trace_lambda else None
    sx = np.empty((gammas.size, p.nnz)) if stage_x else None
    eq = _eq_mask(p, is_eq)
    rc = _load().dualip_oracle_solve(p.I, p.J, p.m, _ptr(p.row_ptr), _ptr(p.item_idx), _ptr(p.c), _ptr(p.a),
                                     _ptr(p.b), p.proj_kind, p.p0, p.p1, _ptr(gammas), gammas.size, _ptr(iters),
                                     1 if momentum else 0, 1 if jacobi else 0, _ptr(eq), 1 if adaptive else 0, float(eta_min),
                                     float(eta_max), 0 if p.count_M is None else 1, 0.0 if p.count_M is None else float(p.count_M),
                                     _ptr(lam), _ptr(x), _ptr(sc), _ptr(fg),
                                     _ptr(tg), _ptr(ti), _ptr(t2), _ptr(tgrad), _ptr(tlam), _ptr(te), _ptr(sx))
    if rc != 0:
        raise MemoryError("oracle solve failed")
    final = GradResult(sc[0], sc[1], sc[2], sc[3], sc[4], fg, x, sc[5])
    return SolveResult(lam, x, final, tg, ti, t2, tgrad, tlam, sx, te)
