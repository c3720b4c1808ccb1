"""ctypes binding of include/dualip.h -- argument marshalling only; every step of the path runs in the CUDA
kernels behind the C ABI.  Same names as the C entry points: Problem.create / grad / solve / set_c / info.

torch is used for device memory and streams: device tensors are passed as raw pointers, host numpy arrays
are passed as host pointers (the library stages them itself).
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

PROJ_SIMPLEX_INEQ, PROJ_BOX, PROJ_BOXCUT, PROJ_SIMPLEX_EQ = 0, 1, 2, 3
RED_AUTO, RED_SMEM, RED_GLOBAL, RED_CSC = 0, 1, 2, 3
PRECOND_NONE, PRECOND_JACOBI = 0, 1
STEP_FIXED, STEP_ADAPTIVE = 0, 1
STATIC_MAX_DUALS = 28672          # DUALIP_STATIC_MAX_DUALS of include/dualip.h: largest J*m dualip_grad_static accepts
ETOOBIG = -7
ESTALE = -8
EHOOK = -9

EXPORTED_SYMBOLS = ("dualip_opts_default", "dualip_create", "dualip_grad", "dualip_solve", "dualip_set_c",
                    "dualip_set_equality_rows", "dualip_set_global_count", "dualip_set_reduce_hook", "dualip_get_shard_extents",
                    "dualip_get_column_stats", "dualip_set_shard_constants", "dualip_eval_partial", "dualip_export_accumulators",
                    "dualip_import_accumulators", "dualip_set_profiling", "dualip_get_info", "dualip_get_csc", "dualip_destroy",
                    "dualip_strerror", "dualip_grad_static")

_HERE = os.path.dirname(os.path.abspath(__file__))


class DualipError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"dualip error {code}: {msg}")
        self.code = code


class Tuning(ctypes.Structure):
    _fields_ = [("direct_kernel", ctypes.c_int32), ("stages", ctypes.c_int32), ("tile_units", ctypes.c_int32),
                ("lambda_plan", ctypes.c_int32), ("step_deal", ctypes.c_int32)]


class Opts(ctypes.Structure):
    _fields_ = [("projection", ctypes.c_int32), ("p0", ctypes.c_double), ("p1", ctypes.c_double),
                ("reduction", ctypes.c_int32), ("borrow", ctypes.c_int32), ("validate", ctypes.c_int32),
                ("momentum", ctypes.c_int32), ("group_lanes", ctypes.c_int32), ("grid_ctas", ctypes.c_int32),
                ("use_graph", ctypes.c_int32), ("tuning", Tuning), ("precondition", ctypes.c_int32),
                ("step_rule", ctypes.c_int32), ("eta_min", ctypes.c_double), ("eta_max", ctypes.c_double)]


class Scalars(ctypes.Structure):
    _fields_ = [("g", ctypes.c_double), ("obj", ctypes.c_double), ("reg", ctypes.c_double),
                ("r_inf", ctypes.c_double), ("r_2", ctypes.c_double), ("gap", ctypes.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}

    def table4(self):
        """The fields behind the paper's solution-quality report (Table 4), selected and renamed, nothing
        computed here: the two parts of the primal objective of the ridge problem (c'x and gamma/2 |x|^2, whose sum is Table 4's
        "primal"), the dual objective, the SIGNED primal-dual gap (obj + reg) - g as the kernel's epilogue formed it (Table 4
        prints its absolute value), and the maximum positive constraint violation ("slack")."""
        return {"primal_obj": self.obj, "primal_reg": self.reg, "dual": self.g, "gap": self.gap, "slack": self.r_inf}


class ShardExtents(ctypes.Structure):
    _fields_ = [("I", ctypes.c_int64), ("nnz", ctypes.c_int64), ("max_abs_a", ctypes.c_float), ("max_abs_c", ctypes.c_float)]


# int hook(void* user, int64_t* accumulators_dev, int64_t n_words, const double* lambda_eval_dev, double gamma, void* stream)
REDUCE_HOOK = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_double, ctypes.c_void_p)


class _Trace(ctypes.Structure):
    _fields_ = [("capacity", ctypes.c_int64), ("g", ctypes.c_void_p), ("r_inf", ctypes.c_void_p),
                ("r_2", ctypes.c_void_p), ("grad", ctypes.c_void_p), ("lam", ctypes.c_void_p), ("eta", ctypes.c_void_p)]


class Info(ctypes.Structure):
    _fields_ = [("I", ctypes.c_int64), ("nnz", ctypes.c_int64), ("J", ctypes.c_int32), ("m", ctypes.c_int32),
                ("L", ctypes.c_double), ("max_row_len", ctypes.c_int64), ("group_lanes", ctypes.c_int32),
                ("chunk_regs", ctypes.c_int32), ("reduction", ctypes.c_int32), ("lambda_in_smem", ctypes.c_int32),
                ("grid_ctas", ctypes.c_int32), ("block_threads", ctypes.c_int32), ("smem_bytes", ctypes.c_int64),
                ("bytes_resident", ctypes.c_int64), ("launches", ctypes.c_int64), ("fix_scale_s", ctypes.c_double),
                ("streaming", ctypes.c_int32), ("stages", ctypes.c_int32), ("tile_units", ctypes.c_int64), ("ntiles", ctypes.c_int64),
                ("grad_kernel_ms", ctypes.c_double), ("grad_kernel_count", ctypes.c_int64),
                ("precondition", ctypes.c_int32), ("pad0", ctypes.c_int32), ("L_step", ctypes.c_double),
                ("duals", ctypes.c_int32), ("lambda_lo_smem", ctypes.c_int32), ("checked_build", ctypes.c_int32),
                ("checks_failed", ctypes.c_int32), ("long_rows", ctypes.c_int64), ("long_row_threshold", ctypes.c_int64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def lib_path() -> str:
    """The in-tree library (there is no other: no override, no fallback)."""
    return os.path.join(_HERE, "libdualip_b200.so")


_lib = None


def load_library():
    """dlopen the in-tree CUDA library; fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: run `python -m paper_2606_07777_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        lib = ctypes.CDLL(path)
        vp, i32, i64, d = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
        lib.dualip_opts_default.argtypes = [ctypes.POINTER(Opts)]
        lib.dualip_opts_default.restype = None
        lib.dualip_create.argtypes = [ctypes.POINTER(vp), i64, i32, i32, vp, vp, vp, vp, vp, ctypes.POINTER(Opts), vp]
        lib.dualip_grad.argtypes = [vp, vp, d, vp, vp, vp, vp]
        lib.dualip_solve.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, ctypes.POINTER(_Trace), vp]
        lib.dualip_set_c.argtypes = [vp, vp, vp]
        lib.dualip_set_equality_rows.argtypes = [vp, vp, vp]
        lib.dualip_set_global_count.argtypes = [vp, i32, d, vp]
        lib.dualip_set_reduce_hook.argtypes = [vp, REDUCE_HOOK, vp]
        lib.dualip_get_shard_extents.argtypes = [vp, ctypes.POINTER(ShardExtents)]
        lib.dualip_get_column_stats.argtypes = [vp, ctypes.POINTER(ShardExtents), vp, vp]
        lib.dualip_set_shard_constants.argtypes = [vp, ctypes.POINTER(ShardExtents), vp, vp]
        lib.dualip_eval_partial.argtypes = [vp, vp, d, vp, vp]
        lib.dualip_export_accumulators.argtypes = [vp, vp, i32, vp]
        lib.dualip_import_accumulators.argtypes = [vp, vp, i32, vp]
        lib.dualip_get_info.argtypes = [vp, ctypes.POINTER(Info)]
        lib.dualip_set_profiling.argtypes = [vp, ctypes.c_int]
        lib.dualip_get_csc.argtypes = [vp, vp, vp, vp]
        lib.dualip_get_csc.restype = ctypes.c_int
        lib.dualip_grad_static.argtypes = [i64, i32, i32, vp, vp, vp, vp, vp, i32, d, d, vp, d, vp, vp, vp, vp]
        lib.dualip_grad_static.restype = ctypes.c_int
        lib.dualip_destroy.argtypes = [vp]
        lib.dualip_destroy.restype = None
        lib.dualip_strerror.argtypes = [ctypes.c_int]
        lib.dualip_strerror.restype = ctypes.c_char_p
        for f in ("dualip_create", "dualip_grad", "dualip_solve", "dualip_set_c", "dualip_set_equality_rows", "dualip_set_global_count",
                  "dualip_get_info", "dualip_set_profiling", "dualip_set_reduce_hook", "dualip_get_shard_extents",
                  "dualip_get_column_stats", "dualip_set_shard_constants", "dualip_eval_partial", "dualip_export_accumulators",
                  "dualip_import_accumulators"):
            getattr(lib, f).restype = ctypes.c_int
        _lib = lib
    return _lib


def _check(rc: int):
    if rc != 0:
        raise DualipError(rc, load_library().dualip_strerror(rc).decode())


def _ptr(t, dtype=None, keep=None):
    """Raw pointer of a torch tensor (device or host) or numpy array; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        if dtype is not None and t.dtype != dtype:
            raise TypeError(f"expected {dtype}, got {t.dtype}")
        if not t.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return ctypes.c_void_p(t.ctypes.data)
    import torch
    if isinstance(t, torch.Tensor):
        if not t.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if dtype is not None and np.dtype(str(t.dtype).replace("torch.", "")) != dtype:
            raise TypeError(f"expected {dtype}, got {t.dtype}")
        return ctypes.c_void_p(t.data_ptr())
    raise TypeError(type(t))


def make_opts(projection=PROJ_SIMPLEX_INEQ, p0=1.0, p1=0.0, reduction=RED_AUTO, borrow=False, validate=True,
              momentum=True, group_lanes=0, grid_ctas=0, use_graph=False, direct_kernel=False, jacobi=False, stages=0, tile_units=0,
              adaptive=False, eta_min=1e-5, eta_max=1e-1, lambda_plan=0, step_deal=0) -> Opts:
    o = Opts()
    load_library().dualip_opts_default(ctypes.byref(o))
    o.projection, o.p0, o.p1, o.reduction = projection, p0, p1, reduction
    o.borrow, o.validate, o.momentum = int(borrow), int(validate), int(momentum)
    o.group_lanes, o.grid_ctas, o.use_graph = group_lanes, grid_ctas, int(use_graph)
    o.tuning.direct_kernel = 1 if direct_kernel else 0
    o.tuning.stages, o.tuning.tile_units, o.tuning.lambda_plan, o.tuning.step_deal = stages, tile_units, lambda_plan, step_deal
    o.precondition = PRECOND_JACOBI if jacobi else PRECOND_NONE
    o.step_rule = STEP_ADAPTIVE if adaptive else STEP_FIXED
    o.eta_min, o.eta_max = float(eta_min), float(eta_max)
    return o


def _stream_ptr(stream):
    if stream is None:
        import torch
        if torch.cuda.is_available():
            return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
        return None
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def grad_static(I, J, m, row_ptr, item_idx, c, a, b, lam, gamma: float, projection=PROJ_SIMPLEX_INEQ, p0=1.0, p1=0.0,
                grad=None, scalars=None, x=None, stream=None):
    """dualip_grad_static: one gradient evaluation with no handle and no allocation, for callers that are not allowed to
    allocate device memory where they run (include/dualip.h says who and why).  Every argument is a CUDA tensor used in place:
    row_ptr int64[I+1], item_idx int32[nnz], c fp32[nnz], a fp32[nnz*m], b fp32[J*m], lam fp64[J*m] in; grad fp64[J*m],
    scalars fp64[6] = (g, obj, reg, r_inf, r_2, gap), x fp32[nnz] out, each optional.  J*m above STATIC_MAX_DUALS raises
    DualipError with code ETOOBIG.  The outputs are ready once `stream` is; calls that overlap on the GPU race on the
    library's one scratch array, so keep them on one stream."""
    for name, t in (("row_ptr", row_ptr), ("item_idx", item_idx), ("c", c), ("a", a), ("b", b), ("lam", lam), ("grad", grad),
                    ("scalars", scalars), ("x", x)):
        if t is not None and not getattr(t, "is_cuda", False):
            raise TypeError(f"{name} must be a CUDA tensor: dualip_grad_static cannot stage host memory without allocating")
    if scalars is not None and scalars.numel() < 6:
        raise ValueError("scalars needs 6 fp64 entries")
    _check(load_library().dualip_grad_static(I, J, m, _ptr(row_ptr, np.int64), _ptr(item_idx, np.int32), _ptr(c, np.float32),
                                             _ptr(a, np.float32), _ptr(b, np.float32), int(projection), float(p0), float(p1),
                                             _ptr(lam, np.float64), float(gamma), _ptr(grad, np.float64),
                                             _ptr(scalars, np.float64), _ptr(x, np.float32), _stream_ptr(stream)))


class Problem:
    """Handle of a device-resident matching LP (dualip_t*)."""

    def __init__(self, handle, I, J, m, nnz, keep):
        self._h, self.I, self.J, self.m, self.nnz, self._keep = handle, I, J, m, nnz, keep
        self.duals = J * m          # length of lambda / grad vectors (+ 1 while the global-count row is on)

    @classmethod
    def create(cls, I, J, m, row_ptr, item_idx, c, a, b, opts: Opts | None = None, stream=None) -> "Problem":
        """dualip_create: per-user CSR rows (row_ptr int64, item_idx int32, c fp32, a fp32[nnz*m]) + b fp32[J*m];
        each array a torch tensor (CUDA or CPU) or a numpy array."""
        lib = load_library()
        h = ctypes.c_void_p()
        rc = lib.dualip_create(ctypes.byref(h), I, J, m, _ptr(row_ptr, np.int64), _ptr(item_idx, np.int32),
                               _ptr(c, np.float32), _ptr(a, np.float32), _ptr(b, np.float32),
                               ctypes.byref(opts) if opts is not None else None, _stream_ptr(stream))
        _check(rc)
        nnz = int(row_ptr[-1])
        keep = (row_ptr, item_idx, c, a) if (opts is not None and opts.borrow) else None
        return cls(h, I, J, m, nnz, keep)

    def grad(self, lam, gamma: float, grad=None, scalars=None, x=None, stream=None):
        """dualip_grad: lam fp64[J*m] in; grad fp64[J*m], x fp32[nnz] out (tensors / arrays or None).
        `scalars`: a Scalars() to fill, a 5-element fp64 device tensor, or None.  Returns `scalars`."""
        sp = ctypes.byref(scalars) if isinstance(scalars, Scalars) else _ptr(scalars, np.float64)
        if isinstance(scalars, Scalars):
            sp = ctypes.cast(sp, ctypes.c_void_p)
        self._checked(load_library().dualip_grad(self._h, _ptr(lam, np.float64), float(gamma), _ptr(grad, np.float64), sp,
                                                 _ptr(x, np.float32), _stream_ptr(stream)))
        return scalars

    def solve(self, gammas, iters, lam, x=None, scalars=None, grad=None, trace=None, stream=None):
        """dualip_solve: lam fp64[J*m] in/out.  trace: dict with optional device tensors under the keys
        'g','r_inf','r_2','eta' (fp64[T]), 'grad','lambda' (fp64[T*duals]); T = sum(iters)."""
        gam = np.ascontiguousarray(np.asarray(gammas, dtype=np.float64))
        its = np.ascontiguousarray(np.asarray(iters, dtype=np.int32))
        if gam.shape != its.shape or gam.ndim != 1:
            raise ValueError("gammas and iters must be 1-D of equal length")
        tr = None
        if trace is not None:
            tr = _Trace()
            tr.capacity = int(its.sum())
            for key, field in (("g", "g"), ("r_inf", "r_inf"), ("r_2", "r_2"), ("grad", "grad"), ("lambda", "lam"), ("eta", "eta")):
                t = trace.get(key)
                if t is not None:
                    if not t.is_cuda:
                        raise ValueError("trace buffers must be CUDA tensors")
                    need = tr.capacity * (self.duals if key in ("grad", "lambda") else 1)
                    if t.numel() < need:
                        raise ValueError(f"trace['{key}'] too small")
                    setattr(tr, field, t.data_ptr())
        sp = ctypes.byref(scalars) if isinstance(scalars, Scalars) else _ptr(scalars, np.float64)
        if isinstance(scalars, Scalars):
            sp = ctypes.cast(sp, ctypes.c_void_p)
        self._checked(load_library().dualip_solve(self._h, _ptr(gam), gam.size, _ptr(its), _ptr(lam, np.float64),
                                                  _ptr(x, np.float32), sp, _ptr(grad, np.float64),
                                                  ctypes.byref(tr) if tr is not None else None, _stream_ptr(stream)))
        return scalars

    def set_c(self, c_new, stream=None):
        _check(load_library().dualip_set_c(self._h, _ptr(c_new, np.float32), _stream_ptr(stream)))
        if self._keep is not None:
            self._keep = self._keep + (c_new,)

    def set_equality_rows(self, is_equality, stream=None):
        """dualip_set_equality_rows: uint8 mask over the J*m coupling rows (tensor / array), or None for all-inequality."""
        _check(load_library().dualip_set_equality_rows(self._h, _ptr(is_equality, np.uint8), _stream_ptr(stream)))

    def set_global_count(self, M, stream=None):
        """dualip_set_global_count: M = right-hand side of sum x <= M (one more dual at the end of every dual-sized vector),
        or None to switch the row off."""
        _check(load_library().dualip_set_global_count(self._h, 0 if M is None else 1, 0.0 if M is None else float(M), _stream_ptr(stream)))
        self.duals = self.J * self.m + (0 if M is None else 1)

    # ---- user-sharded multi-GPU (include/dualip.h, "user-sharded multi-GPU"): thin wrappers, see sharded.py ----
    @property
    def acc_words(self) -> int:
        return self.J * self.m + 3

    def set_reduce_hook(self, fn):
        """fn(acc_ptr:int, n_words:int, lam_ptr:int, gamma:float, stream:int) or None; stream is the raw cudaStream_t (0 = the
        default stream) everything fn enqueues must go to.  fn returns None / 0, or non-zero to abandon the evaluation.  An
        exception raised in fn cannot cross the C frames: it is caught here, the library is told the hook failed, and the
        grad / solve call that triggered it raises DualipError(EHOOK) from it.  The ctypes thunk is kept alive here."""
        def thunk(user, acc, n, lam, gamma, st):
            try:
                r = fn(acc, n, lam, gamma, st or 0)
                return 0 if r is None else int(r)
            except BaseException as exc:          # noqa: BLE001 -- must not propagate into the C caller
                self._hook_error = exc
                return 1
        self._hook_error = None
        self._hook = REDUCE_HOOK(thunk) if fn else REDUCE_HOOK()
        _check(load_library().dualip_set_reduce_hook(self._h, self._hook, None))

    def _checked(self, rc: int):
        """_check, chaining the exception a reduce hook raised during the call (if any)."""
        err, self._hook_error = getattr(self, "_hook_error", None), None
        if rc != 0 and err is not None:
            raise DualipError(rc, load_library().dualip_strerror(rc).decode()) from err
        _check(rc)

    def shard_extents(self) -> ShardExtents:
        e = ShardExtents()
        _check(load_library().dualip_get_shard_extents(self._h, ctypes.byref(e)))
        return e

    def column_stats(self, global_extents: ShardExtents, out, stream=None):
        _check(load_library().dualip_get_column_stats(self._h, ctypes.byref(global_extents), _ptr(out, np.int64), _stream_ptr(stream)))
        return out

    def set_shard_constants(self, global_extents: ShardExtents, summed, stream=None):
        _check(load_library().dualip_set_shard_constants(self._h, ctypes.byref(global_extents), _ptr(summed, np.int64), _stream_ptr(stream)))

    def eval_partial(self, lam, gamma: float, x=None, stream=None):
        """lam: a CUDA tensor, or a raw device pointer (int) as handed to a reduce hook."""
        lp = ctypes.c_void_p(lam) if isinstance(lam, int) else _ptr(lam, np.float64)
        _check(load_library().dualip_eval_partial(self._h, lp, float(gamma), _ptr(x, np.float32), _stream_ptr(stream)))

    def export_accumulators(self, out, clear=True, stream=None):
        _check(load_library().dualip_export_accumulators(self._h, _ptr(out, np.int64), int(clear), _stream_ptr(stream)))
        return out

    def import_accumulators(self, acc, accumulate=False, stream=None):
        _check(load_library().dualip_import_accumulators(self._h, _ptr(acc, np.int64), int(accumulate), _stream_ptr(stream)))

    def get_csc(self, col_ptr=None, perm=None, stream=None):
        """dualip_get_csc: fills col_ptr int64[J+1] and perm int64[nnz] (tensors / arrays or None)."""
        _check(load_library().dualip_get_csc(self._h, _ptr(col_ptr, np.int64), _ptr(perm, np.int64), _stream_ptr(stream)))

    def set_profiling(self, on: bool):
        _check(load_library().dualip_set_profiling(self._h, int(on)))

    def info(self) -> Info:
        inf = Info()
        _check(load_library().dualip_get_info(self._h, ctypes.byref(inf)))
        return inf

    def destroy(self):
        if self._h:
            load_library().dualip_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
