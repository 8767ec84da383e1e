"""Thin Python binding of the SABLE B200 C-ABI library (include/sable.h) -- argument marshalling only.

Every step of the path (mismatch, Jacobian fill, LU refactor, triangular solves, masking) runs in the CUDA
kernels of `csrc/`; PyTorch is used by callers for device memory and streams only.  There is no CPU fallback:
if `libsable.so` is missing, `lib()` raises.  Build it with `python -m paper_2606_07099_b200.build` (nvcc,
sm_100a) or `__graft_entry__.build()`.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsable.so")
_lib = None

PQ, PV, SLACK = 0, 1, 2
FP64, MIXED = 0, 1
FUSED, STAGED = 0, 1
STATUS = {0: "OK", 1: "INVALID_ARG", 2: "STRUCTURE", 3: "ALLOC", 4: "CUDA", 5: "STATE"}


class SableError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"sable: {STATUS.get(status, status)}: {msg}")
        self.status = status


class Tuning(C.Structure):
    _fields_ = [("group", C.c_int32), ("ctas_per_sm", C.c_int32), ("on_chip", C.c_int32), ("ring_slots", C.c_int32),
                ("ring_slot_bytes", C.c_int32), ("front_nodes", C.c_int32), ("front_kb", C.c_int32),
                ("threads_stage", C.c_int32), ("threads_lin", C.c_int32), ("timing", C.c_int32), ("cluster", C.c_int32)]


class Options(C.Structure):
    _fields_ = [("max_batch", C.c_int32), ("precision", C.c_int32), ("keep_factors", C.c_int32),
                ("mode", C.c_int32), ("device", C.c_int32), ("threads", C.c_int32), ("ir_sweeps", C.c_int32),
                ("tune", Tuning)]


class Info(C.Structure):
    _fields_ = [("n_bus", C.c_int32), ("n_pq", C.c_int32), ("n_pv", C.c_int32), ("n", C.c_int32),
                ("nnz_y", C.c_int32), ("nnz_j", C.c_int32), ("nnz_lu", C.c_int32), ("n_node", C.c_int32),
                ("n_pair", C.c_int32), ("n_pair_j", C.c_int32), ("n_level", C.c_int32),
                ("n_term", C.c_int64), ("n_term_diag", C.c_int64), ("lu_flops", C.c_int64),
                ("factor_bytes", C.c_int64), ("bytes_iter_m0", C.c_int64), ("bytes_adjoint_m0", C.c_int64),
                ("smem_bytes", C.c_int32), ("placement", C.c_int32), ("threads", C.c_int32),
                ("ctas_per_sm", C.c_int32), ("slots_per_cta", C.c_int32), ("cut_level", C.c_int32),
                ("front_k", C.c_int32), ("front_level", C.c_int32), ("threads_lin", C.c_int32), ("threads_stage", C.c_int32),
                ("cluster", C.c_int32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


EXPORTS = ["sable_create", "sable_default_options", "sable_solve", "sable_adjoint", "sable_get_pivot_flags", "sable_recover",
           "sable_layer_backward", "sable_adjoint_refined", "sable_solve_host", "sable_adjoint_host",
           "sable_get_info", "sable_last_error", "sable_destroy", "sable_launch_count", "sable_debug_pattern",
           "sable_debug_mismatch", "sable_debug_jacobian", "sable_debug_linear_solve", "sable_debug_timing",
           "sable_debug_stage_times", "sable_injections_static"]

STATIC_SCRATCH_BYTES = 8 << 20      # SABLE_STATIC_SCRATCH_BYTES of include/sable.h


def lib():
    """Load libsable.so; raises (no fallback) if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2606_07099_b200.build` (needs nvcc)")
        L = C.CDLL(LIB_PATH)
        L.sable_last_error.restype = C.c_char_p
        L.sable_last_error.argtypes = [C.c_void_p]
        L.sable_launch_count.restype = C.c_int64
        L.sable_launch_count.argtypes = [C.c_void_p]
        L.sable_destroy.restype = None
        L.sable_destroy.argtypes = [C.c_void_p]
        L.sable_default_options.restype = Options
        L.sable_default_options.argtypes = []
        _lib = L
    return _lib


def _hp(a, dtype):
    """host numpy array -> pointer (keeps a reference alive through the returned tuple)."""
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data_as(C.c_void_p)


def _dp(t, shape=None, dtype=None, device=None):
    """torch CUDA tensor (or None) -> device pointer.  With `shape` / `dtype` / `device` given the tensor is checked
    against them first: the kernels trust the boundary arrays' sizes."""
    if t is None:
        return C.c_void_p(0)
    if not (t.is_cuda and t.is_contiguous()):
        raise ValueError("device arrays must be contiguous CUDA tensors")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {tuple(t.shape)}")
    if device is not None and t.device.index != device:
        raise ValueError(f"tensor lives on cuda:{t.device.index}, the context on cuda:{device}")
    return C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Context:
    """Owns one `sable_ctx*`.  Method names follow the C calls (sable_solve -> .solve, ...)."""

    def __init__(self, n_bus, row_ptr, col_idx, y_re, y_im, bus_type, slack, max_batch=1, precision=FP64,
                 keep_factors=True, mode=FUSED, device=0, threads=0, ir_sweeps=0, **tune):
        """`tune`: fields of sable_tuning (group, ctas_per_sm, on_chip, ring_slots, ring_slot_bytes, front_nodes, front_kb,
        threads_stage, threads_lin, timing); anything not given stays automatic."""
        L = lib()
        keep = []
        ptrs = []
        for a, dt in ((row_ptr, np.int32), (col_idx, np.int32), (y_re, np.float64), (y_im, np.float64),
                      (bus_type, np.uint8)):
            arr, p = _hp(a, dt)
            keep.append(arr)
            ptrs.append(p)
        opt = L.sable_default_options()
        opt.max_batch, opt.precision, opt.keep_factors = int(max_batch), int(precision), int(bool(keep_factors))
        opt.mode, opt.device, opt.threads = int(mode), int(device), int(threads)
        opt.ir_sweeps = int(ir_sweeps)
        for k, v in tune.items():
            if not hasattr(opt.tune, k):
                raise TypeError(f"unknown tuning field {k!r}")
            setattr(opt.tune, k, int(v))
        self._h = C.c_void_p(0)
        st = L.sable_create(C.c_int32(int(n_bus)), *ptrs, C.c_int32(int(slack)), C.byref(opt), C.byref(self._h))
        if st != 0:
            raise SableError(st, (L.sable_last_error(None) or b"").decode())
        self.n_bus = int(n_bus)
        self.max_batch = int(max_batch)
        self.device = int(device)
        self.info = self.get_info()

    # -- plumbing ---------------------------------------------------------------------------------
    def _check(self, st):
        if st != 0:
            raise SableError(st, (lib().sable_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().sable_destroy(self._h)
            self._h = C.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def get_info(self) -> dict:
        info = Info()
        self._check(lib().sable_get_info(self._h, C.byref(info)))
        return info.as_dict()

    def launch_count(self) -> int:
        return int(lib().sable_launch_count(self._h))

    # -- device-pointer calls (torch CUDA tensors, float64 [batch][n_bus]) ------------------------------
    def _bn(self, t):
        """pointer of a float64 [batch][n_bus] tensor on this context's device (batch read from the first argument)."""
        return _dp(t, (self._batch, self.n_bus), self._f64, self.device)

    def _begin(self, first):
        import torch
        self._f64 = torch.float64
        self._batch = int(first.shape[0])
        return self._batch

    def solve(self, p_spec, q_spec, v_set, vm0=None, va0=None, tol=1e-8, max_it=20, out=None):
        """sable_solve.  Returns dict(vm, va, iterations, converged, final_norm) of torch CUDA tensors.
        Asynchronous on torch's current stream."""
        import torch
        batch = self._begin(p_spec)
        dev = p_spec.device
        if out is None:
            out = dict(vm=torch.empty((batch, self.n_bus), dtype=torch.float64, device=dev),
                       va=torch.empty((batch, self.n_bus), dtype=torch.float64, device=dev),
                       iterations=torch.empty(batch, dtype=torch.int32, device=dev),
                       converged=torch.empty(batch, dtype=torch.uint8, device=dev),
                       final_norm=torch.empty(batch, dtype=torch.float64, device=dev))
        self._check(lib().sable_solve(self._h, C.c_int32(batch), self._bn(p_spec), self._bn(q_spec), self._bn(v_set), self._bn(vm0),
                                      self._bn(va0), C.c_double(tol), C.c_int32(int(max_it)), self._bn(out["vm"]),
                                      self._bn(out["va"]), _dp(out["iterations"], (batch,), torch.int32, self.device),
                                      _dp(out["converged"], (batch,), torch.uint8, self.device),
                                      _dp(out["final_norm"], (batch,), torch.float64, self.device), _stream()))
        return out

    def pivot_flags(self, batch):
        """sable_get_pivot_flags of the last solve: int32 [batch], bit 0 = a tiny pivot in some refactorisation, bit 1 = in the last."""
        import torch
        flags = torch.empty(int(batch), dtype=torch.int32, device=torch.device("cuda", self.device))
        self._check(lib().sable_get_pivot_flags(self._h, C.c_int32(int(batch)), _dp(flags), _stream()))
        return flags

    def adjoint(self, g_va, g_vm, out=None):
        """sable_adjoint.  Returns (lam_p, lam_q)."""
        import torch
        batch = self._begin(g_va)
        if out is None:
            out = (torch.empty_like(g_va), torch.empty_like(g_vm))
        self._check(lib().sable_adjoint(self._h, C.c_int32(batch), self._bn(g_va), self._bn(g_vm), self._bn(out[0]), self._bn(out[1]),
                                        _stream()))
        return out

    def adjoint_refined(self, vm, va, g_va, g_vm, sweeps=2, out=None):
        """sable_adjoint_refined: the adjoint of eq. 14 with `sweeps` FP64 refinement sweeps.  Returns (lam_p, lam_q)."""
        import torch
        batch = self._begin(g_va)
        if out is None:
            out = (torch.empty_like(g_va), torch.empty_like(g_vm))
        self._check(lib().sable_adjoint_refined(self._h, C.c_int32(batch), self._bn(vm), self._bn(va), self._bn(g_va), self._bn(g_vm),
                                                C.c_int32(int(sweeps)), self._bn(out[0]), self._bn(out[1]), _stream()))
        return out

    def recover(self, vm, va, out=None):
        """sable_recover (Step-2 explicit recovery).  Returns (p_inj, q_inj): calculated net injections at every bus."""
        import torch
        batch = self._begin(vm)
        if out is None:
            out = (torch.empty_like(vm), torch.empty_like(vm))
        self._check(lib().sable_recover(self._h, C.c_int32(batch), self._bn(vm), self._bn(va), self._bn(out[0]), self._bn(out[1]), _stream()))
        return out

    def layer_backward(self, vm, va, gl_pg, gl_qg, gl_vm, gl_va, out=None):
        """sable_layer_backward (eqs. 10-16).  Returns (dx_pg, dx_vm)."""
        import torch
        batch = self._begin(vm)
        if out is None:
            out = (torch.empty_like(vm), torch.empty_like(vm))
        self._check(lib().sable_layer_backward(self._h, C.c_int32(batch), self._bn(vm), self._bn(va), self._bn(gl_pg), self._bn(gl_qg),
                                               self._bn(gl_vm), self._bn(gl_va), self._bn(out[0]), self._bn(out[1]), _stream()))
        return out

    def stage_times(self, p_spec, q_spec, v_set, reps=1):
        """sable_debug_stage_times: mean ms of the mismatch + fill launch and of the refactor + solve launch over three Newton
        iterations of the whole batch in the default workspace layout (median over `reps` calls)."""
        batch = self._begin(p_spec)
        a, b = C.c_double(0), C.c_double(0)
        ta, tb = [], []
        for _ in range(max(1, int(reps))):
            self._check(lib().sable_debug_stage_times(self._h, C.c_int32(batch), self._bn(p_spec), self._bn(q_spec), self._bn(v_set),
                                                      C.byref(a), C.byref(b), _stream()))
            ta.append(a.value)
            tb.append(b.value)
        return {"mismatch_fill_ms": float(np.median(ta)), "factor_solve_ms": float(np.median(tb))}

    # -- host-buffer calls (numpy) ----------------------------------------------------------------------
    def solve_host(self, p_spec, q_spec, v_set, vm0=None, va0=None, tol=1e-8, max_it=20, out=None):
        batch = int(p_spec.shape[0])
        if out is None:
            out = dict(vm=np.empty((batch, self.n_bus)), va=np.empty((batch, self.n_bus)),
                       iterations=np.empty(batch, dtype=np.int32), converged=np.empty(batch, dtype=np.uint8),
                       final_norm=np.empty(batch))
        hp = lambda a: C.c_void_p(0) if a is None else C.c_void_p(a.ctypes.data)
        for a in (p_spec, q_spec, v_set, vm0, va0):
            assert a is None or (a.dtype == np.float64 and a.flags.c_contiguous)
        self._check(lib().sable_solve_host(self._h, C.c_int32(batch), hp(p_spec), hp(q_spec), hp(v_set), hp(vm0),
                                           hp(va0), C.c_double(tol), C.c_int32(int(max_it)), hp(out["vm"]),
                                           hp(out["va"]), hp(out["iterations"]), hp(out["converged"]),
                                           hp(out["final_norm"])))
        return out

    def adjoint_host(self, g_va, g_vm, out=None):
        batch = int(g_va.shape[0])
        if out is None:
            out = (np.empty_like(g_va), np.empty_like(g_vm))
        for a in (g_va, g_vm):
            assert a.dtype == np.float64 and a.flags.c_contiguous
        self._check(lib().sable_adjoint_host(self._h, C.c_int32(batch), C.c_void_p(g_va.ctypes.data),
                                             C.c_void_p(g_vm.ctypes.data), C.c_void_p(out[0].ctypes.data),
                                             C.c_void_p(out[1].ctypes.data)))
        return out

    # -- debug exports ------------------------------------------------------------------------------------
    def debug_pattern(self) -> dict:
        I = self.info
        nn, npair, nt = I["n_node"], I["n_pair"], I["n_term"]
        a = dict(node_bus=np.zeros(nn, np.int32), node_level=np.zeros(nn, np.int32), pair_ptr=np.zeros(nn + 1, np.int32),
                 pair_col=np.zeros(npair, np.int32), pair_in_j=np.zeros(npair, np.uint8),
                 term_ptr=np.zeros(npair + 1, np.int32), term_a=np.zeros(nt, np.int32), term_b=np.zeros(nt, np.int32),
                 dterm_ptr=np.zeros(nn + 1, np.int32), dterm=np.zeros(npair, np.int32))
        order = ["node_bus", "node_level", "pair_ptr", "pair_col", "pair_in_j", "term_ptr", "term_a", "term_b",
                 "dterm_ptr", "dterm"]
        self._check(lib().sable_debug_pattern(self._h, *[C.c_void_p(a[k].ctypes.data) for k in order]))
        return a

    def debug_timing(self):
        """Per-phase cycle counters of CTA 0 (needs timing=1 at create).
        Returns (per_level [L][2] = accumulate / backward cycles, dict(decide_output, trips, refill_init, mismatch_norm, front_*))."""
        L = self.info["n_level"]
        buf = np.zeros(4 * L + 4, np.uint64)
        self._check(lib().sable_debug_timing(self._h, C.c_void_p(buf.ctypes.data), C.c_int32(buf.size)))
        return (buf[:4 * L].reshape(L, 4)[:, [0, 2]].astype(np.int64),
                dict(decide_output=int(buf[4 * L]), trips=int(buf[4 * L + 1]), refill_init=int(buf[4 * L + 2]),
                     mismatch_norm=int(buf[4 * L + 3]), front_assemble=int(buf[3]), front_factor=int(buf[7]) if L > 1 else 0,
                     front_backward=int(buf[11]) if L > 2 else 0))

    def debug_mismatch(self, p_spec, q_spec, vm, va):
        import torch
        batch = int(vm.shape[0])
        f_p, f_q = torch.empty_like(vm), torch.empty_like(vm)
        norm = torch.empty(batch, dtype=torch.float64, device=vm.device)
        self._check(lib().sable_debug_mismatch(self._h, C.c_int32(batch), _dp(p_spec), _dp(q_spec), _dp(vm), _dp(va),
                                               _dp(f_p), _dp(f_q), _dp(norm), _stream()))
        return f_p, f_q, norm

    def debug_jacobian(self, vm, va):
        import torch
        batch = int(vm.shape[0])
        diag = torch.empty((batch, self.info["n_node"], 4), dtype=torch.float64, device=vm.device)
        pairs = torch.empty((batch, self.info["n_pair"], 8), dtype=torch.float64, device=vm.device)
        self._check(lib().sable_debug_jacobian(self._h, C.c_int32(batch), _dp(vm), _dp(va), _dp(diag), _dp(pairs),
                                               _stream()))
        return diag, pairs

    def debug_linear_solve(self, vm, va, rhs_p, rhs_q, transpose=False):
        import torch
        batch = int(vm.shape[0])
        x_p, x_q = torch.empty_like(vm), torch.empty_like(vm)
        self._check(lib().sable_debug_linear_solve(self._h, C.c_int32(batch), _dp(vm), _dp(va), _dp(rhs_p), _dp(rhs_q),
                                                   C.c_int32(int(bool(transpose))), _dp(x_p), _dp(x_q), _stream()))
        return x_p, x_q


def sable_create(n_bus, row_ptr, col_idx, y_re, y_im, bus_type, slack, **opt) -> Context:
    return Context(n_bus, row_ptr, col_idx, y_re, y_im, bus_type, slack, **opt)


def injections_static(row_ptr, col_idx, y_re, y_im, vm, va, out=None):
    """sable_injections_static: the Step-2 recovery without a context and without any allocation inside the library (its
    scratch is a static device array of STATIC_SCRATCH_BYTES shared by all calls -- calls that overlap on the GPU race).
    Everything is a CUDA tensor on the current device: Y_bus CSR (int32 row_ptr [n_bus+1], int32 col_idx, float64 y_re, y_im),
    vm, va [batch][n_bus] float64.  Returns (p_inj, q_inj); pass `out` to keep the call free of torch allocations too."""
    import torch
    n_bus, batch = int(row_ptr.shape[0]) - 1, int(vm.shape[0])
    dv = torch.cuda.current_device()
    if out is None:
        out = (torch.empty_like(vm), torch.empty_like(vm))
    nnz = tuple(col_idx.shape)
    err = C.create_string_buffer(512)
    st = lib().sable_injections_static(
        C.c_int32(n_bus), C.c_int32(batch), _dp(row_ptr, (n_bus + 1,), torch.int32, dv), _dp(col_idx, nnz, torch.int32, dv),
        _dp(y_re, nnz, torch.float64, dv), _dp(y_im, nnz, torch.float64, dv), _dp(vm, (batch, n_bus), torch.float64, dv),
        _dp(va, (batch, n_bus), torch.float64, dv), _dp(out[0], (batch, n_bus), torch.float64, dv),
        _dp(out[1], (batch, n_bus), torch.float64, dv), _stream(), err, C.c_int32(len(err)))
    if st != 0:
        raise SableError(st, err.value.decode())
    return out
