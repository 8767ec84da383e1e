"""CPU FP64 oracle for SABLE's batched NR power flow + adjoint -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import
this package.  It never imports `paper_2606_07099_b200` and shares no code with the CUDA path.
The arithmetic lives in `sable_oracle.c` (plain C, FP64, each function citing the PAPER.md passage it
follows); this file only compiles it with gcc and marshals numpy arrays through ctypes.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): 2-bus closed form, hand-derived 3-bus example
(tests/golden/), Jacobian vs central finite differences and vs the complex-matrix identities,
power balance vs branch losses, adjoint vs finite-difference sensitivities, dense vs sparse vs scipy
solves, permutation / batch-composition invariance; the implicit-layer backward (numpy, below) is pinned by finite
differences of the whole layer (tests/test_oracle_layer.py); the mixed-precision loop with inner refinement sweeps
(`nr_mixed_ir`, a Python loop over the C steps) is pinned to the C oracle's mixed mode at 0 sweeps and to the FP64 Newton
history at 3 (tests/test_oracle_pins.py).  No function of this oracle is "parity unpinned".
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sable_oracle.c")
_LIB = os.path.join(_HERE, "libsable_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-Wall", "-o", tmp,
                               _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_mismatch.restype = C.c_double
    return _lib


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _u8(a):
    return np.ascontiguousarray(a, dtype=np.uint8)


def ybus(n_bus, f, t, r, x, b):
    """Y_bus CSR from a pi-model branch list.  Returns (row_ptr, col, G, B)."""
    f, t, r, x, b = _i32(f), _i32(t), _f64(r), _f64(x), _f64(b)
    L = lib()
    nnz = L.oracle_ybus(int(n_bus), int(f.shape[0]), _p(f, C.c_int), _p(t, C.c_int), _p(r, C.c_double),
                        _p(x, C.c_double), _p(b, C.c_double), None, None, None, None)
    row_ptr = np.zeros(n_bus + 1, dtype=np.int32)
    col = np.zeros(nnz, dtype=np.int32)
    g = np.zeros(nnz)
    bb = np.zeros(nnz)
    L.oracle_ybus(int(n_bus), int(f.shape[0]), _p(f, C.c_int), _p(t, C.c_int), _p(r, C.c_double),
                  _p(x, C.c_double), _p(b, C.c_double), _p(row_ptr, C.c_int), _p(col, C.c_int),
                  _p(g, C.c_double), _p(bb, C.c_double))
    return row_ptr, col, g, bb


def index_maps(bus_type):
    bus_type = _u8(bus_type)
    nb = bus_type.shape[0]
    th = np.zeros(nb, dtype=np.int32)
    vmx = np.zeros(nb, dtype=np.int32)
    n = lib().oracle_index_maps(nb, _p(bus_type, C.c_uint8), _p(th, C.c_int), _p(vmx, C.c_int))
    return n, th, vmx


def injections(Y, vm, va):
    row_ptr, col, g, bb = Y
    vm, va = _f64(vm), _f64(va)
    nb = vm.shape[0]
    P = np.zeros(nb)
    Q = np.zeros(nb)
    lib().oracle_injections(nb, _p(row_ptr, C.c_int), _p(col, C.c_int), _p(g, C.c_double), _p(bb, C.c_double),
                            _p(vm, C.c_double), _p(va, C.c_double), _p(P, C.c_double), _p(Q, C.c_double))
    return P, Q


def mismatch(Y, bus_type, p_spec, q_spec, vm, va):
    """One scenario.  Returns (F [n] in oracle order, inf-norm, P, Q)."""
    row_ptr, col, g, bb = Y
    bus_type = _u8(bus_type)
    p_spec, q_spec, vm, va = _f64(p_spec), _f64(q_spec), _f64(vm), _f64(va)
    nb = vm.shape[0]
    n, th, vmx = index_maps(bus_type)
    F = np.zeros(max(n, 1))
    P = np.zeros(nb)
    Q = np.zeros(nb)
    r = lib().oracle_mismatch(nb, _p(row_ptr, C.c_int), _p(col, C.c_int), _p(g, C.c_double), _p(bb, C.c_double),
                              _p(bus_type, C.c_uint8), _p(p_spec, C.c_double), _p(q_spec, C.c_double),
                              _p(vm, C.c_double), _p(va, C.c_double), _p(th, C.c_int), _p(vmx, C.c_int),
                              _p(F, C.c_double), _p(P, C.c_double), _p(Q, C.c_double))
    return F[:n], r, P, Q


def jacobian(Y, bus_type, vm, va):
    """One scenario.  Returns (n, rows, cols, vals) of J1 in COO, oracle order."""
    row_ptr, col, g, bb = Y
    bus_type = _u8(bus_type)
    vm, va = _f64(vm), _f64(va)
    nb = vm.shape[0]
    n, th, vmx = index_maps(bus_type)
    P, Q = injections(Y, vm, va)
    cap = 4 * int(row_ptr[nb]) + 4 * nb
    jr = np.zeros(cap, dtype=np.int32)
    jc = np.zeros(cap, dtype=np.int32)
    jv = np.zeros(cap)
    m = lib().oracle_jacobian_coo(nb, _p(row_ptr, C.c_int), _p(col, C.c_int), _p(g, C.c_double),
                                  _p(bb, C.c_double), _p(vm, C.c_double), _p(va, C.c_double), _p(P, C.c_double),
                                  _p(Q, C.c_double), _p(th, C.c_int), _p(vmx, C.c_int), _p(jr, C.c_int),
                                  _p(jc, C.c_int), _p(jv, C.c_double))
    return n, jr[:m].copy(), jc[:m].copy(), jv[:m].copy()


def jacobian_dense(Y, bus_type, vm, va):
    n, jr, jc, jv = jacobian(Y, bus_type, vm, va)
    J = np.zeros((n, n))
    np.add.at(J, (jr, jc), jv)
    return J


def linear_solve(n, jr, jc, jv, rhs, method=0, transpose=False, mixed=False):
    jr, jc, jv = _i32(jr), _i32(jc), _f64(jv)
    x = np.array(rhs, dtype=np.float64, copy=True)
    rc = lib().oracle_linear_solve(int(n), int(jv.shape[0]), _p(jr, C.c_int), _p(jc, C.c_int), _p(jv, C.c_double),
                                   _p(x, C.c_double), int(method), int(bool(transpose)), int(bool(mixed)))
    if rc:
        raise np.linalg.LinAlgError("oracle: singular matrix")
    return x


def nr_batch(Y, bus_type, p_spec, q_spec, v_set, vm0=None, va0=None, tol=1e-8, max_it=20, method=1,
             mixed=False, n_threads=0, want_hist=False):
    """Batched Newton-Raphson.  Returns dict(vm, va, iterations, converged, final_norm, threads[, hist])."""
    row_ptr, col, g, bb = Y
    bus_type = _u8(bus_type)
    p_spec, q_spec, v_set = _f64(p_spec), _f64(q_spec), _f64(v_set)
    vm0, va0 = _f64(vm0), _f64(va0)
    batch, nb = p_spec.shape
    vm = np.zeros((batch, nb))
    va = np.zeros((batch, nb))
    it = np.zeros(batch, dtype=np.int32)
    conv = np.zeros(batch, dtype=np.uint8)
    fn = np.zeros(batch)
    hist = np.zeros((batch, max_it + 1)) if want_hist else None
    used = lib().oracle_nr_batch(nb, _p(row_ptr, C.c_int), _p(col, C.c_int), _p(g, C.c_double), _p(bb, C.c_double),
                                 _p(bus_type, C.c_uint8), batch, _p(p_spec, C.c_double), _p(q_spec, C.c_double),
                                 _p(v_set, C.c_double), _p(vm0, C.c_double), _p(va0, C.c_double),
                                 C.c_double(tol), int(max_it), int(method), int(bool(mixed)), int(n_threads),
                                 _p(vm, C.c_double), _p(va, C.c_double), _p(it, C.c_int), _p(conv, C.c_uint8),
                                 _p(fn, C.c_double), _p(hist, C.c_double))
    out = dict(vm=vm, va=va, iterations=it, converged=conv, final_norm=fn, threads=used)
    if want_hist:
        out["hist"] = hist
    return out


def nr_mixed_ir(Y, bus_type, p_spec, q_spec, v_set, tol=1e-8, max_it=20, ir_sweeps=0, method=1):
    """One scenario: Newton-Raphson whose linear solves run in FP32 (Table I: "solver copy SP") and are
    then refined by `ir_sweeps` inner sweeps (SURVEY.md section 8(c) reading 15): r = -F1 - J1 dz with J1, F1 in FP64,
    J1 c = r solved in FP32, dz += c in FP64.  Loop convention and update as oracle_nr_batch (eq. 7-8).
    Plain Python over the oracle's own mismatch / Jacobian / linear-solve steps; the FP64 product J1 dz is a numpy
    scatter-add over the COO entries.  Returns dict(vm, va, iterations, converged, final_norm, hist)."""
    bus_type = _u8(bus_type)
    p_spec, q_spec, v_set = _f64(p_spec), _f64(q_spec), _f64(v_set)
    n, th, vmx = index_maps(bus_type)
    vm = np.where(bus_type == 0, 1.0, v_set).astype(np.float64)        # PAPER.md:287 flat start; PV / slack at setpoint
    va = np.zeros_like(vm)
    hist = np.full(max_it + 1, np.nan)
    it, conv = 0, 0
    while True:
        F, r, _, _ = mismatch(Y, bus_type, p_spec, q_spec, vm, va)
        hist[it] = r
        if r <= tol:
            conv = 1
            break
        if it == max_it or not np.isfinite(r):
            break
        _, jr, jc, jv = jacobian(Y, bus_type, vm, va)
        dz = linear_solve(n, jr, jc, jv, -F, method=method, mixed=True)
        for _ in range(int(ir_sweeps)):
            res = -F.copy()
            np.subtract.at(res, jr, jv * dz[jc])                       # r = -F1 - J1 dz, FP64
            dz = dz + linear_solve(n, jr, jc, jv, res, method=method, mixed=True)
        va = va + np.where(th >= 0, dz[np.maximum(th, 0)], 0.0)
        vm = vm + np.where(vmx >= 0, dz[np.maximum(vmx, 0)], 0.0)
        it += 1
    return dict(vm=vm, va=va, iterations=it if conv else max_it, converged=conv, final_norm=r, hist=hist)


def adjoint_batch(Y, bus_type, vm, va, g_va, g_vm, method=1, mixed=False, n_threads=0):
    """J1(V)^T lambda = g per scenario.  Returns (lam_p, lam_q, threads)."""
    row_ptr, col, g, bb = Y
    bus_type = _u8(bus_type)
    vm, va, g_va, g_vm = _f64(vm), _f64(va), _f64(g_va), _f64(g_vm)
    batch, nb = vm.shape
    lp = np.zeros((batch, nb))
    lq = np.zeros((batch, nb))
    used = lib().oracle_adjoint_batch(nb, _p(row_ptr, C.c_int), _p(col, C.c_int), _p(g, C.c_double),
                                      _p(bb, C.c_double), _p(bus_type, C.c_uint8), batch, _p(vm, C.c_double),
                                      _p(va, C.c_double), _p(g_va, C.c_double), _p(g_vm, C.c_double), int(method),
                                      int(bool(mixed)), int(n_threads), _p(lp, C.c_double), _p(lq, C.c_double))
    return lp, lq, used


# ---- NEXT row 2: implicit-layer backward (eqs. 10-16) -----------------------------------------------
def full_jacobians(Y, vm, va):
    """Dense dS/dtheta and dS/dVm of S = V o conj(Ybus V) for ALL buses (complex n_bus x n_bus), by the complex-matrix
    identities  dS/dtheta = j diag(V) conj(diag(I) - Y diag(V)),  dS/dVm = diag(V) conj(Y diag(V/|V|)) + conj(diag(I)) diag(V/|V|).
    The base Jacobian of eq. (2) is made of their real / imaginary parts."""
    row_ptr, col, g, bb = Y
    nb = vm.shape[0]
    Yd = np.zeros((nb, nb), dtype=complex)
    for i in range(nb):
        sl = slice(row_ptr[i], row_ptr[i + 1])
        np.add.at(Yd[i], col[sl], g[sl] + 1j * bb[sl])
    V = vm * np.exp(1j * va)
    I = Yd @ V
    E = V / np.abs(V)
    dS_dth = 1j * np.diag(V) @ np.conj(np.diag(I) - Yd @ np.diag(V))
    dS_dvm = np.diag(V) @ np.conj(Yd @ np.diag(E)) + np.conj(np.diag(I)) @ np.diag(E)
    return dS_dth, dS_dvm


def layer_backward(Y, bus_type, vm, va, gl_pg, gl_qg, gl_vm, gl_va):
    """dL/dx of the embedded PF layer for ONE scenario at the converged (vm, va), following PAPER.md eqs. (10)-(16).

    Layer: input x = [p_g at PV buses; Vm at PV and slack buses] (eq. 3); Step 1 solves F1 = 0 for
    z1 = [Vm at PQ; theta at non-slack] (eq. 4, 6); Step 2 reads z2 = [p_g at the slack; q_g at PV and slack] off the
    unused rows (eq. 5, 9): p_g = P(V) + p_d, q_g = Q(V) + q_d.  Given the partials of a scalar loss w.r.t. the output
    buffer y -- gl_pg (used at PV and slack), gl_qg (PV and slack), gl_vm (all buses), gl_va (non-slack) -- returns
    (dx_pg [n_bus], nonzero at PV; dx_vm [n_bus], nonzero at PV and slack).

    Sign convention of this repository: F = S_calc - S_spec, so dz2/dv = +d(S_calc rows)/dv and dF1/dp_g = -1; the
    paper writes F = spec - calc, which flips the sign of lambda and of J2, J3 but not of dL/dx."""
    bus_type = np.asarray(bus_type)
    nb = vm.shape[0]
    pq = bus_type == 0
    pv = bus_type == 1
    sl = bus_type == 2
    nonslack = ~sl
    gen = pv | sl                                   # B \\ D
    dS_dth, dS_dvm = full_jacobians(Y, vm, va)
    dP_dth, dQ_dth, dP_dvm, dQ_dvm = dS_dth.real, dS_dth.imag, dS_dvm.real, dS_dvm.imag
    # eq. (11)-(12): Step-2 contribution on the voltage coordinates, v2 = (dz2/dv)^T dL/dz2
    v2_th = dP_dth[sl].T @ gl_pg[sl] + dQ_dth[gen].T @ gl_qg[gen]
    v2_vm = dP_dvm[sl].T @ gl_pg[sl] + dQ_dvm[gen].T @ gl_qg[gen]
    # eq. (13)
    g_th = np.where(nonslack, gl_va + v2_th, 0.0)
    g_vm = gl_vm + v2_vm
    # eq. (14): J1^T lambda = g_z1, unknown / equation order [theta non-slack; Vm PQ] / [P non-slack; Q PQ]
    ns, pqi = np.flatnonzero(nonslack), np.flatnonzero(pq)
    J1 = np.block([[dP_dth[np.ix_(ns, ns)], dP_dvm[np.ix_(ns, pqi)]], [dQ_dth[np.ix_(pqi, ns)], dQ_dvm[np.ix_(pqi, pqi)]]])
    lam = np.linalg.solve(J1.T, np.concatenate([g_th[ns], g_vm[pqi]]))
    lam_p = np.zeros(nb); lam_q = np.zeros(nb)
    lam_p[ns] = lam[: len(ns)]; lam_q[pqi] = lam[len(ns):]
    # eq. (15)-(16): dF1/dp_g,PV = -I on the P rows of PV buses; J3 = dF1/dVm at PV and slack buses
    dx_pg = np.where(pv, gl_pg + lam_p, 0.0)
    J3T_lam = dP_dvm[ns].T @ lam_p[ns] + dQ_dvm[pqi].T @ lam_q[pqi]
    dx_vm = np.where(gen, g_vm - J3T_lam, 0.0)
    return dx_pg, dx_vm


def full_jacobians_sparse(Y, vm, va):
    """The same complex-matrix identities as full_jacobians, as scipy.sparse matrices (for grids where the dense
    n_bus x n_bus form does not fit): dS/dtheta = j diag(V) conj(diag(I) - Y diag(V)),
    dS/dVm = diag(V) conj(Y diag(V/|V|)) + conj(diag(I)) diag(V/|V|)."""
    import scipy.sparse as sp
    row_ptr, col, g, bb = Y
    nb = vm.shape[0]
    Ys = sp.csr_matrix((g + 1j * bb, col, row_ptr), shape=(nb, nb))
    V = vm * np.exp(1j * va)
    I = Ys @ V
    E = V / np.abs(V)
    dg = lambda v: sp.diags(v, format="csr")
    dS_dth = (1j * dg(V) @ (dg(I) - Ys @ dg(V)).conj()).tocsr()
    dS_dvm = (dg(V) @ (Ys @ dg(E)).conj() + dg(np.conj(I)) @ dg(E)).tocsr()
    return dS_dth, dS_dvm


def layer_backward_sparse(Y, bus_type, vm, va, gl_pg, gl_qg, gl_vm, gl_va):
    """layer_backward (eqs. 10-16) restated line by line on scipy.sparse matrices, with the adjoint system of
    eq. (14) solved by scipy's SuperLU; for grids where the dense form is too large.  Pinned against the dense form on
    configs 1-3 and by finite differences of the whole layer on config 4 (tests/test_oracle_layer.py)."""
    import scipy.sparse as sp
    import scipy.sparse.linalg as spla
    bus_type = np.asarray(bus_type)
    nb = vm.shape[0]
    pq = bus_type == 0
    pv = bus_type == 1
    sl = bus_type == 2
    nonslack = ~sl
    gen = pv | sl
    dS_dth, dS_dvm = full_jacobians_sparse(Y, vm, va)
    dP_dth, dQ_dth, dP_dvm, dQ_dvm = dS_dth.real.tocsr(), dS_dth.imag.tocsr(), dS_dvm.real.tocsr(), dS_dvm.imag.tocsr()
    sli, geni = np.flatnonzero(sl), np.flatnonzero(gen)
    ns, pqi = np.flatnonzero(nonslack), np.flatnonzero(pq)
    # eq. (11)-(12)
    v2_th = dP_dth[sli].T @ gl_pg[sli] + dQ_dth[geni].T @ gl_qg[geni]
    v2_vm = dP_dvm[sli].T @ gl_pg[sli] + dQ_dvm[geni].T @ gl_qg[geni]
    # eq. (13)
    g_th = np.where(nonslack, gl_va + v2_th, 0.0)
    g_vm = gl_vm + v2_vm
    # eq. (14)
    J1 = sp.bmat([[dP_dth[ns][:, ns], dP_dvm[ns][:, pqi]], [dQ_dth[pqi][:, ns], dQ_dvm[pqi][:, pqi]]], format="csc")
    lam = spla.splu(J1.T.tocsc()).solve(np.concatenate([g_th[ns], g_vm[pqi]]))
    lam_p = np.zeros(nb); lam_q = np.zeros(nb)
    lam_p[ns] = lam[: len(ns)]; lam_q[pqi] = lam[len(ns):]
    # eq. (15)-(16)
    dx_pg = np.where(pv, gl_pg + lam_p, 0.0)
    J3T_lam = dP_dvm[ns].T @ lam_p[ns] + dQ_dvm[pqi].T @ lam_q[pqi]
    dx_vm = np.where(gen, g_vm - J3T_lam, 0.0)
    return dx_pg, dx_vm
