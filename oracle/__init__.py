"""ORACLE — TEST INFRASTRUCTURE ONLY (ctypes loader for oracle/oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It shares no code with paper_2601_21310_b200 and never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "oracle.cpp")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.cpp with g++ (no FMA contraction so the Q7 evaluation order is what the source says)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                               _SRC, "-o", _SO])
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        dp, up, ip = C.POINTER(C.c_double), C.POINTER(C.c_uint64), C.POINTER(C.c_int64)
        L.orc_diagonal.restype = C.c_double
        L.orc_diagonal.argtypes = [C.c_int, dp, dp, C.c_double, up]
        L.orc_element.restype = C.c_double
        L.orc_element.argtypes = [C.c_int, dp, dp, C.c_double, up, up]
        L.orc_connections.restype = C.c_int64
        L.orc_connections.argtypes = [C.c_int, dp, dp, C.c_double, up, C.c_double, up, dp, C.c_int64, ip]
        L.orc_dense.restype = None
        L.orc_dense.argtypes = [C.c_int, dp, dp, C.c_double, up, C.c_int64, dp]
        L.orc_zobrist.restype = C.c_uint64
        L.orc_zobrist.argtypes = [up]
        L.orc_ham_build.restype = C.c_void_p
        L.orc_ham_build.argtypes = [C.c_int, dp, dp, C.c_double, up, C.c_int64, C.c_double, ip, C.c_int64]
        L.orc_csr_nnz.restype = C.c_int64
        L.orc_csr_nnz.argtypes = [C.c_void_p]
        L.orc_csr_copy.restype = None
        L.orc_csr_copy.argtypes = [C.c_void_p, ip, C.POINTER(C.c_int32), dp]
        L.orc_csr_free.restype = None
        L.orc_csr_free.argtypes = [C.c_void_p]
        L.orc_energy.restype = None
        L.orc_energy.argtypes = [C.c_int64, ip, C.POINTER(C.c_int32), dp, dp, dp, dp, dp]
        L.orc_residual.restype = None
        L.orc_residual.argtypes = [C.c_int64, ip, C.POINTER(C.c_int32), dp, dp, C.c_double, dp, dp]
        L.orc_pt2.restype = None
        L.orc_pt2.argtypes = [C.c_int, dp, dp, C.c_double, up, C.c_int64, dp, C.c_double, C.c_double, C.c_int,
                              C.c_int, C.c_int, dp, ip, ip, dp, dp, dp]
        L.orc_expand.restype = C.c_int64
        L.orc_expand.argtypes = [C.c_int, dp, dp, C.c_double, up, C.c_int64, dp, C.c_double, up, dp, dp, dp, C.c_int64]
        L.orc_hsp_build.restype = C.c_void_p
        L.orc_hsp_build.argtypes = [C.c_int, dp, dp, C.c_double, up, C.c_int64, dp, C.c_double, up, C.c_int64]
        L.orc_use_lists.restype = C.c_int
        L.orc_use_lists.argtypes = [C.c_int]
        L.orc_complete_sum.restype = None
        L.orc_complete_sum.argtypes = [C.c_int, dp, dp, C.c_double, up, C.c_int64, dp, up, C.c_int64, dp]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _u(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint64))


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _u64(a):
    return np.ascontiguousarray(a, dtype=np.uint64)


def num_threads() -> int:
    return lib().orc_num_threads()


def diagonal(n, h1, eri, e_core, det) -> float:
    h1, eri, det = _f64(h1), _f64(eri), _u64(det)
    return lib().orc_diagonal(n, _d(h1), _d(eri), e_core, _u(det))


def element(n, h1, eri, e_core, x, y) -> float:
    h1, eri, x, y = _f64(h1), _f64(eri), _u64(x), _u64(y)
    return lib().orc_element(n, _d(h1), _d(eri), e_core, _u(x), _u(y))


def dense(n, h1, eri, e_core, dets):
    """Dense matrix <D_r|H|D_c> over `dets` via element() (pins only)."""
    h1, eri, dets = _f64(h1), _f64(eri), _u64(dets)
    nd = dets.shape[0]
    out = np.empty((nd, nd), dtype=np.float64)
    lib().orc_dense(n, _d(h1), _d(eri), e_core, _u(dets), nd, _d(out))
    return out


def zobrist(det) -> int:
    det = _u64(det)
    return lib().orc_zobrist(_u(det))


def connections(n, h1, eri, e_core, det, tau):
    """Sorted screened connection list of one source: (keys uint64 [m,2], h fp64 [m], visited)."""
    h1, eri, det = _f64(h1), _f64(eri), _u64(det)
    vis = C.c_int64(0)
    cap = 1 << 12
    while True:
        keys = np.empty((cap, 2), dtype=np.uint64)
        hv = np.empty(cap, dtype=np.float64)
        m = lib().orc_connections(n, _d(h1), _d(eri), e_core, _u(det), tau, _u(keys), _d(hv), cap, C.byref(vis))
        if m <= cap:
            return keys[:m].copy(), hv[:m].copy(), vis.value
        cap = int(m)


def ham_build(n, h1, eri, e_core, dets, eps, rows=None):
    """CSR H_SS: (row_ptr int64 [|S|+1], col int32 [nnz], val fp64 [nnz]).  rows: optional subset of rows to build."""
    h1, eri, dets = _f64(h1), _f64(eri), _u64(dets)
    nd = dets.shape[0]
    if rows is None:
        hnd = lib().orc_ham_build(n, _d(h1), _d(eri), e_core, _u(dets), nd, eps, None, 0)
    else:
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        hnd = lib().orc_ham_build(n, _d(h1), _d(eri), e_core, _u(dets), nd, eps, _i(rows), rows.shape[0])
    nnz = lib().orc_csr_nnz(hnd)
    row_ptr = np.empty(nd + 1, dtype=np.int64)
    col = np.empty(nnz, dtype=np.int32)
    val = np.empty(nnz, dtype=np.float64)
    lib().orc_csr_copy(hnd, _i(row_ptr), col.ctypes.data_as(C.POINTER(C.c_int32)), _d(val))
    lib().orc_csr_free(hnd)
    return row_ptr, col, val


def energy(row_ptr, col, val, psi, want_y=False):
    """(E_S, psi^T psi[, y = H psi])."""
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col = np.ascontiguousarray(col, dtype=np.int32)
    val, psi = _f64(val), _f64(psi)
    nd = psi.shape[0]
    e, n2 = C.c_double(0), C.c_double(0)
    y = np.empty(nd, dtype=np.float64)
    lib().orc_energy(nd, _i(row_ptr), col.ctypes.data_as(C.POINTER(C.c_int32)), _d(val), _d(psi), C.byref(e),
                     C.byref(n2), _d(y))
    return (e.value, n2.value, y) if want_y else (e.value, n2.value)


def ediag(row_ptr, col, val):
    """E_diag = lambda_min(H_VV) ("diagnostic post-hoc diagonalization energy").  The plain definition through
    a library eigensolver: LAPACK on the dense matrix up to 4000 rows, ARPACK (scipy eigsh, smallest algebraic) beyond."""
    import scipy.sparse as sp
    nd = len(row_ptr) - 1
    A = sp.csr_matrix((_f64(val), np.ascontiguousarray(col, dtype=np.int32), np.ascontiguousarray(row_ptr, dtype=np.int64)),
                      shape=(nd, nd))
    if nd <= 4000:
        return float(np.linalg.eigvalsh(A.toarray())[0])
    from scipy.sparse.linalg import eigsh
    w = eigsh(A, k=1, which="SA", tol=1e-13, maxiter=20000, return_eigenvectors=False)
    return float(w[0])


def expand(n, h1, eri, e_core, dets, psi, eps2):
    """Perturbative set P of Eq. 14: (keys [|P|, 2] sorted ascending, score = max_i |H_ai psi_i|, v = sum_i H_ai psi_i, H_aa)."""
    h1, eri, dets, psi = _f64(h1), _f64(eri), _u64(dets), _f64(psi)
    m = lib().orc_expand(n, _d(h1), _d(eri), e_core, _u(dets), dets.shape[0], _d(psi), eps2, None, None, None, None, 0)
    keys = np.zeros((m, 2), dtype=np.uint64)
    score, v, haa = np.zeros(m), np.zeros(m), np.zeros(m)
    if m:
        lib().orc_expand(n, _d(h1), _d(eri), e_core, _u(dets), dets.shape[0], _d(psi), eps2, _u(keys), _d(score), _d(v), _d(haa), m)
    return keys, score, v, haa


def use_lists(on):
    """Switch conn(D, tau) in connections / ham_build / pt2 between the plain definition (False, the default every parity test
    uses) and the paper's CPU algorithm - per-pair lists sorted by magnitude, walked with the early exit - which
    is only the second timed CPU baseline of bench.py.  Returns the previous setting."""
    return bool(lib().orc_use_lists(1 if on else 0))


def complete_sum(n, h1, eri, e_core, dets, psi, pkeys):
    """v_a = sum over ALL i in V of H_ai psi_i (the full <x|H|Psi_V> of Eq. 13) for the sorted key list `pkeys`."""
    h1, eri, dets, psi, pkeys = _f64(h1), _f64(eri), _u64(dets), _f64(psi), _u64(pkeys)
    v = np.zeros(pkeys.shape[0])
    if pkeys.shape[0]:
        lib().orc_complete_sum(n, _d(h1), _d(eri), e_core, _u(dets), dets.shape[0], _d(psi), _u(pkeys), pkeys.shape[0], _d(v))
    return v


def hsp_build(n, h1, eri, e_core, dets, psi, eps2, pkeys):
    """CSR H_VP (rows = determinants of V, columns = indices into the sorted key list `pkeys`), couplings screened by
    tau_i = eps2 / |psi_i| as in expand(); (row_ptr int64 [nd+1], col int32 [nnz], val fp64 [nnz])."""
    h1, eri, dets, psi, pkeys = _f64(h1), _f64(eri), _u64(dets), _f64(psi), _u64(pkeys)
    nd = dets.shape[0]
    hnd = lib().orc_hsp_build(n, _d(h1), _d(eri), e_core, _u(dets), nd, _d(psi), eps2, _u(pkeys), pkeys.shape[0])
    nnz = lib().orc_csr_nnz(hnd)
    row_ptr = np.empty(nd + 1, dtype=np.int64)
    col = np.empty(nnz, dtype=np.int32)
    val = np.empty(nnz, dtype=np.float64)
    lib().orc_csr_copy(hnd, _i(row_ptr), col.ctypes.data_as(C.POINTER(C.c_int32)), _d(val))
    lib().orc_csr_free(hnd)
    return row_ptr, col, val


def residual(row_ptr, col, val, psi, e_s):
    """(r = H_SS psi - e_s psi, internal term of Eq. 13 = sum_i r_i^2 / (e_s - H_ii) / psi^T psi)."""
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col = np.ascontiguousarray(col, dtype=np.int32)
    val, psi = _f64(val), _f64(psi)
    nd = psi.shape[0]
    r = np.empty(nd, dtype=np.float64)
    out = C.c_double(0)
    lib().orc_residual(nd, _i(row_ptr), col.ctypes.data_as(C.POINTER(C.c_int32)), _d(val), _d(psi), float(e_s), _d(r),
                       C.byref(out))
    return r, out.value


def pt2(n, h1, eri, e_core, dets, psi, e_s, eps2, n_parts=1, part_begin=0, part_end=None):
    """dict(pt2, n_external, n_contrib, part_sums, sum_abs, min_abs_den) over classes [part_begin, part_end)."""
    h1, eri, dets, psi = _f64(h1), _f64(eri), _u64(dets), _f64(psi)
    if part_end is None:
        part_end = n_parts
    out, sabs, mden = C.c_double(0), C.c_double(0), C.c_double(0)
    next_, ncon = C.c_int64(0), C.c_int64(0)
    ps = np.zeros(n_parts, dtype=np.float64)
    lib().orc_pt2(n, _d(h1), _d(eri), e_core, _u(dets), dets.shape[0], _d(psi), e_s, eps2, n_parts, part_begin,
                  part_end, C.byref(out), C.byref(next_), C.byref(ncon), _d(ps), C.byref(sabs), C.byref(mden))
    return dict(pt2=out.value, n_external=next_.value, n_contrib=ncon.value, part_sums=ps, sum_abs=sabs.value,
                min_abs_den=mden.value)
