from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_PKG, "libdetham.so")
_lib = None

STATUS = {0: "DH_OK", 1: "DH_EINVAL", 2: "DH_EUNSORTED", 3: "DH_EPOPCOUNT", 4: "DH_ENOMEM", 5: "DH_ETABLEFULL", 6: "DH_ECUDA"}

# every symbol include/detham.h declares
SYMBOLS = ["detham_create", "detham_set_subspace", "detham_ham_build", "detham_build_config", "detham_csr", "detham_csr_copy", "detham_energy", "detham_energy_static", "detham_energy_static_error", "detham_residual", "detham_ediag",
           "detham_pt2_config", "detham_pt2_set_options", "detham_trim", "detham_count_screened", "detham_pt2", "detham_expand", "detham_hsp_build", "detham_complete_sum", "detham_hsp_csr", "detham_hsp_csr_copy", "detham_pt2_partials", "detham_solve_host", "detham_connections",
           "detham_diagonals", "detham_get_counters", "detham_destroy", "detham_strerror", "detham_last_cuda_error"]


class Counters(C.Structure):
    _fields_ = [("nnz", C.c_int64), ("build_generated", C.c_int64), ("pt2_generated", C.c_int64),
                ("pt2_contrib", C.c_int64), ("pt2_external", C.c_int64), ("pt2_parts", C.c_int32),
                ("pt2_max_probe", C.c_int32), ("pt2_table_slots", C.c_int64), ("pt2_probe_parts", C.c_int64), ("pt2_sum_abs", C.c_double),
                ("pt2_min_abs_den", C.c_double), ("ms_store", C.c_double), ("ms_build_count", C.c_double),
                ("ms_build_fill", C.c_double), ("ms_energy", C.c_double), ("ms_pt2_plan", C.c_double),
                ("ms_pt2_accum", C.c_double), ("ms_pt2_scan", C.c_double),
                ("hsp_nnz", C.c_int64), ("hsp_generated", C.c_int64), ("ms_hsp_build", C.c_double),
                ("ms_hsp_fill", C.c_double), ("pt2_binned", C.c_int64), ("pt2_stream_bins", C.c_int64), ("build_pairs", C.c_int64)]


class Pt2Options(C.Structure):
    """detham_pt2_options (include/detham.h); zero in every field = the defaults."""
    _fields_ = [("mode", C.c_int32), ("n_parts", C.c_int32), ("table_slots", C.c_int64), ("table_load", C.c_double),
                ("max_table_gb", C.c_double), ("small_den", C.c_double), ("stream_bins", C.c_int32), ("table_regions", C.c_int32),
                ("stream_ring_mb", C.c_double), ("stream_load", C.c_double), ("stream_pool_frac", C.c_double),
                ("stream_pool_gb", C.c_double)]

MODES = {"auto": 0, "table": 1, "stream": 2}


class DethamError(RuntimeError):
    def __init__(self, status, text, cuda=""):
        self.status = STATUS.get(status, str(status))
        super().__init__(f"{self.status}: {text}" + (f" [{cuda}]" if cuda else ""))


def use_checked_library():
    """Make this process load libdetham_checked.so (the same sources built with -DDETHAM_CHECKED: device asserts at every
    computed index).  Call before the first context is created."""
    global _SO
    if _lib is not None:
        raise RuntimeError("the library is already loaded")
    _SO = os.path.join(_PKG, "libdetham_checked.so")


def load_library():
    """dlopen the in-tree libdetham.so (built by paper_2601_21310_b200.build).  Fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise ImportError(f"{_SO} not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    L = C.CDLL(_SO)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)
    L.detham_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, vp, vp, C.c_double, vp]
    L.detham_set_subspace.argtypes = [vp, vp, C.c_int64]
    L.detham_ham_build.argtypes = [vp, C.c_double, ip]
    L.detham_build_config.argtypes = [vp, C.c_int]
    L.detham_csr.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    L.detham_csr_copy.argtypes = [vp, vp, vp, vp]
    L.detham_energy.argtypes = [vp, vp, dp, dp, vp]
    L.detham_energy_static.argtypes = [vp, vp, vp, vp, C.c_int64, C.c_int64, vp, vp, vp]
    L.detham_energy_static_error.argtypes = []
    L.detham_energy_static_error.restype = C.c_char_p
    L.detham_residual.argtypes = [vp, vp, C.c_double, vp, dp]
    L.detham_ediag.argtypes = [vp, vp, C.c_double, C.c_int, dp, C.POINTER(C.c_int), dp, C.POINTER(C.c_int)]
    L.detham_pt2_config.argtypes = [vp, C.c_int64, C.c_int]
    L.detham_pt2_set_options.argtypes = [vp, C.POINTER(Pt2Options)]
    L.detham_trim.argtypes = [vp]
    L.detham_count_screened.argtypes = [vp, vp, C.c_double, ip]
    L.detham_pt2.argtypes = [vp, vp, C.c_double, C.c_double, dp, ip, ip]
    L.detham_expand.argtypes = [vp, vp, C.c_double, vp, vp, vp, vp, C.c_int64, ip]
    L.detham_hsp_build.argtypes = [vp, vp, C.c_double, vp, C.c_int64, ip]
    L.detham_complete_sum.argtypes = [vp, vp, vp, C.c_int64, vp]
    L.detham_hsp_csr.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    L.detham_hsp_csr_copy.argtypes = [vp, vp, vp, vp]
    L.detham_pt2_partials.argtypes = [vp, dp, C.c_int, C.POINTER(C.c_int)]
    L.detham_solve_host.argtypes = [vp, vp, vp, C.c_int64, C.c_double, C.c_double, dp, dp, ip, ip]
    L.detham_connections.argtypes = [vp, C.c_int64, C.c_double, vp, vp, C.c_int64, ip]
    L.detham_diagonals.argtypes = [vp, vp, C.c_int64, vp]
    L.detham_get_counters.argtypes = [vp, C.POINTER(Counters)]
    L.detham_destroy.argtypes = [vp]
    L.detham_destroy.restype = None
    L.detham_strerror.argtypes = [C.c_int]
    L.detham_strerror.restype = C.c_char_p
    L.detham_last_cuda_error.argtypes = [vp]
    L.detham_last_cuda_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name not in ("detham_destroy", "detham_strerror", "detham_last_cuda_error", "detham_energy_static_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _dev_u64(t):
    """torch CUDA tensor holding [m, 2] 64-bit words (int64 or uint64 bit patterns) -> (pointer, m)."""
    import torch
    assert t.is_cuda and t.is_contiguous() and t.dtype in (torch.int64, torch.uint64) and t.dim() == 2 and t.shape[1] == 2
    return t.data_ptr(), t.shape[0]


class Detham:
    """One context = one integral set on one GPU.  Method names follow include/detham.h."""

    def __init__(self, n_orb, n_alpha, n_beta, h1, eri, e_core=0.0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise DethamError(6, "no CUDA device: the detham hot path has no CPU fallback")
        self._L = load_library()
        self._h = C.c_void_p()
        self.n_orb, self.n_alpha, self.n_beta = n_orb, n_alpha, n_beta
        h1 = np.ascontiguousarray(h1, dtype=np.float64)
        eri = np.ascontiguousarray(eri, dtype=np.float64)
        npair = n_orb * (n_orb + 1) // 2
        if h1.size != n_orb * n_orb or eri.size != npair * (npair + 1) // 2:
            raise DethamError(1, "h1 / eri have the wrong size")
        self._stream = stream
        sp = C.c_void_p(stream.cuda_stream) if stream is not None else None
        self._check(self._L.detham_create(C.byref(self._h), n_orb, n_alpha, n_beta, h1.ctypes.data, eri.ctypes.data,
                                          float(e_core), sp))
        self._dets = None
        self.n_dets = 0

    def _check(self, st):
        if st != 0:
            cuda = self._L.detham_last_cuda_error(self._h).decode() if self._h else ""
            raise DethamError(st, self._L.detham_strerror(st).decode(), cuda)

    def set_subspace(self, dets):
        """dets: torch CUDA tensor [|S|, 2] int64/uint64 (alpha, beta words), or a numpy uint64 array (uploaded)."""
        import torch
        if isinstance(dets, np.ndarray):
            dets = torch.from_numpy(np.ascontiguousarray(dets, dtype=np.uint64).view(np.int64)).cuda()
        ptr, m = _dev_u64(dets)
        self._dets = dets  # keep the borrowed buffer alive
        self._check(self._L.detham_set_subspace(self._h, ptr, m))
        self.n_dets = m
        self._last_external = 0

    def build_config(self, method=0):
        """How ham_build finds connections: 0 library's choice, 1 heat-bath list walk, 2 by excitation degree (pairs of S)."""
        self._check(self._L.detham_build_config(self._h, int(method)))

    def ham_build(self, eps):
        nnz = C.c_int64(0)
        self._check(self._L.detham_ham_build(self._h, float(eps), C.byref(nnz)))
        self.nnz = nnz.value
        return nnz.value

    def csr(self):
        """(row_ptr int64 [|S|+1], col int32 [nnz], val fp64 [nnz]) as new torch CUDA tensors (device-to-device copy)."""
        import torch
        rp = torch.empty(self.n_dets + 1, dtype=torch.int64, device="cuda")
        col = torch.empty(self.nnz, dtype=torch.int32, device="cuda")
        val = torch.empty(self.nnz, dtype=torch.float64, device="cuda")
        self._check(self._L.detham_csr_copy(self._h, rp.data_ptr(), col.data_ptr(), val.data_ptr()))
        return rp, col, val

    def csr_pointers(self):
        a, b, c = C.c_void_p(), C.c_void_p(), C.c_void_p()
        self._check(self._L.detham_csr(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return a.value, b.value, c.value

    def energy(self, psi, want_y=False):
        import torch
        assert psi.is_cuda and psi.dtype == torch.float64 and psi.is_contiguous() and psi.numel() == self.n_dets
        e, n2 = C.c_double(0), C.c_double(0)
        y = torch.empty_like(psi) if want_y else None
        self._check(self._L.detham_energy(self._h, psi.data_ptr(), C.byref(e), C.byref(n2), y.data_ptr() if want_y else None))
        return (e.value, n2.value, y) if want_y else (e.value, n2.value)

    def residual(self, psi, e_s, want_r=True):
        """(r = H_SS psi - e_s psi as a CUDA tensor or None, internal term of Eq. 13)."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.float64 and psi.is_contiguous() and psi.numel() == self.n_dets
        out = C.c_double(0)
        r = torch.empty_like(psi) if want_r else None
        self._check(self._L.detham_residual(self._h, psi.data_ptr(), float(e_s), r.data_ptr() if want_r else None, C.byref(out)))
        return r, out.value

    def ediag(self, v0=None, tol=1e-12, max_iter=500):
        """(E_diag = lambda_min(H_SS), Lanczos steps taken).  `self.ediag_residual` = residual norm of the Ritz pair returned,
        `self.ediag_converged` = whether the stopping rule of include/detham.h was met (False: max_iter reached; a warning is
        issued, the value is an upper bound only)."""
        import torch
        if v0 is not None:
            assert v0.is_cuda and v0.dtype == torch.float64 and v0.is_contiguous() and v0.numel() == self.n_dets
        e, it, res, conv = C.c_double(0), C.c_int(0), C.c_double(0), C.c_int(0)
        self._check(self._L.detham_ediag(self._h, v0.data_ptr() if v0 is not None else None, float(tol), int(max_iter),
                                         C.byref(e), C.byref(it), C.byref(res), C.byref(conv)))
        self.ediag_residual, self.ediag_converged = res.value, bool(conv.value)
        if not self.ediag_converged:
            import warnings
            warnings.warn(f"detham_ediag: not converged after {it.value} steps (residual {res.value:.3g})")
        return e.value, it.value

    def expand(self, psi, eps2):
        """Perturbative set P of Eq. 14 as CUDA tensors: (keys int64 [|P|, 2] sorted, score, v, H_aa).

        The buffers are sized from the external count of the last pt2() on this context when there is one (same S: the usual
        case, one enumeration); otherwise, or if that was too small, a sizing call (cap = 0) runs first."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.float64 and psi.is_contiguous() and psi.numel() == self.n_dets
        m = C.c_int64(0)
        cap = int(getattr(self, "_last_external", 0))
        for _ in range(3):
            keys = torch.empty((cap, 2), dtype=torch.int64, device=psi.device)
            score, v, haa = (torch.empty(cap, dtype=torch.float64, device=psi.device) for _ in range(3))
            st = self._L.detham_expand(self._h, psi.data_ptr(), float(eps2), keys.data_ptr() if cap else None,
                                       score.data_ptr() if cap else None, v.data_ptr() if cap else None,
                                       haa.data_ptr() if cap else None, cap, C.byref(m))
            if st == 0:
                n = m.value
                return keys[:n], score[:n], v[:n], haa[:n]
            if st == 1 and m.value > cap:      # DH_EINVAL with *n_out set: the set needs m.value entries
                cap = m.value
                del keys, score, v, haa
                continue
            self._check(st)
        raise DethamError(1, "detham_expand did not settle on a buffer size")

    def hsp_build(self, psi, eps2, pkeys):
        """H_SP in CSR against the sorted key list `pkeys` (CUDA [m, 2] int64/uint64, e.g. expand()'s keys); returns nnz."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.float64 and psi.is_contiguous() and psi.numel() == self.n_dets
        ptr, m = _dev_u64(pkeys)
        nnz = C.c_int64(0)
        self._check(self._L.detham_hsp_build(self._h, psi.data_ptr(), float(eps2), ptr if m else None, m, C.byref(nnz)))
        self.hsp_nnz = nnz.value
        return nnz.value

    def complete_sum(self, psi, pkeys):
        """v_a = sum over ALL i in S of H_ai psi_i (the full <x|H|Psi_V> of Eq. 13) for the sorted CUDA key tensor `pkeys` [m, 2]."""
        import torch
        assert psi.is_cuda and psi.dtype == torch.float64 and psi.is_contiguous() and psi.numel() == self.n_dets
        ptr, m = _dev_u64(pkeys) if pkeys.numel() else (None, 0)
        v = torch.empty(m, dtype=torch.float64, device="cuda")
        self._check(self._L.detham_complete_sum(self._h, psi.data_ptr(), ptr, m, v.data_ptr() if m else None))
        return v

    def hsp_csr(self):
        """(row_ptr int64 [|S|+1], col int32 [nnz], val fp64 [nnz]) of H_SP as new torch CUDA tensors."""
        import torch
        rp = torch.empty(self.n_dets + 1, dtype=torch.int64, device="cuda")
        col = torch.empty(self.hsp_nnz, dtype=torch.int32, device="cuda")
        val = torch.empty(self.hsp_nnz, dtype=torch.float64, device="cuda")
        self._check(self._L.detham_hsp_csr_copy(self._h, rp.data_ptr(), col.data_ptr(), val.data_ptr()))
        return rp, col, val

    def pt2_config(self, table_slots=0, n_parts=0):
        self._check(self._L.detham_pt2_config(self._h, int(table_slots), int(n_parts)))

    def pt2_set_options(self, **kw):
        """Set every option of pt2 (detham_pt2_options); fields not named go back to their defaults.  mode: "auto" | "table" |
        "stream" or 0 | 1 | 2.  No arguments = all defaults."""
        o = Pt2Options()
        for k, v in kw.items():
            if k == "mode" and isinstance(v, str):
                v = MODES[v]
            if not hasattr(o, k):
                raise DethamError(1, f"unknown pt2 option {k}")
            setattr(o, k, v)
        self._check(self._L.detham_pt2_set_options(self._h, C.byref(o)))

    def count_screened(self, thr, psi=None):
        """Size of the screened connection lists summed over the sources (psi None: tau = thr; else tau_i = thr / |psi_i|)."""
        n = C.c_int64(0)
        self._check(self._L.detham_count_screened(self._h, psi.data_ptr() if psi is not None else None, float(thr), C.byref(n)))
        return n.value

    def trim(self):
        self._check(self._L.detham_trim(self._h))

    def pt2(self, psi, e_s, eps2):
        import torch
        assert psi.is_cuda and psi.dtype == torch.float64 and psi.is_contiguous() and psi.numel() == self.n_dets
        out = C.c_double(0)
        ne, nc = C.c_int64(0), C.c_int64(0)
        self._check(self._L.detham_pt2(self._h, psi.data_ptr(), float(e_s), float(eps2), C.byref(out), C.byref(ne), C.byref(nc)))
        self._last_external = ne.value
        return out.value, ne.value, nc.value

    def pt2_partials(self):
        buf = (C.c_double * 1024)()
        m = C.c_int(0)
        self._check(self._L.detham_pt2_partials(self._h, buf, 1024, C.byref(m)))
        return np.array(buf[: m.value])

    def solve_host(self, dets_host, psi_host, eps, eps2):
        """Whole path from HOST numpy buffers: returns (E_S, PT2, nnz, n_external)."""
        dets_host = np.ascontiguousarray(dets_host, dtype=np.uint64)
        psi_host = np.ascontiguousarray(psi_host, dtype=np.float64)
        e, p = C.c_double(0), C.c_double(0)
        nnz, ne = C.c_int64(0), C.c_int64(0)
        self._check(self._L.detham_solve_host(self._h, dets_host.ctypes.data, psi_host.ctypes.data, dets_host.shape[0],
                                              float(eps), float(eps2), C.byref(e), C.byref(p), C.byref(nnz), C.byref(ne)))
        self.n_dets, self.nnz = dets_host.shape[0], nnz.value
        return e.value, p.value, nnz.value, ne.value

    def connections(self, row, tau):
        n, na, nb = self.n_orb, self.n_alpha, self.n_beta
        c2 = lambda x: x * (x - 1) // 2
        cap = na * (n - na) + nb * (n - nb) + c2(na) * c2(n - na) + c2(nb) * c2(n - nb) + na * nb * (n - na) * (n - nb)
        keys = np.empty((max(cap, 1), 2), dtype=np.uint64)
        h = np.empty(max(cap, 1), dtype=np.float64)
        m = C.c_int64(0)
        self._check(self._L.detham_connections(self._h, int(row), float(tau), keys.ctypes.data, h.ctypes.data, cap, C.byref(m)))
        return keys[: m.value].copy(), h[: m.value].copy()

    def diagonals(self, dets):
        import torch
        ptr, m = _dev_u64(dets)
        out = torch.empty(m, dtype=torch.float64, device="cuda")
        self._check(self._L.detham_diagonals(self._h, ptr, m, out.data_ptr()))
        return out

    def counters(self):
        c = Counters()
        self._check(self._L.detham_get_counters(self._h, C.byref(c)))
        return {f[0]: getattr(c, f[0]) for f in Counters._fields_}

    def close(self):
        if self._h:
            self._L.detham_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


ENERGY_STATIC_MAX_ROWS = 8388608  # DETHAM_ENERGY_STATIC_MAX_ROWS of include/detham.h


def energy_static(row_ptr, col, val, psi, n_dets=None, nnz=None, want_y=False, out=None, y=None, stream=None):
    """detham_energy_static: the energy step on a caller-held CSR with the scratch in a static device array of the library - the
    C call allocates nothing, needs no context and does not synchronise.  row_ptr / col / val: torch CUDA tensors, or raw device
    pointers (e.g. Detham.csr_pointers()) with `n_dets` and `nnz` given.  `out` (float64 [3] CUDA) and `y` are created here unless
    passed in.  Returns out = {psi^T H psi, psi^T psi, E_S} (device; read it after synchronising), and y if want_y."""
    import torch
    if not torch.cuda.is_available():
        raise DethamError(6, "no CUDA device: the detham hot path has no CPU fallback")
    L = load_library()
    assert psi.is_cuda and psi.dtype == torch.float64 and psi.is_contiguous()
    ptrs = []
    for t, dt in ((row_ptr, torch.int64), (col, torch.int32), (val, torch.float64)):
        if isinstance(t, int):
            ptrs.append(t)
        else:
            assert t.is_cuda and t.dtype == dt and t.is_contiguous()
            ptrs.append(t.data_ptr())
    if n_dets is None:
        n_dets = psi.numel()
    if nnz is None:
        nnz = val.numel()
    if out is None:
        out = torch.empty(3, dtype=torch.float64, device=psi.device)
    if want_y and y is None:
        y = torch.empty_like(psi)
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 3
    sp = C.c_void_p(stream.cuda_stream) if stream is not None else C.c_void_p(torch.cuda.current_stream().cuda_stream)
    st = L.detham_energy_static(ptrs[0], ptrs[1], ptrs[2], psi.data_ptr(), int(n_dets), int(nnz),
                                y.data_ptr() if want_y else None, out.data_ptr(), sp)
    if st != 0:
        raise DethamError(st, L.detham_strerror(st).decode(), L.detham_energy_static_error().decode())
    return (out, y) if want_y else out


def create(n_orb, n_alpha, n_beta, h1, eri, e_core=0.0, stream=None) -> Detham:
    return Detham(n_orb, n_alpha, n_beta, h1, eri, e_core, stream)
