"""ctypes binding of include/qsgw.h.  Function names mirror the C ABI (qsgw_* -> methods of
Chi0Context); tensors are torch CUDA tensors (device memory + streams only) whose data_ptr()
is passed straight through.  No arithmetic of the method happens here, and there is no CPU
fallback: if libqsgw.so is missing or no sm_100 GPU is present the calls raise QsgwError.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

from .build import LIB_PATH

PREC_FP64, PREC_MIXED = 0, 1
STAGE_ZMEL, STAGE_WEIGHTS, STAGE_CHI0, STAGE_FINALIZE = 0, 1, 2, 3
_STATUS = {0: "QSGW_OK", 1: "QSGW_ERR_INVALID_ARG", 2: "QSGW_ERR_SHAPE", 3: "QSGW_ERR_STATE",
           4: "QSGW_ERR_ALLOC", 5: "QSGW_ERR_CUDA", 6: "QSGW_ERR_UNSUPPORTED"}


class QsgwError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_STATUS.get(code, code)}: {msg}")
        self.code = code


class _Desc(C.Structure):
    _fields_ = [("n_sites", C.c_int32), ("h_orb_per_site", C.POINTER(C.c_int32)),
                ("h_pb_per_site", C.POINTER(C.c_int32)), ("n_freq", C.c_int32),
                ("h_omega", C.POINTER(C.c_double)), ("n_k", C.c_int32), ("max_n_o", C.c_int32),
                ("max_n_u", C.c_int32), ("precision", C.c_int32), ("occ_tol", C.c_double),
                ("workspace_bytes", C.c_size_t)]


_lib = None


def library_path() -> str:
    return LIB_PATH


def lib() -> C.CDLL:
    """Load libqsgw.so (built in-tree by paper_2506_03477_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise QsgwError(6, f"{LIB_PATH} not found: run `python -m paper_2506_03477_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, dp = C.c_void_p, C.c_int32, C.c_int64, C.c_void_p
    L.qsgw_create.argtypes = [C.POINTER(_Desc), vp, C.POINTER(vp)]
    L.qsgw_set_product_tensor.argtypes = [vp, vp]
    L.qsgw_zmel_build.argtypes = [vp, vp, i64, vp, i64, i32, i32, i32, i32, vp]
    L.qsgw_chi0_accumulate.argtypes = [vp, vp, dp, dp, dp, dp, i32, i32]
    L.qsgw_chi0_add_kpoint.argtypes = [vp, vp, i64, vp, i64, dp, dp, dp, dp, i32, i32]
    L.qsgw_chi0_add_kpoints.argtypes = [vp, vp, i64, i64, vp, i64, i64, dp, dp, dp, dp, i32, i32, i32]
    L.qsgw_chi0_finalize.argtypes = [vp, vp]
    L.qsgw_reset.argtypes = [vp]
    L.qsgw_sync.argtypes = [vp]
    L.qsgw_destroy.argtypes = [vp]
    L.qsgw_destroy.restype = None
    L.qsgw_chi0_run_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, vp, C.POINTER(i64)]
    L.qsgw_set_option.argtypes = [vp, C.c_char_p, i64]
    L.qsgw_sigc_imag_accumulate.argtypes = [vp, vp, dp, dp, vp, i32, i32, vp]
    L.qsgw_imchi_add_batch.argtypes = [vp, vp, i64, vp, i64, i32, i32, i32, i32, vp, vp, dp, i32]
    L.qsgw_hilbert_to_imag_axis.argtypes = [i32, i32, dp, i32, dp, vp, vp, vp]
    L.qsgw_hilbert_to_real_axis.argtypes = [i32, i32, dp, i32, dp, vp, vp, vp]
    L.qsgw_mixed_stats.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(C.c_double)]
    L.qsgw_coulomb_eigenbasis.argtypes = [i32, vp, vp, vp, vp, C.POINTER(i32), C.POINTER(i32), vp]
    L.qsgw_zmel_ipw_build.argtypes = [C.POINTER(i32), vp, i32, vp, i32, vp, i32, vp, vp, i64, i32, vp, i64, i32, vp, i64, vp]
    for name in ("qsgw_create", "qsgw_set_product_tensor", "qsgw_zmel_build", "qsgw_chi0_accumulate",
                 "qsgw_chi0_add_kpoint", "qsgw_chi0_finalize", "qsgw_reset", "qsgw_sync",
                 "qsgw_chi0_run_host", "qsgw_n_m", "qsgw_n_b", "qsgw_set_option", "qsgw_mixed_stats", "qsgw_wc_from_chi0",
                 "qsgw_sigc_imag_accumulate", "qsgw_chi0_add_kpoints", "qsgw_imchi_add_batch",
                 "qsgw_hilbert_to_imag_axis", "qsgw_hilbert_to_real_axis", "qsgw_zmel_ipw_build", "qsgw_coulomb_eigenbasis",
                 "qsgw_chi0_to_coulomb_basis"):
        getattr(L, name).restype = i32
    for name in ("qsgw_last_error", "qsgw_last_create_error", "qsgw_version"):
        getattr(L, name).restype = C.c_char_p
    L.qsgw_last_error.argtypes = [vp]
    for name in ("qsgw_kernel_launches", "qsgw_pairs_accumulated"):
        getattr(L, name).restype = i64
        getattr(L, name).argtypes = [vp]
    L.qsgw_set_stage_timing.argtypes = [vp, i32]
    L.qsgw_set_stage_timing.restype = i32
    L.qsgw_stage_time_ms.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(i64)]
    L.qsgw_stage_time_ms.restype = i32
    L.qsgw_probe_peak.argtypes = [i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.qsgw_probe_peak.restype = i32
    L.qsgw_device_bytes.restype = C.c_size_t
    L.qsgw_device_bytes.argtypes = [vp]
    L.qsgw_n_m.argtypes = [vp]
    L.qsgw_n_b.argtypes = [vp]
    L.qsgw_wc_from_chi0.argtypes = [i32, i32, vp, vp, vp, vp, vp]
    L.qsgw_chi0_to_coulomb_basis.argtypes = [i32, i32, vp, vp, vp, vp]
    L.qsgw_chi0_to_coulomb_basis_static.argtypes = [i32, i32, vp, vp, vp, vp]
    L.qsgw_chi0_to_coulomb_basis_static.restype = i32
    _lib = L
    return L


def version() -> str:
    return lib().qsgw_version().decode()


def _make_desc(orb_per_site, pb_per_site, omega, n_k, max_n_o, max_n_u, precision, occ_tol,
               workspace_bytes):
    s = len(orb_per_site)
    orb = (C.c_int32 * s)(*[int(x) for x in orb_per_site])
    pb = (C.c_int32 * len(pb_per_site))(*[int(x) for x in pb_per_site])
    om = (C.c_double * len(omega))(*[float(x) for x in omega])
    d = _Desc(s, orb, pb, len(omega), om, int(n_k), int(max_n_o), int(max_n_u), int(precision),
              float(occ_tol), int(workspace_bytes))
    d._keep = (orb, pb, om)
    return d


def _ptr(t, dtype=None):
    """data_ptr of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("expected a torch CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return C.c_void_p(t.data_ptr())


PEAK_FP64_MMA, PEAK_TF32_MMA, PEAK_F16_MMA = 0, 1, 2


def probe_peak(kind: int = PEAK_FP64_MMA):
    """qsgw_probe_peak: (TFLOP/s, ms) of the register-resident MMA issue-rate loop on this device."""
    L = lib()
    tf, ms = C.c_double(0.0), C.c_double(0.0)
    rc = L.qsgw_probe_peak(int(kind), C.byref(tf), C.byref(ms))
    if rc != 0:
        raise QsgwError(rc, L.qsgw_last_create_error().decode())
    return float(tf.value), float(ms.value)


class Chi0Context:
    """One (q, spin) polarization build.  Methods map 1:1 to the qsgw_* entry points."""

    def __init__(self, orb_per_site: Sequence[int], pb_per_site: Sequence[int], omega, n_k: int,
                 max_n_o: int, max_n_u: int, precision: int = PREC_FP64, occ_tol: float = 1e-12,
                 workspace_bytes: int = 0, stream=None):
        import torch
        self._L = lib()
        self._h = C.c_void_p()
        self.n_freq = len(omega)
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.current_stream()
        self._stream = stream
        sp = C.c_void_p(stream.cuda_stream) if stream is not None else None
        d = _make_desc(orb_per_site, pb_per_site, omega, n_k, max_n_o, max_n_u, precision, occ_tol,
                       workspace_bytes)
        rc = self._L.qsgw_create(C.byref(d), sp, C.byref(self._h))
        if rc != 0:
            self._h = C.c_void_p()
            raise QsgwError(rc, self._L.qsgw_last_create_error().decode())
        self.n_m = self._L.qsgw_n_m(self._h)
        self.n_b = self._L.qsgw_n_b(self._h)

    def _check(self, rc: int):
        if rc != 0:
            raise QsgwError(rc, self._L.qsgw_last_error(self._h).decode())

    def set_product_tensor(self, d_P):
        import torch
        self._check(self._L.qsgw_set_product_tensor(self._h, _ptr(d_P, torch.complex128)))

    def zmel_build(self, d_Ck, d_Ckq, n_begin: int, n_o: int, np_begin: int, n_u: int, d_z_out=None,
                   ld_k: Optional[int] = None, ld_kq: Optional[int] = None):
        import torch
        ld_k = d_Ck.shape[-1] if ld_k is None else ld_k
        ld_kq = d_Ckq.shape[-1] if ld_kq is None else ld_kq
        self._check(self._L.qsgw_zmel_build(self._h, _ptr(d_Ck, torch.complex128), ld_k,
                                            _ptr(d_Ckq, torch.complex128), ld_kq, n_begin, n_o,
                                            np_begin, n_u, _ptr(d_z_out, torch.complex128)))

    def chi0_accumulate(self, d_eps_k, d_f_k, d_eps_kq, d_f_kq, n_o: int, n_u: int, d_z=None):
        import torch
        f64 = torch.float64
        self._check(self._L.qsgw_chi0_accumulate(self._h, _ptr(d_z, torch.complex128),
                                                 _ptr(d_eps_k, f64), _ptr(d_f_k, f64),
                                                 _ptr(d_eps_kq, f64), _ptr(d_f_kq, f64), n_o, n_u))

    def chi0_add_kpoint(self, d_Ck, d_Ckq, d_eps_k, d_f_k, d_eps_kq, d_f_kq):
        import torch
        f64 = torch.float64
        self._check(self._L.qsgw_chi0_add_kpoint(
            self._h, _ptr(d_Ck, torch.complex128), d_Ck.shape[-1], _ptr(d_Ckq, torch.complex128),
            d_Ckq.shape[-1], _ptr(d_eps_k, f64), _ptr(d_f_k, f64), _ptr(d_eps_kq, f64),
            _ptr(d_f_kq, f64), d_Ck.shape[0], d_Ckq.shape[0]))

    def chi0_add_kpoints(self, d_Ck, d_Ckq, d_eps_k, d_f_k, d_eps_kq, d_f_kq):
        """All k-points of contiguous arrays d_Ck [n_k][n_o][N_b], d_Ckq [n_k][n_u][N_b], d_eps_k/d_f_k [n_k][n_o],
        d_eps_kq/d_f_kq [n_k][n_u] in one call."""
        import torch
        f64 = torch.float64
        n_k, n_o, ld = d_Ck.shape
        n_u = d_Ckq.shape[1]
        self._check(self._L.qsgw_chi0_add_kpoints(
            self._h, _ptr(d_Ck, torch.complex128), ld, n_o * ld, _ptr(d_Ckq, torch.complex128), d_Ckq.shape[2],
            n_u * d_Ckq.shape[2], _ptr(d_eps_k, f64), _ptr(d_f_k, f64), _ptr(d_eps_kq, f64), _ptr(d_f_kq, f64),
            n_o, n_u, n_k))

    def chi0_finalize(self, d_chi0_out=None):
        import torch
        if d_chi0_out is None:
            d_chi0_out = torch.empty((self.n_freq, self.n_m, self.n_m), dtype=torch.complex128,
                                     device="cuda")
        self._check(self._L.qsgw_chi0_finalize(self._h, _ptr(d_chi0_out, torch.complex128)))
        return d_chi0_out

    def sigc_imag_accumulate(self, d_eps_q, d_eps_qk, d_wc, n_all: int, n_qp: int, d_sigc, d_z=None):
        """I^c of Eq. (22) for one k-point and one batch of intermediate states, added into d_sigc [n_qp][n_qp]."""
        import torch
        f64 = torch.float64
        self._check(self._L.qsgw_sigc_imag_accumulate(self._h, _ptr(d_z, torch.complex128), _ptr(d_eps_q, f64),
                                                      _ptr(d_eps_qk, f64), _ptr(d_wc, torch.complex128), n_all, n_qp,
                                                      _ptr(d_sigc, torch.complex128)))

    def imchi_add_batch(self, d_Ck, d_Ckq, n_begin: int, n_o: int, np_begin: int, n_u: int, d_bin_ptr, d_pair, d_w):
        """Binned spectral part (Eq. 15, Alg. 1 lines 12-21) of one k-point / band batch; CSR-by-bin weights."""
        import torch
        nnz = int(d_pair.shape[0]) if d_pair is not None else 0
        self._check(self._L.qsgw_imchi_add_batch(
            self._h, _ptr(d_Ck, torch.complex128), d_Ck.shape[-1], _ptr(d_Ckq, torch.complex128), d_Ckq.shape[-1],
            n_begin, n_o, np_begin, n_u, _ptr(d_bin_ptr, torch.int32), _ptr(d_pair, torch.int32) if nnz else None,
            _ptr(d_w, torch.float64) if nnz else None, nnz))

    def reset(self):
        self._check(self._L.qsgw_reset(self._h))

    def sync(self):
        self._check(self._L.qsgw_sync(self._h))

    def set_option(self, key: str, value: int):
        self._check(self._L.qsgw_set_option(self._h, key.encode(), int(value)))

    def mixed_stats(self):
        """qsgw_mixed_stats: (stage (b) launches, launches with E5M2 corrections, smallest P_eff); synchronises."""
        n, n8, pe = C.c_int64(0), C.c_int64(0), C.c_double(0.0)
        self._check(self._L.qsgw_mixed_stats(self._h, C.byref(n), C.byref(n8), C.byref(pe)))
        return int(n.value), int(n8.value), float(pe.value)

    def run_host(self, P, Ck, Ckq, eps_k, f_k, eps_kq, f_kq, out=None):
        """qsgw_chi0_run_host: whole job from HOST (NumPy) buffers on this context; returns (chi0, launches)."""
        import numpy as np
        n_k, n_o, _ = Ck.shape
        n_u = Ckq.shape[1]
        arrs = [np.ascontiguousarray(a, dtype=dt) for a, dt in
                ((P, np.complex128), (Ck, np.complex128), (Ckq, np.complex128), (eps_k, np.float64),
                 (f_k, np.float64), (eps_kq, np.float64), (f_kq, np.float64))]
        if out is None:
            out = np.empty((self.n_freq, self.n_m, self.n_m), dtype=np.complex128)
        launches = C.c_int64(0)
        self._check(self._L.qsgw_chi0_run_host(self._h, *[a.ctypes.data_as(C.c_void_p) for a in arrs], n_k, n_o,
                                               n_u, out.ctypes.data_as(C.c_void_p), C.byref(launches)))
        return out, int(launches.value)

    def set_stage_timing(self, enable: bool):
        self._check(self._L.qsgw_set_stage_timing(self._h, int(bool(enable))))

    def stage_time_ms(self, stage: int):
        """(summed event time in ms, launches) of `stage` since set_stage_timing; synchronises."""
        ms, n = C.c_double(0.0), C.c_int64(0)
        self._check(self._L.qsgw_stage_time_ms(self._h, int(stage), C.byref(ms), C.byref(n)))
        return float(ms.value), int(n.value)

    @property
    def kernel_launches(self) -> int:
        return int(self._L.qsgw_kernel_launches(self._h))

    @property
    def pairs_accumulated(self) -> int:
        return int(self._L.qsgw_pairs_accumulated(self._h))

    @property
    def device_bytes(self) -> int:
        return int(self._L.qsgw_device_bytes(self._h))

    def destroy(self):
        if self._h:
            self._L.qsgw_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def wc_from_chi0(chi0, v, out=None, info=None):
    """qsgw_wc_from_chi0: W^c[j] = sqrt(v) ((1 - sqrt(v) chi0[j] sqrt(v))^-1 - 1) sqrt(v) on the current
    torch stream.  chi0: complex128 CUDA tensor [n_freq][N_M][N_M]; v: float64 CUDA tensor [N_M].
    Returns (W^c, info) -- info is an int32 CUDA tensor (0 = all pivots positive), not synchronised."""
    import torch
    L = lib()
    n_freq, n_m = int(chi0.shape[0]), int(chi0.shape[1])
    if out is None:
        out = torch.empty_like(chi0)
    if info is None:
        info = torch.zeros(1, dtype=torch.int32, device=chi0.device)
    stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc = L.qsgw_wc_from_chi0(n_m, n_freq, _ptr(chi0, torch.complex128), _ptr(v, torch.float64),
                             _ptr(out, torch.complex128), _ptr(info, torch.int32), stream)
    if rc != 0:
        raise QsgwError(rc, L.qsgw_last_create_error().decode())
    return out, info


def chi0_to_coulomb_basis(chi0, U, out=None):
    """qsgw_chi0_to_coulomb_basis: U^H chi0[j] U for every frequency on the current torch stream."""
    import torch
    L = lib()
    n_freq, n_m = int(chi0.shape[0]), int(chi0.shape[1])
    if out is None:
        out = torch.empty_like(chi0)
    stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc = L.qsgw_chi0_to_coulomb_basis(n_m, n_freq, _ptr(chi0, torch.complex128), _ptr(U, torch.complex128),
                                      _ptr(out, torch.complex128), stream)
    if rc != 0:
        raise QsgwError(rc, L.qsgw_last_create_error().decode())
    return out


def chi0_to_coulomb_basis_static(chi0, U, out):
    """qsgw_chi0_to_coulomb_basis_static: the same rotation on the library's file-scope device scratch; the call allocates
    nothing (the caller passes `out`).  Limit (2 n_freq + 1) ceil64(N_M)^2 <= 33 * 256 * 256; calls that overlap on the GPU race."""
    import torch
    L = lib()
    n_freq, n_m = int(chi0.shape[0]), int(chi0.shape[1])
    stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc = L.qsgw_chi0_to_coulomb_basis_static(n_m, n_freq, _ptr(chi0, torch.complex128), _ptr(U, torch.complex128),
                                             _ptr(out, torch.complex128), stream)
    if rc != 0:
        raise QsgwError(rc, L.qsgw_last_create_error().decode())
    return out


def hilbert_to_real_axis(A, edges, omega_out, out=None):
    """Eq. (18) for real-axis targets (principal value): qsgw_hilbert_to_real_axis."""
    return hilbert_to_imag_axis(A, edges, omega_out, out=out, _real=True)


def hilbert_to_imag_axis(A, edges, omega_out, out=None, _real=False):
    """Eq. (18) on the imaginary axis: out[i] = sum_j K[i][j] A[j] (qsgw_hilbert_to_imag_axis)."""
    import torch
    n_bins, n_m = int(A.shape[0]), int(A.shape[1])
    n_out = int(omega_out.shape[0])
    if out is None:
        out = torch.empty((n_out, n_m, n_m), dtype=torch.complex128, device=A.device)
    st = torch.cuda.current_stream(A.device).cuda_stream
    fn = lib().qsgw_hilbert_to_real_axis if _real else lib().qsgw_hilbert_to_imag_axis
    rc = fn(n_m, n_bins, _ptr(edges, torch.float64), n_out, _ptr(omega_out, torch.float64),
                                         _ptr(A, torch.complex128), _ptr(out, torch.complex128), C.c_void_p(st))
    if rc != 0:
        raise QsgwError(rc, lib().qsgw_last_create_error().decode())
    return out


def zmel_ipw_build(L, theta, g_kq, g_k, g_ipw, Bk, Bkq, out=None, col_offset=0):
    """IPW block of the matrix elements (qsgw_zmel_ipw_build): z[n, n', I] into out[:, :, col_offset:col_offset + n_ipw].

    L: three ints (host); theta complex128 (2 L0 + 1, 2 L1 + 1, 2 L2 + 1); g_*: int32 (N, 3); Bk (n_o, N_k), Bkq (n_u, N_kq).
    out: complex128 (n_o, n_u, ld_z) or None (allocated with ld_z = n_ipw)."""
    import torch
    n_o, n_u, n_ipw = int(Bk.shape[0]), int(Bkq.shape[0]), int(g_ipw.shape[0])
    if out is None:
        out = torch.empty((n_o, n_u, n_ipw), dtype=torch.complex128, device=Bk.device)
    if out.shape[0] != n_o or out.shape[1] != n_u or col_offset < 0 or col_offset + n_ipw > out.shape[2] or not out.is_contiguous():
        raise QsgwError(2, "out must be a contiguous (n_o, n_u, >= col_offset + n_ipw) tensor")
    hl = (C.c_int32 * 3)(int(L[0]), int(L[1]), int(L[2]))
    if tuple(theta.shape) != tuple(2 * int(l) + 1 for l in L):
        raise QsgwError(2, "theta must have shape (2 L0 + 1, 2 L1 + 1, 2 L2 + 1)")
    st = torch.cuda.current_stream(Bk.device).cuda_stream
    zp = C.c_void_p(_ptr(out, torch.complex128).value + 16 * int(col_offset))
    rc = lib().qsgw_zmel_ipw_build(hl, _ptr(theta, torch.complex128), int(g_kq.shape[0]), _ptr(g_kq, torch.int32),
                                   int(g_k.shape[0]), _ptr(g_k, torch.int32), n_ipw, _ptr(g_ipw, torch.int32),
                                   _ptr(Bk, torch.complex128), int(Bk.shape[1]), n_o, _ptr(Bkq, torch.complex128),
                                   int(Bkq.shape[1]), n_u, zp, int(out.shape[2]), C.c_void_p(st))
    if rc != 0:
        raise QsgwError(rc, lib().qsgw_last_create_error().decode())
    return out


def coulomb_eigenbasis(v, O):
    """Generalized eigenproblem (v - v_mu O) z = 0 of the mixed product basis (qsgw_coulomb_eigenbasis):
    returns (v_mu [N_M] float64 descending, U [N_M, N_M] complex128 with U[I, mu] = z_{mu I}, sweeps)."""
    import torch
    n = int(v.shape[0])
    vmu = torch.empty((n,), dtype=torch.float64, device=v.device)
    U = torch.empty((n, n), dtype=torch.complex128, device=v.device)
    info, sweeps = C.c_int32(0), C.c_int32(0)
    st = torch.cuda.current_stream(v.device).cuda_stream
    rc = lib().qsgw_coulomb_eigenbasis(n, _ptr(v, torch.complex128), _ptr(O, torch.complex128), _ptr(vmu, torch.float64),
                                       _ptr(U, torch.complex128), C.byref(info), C.byref(sweeps), C.c_void_p(st))
    if rc != 0:
        raise QsgwError(rc, lib().qsgw_last_create_error().decode() + f" (info = {info.value})")
    return vmu, U, int(sweeps.value)


def set_global_option(key: str, value: int):
    """qsgw_set_option(NULL, key, value): process-wide options ("wc_graph")."""
    L = lib()
    rc = L.qsgw_set_option(None, key.encode(), int(value))
    if rc != 0:
        raise QsgwError(rc, L.qsgw_last_create_error().decode())


def chi0_run_host(orb_per_site, pb_per_site, omega, P, Ck, Ckq, eps_k, f_k, eps_kq, f_kq,
                  max_n_o: int, max_n_u: int, precision: int = PREC_FP64, occ_tol: float = 1e-12,
                  out=None):
    """One-shot convenience: create a context, qsgw_chi0_run_host, destroy it; returns (chi0, kernel_launches).
    Repeated jobs should keep a Chi0Context and call its run_host (no per-call allocation)."""
    ctx = Chi0Context(orb_per_site, pb_per_site, omega, Ck.shape[0], max_n_o, max_n_u, precision=precision,
                      occ_tol=occ_tol)
    try:
        return ctx.run_host(P, Ck, Ckq, eps_k, f_k, eps_kq, f_kq, out=out)
    finally:
        ctx.destroy()
