"""paper_2202_00832_b200 -- Python binding of liblo_afqmc.so (B200-native LO-AFQMC local energy).

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C ABI declared in
include/lo_afqmc.h.  torch is used for device memory and streams.  There is no CPU fallback: if the
library cannot be built or loaded, importing works but every call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

LO_SETUP_GPU_SVD = 1
LO_SETUP_PROPAGATOR = 2
LO_SETUP_NO_PRESCREEN = 4
LO_SETUP_RANDOMIZED_SVD = 8
K_NAMES = ("overlap", "inverse", "theta", "coulomb", "exchange", "finalize", "propagator")
_STATUS = {0: "LO_OK", 1: "LO_EINVAL", 2: "LO_ENOMEM", 3: "LO_ECUDA", 5: "LO_EINTERNAL"}
EXPORTS = ("lo_setup", "lo_info_get", "lo_ranks", "lo_factor_pair", "lo_factor_all", "lo_retruncate", "lo_screen_pairs", "lo_local_energy",
           "lo_local_energy_host", "lo_set_cas_trial", "lo_set_cas_trial_beta", "lo_local_energy_cas", "lo_set_coulomb_mode", "lo_set_exchange_mode", "lo_coulomb_x", "lo_propagator", "lo_propagator_buffer", "lo_propagator_host", "lo_theta_host", "lo_timing_enable", "lo_timing_get", "lo_flops_per_walker",
           "lo_measure_peak", "lo_theta_noalloc_init", "lo_theta_noalloc", "lo_free", "lo_last_error", "lo_version")


class LoError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (_STATUS.get(status, status), msg))
        self.status = status


class LoInfo(C.Structure):
    _fields_ = [("N", C.c_int), ("n_chol", C.c_int), ("n_spin", C.c_int), ("n_occ", C.c_int * 2), ("N_pad", C.c_int),
                ("n_pairs", C.c_longlong * 2), ("sum_rank", C.c_longlong * 2), ("sum_rank_padded", C.c_longlong),
                ("max_rank", C.c_int), ("min_rank", C.c_int), ("factor_bytes", C.c_ulonglong), ("lbar_bytes", C.c_ulonglong),
                ("workspace_bytes", C.c_ulonglong), ("threshold", C.c_double), ("device", C.c_int), ("max_walkers", C.c_int),
                ("setup_on_gpu", C.c_int), ("n_tiles", C.c_longlong), ("svd_sweeps_max", C.c_int), ("svd_offdiag_max", C.c_double),
                ("setup_seconds", C.c_double), ("setup_svd_seconds", C.c_double), ("rsvd_sketch", C.c_int),
                ("n_pairs_rsvd", C.c_longlong), ("n_pairs_prescreened", C.c_longlong),
                ("n_pairs_energy_screened", C.c_longlong), ("energy_screen_cutoff", C.c_double), ("energy_screen_bound", C.c_double),
                ("exchange_mode", C.c_int), ("int8_bytes", C.c_ulonglong)]


_lib = None


def lib():
    """Load (building first if needed) liblo_afqmc.so.  Raises if it cannot be built: there is no fallback."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, ci, cd = C.c_void_p, C.c_int, C.c_double
        L.lo_setup.argtypes = [ci, ci, ci, C.POINTER(ci), vp, vp, vp, vp, cd, ci, ci, C.c_uint, C.POINTER(vp)]
        L.lo_info_get.argtypes = [vp, C.POINTER(LoInfo)]
        L.lo_ranks.argtypes = [vp, ci, vp]
        L.lo_factor_pair.argtypes = [vp, ci, ci, ci, vp, vp, vp]
        L.lo_factor_all.argtypes = [vp, ci, vp, vp, vp]
        L.lo_retruncate.argtypes = [vp, cd, C.POINTER(vp)]
        L.lo_screen_pairs.argtypes = [vp, cd, C.POINTER(vp)]
        L.lo_local_energy.argtypes = [vp, ci, vp, vp, vp, vp, vp, vp, vp, vp]
        L.lo_local_energy_host.argtypes = [vp, ci, vp, vp, vp, vp, vp]
        L.lo_coulomb_x.argtypes = [vp, C.POINTER(vp), C.POINTER(ci)]
        L.lo_theta_host.argtypes = [vp, ci, ci, vp]
        L.lo_set_coulomb_mode.argtypes = [vp, ci]
        L.lo_set_exchange_mode.argtypes = [vp, ci]
        L.lo_set_cas_trial.argtypes = [vp, ci, ci, ci, vp, vp, vp, ci, ci]
        L.lo_set_cas_trial_beta.argtypes = [vp, ci, vp, vp]
        L.lo_local_energy_cas.argtypes = [vp, ci, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.lo_propagator.argtypes = [vp, ci, vp, vp]
        L.lo_propagator_buffer.argtypes = [vp, C.POINTER(vp), C.POINTER(ci), C.POINTER(C.c_longlong)]
        L.lo_propagator_host.argtypes = [vp, ci, vp]
        L.lo_timing_enable.argtypes = [vp, ci]
        L.lo_timing_get.argtypes = [vp, C.POINTER(cd), C.POINTER(C.c_longlong)]
        L.lo_flops_per_walker.argtypes = [vp, C.POINTER(cd)]
        L.lo_measure_peak.argtypes = [ci, ci, C.POINTER(cd)]
        L.lo_theta_noalloc_init.argtypes = [ci]
        L.lo_theta_noalloc.argtypes = [ci, ci, ci, ci, vp, vp, vp, ci, vp, vp]
        L.lo_free.argtypes = [vp]
        L.lo_free.restype = None
        L.lo_last_error.restype = C.c_char_p
        L.lo_version.restype = C.c_char_p
        _lib = L
    return _lib


def library_path() -> str:
    return _build.LIB


def _check(st):
    if st != 0:
        raise LoError(st, lib().lo_last_error().decode())


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def measure_peak(kind: str, device: int = 0) -> float:
    """In-run roofline denominators: 'dmma' / 'dfma' in TFLOP/s, 'hbm' in GB/s; the gated INT8-slicing probe on tcgen05
    (DESIGN.md 10.1): 'int8_tile_us' (microseconds per 128 x 128 x 384 tile) and 'int8_tile_err' (error against fp64)."""
    v = C.c_double(0)
    _check(lib().lo_measure_peak(device, {"dmma": 0, "dfma": 1, "hbm": 2, "int8_tile_us": 3, "int8_tile_err": 4}[kind], C.byref(v)))
    return v.value


LO_NOALLOC_SCRATCH_BYTES = 4 << 20


def theta_noalloc_init(device: int = 0):
    """lo_theta_noalloc_init: fetch the device address of the static scratch array (once per device, before any capture)."""
    _check(lib().lo_theta_noalloc_init(int(device)))


def theta_noalloc(psi, phi, thetaT, status, stream=None):
    """lo_theta_noalloc: Theta = Phi (Psi^T Phi)^-1 with no allocation (scratch in a static device array of 4 MiB).
    All arguments are torch CUDA tensors the caller owns: psi float64 [N, n_occ], phi complex128 [n_w, N, n_occ],
    thetaT float64 [n_occ, ld_w, N_pad] (OUT, Theta^T panels), status int32 [n_w] (OUT).  Asynchronous on `stream`."""
    import torch
    if not (psi.is_cuda and phi.is_cuda and thetaT.is_cuda and status.is_cuda):
        raise ValueError("theta_noalloc: all tensors must be CUDA tensors")
    if psi.dtype != torch.float64 or phi.dtype != torch.complex128 or thetaT.dtype != torch.float64 or status.dtype != torch.int32:
        raise ValueError("theta_noalloc: psi/thetaT float64, phi complex128, status int32")
    if not (psi.is_contiguous() and phi.is_contiguous() and thetaT.is_contiguous() and status.is_contiguous()):
        raise ValueError("theta_noalloc: tensors must be contiguous")
    n_w, N, O = phi.shape
    if tuple(psi.shape) != (N, O) or thetaT.dim() != 3 or thetaT.shape[0] != O or thetaT.shape[2] != (N + 15) // 16 * 16 or status.numel() < n_w:
        raise ValueError("theta_noalloc: shapes psi [N, O], phi [n_w, N, O], thetaT [O, ld_w, ceil16(N)], status [n_w]")
    s = torch.cuda.current_stream(phi.device) if stream is None else stream
    _check(lib().lo_theta_noalloc(phi.device.index, N, O, n_w, C.c_void_p(psi.data_ptr()), C.c_void_p(phi.data_ptr()),
                                  C.c_void_p(thetaT.data_ptr()), int(thetaT.shape[1]), C.c_void_p(status.data_ptr()), C.c_void_p(s.cuda_stream)))


class Factors:
    """Owner of a lo_factors handle (lo_setup ... lo_free)."""

    def __init__(self, handle):
        self._h = C.c_void_p(handle)

    @classmethod
    def setup(cls, h, L, psis, threshold, device=0, max_walkers=1, gpu_svd=False, propagator=False, prescreen=True, rsvd=0):
        """lo_setup: h [N,N], L [n_chol,N,N], psis = [psi] (closed shell) or [psi_a, psi_b]; host numpy arrays.
        rsvd = k > 0: LO_SETUP_RANDOMIZED_SVD with a sketch of k rows (a multiple of 16)."""
        h, L = _np(h, np.float64), _np(L, np.float64)
        psis = [_np(p, np.float64) for p in psis]
        N, n_chol = h.shape[0], L.shape[0]
        n_occ = (C.c_int * 2)(*([p.shape[1] for p in psis] + [0])[:2])
        out = C.c_void_p()
        st = lib().lo_setup(N, n_chol, len(psis), n_occ, h.ctypes.data, L.ctypes.data, psis[0].ctypes.data,
                            psis[1].ctypes.data if len(psis) == 2 else None, float(threshold), int(device), int(max_walkers),
                            (LO_SETUP_GPU_SVD if gpu_svd else 0) | (LO_SETUP_PROPAGATOR if propagator else 0) |
                            (0 if prescreen else LO_SETUP_NO_PRESCREEN) |
                            ((LO_SETUP_RANDOMIZED_SVD | ((int(rsvd) // 16) << 8)) if rsvd else 0), C.byref(out))
        _check(st)
        return cls(out.value)

    def free(self):
        if self._h:
            lib().lo_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass

    def info(self) -> LoInfo:
        info = LoInfo()
        _check(lib().lo_info_get(self._h, C.byref(info)))
        return info

    def ranks(self, spin=0) -> np.ndarray:
        r = np.zeros(self.info().n_pairs[spin], dtype=np.int32)
        _check(lib().lo_ranks(self._h, spin, r.ctypes.data))
        return r

    def factor_pair(self, spin, i, j):
        info = self.info()
        O = info.n_occ[spin]
        k = i * O - i * (i - 1) // 2 + (j - i)
        r = int(self.ranks(spin)[k])
        U, s, W = np.zeros((r, info.N)), np.zeros(r), np.zeros((r, info.N))
        _check(lib().lo_factor_pair(self._h, spin, i, j, U.ctypes.data, s.ctypes.data, W.ctypes.data))
        return U, s, W

    def factor_all(self, spin=0):
        info = self.info()
        R = int(info.sum_rank[spin])
        U, s, W = np.zeros((R, info.N)), np.zeros(R), np.zeros((R, info.N))
        _check(lib().lo_factor_all(self._h, spin, U.ctypes.data, s.ctypes.data, W.ctypes.data))
        return U, s, W

    def factor_range(self, spin, k0, k1):
        """Factors of the pairs [k0, k1) of one spin (lo_ranks order), rows back to back: (ranks, U, sigma, W).
        One lo_factor_pair call per pair; for factor sets too large to copy to the host in one piece."""
        info = self.info()
        O, N = info.n_occ[spin], info.N
        r = self.ranks(spin)[k0:k1]
        off = np.concatenate([[0], np.cumsum(r)]).astype(np.int64)
        U, s, W = np.zeros((int(off[-1]), N)), np.zeros(int(off[-1])), np.zeros((int(off[-1]), N))
        ii, jj = np.triu_indices(O)
        L = lib()
        for n, k in enumerate(range(k0, k1)):
            if r[n] == 0:
                continue
            a = int(off[n])
            _check(L.lo_factor_pair(self._h, spin, int(ii[k]), int(jj[k]), U[a:].ctypes.data, s[a:].ctypes.data, W[a:].ctypes.data))
        return r, U, s, W

    def retruncate(self, threshold) -> "Factors":
        out = C.c_void_p()
        _check(lib().lo_retruncate(self._h, float(threshold), C.byref(out)))
        return Factors(out.value)

    def _check_phis(self, phis, n_cols, what):
        """Argument checks the C ABI cannot make on raw pointers: dtype, device, shape [n_w, N, n_cols[s]] per spin and one
        n_w for all spins.  Returns (contiguous tensors, n_w, device)."""
        import torch
        info = self.info()
        if len(phis) != len(n_cols):
            raise LoError(1, "%s: %d walker tensor(s) given, the factor set needs %d" % (what, len(phis), len(n_cols)))
        out = []
        for s, p in enumerate(phis):
            if not isinstance(p, torch.Tensor) or p.dtype != torch.complex128 or not p.is_cuda:
                raise LoError(1, "%s: phi must be a CUDA complex128 tensor" % what)
            if p.device.index != info.device:
                raise LoError(1, "%s: phi is on cuda:%s, the factor set on cuda:%d" % (what, p.device.index, info.device))
            if p.dim() != 3 or p.shape[1] != info.N or p.shape[2] != n_cols[s] or p.shape[0] != phis[0].shape[0]:
                raise LoError(1, "%s: phi[%d] has shape %s, expected [n_w=%d, N=%d, %d]" % (what, s, tuple(p.shape), phis[0].shape[0], info.N, n_cols[s]))
            out.append(p if p.is_contiguous() else p.contiguous())
        return out, int(phis[0].shape[0]), phis[0].device

    @staticmethod
    def _on_stream(stream, dev, *tensors):
        """Tensors allocated by the caching allocator on the current stream but used on `stream`: tell the allocator."""
        import torch
        if stream is not None and stream != torch.cuda.current_stream(dev):
            for t in tensors:
                if t is not None:
                    t.record_stream(stream)

    def screen_pairs(self, pair_cutoff) -> "Factors":
        """lo_screen_pairs: drop every pair with m_ij sigma_1 <= pair_cutoff."""
        out = C.c_void_p()
        _check(lib().lo_screen_pairs(self._h, float(pair_cutoff), C.byref(out)))
        return Factors(out.value)

    def local_energy(self, phis, parts=True, status=True, stream=None):
        """lo_local_energy on torch CUDA tensors phis = [phi_a(, phi_b)], complex128 [n_w,N,O].  Asynchronous on the
        current (or given) torch stream.  Returns (E_L, E1, E_J, E_K, status) torch tensors (None where not requested)."""
        import torch
        info = self.info()
        phis, n_w, dev = self._check_phis(list(phis), list(info.n_occ)[:info.n_spin], "local_energy")
        s = torch.cuda.current_stream(dev) if stream is None else stream
        E = torch.empty((4 if parts else 1, n_w), dtype=torch.complex128, device=dev)
        st_t = torch.empty(n_w, dtype=torch.int32, device=dev) if status else None
        self._on_stream(stream, dev, E, st_t, *phis)
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        _check(lib().lo_local_energy(self._h, n_w, ptr(phis[0]), ptr(phis[1]) if len(phis) == 2 else None, ptr(E[0]),
                                     ptr(E[1]) if parts else None, ptr(E[2]) if parts else None, ptr(E[3]) if parts else None,
                                     ptr(st_t), C.c_void_p(s.cuda_stream)))
        return (E[0], E[1], E[2], E[3], st_t) if parts else (E[0], None, None, None, st_t)

    def local_energy_host(self, phis_host, E_host=None, status_host=None, stream=None):
        """lo_local_energy_host: numpy (or pinned torch CPU) complex128 inputs [n_w,N,O]; copies in, runs, copies
        E [n_w,4] = (E_L,E1,E_J,E_K) and status back, synchronises."""
        import torch
        info = self.info()
        n_w = phis_host[0].shape[0]
        if len(phis_host) != info.n_spin:
            raise LoError(1, "local_energy_host: %d walker array(s) given, the factor set needs %d" % (len(phis_host), info.n_spin))
        for sp, a in enumerate(phis_host):
            if tuple(a.shape) != (n_w, info.N, info.n_occ[sp]) or str(a.dtype).split(".")[-1] != "complex128":
                raise LoError(1, "local_energy_host: phi[%d] must be complex128 [n_w=%d, N=%d, %d], got %s %s" % (
                    sp, n_w, info.N, info.n_occ[sp], a.dtype, tuple(a.shape)))
            if not (a.is_contiguous() if hasattr(a, "is_contiguous") else a.flags["C_CONTIGUOUS"]):
                raise LoError(1, "local_energy_host: phi[%d] must be contiguous" % sp)
        if E_host is None:
            E_host = np.empty((n_w, 4), dtype=np.complex128)
        if status_host is None:
            status_host = np.empty(n_w, dtype=np.int32)
        dp = lambda a: C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data)
        s = torch.cuda.current_stream() if stream is None else stream
        _check(lib().lo_local_energy_host(self._h, n_w, dp(phis_host[0]), dp(phis_host[1]) if len(phis_host) == 2 else None,
                                          dp(E_host), dp(status_host), C.c_void_p(s.cuda_stream)))
        return E_host, status_host

    def theta_host(self, spin, n_w) -> np.ndarray:
        info = self.info()
        th = np.empty((n_w, info.N, info.n_occ[spin]), dtype=np.complex128)
        _check(lib().lo_theta_host(self._h, spin, n_w, th.ctypes.data))
        return th

    def coulomb_x(self):
        """Device pointer and leading dimension of X[g][w] (complex128) from the last call."""
        p, ld = C.c_void_p(), C.c_int()
        _check(lib().lo_coulomb_x(self._h, C.byref(p), C.byref(ld)))
        return p.value, ld.value

    def set_cas_trial(self, n_ref, holes, parts, coef, max_real_walkers, smw_energy=False):
        """lo_set_cas_trial: holes/parts int32 [n_det, max_exc] (-1 padded), coef [n_det]; smw_energy selects the
        rearranged sums of Eq. 21-23 (LO_CAS_SMW_ENERGY) instead of direct summation over determinants."""
        holes, parts, coef = _np(holes, np.int32), _np(parts, np.int32), _np(coef, np.float64)
        n_det, max_exc = holes.shape
        _check(lib().lo_set_cas_trial(self._h, int(n_ref), n_det, max_exc, holes.ctypes.data, parts.ctypes.data, coef.ctypes.data,
                                      int(max_real_walkers), 1 if smw_energy else 0))
        self._cas_n_ref = [int(n_ref)]

    def set_cas_trial_beta(self, n_ref_b, holes_b, parts_b):
        """lo_set_cas_trial_beta: beta strings of an unrestricted trial (after set_cas_trial with the alpha strings)."""
        holes_b, parts_b = _np(holes_b, np.int32), _np(parts_b, np.int32)
        _check(lib().lo_set_cas_trial_beta(self._h, int(n_ref_b), holes_b.ctypes.data, parts_b.ctypes.data))
        self._cas_n_ref = [self._cas_n_ref[0], int(n_ref_b)]

    def local_energy_cas(self, phi, phi_b=None, stream=None):
        """lo_local_energy_cas on a torch CUDA complex128 tensor [n_w, N, n_ref]; returns (E [5, n_w] = E_L, E1, E_J,
        E_K, overlap ratio; status [n_w]) torch tensors.  Asynchronous on the current (or given) stream."""
        import torch
        if getattr(self, "_cas_n_ref", None) is None:
            raise LoError(1, "local_energy_cas: call set_cas_trial first")
        phis, n_w, dev = self._check_phis([phi] if phi_b is None else [phi, phi_b], self._cas_n_ref, "local_energy_cas")
        phi, phi_b = phis[0], (phis[1] if phi_b is not None else None)
        s = torch.cuda.current_stream(dev) if stream is None else stream
        E = torch.empty((5, n_w), dtype=torch.complex128, device=dev)
        st_t = torch.empty(n_w, dtype=torch.int32, device=dev)
        self._on_stream(stream, dev, E, st_t, *phis)
        ptr = lambda t: C.c_void_p(t.data_ptr())
        _check(lib().lo_local_energy_cas(self._h, n_w, ptr(phi), ptr(phi_b) if phi_b is not None else None, ptr(E[0]), ptr(E[1]), ptr(E[2]), ptr(E[3]), ptr(E[4]), ptr(st_t),
                                         C.c_void_p(s.cuda_stream)))
        return E, st_t

    def set_coulomb_mode(self, compressed: bool):
        """lo_set_coulomb_mode: E_J from the compressed pair factors (Eq. 19/22, paper-literal) or the Cholesky route."""
        _check(lib().lo_set_coulomb_mode(self._h, 1 if compressed else 0))

    def set_exchange_mode(self, int8: bool):
        """lo_set_exchange_mode: exchange projections from INT8 digit slices on the tcgen05 tensor cores (True) or on the FP64
        tensor pipe (False, the default).  The first switch to INT8 slices the factor rows (synchronous)."""
        _check(lib().lo_set_exchange_mode(self._h, 1 if int8 else 0))

    def propagator(self, x, stream=None):
        """lo_propagator: x = torch CUDA complex128 [n_w, n_chol] (shifted auxiliary fields); forms
        B_w = sum_g x[w,g] L^g into the library's buffer (see propagator_buffer / propagator_host).  Asynchronous."""
        import torch
        info = self.info()
        if x.dtype != torch.complex128 or not x.is_cuda or x.device.index != info.device:
            raise LoError(1, "propagator: x must be a complex128 tensor on cuda:%d" % info.device)
        if x.dim() != 2 or x.shape[1] != info.n_chol:
            raise LoError(1, "propagator: x has shape %s, expected [n_w, n_chol=%d]" % (tuple(x.shape), info.n_chol))
        x = x if x.is_contiguous() else x.contiguous()
        s = torch.cuda.current_stream(x.device) if stream is None else stream
        self._on_stream(stream, x.device, x)
        _check(lib().lo_propagator(self._h, int(x.shape[0]), C.c_void_p(x.data_ptr()), C.c_void_p(s.cuda_stream)))
        return x

    def propagator_buffer(self):
        """(device pointer, ld, n_rows) of the packed upper-triangle result, complex128 [n_rows][ld], walker fastest."""
        p, ld, n = C.c_void_p(), C.c_int(), C.c_longlong()
        _check(lib().lo_propagator_buffer(self._h, C.byref(p), C.byref(ld), C.byref(n)))
        return p.value, ld.value, n.value

    def propagator_host(self, w) -> np.ndarray:
        N = self.info().N
        B = np.empty((N, N), dtype=np.complex128)
        _check(lib().lo_propagator_host(self._h, int(w), B.ctypes.data))
        return B

    def timing_enable(self, on=True):
        _check(lib().lo_timing_enable(self._h, 1 if on else 0))

    def timing_get(self):
        ms = (C.c_double * len(K_NAMES))()
        n = (C.c_longlong * len(K_NAMES))()
        _check(lib().lo_timing_get(self._h, ms, n))
        return {k: (ms[i], n[i]) for i, k in enumerate(K_NAMES)}

    def flops_per_walker(self):
        fl = (C.c_double * len(K_NAMES))()
        _check(lib().lo_flops_per_walker(self._h, fl))
        return {k: fl[i] for i, k in enumerate(K_NAMES)}
