"""dfjk -- B200-native density-fitted Coulomb/exchange build (``get_jk``).

Thin ctypes binding over ``libdfjk.so`` (C ABI in ``include/dfjk.h``; kernels in
``csrc/``).  Argument marshalling only: every step of the path runs in the
library's sm_100a kernels.  PyTorch is used for device memory and streams.

There is NO CPU fallback: if the shared library is missing or no CUDA device is
present, the calls raise.  This package never imports ``oracle``.

Paper: ``jmat, kmat = get_jk(mol, dm)`` with the integrals
density-fitted (Eq. 1-3).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

__all__ = ["build", "lib", "build_b", "df_diag_noalloc", "noalloc_max_nao", "device_info", "probe_fp64_peak", "DFJK", "DFJKError", "SYMBOLS", "KERNELS", "LIB_PATH", "HEADER_PATH"]

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdfjk.so")
CSRC = os.path.join(_HERE, "csrc")
HEADER_PATH = os.path.join(os.path.dirname(_HERE), "include", "dfjk.h")

# every symbol include/dfjk.h declares
SYMBOLS = (
    "dfjk_create", "dfjk_get_jk", "dfjk_get_jk_u", "dfjk_get_jk_host", "dfjk_get_d",
    "dfjk_set_option", "dfjk_workspace_bytes", "dfjk_destroy", "dfjk_last_error",
    "dfjk_version", "dfjk_launch_count", "dfjk_kernel_time",
    "dfjk_get_jk_pair", "dfjk_get_jk_dm", "dfjk_get_jk_dms", "dfjk_get_df_diag",
    "dfjk_build_b", "dfjk_scf_rhf", "dfjk_probe_dmma_peak",
    "dfjk_get_jk_u_host", "dfjk_scf_uhf", "dfjk_device_info", "dfjk_scf_timing",
    "dfjk_df_diag_noalloc", "dfjk_noalloc_max_nao", "dfjk_get_jk_pairs",
)

# DFJK_KERNEL_* ids of include/dfjk.h
KERNELS = {"K0": 0, "J0": 1, "J1": 2, "J1R": 3, "J2": 4, "J3": 5, "K1": 6, "K2": 7, "K3": 8}

_lib = None


class DFJKError(RuntimeError):
    """A dfjk_* call returned a negative code."""


def build(force: bool = False) -> str:
    """Compile ``libdfjk.so`` in-tree with nvcc for sm_100a (see csrc/Makefile)."""
    if force:
        subprocess.run(["make", "-C", CSRC, "clean"], check=True, stdout=subprocess.DEVNULL)
    subprocess.run(["make", "-C", CSRC, "-j8"], check=True, stdout=subprocess.DEVNULL)
    return LIB_PATH


def lib() -> ctypes.CDLL:
    """Load the C-ABI library (raises if it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise DFJKError(f"{LIB_PATH} is missing: run paper_2506_06661_b200.build() "
                        "(or __graft_entry__.build()); there is no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
    L.dfjk_create.restype = vp
    L.dfjk_create.argtypes = [i64, i64, vp]
    L.dfjk_get_jk.restype = ci
    L.dfjk_get_jk.argtypes = [vp, vp, i64, vp, vp, vp]
    L.dfjk_get_jk_u.restype = ci
    L.dfjk_get_jk_u.argtypes = [vp, vp, i64, vp, i64, vp, vp, vp, vp]
    L.dfjk_get_jk_pair.restype = ci
    L.dfjk_get_jk_pair.argtypes = [vp, vp, vp, i64, vp, vp, vp]
    L.dfjk_get_jk_pairs.restype = ci
    L.dfjk_get_jk_pairs.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp]
    L.dfjk_get_jk_dm.restype = ci
    L.dfjk_get_jk_dm.argtypes = [vp, vp, vp, vp, vp]
    L.dfjk_get_jk_dms.restype = ci
    L.dfjk_get_jk_dms.argtypes = [vp, i64, vp, vp, vp, vp]
    L.dfjk_scf_rhf.restype = ci
    L.dfjk_scf_rhf.argtypes = [vp, vp, vp, i64, i64, ctypes.c_double, i64, vp, vp, vp, vp,
                               ctypes.POINTER(ctypes.c_double), ctypes.POINTER(i64),
                               ctypes.POINTER(ci), vp]
    L.dfjk_probe_dmma_peak.restype = ci
    L.dfjk_probe_dmma_peak.argtypes = [ctypes.POINTER(ctypes.c_double)]
    L.dfjk_scf_uhf.restype = ci
    L.dfjk_scf_uhf.argtypes = [vp, vp, vp, i64, i64, i64, ctypes.c_double, i64, vp, vp, vp, vp, vp, vp,
                               ctypes.POINTER(ctypes.c_double), ctypes.POINTER(i64),
                               ctypes.POINTER(ci), vp]
    L.dfjk_scf_timing.restype = ci
    L.dfjk_scf_timing.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(ctypes.c_double),
                                  ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    L.dfjk_device_info.restype = ci
    L.dfjk_device_info.argtypes = [ctypes.POINTER(ci), ctypes.POINTER(ci), ctypes.POINTER(i64)]
    L.dfjk_build_b.restype = ci
    L.dfjk_build_b.argtypes = [i64, i64, vp, vp, vp, vp]
    L.dfjk_get_df_diag.restype = ci
    L.dfjk_get_df_diag.argtypes = [vp, vp, vp]
    L.dfjk_df_diag_noalloc.restype = ci
    L.dfjk_df_diag_noalloc.argtypes = [i64, i64, vp, vp, vp]
    L.dfjk_noalloc_max_nao.restype = i64
    L.dfjk_noalloc_max_nao.argtypes = []
    L.dfjk_get_jk_host.restype = ci
    L.dfjk_get_jk_host.argtypes = [vp, vp, i64, vp, vp]
    L.dfjk_get_jk_u_host.restype = ci
    L.dfjk_get_jk_u_host.argtypes = [vp, vp, i64, vp, i64, vp, vp, vp]
    L.dfjk_get_d.restype = ci
    L.dfjk_get_d.argtypes = [vp, vp, vp]
    L.dfjk_set_option.restype = ci
    L.dfjk_set_option.argtypes = [vp, ctypes.c_char_p, i64]
    L.dfjk_workspace_bytes.restype = i64
    L.dfjk_workspace_bytes.argtypes = [vp]
    L.dfjk_destroy.restype = ci
    L.dfjk_destroy.argtypes = [vp]
    L.dfjk_last_error.restype = ctypes.c_char_p
    L.dfjk_last_error.argtypes = []
    L.dfjk_version.restype = ctypes.c_char_p
    L.dfjk_version.argtypes = []
    L.dfjk_launch_count.restype = i64
    L.dfjk_launch_count.argtypes = [vp]
    L.dfjk_kernel_time.restype = ci
    L.dfjk_kernel_time.argtypes = [vp, ci, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(i64)]
    _lib = L
    return L


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise DFJKError(f"{what} failed ({rc}): {lib().dfjk_last_error().decode()}")


def _dev_f64(t, name: str, numel: Optional[int] = None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64
            and t.is_contiguous()):
        raise ValueError(f"{name} must be a contiguous CUDA float64 tensor")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name} has {t.numel()} elements, expected {numel}")
    return t.data_ptr()


def probe_fp64_peak() -> float:
    """Sustained FP64 TFLOP/s of a register-only DMMA loop on the current device."""
    v = ctypes.c_double(0.0)
    _check(lib().dfjk_probe_dmma_peak(ctypes.byref(v)), "dfjk_probe_dmma_peak")
    return v.value


def device_info() -> dict:
    """SM count, peak SM clock (kHz), L2 bytes of the current device, and the FP64 peak derived from
    them (SMs x 64 FMA/clk x 2 x clock, TFLOP/s) -- the roofline denominators' raw material."""
    sms, khz, l2 = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_int64(0)
    _check(lib().dfjk_device_info(ctypes.byref(sms), ctypes.byref(khz), ctypes.byref(l2)), "dfjk_device_info")
    return {"sm_count": sms.value, "sm_clock_khz": khz.value, "l2_bytes": l2.value,
            "fp64_peak_tflops": sms.value * 64 * 2 * khz.value * 1e3 / 1e12}


def build_b(M, R_packed, nao: int, stream=None):
    """Eq. 2-3 on the device, IN PLACE: ``M`` (naux x naux, SPD) becomes its
    Cholesky factor L (lower triangle), ``R_packed`` ([naux][npair] raw 3-centre tensor) becomes
    B = L^-1 R.  Returns the device int64 ``info`` flag (0 = ok, j+1 = pivot j not positive)."""
    import torch
    nao = int(nao)
    naux = int(R_packed.shape[0])
    if R_packed.dim() != 2 or R_packed.shape[1] != nao * (nao + 1) // 2:
        raise ValueError("R_packed must be [naux][nao(nao+1)/2]")
    if M.dim() != 2 or tuple(M.shape) != (naux, naux):
        raise ValueError("M must be naux x naux")
    mp, rp = _dev_f64(M, "M"), _dev_f64(R_packed, "R_packed")
    with torch.cuda.device(R_packed.device):
        info = torch.zeros(1, dtype=torch.int64, device=R_packed.device)
        st = (stream or torch.cuda.current_stream(R_packed.device)).cuda_stream
        _check(lib().dfjk_build_b(naux, nao, mp, rp, info.data_ptr(), st), "dfjk_build_b")
    return info


def noalloc_max_nao() -> int:
    """Largest nao ``df_diag_noalloc`` accepts (its scratch is a fixed 8 MiB array in the library)."""
    return int(lib().dfjk_noalloc_max_nao())


def df_diag_noalloc(B_packed, nao: int, out, stream=None):
    """``out[mu][nu] = sum_P B_P[mu,nu]^2`` (Eq. 7) through ``dfjk_df_diag_noalloc``:
    no handle and no device allocation anywhere, for callers that cannot allocate -- code living
    inside another framework's memory pool, code under a no-allocation-after-start-up rule, or a
    process whose HBM is already full of B.  That is why ``out`` (nao x nao CUDA float64) is the
    caller's buffer and not created here.  ``nao <= noalloc_max_nao()``; larger sizes raise.

    All calls on a device share one scratch array inside the library: issue them on one stream (or
    order them with events), never concurrently.  Make the first call on a device during start-up,
    outside any stream capture (it looks up the array's device address once)."""
    import torch
    nao = int(nao)
    npair = nao * (nao + 1) // 2
    if B_packed.dim() != 2 or B_packed.shape[1] != npair:
        raise ValueError(f"B_packed must be [naux][{npair}]")
    bp = _dev_f64(B_packed, "B_packed")
    op = _dev_f64(out, "out", nao * nao)
    with torch.cuda.device(B_packed.device):
        st = (stream or torch.cuda.current_stream(B_packed.device)).cuda_stream
        _check(lib().dfjk_df_diag_noalloc(int(B_packed.shape[0]), nao, bp, op, st), "dfjk_df_diag_noalloc")
    return out


class DFJK:
    """Handle on a device-resident packed DF tensor ``B[naux][nao(nao+1)/2]``.

    ``B`` is borrowed (never copied; up to 96 GB) and must outlive the handle.
    """

    def __init__(self, B_packed, nao: int):
        import torch
        self._h = None
        if not (isinstance(B_packed, torch.Tensor) and B_packed.is_cuda):
            raise ValueError("B_packed must be a CUDA tensor (there is no CPU path)")
        nao = int(nao)
        npair = nao * (nao + 1) // 2
        if B_packed.dim() != 2 or B_packed.shape[1] != npair:
            raise ValueError(f"B_packed must be [naux][{npair}]")
        ptr = _dev_f64(B_packed, "B_packed")
        self.B = B_packed                      # keep the borrowed tensor alive
        self.nao, self.naux, self.npair = nao, int(B_packed.shape[0]), npair
        self.device = B_packed.device
        with torch.cuda.device(self.device):
            self._h = lib().dfjk_create(self.naux, nao, ptr)
        if not self._h:
            raise DFJKError("dfjk_create failed: " + lib().dfjk_last_error().decode())

    # -- restricted: D = 2 C C^T
    def get_jk(self, C_occ, with_j: bool = True, with_k: bool = True, out_j=None, out_k=None,
               stream=None) -> Tuple[Optional["torch.Tensor"], Optional["torch.Tensor"]]:
        import torch
        if C_occ.dim() != 2 or C_occ.shape[0] != self.nao:
            raise ValueError("C_occ must be nao x nocc")
        cp = _dev_f64(C_occ, "C_occ")
        n2 = self.nao * self.nao
        J = (out_j if out_j is not None else torch.empty(self.nao, self.nao, dtype=torch.float64,
                                                         device=self.device)) if with_j else None
        K = (out_k if out_k is not None else torch.empty(self.nao, self.nao, dtype=torch.float64,
                                                         device=self.device)) if with_k else None
        jp = _dev_f64(J, "J", n2) if with_j else None
        kp = _dev_f64(K, "K", n2) if with_k else None
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            _check(lib().dfjk_get_jk(self._h, cp, int(C_occ.shape[1]), jp, kp, st), "dfjk_get_jk")
        return J, K

    # -- unrestricted: D_s = C_s C_s^T, J = J[D_a + D_b]
    def get_jk_u(self, C_a, C_b, with_j: bool = True, with_k: bool = True, stream=None):
        import torch
        for C in (C_a, C_b):
            if C.dim() != 2 or C.shape[0] != self.nao:
                raise ValueError("C_a, C_b must be nao x nocc")
        ap, bp = _dev_f64(C_a, "C_a"), _dev_f64(C_b, "C_b")
        mk = lambda: torch.empty(self.nao, self.nao, dtype=torch.float64, device=self.device)
        J = mk() if with_j else None
        Ka, Kb = (mk(), mk()) if with_k else (None, None)
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            _check(lib().dfjk_get_jk_u(self._h, ap, int(C_a.shape[1]), bp, int(C_b.shape[1]),
                                       J.data_ptr() if with_j else None,
                                       Ka.data_ptr() if with_k else None,
                                       Kb.data_ptr() if with_k else None, st), "dfjk_get_jk_u")
        return J, Ka, Kb

    # -- general densities: dm = C1 C2^T (pair) or a raw nao x nao matrix; J, K linear in dm
    def _out(self, with_it: bool, lead=()):
        import torch
        return torch.empty(*lead, self.nao, self.nao, dtype=torch.float64,
                           device=self.device) if with_it else None

    def get_jk_pair(self, C1, C2, with_j: bool = True, with_k: bool = True, stream=None):
        import torch
        if C1.dim() != 2 or C1.shape[0] != self.nao or C1.shape != C2.shape:
            raise ValueError("C1, C2 must both be nao x ncol")
        p1, p2 = _dev_f64(C1, "C1"), _dev_f64(C2, "C2")
        J, K = self._out(with_j), self._out(with_k)
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            _check(lib().dfjk_get_jk_pair(self._h, p1, p2, int(C1.shape[1]),
                                          J.data_ptr() if with_j else None,
                                          K.data_ptr() if with_k else None, st), "dfjk_get_jk_pair")
        return J, K

    def get_jk_dm(self, dm, with_j: bool = True, with_k: bool = True, stream=None):
        """dm: nao x nao (one density) or ndm x nao x nao (a batch)."""
        import torch
        batched = dm.dim() == 3
        if dm.shape[-2:] != (self.nao, self.nao) or dm.dim() not in (2, 3):
            raise ValueError("dm must be nao x nao or ndm x nao x nao")
        dp = _dev_f64(dm, "dm")
        lead = (dm.shape[0],) if batched else ()
        J, K = self._out(with_j, lead), self._out(with_k, lead)
        jp, kp = (J.data_ptr() if with_j else None), (K.data_ptr() if with_k else None)
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            if batched:
                _check(lib().dfjk_get_jk_dms(self._h, int(dm.shape[0]), dp, jp, kp, st), "dfjk_get_jk_dms")
            else:
                _check(lib().dfjk_get_jk_dm(self._h, dp, jp, kp, st), "dfjk_get_jk_dm")
        return J, K

    # -- host buffers in, host buffers out (B stays resident); synchronous
    def get_jk_host(self, C_occ_host, J_host=None, K_host=None):
        import torch
        for t, name in ((C_occ_host, "C_occ_host"), (J_host, "J_host"), (K_host, "K_host")):
            if t is not None and not (isinstance(t, torch.Tensor) and not t.is_cuda
                                      and t.dtype == torch.float64 and t.is_contiguous()):
                raise ValueError(f"{name} must be a contiguous CPU float64 tensor")
        if C_occ_host.dim() != 2 or C_occ_host.shape[0] != self.nao:
            raise ValueError("C_occ_host must be nao x nocc")
        for t in (J_host, K_host):
            if t is not None and t.numel() != self.nao * self.nao:
                raise ValueError("J_host / K_host must be nao x nao")
        with torch.cuda.device(self.device):
            _check(lib().dfjk_get_jk_host(self._h, C_occ_host.data_ptr(), int(C_occ_host.shape[1]),
                                          J_host.data_ptr() if J_host is not None else None,
                                          K_host.data_ptr() if K_host is not None else None),
                   "dfjk_get_jk_host")
        return J_host, K_host

    def scf_rhf(self, hcore, S, nocc: int, max_iter: int = 50, conv_tol: float = 1e-10,
                diis_space: int = 8, stream=None):
        """Closed-shell DF-SCF around get_jk (dfjk_scf_rhf; synchronous).  Returns a dict with
        converged, e_hist (list), C, mo_energy, D, F (device tensors)."""
        import torch
        n2 = self.nao * self.nao
        hp, sp = _dev_f64(hcore, "hcore", n2), _dev_f64(S, "S", n2)
        C, D, F = self._out(True), self._out(True), self._out(True)
        eps = torch.empty(self.nao, dtype=torch.float64, device=self.device)
        e_hist = (ctypes.c_double * int(max_iter))()
        n_iter, conv = ctypes.c_int64(0), ctypes.c_int(0)
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            _check(lib().dfjk_scf_rhf(self._h, hp, sp, int(nocc), int(max_iter), float(conv_tol),
                                      int(diis_space), C.data_ptr(), eps.data_ptr(), D.data_ptr(),
                                      F.data_ptr(), e_hist, ctypes.byref(n_iter), ctypes.byref(conv), st),
                   "dfjk_scf_rhf")
        return dict(converged=bool(conv.value), e_hist=list(e_hist[:n_iter.value]), C=C,
                    mo_energy=eps, D=D, F=F, timing=self.scf_timing())

    def scf_uhf(self, hcore, S, nocc_a: int, nocc_b: int, max_iter: int = 50, conv_tol: float = 1e-10,
                diis_space: int = 8, stream=None):
        """Unrestricted DF-SCF around get_jk_u (dfjk_scf_uhf; synchronous).  Returns a dict with
        converged, e_hist and two-element lists C, mo_energy, D."""
        import torch
        n2 = self.nao * self.nao
        hp, sp = _dev_f64(hcore, "hcore", n2), _dev_f64(S, "S", n2)
        C = [self._out(True), self._out(True)]
        D = [self._out(True), self._out(True)]
        eps = [torch.empty(self.nao, dtype=torch.float64, device=self.device) for _ in range(2)]
        e_hist = (ctypes.c_double * int(max_iter))()
        n_iter, conv = ctypes.c_int64(0), ctypes.c_int(0)
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            _check(lib().dfjk_scf_uhf(self._h, hp, sp, int(nocc_a), int(nocc_b), int(max_iter),
                                      float(conv_tol), int(diis_space), C[0].data_ptr(), C[1].data_ptr(),
                                      eps[0].data_ptr(), eps[1].data_ptr(), D[0].data_ptr(), D[1].data_ptr(),
                                      e_hist, ctypes.byref(n_iter), ctypes.byref(conv), st), "dfjk_scf_uhf")
        return dict(converged=bool(conv.value), e_hist=list(e_hist[:n_iter.value]), C=C, mo_energy=eps, D=D,
                    timing=self.scf_timing())

    def scf_timing(self) -> Optional[dict]:
        """ms per iteration of the last SCF run: get_jk, eigensolver (cuSOLVER Dsygvd), everything else.
        None when the library has no valid timing on record (no run yet, or its events failed)."""
        it, a, b, c = ctypes.c_int64(0), ctypes.c_double(0), ctypes.c_double(0), ctypes.c_double(0)
        if lib().dfjk_scf_timing(self._h, ctypes.byref(it), ctypes.byref(a), ctypes.byref(b),
                                 ctypes.byref(c)) != 0:
            return None
        n = max(it.value, 1)
        return {"iterations": it.value, "get_jk": a.value / n, "eigensolver": b.value / n, "glue": c.value / n}

    def get_jk_pairs(self, C1s, C2s, with_j: bool = True, with_k: bool = True, stream=None):
        """Several factored densities dm_i = C1_i C2_i^T from one sweep over B (dfjk_get_jk_pairs): one
        half transform over all factors side by side, one axpy pass for all J_i.  ``C1s`` / ``C2s`` are
        sequences of nao x ncol_i CUDA float64 tensors.  Returns (list of J_i or None, list of K_i or None)."""
        import torch
        n = len(C1s)
        if n < 1 or len(C2s) != n:
            raise ValueError("C1s and C2s must be non-empty sequences of the same length")
        ncols = (ctypes.c_int64 * n)()
        p1, p2 = (ctypes.c_void_p * n)(), (ctypes.c_void_p * n)()
        for i, (a, b) in enumerate(zip(C1s, C2s)):
            if a.dim() != 2 or a.shape[0] != self.nao or tuple(b.shape) != tuple(a.shape):
                raise ValueError("C1_i and C2_i must both be nao x ncol_i")
            p1[i], p2[i], ncols[i] = _dev_f64(a, "C1"), _dev_f64(b, "C2"), int(a.shape[1])
        Js = [self._out(True) for _ in range(n)] if with_j else None
        Ks = [self._out(True) for _ in range(n)] if with_k else None
        pj = (ctypes.c_void_p * n)(*[t.data_ptr() for t in Js]) if with_j else None
        pk = (ctypes.c_void_p * n)(*[t.data_ptr() for t in Ks]) if with_k else None
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            _check(lib().dfjk_get_jk_pairs(self._h, n, p1, p2, ncols, pj, pk, st), "dfjk_get_jk_pairs")
        return Js, Ks

    def get_df_diag(self, stream=None):
        """diag[mu][nu] = sum_P B_P[mu,nu]^2, the DF term of Eq. 7."""
        import torch
        out = self._out(True)
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            _check(lib().dfjk_get_df_diag(self._h, out.data_ptr(), st), "dfjk_get_df_diag")
        return out

    def get_jk_u_host(self, C_a_host, C_b_host, J_host=None, K_a_host=None, K_b_host=None):
        """Unrestricted build with host orbitals / results (synchronous; B stays resident)."""
        import torch
        for t, name in ((C_a_host, "C_a_host"), (C_b_host, "C_b_host"), (J_host, "J_host"),
                        (K_a_host, "K_a_host"), (K_b_host, "K_b_host")):
            if t is not None and not (isinstance(t, torch.Tensor) and not t.is_cuda
                                      and t.dtype == torch.float64 and t.is_contiguous()):
                raise ValueError(f"{name} must be a contiguous CPU float64 tensor")
        for C in (C_a_host, C_b_host):
            if C.dim() != 2 or C.shape[0] != self.nao:
                raise ValueError("C_a_host, C_b_host must be nao x nocc")
        for t in (J_host, K_a_host, K_b_host):
            if t is not None and t.numel() != self.nao * self.nao:
                raise ValueError("J_host / K_host must be nao x nao")
        ptr = lambda t: t.data_ptr() if t is not None else None
        with torch.cuda.device(self.device):
            _check(lib().dfjk_get_jk_u_host(self._h, C_a_host.data_ptr(), int(C_a_host.shape[1]),
                                            C_b_host.data_ptr(), int(C_b_host.shape[1]),
                                            ptr(J_host), ptr(K_a_host), ptr(K_b_host)), "dfjk_get_jk_u_host")
        return J_host, K_a_host, K_b_host

    def get_d(self, stream=None):
        """Fitting coefficients d_P of the most recent J build (debug getter)."""
        import torch
        d = torch.empty(self.naux, dtype=torch.float64, device=self.device)
        with torch.cuda.device(self.device):
            st = (stream or torch.cuda.current_stream(self.device)).cuda_stream
            _check(lib().dfjk_get_d(self._h, d.data_ptr(), st), "dfjk_get_d")
        return d

    def set_option(self, name: str, value: int) -> None:
        _check(lib().dfjk_set_option(self._h, name.encode(), int(value)), "dfjk_set_option")

    @property
    def launch_count(self) -> int:
        return int(lib().dfjk_launch_count(self._h))

    def kernel_time(self, kernel: str) -> Tuple[float, int]:
        """(total ms, launches) of one kernel since ``set_option("time_kernels", 1)``."""
        ms, n = ctypes.c_double(0.0), ctypes.c_int64(0)
        _check(lib().dfjk_kernel_time(self._h, KERNELS[kernel], ctypes.byref(ms), ctypes.byref(n)),
               "dfjk_kernel_time")
        return ms.value, n.value

    @property
    def workspace_bytes(self) -> int:
        return int(lib().dfjk_workspace_bytes(self._h))

    def close(self) -> None:
        if self._h:
            import torch
            torch.cuda.synchronize(self.device)
            lib().dfjk_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
