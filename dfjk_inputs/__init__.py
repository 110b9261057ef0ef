"""Seeded synthetic inputs for the DF-JK hot path (BASELINE.json configs 1-5).

INPUT GENERATION ONLY: this package holds none of the method's arithmetic (no
density, no contraction).  It serves the oracle's tests, the CUDA parity tests,
``smoke()`` and ``bench.py`` with the same bytes; it imports neither ``oracle``
nor ``paper_2506_06661_b200``.

Recipe (BASELINE.json ``configs``):
  x_mu = sort(U(0,10));  a_P = U(0.05,1) exp(-P/naux);  z ~ N(0,1) per packed index
  Bp[P][mu(mu+1)/2+nu] = a_P exp(-(x_mu-x_nu)^2/4) (1 + 0.1 z)
  C_occ = Q of QR(N(0,1)^{nao x nocc});  later calls either fresh (cfg 2) or
  C_{k+1} = orth(exp(eps A_k) C_k), A_k antisymmetric N(0,1), eps = 1e-2 (cfg 3-5).
These stand in for the real-molecule DF tensors the paper runs on (PAPER.md:106,
312, 295), which need PySCF/libcint and basis-set data that are not available.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import List, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_HOST_LIB = os.path.join(_HERE, "libdfjk_gen_host.so")
_DEV_LIB = os.path.join(_HERE, "libdfjk_gen_device.so")
_host = None
_dev = None

STREAM_X, STREAM_A, STREAM_Z, STREAM_Y, STREAM_C, STREAM_ROT = 0, 1, 2, 3, 10, 1000


@dataclass(frozen=True)
class Config:
    index: int
    name: str
    seed: int
    nao: int
    naux: int
    nocc: Tuple[int, ...]          # one entry restricted, two unrestricted
    calls: int
    schedule: str                  # "single" | "fresh" | "rotate"

    @property
    def npair(self) -> int:
        return self.nao * (self.nao + 1) // 2

    @property
    def b_bytes(self) -> int:
        return self.naux * self.npair * 8

    @property
    def weights(self) -> Tuple[float, ...]:
        return (2.0,) if len(self.nocc) == 1 else (1.0,) * len(self.nocc)


CONFIGS = {
    1: Config(1, "tiny", 0, 48, 160, (5,), 1, "single"),
    2: Config(2, "small", 1, 290, 900, (25,), 10, "fresh"),
    3: Config(3, "medium", 2, 800, 2600, (66,), 10, "rotate"),
    4: Config(4, "large", 3, 1600, 5000, (130,), 5, "rotate"),
    5: Config(5, "unrestricted", 4, 2000, 6000, (170, 160), 3, "rotate"),
    # not a BASELINE.json config: the LRDF shape of PAPER.md:433-450 ("the auxiliary dimension
    # needed is approximately only 1/10 of the size of the orbital basis"): few, long rows
    6: Config(6, "lrdf-shape", 5, 4000, 400, (330,), 3, "rotate"),
}


def custom_config(nao: int, naux: int, nocc, seed: int = 7, calls: int = 1,
                  schedule: str = "fresh", name: str = "custom") -> Config:
    nocc = tuple(int(n) for n in (nocc if isinstance(nocc, (tuple, list)) else (nocc,)))
    return Config(0, name, seed, int(nao), int(naux), nocc, calls, schedule)


def build(force: bool = False) -> None:
    """Compile the host (gcc) and device (nvcc, sm_100a) generator libraries."""
    core = os.path.join(_HERE, "gen_core.h")
    src = os.path.join(_HERE, "gen_host.c")
    if force or not os.path.exists(_HOST_LIB) or \
            os.path.getmtime(_HOST_LIB) < max(os.path.getmtime(src), os.path.getmtime(core)):
        subprocess.run(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall",
                        "-o", _HOST_LIB, src, "-lm"], check=True)
    src = os.path.join(_HERE, "gen_device.cu")
    if force or not os.path.exists(_DEV_LIB) or \
            os.path.getmtime(_DEV_LIB) < max(os.path.getmtime(src), os.path.getmtime(core)):
        subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3",
                        "-lineinfo", "-shared", "-Xcompiler", "-fPIC",
                        "-o", _DEV_LIB, src], check=True)


def _hostlib():
    global _host
    if _host is None:
        if not os.path.exists(_HOST_LIB):
            build()
        lib = ctypes.CDLL(_HOST_LIB)
        lib.gen_uniform.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int64, ctypes.c_void_p]
        lib.gen_normals.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int64, ctypes.c_void_p]
        lib.gen_bits_host.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int64, ctypes.c_void_p]
        lib.gen_fill_B_rows_host.restype = ctypes.c_int
        lib.gen_fill_B_rows_host.argtypes = [
            ctypes.c_uint64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p]
        _host = lib
    return _host


def _devlib():
    global _dev
    if _dev is None:
        if not os.path.exists(_DEV_LIB):
            build()
        lib = ctypes.CDLL(_DEV_LIB)
        lib.gen_fill_B_rows_device.restype = ctypes.c_int
        lib.gen_fill_B_rows_device.argtypes = [
            ctypes.c_uint64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
        _dev = lib
    return _dev


def uniform(seed: int, stream: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _hostlib().gen_uniform(seed, stream, n, out.ctypes.data)
    return out


def normals(seed: int, stream: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _hostlib().gen_normals(seed, stream, n, out.ctypes.data)
    return out


def raw_bits(seed: int, stream: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.uint64)
    _hostlib().gen_bits_host(seed, stream, n, out.ctypes.data)
    return out


def centers(cfg: Config) -> np.ndarray:
    """x_mu = sorted U(0,10)."""
    return np.sort(10.0 * uniform(cfg.seed, STREAM_X, cfg.nao))


def aux_scales(cfg: Config) -> np.ndarray:
    """a_P = U(0.05,1) exp(-P/naux), P zero-based."""
    u = uniform(cfg.seed, STREAM_A, cfg.naux)
    P = np.arange(cfg.naux, dtype=np.float64)
    return (0.05 + 0.95 * u) * np.exp(-P / cfg.naux)


def fill_B_host(cfg: Config, P0: int = 0, nrows: int | None = None) -> np.ndarray:
    """Rows P0..P0+nrows-1 of packed B as a [nrows][npair] float64 array (canonical)."""
    if nrows is None:
        nrows = cfg.naux - P0
    x, a = centers(cfg), aux_scales(cfg)
    out = np.empty((nrows, cfg.npair), dtype=np.float64)
    rc = _hostlib().gen_fill_B_rows_host(cfg.seed, cfg.nao, x.ctypes.data, a.ctypes.data,
                                         P0, nrows, out.ctypes.data)
    if rc != 0:
        raise MemoryError("gen_fill_B_rows_host")
    return out


def fill_B_device(cfg: Config, out, P0: int = 0, nrows: int | None = None) -> None:
    """Fill a CUDA torch tensor ``out`` ([nrows][npair], float64, contiguous) in place."""
    import torch
    if nrows is None:
        nrows = cfg.naux - P0
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous()
    assert out.numel() == nrows * cfg.npair
    x = torch.from_numpy(centers(cfg)).to(out.device)
    a = torch.from_numpy(aux_scales(cfg)).to(out.device)
    stream = torch.cuda.current_stream(out.device).cuda_stream
    rc = _devlib().gen_fill_B_rows_device(cfg.seed, cfg.nao, x.data_ptr(), a.data_ptr(),
                                          P0, nrows, out.data_ptr(), stream)
    if rc != 0:
        raise RuntimeError(f"gen_fill_B_rows_device: cuda error {rc}")
    torch.cuda.current_stream(out.device).synchronize()   # x, a must outlive the kernel


def _orth(M: np.ndarray) -> np.ndarray:
    Q, _ = np.linalg.qr(M)
    return np.ascontiguousarray(Q)


def _expm_apply(cfg: Config, call: int, s: int, C: np.ndarray, eps: float = 1e-2) -> np.ndarray:
    """exp(eps A) C by a 30-term Taylor series; A antisymmetric, N(0,1) strict upper."""
    nao = cfg.nao
    G = normals(cfg.seed, STREAM_ROT + 16 * call + s, nao * nao).reshape(nao, nao)
    U = np.triu(G, 1)
    A = U - U.T
    term = C.copy()
    out = C.copy()
    for k in range(1, 31):
        term = (eps / k) * (A @ term)
        out += term
    return out


def orbitals(cfg: Config, call: int = 0) -> List[np.ndarray]:
    """Occupied-orbital blocks C_s (nao x nocc_s, C order) for SCF call ``call``."""
    out = []
    for s, nocc in enumerate(cfg.nocc):
        if cfg.schedule == "rotate":
            C = _orth(normals(cfg.seed, STREAM_C + s, cfg.nao * nocc).reshape(cfg.nao, nocc))
            for k in range(1, call + 1):
                C = _orth(_expm_apply(cfg, k, s, C))
        else:
            C = _orth(normals(cfg.seed, STREAM_C + 16 * call + s,
                              cfg.nao * nocc).reshape(cfg.nao, nocc))
        out.append(C)
    return out


def orbital_sequence(cfg: Config, ncalls: int):
    """Yield the per-call orbital blocks of calls 0..ncalls-1 (same values as ``orbitals``,
    computed incrementally; continues the schedule past ``cfg.calls``)."""
    if cfg.schedule != "rotate":
        for call in range(ncalls):
            yield orbitals(cfg, call)
        return
    cur = orbitals(cfg, 0)
    yield cur
    for k in range(1, ncalls):
        cur = [_orth(_expm_apply(cfg, k, s, C)) for s, C in enumerate(cur)]
        yield cur


def random_orbitals(nao: int, nocc: int, seed: int, orthonormal: bool = True) -> np.ndarray:
    """A free-standing nao x nocc block for tests (optionally NOT orthonormal, reading R8)."""
    M = normals(seed, STREAM_C, nao * nocc).reshape(nao, nocc)
    return _orth(M) if orthonormal else np.ascontiguousarray(M)


def metric(cfg: Config) -> np.ndarray:
    """Synthetic auxiliary metric M_PQ of Eq. 2, naux x naux, symmetric
    positive definite and moderately conditioned (the real Coulomb metric needs an integral engine):
        y_P = U(0,10) (stream 3),   M_PQ = exp(-|y_P - y_Q| / 2) + 0.1 delta_PQ
    (an exponential kernel is positive definite; the 0.1 ridge bounds cond(M) by ~(1+naux)/0.1).
    The raw 3-centre tensor (Q|mu nu) of Eq. 3 is ``fill_B_host`` / ``fill_B_device`` unchanged."""
    y = 10.0 * uniform(cfg.seed, STREAM_Y, cfg.naux)
    M = np.exp(-np.abs(y[:, None] - y[None, :]) / 2.0)
    M[np.diag_indices(cfg.naux)] += 0.1
    return np.ascontiguousarray(M)


def overlap(cfg: Config) -> np.ndarray:
    """Synthetic overlap matrix S of a non-orthogonal basis (SCF driver tests, section 8f rank 4):
    S_mn = 0.7 delta_mn + 0.3 exp(-|x_m - x_n| / 0.5) on the basis-function centres x -- symmetric,
    unit diagonal, positive definite (exponential kernel) and well conditioned."""
    x = centers(cfg)
    S = 0.3 * np.exp(-np.abs(x[:, None] - x[None, :]) / 0.5)
    S[np.diag_indices(cfg.nao)] += 0.7
    return np.ascontiguousarray(S)


def core_hamiltonian(cfg: Config) -> np.ndarray:
    """Synthetic one-electron Hamiltonian with a clear occupied/virtual gap (so that plain DIIS
    converges): every (nao // nocc)-th site is "deep", -(4 + u_m), the others are
    shallow, -(0.5 + 0.5 u_m), u = U(0,1) (stream 4); plus a short-range hopping
    -0.2 exp(-|x_m - x_n|) between different sites.  Symmetric."""
    x = centers(cfg)
    u = uniform(cfg.seed, 4, cfg.nao)
    nocc = cfg.nocc[0]
    deep = np.zeros(cfg.nao, dtype=bool)
    deep[(np.arange(nocc) * cfg.nao) // nocc] = True
    h = -0.2 * np.exp(-np.abs(x[:, None] - x[None, :]))
    h[np.diag_indices(cfg.nao)] = np.where(deep, -(4.0 + u), -(0.5 + 0.5 * u))
    return np.ascontiguousarray(h)
