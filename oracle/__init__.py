"""CPU oracle for the DF-JK hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes binding over ``oracle/dfjk_oracle.c`` (plain C loops, FP64, OpenMP).
Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` may import this package.  It imports
nothing from ``paper_2506_06661_b200`` and the product never imports it.

Definitions and citations live in the C file header (Eq. 1-3,
PAPER.md:96/126-131 ``get_jk``; BASELINE.json north_star for the J/K formulas).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dfjk_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_dfjk.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc: no fast-math, no reassociation, no FMA contraction
    (-ffp-contract=off), AVX2 code generation (x86-64-v3: any host of the last decade) so that the
    axpy-shaped inner loops vectorise.  The results are bit-for-bit those of a plain -O2 build
    (element-wise vectorisation does not reorder any sum); only the full-size parity tests get
    shorter (SURVEY.md section 7 step 1 builds the oracle with -O3 and native vectors)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    subprocess.run(build_command(_LIB, vector=host_has_avx2()), check=True)
    return _LIB


def host_has_avx2() -> bool:
    """True when /proc/cpuinfo lists avx2 and fma (what -march=x86-64-v3 code needs to run)."""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = set(line.split(":", 1)[1].split())
                    return {"avx2", "fma", "bmi2"} <= flags
    except OSError:
        pass
    return False


def build_command(out: str, vector: bool) -> list:
    """The gcc line of the oracle: the AVX2 build (``vector``) or the portable -O2 one a host
    without AVX2 falls back to.  Same arithmetic either way: no fast-math, no reassociation,
    -ffp-contract=off (tests/test_oracle_pins.py compares the two builds bit for bit)."""
    opt = ["-O3", "-march=x86-64-v3"] if vector else ["-O2"]
    return ["gcc", *opt, "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall", "-o", out, _SRC, "-lm"]


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = _open(_LIB)
    return _lib


def _open(path: str):
    """dlopen one build of the oracle and declare its signatures."""
    lib = ctypes.CDLL(path)
    pp = ctypes.POINTER(ctypes.c_void_p)
    lib.oracle_num_threads.restype = ctypes.c_int
    lib.oracle_jk_slab.restype = ctypes.c_int
    lib.oracle_jk_slab.argtypes = [
        ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int,
        pp, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, pp,
        ctypes.c_void_p]
    lib.oracle_bruteforce_jk.restype = ctypes.c_int
    lib.oracle_bruteforce_jk.argtypes = [
        ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int,
        pp, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, pp,
        ctypes.c_void_p]
    lib.oracle_kv_slab.restype = ctypes.c_int
    lib.oracle_kv_slab.argtypes = [
        ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int,
        pp, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, pp]
    lib.oracle_jk_dm_slab.restype = ctypes.c_int
    lib.oracle_jk_dm_slab.argtypes = [
        ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p,
        ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    lib.oracle_jk_pair_slab.restype = ctypes.c_int
    lib.oracle_jk_pair_slab.argtypes = [
        ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int64,
        ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
        ctypes.c_void_p]
    lib.oracle_bruteforce_jk_dm.restype = ctypes.c_int
    lib.oracle_bruteforce_jk_dm.argtypes = [
        ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p,
        ctypes.c_void_p, ctypes.c_void_p]
    lib.oracle_df_diag_slab.restype = ctypes.c_int
    lib.oracle_df_diag_slab.argtypes = [ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p,
                                        ctypes.c_void_p]
    lib.oracle_cholesky_lower.restype = ctypes.c_int
    lib.oracle_cholesky_lower.argtypes = [ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
    lib.oracle_whiten.restype = ctypes.c_int
    lib.oracle_whiten.argtypes = [ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p,
                                  ctypes.c_void_p, ctypes.c_void_p]
    return lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _f64c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr_array(arrs: Sequence[Optional[np.ndarray]]):
    out = (ctypes.c_void_p * len(arrs))()
    for i, a in enumerate(arrs):
        out[i] = None if a is None else a.ctypes.data
    return out


def _check_inputs(Bp, nao, Cs):
    npair = nao * (nao + 1) // 2
    if Bp.ndim != 2 or Bp.shape[1] != npair:
        raise ValueError(f"Bp must be [rows][{npair}], got {Bp.shape}")
    for C in Cs:
        if C.ndim != 2 or C.shape[0] != nao or C.shape[1] < 1:
            raise ValueError("each C must be nao x nocc with nocc >= 1")


class JKAccumulator:
    """Feed packed-B slabs, get J and K_s (oracle_jk_slab; P outermost).

    ``Cs`` is a list of nao x nocc_s arrays, ``w`` their density weights
    (restricted: one set, w=[2.0]; unrestricted: two sets, w=[1.0, 1.0]).
    """

    def __init__(self, nao: int, Cs: Sequence[np.ndarray], w: Sequence[float],
                 with_j: bool = True, with_k: bool = True):
        self.nao = int(nao)
        self.Cs = [_f64c(C) for C in Cs]
        self.w = _f64c(np.asarray(w, dtype=np.float64))
        if len(self.w) != len(self.Cs):
            raise ValueError("one weight per orbital set")
        self.nocc = np.asarray([C.shape[1] for C in self.Cs], dtype=np.int64)
        self.J = np.zeros((nao, nao)) if with_j else None
        self.K = [np.zeros((nao, nao)) for _ in self.Cs] if with_k else None
        self.d = []

    def add_slab(self, Bp_slab: np.ndarray) -> None:
        Bp_slab = _f64c(Bp_slab)
        _check_inputs(Bp_slab, self.nao, self.Cs)
        nrows = Bp_slab.shape[0]
        d = np.zeros(nrows)
        Cp = _ptr_array(self.Cs)
        Kp = _ptr_array(self.K) if self.K is not None else None
        rc = _load().oracle_jk_slab(
            nrows, self.nao, Bp_slab.ctypes.data, len(self.Cs), Cp,
            self.nocc.ctypes.data, self.w.ctypes.data,
            None if self.J is None else self.J.ctypes.data, Kp, d.ctypes.data)
        if rc != 0:
            raise RuntimeError(f"oracle_jk_slab failed: {rc}")
        self.d.append(d)

    def d_vector(self) -> np.ndarray:
        return np.concatenate(self.d) if self.d else np.zeros(0)


def get_jk(Bp: np.ndarray, nao: int, Cs: Sequence[np.ndarray], w: Sequence[float],
           with_j: bool = True, with_k: bool = True):
    """Whole-tensor convenience: returns (J, [K_s], d)."""
    acc = JKAccumulator(nao, Cs, w, with_j, with_k)
    acc.add_slab(Bp)
    return acc.J, acc.K, acc.d_vector()


def get_jk_restricted(Bp: np.ndarray, nao: int, C_occ: np.ndarray):
    """D = 2 C C^T (BASELINE.json north_star): returns (J, K)."""
    J, K, _ = get_jk(Bp, nao, [C_occ], [2.0])
    return J, K[0]


def get_jk_unrestricted(Bp: np.ndarray, nao: int, C_a: np.ndarray, C_b: np.ndarray):
    """D_s = C_s C_s^T, J = J[D_a + D_b] (reading R7): returns (J, K_a, K_b)."""
    J, K, _ = get_jk(Bp, nao, [C_a, C_b], [1.0, 1.0])
    return J, K[0], K[1]


def bruteforce_jk(Bp: np.ndarray, nao: int, Cs: Sequence[np.ndarray],
                  w: Sequence[float]):
    """Explicit 4-index tensor (Eq. 1 materialised), tiny inputs only.

    Returns (J, [K_s], diag) with diag[m][n] = (mn|mn)_DF (Eq. 7's second term).
    """
    Bp = _f64c(Bp)
    Cs = [_f64c(C) for C in Cs]
    _check_inputs(Bp, nao, Cs)
    wv = _f64c(np.asarray(w, dtype=np.float64))
    nocc = np.asarray([C.shape[1] for C in Cs], dtype=np.int64)
    J = np.zeros((nao, nao))
    K = [np.zeros((nao, nao)) for _ in Cs]
    diag = np.zeros((nao, nao))
    rc = _load().oracle_bruteforce_jk(
        Bp.shape[0], nao, Bp.ctypes.data, len(Cs), _ptr_array(Cs),
        nocc.ctypes.data, wv.ctypes.data, J.ctypes.data, _ptr_array(K),
        diag.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_bruteforce_jk failed: {rc}")
    return J, K, diag


class KVAccumulator:
    """K_s @ V from the definition, slab by slab (oracle_kv_slab)."""

    def __init__(self, nao: int, Cs: Sequence[np.ndarray], V: np.ndarray):
        self.nao = int(nao)
        self.Cs = [_f64c(C) for C in Cs]
        self.nocc = np.asarray([C.shape[1] for C in self.Cs], dtype=np.int64)
        self.V = _f64c(V)            # [nvec][nao]
        if self.V.ndim != 2 or self.V.shape[1] != nao:
            raise ValueError("V must be [nvec][nao]")
        self.KV = [np.zeros_like(self.V) for _ in self.Cs]

    def add_slab(self, Bp_slab: np.ndarray) -> None:
        Bp_slab = _f64c(Bp_slab)
        _check_inputs(Bp_slab, self.nao, self.Cs)
        rc = _load().oracle_kv_slab(
            Bp_slab.shape[0], self.nao, Bp_slab.ctypes.data, len(self.Cs),
            _ptr_array(self.Cs), self.nocc.ctypes.data, self.V.shape[0],
            self.V.ctypes.data, _ptr_array(self.KV))
        if rc != 0:
            raise RuntimeError(f"oracle_kv_slab failed: {rc}")


class KBlockAccumulator:
    """Sampled entries of K_s, one by one from the definition (numpy, FP64).

    For a list of row indices S this accumulates, slab by slab,
        K_s[a][b] = sum_P sum_i X_P[S_a][i] X_P[S_b][i],   X_P[mu][i] = sum_nu B(P,mu,nu) C_s[nu][i]
    (the K of the C file header restricted to the |S| x |S| block), with
    B(P,mu,nu) = Bp[P][max(max+1)/2 + min] unpacked by explicit index arithmetic.  Used for
    full-size parity (cfg 3-5) where the whole K is too slow on a CPU; pinned against the
    full oracle K in tests/test_oracle_pins.py.
    """

    def __init__(self, nao: int, Cs: Sequence[np.ndarray], rows: Sequence[int]):
        self.nao = int(nao)
        self.Cs = [_f64c(C) for C in Cs]
        self.rows = np.asarray(rows, dtype=np.int64)
        mu = self.rows[:, None]
        nu = np.arange(self.nao, dtype=np.int64)[None, :]
        a, b = np.maximum(mu, nu), np.minimum(mu, nu)
        self.idx = a * (a + 1) // 2 + b                  # [|S|][nao] packed index of B(P, S_a, nu)
        self.K = [np.zeros((len(self.rows), len(self.rows))) for _ in self.Cs]

    def add_slab(self, Bp_slab: np.ndarray) -> None:
        Bp_slab = np.asarray(Bp_slab, dtype=np.float64)
        for P in range(Bp_slab.shape[0]):
            Bsel = Bp_slab[P][self.idx]                  # [|S|][nao]
            for s, C in enumerate(self.Cs):
                X = Bsel @ C                             # [|S|][nocc]
                self.K[s] += X @ X.T


# ---------------------------------------------------------------- general densities
def get_jk_dm(Bp: np.ndarray, nao: int, dm: np.ndarray, with_j: bool = True,
              with_k: bool = True):
    """J[dm], K[dm] (both linear in dm, any real nao x nao dm; oracle_jk_dm_slab).

    Returns (J, K, d).  PAPER.md:96 ("arbitrary number of density matrices").
    """
    Bp, dm = _f64c(Bp), _f64c(dm)
    _check_inputs(Bp, nao, [])
    if dm.shape != (nao, nao):
        raise ValueError("dm must be nao x nao")
    J = np.zeros((nao, nao)) if with_j else None
    K = np.zeros((nao, nao)) if with_k else None
    d = np.zeros(Bp.shape[0])
    rc = _load().oracle_jk_dm_slab(
        Bp.shape[0], nao, Bp.ctypes.data, dm.ctypes.data,
        None if J is None else J.ctypes.data, None if K is None else K.ctypes.data,
        d.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_jk_dm_slab failed: {rc}")
    return J, K, d


def get_jk_pair(Bp: np.ndarray, nao: int, C1: np.ndarray, C2: np.ndarray,
                with_j: bool = True, with_k: bool = True):
    """dm = C1 C2^T given by its factors: K = sum_P (B_P C1)(B_P C2)^T, J = J[dm]
    (oracle_jk_pair_slab).  Returns (J, K, d)."""
    Bp, C1, C2 = _f64c(Bp), _f64c(C1), _f64c(C2)
    _check_inputs(Bp, nao, [C1, C2])
    if C1.shape != C2.shape:
        raise ValueError("C1 and C2 must have the same shape")
    J = np.zeros((nao, nao)) if with_j else None
    K = np.zeros((nao, nao)) if with_k else None
    d = np.zeros(Bp.shape[0])
    rc = _load().oracle_jk_pair_slab(
        Bp.shape[0], nao, Bp.ctypes.data, C1.shape[1], C1.ctypes.data, C2.ctypes.data,
        None if J is None else J.ctypes.data, None if K is None else K.ctypes.data,
        d.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_jk_pair_slab failed: {rc}")
    return J, K, d


def bruteforce_jk_dm(Bp: np.ndarray, nao: int, dm: np.ndarray):
    """Eq. 1 materialised + textbook J/K with an arbitrary dm (tiny inputs).  Returns (J, K)."""
    Bp, dm = _f64c(Bp), _f64c(dm)
    _check_inputs(Bp, nao, [])
    J, K = np.zeros((nao, nao)), np.zeros((nao, nao))
    rc = _load().oracle_bruteforce_jk_dm(Bp.shape[0], nao, Bp.ctypes.data, dm.ctypes.data,
                                         J.ctypes.data, K.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_bruteforce_jk_dm failed: {rc}")
    return J, K


def df_diag(Bp: np.ndarray, nao: int, out: Optional[np.ndarray] = None) -> np.ndarray:
    """diag[m][n] (+)= sum_P B(P,m,n)^2 -- the DF term of Eq. 7.
    Pass ``out`` to accumulate slab by slab."""
    Bp = _f64c(Bp)
    _check_inputs(Bp, nao, [])
    diag = np.zeros((nao, nao)) if out is None else out
    rc = _load().oracle_df_diag_slab(Bp.shape[0], nao, Bp.ctypes.data, diag.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_df_diag_slab failed: {rc}")
    return diag


# ---------------------------------------------------------------- building B (Eq. 2-3)
def cholesky_lower(M: np.ndarray) -> np.ndarray:
    """L with M = L L^T (Eq. 2), textbook recurrence; raises if M is not SPD."""
    M = _f64c(M)
    if M.ndim != 2 or M.shape[0] != M.shape[1]:
        raise ValueError("M must be square")
    L = np.zeros_like(M)
    rc = _load().oracle_cholesky_lower(M.shape[0], M.ctypes.data, L.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_cholesky_lower failed: {rc} (not positive definite?)")
    return L


def whiten(L: np.ndarray, R: np.ndarray) -> np.ndarray:
    """B = L^-1 R by forward substitution per column (Eq. 3).
    R is [naux][ncols] (the packed raw 3-centre tensor (Q|mu nu))."""
    L, R = _f64c(L), _f64c(R)
    if R.ndim != 2 or L.shape != (R.shape[0], R.shape[0]):
        raise ValueError("L must be naux x naux and R naux x ncols")
    B = np.empty_like(R)
    rc = _load().oracle_whiten(R.shape[0], R.shape[1], L.ctypes.data, R.ctypes.data, B.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_whiten failed: {rc}")
    return B


def build_b(M: np.ndarray, R: np.ndarray):
    """Eq. 2-3 together: returns (L, B)."""
    L = cholesky_lower(M)
    return L, whiten(L, R)
