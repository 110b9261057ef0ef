"""CPU oracle of the DF-RHF SCF loop around get_jk -- TEST INFRASTRUCTURE ONLY
(only tests/ may import it; it shares nothing with the CUDA path).

The paper describes the loop only in words: the mean-field object iterates Fock build ->
diagonalisation -> new density until self-consistency, with DIIS as the default accelerator
(Sec. IV.B; `mf.kernel(dm0=...)` PAPER.md:154-159) and get_jk(dm) -> (vj, vk)
as the step that costs the time.  Written out for a closed-shell
determinant in a non-orthogonal basis (textbook Roothaan-Hall + Pulay DIIS), in this order:

    0. core guess:  hcore C = S C eps                      (generalised symmetric eigenproblem)
    k. C_occ = the nocc lowest orbitals;  D = 2 C_occ C_occ^T
       J, K  = get_jk(C_occ)            (oracle.get_jk: K carries no factor 2, R1)
       F     = hcore + J - K
       E_k   = 1/2 sum_{mu nu} D_{mu nu} (hcore + F)_{mu nu}
       e     = F D S - S D F                               (DIIS error, Pulay)
       stop when k > 0, |E_k - E_{k-1}| <= conv_tol max(1, |E_k|) and max|e| <= sqrt(conv_tol)
       keep the last `diis_space` pairs (F_i, e_i);  B_ij = <e_i, e_j>;
       solve [[B, -1], [-1^T, 0]] [c; lam] = [0; -1];  F_ext = sum_i c_i F_i
       F_ext C = S C eps  -> next orbitals

Library steps: scipy.linalg.eigh (generalised eigenproblem), numpy.linalg.solve (the DIIS system),
numpy matmul.  Pins: tests/test_oracle_scf_pins.py.
"""
from __future__ import annotations

import numpy as np
import scipy.linalg

from . import get_jk


def scf_rhf(Bp, nao, hcore, S, nocc, max_iter=50, conv_tol=1e-10, diis_space=8):
    """Returns dict(converged, e_hist, C, mo_energy, D, F, err_hist)."""
    hcore = np.asarray(hcore, dtype=np.float64)
    S = np.asarray(S, dtype=np.float64)
    mo_energy, C = scipy.linalg.eigh(hcore, S)
    Fs, errs, e_hist, err_hist = [], [], [], []
    converged = False
    F = hcore
    for k in range(max_iter):
        C_occ = np.ascontiguousarray(C[:, :nocc])
        D = 2.0 * C_occ @ C_occ.T
        J, K, _ = get_jk(Bp, nao, [C_occ], [2.0])
        F = hcore + J - K[0]
        E = 0.5 * float(np.sum(D * (hcore + F)))
        e = F @ D @ S - S @ D @ F
        err = float(np.abs(e).max())
        e_hist.append(E)
        err_hist.append(err)
        if k > 0 and abs(E - e_hist[-2]) <= conv_tol * max(1.0, abs(E)) and err <= np.sqrt(conv_tol):
            converged = True
            break
        Fs.append(F)
        errs.append(e)
        if len(Fs) > diis_space:
            Fs.pop(0)
            errs.pop(0)
        m = len(Fs)
        A = np.zeros((m + 1, m + 1))
        for i in range(m):
            for j in range(m):
                A[i, j] = float(np.sum(errs[i] * errs[j]))
        A[:m, m] = A[m, :m] = -1.0
        rhs = np.zeros(m + 1)
        rhs[m] = -1.0
        c = np.linalg.solve(A, rhs)[:m]
        F_ext = sum(ci * Fi for ci, Fi in zip(c, Fs))
        mo_energy, C = scipy.linalg.eigh(F_ext, S)
    return dict(converged=converged, e_hist=np.array(e_hist), err_hist=np.array(err_hist), C=C,
                mo_energy=mo_energy, D=D, F=F)


def scf_uhf(Bp, nao, hcore, S, nocc_a, nocc_b, max_iter=50, conv_tol=1e-10, diis_space=8):
    """Unrestricted (two-spin) counterpart of scf_rhf (the paper's UKS/UHF objects, PAPER.md:172-180,
    264-293), textbook Pople-Nesbet equations with the same DIIS, on the stacked spin blocks:

        D_s = C_s,occ C_s,occ^T (weight 1);  J = J[D_a + D_b];  K_s = K[D_s]   (reading R7)
        F_s = hcore + J - K_s
        E   = 1/2 sum_s sum D_s o (hcore + F_s)
        e_s = F_s D_s S - S D_s F_s;  B_ij = <e_a^i, e_a^j> + <e_b^i, e_b^j>;  err = max_s max|e_s|
        F_s,ext = sum_i c_i F_s^i  (one coefficient vector for both spins);  F_s,ext C_s = S C_s eps_s

    Both spins start from the core guess.  Returns dict(converged, e_hist, err_hist, C, mo_energy, D, F)
    with two-element lists for the per-spin entries.
    """
    hcore = np.asarray(hcore, dtype=np.float64)
    S = np.asarray(S, dtype=np.float64)
    eps0, C0 = scipy.linalg.eigh(hcore, S)
    C = [C0, C0.copy()]
    mo_energy = [eps0, eps0.copy()]
    nocc = (int(nocc_a), int(nocc_b))
    Fs, errs, e_hist, err_hist = [], [], [], []
    converged = False
    for k in range(max_iter):
        Cocc = [np.ascontiguousarray(C[s][:, :nocc[s]]) for s in range(2)]
        D = [Cocc[s] @ Cocc[s].T for s in range(2)]
        J, K, _ = get_jk(Bp, nao, Cocc, [1.0, 1.0])
        F = [hcore + J - K[s] for s in range(2)]
        E = sum(0.5 * float(np.sum(D[s] * (hcore + F[s]))) for s in range(2))
        e = [F[s] @ D[s] @ S - S @ D[s] @ F[s] for s in range(2)]
        err = max(float(np.abs(e[s]).max()) for s in range(2))
        e_hist.append(E)
        err_hist.append(err)
        if k > 0 and abs(E - e_hist[-2]) <= conv_tol * max(1.0, abs(E)) and err <= np.sqrt(conv_tol):
            converged = True
            break
        Fs.append(F)
        errs.append(e)
        if len(Fs) > diis_space:
            Fs.pop(0)
            errs.pop(0)
        m = len(Fs)
        A = np.zeros((m + 1, m + 1))
        for i in range(m):
            for j in range(m):
                A[i, j] = sum(float(np.sum(errs[i][s] * errs[j][s])) for s in range(2))
        A[:m, m] = A[m, :m] = -1.0
        rhs = np.zeros(m + 1)
        rhs[m] = -1.0
        c = np.linalg.solve(A, rhs)[:m]
        for s in range(2):
            F_ext = sum(ci * Fi[s] for ci, Fi in zip(c, Fs))
            mo_energy[s], C[s] = scipy.linalg.eigh(F_ext, S)
    return dict(converged=converged, e_hist=np.array(e_hist), err_hist=np.array(err_hist), C=C,
                mo_energy=mo_energy, D=D, F=F)
