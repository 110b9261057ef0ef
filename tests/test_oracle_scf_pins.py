"""Pins for the SCF-loop oracle (oracle/scf.py).

  * no two-electron term (B = 0): one diagonalisation, E = 2 sum_{i<nocc} eps_i of (hcore, S)
  * stationarity of the converged point: F D S = S D F, F C = S C eps, C^T S C = 1,
    tr(D S) = 2 nocc, D S D = 2 D
  * the energy formula (incl. the factor in front of K, R1) against the textbook RHF energy
    E = sum D h + 1/2 sum_{mnls} D_mn D_ls [(mn|ls) - 1/2 (ml|ns)] over the explicit 4-index tensor
  * variational: E(converged) is below E of any occupied-virtual rotation of the converged orbitals
  * plain Roothaan iteration (diis_space = 1) reaches the same energy
"""
import numpy as np
import pytest
import scipy.linalg

import dfjk_inputs as gi
import oracle
from oracle import scf


def case(nao, naux, nocc, scale, seed=3):
    cfg = gi.custom_config(nao, naux, (nocc,), seed=seed)
    return cfg, gi.fill_B_host(cfg) * scale, gi.core_hamiltonian(cfg), gi.overlap(cfg)


def rhf_energy_4index(Bp, nao, h, C_occ):
    il = np.tril_indices(nao)
    Bf = np.zeros((Bp.shape[0], nao, nao)); Bf[:, il[0], il[1]] = Bp; Bf[:, il[1], il[0]] = Bp
    eri = np.einsum("pmn,pls->mnls", Bf, Bf)                     # Eq. 1
    D = 2.0 * C_occ @ C_occ.T
    return float(np.sum(D * h) + 0.5 * np.einsum("mn,ls,mnls->", D, D, eri)
                 - 0.25 * np.einsum("mn,ls,mlns->", D, D, eri))


def test_no_two_electron_term_is_one_diagonalisation():
    cfg, Bp, h, S = case(14, 5, 3, 0.0)
    r = scf.scf_rhf(Bp, 14, h, S, 3)
    eps = scipy.linalg.eigh(h, S, eigvals_only=True)
    assert r["converged"] and len(r["e_hist"]) == 2
    assert abs(r["e_hist"][-1] - 2.0 * eps[:3].sum()) <= 1e-12 * abs(eps[:3].sum())
    assert np.allclose(r["mo_energy"], eps, rtol=0, atol=1e-12)


def test_converged_point_is_stationary():
    cfg, Bp, h, S = case(24, 70, 4, 0.25)
    r = scf.scf_rhf(Bp, 24, h, S, 4, conv_tol=1e-12)
    assert r["converged"]
    C, D, F, eps = r["C"], r["D"], r["F"], r["mo_energy"]
    assert np.abs(F @ D @ S - S @ D @ F).max() <= 1e-6
    assert np.abs(C.T @ S @ C - np.eye(24)).max() <= 1e-12
    assert abs(np.trace(D @ S) - 8.0) <= 1e-12
    assert np.abs(D @ S @ D - 2.0 * D).max() <= 1e-12
    # the last diagonalised Fock matrix is the DIIS extrapolation, which equals F at convergence
    assert np.abs(F @ C - S @ C * eps).max() <= 1e-5
    assert np.all(np.diff(r["e_hist"])[1:] <= 1e-9)               # monotone after the first step


def test_energy_formula_against_textbook_four_index():
    cfg, Bp, h, S = case(9, 20, 2, 0.3)
    r = scf.scf_rhf(Bp, 9, h, S, 2, max_iter=1)                   # E_0 of the core guess
    C0 = scipy.linalg.eigh(h, S)[1][:, :2]
    assert abs(r["e_hist"][0] - rhf_energy_4index(Bp, 9, h, C0)) <= 1e-12 * abs(r["e_hist"][0])
    r = scf.scf_rhf(Bp, 9, h, S, 2, conv_tol=1e-12)
    assert r["converged"]
    Efin = rhf_energy_4index(Bp, 9, h, r["C"][:, :2])
    assert abs(r["e_hist"][-1] - Efin) <= 1e-9 * abs(Efin)


def test_variational_minimum():
    cfg, Bp, h, S = case(10, 24, 3, 0.3)
    r = scf.scf_rhf(Bp, 10, h, S, 3, conv_tol=1e-12)
    assert r["converged"]
    C, E = r["C"], r["e_hist"][-1]
    rng = np.random.default_rng(0)
    for _ in range(6):
        A = np.zeros((10, 10))
        A[:3, 3:] = 0.05 * rng.standard_normal((3, 7))
        A -= A.T
        Crot = C @ scipy.linalg.expm(A)                           # keeps C^T S C = 1
        assert rhf_energy_4index(Bp, 10, h, Crot[:, :3]) >= E - 1e-10


def test_plain_roothaan_reaches_the_same_energy():
    cfg, Bp, h, S = case(20, 60, 4, 0.1)
    a = scf.scf_rhf(Bp, 20, h, S, 4, conv_tol=1e-11)
    b = scf.scf_rhf(Bp, 20, h, S, 4, conv_tol=1e-11, diis_space=1, max_iter=200)
    assert a["converged"] and b["converged"]
    assert abs(a["e_hist"][-1] - b["e_hist"][-1]) <= 1e-8 * abs(a["e_hist"][-1])
    assert len(a["e_hist"]) <= len(b["e_hist"])


def test_generators_for_the_scf_inputs():
    cfg = gi.custom_config(100, 10, (9,), seed=5)
    S, h = gi.overlap(cfg), gi.core_hamiltonian(cfg)
    assert np.array_equal(S, S.T) and np.array_equal(h, h.T)
    ev = np.linalg.eigvalsh(S)
    assert ev.min() > 0.5 and ev.max() / ev.min() < 100
    eps = scipy.linalg.eigh(h, S, eigvals_only=True)
    assert eps[9] - eps[8] > 1.0                                  # occupied/virtual gap


# ---------------------------------------------------------------- unrestricted
def uhf_energy_4index(Bp, nao, h, Ca, Cb):
    il = np.tril_indices(nao)
    Bf = np.zeros((Bp.shape[0], nao, nao)); Bf[:, il[0], il[1]] = Bp; Bf[:, il[1], il[0]] = Bp
    eri = np.einsum("pmn,pls->mnls", Bf, Bf)
    Da, Db = Ca @ Ca.T, Cb @ Cb.T
    Dt = Da + Db
    return float(np.sum(Dt * h) + 0.5 * np.einsum("mn,ls,mnls->", Dt, Dt, eri)
                 - 0.5 * np.einsum("mn,ls,mlns->", Da, Da, eri) - 0.5 * np.einsum("mn,ls,mlns->", Db, Db, eri))


def test_uhf_reduces_to_rhf_for_a_closed_shell():
    """nocc_a = nocc_b from the same core guess: the spin blocks stay equal, every energy equals RHF's."""
    cfg, Bp, h, S = case(20, 60, 4, 0.3)
    r = scf.scf_rhf(Bp, 20, h, S, 4)
    u = scf.scf_uhf(Bp, 20, h, S, 4, 4)
    assert u["converged"] and len(u["e_hist"]) == len(r["e_hist"])
    assert np.allclose(u["e_hist"], r["e_hist"], rtol=1e-11, atol=0)
    assert np.allclose(u["D"][0] + u["D"][1], r["D"], rtol=0, atol=1e-9)


def test_uhf_energy_formula_and_stationarity():
    cfg, Bp, h, S = case(9, 20, 3, 0.3)
    u = scf.scf_uhf(Bp, 9, h, S, 3, 1, max_iter=1)
    C0 = scipy.linalg.eigh(h, S)[1]
    E0 = uhf_energy_4index(Bp, 9, h, C0[:, :3], C0[:, :1])
    assert abs(u["e_hist"][0] - E0) <= 1e-12 * abs(E0)            # textbook UHF energy, incl. the K factors
    u = scf.scf_uhf(Bp, 9, h, S, 3, 1, conv_tol=1e-12)
    assert u["converged"]
    for s, n in ((0, 3), (1, 1)):
        C, D, F = u["C"][s], u["D"][s], u["F"][s]
        assert np.abs(F @ D @ S - S @ D @ F).max() <= 1e-6
        assert np.abs(C.T @ S @ C - np.eye(9)).max() <= 1e-12
        assert abs(np.trace(D @ S) - n) <= 1e-12
        assert np.abs(D @ S @ D - D).max() <= 1e-12                # idempotent with weight 1
    Efin = uhf_energy_4index(Bp, 9, h, u["C"][0][:, :3], u["C"][1][:, :1])
    assert abs(u["e_hist"][-1] - Efin) <= 1e-9 * abs(Efin)


def test_uhf_no_two_electron_term():
    cfg, Bp, h, S = case(12, 4, 3, 0.0)
    u = scf.scf_uhf(Bp, 12, h, S, 4, 2)
    eps = scipy.linalg.eigh(h, S, eigvals_only=True)
    assert u["converged"] and len(u["e_hist"]) == 2
    assert abs(u["e_hist"][-1] - (eps[:4].sum() + eps[:2].sum())) <= 1e-12 * abs(eps[:4].sum())
