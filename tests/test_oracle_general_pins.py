"""Pins for the general-density oracle functions (oracle_jk_dm_slab, oracle_jk_pair_slab,
oracle_bruteforce_jk_dm) -- SURVEY.md section 8f rank 1.

PAPER.md:96 (get_jk "supports an arbitrary number of density matrices")
and 377 (DF-approximated orbital Hessian of SOSCF: non-idempotent response densities).
With Eq. 1:  J[dm] = sum_P B_P <B_P, dm>,  K[dm] = sum_P B_P dm B_P.

What pins what (no test re-types the oracle's loops):
  * brute force over the explicit 4-index tensor, itself checked against einsum
  * reduction to the occupied-orbital oracle (already pinned): dm = 2 C C^T
  * the dm form against the pair form (two different formulas)
  * linearity, transpose rules, antisymmetric dm, closed forms, single-element probes
  * numpy library reductions on an independently unpacked B
"""
import numpy as np
import pytest

import dfjk_inputs as gi
import oracle

RTOL = 1e-13


def relerr(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / (nb if nb > 0 else 1.0)


def unpack_np(Bp, nao):
    il = np.tril_indices(nao)
    out = np.zeros((Bp.shape[0], nao, nao))
    out[:, il[0], il[1]] = Bp
    out[:, il[1], il[0]] = Bp
    return out


def rand_B(nao, naux, seed):
    return np.random.default_rng(seed).standard_normal((naux, nao * (nao + 1) // 2))


@pytest.mark.parametrize("nao,naux", [(1, 2), (2, 3), (5, 4), (9, 7), (12, 10)])
def test_dm_oracle_vs_bruteforce(nao, naux):
    Bp = rand_B(nao, naux, 40 + nao)
    dm = np.random.default_rng(nao).standard_normal((nao, nao))       # not symmetric
    J, K, _ = oracle.get_jk_dm(Bp, nao, dm)
    Jb, Kb = oracle.bruteforce_jk_dm(Bp, nao, dm)
    assert relerr(J, Jb) < RTOL and relerr(K, Kb) < RTOL


def test_bruteforce_dm_vs_einsum_definition():
    nao, naux = 7, 5
    Bp = rand_B(nao, naux, 3)
    dm = np.random.default_rng(9).standard_normal((nao, nao))
    Bf = unpack_np(Bp, nao)
    eri = np.einsum("pmn,pls->mnls", Bf, Bf)                            # Eq. 1
    Jb, Kb = oracle.bruteforce_jk_dm(Bp, nao, dm)
    assert relerr(Jb, np.einsum("mnls,ls->mn", eri, dm)) < RTOL
    assert relerr(Kb, np.einsum("mlns,ls->mn", eri, dm)) < RTOL


@pytest.mark.parametrize("nao,naux,ncol", [(1, 1, 1), (4, 3, 1), (6, 5, 6), (10, 8, 3), (11, 4, 14)])
def test_pair_oracle_vs_bruteforce_and_dm_form(nao, naux, ncol):
    rng = np.random.default_rng(5 * nao + ncol)
    Bp = rand_B(nao, naux, 70 + nao)
    C1, C2 = rng.standard_normal((nao, ncol)), rng.standard_normal((nao, ncol))
    J, K, d = oracle.get_jk_pair(Bp, nao, C1, C2)
    dm = C1 @ C2.T
    Jb, Kb = oracle.bruteforce_jk_dm(Bp, nao, dm)
    assert relerr(J, Jb) < RTOL and relerr(K, Kb) < RTOL
    Jd, Kd, dd = oracle.get_jk_dm(Bp, nao, dm)
    assert relerr(J, Jd) < RTOL and relerr(K, Kd) < RTOL and relerr(d, dd) < RTOL


def test_reduces_to_occupied_orbital_oracle():
    """dm = 2 C C^T: J equal, K[dm] = 2 K of get_jk (reading R1: K there carries no factor 2);
    pair(C, C) gives K of get_jk exactly and J of the weight-1 density."""
    cfg = gi.CONFIGS[1]
    Bp = gi.fill_B_host(cfg)
    C = gi.orbitals(cfg, 0)[0]
    J0, K0, d0 = oracle.get_jk(Bp, cfg.nao, [C], [2.0])
    J, K, d = oracle.get_jk_dm(Bp, cfg.nao, 2.0 * C @ C.T)
    assert relerr(J, J0) < RTOL and relerr(K, 2.0 * K0[0]) < RTOL and relerr(d, d0) < RTOL
    Jp, Kp, _ = oracle.get_jk_pair(Bp, cfg.nao, C, C)
    assert relerr(Kp, K0[0]) < RTOL and relerr(Jp, 0.5 * J0) < RTOL


def test_linearity_and_transpose_rules():
    nao, naux = 10, 6
    rng = np.random.default_rng(12)
    Bp = rand_B(nao, naux, 8)
    A, Bm = rng.standard_normal((nao, nao)), rng.standard_normal((nao, nao))
    Ja, Ka, _ = oracle.get_jk_dm(Bp, nao, A)
    Jb, Kb, _ = oracle.get_jk_dm(Bp, nao, Bm)
    Jc, Kc, _ = oracle.get_jk_dm(Bp, nao, 0.7 * A - 1.3 * Bm)
    assert relerr(Jc, 0.7 * Ja - 1.3 * Jb) < RTOL and relerr(Kc, 0.7 * Ka - 1.3 * Kb) < RTOL
    Jt, Kt, _ = oracle.get_jk_dm(Bp, nao, A.T)
    assert relerr(Jt, Ja) < RTOL                  # J sees only the symmetric part of dm
    assert relerr(Kt, Ka.T) < RTOL                # K[dm^T] = K[dm]^T
    assert np.abs(Ja - Ja.T).max() <= 1e-14 * np.abs(Ja).max()
    # antisymmetric dm: J = 0 exactly up to rounding, K antisymmetric
    S = A - A.T
    Js, Ks, ds = oracle.get_jk_dm(Bp, nao, S)
    assert np.abs(ds).max() <= 1e-13 * np.abs(S).max() * np.abs(Bp).max() * nao * nao
    assert relerr(Ks, -Ks.T) < RTOL
    # pair: swapping the factors transposes K
    C1, C2 = rng.standard_normal((nao, 4)), rng.standard_normal((nao, 4))
    _, K12, _ = oracle.get_jk_pair(Bp, nao, C1, C2)
    _, K21, _ = oracle.get_jk_pair(Bp, nao, C2, C1)
    assert relerr(K21, K12.T) < RTOL


def test_closed_forms_general():
    """B_P = a_P I  =>  J = (sum a^2) tr(dm) I, K = (sum a^2) dm;
    B_P = u_P u_P^T  =>  J = K^sym-like: K = sum (u^T dm u) u u^T = J."""
    nao, naux = 8, 5
    rng = np.random.default_rng(13)
    a = rng.uniform(0.1, 1.0, naux)
    Bp = np.zeros((naux, nao * (nao + 1) // 2))
    for m in range(nao):
        Bp[:, m * (m + 1) // 2 + m] = a
    dm = rng.standard_normal((nao, nao))
    J, K, d = oracle.get_jk_dm(Bp, nao, dm)
    s = (a ** 2).sum()
    assert relerr(d, a * np.trace(dm)) < RTOL
    assert relerr(J, s * np.trace(dm) * np.eye(nao)) < RTOL
    assert relerr(K, s * dm) < RTOL
    U = rng.standard_normal((naux, nao))
    il = np.tril_indices(nao)
    Bp = np.stack([np.outer(u, u)[il] for u in U])
    J, K, d = oracle.get_jk_dm(Bp, nao, dm)
    q = np.array([u @ dm @ u for u in U])
    ref = sum(qp * np.outer(u, u) for qp, u in zip(q, U))
    assert relerr(d, q) < RTOL and relerr(J, ref) < RTOL and relerr(K, ref) < RTOL


def test_single_element_probes_general():
    """One packed entry at (P, mu, nu) and one dm entry at (l, s): the lit J/K entries by hand."""
    nao = 4
    for mu in range(nao):
        for nu in range(mu + 1):
            Bp = np.zeros((1, nao * (nao + 1) // 2))
            Bp[0, mu * (mu + 1) // 2 + nu] = 2.0
            E = np.zeros((nao, nao)); E[mu, nu] = E[nu, mu] = 2.0
            for l in range(nao):
                for s in range(nao):
                    dm = np.zeros((nao, nao)); dm[l, s] = 3.0
                    J, K, d = oracle.get_jk_dm(Bp, nao, dm)
                    assert d[0] == 3.0 * E[l, s]
                    assert np.array_equal(J, 3.0 * E[l, s] * E)
                    assert np.array_equal(K, 3.0 * np.outer(E[:, l], E[:, s]))


@pytest.mark.parametrize("cfg_id", [1])
def test_library_reduction_general(cfg_id):
    cfg = gi.CONFIGS[cfg_id]
    Bp = gi.fill_B_host(cfg)
    nao = cfg.nao
    rng = np.random.default_rng(17)
    dm = rng.standard_normal((nao, nao))
    J, K, d = oracle.get_jk_dm(Bp, nao, dm)
    Bf = unpack_np(Bp, nao)
    dref = np.einsum("pls,ls->p", Bf, dm)
    assert relerr(d, dref) < 1e-12
    assert relerr(J, np.einsum("p,pmn->mn", dref, Bf)) < 1e-12
    assert relerr(K, sum(Bf[p] @ dm @ Bf[p] for p in range(cfg.naux))) < 1e-12
    C1, C2 = rng.standard_normal((nao, 7)), rng.standard_normal((nao, 7))
    Jp, Kp, _ = oracle.get_jk_pair(Bp, nao, C1, C2)
    X1, X2 = Bf @ C1, Bf @ C2
    assert relerr(Kp, np.einsum("pmi,pni->mn", X1, X2)) < 1e-12
    assert relerr(Jp, np.einsum("p,pmn->mn", np.einsum("pls,ls->p", Bf, C1 @ C2.T), Bf)) < 1e-12


# ---------------------------------------------------------------- Eq. 7 DF diagonal
def test_df_diag_pins():
    """oracle.df_diag against the materialised (mn|mn) of the brute force, numpy, the trace
    identity and K[C = I]'s diagonal (K = sum_P B_P^2  =>  K[m][m] = sum_n diag[m][n])."""
    nao, naux = 9, 6
    Bp = rand_B(nao, naux, 23)
    diag = oracle.df_diag(Bp, nao)
    _, _, diag_bf = oracle.bruteforce_jk(Bp, nao, [np.eye(nao)], [2.0])
    assert relerr(diag, diag_bf) < RTOL
    Bf = unpack_np(Bp, nao)
    assert relerr(diag, (Bf ** 2).sum(0)) < RTOL
    assert np.array_equal(diag, diag.T)
    assert abs(diag.sum() - sum(np.linalg.norm(Bf[p]) ** 2 for p in range(naux))) <= 1e-12 * diag.sum()
    _, K, _ = oracle.get_jk(Bp, nao, [np.eye(nao)], [2.0])
    assert relerr(diag.sum(1), np.diag(K[0])) < RTOL
    # slab accumulation
    acc = oracle.df_diag(Bp[:2], nao)
    oracle.df_diag(Bp[2:], nao, out=acc)
    assert relerr(acc, diag) < RTOL
    # single-element probe
    Bp1 = np.zeros((2, nao * (nao + 1) // 2)); Bp1[1, 4 * 5 // 2 + 2] = 3.0     # (mu, nu) = (4, 2)
    d1 = oracle.df_diag(Bp1, nao)
    ref = np.zeros((nao, nao)); ref[4, 2] = ref[2, 4] = 9.0
    assert np.array_equal(d1, ref)


def test_pair_form_is_the_orbital_derivative_of_the_occupied_build():
    """What the DF orbital Hessian of SOSCF contracts: for an orbital change
    C -> C + eps V the restricted build changes, to first order, by the PAIR build of (C, V):
        dJ = 4 eps J[C V^T],   dK = eps (K[C V^T] + K[C V^T]^T).
    J and K are exactly quadratic in C, so a central difference gives the derivative up to rounding;
    this pins oracle_jk_pair_slab against oracle_jk_slab (two different code paths)."""
    nao, naux, nocc = 12, 9, 3
    rng = np.random.default_rng(44)
    Bp = rand_B(nao, naux, 5)
    C = np.linalg.qr(rng.standard_normal((nao, nocc)))[0]
    V = rng.standard_normal((nao, nocc))
    eps = 1e-3
    Jp, Kp, _ = oracle.get_jk(Bp, nao, [C + eps * V], [2.0])
    Jm, Km, _ = oracle.get_jk(Bp, nao, [C - eps * V], [2.0])
    J1, K1, _ = oracle.get_jk_pair(Bp, nao, C, V)
    assert relerr((Jp - Jm) / (2 * eps), 4.0 * J1) < 1e-10
    assert relerr((Kp[0] - Km[0]) / (2 * eps), K1 + K1.T) < 1e-10
