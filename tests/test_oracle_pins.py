"""Pins for the CPU oracle (oracle/dfjk_oracle.c) -- none of them re-types its loops.

What pins what:
  * hand-worked 2x2 fixture (tests/golden/hand_2x2.txt)
  * brute force over the explicit 4-index tensor, Eq. 1 materialised
  * closed forms A/B/C, single-element probes of the packed index
  * invariants: symmetry, K >= 0, E_J = 1/2 tr(DJ) = 1/2 sum d_P^2, tr(DK) = 2 sum ||C^T B_P C||_F^2
  * structure: column-concatenation additivity, C -> C U, permutation of P, scaling
  * library reductions (numpy DGEMV / matmul on an independently unpacked B)
  * Eq. 7 identity: (mn|mn)_DF = sum_P B_Pmn^2
A plausible slip (dropped term, wrong sign/index, transposed operand, missing
weight) fails at least one of them.
"""
import os

import numpy as np
import pytest

import dfjk_inputs as gi
import oracle

RTOL = 1e-13


def relerr(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / (nb if nb > 0 else 1.0)


def unpack_np(Bp, nao):
    """Independent unpack with numpy tril_indices."""
    il = np.tril_indices(nao)
    out = np.zeros((Bp.shape[0], nao, nao))
    out[:, il[0], il[1]] = Bp
    out[:, il[1], il[0]] = Bp
    return out


def rand_case(nao, naux, noccs, seed, orthonormal=True):
    rng = np.random.default_rng(seed)
    npair = nao * (nao + 1) // 2
    Bp = rng.standard_normal((naux, npair))
    Cs = []
    for n in noccs:
        M = rng.standard_normal((nao, n))
        Cs.append(np.linalg.qr(M)[0] if orthonormal else M)
    return Bp, [np.ascontiguousarray(C) for C in Cs]


# ---------------------------------------------------------------- golden
def test_hand_worked_fixture(repo_root):
    vals = {}
    with open(os.path.join(repo_root, "tests", "golden", "hand_2x2.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            vals[k] = np.array([float(x) for x in v])
    nao, naux, nocc = int(vals["nao"][0]), int(vals["naux"][0]), int(vals["nocc"][0])
    Bp = vals["Bp"].reshape(naux, -1)
    C = vals["C"].reshape(nao, nocc)
    J, K, d = oracle.get_jk(Bp, nao, [C], [2.0])
    assert np.array_equal(d, vals["d"])
    assert np.array_equal(J.ravel(), vals["J"])
    assert np.array_equal(K[0].ravel(), vals["K"])
    Jb, Kb, _ = oracle.bruteforce_jk(Bp, nao, [C], [2.0])
    assert np.array_equal(Jb.ravel(), vals["J"])
    assert np.array_equal(Kb[0].ravel(), vals["K"])


# ---------------------------------------------------------------- brute force
@pytest.mark.parametrize("nao,naux,noccs,w", [
    (1, 3, (1,), (2.0,)),
    (2, 1, (1,), (2.0,)),
    (5, 7, (2,), (2.0,)),
    (7, 4, (7,), (2.0,)),
    (12, 20, (3,), (2.0,)),
    (9, 11, (4, 3), (1.0, 1.0)),
    (6, 5, (2, 1, 3), (0.5, 1.5, -1.0)),
])
@pytest.mark.parametrize("orthonormal", [True, False])
def test_oracle_vs_bruteforce(nao, naux, noccs, w, orthonormal):
    Bp, Cs = rand_case(nao, naux, noccs, 100 + nao, orthonormal)
    J, K, _ = oracle.get_jk(Bp, nao, Cs, w)
    Jb, Kb, _ = oracle.bruteforce_jk(Bp, nao, Cs, w)
    assert relerr(J, Jb) < RTOL
    for s in range(len(Cs)):
        assert relerr(K[s], Kb[s]) < RTOL


def test_bruteforce_vs_einsum_definition():
    """The brute force itself against Eq. 1 + textbook J/K written with einsum."""
    nao, naux = 8, 6
    Bp, Cs = rand_case(nao, naux, (3, 2), 5, orthonormal=False)
    Bf = unpack_np(Bp, nao)
    eri = np.einsum("pmn,pls->mnls", Bf, Bf)
    w = (1.0, 1.0)
    D = sum(wi * C @ C.T for wi, C in zip(w, Cs))
    Jb, Kb, diag = oracle.bruteforce_jk(Bp, nao, Cs, w)
    assert relerr(Jb, np.einsum("mnls,ls->mn", eri, D)) < RTOL
    for s, C in enumerate(Cs):
        assert relerr(Kb[s], np.einsum("mlns,ls->mn", eri, C @ C.T)) < RTOL
    # Eq. 7: DF diagonal (mn|mn) = sum_P B_Pmn^2
    assert relerr(diag, (Bf ** 2).sum(0)) < RTOL


# ---------------------------------------------------------------- invariants
@pytest.mark.parametrize("cfg_id", [1])
def test_invariants_cfg(cfg_id):
    cfg = gi.CONFIGS[cfg_id]
    Bp = gi.fill_B_host(cfg)
    C = gi.orbitals(cfg, 0)[0]
    J, K, d = oracle.get_jk(Bp, cfg.nao, [C], [2.0])
    K = K[0]
    D = 2.0 * C @ C.T
    assert np.abs(J - J.T).max() <= 1e-14 * np.abs(J).max()
    assert np.abs(K - K.T).max() <= 1e-14 * np.abs(K).max()
    # E_J = 1/2 tr(D J) = 1/2 sum_P d_P^2
    assert abs(0.5 * np.trace(D @ J) - 0.5 * (d ** 2).sum()) <= 1e-12 * 0.5 * (d ** 2).sum()
    # tr(D K) = 2 sum_P ||C^T B_P C||_F^2
    Bf = unpack_np(Bp, cfg.nao)
    rhs = 2.0 * sum(np.linalg.norm(C.T @ Bf[p] @ C) ** 2 for p in range(cfg.naux))
    assert abs(np.trace(D @ K) - rhs) <= 1e-12 * rhs
    # K positive semidefinite
    ev = np.linalg.eigvalsh(0.5 * (K + K.T))
    assert ev.min() >= -1e-12 * np.linalg.norm(K)


def test_psd_quadratic_form_random():
    Bp, Cs = rand_case(10, 9, (4,), 77, orthonormal=False)
    _, K, _ = oracle.get_jk(Bp, 10, Cs, [2.0])
    rng = np.random.default_rng(1)
    Bf = unpack_np(Bp, 10)
    for _ in range(5):
        v = rng.standard_normal(10)
        q = v @ K[0] @ v
        ref = sum(np.linalg.norm((Bf[p] @ Cs[0]).T @ v) ** 2 for p in range(9))
        assert q >= 0 and abs(q - ref) <= 1e-12 * ref


# ---------------------------------------------------------------- closed forms
def test_closed_form_A_scaled_identity():
    """B_P = a_P I  =>  J = (sum a_P^2) * 2 nocc * I,  K = (sum a_P^2) C C^T."""
    nao, naux, nocc = 9, 6, 4
    rng = np.random.default_rng(3)
    a = rng.uniform(0.1, 1.0, naux)
    Bp = np.zeros((naux, nao * (nao + 1) // 2))
    for m in range(nao):
        Bp[:, m * (m + 1) // 2 + m] = a
    C = np.linalg.qr(rng.standard_normal((nao, nocc)))[0]
    J, K, d = oracle.get_jk(Bp, nao, [C], [2.0])
    s = (a ** 2).sum()
    assert relerr(d, a * 2 * nocc) < RTOL
    assert relerr(J, s * 2 * nocc * np.eye(nao)) < RTOL
    assert relerr(K[0], s * C @ C.T) < RTOL


def test_closed_form_B_rank_one():
    """B_P = u_P u_P^T  =>  d_P = 2 ||C^T u_P||^2, J = sum d_P u u^T, K = J / 2."""
    nao, naux, nocc = 8, 5, 3
    rng = np.random.default_rng(4)
    U = rng.standard_normal((naux, nao))
    il = np.tril_indices(nao)
    Bp = np.stack([np.outer(u, u)[il] for u in U])
    C = rng.standard_normal((nao, nocc))
    J, K, d = oracle.get_jk(Bp, nao, [C], [2.0])
    dref = np.array([2 * np.linalg.norm(C.T @ u) ** 2 for u in U])
    Jref = sum(dp * np.outer(u, u) for dp, u in zip(dref, U))
    assert relerr(d, dref) < RTOL
    assert relerr(J, Jref) < RTOL
    assert relerr(K[0], 0.5 * Jref) < RTOL


def test_closed_form_C_full_orthogonal():
    """nocc = nao, C orthogonal => D = 2I, J = 2 sum tr(B_P) B_P, K = sum B_P^2."""
    nao, naux = 7, 6
    Bp, Cs = rand_case(nao, naux, (nao,), 9)
    J, K, d = oracle.get_jk(Bp, nao, Cs, [2.0])
    Bf = unpack_np(Bp, nao)
    tr = np.trace(Bf, axis1=1, axis2=2)
    assert relerr(d, 2 * tr) < RTOL
    assert relerr(J, 2 * np.einsum("p,pmn->mn", tr, Bf)) < RTOL
    assert relerr(K[0], sum(Bf[p] @ Bf[p] for p in range(naux))) < RTOL


def test_single_element_probes_nao5():
    """One non-zero packed entry at (P, mu, nu) lights exactly the predicted J/K entries."""
    nao, naux = 5, 2
    rng = np.random.default_rng(11)
    C = rng.standard_normal((nao, 2))
    G = C @ C.T
    for mu in range(nao):
        for nu in range(mu + 1):
            Bp = np.zeros((naux, nao * (nao + 1) // 2))
            Bp[1, mu * (mu + 1) // 2 + nu] = 1.5
            E = np.zeros((nao, nao))
            E[mu, nu] = E[nu, mu] = 1.5
            J, K, d = oracle.get_jk(Bp, nao, [C], [2.0])
            assert d[0] == 0.0
            assert abs(d[1] - 2.0 * (E * G).sum()) < 1e-13
            assert relerr(J, 2.0 * (E * G).sum() * E) < RTOL
            assert relerr(K[0], E @ G @ E) < RTOL


# ---------------------------------------------------------------- structure
def test_structure_properties():
    nao, naux = 11, 8
    Bp, (C1, C2) = rand_case(nao, naux, (3, 4), 21, orthonormal=False)
    J1, K1, _ = oracle.get_jk(Bp, nao, [C1], [2.0])
    J2, K2, _ = oracle.get_jk(Bp, nao, [C2], [2.0])
    J12, K12, _ = oracle.get_jk(Bp, nao, [np.hstack([C1, C2])], [2.0])
    assert relerr(J12, J1 + J2) < RTOL              # column-concatenation additivity
    assert relerr(K12[0], K1[0] + K2[0]) < RTOL
    # two-set call == concatenated restricted call with w=1 (unrestricted J, reading R7)
    Ju, Ku, _ = oracle.get_jk(Bp, nao, [C1, C2], [1.0, 1.0])
    assert relerr(Ju, 0.5 * (J1 + J2)) < RTOL
    assert relerr(Ku[0], K1[0]) < RTOL and relerr(Ku[1], K2[0]) < RTOL
    # C -> C U, U orthogonal
    U = np.linalg.qr(np.random.default_rng(5).standard_normal((3, 3)))[0]
    Jr, Kr, _ = oracle.get_jk(Bp, nao, [C1 @ U], [2.0])
    assert relerr(Jr, J1) < RTOL and relerr(Kr[0], K1[0]) < RTOL
    # permutation of P
    perm = np.random.default_rng(6).permutation(naux)
    Jp, Kp, dp = oracle.get_jk(Bp[perm], nao, [C1], [2.0])
    assert relerr(Jp, J1) < RTOL and relerr(Kp[0], K1[0]) < RTOL
    # scaling B_P -> s B_P scales by s^2
    Js, Ks, _ = oracle.get_jk(3.0 * Bp, nao, [C1], [2.0])
    assert relerr(Js, 9.0 * J1) < RTOL and relerr(Ks[0], 9.0 * K1[0]) < RTOL
    # slab feeding == whole tensor
    acc = oracle.JKAccumulator(nao, [C1], [2.0])
    acc.add_slab(Bp[:3]); acc.add_slab(Bp[3:])
    assert relerr(acc.J, J1) < RTOL and relerr(acc.K[0], K1[0]) < RTOL


# ---------------------------------------------------------------- library reductions
@pytest.mark.parametrize("cfg_id", [1, 2])
def test_library_reduction(cfg_id):
    cfg = gi.CONFIGS[cfg_id]
    Bp = gi.fill_B_host(cfg)
    C = gi.orbitals(cfg, 0)[0]
    nao = cfg.nao
    J, K, d = oracle.get_jk(Bp, nao, [C], [2.0])
    D = 2.0 * C @ C.T
    il = np.tril_indices(nao)
    Dt = D[il] * np.where(il[0] == il[1], 1.0, 2.0)
    dref = Bp @ Dt                                  # DGEMV over the packed rows
    Jp = Bp.T @ dref
    Jref = np.zeros((nao, nao)); Jref[il] = Jp; Jref.T[il] = Jp
    assert relerr(d, dref) < 1e-12
    assert relerr(J, Jref) < 1e-12
    Kref = np.zeros((nao, nao))
    for p0 in range(0, cfg.naux, 64):
        X = unpack_np(Bp[p0:p0 + 64], nao) @ C      # [p][mu][i]
        Kref += np.einsum("pmi,pni->mn", X, X)
    assert relerr(K[0], Kref) < 1e-12


# ---------------------------------------------------------------- matvec form
def test_kv_slab_matches_full_K():
    cfg = gi.CONFIGS[1]
    Bp = gi.fill_B_host(cfg)
    Cs = gi.orbitals(cfg, 0)
    _, K, _ = oracle.get_jk(Bp, cfg.nao, Cs, [2.0])
    V = np.random.default_rng(2).standard_normal((3, cfg.nao))
    kv = oracle.KVAccumulator(cfg.nao, Cs, V)
    kv.add_slab(Bp[:50]); kv.add_slab(Bp[50:])
    assert relerr(kv.KV[0], V @ K[0]) < 1e-13       # K symmetric: rows of V K = (K v)^T
    # and from numpy, not the oracle: K v = sum_P B_P C C^T B_P v
    Bf = unpack_np(Bp, cfg.nao)
    C = Cs[0]
    ref = np.stack([sum(Bf[p] @ (C @ (C.T @ (Bf[p] @ v))) for p in range(cfg.naux)) for v in V])
    assert relerr(kv.KV[0], ref) < 1e-13


def test_kv_two_sets_nonorthonormal():
    Bp, Cs = rand_case(9, 7, (2, 5), 31, orthonormal=False)
    _, K, _ = oracle.get_jk(Bp, 9, Cs, [1.0, 1.0])
    V = np.random.default_rng(8).standard_normal((2, 9))
    kv = oracle.KVAccumulator(9, Cs, V)
    kv.add_slab(Bp)
    for s in range(2):
        assert relerr(kv.KV[s], V @ K[s]) < 1e-13


def test_argument_validation():
    Bp, Cs = rand_case(4, 3, (2,), 1)
    with pytest.raises(ValueError):
        oracle.get_jk(Bp[:, :-1], 4, Cs, [2.0])
    with pytest.raises(ValueError):
        oracle.get_jk(Bp, 4, [Cs[0][:3]], [2.0])


def test_k_block_matches_full_K():
    """KBlockAccumulator (sampled K entries from the definition) against the full oracle K
    and against numpy on an independently unpacked B."""
    cfg = gi.CONFIGS[1]
    Bp = gi.fill_B_host(cfg)
    Cs = [gi.random_orbitals(cfg.nao, 5, 3), gi.random_orbitals(cfg.nao, 3, 4, orthonormal=False)]
    _, K, _ = oracle.get_jk(Bp, cfg.nao, Cs, [1.0, 1.0])
    rows = [0, 1, 7, 31, 32, 47]
    kb = oracle.KBlockAccumulator(cfg.nao, Cs, rows)
    kb.add_slab(Bp[:70]); kb.add_slab(Bp[70:])
    Bf = unpack_np(Bp, cfg.nao)
    for s, C in enumerate(Cs):
        assert relerr(kb.K[s], K[s][np.ix_(rows, rows)]) < 1e-13
        X = Bf[:, rows, :] @ C
        assert relerr(kb.K[s], np.einsum("pai,pbi->ab", X, X)) < 1e-13


def test_vectorised_and_portable_builds_agree_bitwise(tmp_path, monkeypatch):
    """The oracle is normally built -O3 -march=x86-64-v3 (AVX2) and falls back to plain -O2 on a host
    without AVX2 (oracle.build_command).  Neither build may reassociate a sum or contract an FMA, so
    d, J, K -- and the general-density and whitening routines -- must come out bit for bit the same."""
    import subprocess
    if not oracle.host_has_avx2():
        pytest.skip("this host cannot run the AVX2 build")
    libs = {}
    for name, vector in (("vec", True), ("o2", False)):
        out = str(tmp_path / f"liboracle_{name}.so")
        subprocess.run(oracle.build_command(out, vector=vector), check=True)
        libs[name] = oracle._open(out)
    nao, naux = 37, 11
    Bp, Cs = rand_case(nao, naux, (5, 3), seed=99, orthonormal=False)
    rng = np.random.default_rng(5)
    dm = rng.standard_normal((nao, nao))
    M = rng.standard_normal((naux, naux))
    M = M @ M.T + naux * np.eye(naux)
    res = {}
    for name, lib in libs.items():
        monkeypatch.setattr(oracle, "_lib", lib)
        J, K, d = oracle.get_jk(Bp, nao, Cs, [1.0, 0.5])
        Jd, Kd, _ = oracle.get_jk_dm(Bp, nao, dm)
        L = oracle.cholesky_lower(M)
        res[name] = [J, *K, d, Jd, Kd, oracle.df_diag(Bp, nao), L, oracle.whiten(L, Bp)]
    for a, b in zip(res["vec"], res["o2"]):
        assert np.array_equal(a, b)
