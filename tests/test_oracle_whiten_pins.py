"""Pins for the oracle of Eq. 2-3: M = L L^T, B = L^-1 (Q|mu nu).

  * hand-worked 2x2 fixture (tests/golden/hand_whiten_2x2.txt), exact
  * library routines: numpy.linalg.cholesky, scipy.linalg.solve_triangular
  * reconstruction L L^T = M and L B = R; L lower triangular with positive diagonal
  * the resolution-of-identity form the whitening exists for (Eq. 1 with Eq. 2-3 inserted):
        sum_P B_P,mn B_P,ls = sum_QQ' (mn|Q) (M^-1)_QQ' (Q'|ls)
  * special cases: M = I (B = R), diagonal M (B = R / sqrt(diag)), non-SPD M is refused
"""
import os

import numpy as np
import pytest
import scipy.linalg

import dfjk_inputs as gi
import oracle


def relerr(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / (nb if nb > 0 else 1.0)


def test_hand_worked_fixture(repo_root):
    vals = {}
    with open(os.path.join(repo_root, "tests", "golden", "hand_whiten_2x2.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            vals[k] = np.array([float(x) for x in v])
    n, nc = int(vals["n"][0]), int(vals["ncols"][0])
    L, B = oracle.build_b(vals["M"].reshape(n, n), vals["R"].reshape(n, nc))
    assert np.array_equal(L.ravel(), vals["L"])
    assert np.array_equal(B.ravel(), vals["B"])


@pytest.mark.parametrize("nao,naux", [(3, 1), (5, 9), (12, 40), (20, 131), (30, 300)])
def test_against_library_routines(nao, naux):
    cfg = gi.custom_config(nao, naux, (1,), seed=naux)
    M, R = gi.metric(cfg), gi.fill_B_host(cfg)
    L, B = oracle.build_b(M, R)
    Lref = np.linalg.cholesky(M)
    assert relerr(L, Lref) < 1e-13
    assert np.array_equal(L, np.tril(L)) and (np.diag(L) > 0).all()
    assert relerr(B, scipy.linalg.solve_triangular(Lref, R, lower=True)) < 1e-12
    assert relerr(L @ L.T, M) < 1e-14
    assert relerr(L @ B, R) < 1e-13


def test_resolution_of_identity_form():
    """Eq. 1 with Eq. 2-3: B^T B = R^T M^-1 R, and J/K from B equal J/K from the RI integrals."""
    cfg = gi.custom_config(6, 25, (2,), seed=4)
    M, R = gi.metric(cfg), gi.fill_B_host(cfg)
    _, B = oracle.build_b(M, R)
    assert relerr(B.T @ B, R.T @ np.linalg.solve(M, R)) < 1e-11
    # the brute-force 4-index tensor built from B equals the one built from R M^-1 R
    nao = cfg.nao
    il = np.tril_indices(nao)
    Rf = np.zeros((cfg.naux, nao, nao)); Rf[:, il[0], il[1]] = R; Rf[:, il[1], il[0]] = R
    eri = np.einsum("qmn,qp,pls->mnls", Rf, np.linalg.inv(M), Rf)
    C = gi.random_orbitals(nao, 2, 1)
    D = 2.0 * C @ C.T
    J, K, _ = oracle.get_jk(B, nao, [C], [2.0])
    assert relerr(J, np.einsum("mnls,ls->mn", eri, D)) < 1e-11
    assert relerr(K[0], np.einsum("mlns,ls->mn", eri, C @ C.T)) < 1e-11


def test_special_cases():
    rng = np.random.default_rng(0)
    R = rng.standard_normal((7, 10))
    L, B = oracle.build_b(np.eye(7), R)
    assert np.array_equal(L, np.eye(7)) and np.array_equal(B, R)
    dg = rng.uniform(0.5, 2.0, 7)
    L, B = oracle.build_b(np.diag(dg), R)
    assert relerr(np.diag(L), np.sqrt(dg)) < 1e-15
    assert relerr(B, R / np.sqrt(dg)[:, None]) < 1e-15
    # only the lower triangle of M is read
    M = gi.metric(gi.custom_config(4, 7, (1,), seed=2))
    Mu = M.copy(); Mu[np.triu_indices(7, 1)] = 123.0
    assert np.array_equal(oracle.cholesky_lower(Mu), oracle.cholesky_lower(M))
    with pytest.raises(RuntimeError):
        oracle.cholesky_lower(np.array([[1.0, 2.0], [2.0, 1.0]]))        # indefinite


def test_metric_generator_is_spd_and_well_conditioned():
    cfg = gi.custom_config(4, 400, (1,), seed=9)
    M = gi.metric(cfg)
    assert np.array_equal(M, M.T)
    ev = np.linalg.eigvalsh(M)
    assert ev.min() > 0.09 and ev.max() / ev.min() < 1e4
