"""GPU parity of the general-density entry points (dfjk_get_jk_pair / _dm / _dms) against the
CPU oracle, element by element.

Bar: relative Frobenius error <= 1e-11 for J and K, FP64, full matrices (north_star tolerance).
Shapes span several 128 x 128 K tiles (full, non-symmetric tile grid), ragged tails, odd npair,
ncol = 1 ... nao, several X chunks and k splits.
"""
import numpy as np
import pytest

import dfjk_inputs as gi
import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-11


def relerr(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / (nb if nb > 0 else 1.0)


@pytest.fixture(scope="module")
def dfjk():
    import paper_2506_06661_b200 as pkg
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    pkg.lib()
    return pkg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_B(nao, naux, seed):
    return gi.fill_B_host(gi.custom_config(nao, naux, (1,), seed=seed))


@pytest.mark.parametrize("nao,naux,ncol", [
    (1, 1, 1),
    (2, 3, 2),
    (5, 7, 3),
    (17, 9, 17),         # ncol = nao
    (33, 5, 8),
    (64, 16, 9),
    (129, 12, 31),       # 2 x 2 tiles, ragged
    (200, 40, 13),
    (290, 60, 25),       # 3 x 3 tiles, npair odd
    (300, 7, 130),
])
def test_pair_parity(dfjk, nao, naux, ncol):
    Bp = make_B(nao, naux, 100 + nao)
    rng = np.random.default_rng(nao + ncol)
    C1, C2 = rng.standard_normal((nao, ncol)), rng.standard_normal((nao, ncol))
    h = dfjk.DFJK(dev(Bp), nao)
    Jo, Ko, do = oracle.get_jk_pair(Bp, nao, C1, C2)
    h.set_option("k2_panel_kb", 64)
    for fused, k2_panel in ((1, 0), (0, 0), (1, 1)):   # d_P read off X = B_P C1 (default) or by a pass
        h.set_option("j_fused", fused)                  # over B; both full-product K2 kernels
        h.set_option("k2_panel", k2_panel)
        J, K = h.get_jk_pair(dev(C1), dev(C2))
        d = h.get_d()
        torch.cuda.synchronize()
        assert relerr(d.cpu().numpy(), do) <= TOL
        assert relerr(J.cpu().numpy(), Jo) <= TOL
        assert relerr(K.cpu().numpy(), Ko) <= TOL
    h.close()


def test_pair_parity_widest_column_block(dfjk):
    """ncol = nao = 808: the column block [C1|C2] is 2 nao wide, the widest the handle is sized for.
    J1X then deals two 256-unit tiles to each CTA (its block count is capped so that the d-partial
    workspace stays small), with a ragged last CTA; d, J and K against the oracle."""
    nao, naux, ncol = 808, 5, 808
    Bp = make_B(nao, naux, 4242)
    rng = np.random.default_rng(77)
    C1, C2 = rng.standard_normal((nao, ncol)), rng.standard_normal((nao, ncol))
    h = dfjk.DFJK(dev(Bp), nao)
    assert h.workspace_bytes < 3.2e9
    Jo, Ko, do = oracle.get_jk_pair(Bp, nao, C1, C2)
    J, K = h.get_jk_pair(dev(C1), dev(C2))
    d = h.get_d()
    torch.cuda.synchronize()
    assert relerr(d.cpu().numpy(), do) <= TOL
    assert relerr(J.cpu().numpy(), Jo) <= TOL
    assert relerr(K.cpu().numpy(), Ko) <= TOL
    h.close()


@pytest.mark.parametrize("nao,naux", [(1, 2), (3, 4), (31, 6), (130, 9), (257, 5)])
def test_dm_parity(dfjk, nao, naux):
    Bp = make_B(nao, naux, 300 + nao)
    dm = np.random.default_rng(nao).standard_normal((nao, nao))       # neither symmetric nor PSD
    h = dfjk.DFJK(dev(Bp), nao)
    Jo, Ko, _ = oracle.get_jk_dm(Bp, nao, dm)
    h.set_option("k2_panel_kb", 64)
    for k2_panel in (0, 1):
        h.set_option("k2_panel", k2_panel)
        J, K = h.get_jk_dm(dev(dm))
        torch.cuda.synchronize()
        assert relerr(J.cpu().numpy(), Jo) <= TOL
        assert relerr(K.cpu().numpy(), Ko) <= TOL
    h.close()


def test_dm_batch_and_options(dfjk):
    nao, naux = 150, 11
    Bp = make_B(nao, naux, 7)
    rng = np.random.default_rng(3)
    dms = rng.standard_normal((3, nao, nao))
    dms[1] = dms[1] + dms[1].T                                       # one symmetric member
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("k_chunk", 3)                                       # several X chunks
    h.set_option("k_splits", 2)
    J, K = h.get_jk_dm(dev(dms))
    torch.cuda.synchronize()
    for i in range(3):
        Jo, Ko, _ = oracle.get_jk_dm(Bp, nao, dms[i])
        assert relerr(J[i].cpu().numpy(), Jo) <= TOL
        assert relerr(K[i].cpu().numpy(), Ko) <= TOL
    # J only / K only
    Jonly, none = h.get_jk_dm(dev(dms[0]), with_k=False)
    assert none is None and torch.equal(Jonly, J[0])
    none, Konly = h.get_jk_dm(dev(dms[0]), with_j=False)
    assert none is None and torch.equal(Konly, K[0])                 # deterministic: bitwise repeatable
    h.close()


def test_general_reduces_to_restricted(dfjk):
    """pair(C, C) K == get_jk K; dm = 2 C C^T: same J, K[dm] = 2 K (reading R1)."""
    cfg = gi.CONFIGS[1]
    Bp = gi.fill_B_host(cfg)
    C = gi.orbitals(cfg, 0)[0]
    h = dfjk.DFJK(dev(Bp), cfg.nao)
    J0, K0 = h.get_jk(dev(C))
    Jp, Kp = h.get_jk_pair(dev(C), dev(C))
    Jd, Kd = h.get_jk_dm(dev(2.0 * C @ C.T))
    torch.cuda.synchronize()
    assert relerr(Kp.cpu().numpy(), K0.cpu().numpy()) <= 1e-13
    assert relerr(2.0 * Jp.cpu().numpy(), J0.cpu().numpy()) <= 1e-13
    assert relerr(Jd.cpu().numpy(), J0.cpu().numpy()) <= 1e-13
    assert relerr(Kd.cpu().numpy(), 2.0 * K0.cpu().numpy()) <= 1e-13
    h.close()


def test_general_after_restricted_call_shares_workspace(dfjk):
    """Interleaved calls on one handle (different Ccat widths, split counts) stay correct."""
    nao, naux = 140, 10
    Bp = make_B(nao, naux, 21)
    rng = np.random.default_rng(5)
    C = gi.random_orbitals(nao, 12, 4)
    C1, C2 = rng.standard_normal((nao, 5)), rng.standard_normal((nao, 5))
    h = dfjk.DFJK(dev(Bp), nao)
    for _ in range(2):
        J, K = h.get_jk(dev(C))
        Jp, Kp = h.get_jk_pair(dev(C1), dev(C2))
    torch.cuda.synchronize()
    Jo, Ko, _ = oracle.get_jk(Bp, nao, [C], [2.0])
    Jpo, Kpo, _ = oracle.get_jk_pair(Bp, nao, C1, C2)
    assert relerr(J.cpu().numpy(), Jo) <= TOL and relerr(K.cpu().numpy(), Ko[0]) <= TOL
    assert relerr(Jp.cpu().numpy(), Jpo) <= TOL and relerr(Kp.cpu().numpy(), Kpo) <= TOL
    h.close()


def test_general_error_paths(dfjk):
    nao, naux = 6, 3
    h = dfjk.DFJK(dev(make_B(nao, naux, 1)), nao)
    C = dev(np.ones((nao, 2)))
    with pytest.raises(ValueError):
        h.get_jk_pair(C, dev(np.ones((nao, 3))))
    with pytest.raises(dfjk.DFJKError):
        h.get_jk_pair(C, C, with_j=False, with_k=False)
    with pytest.raises(ValueError):
        h.get_jk_dm(dev(np.ones((nao, nao + 1))))
    L = dfjk.lib()
    assert L.dfjk_get_jk_pair(h._h, C.data_ptr(), None, 2, None, C.data_ptr(), None) == -1
    assert L.dfjk_get_jk_pair(h._h, C.data_ptr(), C.data_ptr(), nao + 1, None, C.data_ptr(), None) == -1
    assert L.dfjk_get_jk_dm(None, None, None, None, None) == -1
    assert L.dfjk_get_jk_dms(h._h, 0, C.data_ptr(), C.data_ptr(), None, None) == -1
    h.close()


@pytest.mark.parametrize("nao,naux", [(1, 1), (5, 7), (64, 16), (129, 12), (290, 60)])
def test_df_diag_parity(dfjk, nao, naux):
    """Eq. 7's DF diagonal sum_P B_Pmn^2 against the oracle."""
    Bp = make_B(nao, naux, 500 + nao)
    h = dfjk.DFJK(dev(Bp), nao)
    diag = h.get_df_diag()
    torch.cuda.synchronize()
    assert relerr(diag.cpu().numpy(), oracle.df_diag(Bp, nao)) <= TOL
    h.close()


def test_pair_is_the_orbital_derivative_of_get_jk_on_the_device(dfjk):
    """SOSCF's use of the pair form: the first-order change of get_jk under
    C -> C + eps V is 4 eps J_pair(C, V) and eps (K_pair + K_pair^T).  J and K are quadratic in C, so
    the central difference of two get_jk calls is exact up to rounding -- a cross-check of the pair
    kernels (full DMMA product, J from X) against the SYRK path that needs no oracle at all."""
    nao, naux, nocc = 200, 30, 17
    Bp = make_B(nao, naux, 9)
    rng = np.random.default_rng(2)
    C = gi.random_orbitals(nao, nocc, 3)
    V = rng.standard_normal((nao, nocc))
    eps = 1e-3
    h = dfjk.DFJK(dev(Bp), nao)
    Jp, Kp = h.get_jk(dev(C + eps * V))
    Jm, Km = h.get_jk(dev(C - eps * V))
    J1, K1 = h.get_jk_pair(dev(C), dev(V))
    torch.cuda.synchronize()
    dJ = ((Jp - Jm) / (2 * eps)).cpu().numpy()
    dK = ((Kp - Km) / (2 * eps)).cpu().numpy()
    K1n = K1.cpu().numpy()
    assert relerr(dJ, 4.0 * J1.cpu().numpy()) <= 1e-9
    assert relerr(dK, K1n + K1n.T) <= 1e-9
    h.close()


@pytest.mark.parametrize("nao,naux,ncols", [
    (64, 16, (5,)),                               # nbatch 1
    (129, 12, (1, 31)),                           # ncol 1 beside a wide one
    (200, 40, (13, 8, 3)),
    (150, 11, (150, 4, 150, 9, 20)),              # ncol = nao twice: the batch overflows ldc_max, three K1 sweeps
    (290, 30, (8, 8, 8, 8, 8, 8, 8, 8)),          # the SOSCF shape: 8 trial vectors of 8 columns, 3 x 3 tiles
    (300, 7, (3, 130, 7, 7, 1, 2, 64, 9, 11, 5)), # more than DFJK_MAX_BATCH = 8: two sub-batches
])
def test_pairs_batch_parity(dfjk, nao, naux, ncols):
    """dfjk_get_jk_pairs: every density of a batch against the oracle's single-pair result, on both K2
    kernels, fused and two-pass d, several X chunks, J-only and K-only batches; with d from the dot
    pass J is bitwise that of the single-pair call (same summation order per density)."""
    Bp = make_B(nao, naux, 900 + nao)
    rng = np.random.default_rng(nao + len(ncols))
    C1s = [rng.standard_normal((nao, c)) for c in ncols]
    C2s = [rng.standard_normal((nao, c)) for c in ncols]
    ref = [oracle.get_jk_pair(Bp, nao, a, b) for a, b in zip(C1s, C2s)]
    d1, d2 = [dev(a) for a in C1s], [dev(b) for b in C2s]
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("k2_panel_kb", 64)
    h.set_option("k_chunk", max(1, naux // 3))
    for fused, k2_panel in ((1, 0), (0, 0), (1, 1)):
        h.set_option("j_fused", fused)
        h.set_option("k2_panel", k2_panel)
        Js, Ks = h.get_jk_pairs(d1, d2)
        torch.cuda.synchronize()
        for i, (Jo, Ko, _) in enumerate(ref):
            assert relerr(Js[i].cpu().numpy(), Jo) <= TOL, (i, fused, k2_panel)
            assert relerr(Ks[i].cpu().numpy(), Ko) <= TOL, (i, fused, k2_panel)
        if fused == 0:                      # d from the dot pass over B: the same sums in the same order
            J1, _ = h.get_jk_pair(d1[-1], d2[-1])
            torch.cuda.synchronize()
            assert torch.equal(J1, Js[-1])
    h.set_option("j_fused", 1)
    Js, none = h.get_jk_pairs(d1, d2, with_k=False)
    none2, Ks = h.get_jk_pairs(d1, d2, with_j=False)
    torch.cuda.synchronize()
    assert none is None and none2 is None
    for i, (Jo, Ko, _) in enumerate(ref):
        assert relerr(Js[i].cpu().numpy(), Jo) <= TOL and relerr(Ks[i].cpu().numpy(), Ko) <= TOL
    h.close()


def test_dms_batch_shares_the_axpy_pass(dfjk):
    """dfjk_get_jk_dms with 10 raw densities (two sub-batches): J and K per density against the oracle;
    the J pass count is ndm + 2 streaming kernels per sub-batch instead of 2 per density."""
    nao, naux, ndm = 130, 9, 10
    Bp = make_B(nao, naux, 55)
    dms = np.random.default_rng(8).standard_normal((ndm, nao, nao))
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("time_kernels", 1)
    J, K = h.get_jk_dm(dev(dms))
    torch.cuda.synchronize()
    assert h.kernel_time("J2")[1] == 2 and h.kernel_time("J1")[1] == ndm
    for i in range(ndm):
        Jo, Ko, _ = oracle.get_jk_dm(Bp, nao, dms[i])
        assert relerr(J[i].cpu().numpy(), Jo) <= TOL and relerr(K[i].cpu().numpy(), Ko) <= TOL
    h.close()


def test_pairs_error_paths(dfjk):
    nao, naux = 6, 3
    h = dfjk.DFJK(dev(make_B(nao, naux, 1)), nao)
    C = dev(np.ones((nao, 2)))
    with pytest.raises(ValueError):
        h.get_jk_pairs([C], [C, C])
    with pytest.raises(ValueError):
        h.get_jk_pairs([C], [dev(np.ones((nao, 3)))])
    with pytest.raises(dfjk.DFJKError):
        h.get_jk_pairs([C], [C], with_j=False, with_k=False)
    h.close()
