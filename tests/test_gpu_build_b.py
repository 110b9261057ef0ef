"""GPU parity of dfjk_build_b (Eq. 2-3: M = L L^T, B = L^-1 (Q|mu nu)) against
the CPU oracle (textbook Cholesky recurrence + per-column forward substitution), element by element.

Tolerance: relative Frobenius error <= 1e-11 on L and on B.  Both sides are backward stable; they
differ by O(cond(L) eps) and the synthetic metric (dfjk_inputs.metric) has cond(M) < 1e4, so 1e-11
leaves > 2 orders of headroom while any indexing slip or reduced-precision step fails it.
Shapes: one ragged block, exactly one / several 128-row blocks, ragged last block of 1 and of 127
rows, npair odd (rows only 8-byte aligned) and even, npair below / equal to / above the 128-column
tile, so that the bulk-copy path, the alignment shift and the element-wise edge tile all run.
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


@pytest.mark.parametrize("nao,naux", [
    (1, 1), (3, 2), (5, 9), (12, 40),
    (15, 128),          # npair = 120 < one column tile, exactly one row block
    (16, 129),          # npair = 136, ragged last block of one row
    (17, 255),          # npair = 153 (odd), last block of 127 rows
    (22, 256),          # npair = 253 (odd), two full blocks
    (30, 300),          # npair = 465 (odd), three blocks
    (63, 200),          # npair = 2016 (even), 16 column tiles
    (64, 391),          # npair = 2080, four blocks, ragged
])
def test_build_b_parity(dfjk, nao, naux):
    cfg = gi.custom_config(nao, naux, (1,), seed=1000 + naux)
    M, R = gi.metric(cfg), gi.fill_B_host(cfg)
    Lo, Bo = oracle.build_b(M, R)
    Md, Rd = dev(M), dev(R)
    info = dfjk.build_b(Md, Rd, nao)
    torch.cuda.synchronize()
    assert int(info.item()) == 0
    Lg = np.tril(Md.cpu().numpy())
    assert relerr(Lg, Lo) <= TOL
    assert relerr(Rd.cpu().numpy(), Bo) <= TOL
    # the strict upper triangle of M is untouched outside the diagonal blocks
    Mg = Md.cpu().numpy()
    for i in range(0, naux, 128):
        assert np.array_equal(Mg[i:i + 128, i + 128:], M[i:i + 128, i + 128:])


def test_build_b_then_get_jk(dfjk):
    """The whole chain Eq. 2-3 -> get_jk on the device against the oracle's chain."""
    nao, naux, nocc = 40, 150, 6
    cfg = gi.custom_config(nao, naux, (nocc,), seed=77)
    M, R = gi.metric(cfg), gi.fill_B_host(cfg)
    C = gi.random_orbitals(nao, nocc, 5)
    _, Bo = oracle.build_b(M, R)
    Jo, Ko, _ = oracle.get_jk(Bo, nao, [C], [2.0])
    Md, Rd = dev(M), dev(R)
    dfjk.build_b(Md, Rd, nao)
    h = dfjk.DFJK(Rd, nao)
    J, K = h.get_jk(dev(C))
    torch.cuda.synchronize()
    assert relerr(J.cpu().numpy(), Jo) <= TOL and relerr(K.cpu().numpy(), Ko[0]) <= TOL
    h.close()


def test_build_b_flags_indefinite_metric_and_bad_arguments(dfjk):
    nao, naux = 6, 140
    cfg = gi.custom_config(nao, naux, (1,), seed=3)
    M, R = gi.metric(cfg), gi.fill_B_host(cfg)
    M[133, 133] = -1.0                                   # pivot 133 (second block) goes negative
    info = dfjk.build_b(dev(M), dev(R), nao)
    torch.cuda.synchronize()
    assert int(info.item()) == 134
    with pytest.raises(ValueError):
        dfjk.build_b(dev(M[:, :-1]), dev(R), nao)
    L = dfjk.lib()
    assert L.dfjk_build_b(0, nao, 16, 16, None, None) == -1
    host = np.zeros(64)
    assert L.dfjk_build_b(2, 2, host.ctypes.data & ~15, host.ctypes.data & ~15, None, None) == -1
    assert b"device" in L.dfjk_last_error()


def test_build_b_is_deterministic(dfjk):
    cfg = gi.custom_config(30, 260, (1,), seed=8)
    M, R = gi.metric(cfg), gi.fill_B_host(cfg)
    outs = []
    for _ in range(2):
        Md, Rd = dev(M), dev(R)
        dfjk.build_b(Md, Rd, 30)
        torch.cuda.synchronize()
        outs.append((Md.cpu().numpy(), Rd.cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
