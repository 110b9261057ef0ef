"""GPU parity of the DF-RHF SCF driver (dfjk_scf_rhf) against the SCF oracle (oracle/scf.py), both
running Roothaan-Hall + Pulay DIIS in the same order (PAPER.md:154-159,
258-262).

What is compared: the energy of EVERY iteration, the iteration count and convergence flag, and
the converged density and Fock matrices (unique, unlike the orbitals' signs).  Tolerances: the first
energy (core guess, one get_jk) to 1e-11 relative; later iterations to 1e-9, because each
diagonalisation and DIIS solve amplifies the ~1e-15 differences of the two FP64 paths by the
inverse orbital gap and the DIIS condition number; the converged energy to 1e-11 (it is stationary:
second order in the orbital error); D and F to 1e-7 (first order in it, at conv_tol = 1e-10).
"""
import numpy as np
import pytest

import dfjk_inputs as gi
import oracle
from oracle import scf

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


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


@pytest.mark.parametrize("nao,naux,nocc,scale,diis", [
    (14, 30, 3, 0.0, 8),         # no two-electron term: one diagonalisation
    (20, 60, 4, 0.3, 8),
    (48, 160, 5, 0.2, 8),
    (60, 200, 10, 0.3, 3),       # small DIIS space: the ring buffer wraps
    (150, 400, 13, 0.2, 8),      # 2 x 2 K tiles
    (290, 300, 25, 0.1, 6),      # npair odd, 3 x 3 tiles
])
def test_scf_matches_oracle(dfjk, nao, naux, nocc, scale, diis):
    cfg = gi.custom_config(nao, naux, (nocc,), seed=3)
    Bp = gi.fill_B_host(cfg) * scale
    h, S = gi.core_hamiltonian(cfg), gi.overlap(cfg)
    ref = scf.scf_rhf(Bp, nao, h, S, nocc, conv_tol=1e-10, diis_space=diis)
    hd = dfjk.DFJK(dev(Bp), nao)
    out = hd.scf_rhf(dev(h), dev(S), nocc, conv_tol=1e-10, diis_space=diis)
    assert out["converged"] == ref["converged"] == True
    e, eo = np.array(out["e_hist"]), ref["e_hist"]
    assert len(e) == len(eo)
    assert abs(e[0] - eo[0]) <= 1e-11 * abs(eo[0])
    assert np.all(np.abs(e - eo) <= 1e-9 * np.abs(eo))
    assert abs(e[-1] - eo[-1]) <= 1e-11 * abs(eo[-1])
    assert relerr(out["D"].cpu().numpy(), ref["D"]) <= 1e-7
    assert relerr(out["F"].cpu().numpy(), ref["F"]) <= 1e-7
    assert relerr(out["mo_energy"].cpu().numpy(), ref["mo_energy"]) <= 1e-7
    C = out["C"].cpu().numpy()
    assert np.abs(C.T @ S @ C - np.eye(nao)).max() <= 1e-10            # orbitals S-orthonormal
    D = out["D"].cpu().numpy()
    assert abs(np.trace(D @ S) - 2 * nocc) <= 1e-9
    hd.close()


def test_scf_not_converged_and_errors(dfjk):
    cfg = gi.custom_config(20, 60, (4,), seed=3)
    Bp = gi.fill_B_host(cfg) * 0.3
    h, S = gi.core_hamiltonian(cfg), gi.overlap(cfg)
    hd = dfjk.DFJK(dev(Bp), 20)
    out = hd.scf_rhf(dev(h), dev(S), 4, max_iter=2)
    ref = scf.scf_rhf(Bp, 20, h, S, 4, max_iter=2)
    assert not out["converged"] and len(out["e_hist"]) == 2
    assert np.all(np.abs(np.array(out["e_hist"]) - ref["e_hist"]) <= 1e-10 * np.abs(ref["e_hist"]))
    with pytest.raises(dfjk.DFJKError):
        hd.scf_rhf(dev(h), dev(S), 4, diis_space=17)
    with pytest.raises(dfjk.DFJKError):
        hd.scf_rhf(dev(h), dev(S), 21)
    with pytest.raises(dfjk.DFJKError):                                  # S not positive definite
        hd.scf_rhf(dev(h), dev(-S), 4)
    hd.close()


@pytest.mark.parametrize("nao,naux,na,nb,scale,diis", [
    (20, 60, 5, 3, 0.3, 8),
    (48, 160, 6, 5, 0.2, 3),      # small DIIS space: the ring wraps
    (150, 400, 14, 12, 0.2, 8),
    (290, 300, 26, 24, 0.1, 6),
])
def test_uhf_matches_oracle(dfjk, nao, naux, na, nb, scale, diis):
    """dfjk_scf_uhf against oracle.scf.scf_uhf: every iteration's energy, the spin densities and
    orbital energies (same tolerances as the restricted test)."""
    cfg = gi.custom_config(nao, naux, (na,), seed=3)
    Bp = gi.fill_B_host(cfg) * scale
    h, S = gi.core_hamiltonian(cfg), gi.overlap(cfg)
    ref = scf.scf_uhf(Bp, nao, h, S, na, nb, conv_tol=1e-10, diis_space=diis)
    hd = dfjk.DFJK(dev(Bp), nao)
    out = hd.scf_uhf(dev(h), dev(S), na, nb, conv_tol=1e-10, diis_space=diis)
    assert out["converged"] == ref["converged"] == True
    e, eo = np.array(out["e_hist"]), ref["e_hist"]
    assert len(e) == len(eo)
    assert abs(e[0] - eo[0]) <= 1e-11 * abs(eo[0])
    assert np.all(np.abs(e - eo) <= 1e-9 * np.abs(eo))
    assert abs(e[-1] - eo[-1]) <= 1e-11 * abs(eo[-1])
    for s, n in ((0, na), (1, nb)):
        assert relerr(out["D"][s].cpu().numpy(), ref["D"][s]) <= 1e-7
        assert relerr(out["mo_energy"][s].cpu().numpy(), ref["mo_energy"][s]) <= 1e-7
        C = out["C"][s].cpu().numpy()
        assert np.abs(C.T @ S @ C - np.eye(nao)).max() <= 1e-10
        assert abs(np.trace(out["D"][s].cpu().numpy() @ S) - n) <= 1e-9
    hd.close()


def test_uhf_closed_shell_equals_rhf_on_the_device(dfjk):
    cfg = gi.custom_config(48, 160, (5,), seed=3)
    Bp = gi.fill_B_host(cfg) * 0.2
    h, S = gi.core_hamiltonian(cfg), gi.overlap(cfg)
    hd = dfjk.DFJK(dev(Bp), 48)
    r = hd.scf_rhf(dev(h), dev(S), 5)
    u = hd.scf_uhf(dev(h), dev(S), 5, 5)
    assert r["converged"] and u["converged"] and len(r["e_hist"]) == len(u["e_hist"])
    assert np.allclose(u["e_hist"], r["e_hist"], rtol=1e-11, atol=0)
    assert relerr((u["D"][0] + u["D"][1]).cpu().numpy(), r["D"].cpu().numpy()) <= 1e-8
    hd.close()
