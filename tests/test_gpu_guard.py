"""Bounds checks of our own (compute-sanitizer is closed on this GPU pool; profiles/r03_sanitizer.md).

Parity says the values are right; it does not say that no kernel looked outside its arrays.  K1 stages
the packed triangle with bulk copies that start one element before a packed row and run past its
end when the row is misaligned (k1_half_transform.cu), special-cases the last row of the last P so as
not to read past the end of B, and J1 / J2 issue 128-bit loads on the 16-byte grid of the flat array.
Two kinds of guard catch a wrong access there without a tool:

  * poison: B, the orbitals and the outputs sit inside larger buffers whose surroundings hold NaN (a
    sentinel for the outputs).  An out-of-bounds READ that reaches the arithmetic -- even multiplied
    by a zero of the padding -- turns the result into NaN; an out-of-bounds WRITE changes a sentinel.
  * unmapped pages: B is placed flush against the END (and, in a second run, the START) of a range
    mapped with the CUDA virtual-memory API, with reserved but unmapped address space on both sides.
    Any access outside B -- used or not -- is then an illegal-address fault.  That run happens in a
    child process, so a fault fails this test without taking the pytest process's context with it.

Shapes are ragged (nao not a multiple of 128 or 32, odd npair and odd naux so that rows alternate
between the two 16-byte alignment classes and the tensor ends on an odd element), on both K2 kernels.
"""
import os
import subprocess
import sys

import numpy as np
import pytest

import dfjk_inputs as gi
import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-11
GUARD = 4096            # doubles on each side (even: B keeps its 16-byte alignment)
SENTINEL = -777.25


def relerr(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / (nb if nb > 0 else 1.0)


@pytest.fixture(scope="module")
def dfjk():
    import paper_2506_06661_b200 as pkg
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    pkg.lib()
    return pkg


def embed(a, fill):
    """a copy of `a` in the middle of a buffer filled with `fill`; returns (view, whole buffer)"""
    a = np.ascontiguousarray(a, dtype=np.float64)
    buf = torch.full((a.size + 2 * GUARD,), fill, dtype=torch.float64, device="cuda")
    view = buf[GUARD:GUARD + a.size].view(*a.shape)
    view.copy_(torch.from_numpy(a))
    return view, buf


def out_buffer(nao):
    buf = torch.full((nao * nao + 2 * GUARD,), SENTINEL, dtype=torch.float64, device="cuda")
    return buf[GUARD:GUARD + nao * nao].view(nao, nao), buf


def guards_intact(buf, n):
    return bool((buf[:GUARD] == SENTINEL).all()) and bool((buf[GUARD + n:] == SENTINEL).all())


@pytest.mark.parametrize("nao,naux,nocc", [
    (129, 11, 3),        # npair odd (8385), naux odd: B ends on an odd element; 2 x 2 tiles
    (190, 7, 12),
    (290, 9, 25),        # npair odd, 3 x 3 tiles
    (417, 5, 40),        # 4 x 4 tiles, 33-row last block
    (700, 3, 20),        # automatic K2P size class
])
def test_poisoned_surroundings(dfjk, nao, naux, nocc):
    Bp = gi.fill_B_host(gi.custom_config(nao, naux, (nocc,), seed=nao))
    C = gi.random_orbitals(nao, nocc, nao + 1)
    rng = np.random.default_rng(nao)
    C2 = rng.standard_normal((nao, nocc))
    dm = rng.standard_normal((nao, nao))
    nan = float("nan")
    Bd, _ = embed(Bp, nan)
    Cd, _ = embed(C, nan)
    C2d, _ = embed(C2, nan)
    dmd, _ = embed(dm, nan)
    Jo, Ko = oracle.get_jk_restricted(Bp, nao, C)
    Jpo, Kpo, _ = oracle.get_jk_pair(Bp, nao, C, C2)
    Jdo, Kdo, _ = oracle.get_jk_dm(Bp, nao, dm)
    h = dfjk.DFJK(Bd, nao)
    h.set_option("k2_panel_kb", 64)
    h.set_option("k_chunk", max(1, naux // 2))            # several X chunks, a short last one
    for k2_panel in (0, 1):
        h.set_option("k2_panel", k2_panel)
        for fused in (1, 0):
            h.set_option("j_fused", fused)
            J, jbuf = out_buffer(nao)
            K, kbuf = out_buffer(nao)
            for _ in range(3):                            # plain launch, graph capture, graph replay
                h.get_jk(Cd, out_j=J, out_k=K)
            torch.cuda.synchronize()
            assert relerr(J.cpu().numpy(), Jo) <= TOL and relerr(K.cpu().numpy(), Ko) <= TOL
            assert guards_intact(jbuf, nao * nao) and guards_intact(kbuf, nao * nao)
        Jp, Kp = h.get_jk_pair(Cd, C2d)
        Jd, Kd = h.get_jk_dm(dmd)
        torch.cuda.synchronize()
        assert relerr(Jp.cpu().numpy(), Jpo) <= TOL and relerr(Kp.cpu().numpy(), Kpo) <= TOL
        assert relerr(Jd.cpu().numpy(), Jdo) <= TOL and relerr(Kd.cpu().numpy(), Kdo) <= TOL
    want = oracle.df_diag(Bp, nao)
    diag, dbuf = out_buffer(nao)
    dfjk.df_diag_noalloc(Bd, nao, diag)
    torch.cuda.synchronize()
    assert relerr(diag.cpu().numpy(), want) <= TOL and guards_intact(dbuf, nao * nao)
    assert relerr(h.get_df_diag().cpu().numpy(), want) <= TOL
    h.close()


@pytest.mark.parametrize("nao,naux,na,nb", [(129, 11, 3, 2), (290, 9, 25, 24), (417, 5, 40, 33), (700, 3, 20, 20)])
def test_poisoned_workspace(dfjk, nao, naux, na, nb):
    """initcheck of our own: the handle's whole workspace (X and its padding, Kpart slabs, d partials,
    Jp partials, packed orbitals, K2P counters) is filled with NaN bytes before EVERY call, so a
    kernel that reads workspace which no earlier kernel of the same call has written cannot pass."""
    Bp = gi.fill_B_host(gi.custom_config(nao, naux, (na, nb), seed=nao + 7))
    Ca, Cb = gi.random_orbitals(nao, na, 1), gi.random_orbitals(nao, nb, 2)
    rng = np.random.default_rng(nao)
    V = rng.standard_normal((nao, na))
    dm = rng.standard_normal((nao, nao))
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Jo, Ko = oracle.get_jk_restricted(Bp, nao, Ca)
    Ju, Kao, Kbo = oracle.get_jk_unrestricted(Bp, nao, Ca, Cb)
    Jpo, Kpo, _ = oracle.get_jk_pair(Bp, nao, Ca, V)
    Jdo, Kdo, _ = oracle.get_jk_dm(Bp, nao, dm)
    want_diag = oracle.df_diag(Bp, nao)
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("graph", 0)                  # a replayed graph is the same launch sequence; keep every call plain
    h.set_option("k2_panel_kb", 64)
    h.set_option("k_chunk", max(1, naux // 2))
    ok = lambda got, want: relerr(got.cpu().numpy(), want) <= TOL

    def fresh(call):
        h.set_option("poison_workspace", 1)
        out = call()
        torch.cuda.synchronize()
        return out

    for k2_panel in (0, 1):
        h.set_option("k2_panel", k2_panel)
        for fused in (1, 0):
            h.set_option("j_fused", fused)
            J, K = fresh(lambda: h.get_jk(dev(Ca)))
            assert ok(J, Jo) and ok(K, Ko), (k2_panel, fused)
            J, Ka, Kb = fresh(lambda: h.get_jk_u(dev(Ca), dev(Cb)))
            assert ok(J, Ju) and ok(Ka, Kao) and ok(Kb, Kbo), (k2_panel, fused)
            J, K = fresh(lambda: h.get_jk_pair(dev(Ca), dev(V)))
            assert ok(J, Jpo) and ok(K, Kpo), (k2_panel, fused)
        J, K = fresh(lambda: h.get_jk_dm(dev(dm)))
        assert ok(J, Jdo) and ok(K, Kdo), k2_panel
        J, _ = fresh(lambda: h.get_jk(dev(Ca), with_k=False))
        _, K = fresh(lambda: h.get_jk(dev(Ca), with_j=False))
        assert ok(J, Jo) and ok(K, Ko), k2_panel
    assert ok(fresh(lambda: h.get_df_diag()), want_diag)
    h.close()


def test_build_b_poisoned_surroundings(dfjk):
    nao, naux = 33, 261                                   # 3 block rows of the blocked Cholesky, ragged
    cfg = gi.custom_config(nao, naux, (1,), seed=5)
    M, R = gi.metric(cfg), gi.fill_B_host(cfg)
    Lo, Bo = oracle.build_b(M, R)
    nan = float("nan")
    Md, mbuf = embed(M, nan)
    Rd, rbuf = embed(R, nan)
    info = dfjk.build_b(Md, Rd, nao)
    torch.cuda.synchronize()
    assert int(info.item()) == 0
    assert relerr(torch.tril(Md).cpu().numpy(), np.tril(Lo)) <= TOL
    assert relerr(Rd.cpu().numpy(), Bo) <= TOL
    for buf, n in ((mbuf, M.size), (rbuf, R.size)):       # nothing written outside M and R
        assert bool(torch.isnan(buf[:GUARD]).all()) and bool(torch.isnan(buf[GUARD + n:]).all())


_CHILD = r"""
import sys
import numpy as np
import torch
from cuda.bindings import driver as drv
import dfjk_inputs as gi
import oracle
import paper_2506_06661_b200 as dfjk

def ck(r):
    if r[0] != drv.CUresult.CUDA_SUCCESS:
        print("VMM-UNAVAILABLE", r[0]); sys.exit(77)
    return r[1] if len(r) == 2 else r[1:]

def relerr(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)

torch.zeros(1, device="cuda"); torch.cuda.synchronize()
L = dfjk.lib()
prop = drv.CUmemAllocationProp()
prop.type = drv.CUmemAllocationType.CU_MEM_ALLOCATION_TYPE_PINNED
prop.location.type = drv.CUmemLocationType.CU_MEM_LOCATION_TYPE_DEVICE
prop.location.id = 0
gran = int(ck(drv.cuMemGetAllocationGranularity(prop, drv.CUmemAllocationGranularity_flags.CU_MEM_ALLOC_GRANULARITY_MINIMUM)))
acc = drv.CUmemAccessDesc()
acc.location.type = drv.CUmemLocationType.CU_MEM_LOCATION_TYPE_DEVICE
acc.location.id = 0
acc.flags = drv.CUmemAccess_flags.CU_MEM_ACCESS_FLAGS_PROT_READWRITE

def mapped_range(nbytes):
    size = (nbytes + gran - 1) // gran * gran
    va = int(ck(drv.cuMemAddressReserve(size + 2 * gran, gran, 0, 0)))     # unmapped page before and after
    hnd = ck(drv.cuMemCreate(size, prop, 0))
    ck(drv.cuMemMap(va + gran, size, 0, hnd, 0))
    ck(drv.cuMemSetAccess(va + gran, size, [acc], 1))
    return va + gran, size

for nao, naux, nocc in ((129, 12, 3), (290, 10, 25), (417, 6, 40), (700, 4, 20)):
    Bp = gi.fill_B_host(gi.custom_config(nao, naux, (nocc,), seed=nao))
    assert Bp.size % 2 == 0                                # the end-flush pointer must stay 16-byte aligned
    C = gi.random_orbitals(nao, nocc, nao + 1)
    C2 = np.random.default_rng(nao).standard_normal((nao, nocc))
    Jo, Ko = oracle.get_jk_restricted(Bp, nao, C)
    Jpo, Kpo, _ = oracle.get_jk_pair(Bp, nao, C, C2)
    want = oracle.df_diag(Bp, nao)
    src = torch.from_numpy(Bp).cuda()
    Cd, C2d = torch.from_numpy(C).cuda(), torch.from_numpy(C2).cuda()
    base, size = mapped_range(Bp.nbytes)
    for where, ptr in (("end", base + size - Bp.nbytes), ("start", base)):
        if where == "start" and size == Bp.nbytes:
            continue
        ck(drv.cuMemcpyDtoD(ptr, src.data_ptr(), Bp.nbytes))
        torch.cuda.synchronize()
        h = L.dfjk_create(naux, nao, ptr)
        assert h, L.dfjk_last_error()
        assert L.dfjk_set_option(h, b"k2_panel_kb", 64) == 0
        assert L.dfjk_set_option(h, b"k_chunk", max(1, naux // 2)) == 0
        st = torch.cuda.current_stream().cuda_stream
        for k2_panel in (0, 1):
            assert L.dfjk_set_option(h, b"k2_panel", k2_panel) == 0
            for fused in (1, 0):
                assert L.dfjk_set_option(h, b"j_fused", fused) == 0
                J = torch.empty(nao, nao, dtype=torch.float64, device="cuda"); K = torch.empty_like(J)
                for _ in range(2):
                    assert L.dfjk_get_jk(h, Cd.data_ptr(), nocc, J.data_ptr(), K.data_ptr(), st) == 0, L.dfjk_last_error()
                torch.cuda.synchronize()
                assert relerr(J.cpu().numpy(), Jo) <= 1e-11 and relerr(K.cpu().numpy(), Ko) <= 1e-11
            Jp = torch.empty(nao, nao, dtype=torch.float64, device="cuda"); Kp = torch.empty_like(Jp)
            assert L.dfjk_get_jk_pair(h, Cd.data_ptr(), C2d.data_ptr(), nocc, Jp.data_ptr(), Kp.data_ptr(), st) == 0
            torch.cuda.synchronize()
            assert relerr(Jp.cpu().numpy(), Jpo) <= 1e-11 and relerr(Kp.cpu().numpy(), Kpo) <= 1e-11
        d1 = torch.empty(nao, nao, dtype=torch.float64, device="cuda"); d2 = torch.empty_like(d1)
        assert L.dfjk_get_df_diag(h, d1.data_ptr(), st) == 0
        assert L.dfjk_df_diag_noalloc(naux, nao, ptr, d2.data_ptr(), st) == 0, L.dfjk_last_error()
        torch.cuda.synchronize()
        assert relerr(d1.cpu().numpy(), want) <= 1e-11 and relerr(d2.cpu().numpy(), want) <= 1e-11
        L.dfjk_destroy(h)
        print("ok", nao, naux, nocc, where, flush=True)
print("GUARD-PAGES-OK")
"""


def test_b_flush_against_unmapped_pages(dfjk, repo_root):
    """B at the very end / very start of a mapped range, unmapped address space beyond: any access
    outside B faults.  Child process (a fault would poison this process's CUDA context)."""
    env = dict(os.environ, PYTHONPATH=repo_root + os.pathsep + os.environ.get("PYTHONPATH", ""))
    r = subprocess.run([sys.executable, "-c", _CHILD], cwd=repo_root, env=env, capture_output=True,
                       text=True, timeout=600)
    if r.returncode == 77 and "VMM-UNAVAILABLE" in r.stdout:
        pytest.skip("CUDA virtual-memory API not usable here: " + r.stdout.strip().splitlines()[-1])
    assert r.returncode == 0 and "GUARD-PAGES-OK" in r.stdout, (r.stdout[-2000:], r.stderr[-3000:])
