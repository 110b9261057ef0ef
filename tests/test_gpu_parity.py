"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): relative Frobenius error <= 1e-11 for J and every K, FP64,
on the full matrices.  Sizes here are ones the oracle finishes in seconds but that span
several 128-row tiles, several 16-column k-chunks, several 4096-pair J chunks and ragged tails.
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
    pkg.lib()                      # fails loudly if libdfjk.so is missing
    return pkg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_restricted(pkg, Bp, nao, C, **opts):
    Bd = dev(Bp)
    h = pkg.DFJK(Bd, nao)
    for k, v in opts.items():
        h.set_option(k, v)
    J, K = h.get_jk(dev(C))
    d = h.get_d()
    torch.cuda.synchronize()
    out = J.cpu().numpy(), K.cpu().numpy(), d.cpu().numpy()
    h.close()
    return out


def rand_case(nao, naux, noccs, seed, orthonormal=True):
    cfg = gi.custom_config(nao, naux, noccs, seed=seed)
    Bp = gi.fill_B_host(cfg)
    Cs = [gi.random_orbitals(nao, n, seed + 11 * i, orthonormal) for i, n in enumerate(noccs)]
    return Bp, Cs


@pytest.mark.parametrize("cfg_id", [1, 2])
def test_baseline_configs_all_calls(dfjk, cfg_id):
    cfg = gi.CONFIGS[cfg_id]
    Bp = gi.fill_B_host(cfg)
    Bd = dev(Bp)
    h = dfjk.DFJK(Bd, cfg.nao)
    for call in range(cfg.calls):                 # every call of the schedule (cfg 2: 10 fresh C_occ)
        C = gi.orbitals(cfg, call)[0]
        J, K = h.get_jk(dev(C))
        d = h.get_d()
        torch.cuda.synchronize()
        Jo, Ko, do = oracle.get_jk(Bp, cfg.nao, [C], [2.0])
        assert relerr(d.cpu().numpy(), do) <= TOL
        assert relerr(J.cpu().numpy(), Jo) <= TOL
        assert relerr(K.cpu().numpy(), Ko[0]) <= TOL
    h.close()


@pytest.mark.parametrize("nao,naux,nocc", [
    (1, 1, 1),          # npair = 1
    (2, 3, 1),
    (5, 7, 5),          # nocc = nao
    (17, 9, 7),
    (33, 5, 8),
    (64, 16, 9),
    (129, 10, 3),       # one row past a 128 tile; odd npair
    (130, 12, 17),      # npair odd (nao mod 4 == 2)
    (200, 21, 140),     # nocc > 136: two N tiles in K1
    (257, 6, 31),
    (300, 40, 300),     # nocc = nao, three N tiles
    (150, 11, 10),      # ragged last block of 22 rows: K1 batches it over 4 P, naux not a multiple of 4
    (190, 7, 12),       # 62 rows: batched over 2 P, odd naux (the last ragged item holds one P)
    (280, 9, 20),       # 24 rows after two full blocks
    (400, 13, 30),      # 16 rows after three full blocks: batched over 8 P
    (96, 5, 40),        # a single row block of 96 rows: not batched
])
@pytest.mark.parametrize("k2_panel", [0, 1])       # both K2 kernels (the default picks by size)
def test_ragged_shapes(dfjk, nao, naux, nocc, k2_panel):
    Bp, (C,) = rand_case(nao, naux, (nocc,), seed=nao + naux)
    J, K, d = run_restricted(dfjk, Bp, nao, C, k2_panel=k2_panel, k2_panel_kb=64)
    Jo, Ko, do = oracle.get_jk(Bp, nao, [C], [2.0])
    assert relerr(d, do) <= TOL
    assert relerr(J, Jo) <= TOL
    assert relerr(K, Ko[0]) <= TOL
    assert np.array_equal(J, J.T) and np.array_equal(K, K.T)   # mirrored, bit for bit


def test_non_orthonormal_orbitals(dfjk):
    Bp, (C,) = rand_case(150, 30, (20,), seed=5, orthonormal=False)
    J, K, _ = run_restricted(dfjk, Bp, 150, C)
    Jo, Ko, _ = oracle.get_jk(Bp, 150, [C], [2.0])
    assert relerr(J, Jo) <= TOL and relerr(K, Ko[0]) <= TOL


@pytest.mark.parametrize("opts", [dict(k_chunk=1), dict(k_chunk=3), dict(k_chunk=4, k_splits=1),
                                  dict(k_chunk=7, k_splits=2), dict(j_fused=0), dict(j_fused=0, k_chunk=5),
                                  dict(k2_panel=1), dict(k2_panel=1, k_chunk=3, k_splits=1),
                                  dict(k2_panel=1, k_chunk=7, k_splits=2, k2_panel_kb=64),
                                  dict(k2_panel=1, k2_panel_kb=64, graph=0)])
def test_chunk_and_split_options(dfjk, opts):
    Bp, (C,) = rand_case(260, 23, (13,), seed=3)
    J, K, _ = run_restricted(dfjk, Bp, 260, C, **opts)
    Jo, Ko, _ = oracle.get_jk(Bp, 260, [C], [2.0])
    assert relerr(J, Jo) <= TOL and relerr(K, Ko[0]) <= TOL


@pytest.mark.parametrize("nao,naux,nocc", [(290, 60, 25), (48, 40, 5), (400, 30, 33)])
def test_weighted_splits(dfjk, nao, naux, nocc):
    """The split kernel with per-tile split counts (k2_weighted = 1) and with one count for all tiles
    (0) against the oracle; the automatic choice must be one of the two, bit for bit."""
    Bp, (C,) = rand_case(nao, naux, (nocc,), seed=7 * nao + nocc)
    Jo, Ko, _ = oracle.get_jk(Bp, nao, [C], [2.0])
    res = {}
    for w in (0, 1, 2):
        J, K, _ = run_restricted(dfjk, Bp, nao, C, k2_panel=0, k2_weighted=w)
        assert relerr(J, Jo) <= TOL and relerr(K, Ko[0]) <= TOL, w
        assert np.array_equal(K, K.T)
        res[w] = K
    assert np.array_equal(res[2], res[0]) or np.array_equal(res[2], res[1])


def test_panel_kernel_repeatable(dfjk):
    """K2P with many short panels and few slabs: the slab adds of one (slab, tile) are chained across
    CTAs by a release/acquire counter, so repeat calls must agree bit for bit."""
    nao, naux, nocc = 260, 300, 20
    Bp, (C,) = rand_case(nao, naux, (nocc,), seed=99)
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("k2_panel", 1)
    h.set_option("k2_panel_kb", 64)
    Cd = dev(C)
    ref = h.get_jk(Cd)
    torch.cuda.synchronize()
    Jo, Ko, _ = oracle.get_jk(Bp, nao, [C], [2.0])
    assert relerr(ref[1].cpu().numpy(), Ko[0]) <= TOL
    for _ in range(5):
        again = h.get_jk(Cd)
        torch.cuda.synchronize()
        assert torch.equal(again[0], ref[0]) and torch.equal(again[1], ref[1])
    h.close()


@pytest.mark.parametrize("nao,naux,nocc,chunk", [(656, 301, 57, 77), (736, 203, 140, 50), (1000, 150, 90, 0)])
def test_midsize_ragged_multichunk(dfjk, nao, naux, nocc, chunk):
    """Mid-size shapes against the full oracle: a 16-row (656), 96-row (736) and 104-row (1000) last
    block, chunks whose length is not a multiple of K1's batching group (partial last groups in every
    chunk), two N tiles (nocc 140), both K2 kernels, unrestricted on top of the restricted call."""
    Bp, (C,) = rand_case(nao, naux, (nocc,), seed=nao + 3)
    Jo, Ko, _ = oracle.get_jk(Bp, nao, [C], [2.0])
    for k2_panel in (0, 1):
        J, K, _ = run_restricted(dfjk, Bp, nao, C, k_chunk=chunk, k2_panel=k2_panel, k2_panel_kb=512)
        assert relerr(J, Jo) <= TOL and relerr(K, Ko[0]) <= TOL, k2_panel
        assert np.array_equal(K, K.T)
    Cb = gi.random_orbitals(nao, nocc - 7, 4242)
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("k_chunk", chunk)
    Ju, Ka, Kb = h.get_jk_u(dev(C), dev(Cb))
    torch.cuda.synchronize()
    Juo, Kao, Kbo = oracle.get_jk_unrestricted(Bp, nao, C, Cb)
    assert relerr(Ju.cpu().numpy(), Juo) <= TOL
    assert relerr(Ka.cpu().numpy(), Kao) <= TOL and relerr(Kb.cpu().numpy(), Kbo) <= TOL
    h.close()


def test_panel_kernel_stress_all_sms(dfjk):
    """K2P with every SM busy (nao = 900: 36 tiles, hundreds of short panels, one or two slabs): ten
    calls must agree bit for bit with each other (the cross-CTA chains of `red` adds are ordered by
    release/acquire counters) and, up to summation order, with the split kernel."""
    cfg = gi.custom_config(900, 700, (70,), seed=123)
    B = torch.empty(cfg.naux, cfg.npair, dtype=torch.float64, device="cuda")
    gi.fill_B_device(cfg, B)
    C = dev(gi.random_orbitals(cfg.nao, 70, 5))
    h = dfjk.DFJK(B, cfg.nao)
    h.set_option("k2_panel", 0)
    _, Ksplit = h.get_jk(C, with_j=False)
    h.set_option("k2_panel", 1)
    h.set_option("k2_panel_kb", 1024)
    _, Kref = h.get_jk(C, with_j=False)
    torch.cuda.synchronize()
    assert relerr(Kref.cpu().numpy(), Ksplit.cpu().numpy()) <= 1e-13
    assert torch.equal(Kref, Kref.T)
    for _ in range(10):
        _, K = h.get_jk(C, with_j=False)
        torch.cuda.synchronize()
        assert torch.equal(K, Kref)
    h.close()


@pytest.mark.parametrize("fused,k2_panel", [(1, 0), (0, 0), (1, 1)])
def test_unrestricted(dfjk, fused, k2_panel):
    nao, naux = 210, 33
    Bp, (Ca, Cb) = rand_case(nao, naux, (19, 14), seed=8)
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("j_fused", fused)      # d_P from the half-transformed X (default) or by a pass over B
    h.set_option("k2_panel", k2_panel)
    h.set_option("k2_panel_kb", 64)
    J, Ka, Kb = h.get_jk_u(dev(Ca), dev(Cb))
    d = h.get_d()
    torch.cuda.synchronize()
    Jo, Kao, Kbo = oracle.get_jk_unrestricted(Bp, nao, Ca, Cb)
    _, _, do = oracle.get_jk(Bp, nao, [Ca, Cb], [1.0, 1.0], with_k=False)
    assert relerr(d.cpu().numpy(), do) <= TOL
    assert relerr(J.cpu().numpy(), Jo) <= TOL
    assert relerr(Ka.cpu().numpy(), Kao) <= TOL
    assert relerr(Kb.cpu().numpy(), Kbo) <= TOL
    h.close()


def test_j_only_k_only_and_repeatability(dfjk):
    nao = 190
    Bp, (C,) = rand_case(nao, 25, (11,), seed=2)
    h = dfjk.DFJK(dev(Bp), nao)
    Cd = dev(C)
    J1, K1 = h.get_jk(Cd)
    J2, none_k = h.get_jk(Cd, with_k=False)
    none_j, K2 = h.get_jk(Cd, with_j=False)
    torch.cuda.synchronize()
    assert none_k is None and none_j is None
    # K is the same kernel sequence either way; J of a J-only call comes from two passes over B, J of a
    # J+K call from the fused route (d_P read off X): same numbers up to summation order
    assert torch.equal(K1, K2)
    assert relerr(J2.cpu().numpy(), J1.cpu().numpy()) <= 1e-13
    # deterministic reductions: repeat calls are bitwise identical
    J3, K3 = h.get_jk(Cd)
    J4, _ = h.get_jk(Cd, with_k=False)
    torch.cuda.synchronize()
    assert torch.equal(J1, J3) and torch.equal(K1, K3) and torch.equal(J2, J4)
    # outputs are overwritten, not accumulated
    Jpre = torch.full((nao, nao), 7.0, dtype=torch.float64, device="cuda")
    Kpre = torch.full((nao, nao), -3.0, dtype=torch.float64, device="cuda")
    h.get_jk(Cd, out_j=Jpre, out_k=Kpre)
    torch.cuda.synchronize()
    assert torch.equal(Jpre, J1) and torch.equal(Kpre, K1)
    h.close()


def test_side_stream(dfjk):
    nao = 100
    Bp, (C,) = rand_case(nao, 12, (6,), seed=4)
    h = dfjk.DFJK(dev(Bp), nao)
    Cd = dev(C)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        J, K = h.get_jk(Cd)
    s.synchronize()
    Jo, Ko, _ = oracle.get_jk(Bp, nao, [C], [2.0])
    assert relerr(J.cpu().numpy(), Jo) <= TOL and relerr(K.cpu().numpy(), Ko[0]) <= TOL
    h.close()


def test_host_entry_point(dfjk):
    nao = 140
    Bp, (C,) = rand_case(nao, 18, (9,), seed=6)
    h = dfjk.DFJK(dev(Bp), nao)
    Ch = torch.from_numpy(C).pin_memory()
    Jh = torch.empty(nao, nao, dtype=torch.float64).pin_memory()
    Kh = torch.empty(nao, nao, dtype=torch.float64).pin_memory()
    h.get_jk_host(Ch, Jh, Kh)
    Jo, Ko, _ = oracle.get_jk(Bp, nao, [C], [2.0])
    assert relerr(Jh.numpy(), Jo) <= TOL and relerr(Kh.numpy(), Ko[0]) <= TOL
    # unrestricted host entry
    Ca, Cb = gi.random_orbitals(nao, 7, 21), gi.random_orbitals(nao, 5, 22)
    Kah = torch.empty(nao, nao, dtype=torch.float64).pin_memory()
    Kbh = torch.empty(nao, nao, dtype=torch.float64).pin_memory()
    h.get_jk_u_host(torch.from_numpy(Ca).pin_memory(), torch.from_numpy(Cb).pin_memory(), Jh, Kah, Kbh)
    Juo, Kao, Kbo = oracle.get_jk_unrestricted(Bp, nao, Ca, Cb)
    assert relerr(Jh.numpy(), Juo) <= TOL and relerr(Kah.numpy(), Kao) <= TOL and relerr(Kbh.numpy(), Kbo) <= TOL
    # pageable memory is accepted too
    Jp = torch.empty(nao, nao, dtype=torch.float64)
    h.get_jk_host(torch.from_numpy(C), Jp, None)
    assert relerr(Jp.numpy(), Jo) <= TOL
    h.close()


def test_single_element_probe_on_gpu(dfjk):
    """One non-zero packed entry lights exactly the entries the definition predicts."""
    nao, naux = 37, 3
    C = gi.random_orbitals(nao, 4, 99, orthonormal=False)
    G = C @ C.T
    for (mu, nu) in [(0, 0), (36, 0), (36, 36), (20, 7), (17, 16)]:
        Bp = np.zeros((naux, nao * (nao + 1) // 2))
        Bp[2, mu * (mu + 1) // 2 + nu] = 1.5
        E = np.zeros((nao, nao)); E[mu, nu] = E[nu, mu] = 1.5
        J, K, d = run_restricted(dfjk, Bp, nao, C)
        assert d[0] == 0.0 and d[1] == 0.0
        assert abs(d[2] - 2.0 * (E * G).sum()) <= 1e-13 * max(1.0, abs(d[2]))
        assert relerr(J, 2.0 * (E * G).sum() * E) <= 1e-13
        assert relerr(K, E @ G @ E) <= 1e-13


def test_error_paths(dfjk):
    L = dfjk.lib()
    nao = 8
    Bp, (C,) = rand_case(nao, 4, (3,), seed=1)
    Bd, Cd = dev(Bp), dev(C)
    out = torch.empty(nao, nao, dtype=torch.float64, device="cuda")
    assert not L.dfjk_create(0, nao, Bd.data_ptr()) and b"naux" in L.dfjk_last_error()
    assert not L.dfjk_create(4, 0, Bd.data_ptr())
    assert not L.dfjk_create(4, nao, None)
    assert not L.dfjk_create(4, nao, Bd.data_ptr() + 8) and b"aligned" in L.dfjk_last_error()
    hostbuf = np.zeros(4 * 36)
    assert not L.dfjk_create(4, nao, hostbuf.ctypes.data)
    h = L.dfjk_create(4, nao, Bd.data_ptr())
    assert h
    assert L.dfjk_get_jk(h, Cd.data_ptr(), 0, out.data_ptr(), None, None) == -1
    assert L.dfjk_get_jk(h, Cd.data_ptr(), nao + 1, out.data_ptr(), None, None) == -1
    assert L.dfjk_get_jk(h, None, 3, out.data_ptr(), None, None) == -1
    assert L.dfjk_get_jk(h, Cd.data_ptr(), 3, None, None, None) == -1
    assert L.dfjk_get_jk(None, Cd.data_ptr(), 3, out.data_ptr(), None, None) == -1
    assert L.dfjk_get_d(h, out.data_ptr(), None) == -1          # no J built yet
    assert L.dfjk_set_option(h, b"nonsense", 1) == -1
    assert L.dfjk_get_jk(h, Cd.data_ptr(), 3, out.data_ptr(), None, None) == 0
    assert L.dfjk_last_error() == b""
    torch.cuda.synchronize()
    assert L.dfjk_destroy(h) == 0 and L.dfjk_destroy(None) == 0


def test_seeded_shape_fuzz(dfjk):
    """40 seeded random shapes (nao 1..330, naux 1..24, nocc 1..nao, restricted / unrestricted /
    pair): every tile raggedness the persistent K1, the narrow K2 tiles and the J alignment cases
    can meet, each compared with the oracle in full."""
    rng = np.random.default_rng(20250606)
    for case in range(40):
        nao = int(rng.choice([rng.integers(1, 40), rng.integers(40, 140), rng.integers(140, 331)]))
        naux = int(rng.integers(1, 25))
        kind = case % 3
        if kind == 0:
            nocc = int(rng.integers(1, nao + 1))
            Bp, (C,) = rand_case(nao, naux, (nocc,), seed=1000 + case, orthonormal=bool(case & 1))
            J, K, d = run_restricted(dfjk, Bp, nao, C, k2_panel=(case // 3) % 2, k2_panel_kb=64)
            Jo, Ko, do = oracle.get_jk(Bp, nao, [C], [2.0])
            errs = [relerr(d, do), relerr(J, Jo), relerr(K, Ko[0])]
        elif kind == 1:
            na, nb = int(rng.integers(1, nao + 1)), int(rng.integers(1, nao + 1))
            Bp, (Ca, Cb) = rand_case(nao, naux, (na, nb), seed=1000 + case)
            h = dfjk.DFJK(dev(Bp), nao)
            h.set_option("k2_panel", (case // 3) % 2)
            h.set_option("k2_panel_kb", 64)
            J, Ka, Kb = h.get_jk_u(dev(Ca), dev(Cb))
            torch.cuda.synchronize()
            Jo, Kao, Kbo = oracle.get_jk_unrestricted(Bp, nao, Ca, Cb)
            errs = [relerr(J.cpu().numpy(), Jo), relerr(Ka.cpu().numpy(), Kao), relerr(Kb.cpu().numpy(), Kbo)]
            h.close()
        else:
            ncol = int(rng.integers(1, nao + 1))
            Bp, (C1, C2) = rand_case(nao, naux, (ncol, ncol), seed=1000 + case, orthonormal=False)
            h = dfjk.DFJK(dev(Bp), nao)
            h.set_option("k2_panel", (case // 3) % 2)
            h.set_option("k2_panel_kb", 64)
            J, K = h.get_jk_pair(dev(C1), dev(C2))
            torch.cuda.synchronize()
            Jo, Ko, _ = oracle.get_jk_pair(Bp, nao, C1, C2)
            errs = [relerr(J.cpu().numpy(), Jo), relerr(K.cpu().numpy(), Ko)]
            h.close()
        assert max(errs) <= TOL, (case, kind, nao, naux, errs)


def test_cuda_graph_capture_and_replay(dfjk):
    """dfjk_get_jk only enqueues kernels (no allocation, no host sync), so a caller can capture it in
    a CUDA graph and replay it per SCF iteration: one graph launch instead of 17 kernel launches
    (what makes the launch-bound small configs cheap).  The replay must see new C_occ contents."""
    cfg = gi.CONFIGS[1]
    Bp = gi.fill_B_host(cfg)
    h = dfjk.DFJK(dev(Bp), cfg.nao)
    C_static = dev(gi.orbitals(cfg, 0)[0])
    J = torch.empty(cfg.nao, cfg.nao, dtype=torch.float64, device="cuda")
    K = torch.empty_like(J)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        h.get_jk(C_static, out_j=J, out_k=K)             # warm-up outside the capture
    s.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        h.get_jk(C_static, out_j=J, out_k=K)
    for seed in (5, 6):
        C = gi.random_orbitals(cfg.nao, cfg.nocc[0], seed)
        C_static.copy_(torch.from_numpy(C))
        g.replay()
        torch.cuda.synchronize()
        Jo, Ko, _ = oracle.get_jk(Bp, cfg.nao, [C], [2.0])
        assert relerr(J.cpu().numpy(), Jo) <= TOL and relerr(K.cpu().numpy(), Ko[0]) <= TOL
    del g
    h.close()


def test_internal_graph_replay_matches_plain_launches(dfjk):
    """The handle's own CUDA graph ("graph" option, default on): the first call of a shape launches
    kernel by kernel, the second captures, later ones replay.  Every call gets FRESH orbital and
    output tensors (the replay must not remember pointers), interleaved with other shapes, and must
    equal the graph-free handle bit for bit and the oracle to tolerance."""
    nao, naux = 150, 19
    Bp, _ = rand_case(nao, naux, (7,), seed=31)
    Bd = dev(Bp)
    h, hp = dfjk.DFJK(Bd, nao), dfjk.DFJK(Bd, nao)
    hp.set_option("graph", 0)
    n0 = h.launch_count
    for it in range(6):
        nocc = 7 if it != 3 else 11                     # another shape in between (its own slot)
        C = gi.random_orbitals(nao, nocc, 400 + it)
        J, K = h.get_jk(dev(C))
        Jp, Kp = hp.get_jk(dev(C))
        d, dp = h.get_d(), hp.get_d()
        Jonly = h.get_jk(dev(C), with_k=False)[0]       # a third shape (J only)
        torch.cuda.synchronize()
        assert torch.equal(J, Jp) and torch.equal(K, Kp) and torch.equal(d, dp), it
        Jo, Ko, do = oracle.get_jk(Bp, nao, [C], [2.0])
        assert relerr(J.cpu().numpy(), Jo) <= TOL and relerr(K.cpu().numpy(), Ko[0]) <= TOL
        assert relerr(Jonly.cpu().numpy(), Jo) <= TOL and relerr(d.cpu().numpy(), do) <= TOL
    # the launch counter counts replayed kernels too: J+K calls cost the same on both handles, the
    # extra J-only calls on h add to it
    assert h.launch_count - n0 > hp.launch_count
    # unrestricted replay
    Ca, Cb = gi.random_orbitals(nao, 9, 1), gi.random_orbitals(nao, 5, 2)
    for it in range(3):
        J, Ka, Kb = h.get_jk_u(dev(Ca), dev(Cb))
        Jp, Kap, Kbp = hp.get_jk_u(dev(Ca), dev(Cb))
        torch.cuda.synchronize()
        assert torch.equal(J, Jp) and torch.equal(Ka, Kap) and torch.equal(Kb, Kbp)
    Jo, Kao, Kbo = oracle.get_jk_unrestricted(Bp, nao, Ca, Cb)
    assert relerr(J.cpu().numpy(), Jo) <= TOL and relerr(Ka.cpu().numpy(), Kao) <= TOL
    assert relerr(Kb.cpu().numpy(), Kbo) <= TOL
    h.close(); hp.close()


def test_two_handles_from_two_host_threads(dfjk):
    """Two host threads, each with its own handle and stream, first use of every kernel racing on
    the shared-memory opt-in (k_common.cuh ensure_dynamic_smem) and on the thread-local error text."""
    import threading
    shapes = [(131, 14, 9, 77), (197, 11, 141, 78)]       # different NT8 instantiations of K1
    cases = [rand_case(nao, naux, (nocc,), seed=seed) for nao, naux, nocc, seed in shapes]
    results, errors = [None, None], []
    start = threading.Barrier(2)

    def work(i):
        try:
            nao = shapes[i][0]
            Bp, (C,) = cases[i]
            torch.cuda.set_device(0)
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                h = dfjk.DFJK(dev(Bp), nao)
                start.wait(timeout=60)
                outs = []
                for _ in range(4):
                    J, K = h.get_jk(dev(C))
                    outs.append((J, K))
                s.synchronize()
                results[i] = [(J.cpu().numpy(), K.cpu().numpy()) for J, K in outs]
                h.close()
        except Exception as e:          # noqa: BLE001
            errors.append((i, repr(e)))

    ts = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in ts:
        t.start()
    for t in ts:
        t.join(300)
    assert not errors, errors
    for i, (nao, naux, nocc, seed) in enumerate(shapes):
        Bp, (C,) = cases[i]
        Jo, Ko, _ = oracle.get_jk(Bp, nao, [C], [2.0])
        for J, K in results[i]:
            assert relerr(J, Jo) <= TOL and relerr(K, Ko[0]) <= TOL


def test_kernel_timing_ring_grows(dfjk):
    """More than the initial 1024 event pairs: the ring grows instead of silently dropping launches."""
    nao = 40
    Bp, (C,) = rand_case(nao, 6, (3,), seed=9)
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("k_chunk", 1)                            # 6 chunks -> ~25 launches per call
    h.set_option("time_kernels", 1)
    Cd = dev(C)
    n0 = h.launch_count
    for _ in range(100):
        h.get_jk(Cd)
    torch.cuda.synchronize()
    total = sum(h.kernel_time(k)[1] for k in dfjk.KERNELS)
    assert total == h.launch_count - n0 and total > 1024
    h.close()
