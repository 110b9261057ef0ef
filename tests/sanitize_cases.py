"""Small driver for `compute-sanitizer` ("race detection / sanitizers").

Not a pytest file (pytest does not collect it): run it plainly first, then under ONE tool per GPU call,

    python tests/sanitize_cases.py
    compute-sanitizer --tool memcheck  python tests/sanitize_cases.py
    compute-sanitizer --tool initcheck python tests/sanitize_cases.py
    compute-sanitizer --tool racecheck python tests/sanitize_cases.py

It walks every kernel family of libdfjk.so through the code paths where an out-of-bounds,
uninitialised or racy access could hide behind a green parity test: the packed-triangle TMA row
copies of K1 that start one element before a row and run past its end, the special-cased last row
of the last P, the mbarrier rings, the cross-CTA flag chains of the panel-synchronous K2, padded
workspace read by later kernels.  Shapes: BASELINE configs 1 and 2 (one call), ragged nao / naux /
nocc, unrestricted, pair and raw-dm densities, dfjk_build_b, the SCF driver, the Eq. 7 diagonal with
and without a handle -- each K build on BOTH K2 kernels (k2_panel 0 / 1 with 64 KB panels, so that
even these small problems are cut into several panels and slabs).

Every result is also compared with the CPU oracle (1e-11 relative Frobenius), so a tool run that
ends with "0 errors" has checked the same values the parity tests do.  Exit status 0 = all cases ran
and agreed.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

import dfjk_inputs as gi  # noqa: E402
import oracle  # noqa: E402
from oracle import scf as oscf  # noqa: E402
import paper_2506_06661_b200 as dfjk  # noqa: E402

TOL = 1e-11


def relerr(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / (nb if nb > 0 else 1.0)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check(name, got, want, tol=TOL):
    e = relerr(got.cpu().numpy() if hasattr(got, "cpu") else got, want)
    print(f"  {name}: relF = {e:.2e}", flush=True)
    if not e <= tol:
        raise SystemExit(f"sanitize_cases: {name} disagrees with the oracle ({e:.3e} > {tol})")


def both_k2(h):
    """the two K2 kernels, panels short enough that small problems still use several panels / slabs"""
    h.set_option("k2_panel_kb", 64)
    for k2_panel in (0, 1):
        h.set_option("k2_panel", k2_panel)
        yield k2_panel


def restricted(nao, naux, nocc, seed, Bp=None, C=None, k_chunk=0):
    print(f"restricted nao={nao} naux={naux} nocc={nocc}", flush=True)
    if Bp is None:
        Bp = gi.fill_B_host(gi.custom_config(nao, naux, (nocc,), seed=seed))
        C = gi.random_orbitals(nao, nocc, seed + 1)
    Jo, Ko = oracle.get_jk_restricted(Bp, nao, C)
    h = dfjk.DFJK(dev(Bp), nao)
    if k_chunk:
        h.set_option("k_chunk", k_chunk)
    for p in both_k2(h):
        for fused in (1, 0):
            h.set_option("j_fused", fused)
            for rep in range(2):                       # second call of a shape captures / replays a graph
                J, K = h.get_jk(dev(C))
            torch.cuda.synchronize()
            check(f"J k2_panel={p} j_fused={fused}", J, Jo)
            check(f"K k2_panel={p} j_fused={fused}", K, Ko)
    Jonly, _ = h.get_jk(dev(C), with_k=False)
    _, Konly = h.get_jk(dev(C), with_j=False)
    torch.cuda.synchronize()
    check("J only", Jonly, Jo)
    check("K only", Konly, Ko)
    h.close()


def unrestricted(nao, naux, na, nb, seed):
    print(f"unrestricted nao={nao} naux={naux} nocc=({na},{nb})", flush=True)
    Bp = gi.fill_B_host(gi.custom_config(nao, naux, (na, nb), seed=seed))
    Ca, Cb = gi.random_orbitals(nao, na, seed + 1), gi.random_orbitals(nao, nb, seed + 2)
    Jo, Kao, Kbo = oracle.get_jk_unrestricted(Bp, nao, Ca, Cb)
    h = dfjk.DFJK(dev(Bp), nao)
    h.set_option("k_chunk", max(1, naux // 3))         # several X chunks: the accumulate path
    for p in both_k2(h):
        J, Ka, Kb = h.get_jk_u(dev(Ca), dev(Cb))
        torch.cuda.synchronize()
        check(f"J k2_panel={p}", J, Jo)
        check(f"K_a k2_panel={p}", Ka, Kao)
        check(f"K_b k2_panel={p}", Kb, Kbo)
    h.close()


def general(nao, naux, ncol, seed):
    print(f"pair / raw dm nao={nao} naux={naux} ncol={ncol}", flush=True)
    Bp = gi.fill_B_host(gi.custom_config(nao, naux, (1,), seed=seed))
    rng = np.random.default_rng(seed)
    C1, C2 = rng.standard_normal((nao, ncol)), rng.standard_normal((nao, ncol))
    dm = rng.standard_normal((nao, nao))
    Jpo, Kpo, _ = oracle.get_jk_pair(Bp, nao, C1, C2)
    Jdo, Kdo, _ = oracle.get_jk_dm(Bp, nao, dm)
    h = dfjk.DFJK(dev(Bp), nao)
    for p in both_k2(h):
        for fused in (1, 0):
            h.set_option("j_fused", fused)
            J, K = h.get_jk_pair(dev(C1), dev(C2))
            torch.cuda.synchronize()
            check(f"pair J k2_panel={p} j_fused={fused}", J, Jpo)
            check(f"pair K k2_panel={p} j_fused={fused}", K, Kpo)
        J, K = h.get_jk_dm(dev(dm))
        torch.cuda.synchronize()
        check(f"dm J k2_panel={p}", J, Jdo)
        check(f"dm K k2_panel={p}", K, Kdo)
    diag = h.get_df_diag()
    out = torch.empty(nao, nao, dtype=torch.float64, device="cuda")
    dfjk.df_diag_noalloc(h.B, nao, out)
    torch.cuda.synchronize()
    want = oracle.df_diag(Bp, nao)
    check("df_diag (handle)", diag, want)
    check("df_diag (no-alloc)", out, want)
    h.close()


def build_b(nao, naux, seed):
    print(f"build_b nao={nao} naux={naux}", flush=True)
    cfg = gi.custom_config(nao, naux, (1,), seed=seed)
    M, R = gi.metric(cfg), gi.fill_B_host(cfg)
    Lo, Bo = oracle.build_b(M, R)
    Md, Rd = dev(M), dev(R)
    info = dfjk.build_b(Md, Rd, nao)
    torch.cuda.synchronize()
    assert int(info.item()) == 0
    check("L", torch.tril(Md), np.tril(Lo))
    check("B", Rd, Bo)


def scf_case(nao, naux, nocc, seed):
    print(f"scf nao={nao} naux={naux} nocc={nocc}", flush=True)
    cfg = gi.custom_config(nao, naux, (nocc,), seed=seed)
    Bp = gi.fill_B_host(cfg) * 0.3
    hc, S = gi.core_hamiltonian(cfg), gi.overlap(cfg)
    ref = oscf.scf_rhf(Bp, nao, hc, S, nocc, conv_tol=1e-10, diis_space=4)
    h = dfjk.DFJK(dev(Bp), nao)
    out = h.scf_rhf(dev(hc), dev(S), nocc, conv_tol=1e-10, diis_space=4)
    e, eo = np.array(out["e_hist"]), np.array(ref["e_hist"])
    assert out["converged"] and len(e) == len(eo)
    check("E per iteration", e, eo, 1e-9)
    u = h.scf_uhf(dev(hc), dev(S), nocc, nocc - 1, conv_tol=1e-10, diis_space=4)
    refu = oscf.scf_uhf(Bp, nao, hc, S, nocc, nocc - 1, conv_tol=1e-10, diis_space=4)
    assert u["converged"]
    check("UHF E per iteration", np.array(u["e_hist"]), np.array(refu["e_hist"]), 1e-9)
    h.close()


def main():
    assert torch.cuda.is_available(), "sanitize_cases needs a CUDA device"
    torch.cuda.set_device(0)
    dfjk.lib()
    for cid in (1, 2):                                 # BASELINE.json configs[0], configs[1]
        cfg = gi.CONFIGS[cid]
        restricted(cfg.nao, cfg.naux, cfg.nocc[0], 0, Bp=gi.fill_B_host(cfg), C=gi.orbitals(cfg, 0)[0])
    for nao, naux, nocc in ((129, 10, 3), (150, 11, 10), (190, 7, 12), (400, 13, 30), (96, 5, 40)):
        restricted(nao, naux, nocc, 1000 + nao, k_chunk=max(1, naux // 2))
    restricted(700, 9, 20, 5)                          # 6 x 6 tiles: the automatic K2P size class
    unrestricted(150, 11, 10, 7, 21)
    unrestricted(300, 9, 33, 30, 22)
    general(129, 10, 31, 31)
    general(200, 8, 13, 32)
    build_b(40, 200, 41)
    build_b(24, 300, 42)
    scf_case(60, 200, 10, 3)
    print("sanitize_cases: all cases agree with the oracle", flush=True)


if __name__ == "__main__":
    main()
