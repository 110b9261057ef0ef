#!/usr/bin/env python
"""bench.py -- DF get_jk throughput on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path: one ``dfjk_get_jk`` (J and K, SURVEY.md
section 8a rows J0-J3, K0-K3) for one fresh C_occ of the config's call schedule, B
resident in HBM.  Default workload = BASELINE.json configs[3] (nao=1600, naux=5000,
nocc=130: the config the metric's roofline target is quoted on; 51 GB fits one GPU).

  value      algorithmic GFLOP/s of the whole job (all ranks), inputs resident in HBM
  e2e        the same through dfjk_get_jk_host: C_occ from pinned HOST memory, J and K
             back to pinned HOST memory inside the timed region (B stays resident:
             it is the handle's state, built once per geometry like the paper's with_df)
  roofline   dominant kernel (K1 half transform, 2/3 of the flops): DMMA on the FP64 pipe
  cpu_baseline  the oracle on this box's host cores, on a bounded row-slab sample

Multi-GPU (--gpus N under torchrun): the path does not shard (north_star: one GPU, no
collectives) => N independent replicas, weak scaling, no data-path collective.
``--impl reference`` times the CPU oracle as it stands (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import dfjk_inputs as gi  # noqa: E402

FP64_PEAK_FALLBACK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # only if the device cannot be queried
HBM_FALLBACK_GBS = 6650.0


def flops_j(cfg):
    return 4.0 * cfg.naux * cfg.npair


def flops_k1(cfg):
    return 2.0 * cfg.naux * cfg.nao ** 2 * sum(cfg.nocc)


def flops_k2(cfg):
    return 1.0 * cfg.naux * cfg.nao * (cfg.nao + 1) * sum(cfg.nocc)


def flops_step(cfg):
    return flops_j(cfg) + flops_k1(cfg) + flops_k2(cfg)


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": HBM_FALLBACK_GBS}, "fallback"


def fp64_peak(pkg):
    """FP64 roofline denominator, read from the device: derived = SMs x 64 FMA/clk x 2 x peak SM
    clock (dfjk_device_info), probe = the register-only DMMA loop (dfjk_probe_dmma_peak) measured in
    this run; fractions are quoted against the smaller of the two, so that neither a different SKU
    nor a capped box can flatter them."""
    try:
        info = pkg.device_info()
        derived = info["fp64_peak_tflops"]
    except Exception:
        info, derived = {}, FP64_PEAK_FALLBACK_TFLOPS
    probe = pkg.probe_fp64_peak()
    used = min(derived, probe) if probe > 0 else derived
    return {"peak": used, "derived_tflops": derived, "probe_tflops": probe,
            "sm_count": info.get("sm_count"), "sm_clock_khz": info.get("sm_clock_khz"),
            "source": f"min(derived, probe): derived = {info.get('sm_count')} SM x 64 FP64 FMA/clk x 2 x "
                      f"{info.get('sm_clock_khz', 0) / 1e6:.3f} GHz (dfjk_device_info), probe = "
                      "dfjk_probe_dmma_peak's register-only DMMA.8x8x4 loop measured in this run; "
                      "sm_100a has no tcgen05 FP64 kind"}


def max_over_ranks(x, dist=None, device="cpu"):
    """MAX over ranks of a host scalar (the timing rule: a multi-GPU step takes as long as its
    slowest replica).  dist=None (single process) returns x."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(flops_per_step, steps, total_ms, world):
    """Aggregate GFLOP/s of `world` independent replicas ("replicas only", weak scaling): every
    rank does `steps` steps of flops_per_step in the max-over-ranks time total_ms."""
    return world * flops_per_step * steps / (total_ms * 1e-3) / 1e9


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "power_w": float(np.median(pw)) if pw else None,
                "reasons": sorted(reasons)}


def oracle_full(cfg, call=0, slab=250):
    """Time the oracle (as it stands) on ALL rows of the config's B, fed slab by slab (the tensor is up
    to 96 GB: it is generated, consumed and dropped 250 rows at a time; only the oracle's own time is
    summed, not the generator's).  Returns seconds, threads."""
    import oracle
    Cs = gi.orbitals(cfg, call)
    warm = oracle.JKAccumulator(cfg.nao, Cs, cfg.weights)
    warm.add_slab(gi.fill_B_host(cfg, 0, 1))   # touch the code path / page in
    acc = oracle.JKAccumulator(cfg.nao, Cs, cfg.weights)
    t = 0.0
    for P0 in range(0, cfg.naux, slab):
        Bp = gi.fill_B_host(cfg, P0, min(slab, cfg.naux - P0))
        t0 = time.perf_counter()
        acc.add_slab(Bp)
        t += time.perf_counter() - t0
    return t, oracle.num_threads()


def oracle_sample(cfg, rows, call=0):
    """Time the oracle (as it stands) on `rows` rows of the config's B. Returns seconds, threads."""
    import oracle
    Bp = gi.fill_B_host(cfg, 0, rows)
    Cs = gi.orbitals(cfg, call)
    acc = oracle.JKAccumulator(cfg.nao, Cs, cfg.weights)
    acc.add_slab(Bp[:1])                       # touch the code path / page in
    acc = oracle.JKAccumulator(cfg.nao, Cs, cfg.weights)
    t0 = time.perf_counter()
    acc.add_slab(Bp)
    return time.perf_counter() - t0, oracle.num_threads()


def size_sample(cfg, target_s):
    """Grow the row-slab until the oracle takes about target_s seconds (or all rows)."""
    rows = min(4, cfg.naux)
    while True:
        t, threads = oracle_sample(cfg, rows)
        if t >= target_s / 3 or rows >= cfg.naux:
            return rows, t, threads
        rows = int(min(cfg.naux, max(2 * rows, 0.8 * rows * target_s / max(t, 1e-6))))


def run_reference(args, cfg):
    """--impl reference: the CPU oracle on this box's host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    per_row = flops_step(cfg) / cfg.naux
    # size the per-step sample from one pilot row-slab: aim at ~5 s per step
    rows, _, threads = size_sample(cfg, 5.0)
    Bp = gi.fill_B_host(cfg, 0, rows)
    times = []
    for step in range(args.warmup + args.steps):
        Cs = gi.orbitals(cfg, 0)
        acc = oracle.JKAccumulator(cfg.nao, Cs, cfg.weights)
        t0 = time.perf_counter()
        acc.add_slab(Bp)
        dt = time.perf_counter() - t0
        if step >= args.warmup:
            times.append(dt)
    t = float(np.mean(times))
    val = per_row * rows / t / 1e9
    sample = f"{rows} of {cfg.naux} auxiliary rows of cfg {cfg.index} per step (J and K, full nao)"
    print(json.dumps({
        "impl": "reference", "metric": "df_get_jk_gflops_fp64", "value": val, "unit": "GFLOP/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t * 1e3, "ms_per_step_scaled": t * 1e3 * cfg.naux / rows,
        "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, args),
        "cpu_baseline": {"value": val, "unit": "GFLOP/s", "cores": threads, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "note": "ms_per_step is the MEASURED time of one step = the oracle on the row sample; "
                "ms_per_step_scaled extrapolates it to all naux rows (the oracle is linear in P); value "
                "is a rate: algorithmic flops of the sample (4 npair + 3 nao^2 nocc per row) over the "
                "measured time, the oracle itself does the full-square work",
    }))


def workload_config(cfg, args, fused=True):
    origin = (f"BASELINE.json configs[{cfg.index - 1}]" if cfg.index <= 5 else
              "LRDF-shaped workload (PAPER.md:433-450, naux = nao/10; not a BASELINE config)")
    passes = ("twice (K1's unpack, J2's axpy; d_P is read off the half-transformed X)" if fused else
              "three times (J1 dot, J2 axpy, K1's unpack)")
    return {"workload": f"{origin} '{cfg.name}': nao={cfg.nao} "
                        f"naux={cfg.naux} nocc={'+'.join(map(str, cfg.nocc))} seed={cfg.seed}",
            "nao": cfg.nao, "naux": cfg.naux, "nocc": list(cfg.nocc),
            "b_bytes": cfg.b_bytes, "calls_per_step": 1,
            "l2": f"inputs larger than L2: every step streams the packed B ({cfg.b_bytes / 1e9:.1f} GB) {passes}"
                  if cfg.b_bytes > (1 << 30) else "L2 flushed between steps (256 MB write)",
            "parallelism": f"replicas x{args.gpus}" if args.gpus > 1 else "single GPU"}


class Workload:
    """One config resident on the device: B generated in place, a handle, the call schedule."""

    def __init__(self, pkg, cfg, dev, ncalls):
        import torch
        self.pkg, self.cfg, self.dev = pkg, cfg, dev
        self.unrestricted = len(cfg.nocc) == 2
        self.B = torch.empty(cfg.naux, cfg.npair, dtype=torch.float64, device=dev)
        gi.fill_B_device(cfg, self.B)
        self.h = pkg.DFJK(self.B, cfg.nao)
        self.Cs_host = list(gi.orbital_sequence(cfg, ncalls))          # [call][set] numpy, host
        self.Cs_dev = [[torch.from_numpy(C).to(dev) for C in sets] for sets in self.Cs_host]
        self.flush = (None if cfg.b_bytes > (1 << 30)
                      else torch.empty(256 << 20, dtype=torch.uint8, device=dev))

    def step(self, k, **kw):
        sets = self.Cs_dev[k % len(self.Cs_dev)]
        if self.unrestricted:
            return self.h.get_jk_u(sets[0], sets[1], **kw)
        return self.h.get_jk(sets[0], **kw)

    def close(self):
        import torch
        self.h.close()
        del self.B, self.Cs_dev, self.flush
        torch.cuda.empty_cache()


def timed_steps(wl, first, steps, barrier, local, step_fn=None):
    """`steps` steps bracketed by CUDA events on the launching stream, barrier + synchronize on both
    sides, clocks sampled meanwhile.  Per-kernel event brackets are OFF here (they would sit inside
    the timed region); kernel_breakdown() collects them from an untimed pass over the same calls."""
    import torch
    wl.h.set_option("time_kernels", 0)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(steps)]
    step_fn = step_fn or wl.step
    launches0 = wl.h.launch_count
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    for k in range(steps):
        if wl.flush is not None:
            wl.flush.fill_(k & 0xFF)
        ev[k][0].record()
        step_fn(first + k)
        ev[k][1].record()
    barrier()
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    return step_ms, clocks, wl.h.launch_count - launches0


def kernel_breakdown(wl, first, steps, **kw):
    """Per-kernel CUDA-event times (ms per step) of the same calls, launched again OUTSIDE the
    timed region with the library's event brackets on."""
    import torch
    wl.h.set_option("time_kernels", 1)
    for k in range(steps):
        wl.step(first + k, **kw)
    torch.cuda.synchronize()
    kt = {name: wl.h.kernel_time(name) for name in wl.pkg.KERNELS}
    wl.h.set_option("time_kernels", 0)
    return {n: (ms / steps, cnt) for n, (ms, cnt) in kt.items()}


def j_and_k_summary(cfg, kt, peak, hbm, peak_src):
    """J / K sub-records from a per-step kernel breakdown."""
    k1, k2 = kt["K1"][0], kt["K2"][0]
    j_ms = sum(kt[n][0] for n in ("J0", "J1", "J1R", "J2", "J3"))
    k_ms = sum(kt[n][0] for n in ("K1", "K2", "K3"))
    j2 = kt["J2"][0]
    kf = flops_k1(cfg) + flops_k2(cfg)
    return ({"ms": j_ms, "fused": True, "stream_ms": j2, "bytes": cfg.b_bytes,
             "gbs": cfg.b_bytes / (j2 * 1e-3) / 1e9 if j2 > 0 else None,
             "hbm_peak_gbs": hbm, "peak_source": peak_src,
             "frac": cfg.b_bytes / (j2 * 1e-3) / 1e9 / hbm if j2 > 0 else None,
             "d_from_x_ms": kt["J1"][0]},
            {"ms": k_ms, "tflops": kf / (k_ms * 1e-3) / 1e12 if k_ms > 0 else None,
             "frac_fp64_peak": kf / (k_ms * 1e-3) / 1e12 / peak if k_ms > 0 else None,
             "k1_ms": k1, "k2_ms": k2,
             "k1_tflops": flops_k1(cfg) / (k1 * 1e-3) / 1e12 if k1 > 0 else None,
             "k2_tflops": flops_k2(cfg) / (k2 * 1e-3) / 1e12 if k2 > 0 else None})


def two_pass_j(wl, first, n, hbm):
    """north_star's J path as written -- two plain streaming passes over B (J1 dot, J2 axpy) -- timed
    on J-only calls outside the timed region: 2|B| bytes over t_J1 + t_J2."""
    wl.h.set_option("j_fused", 0)
    kt = kernel_breakdown(wl, first, n, with_k=False)
    wl.h.set_option("j_fused", 1)
    t2 = kt["J1"][0] + kt["J2"][0]
    gbs = 2 * wl.cfg.b_bytes / (t2 * 1e-3) / 1e9 if t2 > 0 else None
    return {"stream_ms": t2, "bytes": 2 * wl.cfg.b_bytes, "gbs": gbs,
            "frac": gbs / hbm if gbs else None}


def other_workloads(pkg, wl4, args, dev, local, barrier, peak, hbm, peak_src):
    """Short timed passes (3 warm-up + 3 steps each, same protocol) of the workloads the headline does
    not cover, so that every number quoted in DESIGN.md is observed in the driver's own run:
    the section-8f operations at cfg 4 (on the resident B), then BASELINE configs 3, 5, 2, 1 and the
    LRDF shape."""
    import torch
    out = {}      # the section-8f operations at cfg 4: run first (B is resident), emitted LAST (see the end)
    W, K = 3, 3
    cc = lambda c: {"sm_mhz": c.get("sm_mhz"), "reasons": c.get("reasons")}   # the driver keeps only the tail of
    cfg = wl4.cfg                                                             # stdout: every entry stays short
    nao, naux, nocc = cfg.nao, cfg.naux, cfg.nocc[0]
    rng = np.random.default_rng(cfg.seed)

    def timed(run, prep=None, warm=W, steps=K):
        for _ in range(warm):
            if prep:
                prep()
            run()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        sampler = ClockSampler(local)
        barrier()
        sampler.start()
        for k in range(steps):
            if prep:
                prep()
            ev[k][0].record()
            run()
            ev[k][1].record()
        barrier()
        clocks = sampler.stop()
        return float(np.median([a.elapsed_time(b) for a, b in ev])), clocks

    # -- section 8f rank 1: the pair form (response-like density by its factors)
    C1 = torch.from_numpy(rng.standard_normal((nao, nocc))).to(dev)
    C2 = torch.from_numpy(rng.standard_normal((nao, nocc))).to(dev)
    ms, clocks = timed(lambda: wl4.h.get_jk_pair(C1, C2))
    fl = flops_j(cfg) + 2.0 * naux * nao ** 2 * (2 * nocc) + 2.0 * naux * nao ** 2 * nocc
    out["cfg4_pair"] = {"op": f"get_jk_pair ncol={nocc}", "ms": ms, "frac_fp64_peak": fl / ms / 1e9 / peak, **cc(clocks)}
    # -- section 8f rank 1, batch half: several pairs from one sweep over B against the same pairs one by one
    for nb, nc in ((8, 8), (4, 32)):
        A = [torch.from_numpy(rng.standard_normal((nao, nc))).to(dev) for _ in range(nb)]
        Bf = [torch.from_numpy(rng.standard_normal((nao, nc))).to(dev) for _ in range(nb)]
        ms_b, clocks = timed(lambda: wl4.h.get_jk_pairs(A, Bf))
        ms_1, _ = timed(lambda: [wl4.h.get_jk_pair(a, b) for a, b in zip(A, Bf)])
        wl4.h.set_option("time_kernels", 1)
        wl4.h.get_jk_pairs(A, Bf)
        torch.cuda.synchronize()
        k1_ms, k1_n = wl4.h.kernel_time("K1")
        j2_ms, j2_n = wl4.h.kernel_time("J2")
        wl4.h.set_option("time_kernels", 0)
        k1_fl = 2.0 * naux * nao ** 2 * (2 * nb * ((nc + 7) // 8 * 8))
        out[f"cfg4_pairs_{nb}x{nc}"] = {"op": f"get_jk_pairs: {nb} pairs of ncol {nc} in one call", "ms": ms_b,
                                        "ms_one_by_one": ms_1, "ratio": ms_b / ms_1, "k1_ms": k1_ms, "k1_launches": k1_n,
                                        "k1_frac_fp64_peak": k1_fl / k1_ms / 1e9 / peak if k1_ms > 0 else None,
                                        "j2_ms": j2_ms, "j2_passes": j2_n, **cc(clocks)}
        del A, Bf
    # -- section 8f rank 3: Eq. 7's DF diagonal, one pass over B
    ms, clocks = timed(lambda: wl4.h.get_df_diag())
    out["cfg4_diag"] = {"op": "get_df_diag (Eq. 7)", "ms": ms, "gbs": cfg.b_bytes / ms / 1e6,
                        "frac_hbm": cfg.b_bytes / ms / 1e6 / hbm, **cc(clocks)}
    # -- the north_star configuration of the whole step: J by two plain passes over B (j_fused = 0)
    wl4.h.set_option("j_fused", 0)
    ms, clocks = timed(lambda: wl4.step(0))
    wl4.h.set_option("j_fused", 1)
    out["cfg4_two_pass_j"] = {"op": "get_jk, j_fused=0 (J1 dot + J2 axpy)", "ms": ms,
                              "gflops": flops_step(cfg) / ms / 1e6, **cc(clocks)}
    # -- section 8f rank 4: the SCF driver, 4 fixed iterations (B scaled so the two-electron term is a
    #    perturbation; build_b below regenerates B)
    try:
        wl4.B.mul_(0.02)
        hc = torch.from_numpy(gi.core_hamiltonian(cfg)).to(dev)
        S = torch.from_numpy(gi.overlap(cfg)).to(dev)
        res = {}
        ms, clocks = timed(lambda: res.update(wl4.h.scf_rhf(hc, S, nocc, max_iter=4, conv_tol=1e-300)), warm=1, steps=1)
        tm = res.get("timing") or {}
        out["cfg4_scf"] = {"op": "scf_rhf, 4 iterations", "ms_per_iteration": ms / 4, "get_jk_ms": tm.get("get_jk"),
                           "eig_ms": tm.get("eigensolver"), "glue_ms": tm.get("glue"), **cc(clocks)}
        del hc, S
    except Exception as e:
        out["cfg4_scf"] = {"error": repr(e)[:120]}
    # -- section 8f rank 2: building B in place (once: 1 warm-up + 1 timed, ~1 s each)
    Mh = torch.from_numpy(gi.metric(cfg)).pin_memory()
    Md = torch.empty(naux, naux, dtype=torch.float64, device=dev)

    def prep():
        Md.copy_(Mh, non_blocking=True)
        gi.fill_B_device(cfg, wl4.B)                 # R is overwritten in place: regenerate it
    ms, clocks = timed(lambda: pkg.build_b(Md, wl4.B, nao), prep, warm=1, steps=1)
    fl = float(naux) ** 2 * cfg.npair + float(naux) ** 3 / 3.0
    out["cfg4_build_b"] = {"op": "build_b (Eq. 2-3, in place)", "ms": ms, "frac_fp64_peak": fl / ms / 1e9 / peak, **cc(clocks)}
    del Md, Mh, C1, C2
    wl4.close()
    f_ops, out = out, {}

    for cid in (3, 5, 2, 1, 6):
        c = gi.CONFIGS[cid]
        free, _ = torch.cuda.mem_get_info()
        if free < c.b_bytes + (6 << 30):
            out[f"cfg{cid}"] = {"skipped": f"needs {c.b_bytes / 1e9:.0f} GB of free device memory"}
            continue
        # sub-millisecond configs: enough warm-up and timed steps for the SM clock to have ramped up
        # (3 + 3 steps of 0.05-0.6 ms after an idle gap read 15-20 % slow now and then)
        Wc, Kc = (W, K) if c.b_bytes > (1 << 30) else (30, 30)
        wl = Workload(pkg, c, dev, Wc + Kc)
        for k in range(Wc):
            wl.step(k)
        step_ms, clocks, launches = timed_steps(wl, Wc, Kc, barrier, local)
        kt = kernel_breakdown(wl, Wc, min(Kc, 5))
        j, kk = j_and_k_summary(c, kt, peak, hbm, peak_src)
        ms = float(np.mean(step_ms))
        rec = {"shape": f"nao {c.nao} naux {c.naux} nocc {'+'.join(map(str, c.nocc))}", "ms_per_step": ms, "steps": Kc,
               "gflops": flops_step(c) / ms / 1e6, "launches_per_step": launches / Kc,
               "k_frac_fp64_peak": kk["frac_fp64_peak"], "k1_ms": kk["k1_ms"], "k2_ms": kk["k2_ms"],
               "j_ms": j["ms"], "j_gbs": j["gbs"], **cc(clocks)}
        if c.b_bytes > (1 << 30):
            rec["j_two_pass_gbs"] = two_pass_j(wl, Wc, 2, hbm)["gbs"]
        out[f"cfg{cid}"] = rec
        wl.close()
    out.update(f_ops)          # last in the line: they survive in a record that keeps only the tail of stdout
    return out


def run_ours(args, cfg):
    import torch
    import paper_2506_06661_b200 as pkg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    pkg.lib()
    pk = fp64_peak(pkg) if rank == 0 else None       # device-derived + measured FP64 pipe rate (untimed)
    peaks, peak_src = measured_peaks()
    hbm = float(peaks.get("hbm_gbs", HBM_FALLBACK_GBS))
    wl = Workload(pkg, cfg, dev, args.warmup + args.steps)
    h, unrestricted = wl.h, wl.unrestricted
    for k in range(args.warmup):
        wl.step(k)
    step_fn = None
    if args.graph and not unrestricted:
        # caller-side CUDA graph: one replay per step; the step's C_occ is copied into the captured
        # input buffer inside the timed region
        C_in = wl.Cs_dev[0][0].clone()
        Jg = torch.empty(cfg.nao, cfg.nao, dtype=torch.float64, device=dev)
        Kg = torch.empty_like(Jg)
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            h.get_jk(C_in, out_j=Jg, out_k=Kg)
        side.synchronize()
        graph = torch.cuda.CUDAGraph()
        n0 = h.launch_count
        with torch.cuda.graph(graph, stream=side):
            h.get_jk(C_in, out_j=Jg, out_k=Kg)
        launches_per_replay = h.launch_count - n0     # kernels inside one captured get_jk

        def step_fn(k):
            C_in.copy_(wl.Cs_dev[k][0])
            graph.replay()
        step_fn(0)
    step_ms, clocks, launches = timed_steps(wl, args.warmup, args.steps, barrier, local, step_fn)
    if step_fn is not None:
        launches = launches_per_replay * args.steps   # replays bypass the host-side counter
    total_ms = max_over_ranks(float(sum(step_ms)), dist, dev)
    kt = kernel_breakdown(wl, args.warmup, args.steps)
    two_pass = two_pass_j(wl, args.warmup, min(args.steps, 3), hbm)

    # ---- end to end through the host entry points
    if unrestricted:
        Ch = [[torch.from_numpy(c).pin_memory() for c in s] for s in wl.Cs_host]
        Jh, Kah, Kbh = (torch.empty(cfg.nao, cfg.nao, dtype=torch.float64).pin_memory() for _ in range(3))
        h.get_jk_u_host(Ch[0][0], Ch[0][1], Jh, Kah, Kbh)
        barrier()
        t0 = time.perf_counter()
        for k in range(args.steps):
            h.get_jk_u_host(Ch[args.warmup + k][0], Ch[args.warmup + k][1], Jh, Kah, Kbh)
        e2e_s = max_over_ranks(time.perf_counter() - t0, dist, dev)
        e2e = {"value": whole_job_value(flops_step(cfg), args.steps, e2e_s * 1e3, world), "unit": "GFLOP/s",
               "ms_per_step": e2e_s * 1e3 / args.steps,
               "h2d_bytes_per_step": cfg.nao * sum(cfg.nocc) * 8, "d2h_bytes_per_step": 3 * cfg.nao * cfg.nao * 8,
               "api": "dfjk_get_jk_u_host (pinned host C_a, C_b in, pinned host J, K_a, K_b out; B resident)"}
    else:
        nocc = cfg.nocc[0]
        Ch = [torch.from_numpy(s[0]).pin_memory() for s in wl.Cs_host]
        Jh = torch.empty(cfg.nao, cfg.nao, dtype=torch.float64).pin_memory()
        Kh = torch.empty(cfg.nao, cfg.nao, dtype=torch.float64).pin_memory()
        h.get_jk_host(Ch[0], Jh, Kh)
        barrier()
        t0 = time.perf_counter()
        for k in range(args.steps):
            h.get_jk_host(Ch[args.warmup + k], Jh, Kh)
        e2e_s = time.perf_counter() - t0
        e2e_s = max_over_ranks(e2e_s, dist, dev)
        e2e = {"value": whole_job_value(flops_step(cfg), args.steps, e2e_s * 1e3, world), "unit": "GFLOP/s",
               "ms_per_step": e2e_s * 1e3 / args.steps,
               "h2d_bytes_per_step": cfg.nao * nocc * 8, "d2h_bytes_per_step": 2 * cfg.nao * cfg.nao * 8,
               "api": "dfjk_get_jk_host (pinned host C_occ in, pinned host J and K out; B resident)"}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak = pk["peak"]
    ms_per_step = total_ms / args.steps
    value = whole_job_value(flops_step(cfg), args.steps, total_ms, world)
    k1_ms, k1_n = kt["K1"]                            # ms per step, launches in the breakdown pass
    # DRAM bytes of the dominant kernel from the committed ncu --set full capture
    # (profiles/traffic.csv), scaled from the captured launch's rows to the average launch
    traffic = None
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for row in csv.DictReader(f):
                if int(row["cfg"]) == cfg.index and row["kernel"] == "K1" and k1_n > 0:
                    per_row = (float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])) / float(row["rows_in_launch"])
                    traffic = per_row * cfg.naux * args.steps / k1_n
    except Exception:
        pass
    k1_tflops = flops_k1(cfg) / (k1_ms * 1e-3) / 1e12 if k1_ms > 0 else 0.0
    roofline = {"kernel": "k1_half_transform_kernel (X_P = B_P C, DMMA.8x8x4 on the FP64 pipe)",
                "bound": "alu", "achieved": k1_tflops, "peak": peak, "unit": "TFLOP/s",
                "frac": k1_tflops / peak, "traffic": traffic, "peak_source": pk["source"],
                "peak_derived_tflops": pk["derived_tflops"], "peak_probe_tflops": pk["probe_tflops"],
                "launches": k1_n, "avg_launch_ms": k1_ms * args.steps / max(k1_n, 1),
                "flops_per_launch": flops_k1(cfg) * args.steps / max(k1_n, 1),
                "timing": "CUDA events around each launch on the launching stream, collected from an untimed "
                          "pass over the same calls (the timed steps carry no per-kernel brackets)"}
    j, kk = j_and_k_summary(cfg, kt, peak, hbm, peak_src)
    j["two_pass"] = two_pass
    out = {
        "metric": "df_get_jk_gflops_fp64", "value": value, "unit": "GFLOP/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, args), "clocks": clocks,
        "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "j": j, "k": kk,
        "step_ms": step_ms,
    }
    if step_fn is not None:
        out["config"]["launch"] = "one CUDA-graph replay per step (+ a device copy of C_occ into the captured input)"
    if world == 1:
        if args.cpu_baseline_full or (cfg.index == 4 and not args.cpu_baseline_sample):
            rows, (t, threads) = cfg.naux, oracle_full(cfg)
        else:
            rows, t, threads = size_sample(cfg, 15.0)
        out["cpu_baseline"] = {
            "value": flops_step(cfg) / cfg.naux * rows / t / 1e9, "unit": "GFLOP/s", "cores": threads,
            "kind": "oracle", "seconds": t,
            "sample": (f"all {cfg.naux} rows" if rows == cfg.naux else f"{rows} of {cfg.naux} auxiliary rows")
                      + f" of cfg {cfg.index}, J and K, one call (algorithmic flop count; the oracle does the "
                        "full-square work)"}
        if cfg.index == 4 and not args.no_others and step_fn is None:
            try:
                out["other"] = other_workloads(pkg, wl, args, dev, local, barrier, peak, hbm, peak_src)
            except Exception as e:                     # the headline line must survive
                out["other"] = {"error": repr(e)}
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def run_extra(args, cfg):
    """--op build_b | pair | dm | diag | scf: the section-8f rows, timed alone with CUDA events (one JSON
    line, same keys as the main line where they apply; no cpu_baseline / e2e legs)."""
    import torch
    import paper_2506_06661_b200 as pkg
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    pkg.lib()
    peak = fp64_peak(pkg)["peak"]
    B = torch.empty(cfg.naux, cfg.npair, dtype=torch.float64, device=dev)
    gi.fill_B_device(cfg, B)
    nao, naux, nocc = cfg.nao, cfg.naux, cfg.nocc[0]
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    sampler = ClockSampler(0)
    if args.op == "scf":
        # SCF driver: max_iter fixed iterations of (get_jk + Fock + DIIS + Dsygvd); B scaled so that
        # the two-electron term is a perturbation of the gapped synthetic core Hamiltonian
        B.mul_(0.02)
        h = pkg.DFJK(B, nao)
        hc = torch.from_numpy(gi.core_hamiltonian(cfg)).to(dev)
        S = torch.from_numpy(gi.overlap(cfg)).to(dev)
        iters = 6
        flops = iters * flops_step(cfg)
        what = f"dfjk_scf_rhf: {iters} SCF iterations (get_jk + Fock + DIIS + Dsygvd), flops = get_jk only"
        res = {}
        prep = lambda: None

        def run():
            res.update(h.scf_rhf(hc, S, nocc, max_iter=iters, conv_tol=1e-300))
    elif args.op == "build_b":
        Mh = torch.from_numpy(gi.metric(cfg)).pin_memory()
        Md = torch.empty(naux, naux, dtype=torch.float64, device=dev)
        flops = float(naux) ** 2 * cfg.npair + float(naux) ** 3 / 3.0
        what = "dfjk_build_b: Cholesky of the metric + in-place whitening (Eq. 2-3)"

        def prep():
            Md.copy_(Mh, non_blocking=True)
            gi.fill_B_device(cfg, B)                 # R is overwritten in place: regenerate it

        def run():
            pkg.build_b(Md, B, nao)
    else:
        h = pkg.DFJK(B, nao)
        rng = np.random.default_rng(cfg.seed)
        if args.op == "pair":
            C1 = torch.from_numpy(rng.standard_normal((nao, nocc))).to(dev)
            C2 = torch.from_numpy(rng.standard_normal((nao, nocc))).to(dev)
            flops = flops_j(cfg) + 2.0 * naux * nao ** 2 * (2 * nocc) + 2.0 * naux * nao ** 2 * nocc
            what = f"dfjk_get_jk_pair, ncol={nocc}: J[C1 C2^T] + K = sum_P (B_P C1)(B_P C2)^T"
            run = lambda: h.get_jk_pair(C1, C2)
        elif args.op == "pairs":
            nbp, ncp = 8, 8
            A = [torch.from_numpy(rng.standard_normal((nao, ncp))).to(dev) for _ in range(nbp)]
            Bf = [torch.from_numpy(rng.standard_normal((nao, ncp))).to(dev) for _ in range(nbp)]
            flops = nbp * (flops_j(cfg) + 2.0 * naux * nao ** 2 * (2 * ncp) + 2.0 * naux * nao ** 2 * ncp)
            what = f"dfjk_get_jk_pairs: {nbp} pairs of ncol {ncp} from one sweep over B (one K1 per X chunk, one J2 pass)"
            run = lambda: h.get_jk_pairs(A, Bf)
        elif args.op == "dm":
            dm = torch.from_numpy(rng.standard_normal((nao, nao))).to(dev)
            flops = flops_j(cfg) + 2.0 * naux * nao ** 3 + 2.0 * naux * nao ** 3
            what = "dfjk_get_jk_dm: J[dm], K[dm] = sum_P B_P dm B_P for a raw nao x nao dm"
            run = lambda: h.get_jk_dm(dm)
        else:
            flops = 2.0 * naux * cfg.npair
            what = "dfjk_get_df_diag: sum_P B_Pmn^2 (Eq. 7), one pass over B"
            run = lambda: h.get_df_diag()
        prep = lambda: None
    for _ in range(max(args.warmup, 1)):
        prep(); run()
    torch.cuda.synchronize()
    sampler.start()
    for k in range(args.steps):
        prep()
        ev[k][0].record()
        run()
        ev[k][1].record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = [a.elapsed_time(b) for a, b in ev]
    t = float(np.median(ms))                      # median: one-second steps see the odd outlier
    out = {"metric": f"df_{args.op}_gflops_fp64", "value": flops / (t * 1e-3) / 1e9, "unit": "GFLOP/s",
           "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": t,
           "higher_is_better": True, "dtype": "f64", "data": "synthetic", "op": what,
           "config": workload_config(cfg, args), "clocks": clocks, "step_ms": ms,
           "algorithmic_flops": flops}
    if args.op == "scf":
        out["e_hist"] = res.get("e_hist")
        out["ms_per_iteration"] = t / 6
        out["split_ms_per_iteration"] = res.get("timing")
    if args.op == "diag":
        out["gbs"] = cfg.b_bytes / (t * 1e-3) / 1e9
    else:
        out["frac_fp64_peak"] = flops / (t * 1e-3) / 1e12 / peak
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=sorted(gi.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--graph", action="store_true",
                    help="replay one captured CUDA graph per step (restricted configs; no per-kernel timing)")
    ap.add_argument("--no-others", action="store_true",
                    help="skip the short passes over the other configs / section-8f ops after the cfg-4 headline")
    ap.add_argument("--cpu-baseline-full", action="store_true",
                    help="time the oracle on ALL rows of the config instead of a ~15 s sample (the default at cfg 4: ~40 s)")
    ap.add_argument("--cpu-baseline-sample", action="store_true",
                    help="cfg 4: time the oracle on a ~15 s row sample instead of all 5000 rows")
    ap.add_argument("--op", default="get_jk", choices=["get_jk", "build_b", "pair", "pairs", "dm", "diag", "scf"],
                    help="get_jk (default, the contract line) or one of the section-8f rows")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: warning: fewer than 3 warm-up steps", file=sys.stderr)
    cfg = gi.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    elif args.op != "get_jk":
        run_extra(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
