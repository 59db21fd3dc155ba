#!/usr/bin/env python
"""bench.py -- throughput of the D_w hot path on seeded synthetic fields.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c3] [--impl reference] [--no-solve]

Headline (BASELINE.json `metric`): algorithmic GB/s of one fp32 D_w apply (row a4) on BASELINE config 3
(64x32^3 QCD+QED with C* boundaries = 64x64x32x32 extended sites).  One "step" = one D_w apply on the packed
device layout; `value` = 768 B/site x V / time.  The same JSON line carries the fp64/fp32/fp16 sweep for D_w and
D-hat, BLAS-1 streams, the mixed-precision solves, the end-to-end number through the host-pointer C-ABI call,
the roofline object for the dominant kernel and the oracle timed on the host cores.

Multi-GPU (torchrun): the path shards by right-hand side -- every rank holds the (replicated) gauge field and
applies D_w to its own spinor; there is no data-path collective (weak scaling).  Only timing uses
torch.distributed (barrier, max over ranks).

`--impl reference` times the fp64 CPU oracle (oracle/, test infrastructure) on a bounded slab of the same
workload on the host cores; it is the base contract's reference arm for this tier.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE = 1824                    # 1320 hopping + 504 clover
REALS_DW = 192                          # psi 24 + 4 links x 18 + clover 72 + out 24 (row a4, 18-real links)
REALS_DHAT = 276                        # both passes, per FULL-lattice site (row a5)
PREC_NAME = {0: "fp64", 1: "fp32", 2: "fp16"}
PREC_BYTES = {0: 8, 1: 4, 2: 2}
FALLBACK_HBM_GBS = 6650.0               # /opt/skills/guides/B200_PROFILING.md fallback
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the headline kernel, from committed `ncu --set full` captures,
# keyed by what the capture was taken on: (config, storage precision, stored reals per link, layout).  Any other
# combination reports "traffic": null (a capture of another lattice says nothing about this one).
NCU_TRAFFIC = {
    ("c3", 1, 18, "extended"): (3663867392, "profiles/r2e_dw_sweep_vs_tile_c3.md"),   # 3.256693 GB read + 0.407175 GB write (tile kernel, final tree)
}


def ncu_traffic(config, prec, link_reals, layout):
    t = NCU_TRAFFIC.get((config, prec, link_reals, layout))
    return (t[0], t[1]) if t else (None, None)


def config_object(cfg, V):
    """The `config` object of the JSON line: identical in the CUDA arm and in the reference arm."""
    fp32_ws_gb = V * (24 + 72 + 72 + 24) * 4 / 1e9
    return {"workload": cfg["label"], "sites_per_gpu": V, "layout": "even-odd tiled SoA, 16-byte chunks, 18-real links",
            "l2": f"inputs larger than L2 (fp32 working set {fp32_ws_gb:.1f} GB vs 126 MB), no flush",
            "sharding": "by right-hand side, replicated gauge field"}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def dw_bytes_per_site(prec, link_reals=18):
    """Algorithmic bytes of one D_w site: psi 24 + 4 links x link_reals (18, or 14 = 12-real reconstruct + det) + clover 72 + out 24."""
    b = (REALS_DW - 72 + 4 * link_reals) * PREC_BYTES[prec]
    if prec == 2:
        b += 8                          # fp32 block-float scale, read with psi and written with out
    return b


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", str(self.index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1]))
                mx.append(float(c[2]))
                pw.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        pw.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm),
                "power_w": pw[len(pw) // 2] if pw else None}


def make_fields(cfg, rank):
    import synth
    U = synth.su3_links(cfg["dims"], cfg["eps"], 1)
    A = synth.u1_field(cfg["dims"], 0.3, 2) if cfg["qed"] else None
    from paper_2502_02490_b200 import sharding
    eta = synth.gaussian_spinor(cfg["dims_ext"], sharding.rhs_seed(rank))   # each rank: its own right-hand side (global index = rank)
    return U, A, eta


# ---------------------------------------------------------------------------------------------------------
# reference arm: the oracle, as it stands, on the host cores
# ---------------------------------------------------------------------------------------------------------
def oracle_sample(cfg, U, A, psi, steps, warmup, budget_s=25.0):
    """Times oracle D_w applies on a slab (leading time slices, natural order) of the workload.
    Returns (sites_per_s, cores, sample description, seconds per step)."""
    from oracle import qxd_ref as R
    ref = R.Ref(*cfg["dims"], cfg["bc"])
    ref.gauge_load(U, A, cfg["qel"])
    ref.set_quark(cfg["kappa"], cfg["q"])
    T, X1, L2, L3 = cfg["dims_ext"]
    slice_sites = X1 * L2 * L3
    nslices = max(1, min(T, (1 << 18) // slice_sites))    # ~262k sites per step (~0.5 s on 8 cores)
    n = nslices * slice_sites
    ref.clover_build_range(cfg["csw"], cfg["csw_qed"], 0, n)
    import numpy as np
    out = np.empty((n, 4, 3), dtype=np.complex128)
    for _ in range(warmup):
        ref.apply_Dw_range(psi, out)
    times = []
    t_start = time.perf_counter()
    for _ in range(steps):
        t0 = time.perf_counter()
        ref.apply_Dw_range(psi, out)
        times.append(time.perf_counter() - t0)
        if time.perf_counter() - t_start > budget_s and len(times) >= 3:
            break
    dt = sum(times) / len(times)
    desc = (f"oracle qxd_ref_apply_Dw_range on the first {nslices} time slices ({n} of {ref.V} sites) of {cfg['name']}, "
            f"{len(times)} applies, fp64, OpenMP over sites")
    return n / dt, R.num_threads(), desc, dt, len(times)


def oracle_solve_baseline(cfg, U, A, eta, oref, solves):
    """BASELINE.md §4 / SURVEY.md §8(d) "Oracle timing": the oracle's own even-odd CGNE (fp64, as it stands), timed in full on
    config c2 and for 10 iterations on the benchmarked configuration, the latter EXTRAPOLATED to the iteration count of the
    GPU's fp64/fp32 CGNE (iteration counts of CG on the same system agree to a few per cent between precisions)."""
    import synth
    from oracle import qxd_ref as R
    out = {"cores": R.num_threads(), "kind": "oracle"}
    c2 = synth.config("c2")
    r2 = R.Ref(*c2["dims"], c2["bc"])
    r2.gauge_load(synth.su3_links(c2["dims"], c2["eps"], 1), synth.u1_field(c2["dims"], 0.3, 2) if c2["qed"] else None, c2["qel"])
    r2.set_quark(c2["kappa"], c2["q"])
    r2.clover_build(c2["csw"], c2["csw_qed"])
    e2 = synth.gaussian_spinor(c2["dims_ext"], 3)
    t0 = time.perf_counter()
    _, info = r2.solve(e2, c2["tol"])
    out["c2_full_solve"] = {"seconds": time.perf_counter() - t0, "iters": info["iters"], "relres": info["relres"], "status": info["status"],
                            "tol": c2["tol"], "sites": r2.V}
    del r2, e2
    if oref is not None and cfg["name"] != "c2":
        t0 = time.perf_counter()
        _, info = oref.solve(eta, cfg["tol"], maxiter=10)
        dt = time.perf_counter() - t0
        ref_it = (solves.get("cgne_fp64_fp32") or {}).get("iters")
        out[cfg["name"] + "_10_iterations"] = {"seconds": dt, "iters": info["iters"], "sites": oref.V,
                                               "note": "includes source preparation and reconstruction (3 dslash-like passes)"}
        if ref_it:
            out[cfg["name"] + "_extrapolated_solve"] = {"seconds": dt / max(info["iters"], 1) * ref_it, "iters_assumed": ref_it,
                                                        "note": "EXTRAPOLATION: seconds per oracle iteration x iterations of the GPU fp64/fp32 CGNE"}
    return out


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    U, A, psi = make_fields(cfg, 0)
    rate, cores, desc, dt, done = oracle_sample(cfg, U, A, psi, args.steps, args.warmup, budget_s=150.0)
    gbs = rate * dw_bytes_per_site(1) / 1e9
    line = {
        "impl": "reference", "metric": "Dw_apply_fp32_GBps", "value": gbs, "unit": "GB/s", "n_gpus": args.gpus, "steps": done,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": config_object(cfg, psi.size // 12),
        "note": "sites/s of the fp64 oracle on the host cores x 768 B/site (the fp32 algorithmic bytes of the CUDA arm)",
        "gflops": rate * FLOP_PER_SITE / 1e9,
        "cpu_baseline": {"value": gbs, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": gbs, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------
# CUDA arm
# ---------------------------------------------------------------------------------------------------------
def run_cuda(args, cfg):
    import numpy as np
    import torch
    import synth as synth_mod
    from paper_2502_02490_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the qxd hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    from paper_2502_02490_b200 import sharding

    def max_over_ranks(x):
        return sharding.max_over_ranks(x, dist, dev)

    t_setup = time.perf_counter()
    U, A, eta = make_fields(cfg, rank)
    precs = (B.QXD_F64, B.QXD_F32, B.QXD_F16)
    g = B.Qxd(*cfg["dims"], cfg["bc"], precisions=precs, nrhs=max(1, args.nrhs), device=f"cuda:{local}", pairing=False)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def timed(fn, n):
        """n calls between two events on the library's stream (torch's current stream); ms per call."""
        e0, e1 = ev(), ev()
        torch.cuda.synchronize(dev)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        e1.synchronize()
        return e0.elapsed_time(e1) / n

    e0, e1, e2, e3 = ev(), ev(), ev(), ev()
    Ud = torch.from_numpy(U).to(dev)
    Ad = torch.from_numpy(A).to(dev) if A is not None else None
    e0.record()
    g.gauge_load(Ud, Ad, cfg["qel"])                   # row a2
    e1.record()
    g.set_quark(cfg["kappa"], cfg["q"])                # hop links in 3 precisions
    e2.record()
    g.clover_build(cfg["csw"], cfg["csw_qed"])         # row a3
    e3.record()
    torch.cuda.synchronize(dev)
    setup_ms = {"gauge_load": e0.elapsed_time(e1), "set_quark_hoplinks_x3": e1.elapsed_time(e2), "clover_build_invert": e2.elapsed_time(e3)}
    del Ud, Ad
    V = g.V
    eta_d = torch.from_numpy(eta).to(dev)
    packed = {p: (g.spinor_pack(eta_d, p), g.new_packed(p)) for p in precs}
    setup_s = time.perf_counter() - t_setup

    # ---- headline: K fp32 D_w applies, barrier + synchronize on both sides, max over ranks ---------------
    hp = B.QXD_F32
    pin, pout = packed[hp]
    if args.dw_sweep:
        g.set_dw_sweep(args.dw_sweep)     # experiment: the time-sweep kernel for the headline apply
    step = lambda: g.apply_Dw_packed(pin, pout, hp)
    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = g.launch_count()
    e0, e1 = ev(), ev()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    e1.synchronize()
    barrier()
    launches = g.launch_count() - l0
    ms_step = max_over_ranks(e0.elapsed_time(e1) / args.steps)
    sites_per_s = world * V / (ms_step * 1e-3)
    value = sites_per_s * dw_bytes_per_site(hp) / 1e9
    peak, peak_src = measured_peak()
    per_gpu_gbs = value / world

    # ---- sustained: the same apply kept running for >= args.sustain_s seconds whatever --steps says (a solver runs for
    # 0.3 s, not 11 ms): events every 100 applies, median of the per-100 intervals, clocks sampled over this window only
    sustained = None
    if args.sustain_s > 0:
        s2 = ClockSampler(local)
        nblk = max(3, int(args.sustain_s * 1e3 / (100 * ms_step)) + 1)
        evs = [ev() for _ in range(nblk + 1)]
        torch.cuda.synchronize(dev)
        s2.start()
        evs[0].record()
        for b in range(nblk):
            for _ in range(100):
                step()
            evs[b + 1].record()
        evs[-1].synchronize()
        ck = s2.stop()
        per100 = sorted(evs[b].elapsed_time(evs[b + 1]) / 100 for b in range(nblk))
        ms_med = max_over_ranks(per100[len(per100) // 2])
        gbs = V * dw_bytes_per_site(hp) / (ms_med * 1e-3) / 1e9
        sustained = {"applies": 100 * nblk, "seconds": evs[0].elapsed_time(evs[-1]) * 1e-3, "ms_per_step_median": ms_med,
                     "ms_per_step_min": per100[0], "ms_per_step_max": per100[-1], "value": gbs * world, "unit": "GB/s",
                     "frac": gbs / peak, "frac_of_nominal_8000": gbs / 8000.0, "clocks": ck}
    g.set_dw_sweep(0)
    # the headline sampler ran through the --steps region and the sustained window of the same kernel (a 100 ms nvidia-smi
    # cadence cannot resolve a --steps region of a few ms by itself)
    clocks = sampler.stop()

    # ---- sweep: D_w and D-hat in the three storage precisions, BLAS streams (rank-local numbers) ----------
    # link formats: 18 stored reals (full) and 14 (12-real reconstruct + det W, qxd_set_gauge_reconstruct)
    sweep = {}
    nrep = max(10, min(args.steps, 50))
    for nl, tag in ((18, ""), (14, "_recon12")):
        if args.no_sweep or args.only_multi:
            break
        g.set_gauge_reconstruct(B.QXD_RECON_12 if nl == 14 else B.QXD_RECON_NONE)
        for p in precs:
            a, b = packed[p]
            for _ in range(3):
                g.apply_Dw_packed(a, b, p)
            ms = timed(lambda: g.apply_Dw_packed(a, b, p), nrep)
            hb = g.packed_spinor_bytes(p, half_only=True)
            for _ in range(3):
                g.apply_Dhat_packed(a[:hb], b[:hb], p)
            ms_hat = timed(lambda: g.apply_Dhat_packed(a[:hb], b[:hb], p), nrep)
            bytes_dw = dw_bytes_per_site(p, nl) * V
            # D-hat, both passes, per full-lattice site: 276 reals with 18-real links, 8 x (18 - nl) fewer per even site
            bytes_hat = (REALS_DHAT - 4 * (18 - nl)) * PREC_BYTES[p] * V + (16 * V // 2 if p == 2 else 0)
            e = {"link_reals": nl, "Dw_ms": ms, "Dw_GBps": bytes_dw / ms / 1e6, "Dw_Gflops": FLOP_PER_SITE * V / ms / 1e6,
                 "Dw_frac_of_peak": bytes_dw / ms / 1e6 / peak, "Dhat_ms": ms_hat, "Dhat_GBps": bytes_hat / ms_hat / 1e6,
                 "Dhat_Gflops": FLOP_PER_SITE * V / ms_hat / 1e6}
            if nl == 18:
                ms_axpy = timed(lambda: g.blas_axpy(1e-3, a[:hb], b[:hb], p), nrep)
                e["axpy_GBps"] = 3 * 24 * PREC_BYTES[p] * (V // 2) / ms_axpy / 1e6
            sweep[PREC_NAME[p] + tag] = e
    g.set_gauge_reconstruct(B.QXD_RECON_NONE)

    # ---- multi-RHS D_w (row a10): links and clover blocks read once for a batch of right-hand sides --------
    multi = {}
    if args.nrhs > 1 and (not args.no_sweep or args.only_multi):
        n = args.nrhs
        for p in (B.QXD_F32, B.QXD_F16):
            nb = g.packed_spinor_bytes(p)
            pin = packed[p][0].repeat(n)
            pout = torch.empty_like(pin)
            for _ in range(2):
                g.apply_Dw_multi_packed(pin, pout, p, n)
            ms = timed(lambda: g.apply_Dw_multi_packed(pin, pout, p, n), max(3, nrep // 5))
            reals = 48 + 144.0 / n
            multi[PREC_NAME[p]] = {"nrhs": n, "ms_per_rhs": ms / n, "GBps": reals * PREC_BYTES[p] * V * n / ms / 1e6,
                                   "Gflops": FLOP_PER_SITE * V * n / ms / 1e6, "speedup_vs_single": (sweep[PREC_NAME[p]]["Dw_ms"] * n / ms) if PREC_NAME[p] in sweep else None}
            if n % 4 == 0:      # experimental layout: right-hand sides across lanes (csrc/dslash_ilv.cu)
                qin = torch.empty_like(pin)
                g.multi_interleave(pin, qin, p, n, True)
                for _ in range(2):
                    g.apply_Dw_multi_interleaved(qin, pout, p, n)
                ms_i = timed(lambda: g.apply_Dw_multi_interleaved(qin, pout, p, n), max(3, nrep // 5))
                multi[PREC_NAME[p]]["ms_per_rhs_interleaved"] = ms_i / n
                del qin
            del pin, pout

    # ---- end to end through the host-pointer C-ABI call (H2D + pack + apply + unpack + D2H every step) ------
    eh = torch.from_numpy(eta).pin_memory()
    oh = torch.empty_like(eh).pin_memory()
    n_e2e = 0 if args.no_e2e else 3
    g.apply_Dw_host(eh, oh, hp)
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        g.apply_Dw_host(eh, oh, hp)
    torch.cuda.synchronize(dev)
    barrier()
    e2e_s = max_over_ranks((time.perf_counter() - t0) / max(n_e2e, 1))
    e2e_val = None if args.no_e2e else world * V * dw_bytes_per_site(hp) / e2e_s / 1e9
    io_bytes = V * 24 * 8

    # ---- C*-paired device layout (qxd_set_cstar_pairing): links and clover once per physical site, a site and its mirror
    # image in neighbouring threads.  A different scheme with fewer algorithmic bytes (D_w 120 / 112 reals per site instead
    # of 192 / 176; D-hat 168 / 152 per full-lattice site instead of 276 / 244), reported beside the headline scheme and
    # used for the solves below.
    pairing = cfg["cstar"] > 0 and not args.no_pairing
    if pairing:
        g.close()
        del packed
        torch.cuda.empty_cache()
        g = B.Qxd(*cfg["dims"], cfg["bc"], precisions=precs, nrhs=max(1, args.nrhs), device=f"cuda:{local}", pairing=True)
        Ud = torch.from_numpy(U).to(dev)
        Ad = torch.from_numpy(A).to(dev) if A is not None else None
        g.gauge_load(Ud, Ad, cfg["qel"])
        g.set_quark(cfg["kappa"], cfg["q"])
        ep0, ep1 = ev(), ev()
        ep0.record()
        g.clover_build(cfg["csw"], cfg["csw_qed"])
        ep1.record()
        torch.cuda.synchronize(dev)
        setup_ms["clover_build_invert_paired"] = ep0.elapsed_time(ep1)
        del Ud, Ad
        for nl, tag in ((18, "_paired"), (14, "_paired_recon12")):
            if args.no_sweep or args.only_multi:
                break
            g.set_gauge_reconstruct(B.QXD_RECON_12 if nl == 14 else B.QXD_RECON_NONE)
            for p in precs:
                a, b = g.spinor_pack(eta_d, p), g.new_packed(p)
                for _ in range(3):
                    g.apply_Dw_packed(a, b, p)
                ms = timed(lambda: g.apply_Dw_packed(a, b, p), nrep)
                hb = g.packed_spinor_bytes(p, half_only=True)
                for _ in range(3):
                    g.apply_Dhat_packed(a[:hb], b[:hb], p)
                ms_hat = timed(lambda: g.apply_Dhat_packed(a[:hb], b[:hb], p), nrep)
                reals_dw = 48 + (4 * nl + 72) / 2.0                     # psi + out + half of (links + clover)
                reals_hat = (120 + (8 * nl + 72 + 8 * nl + 72) / 2.0) / 2.0   # per FULL-lattice site: 5 spinor streams + half the gauge data
                bytes_dw = reals_dw * PREC_BYTES[p] * V + (8 * V if p == 2 else 0)
                bytes_hat = reals_hat * PREC_BYTES[p] * V + (16 * V // 2 if p == 2 else 0)
                sweep[PREC_NAME[p] + tag] = {"link_reals": nl, "layout": "C*-paired", "Dw_ms": ms, "Dw_GBps": bytes_dw / ms / 1e6,
                                             "Dw_Gflops": FLOP_PER_SITE * V / ms / 1e6, "Dw_frac_of_peak": bytes_dw / ms / 1e6 / peak,
                                             "Dhat_ms": ms_hat, "Dhat_GBps": bytes_hat / ms_hat / 1e6, "Dhat_Gflops": FLOP_PER_SITE * V / ms_hat / 1e6}
                del a, b
        g.set_gauge_reconstruct(B.QXD_RECON_NONE)

    # ---- row f4: one HMC step's regeneration of the derived fields (new gauge field, same kappa/q/c_sw), lazily -------
    Ud = torch.from_numpy(U).to(dev)
    Ad = torch.from_numpy(A).to(dev) if A is not None else None
    g.set_lazy_refresh(True)

    def new_field():
        g.gauge_load(Ud, Ad, cfg["qel"])
        g.refresh()
    new_field()
    setup_ms["hmc_step_gauge_load_hoplinks_x3_clover"] = timed(new_field, 5)
    g.set_lazy_refresh(False)
    del Ud, Ad

    # ---- solves (rows a7, a8): fp64/fp16 and fp64/fp32 mixed CGNE, BiCGstab ------------------------------
    # Every solve is judged twice: by the library's own fp64 residual (true_res) and, outside the timed region, by
    # ||eta - D_ref psi|| / ||eta|| over the WHOLE lattice with the ORACLE's D_w (true_res_oracle).
    solves = {}
    oref = None
    want_oracle = rank == 0 and world == 1 and not args.no_oracle_residual and not args.no_solve

    def oracle_residual(eta_np, psi_t):
        nonlocal oref
        if not want_oracle:
            return None
        if oref is None:
            from oracle import qxd_ref as R
            oref = R.Ref(*cfg["dims"], cfg["bc"])
            oref.gauge_load(U, A, cfg["qel"])
            oref.set_quark(cfg["kappa"], cfg["q"])
            oref.clover_build(cfg["csw"], cfg["csw_qed"])
        r = eta_np.reshape(-1) - oref.apply_Dw(psi_t.cpu().numpy()).reshape(-1)
        return float(np.linalg.norm(r) / np.linalg.norm(eta_np.reshape(-1)))

    e2e_solve = None
    if not args.no_solve:
        # link format per storage precision as measured best: 14 reals (12-real reconstruct) where the dslash is bandwidth
        # bound (fp64, fp32), 18 reals in fp16 (issue bound)
        g.set_gauge_reconstruct(B.QXD_RECON_12)
        g.set_gauge_reconstruct(B.QXD_RECON_NONE, prec=B.QXD_F16)
        psi_d = torch.empty_like(eta_d)
        runs = [("cgne_fp64_fp16", B.QXD_CGNE, B.QXD_F16, cfg["tol"]), ("cgne_fp64_fp32", B.QXD_CGNE, B.QXD_F32, cfg["tol"]),
                ("bicgstab_fp64_fp32", B.QXD_BICGSTAB, B.QXD_F32, cfg["tol"]), ("bicgstab_fp64_fp16", B.QXD_BICGSTAB, B.QXD_F16, cfg["tol"])]
        if cfg["tol"] > 1e-12:   # the paper's own target for all solves, beside BASELINE.json's 1e-10
            runs += [("cgne_fp64_fp16_tol1e-12", B.QXD_CGNE, B.QXD_F16, 1e-12), ("cgne_fp64_fp32_tol1e-12", B.QXD_CGNE, B.QXD_F32, 1e-12)]
        for name, algo, sl, tol in runs:
            l0 = g.launch_count()
            _, info = g.solve(eta_d, tol, algo=algo, sloppy=sl, delta=0.1, maxiter=args.maxiter, psi=psi_d)
            info["launches"] = g.launch_count() - l0
            info["tol"] = tol
            info["links"] = "fp64/fp32: recon12, fp16: 18 reals"
            info["layout"] = "C*-paired" if pairing else "extended lattice"
            info["true_res_oracle"] = oracle_residual(eta, psi_d)
            solves[name] = info
        # end to end through the host-pointer call (the invertQuda boundary of PAPER.md:73-79): pinned eta in, pinned psi out
        if not args.no_e2e:
            ph = torch.empty_like(eh).pin_memory()
            t0 = time.perf_counter()
            _, info = g.solve_host(eh, ph, cfg["tol"], algo=B.QXD_CGNE, sloppy=B.QXD_F16, delta=0.1, maxiter=args.maxiter)
            e2e_solve = {"seconds": time.perf_counter() - t0, "call": "qxd_solve_host (pinned host fp64 eta in, psi out), fp64/fp16 CGNE",
                         "tol": cfg["tol"], "iters": info["iters"], "status": info["status"], "true_res": info["true_res"],
                         "seconds_device_part": info["seconds"], "h2d_bytes": io_bytes, "d2h_bytes": io_bytes,
                         "true_res_oracle": oracle_residual(eta, ph)}
            del ph
        del psi_d
        if args.nrhs > 1:
            etas = torch.empty((args.nrhs,) + tuple(eta_d.shape), dtype=eta_d.dtype, device=dev)
            etas[0].copy_(eta_d)
            for k in range(1, args.nrhs):
                etas[k].copy_(torch.from_numpy(synth_mod.gaussian_spinor(cfg["dims_ext"], 40 + k)))
            psis = torch.empty_like(etas) if torch.cuda.mem_get_info(dev)[0] > 1.2 * etas.numel() * 16 else None
            for sl, tag, links in ((B.QXD_F32, "fp32", "recon12"), (B.QXD_F16, "fp16", "fp64: recon12, fp16: 18 reals")):
                if psis is None and tag == "fp16":
                    break            # in-place solve (no room for a second batch of spinors): the sources are gone after the first run
                l0 = g.launch_count()
                t0 = time.perf_counter()
                out, infos = g.solve_multi(etas, cfg["tol"], sloppy=sl, delta=0.1, maxiter=args.maxiter, psi=psis if psis is not None else etas)
                torch.cuda.synchronize(dev)
                dt = time.perf_counter() - t0
                kk = args.nrhs - 1
                eta_k = eta if kk == 0 else synth_mod.gaussian_spinor(cfg["dims_ext"], 40 + kk)
                solves[f"cgne_multi{args.nrhs}_fp64_{tag}"] = {
                    "status": max(abs(i["status"]) for i in infos), "iters_max": max(i["iters"] for i in infos),
                    "true_res_max": max(i["true_res"] for i in infos), "seconds": dt, "seconds_per_rhs": dt / args.nrhs,
                    "launches": g.launch_count() - l0, "tol": cfg["tol"], "links": links,
                    "true_res_oracle_last_rhs": oracle_residual(eta_k, out.reshape(etas.shape)[kk])}
            del etas, psis
        g.set_gauge_reconstruct(B.QXD_RECON_NONE)

    # ---- row f3: SAP-preconditioned GCR on the full-lattice D_w (the solver family the paper measures), in a
    # context of its own (the Krylov space is part of the workspace): library default layout, link formats as above
    if not args.no_solve and args.gcr_nkv > 0:
        g.close()
        packed = None                     # the packed sweep spinors of the first context are not needed any more
        torch.cuda.empty_cache()
        gp = (args.gcr_nkv, args.gcr_ncy, args.gcr_nmr)
        dp = (args.dfl_ns, args.dfl_ninv, args.dfl_nkc) if args.dfl_ns > 0 else None
        # the Krylov space and the deflation space are part of the workspace: take the largest number of null vectors that
        # leaves room for the test vectors of the setup (the largest lattices run with fewer, or without the second level)
        g = None
        for ns_try in ([n for n in (dp[0], 16, 8) if n <= dp[0]] if dp else []) + [0]:
            dtry = (ns_try, dp[1], dp[2], 0, args.dfl_chiral) if (dp and ns_try > 0) else None
            try:
                g = B.Qxd(*cfg["dims"], cfg["bc"], precisions=precs, nrhs=1, device=f"cuda:{local}", pairing=(True if pairing else None), gcr=gp, deflation=dtry)
                free = torch.cuda.mem_get_info(dev)[0]
                need = g.packed_spinor_bytes(B.QXD_F32) * ns_try + 5 * g.packed_spinor_bytes(B.QXD_F64)
                if free >= need:
                    break
                g.close()
                g = None
                torch.cuda.empty_cache()
            except torch.OutOfMemoryError:
                g = None
                torch.cuda.empty_cache()
        if dp is not None and (dtry is None or dtry[0] != dp[0]):
            solves["dfl_gcr_sap_fp64_fp16_note"] = f"device memory: {dp[0]} null vectors requested, {ns_try} used"
        dp = dtry
        Ud = torch.from_numpy(U).to(dev)
        Ad = torch.from_numpy(A).to(dev) if A is not None else None
        g.gauge_load(Ud, Ad, cfg["qel"])
        g.set_quark(cfg["kappa"], cfg["q"])
        g.clover_build(cfg["csw"], cfg["csw_qed"])
        del Ud, Ad
        g.set_gauge_reconstruct(B.QXD_RECON_12)
        g.set_gauge_reconstruct(B.QXD_RECON_NONE, prec=B.QXD_F16)
        psi_d = torch.empty_like(eta_d)
        pin = g.spinor_pack(eta_d, B.QXD_F32)
        pout = torch.zeros_like(pin)
        for name, sl in (("gcr_sap_fp64_fp16", B.QXD_F16), ("gcr_sap_fp64_fp32", B.QXD_F32)):
            g.apply_sap(pin, pout, sl)
            sap_ms = timed(lambda: g.apply_sap(pin, pout, sl), 10)
            g.solve(eta_d, cfg["tol"], algo=B.QXD_GCR, sloppy=sl, maxiter=args.maxiter, psi=psi_d)     # warm-up (function attributes, clocks)
            l0 = g.launch_count()
            _, info = g.solve(eta_d, cfg["tol"], algo=B.QXD_GCR, sloppy=sl, maxiter=args.maxiter, psi=psi_d)
            info.update({"launches": g.launch_count() - l0, "tol": cfg["tol"], "nkv": gp[0], "ncy": gp[1], "nmr": gp[2],
                         "sap_ms_per_application": sap_ms, "sap_ms_per_half_step": sap_ms / (2 * gp[1]),
                         "layout": "C*-paired" if pairing else "extended lattice", "block": "128-index tile, both parities (256 sites)",
                         "true_res_oracle": oracle_residual(eta, psi_d)})
            solves[name] = info
        if dp is not None:   # second level: local-coherence deflation (setup per gauge field and quark, timed separately)
            nbv = g.packed_spinor_bytes(B.QXD_F32)
            rnd = torch.empty(dp[0] * nbv, dtype=torch.uint8, device=dev)
            for i in range(dp[0]):
                g.spinor_pack(torch.from_numpy(synth_mod.gaussian_spinor(cfg["dims_ext"], 100 + i)).to(dev), B.QXD_F32, packed=rnd[i * nbv:(i + 1) * nbv])
            t0 = ev(); t1 = ev()
            g.deflation_setup(rnd, B.QXD_F16)
            t0.record()
            g.deflation_setup(rnd, B.QXD_F16)
            t1.record()
            t1.synchronize()
            g.solve(eta_d, cfg["tol"], algo=B.QXD_DFL_GCR, sloppy=B.QXD_F16, maxiter=args.maxiter, psi=psi_d)
            _, info = g.solve(eta_d, cfg["tol"], algo=B.QXD_DFL_GCR, sloppy=B.QXD_F16, maxiter=args.maxiter, psi=psi_d)
            info.update({"tol": cfg["tol"], "nkv": gp[0], "ncy": gp[1], "nmr": gp[2], "ns": dp[0], "ninv": dp[1], "nkc": dp[2], "chirality_split": dp[4],
                         "setup_seconds": t0.elapsed_time(t1) * 1e-3, "layout": "C*-paired" if pairing else "extended lattice",
                         "true_res_oracle": oracle_residual(eta, psi_d)})
            solves["dfl_gcr_sap_fp64_fp16"] = info
            # ---- the regime the second level is for: the same lattice, couplings and U(1) field with SU(3)
            # links that have long-range order (synth.su3_links_smooth), just below the critical hopping parameter
            nck = args.nc_kappa if args.nc_kappa is not None else (0.1238 if cfg["name"] == "c3" else 0.0)
            if nck > 0:
                Us = synth_mod.su3_links_smooth(cfg["dims"], 0.7, 1, 4)
                Ud = torch.from_numpy(Us).to(dev)
                Ad = torch.from_numpy(A).to(dev) if A is not None else None
                g.gauge_load(Ud, Ad, cfg["qel"])
                g.set_quark(nck, cfg["q"])
                g.clover_build(cfg["csw"], cfg["csw_qed"])
                del Ud, Ad
                g.set_gauge_reconstruct(B.QXD_RECON_12)
                g.set_gauge_reconstruct(B.QXD_RECON_NONE, prec=B.QXD_F16)
                oref2 = None
                if want_oracle:
                    from oracle import qxd_ref as R
                    oref2 = R.Ref(*cfg["dims"], cfg["bc"])
                    oref2.gauge_load(Us, A, cfg["qel"])
                    oref2.set_quark(nck, cfg["q"])
                    oref2.clover_build(cfg["csw"], cfg["csw_qed"])
                nc = {"workload": f"{cfg['name']} geometry, couplings and U(1) field; SU(3) links = synth.su3_links_smooth(eps 0.7, every 4 sites); kappa {nck}",
                      "tol": cfg["tol"], "maxiter": 3000}
                # here the inverse-iteration refinement of the deflation space pays (it does not on the white-noise links: DESIGN.md 6a)
                refine = (args.nc_nref, args.nc_refk) if dp[0] <= 2 * (gp[0] - args.nc_refk) else (0, 1)
                g.set_deflation_refine(*refine)
                t0 = ev(); t1 = ev()
                t0.record()
                g.deflation_setup(rnd, B.QXD_F16)
                t1.record()
                t1.synchronize()
                g.set_deflation_refine(0, 1)
                for name, algo in (("cgne_fp64_fp16", B.QXD_CGNE), ("bicgstab_fp64_fp16", B.QXD_BICGSTAB), ("gcr_sap_fp64_fp16", B.QXD_GCR),
                                   ("dfl_gcr_sap_fp64_fp16", B.QXD_DFL_GCR)):
                    reps = 1 if algo == B.QXD_CGNE else 2          # CGNE runs into maxiter here (seconds): once is enough
                    for _ in range(reps):
                        _, info = g.solve(eta_d, cfg["tol"], algo=algo, sloppy=B.QXD_F16, maxiter=3000, psi=psi_d)
                    if oref2 is not None and info["status"] == 0:
                        r = eta.reshape(-1) - oref2.apply_Dw(psi_d.cpu().numpy()).reshape(-1)
                        info["true_res_oracle"] = float(np.linalg.norm(r) / np.linalg.norm(eta.reshape(-1)))
                    nc[name] = info
                nc["dfl_gcr_sap_fp64_fp16"].update({"ns": dp[0], "ninv": dp[1], "nkc": dp[2], "chirality_split": dp[4], "refinement_rounds": refine[0],
                                                    "gcr_steps_per_refinement_solve": refine[1], "setup_seconds": t0.elapsed_time(t1) * 1e-3})
                solves["near_critical"] = nc
                del oref2, Us
            del rnd
        del psi_d, pin, pout

    # ---- CPU baseline: the oracle on this box's host cores (rank 0, N = 1 only) ----------------------------
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rate, cores, desc, dt, done = oracle_sample(cfg, U, A, eta, 40, 1, budget_s=10.0)
        cpu_baseline = {"value": rate * dw_bytes_per_site(hp) / 1e9, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": desc,
                        "sites_per_s": rate, "gflops": rate * FLOP_PER_SITE / 1e9}
        if not args.no_solve:
            cpu_baseline["solve"] = oracle_solve_baseline(cfg, U, A, eta, oref, solves)

    traffic, traffic_src = ncu_traffic(cfg["name"], hp, 18, "extended")
    if rank == 0:
        line = {
            "metric": "Dw_apply_fp32_GBps", "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": config_object(cfg, V),
            "gflops": sites_per_s * FLOP_PER_SITE / 1e9,
            "roofline": {"bound": "hbm", "achieved": per_gpu_gbs, "peak": peak, "unit": "GB/s", "frac": per_gpu_gbs / peak,
                         "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src, "frac_of_nominal_8000": per_gpu_gbs / 8000.0,
                         "kernel": "dslash_k<float, DW_FULL>", "algorithmic_bytes_per_launch": dw_bytes_per_site(hp) * V},
            "e2e": {"value": e2e_val, "unit": "GB/s", "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes, "ms_per_step": e2e_s * 1e3,
                    "call": "qxd_apply_Dw_host (pinned host fp64 in/out, pipelined over time slabs)"},
            "sustained": sustained,
            "e2e_solve": e2e_solve,
            "gpu_launches": launches,
            "clocks": clocks,
            "cpu_baseline": cpu_baseline,
            "sweep": sweep,
            "multi_rhs": multi,
            "solve": solves,
            "setup_ms": setup_ms,
            "setup_s_total": setup_s,
        }
        print(json.dumps(line), flush=True)
    g.close()
    if dist is not None:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------------------
# --decomp domain: the lattice cut into time slabs over the ranks (row f2), strong scaling
# ---------------------------------------------------------------------------------------------------------
def run_domain(args, cfg):
    """One rank per GPU, the GLOBAL lattice of the config cut along time (paper_2502_02490_b200/domain.py): device-side
    projected halos, faces exchanged by NCCL while the interior slabs run, all-reduced solver scalars.  With one rank the
    ghost layers are kept and filled through a real NCCL send/recv to the rank itself, so that the N = 1 line measures the
    cost of the halo path against the plain single-GPU apply.  value = global sites x 768 B / max-over-ranks time."""
    import numpy as np
    import torch
    import torch.distributed as dist
    import synth as synth_mod
    from paper_2502_02490_b200 import binding as B, domain as D, sharding
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the qxd hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world == 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29533")
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    pg = D.ProcessGrid(cfg["dims"], (world, 1, 1, 1), cfg["cstar"])
    lat = D.LocalLattice(pg, rank, antiperiodic=bool(cfg["antiperiodic"]), force_cut=(True, False, False, False))
    U = synth_mod.su3_links(cfg["dims"], cfg["eps"], 1)
    A = synth_mod.u1_field(cfg["dims"], 0.3, 2) if cfg["qed"] else None
    comm = D.TorchComm(dist, self_via_dist=True)
    hp = B.QXD_F32
    ops = {rank: D.GpuRank(lat, U, A, cfg["qel"], cfg["kappa"], cfg["q"], cfg["csw"], cfg["csw_qed"], prec=hp, device=f"cuda:{local}")}
    op = D.GpuOperator(comm, {rank: lat}, ops, overlap=not args.no_overlap)
    eta = synth_mod.gaussian_spinor(cfg["dims_ext"], 3)
    vin = {rank: ops[rank].pack(lat.scatter(eta))}
    vout = op.alloc()
    V = int(np.prod(cfg["dims_ext"]))

    def barrier():
        dist.barrier()
        torch.cuda.synchronize(dev)
    for _ in range(args.warmup):
        op.apply_Dw(vin, vout)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = ops[rank].g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        op.apply_Dw(vin, vout)
    e1.record()
    e1.synchronize()
    barrier()
    launches = ops[rank].g.launch_count() - l0
    ms_step = sharding.max_over_ranks(e0.elapsed_time(e1) / args.steps, dist, dev)
    # keep the same apply running for another ~0.5 s so that the 100 ms nvidia-smi cadence sees the clocks under this load
    for _ in range(max(0, int(500.0 / ms_step) - args.steps)):
        op.apply_Dw(vin, vout)
    torch.cuda.synchronize(dev)
    clocks = sampler.stop()
    value = V * dw_bytes_per_site(hp) / (ms_step * 1e-3) / 1e9
    peak, peak_src = measured_peak()
    # distributed solves: fp64 even-odd CGNE and the mixed fp64/fp32 one with reliable updates (every scalar all-reduced)
    solve = None
    if not args.no_solve:
        hi = {rank: D.GpuRank(lat, U, A, cfg["qel"], cfg["kappa"], cfg["q"], cfg["csw"], cfg["csw_qed"], prec=B.QXD_F64, device=f"cuda:{local}",
                              extra_precisions=(B.QXD_F32, B.QXD_F16))}
        lo = {rank: hi[rank].with_prec(B.QXD_F32)}
        lo16 = {rank: hi[rank].with_prec(B.QXD_F16)}
        op64 = D.GpuOperator(comm, {rank: lat}, hi, overlap=not args.no_overlap)
        op32 = D.GpuOperator(comm, {rank: lat}, lo, overlap=not args.no_overlap)
        op16 = D.GpuOperator(comm, {rank: lat}, lo16, overlap=not args.no_overlap)
        src = {rank: hi[rank].pack(lat.scatter(eta))}
        solve = {}
        for name in ("cgne_fp64_fp32", "cgne_fp64", "cgne_fp64_fp32", "cgne_fp64_fp16", "cgne_fp64_fp16"):   # first pass of the mixed solves: warm-up (allocator)
            barrier()
            t0 = time.perf_counter()
            if name == "cgne_fp64":
                x, info = D.solve_distributed(op64, src, cfg["tol"], maxiter=args.maxiter)
            else:
                x, info = D.solve_distributed_mixed(op64, op32 if name == "cgne_fp64_fp32" else op16, src, cfg["tol"], delta=0.1, maxiter=args.maxiter,
                                                    op_vec=None if name == "cgne_fp64_fp32" else op32)
            barrier()
            solve[name] = {"algo": "distributed even-odd CGNE", "seconds": sharding.max_over_ranks(time.perf_counter() - t0, dist, dev), "iters": info["iters"],
                           "status": info["status"], "true_res": info["true_res_eo"], "tol": cfg["tol"], "n_reliable": info.get("n_reliable")}
        hi[rank].close()
    if rank == 0:
        face = lat.local_ext[1] * lat.local_ext[2] * lat.local_ext[3]
        line = {"metric": "Dw_apply_fp32_GBps", "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": dict(config_object(cfg, V // world), parallelism=f"time-slab domain decomposition over {world} rank(s), "
                               f"local lattice {lat.local_dims[0]} slices incl. 2 x {D.TIME_GHOST} ghost slices",
                               sharding="lattice cut along time; halo = 2 faces x 12 reals per face site per apply, NCCL, overlapped with the interior slabs"),
                "gflops": V * FLOP_PER_SITE / (ms_step * 1e-3) / 1e9,
                "roofline": {"bound": "hbm", "achieved": value / world, "peak": peak, "unit": "GB/s", "frac": value / world / peak, "traffic": None,
                             "peak_source": peak_src, "kernel": "dslash_k<float, DW_FULL> on interior + boundary time slabs",
                             "algorithmic_bytes_per_launch": dw_bytes_per_site(hp) * V // world},
                "e2e": {"value": None, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                        "note": "fields stay on the devices between applies; see the default (right-hand-side sharded) line for the host-pointer path"},
                "halo_bytes_per_step_per_rank": 2 * face * 12 * 4, "gpu_launches": launches, "clocks": clocks, "solve": solve}
        print(json.dumps(line), flush=True)
    ops[rank].close()
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", default="c3")
    ap.add_argument("--maxiter", type=int, default=20000)
    ap.add_argument("--nrhs", type=int, default=12, help="right-hand sides of the multi-RHS D_w / batched solve lines (row a10; 1 = skip)")
    ap.add_argument("--gcr-nkv", type=int, default=16, help="Krylov vectors per GCR cycle (0 = skip the SAP-GCR solves)")
    ap.add_argument("--gcr-ncy", type=int, default=4, help="SAP cycles per preconditioner application")
    ap.add_argument("--gcr-nmr", type=int, default=5, help="minimal-residual steps per SAP block solve")
    ap.add_argument("--dw-sweep", type=int, default=0, help="use the time-sweep D_w kernel with this segment length for the headline apply (0 = tile kernel)")
    ap.add_argument("--dfl-ns", type=int, default=16, help="null vectors of the deflated (two-level) GCR solve (0 = skip)")
    ap.add_argument("--dfl-chiral", type=int, default=1, help="1: null vectors split by chirality (2 ns coarse degrees of freedom per block; ns <= 16)")
    ap.add_argument("--dfl-ninv", type=int, default=8, help="M_sap smoothing passes per null vector in the deflation setup")
    ap.add_argument("--dfl-nkc", type=int, default=12, help="GCR steps of every coarse-grid solve")
    ap.add_argument("--nc-nref", type=int, default=2, help="refinement rounds of the deflation space in the near-critical comparison")
    ap.add_argument("--nc-refk", type=int, default=4, help="deflated GCR steps of every refinement solve there")
    ap.add_argument("--nc-kappa", type=float, default=None,
                    help="hopping parameter of the near-critical solver comparison on smooth links (default: 0.1238 at c3, skipped elsewhere; 0 = skip)")
    ap.add_argument("--decomp", default="rhs", choices=["rhs", "domain"], help="rhs: shard by right-hand side (weak scaling, the default); "
                    "domain: cut the lattice along time over the ranks (strong scaling, row f2)")
    ap.add_argument("--no-overlap", action="store_true", help="--decomp domain: exchange the faces before the interior slabs instead of during them")
    ap.add_argument("--no-pairing", action="store_true", help="keep the extended-lattice layout for the solves (C* configs)")
    ap.add_argument("--no-solve", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the precision sweep (short runs under ncu)")
    ap.add_argument("--only-multi", action="store_true", help="of the sweep, run only the multi-RHS D_w lines (short runs under ncu)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-pointer end-to-end loops (short runs under ncu)")
    ap.add_argument("--sustain-s", type=float, default=1.0, help="seconds of back-to-back applies for the `sustained` figure (0 = skip)")
    ap.add_argument("--no-oracle-residual", action="store_true", help="skip the oracle's whole-lattice true residual of the solves")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    import synth
    cfg = synth.config(args.config)
    cfg["name"] = args.config
    T, L1, L2, L3 = cfg["dims"]
    cfg["label"] = (f"{args.config}: {T}x{L1}x{L2}x{L3} {'QCD+QED' if cfg['qed'] else 'QCD'} Wilson-clover, cstar={cfg['cstar']} "
                    f"(extended {'x'.join(map(str, cfg['dims_ext']))}), eps={cfg['eps']}, kappa={cfg['kappa']}, csw={cfg['csw']}, "
                    f"csw_qed={cfg['csw_qed']}, q={cfg['q']:.4f}")
    if args.impl == "reference":
        run_reference(args, cfg)
    elif args.decomp == "domain":
        run_domain(args, cfg)
    else:
        run_cuda(args, cfg)


if __name__ == "__main__":
    main()
