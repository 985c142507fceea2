#!/usr/bin/env python
"""bench.py -- Gcell-updates/s of the whole FDTD step (E and H updates with CPML, air-water boundary,
source, DTFT, convergence bookkeeping) on BASELINE.json's production config (configs[3]: non-uniform
400x400x200, 5 frequencies), one JSON line on stdout.  See DESIGN.md "Measurement".

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--rd 3] [--impl reference]

A "step" is one pass of Algorithm 1 lines 9-23 over the padded grid.  `value` times K steps with all
inputs resident in HBM (CUDA events on the stream the kernels run on); `e2e` is the same metric through
emm_model_set + emm_run with host buffers.  Multi-GPU = independent replicas (one process per GPU, no
data-path collective: the method does not shard).
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2304_00233_b200 import workloads as W  # noqa: E402

METRIC = "Gcell-updates/s (E+H, fp32), whole FDTD step incl. CPML, air-water BC, source, DTFT"


def build_workload(args, nugrid):
    kw = {}
    if args.workload in ("cfg3", "cfg4", "cfg5"):
        kw = dict(rd=args.rd) if args.rd else {}
        if args.scale != 1.0:
            base = {"cfg3": (200, 120), "cfg4": (400, 200), "cfg5": (256, 160)}[args.workload]
            kw.update(nx=int(base[0] * args.scale) // 2 * 2, nz=int(base[1] * args.scale),
                      n_water=max(4, int(round(28 * args.scale))))
        if args.aux_dx:
            kw["aux_dx"] = args.aux_dx
        w = W.build(args.workload, nugrid, **kw)
        if args.nf:
            w["freqs"] = w["freqs"][: max(args.nf, 0)]       # --nf -1: pure update (no DTFT)
            if args.nf < 0:
                w["receivers"] = np.zeros((0, 3))
    else:
        w = W.build(args.workload, None, **({"rd": args.rd} if args.rd else {}))
    if args.air_route:
        w["grid"] = dict(w["grid"], air_route=args.air_route)
    return w


def describe(w, info, nsrc):
    d = {"workload": "%s: %dx%dx%d cells, rd=%d (order %d), %s, nf=%d, nsrc=%d, padded %dx%dx%d" % (
        w["name"], len(w["x"]) - 1, len(w["y"]) - 1, len(w["z"]) - 1, w["grid"]["rd"], 2 * w["grid"]["rd"],
        "non-uniform" if not info["uniform_xy"] else "uniform x-y", len(w["freqs"]), nsrc, info["N1"], info["N2"], info["N3"]),
        "padded_nodes": info["N1"] * info["N2"] * info["N3"],
        "air_plane": [info["aux_M1"], info["aux_M2"]],
        "l2": "working set (fields + DTFT accumulators) is >> the 126 MB L2; no flush needed"}
    if "air_cluster" in info:             # the CUDA library's grid (the oracle has its own plain transforms)
        d["air_boundary"] = ("none" if info["k0"] < 0 else "one launch per pass: %d-CTA cluster, plane in distributed shared memory" % info["air_cluster"]
                             if info["air_cluster"] else "library 2-D transforms" if info["uniform_xy"] else "separable route, batched 1-D library transforms")
    return d


def algorithmic_bytes(info, nf, nb, kernel, m=1):
    """E kernel reads 3 H, RMWs 3 E, reads 3 dt/eps = 48 B/node; H kernel reads 3 E, RMWs 3 H
    = 36 B/node; each RMWs 3*nf complex accumulators (48*nf B) per DTFT-box node; plus 8 B per active CPML
    memory variable (two per slab membership).  Grouped DTFT with m terms per accumulator pass:
    the closing pass of a group ("E2"/"H2") also reads m-2 earlier levels of its 3 components (12 B per box node each);
    the accumulator-free passes ("E0"/"H0") update out of place into the next buffer of the ring: no extra bytes."""
    N1, N2, N3 = info["N1"], info["N2"], info["N3"]
    N = N1 * N2 * N3
    box = ((info["box_hi1"] - info["box_lo1"] + 1) * (info["box_hi2"] - info["box_lo2"] + 1)
           * (info["box_hi3"] - info["box_lo3"] + 1))
    zs = (2 if info["k0"] < 0 else 1) * nb
    psi = 16 * (2 * nb * N2 * N3 + 2 * nb * N1 * N3 + zs * N1 * N2)
    b = (48 if kernel[0] == "E" else 36) * N + 48 * (0 if kernel[1:] == "0" else nf) * box + psi
    if kernel[1:] == "2":
        b += 12 * max(m - 2, 0) * box
    return b


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                       "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None
        time.sleep(0.3)

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.1)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.strip() == "Active":
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_rate(w_full, budget_s, steps, warmup, args):
    """Oracle (as it stands) on the host cores, on a bounded sample: the same recipe at a size chosen so that
    steps+warmup time steps take about budget_s.  Returns (Mcell/s, seconds per step list, description)."""
    from oracle import emm_oracle as O
    O.build()
    ncores = os.cpu_count() or 1
    # calibrate on a tiny instance of the same recipe
    scale = 0.12
    rate = None
    for _ in range(3):
        a2 = argparse.Namespace(**vars(args))
        a2.scale = scale
        a2.air_route = 0                  # a scheduling option of the CUDA library, not of the method
        w = build_workload(a2, O.nugrid)
        g = O.Grid(w["x"], w["y"], w["z"], **w["grid"])
        g.model_set(w["sigma_h"], w.get("sigma_v"))
        i = g.info()
        n = i["N1"] * i["N2"] * i["N3"]
        g.run_begin(w["sources"][:1], w["freqs"], w["receivers"][:4], dict(fixed_steps=10 ** 6, sparse_dft=0))
        g.run_steps(1)
        t = time.perf_counter()
        g.run_steps(2)
        dt2 = (time.perf_counter() - t) / 2
        g.close()
        rate = n / dt2
        target = min(budget_s * rate / max(steps + warmup, 1), 12e6)   # nodes of a sample that fits the budget (and ~8 GB of host RAM)
        full = None
        if args.workload not in ("cfg1", "cfg2"):
            full = (len(w_full["x"]) - 1) ** 2 * (len(w_full["z"]) - 1) * 1.35
        new_scale = min(1.0, scale * (target / n) ** (1 / 3.0)) if full else 1.0
        if args.workload in ("cfg1", "cfg2") or abs(new_scale - scale) < 0.25 * scale or new_scale <= scale:
            break
        scale = new_scale
    a2 = argparse.Namespace(**vars(args))
    a2.scale = scale
    a2.air_route = 0
    w = build_workload(a2, O.nugrid)
    g = O.Grid(w["x"], w["y"], w["z"], **w["grid"])
    g.model_set(w["sigma_h"], w.get("sigma_v"))
    i = g.info()
    n = i["N1"] * i["N2"] * i["N3"]
    g.run_begin(w["sources"][:1], w["freqs"], w["receivers"][:4], dict(fixed_steps=10 ** 6, sparse_dft=0))
    g.run_steps(warmup)
    t = time.perf_counter()
    g.run_steps(steps)
    el = time.perf_counter() - t
    # the same sample on ONE host thread (1 thread and all cores), one step is enough
    one = None
    try:
        import ctypes
        gomp = ctypes.CDLL("libgomp.so.1")
        gomp.omp_set_num_threads(1)
        t = time.perf_counter()
        g.run_steps(1)
        one = n / (time.perf_counter() - t) / 1e9
        gomp.omp_set_num_threads(ncores)
    except OSError:
        pass
    oracle_rate.one_thread = one
    g.close()
    desc = ("%s recipe at %dx%dx%d cells (padded %dx%dx%d, nf=%d, full-box DTFT), %d steps after %d warm-up, fp64, "
            "gcc -O2 -fopenmp" % (w["name"], len(w["x"]) - 1, len(w["y"]) - 1, len(w["z"]) - 1, i["N1"], i["N2"], i["N3"],
                                  len(w["freqs"]), steps, warmup))
    return n * steps / el / 1e9, el / steps * 1e3, ncores, desc


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w_full = build_workload(args, None) if args.workload in ("cfg1", "cfg2") else None
    if w_full is None:
        from oracle import emm_oracle as O
        O.build()
        w_full = build_workload(args, O.nugrid)
    val, ms, cores, desc = oracle_rate(w_full, 120.0, args.steps, args.warmup, args)
    from oracle import emm_oracle as O
    gi = O.Grid(w_full["x"], w_full["y"], w_full["z"], **w_full["grid"]).info()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "Gcell-updates/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": dict(describe(w_full, gi, 1), workload="%s; the oracle steps a bounded sample of this recipe: %s" % (describe(w_full, gi, 1)["workload"], desc)),
            "cpu_baseline": {"value": val, "unit": "Gcell-updates/s", "cores": cores, "kind": "oracle", "sample": desc,
                             "value_one_thread": getattr(oracle_rate, "one_thread", None)},
            "e2e": {"value": val, "unit": "Gcell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2304_00233_b200 import emm

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    emm.build()
    w = build_workload(args, emm.emm_nugrid)
    nsrc = len(w["sources"]) if w["run"].get("batched") else 1
    srcs = w["sources"][:nsrc]
    K, Wm = args.steps, max(args.warmup, 3)
    g = emm.Grid(w["x"], w["y"], w["z"], **w["grid"])
    g.bind(nsrc=nsrc, nfreq=len(w["freqs"]), max_steps=K + Wm + 8, nrec=len(w["receivers"]), device=dev)
    info = g.info()
    N = info["N1"] * info["N2"] * info["N3"]

    # ---- end to end through the C ABI with host buffers (model upload + run + receiver read-back) ----
    # host inputs in pinned memory (numpy views of pinned torch tensors): the library copies from whatever host pointer it gets
    def pinned(a):
        return torch.from_numpy(np.ascontiguousarray(a, np.float32)).pin_memory().numpy()
    sh = pinned(w["sigma_h"])
    sv = None if w.get("sigma_v") is None else pinned(w["sigma_v"])
    g.model_set(sh, sv)                                        # warm-up of the whole path (plans, kernels, one graph capture)
    g.run(srcs, w["freqs"], w["receivers"], dict(fixed_steps=min(K, 210), batched=1 if nsrc > 1 else 0))
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    g.model_set(sh, sv)
    out, ns = g.run(srcs, w["freqs"], w["receivers"], dict(fixed_steps=K, batched=1 if nsrc > 1 else 0))
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    assert int(ns[0]) == K and np.all(np.isfinite(out))
    h2d = sh.nbytes + (sv.nbytes if sv is not None else 0) + (K + 1) * (len(w["freqs"]) * 16 + 4 + 32)
    d2h = nsrc * len(w["freqs"]) * len(w["receivers"]) * 6 * 16      # accumulators interpolated to the receivers on the device, complex fp64
    if world > 1:
        tt = torch.tensor([t_e2e], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_e2e = float(tt.item())

    # ---- device-resident stepping: K steps timed with CUDA events on the library's stream ----
    g.run_begin(srcs, w["freqs"], w["receivers"], dict(fixed_steps=K + Wm + 4, batched=1 if nsrc > 1 else 0))
    dtft_group = int(g.get("DTFT_GROUP")[0])
    g.run_enqueue(Wm)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(g.stream)            # the library's stream (a torch stream owned by the binding)
    g.run_enqueue(K)
    e1.record(g.stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    launches = g.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    # per-kernel durations of the two update kernels: a second pass over the same state with CUDA events around
    # every launch (emm_profile); in that pass the steps run one kernel after the other (no stream overlap, no
    # CUDA graph) so that each duration is the kernel's own
    # whole DTFT groups only, so that every closing pass of the profile carries the full number of history levels (the
    # algorithmic bytes of the instance table assume the full group)
    Kp = min(K, 48)
    if dtft_group > 1:
        Kp = max(dtft_group, Kp // dtft_group * dtft_group)
    g.run_begin(srcs, w["freqs"], w["receivers"], dict(fixed_steps=Kp + Wm + 4, batched=1 if nsrc > 1 else 0))
    g.run_enqueue(Wm)
    torch.cuda.synchronize()
    g.profile(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(g.stream)
    g.run_enqueue(Kp)
    p1.record(g.stream)
    torch.cuda.synchronize()
    ms_prof = p0.elapsed_time(p1) / Kp
    prof = g.profile_read()
    g.profile(False)
    if world > 1:
        dist.barrier()
        tt = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms = float(tt.item())
    g.run_steps(1)
    for c in ("E1", "H2"):
        assert np.all(np.isfinite(g.get(c)))
    # extra: the same K steps with one DTFT term per step in every step (dtft_pair = -1: the paper's own schedule, L454)
    unpaired = None
    if 0 < len(w["freqs"]) <= 5:
        g.run_begin(srcs, w["freqs"], w["receivers"], dict(fixed_steps=K + Wm + 4, batched=1 if nsrc > 1 else 0, dtft_pair=-1))
        g.run_enqueue(Wm)
        torch.cuda.synchronize()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(g.stream)
        g.run_enqueue(K)
        d1.record(g.stream)
        torch.cuda.synchronize()
        msu = d0.elapsed_time(d1)
        unpaired = {"ms_per_step": msu / K, "value": world * nsrc * N * K / (msu * 1e-3) / 1e9,
                    "note": "dtft_pair=-1: every update kernel adds its one term of Eq. 25 in every step; same sums, twice the accumulator traffic"}
    # extra, not the headline: the same K steps with DTFT decimation at the automatic safe stride
    decim = None
    if len(w["freqs"]) > 0:
        g.run_begin(srcs, w["freqs"], w["receivers"], dict(fixed_steps=K + Wm + 4, batched=1 if nsrc > 1 else 0, dtft_every=-1))
        g.run_enqueue(Wm)
        torch.cuda.synchronize()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(g.stream)
        g.run_enqueue(K)
        d1.record(g.stream)
        torch.cuda.synchronize()
        msd = d0.elapsed_time(d1)
        fmax = 4.0 * float(np.sqrt(max(w["freqs"]) * 1.0))
        m_auto = max(1, min(1000, int(np.floor(1.0 / (g.info()["dt"] * (3.0 * fmax + 2.0 * np.sqrt(max(w["freqs"]) * 1.0)))))))
        decim = {"dtft_every": m_auto, "ms_per_step": msd / K, "value": world * nsrc * N * K / (msd * 1e-3) / 1e9,
                 "note": "only every m-th term of Eq. 25 (fields and J'); same converged step count; not the paper's every-step DTFT"}
    # extra, not the headline: receivers-only DTFT (every term of Eq. 25, but only at the receivers' stencil nodes)
    rec_only = None
    if len(w["freqs"]) > 0 and len(w["receivers"]) > 0:
        g.run_begin(srcs, w["freqs"], w["receivers"], dict(fixed_steps=K + Wm + 4, batched=1 if nsrc > 1 else 0, sparse_dft=1))
        g.run_enqueue(Wm)
        torch.cuda.synchronize()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(g.stream)
        g.run_enqueue(K)
        d1.record(g.stream)
        torch.cuda.synchronize()
        msr = d0.elapsed_time(d1)
        rec_only = {"ms_per_step": msr / K, "value": world * nsrc * N * K / (msr * 1e-3) / 1e9,
                    "note": "sparse_dft=1: same receiver outputs and step counts, no full-grid frequency-domain fields"}
    # extra: configs[3] at 4th order (rd = 2), the order north_star's target sentence names for this grid
    rd2 = None
    if w["name"] == "cfg4" and w["grid"]["rd"] == 3 and args.scale == 1.0 and not args.no_rd2:
        a2 = argparse.Namespace(**vars(args))
        a2.rd = 2
        w2 = build_workload(a2, emm.emm_nugrid)
        g.close()
        g2 = emm.Grid(w2["x"], w2["y"], w2["z"], **w2["grid"])
        g2.bind(nsrc=1, nfreq=len(w2["freqs"]), max_steps=K + Wm + 8, nrec=len(w2["receivers"]), device=dev)
        g2.model_set(w2["sigma_h"], w2.get("sigma_v"))
        i2 = g2.info()
        N2n = i2["N1"] * i2["N2"] * i2["N3"]
        g2.run_begin(w2["sources"][:1], w2["freqs"], w2["receivers"], dict(fixed_steps=K + Wm + 4))
        g2.run_enqueue(Wm)
        torch.cuda.synchronize()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(g2.stream)
        g2.run_enqueue(K)
        d1.record(g2.stream)
        torch.cuda.synchronize()
        ms2 = d0.elapsed_time(d1)
        g2.run_begin(w2["sources"][:1], w2["freqs"], w2["receivers"], dict(fixed_steps=Kp + Wm + 4))
        g2.run_enqueue(Wm)
        torch.cuda.synchronize()
        g2.profile(True)
        g2.run_enqueue(Kp)
        torch.cuda.synchronize()
        prof2 = g2.profile_read()
        g2.profile(False)
        grp2 = int(g2.get("DTFT_GROUP")[0])
        g2.close()
        nb2, nf2 = w2["grid"]["nb"], len(w2["freqs"])
        t2 = sum(v[0] for v in prof2.values())
        b2 = sum(algorithmic_bytes(i2, nf2, nb2, k, grp2) * v[1] for k, v in prof2.items() if v[1] > 0)
        rd2 = {"workload": describe(w2, i2, 1)["workload"], "ms_per_step": ms2 / K, "value": world * N2n * K / (ms2 * 1e-3) / 1e9,
               "kernels_ms_per_launch": {k: v[0] / v[1] for k, v in prof2.items() if v[1] > 0},
               "instances_gbs": {k: algorithmic_bytes(i2, nf2, nb2, k, grp2) / (v[0] / v[1] * 1e-3) / 1e9 for k, v in prof2.items() if v[1] > 0},
               "update_kernels_gbs_time_weighted": b2 / (t2 * 1e-3) / 1e9}
    batched = None
    if nsrc > 1:
        # configs[4]: the same K steps for ONE source alone = what running the sources one after the other costs
        g.run_begin(srcs[:1], w["freqs"], w["receivers"], dict(fixed_steps=K + Wm + 4))
        g.run_enqueue(Wm)
        torch.cuda.synchronize()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(g.stream)
        g.run_enqueue(K)
        s1.record(g.stream)
        torch.cuda.synchronize()
        ms1 = s0.elapsed_time(s1)
        batched = {"nsrc": nsrc, "ms_per_step_per_source_batched": ms / K / nsrc, "ms_per_step_per_source_sequential": ms1 / K,
                   "speedup_vs_sequential": (ms1 / K) / (ms / K / nsrc)}

    if rank == 0:
        value = world * nsrc * N * K / (ms * 1e-3) / 1e9
        peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
        if os.path.exists(peaks_file):
            peak, peak_src = float(json.load(open(peaks_file))["hbm_gbs"]), "of measured (MEASURED_PEAKS.json hbm_gbs)"
        else:
            peak, peak_src = 6650.0, "of fallback (B200_PROFILING.md)"
        # instances of the update kernels in this run (grouped DTFT: E0/H0 = accumulator-free steps, the TMA tile pipeline
        # k_tile; E2/H2 = the pass that closes a group).  `frac` is the time-weighted figure over ALL of them: the
        # algorithmic bytes of every timed launch over the summed launch durations; `kernel` names the instance with the
        # largest share of that time.
        avg = {k: v[0] / v[1] for k, v in prof.items() if v[1] > 0}
        mgrp = dtft_group
        inst = {"E": "k_update<R,NF,E>", "H": "k_update<R,NF,H>", "E0": "k_tile<R,E> (accumulator-free, TMA tile pipeline)",
                "H0": "k_tile<R,H> (accumulator-free, TMA tile pipeline)",
                "E2": "k_update<R,NF,E,PAIR> (closing pass of a DTFT group)", "H2": "k_update<R,NF,H,PAIR> (closing pass of a DTFT group)"}
        nfq, nbq = len(w["freqs"]), w["grid"]["nb"]
        ibytes = {k: nsrc * algorithmic_bytes(info, nfq, nbq, k, mgrp) for k in avg}
        tot_update = sum(v[0] for v in prof.values())
        tot_bytes = sum(ibytes[k] * prof[k][1] for k in avg)
        share = {k: prof[k][0] / tot_update for k in avg}
        dom = max(share, key=share.get)
        achieved = tot_bytes / (tot_update * 1e-3) / 1e9
        traffic = None
        tf = os.path.join(ROOT, "profiles", "ncu_traffic.json")
        if os.path.exists(tf):
            traffic = json.load(open(tf)).get("%s:%s:rd%d:nf%d" % (w["name"], dom, w["grid"]["rd"], len(w["freqs"])))
        roofline = {"bound": "hbm", "kernel": inst[dom], "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "peak_source": peak_src, "traffic": traffic,
                    "what": "time-weighted over every update-kernel launch of the serialised pass: sum of algorithmic bytes / sum of launch durations",
                    "algorithmic_bytes_per_launch": ibytes[dom], "kernel_ms": avg[dom],
                    "kernels_ms_per_launch": avg, "launches": {k: prof[k][1] for k in avg}, "share_of_update_time": share,
                    "instances_gbs": {k: ibytes[k] / (avg[k] * 1e-3) / 1e9 for k in avg},
                    "instances_frac": {k: ibytes[k] / (avg[k] * 1e-3) / 1e9 / peak for k in avg},
                    "dtft_group": mgrp,
                    "update_kernels_ms_per_step": tot_update / Kp,
                    "step_frac_in_update_kernels": tot_update / (ms_prof * Kp),
                    "ms_per_step_serialised": ms_prof,
                    "how": "launch durations from a serialised pass (emm_profile: CUDA events around each launch); `value` is timed with the air-water boundary overlapped on a second stream"}
        # whole step against the same peak: algorithmic bytes of the update kernels of one step (paired DTFT: half of the four
        # passes of a pair), boundary / check-set / injection bytes not counted, over the timed ms per step
        if "E2" in avg:      # a group of m steps: m-1 accumulator-free passes and one closing pass per kernel
            step_bytes = nsrc * sum((mgrp - 1) * algorithmic_bytes(info, nfq, nbq, k + "0", mgrp) + algorithmic_bytes(info, nfq, nbq, k + "2", mgrp)
                                    for k in ("E", "H")) / mgrp
        else:
            step_bytes = nsrc * (algorithmic_bytes(info, nfq, nbq, "E") + algorithmic_bytes(info, nfq, nbq, "H"))
        if rd2:
            rd2["update_kernels_frac_time_weighted"] = rd2["update_kernels_gbs_time_weighted"] / peak
        roofline["whole_step"] = {"algorithmic_bytes_per_step": step_bytes, "achieved": step_bytes / (ms / K * 1e-3) / 1e9,
                                  "frac": step_bytes / (ms / K * 1e-3) / 1e9 / peak,
                                  "note": "update-kernel bytes only, over the whole timed step (boundary, check set and injection included in the time)"}
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            v, cms, cores, desc = oracle_rate(w, 20.0, 3, 1, args)
            cpu = {"value": v, "unit": "Gcell-updates/s", "cores": cores, "kind": "oracle", "sample": desc, "ms_per_step": cms,
                   "value_one_thread": getattr(oracle_rate, "one_thread", None)}
        line = {"metric": METRIC, "value": value, "unit": "Gcell-updates/s", "n_gpus": world, "steps": K, "warmup": Wm,
                "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic", "config": describe(w, info, nsrc), "clocks": clocks,
                "e2e": {"value": world * nsrc * N * K / t_e2e / 1e9, "unit": "Gcell-updates/s", "h2d_bytes_per_step": h2d / K,
                        "d2h_bytes_per_step": d2h / K, "seconds": t_e2e,
                        "what": "emm_model_set (host sigma -> device) + emm_run(fixed_steps=K) (tables up, receivers back)"},
                "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu, "batched": batched,
                "dtft": ("every term of Eq. 25, %d consecutive terms per accumulator pass (emm_run_opts.dtft_pair, default)" % dtft_group) if dtft_group > 1 else "every term of Eq. 25, one per step",
                "dtft_one_term_per_step": unpaired, "dtft_decimation": decim, "receivers_only_dtft": rec_only, "rd2": rd2,
                "multi_gpu": "replicas only: every rank runs the whole workload, no collective on the data path"}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_converge(args):
    """--converge: time to converged (BASELINE.json metric, third part) of the chosen workload through Grid.run, wall
    clock, in the five DTFT schedules; one JSON line.  Not the driver's line (that is the default run)."""
    import torch
    from paper_2304_00233_b200 import emm
    emm.build()
    w = build_workload(args, emm.emm_nugrid)
    g = emm.Grid(w["x"], w["y"], w["z"], **w["grid"])
    g.bind(nsrc=1, nfreq=len(w["freqs"]), max_steps=60000, nrec=len(w["receivers"]), device="cuda:0")
    g.model_set(w["sigma_h"], w.get("sigma_v"))
    info = g.info()
    N = info["N1"] * info["N2"] * info["N3"]
    base = dict(w["run"])
    base.pop("batched", None)
    base["max_steps"] = 60000
    g.run(w["sources"][:1], w["freqs"], w["receivers"], dict(fixed_steps=210))     # warm-up (plans, kernels, graph capture)
    res = {}
    for mode, extra in (("grouped_default", {}), ("pairs", dict(dtft_pair=2)), ("one_term_per_step", dict(dtft_pair=-1)), ("decimated_auto", dict(dtft_every=-1)),
                        ("receivers_only", dict(sparse_dft=1))):
        torch.cuda.synchronize()
        t = time.perf_counter()
        out, ns = g.run(w["sources"][:1], w["freqs"], w["receivers"], dict(base, **extra))
        torch.cuda.synchronize()
        el = time.perf_counter() - t
        res[mode] = {"seconds": el, "steps": int(ns[0]), "gcell_updates_per_s": N * int(ns[0]) / el / 1e9,
                     "largest_receiver_amplitude": float(np.abs(out).max())}
    print(json.dumps({"metric": "time to converged", "config": describe(w, info, 1), "schedules": res}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--rd", type=int, default=0, help="override the FD half length (cfg4: 3 = 6th order as configs[3]; 2 = 4th order)")
    ap.add_argument("--nf", type=int, default=0, help="keep only the first nf frequencies; -1 = none (pure E/H update, no DTFT)")
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the cell counts (debugging only)")
    ap.add_argument("--aux-dx", type=float, default=0.0)
    ap.add_argument("--air-route", type=int, default=0, help="emm_grid_opts.air_route (1 = library / plane-sized route of the air-water boundary)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-rd2", action="store_true", help="skip the extra 4th-order (rd = 2) run of configs[3]")
    ap.add_argument("--converge", action="store_true", help="time to converged in the four DTFT schedules instead of the step benchmark")
    args = ap.parse_args()
    if args.converge:
        run_converge(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
