#!/usr/bin/env python
"""bench.py — one JSON line for the fragment-projected DF-MP2 hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config3] [--impl reference]

A "step" is one pass of the whole hot path (A1-A7: AO->MO transform of every aux row, fused pair kernel,
projector/trace reduction) over one synthetic workload of BASELINE.json:
    config3 (default, the headline)  one cluster o=120 v=1080 nao=1200 naux=4800, packed (P|mu nu) 27.7 GB
    config1                          one cluster o=30 v=270 nao=300 naux=1200
    config2                          96 clusters through sie_dfmp2_batch (clusters/s)
    config4:<k>                      sweep point k in 0..3 (o=64, v=256/512/1024/2048)
    custom:o,v,naux                  one cluster of that shape (nao=o+v): short slices for ncu captures
`value` is algorithmic FP64 TFLOP/s (minimum flops of the method / device time) with the inputs resident in HBM;
`e2e` is the same metric through the C ABI with HOST (pinned) buffers, H2D/D2H inside the timed region.
N > 1 (torchrun): independent replicas, one cluster (batch) per GPU, no data-path collective ("replicas only").
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import ClusterSpec, config_specs, make_cluster  # noqa: E402

METRIC = "DF-MP2 cluster energy: FP64 TFLOP/s (algorithmic) & % of FP64 peak; clusters/s (batched)"
UNIT = "TFLOP/s"
# dram__bytes_read.sum + dram__bytes_write.sum of ONE pair_kernel launch, from the committed ncu --set full
# captures under profiles/ (file named beside each number); None = not captured for that workload.
NCU_PAIR_TRAFFIC_BYTES = {
    "config3": 529.222e9 + 85.369e9,              # profiles/r01_ncu_pair_rev3_config3.md
}


# ------------------------------------------------------------------------------------------------ flop model
def alg_flops(s: ClusterSpec) -> dict:
    """Minimum FP64 flops of the method for one cluster (SURVEY.md §8(d) 'Algorithmic work per cluster')."""
    o, v, nao, naux = s.nocc, s.nvir, s.nao, s.naux
    f = {
        "A1": 2.0 * naux * nao * nao * o,
        "A2": 2.0 * naux * nao * o * v,
        "A3_pair_syrk": 1.0 * o * o * v * (v + 1) * naux,
        "A5_G": 2.0 * o ** 3 * v * v,
    }
    f["pair_kernel"] = f["A3_pair_syrk"] + f["A5_G"]
    f["total"] = f["A1"] + f["A2"] + f["pair_kernel"]
    return f


def exec_pair_flops(s: ClusterSpec, info: dict) -> float:
    """Flops the pair kernel issues on the tensor pipe: TM x TN SYRK tiles (TM = ceil8(ta*nocc)) over ceil(naux/8)
    K-blocks, plus the G update (two DMMA passes of ceil8(o) x ceil8(o) x ceil4(o) per unordered virtual pair)."""
    kblocks = (s.naux + 7) // 8
    main = 2.0 * info["TM"] * info["TN"] * 8 * kblocks * info["ntiles"]
    o8, v = info["o8"], s.nvir
    o4 = (s.nocc + 3) // 4 * 4
    epi = 2.0 * o8 * o8 * o4 * (v * (v + 1))
    return main + epi


def workload_specs(name: str, rank: int):
    """Cluster list of one replica. Replica r > 0 draws its own clusters (cluster_id shifted by 1000 r)."""
    if name.startswith("custom:"):  # profiling slices, e.g. custom:120,216,4800 = a 1/5-virtuals slice of config 3
        o, v, naux = (int(x) for x in name.split(":")[1].split(",")[:3])
        specs = [ClusterSpec(9, 0, o + v, o, v, naux, max(1, o // 2))]
    elif name.startswith("config4"):
        k = int(name.split(":")[1]) if ":" in name else 2
        specs = [config_specs(4)[2 * k]]
    else:
        cid = int(name.replace("config", ""))
        specs = config_specs(cid)
        if cid == 1:
            specs = specs[:1]
    return [s.with_(cluster_id=s.cluster_id + 1000 * rank) for s in specs]


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()

    def summary(self) -> dict:
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])), mx.append(float(f[1])), pw.append(float(f[2]))
            except ValueError:
                continue
            for n, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_min_mhz": min(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------ CPU oracle arm
def oracle_sample(spec: ClusterSpec, n_aux_rows: int = 96, n_j: int = 16, v_sub: int = 256, seed: int = 7):
    """Time the oracle (oracle/dfmp2_oracle.c, as it stands) on a bounded sample of `spec` and extrapolate.

    Sample: (a) O1-O3 for the first `n_aux_rows` aux rows at the full nao/nocc/nvir; (b) O4-O7 for j in [0, n_j),
    all i, the first `v_sub` virtuals (a, b), the FULL aux length, on a B sample drawn N(0, 1/nao) like the real B
    (the real B would need the full O1-O3 pass, hours of long-double loops).  Extrapolation: transform time x
    naux/n_aux_rows; pair time x (nocc/n_j) x (nvir/v_sub)^2 (both loops have equal work per slice).
    Returns (seconds for the whole workload, extrapolated; seconds actually spent; description).
    """
    import oracle  # test infrastructure: allowed here (cpu_baseline / --impl reference legs only)

    x = make_cluster(spec)
    o, v, naux = spec.nocc, spec.nvir, spec.naux
    n_aux_rows = min(n_aux_rows, naux)
    n_j = min(n_j, o)
    v_sub = min(v_sub, v)
    Lb = x.L_block(0, n_aux_rows)
    Bt = np.zeros((o, v, n_aux_rows))
    t0 = time.perf_counter()
    oracle.transform_block(x.C_occ, x.C_vir, Lb, 0, n_aux_rows, Bt)
    t_tr = time.perf_counter() - t0
    rng = np.random.default_rng(seed)
    Bs = rng.standard_normal((o, v_sub, naux)) * spec.nao ** -0.5
    t0 = time.perf_counter()
    G = oracle.pair_G(Bs, x.e_occ, x.e_vir[:v_sub].copy(), 0, n_j)
    oracle.trace(x.P_frag, G)
    t_pair = time.perf_counter() - t0
    total = t_tr * (naux / n_aux_rows) + t_pair * (o / n_j) * (v / v_sub) ** 2
    desc = (f"O1-O3 on aux rows [0,{n_aux_rows}) of {naux}; O4-O7 for j in [0,{n_j}) of {o}, virtuals [0,{v_sub}) of {v}, "
            f"full aux length, B sample ~N(0,1/nao); extrapolated by slice counts")
    return total, t_tr + t_pair, desc


def oracle_workload_seconds(specs, budget_per_cluster=None):
    """Extrapolated oracle seconds for a list of clusters (a batch is sampled on its largest cluster)."""
    import oracle

    big = max(specs, key=lambda s: alg_flops(s)["total"])
    small = alg_flops(big)["total"] < 5e9
    if small:  # tiny cluster: run all of it
        n_rows, n_j, v_sub = big.naux, big.nocc, big.nvir
    else:
        n_rows, n_j, v_sub = 96, 16, min(big.nvir, 256)  # ~15 s of CPU work on 16 cores at config 3
    tot, spent, desc = oracle_sample(big, n_rows, n_j, v_sub)
    rate = alg_flops(big)["total"] / tot  # algorithmic flop/s of the oracle
    secs = sum(alg_flops(s)["total"] for s in specs) / rate
    if len(specs) > 1:
        desc = f"largest of {len(specs)} clusters (o={big.nocc}): " + desc + "; other clusters scaled by algorithmic flops"
    return secs, spent, desc, oracle.threads()


def run_reference(args) -> None:
    """--impl reference: the CPU oracle on the same config / metric / unit (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    specs = workload_specs(args.workload, 0)
    flops = sum(alg_flops(s)["total"] for s in specs)
    for _ in range(args.warmup):
        oracle_workload_seconds(specs)
    times, spent, desc, cores = [], 0.0, "", 0
    for _ in range(args.steps):
        secs, sp, desc, cores = oracle_workload_seconds(specs)
        times.append(secs)
        spent += sp
    sec = sum(times) / len(times)
    val = flops / sec * 1e-12
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": workload_config(args.workload, specs, "n/a (CPU)"),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "extrapolated_s_per_step": sec, "measured_s_per_step": spent / max(1, args.steps)},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "note": "ms_per_step is the oracle's time for the WHOLE workload extrapolated from the timed sample",
    }
    print(json.dumps(line))


def workload_config(name: str, specs, l2_note: str) -> dict:
    s = specs[0]
    cfg = {"workload": name, "clusters": len(specs), "l2": l2_note}
    if len(specs) == 1:
        cfg.update({"nocc": s.nocc, "nvir": s.nvir, "nao": s.nao, "naux": s.naux, "P_frag_rank": s.rank})
    else:
        cfg.update({"nocc_range": [min(x.nocc for x in specs), max(x.nocc for x in specs)], "nvir": "8*nocc", "naux": "36*nocc"})
    cfg["inputs"] = "seeded synthetic (workloads/gen.py): C = QR(Gaussian), packed (P|mu nu) ~ N(0, var 1/nao), e_occ~U[-1.5,-0.3], e_vir~U[0.1,3.0], P=QQ^T"
    return cfg


# ------------------------------------------------------------------------------------------------ multi-process plumbing
def reduce_over_ranks(ms: float, units: float, world: int, device) -> tuple:
    """Replicas only: no data-path collective.  The only exchange is this bookkeeping one after the
    timed region: job time = MAX over ranks of the device time, job work = SUM over ranks of the units processed."""
    if world <= 1:
        return ms, units
    import torch
    import torch.distributed as dist

    t = torch.tensor([ms], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t[0]), float(u[0])


# ------------------------------------------------------------------------------------------------ GPU arm
def run_gpu(args) -> None:
    import torch
    import torch.distributed as dist

    import paper_2412_18553_b200 as sie  # raises if libsie_dfmp2.so is missing: there is no fallback

    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU path. Use --impl reference for the CPU oracle.")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    specs = workload_specs(args.workload, rank)
    single = len(specs) == 1
    ncpu = max(1, min(32, (os.cpu_count() or 8) // max(1, world)))

    # ---- seeded inputs: generated once on the host, straight into pinned buffers (the e2e source), then uploaded
    t_gen = time.perf_counter()
    host, devc = [], []
    for s in specs:
        x = make_cluster(s)
        L = torch.empty((s.naux, s.npair), dtype=torch.float64, pin_memory=True)
        x.L_block(0, s.naux, out=L.numpy(), threads=ncpu)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()  # noqa: E731
        h = dict(nao=s.nao, nocc=s.nocc, nvir=s.nvir, naux=s.naux, C_occ=pin(x.C_occ), C_vir=pin(x.C_vir), L_packed=L,
                 e_occ=pin(x.e_occ), e_vir=pin(x.e_vir), P_frag=None if s.rank <= 0 else pin(x.P_frag))
        host.append(h)
        devc.append({k: (t.to(dev, non_blocking=True) if isinstance(t, torch.Tensor) else t) for k, t in h.items()})
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t_gen
    in_bytes = sum(sum(t.numel() * 8 for t in h.values() if isinstance(t, torch.Tensor)) for h in host)
    out_bytes = sum(8 + s.nocc * s.nocc * 8 for s in specs)

    PROF = sie.SIE_FLAG_PROFILE

    def make_step(data, flags):
        """Returns (step(), results(), timing()) for the device-resident (flags=PROF) or host-I/O arm."""
        hostio = bool(flags & sie.SIE_FLAG_HOST_IO)
        mk = (lambda *sh: torch.zeros(*sh, dtype=torch.float64).pin_memory()) if hostio else (lambda *sh: torch.zeros(*sh, dtype=torch.float64, device=dev))
        outs = [(mk(1), mk(s.nocc, s.nocc)) for s in specs]
        acc = {"ms": {k: 0.0 for k in sie.binding.STAGES}, "launch_groups": {k: 0 for k in sie.binding.STAGES}}

        def add(t):
            for k in acc["ms"]:
                acc["ms"][k] += t["ms"][k]
                acc["launch_groups"][k] += t["launch_groups"][k]

        if single:
            s, d = specs[0], data[0]
            plan0, nbytes = sie.sie_dfmp2_plan(s.nao, s.nocc, s.nvir, s.naux, 0, flags)
            info = sie.sie_dfmp2_plan_info(plan0)
            sie.sie_dfmp2_destroy(plan0)
            ws = sie.alloc_workspace(nbytes, dev)
            pending = []

            def step():
                plan, _ = sie.sie_dfmp2_plan(s.nao, s.nocc, s.nvir, s.naux, 0, flags)
                sie.sie_dfmp2_transform(plan, ws, d["C_occ"], d["C_vir"], d["L_packed"], 0, s.naux, host=hostio)
                sie.sie_dfmp2_energy(plan, ws, d["e_occ"], d["e_vir"], d["P_frag"], outs[0][0], outs[0][1], host=hostio)
                pending.append(plan)

            def timing():
                for plan in pending:
                    add(sie.sie_dfmp2_plan_timing(plan))
                    sie.sie_dfmp2_destroy(plan)
                pending.clear()
                return acc
        else:
            cl = [dict(d, E_out=o_[0], G_out=o_[1]) for d, o_ in zip(data, outs)]
            nbytes = sie.sie_dfmp2_batch_query(cl, flags)
            ws = sie.alloc_workspace(nbytes, dev)
            info = {}

            def step():
                sie.sie_dfmp2_batch(cl, ws, flags)
                if not hostio:
                    torch.cuda.current_stream().synchronize()  # the batch profile is per call: read it before the next one
                add(sie.sie_dfmp2_batch_timing())

            def timing():
                return acc

        def results():
            torch.cuda.synchronize()
            return [float(e[0]) for e, _ in outs]

        return step, results, timing, info, nbytes

    def timed(step, timing, warmup, steps, sampler_index):
        for _ in range(warmup):
            step()
        barrier()
        timing()  # drop the warm-up spans
        for k in timing()["ms"]:
            timing()["ms"][k] = 0.0
            timing()["launch_groups"][k] = 0
        l0 = sie.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(sampler_index) as cs:
            ev0.record()
            for _ in range(steps):
                step()
            ev1.record()
            barrier()
        ms, _ = reduce_over_ranks(ev0.elapsed_time(ev1), 0.0, world, dev)
        return ms / steps, sie.launch_count() - l0, cs.summary()

    phys_index = local
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            phys_index = int(vis.split(",")[local])
        except (ValueError, IndexError):
            pass

    # ---- arm 1: inputs resident in HBM
    step, results, timing, info, ws_bytes = make_step(devc, PROF)
    ms_step, launches, clocks = timed(step, timing, args.warmup, args.steps, phys_index)
    stage = timing()
    E_dev = results()
    del step, results, timing
    torch.cuda.empty_cache()

    # ---- FP64 peak probes (live denominators): DMMA, DFMA, smem-fed DMMA
    probes = {}
    for kind, name in ((0, "dmma_reg"), (1, "dfma_reg"), (2, "dmma_smem")):
        best = 0.0
        for _ in range(3):
            tf, _ms = sie.sie_dfmp2_probe_fp64(kind, 40000 if kind != 2 else 10000, 2 if kind != 2 else 1)
            best = max(best, tf)
        probes[name] = best

    # ---- NEXT-1 (optional): occupied MP2 1-RDM block on the same transformed B, same fused kernel in amplitude mode
    next1 = None
    if args.rdm and single:
        s0, d0 = specs[0], devc[0]
        plan, nb = sie.sie_dfmp2_plan(s0.nao, s0.nocc, s0.nvir, s0.naux, 0, 0)
        ws1 = sie.alloc_workspace(nb, dev)
        sie.sie_dfmp2_transform(plan, ws1, d0["C_occ"], d0["C_vir"], d0["L_packed"], 0, s0.naux)
        gam = torch.zeros(s0.nocc, s0.nocc, dtype=torch.float64, device=dev)
        tr = torch.zeros(1, dtype=torch.float64, device=dev)
        for _ in range(max(1, min(args.warmup, 2))):
            sie.sie_dfmp2_rdm_occ(plan, ws1, d0["e_occ"], d0["e_vir"], gam, tr)
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = max(1, min(args.steps, 3))
        ev0.record()
        for _ in range(reps):
            sie.sie_dfmp2_rdm_occ(plan, ws1, d0["e_occ"], d0["e_vir"], gam, tr)
        ev1.record()
        torch.cuda.synchronize()
        ms_rdm = ev0.elapsed_time(ev1) / reps
        f_rdm = alg_flops(s0)["pair_kernel"]  # same contraction count: SYRK of B plus two o^3 products per virtual pair
        next1 = {"call": "sie_dfmp2_rdm_occ", "ms": ms_rdm, "tflops": f_rdm / (ms_rdm * 1e-3) * 1e-12,
                 "trace_gamma": float(tr.cpu()[0]), "algorithmic_flops": f_rdm, "includes": "pair kernel (amplitude mode) + reduce"}
        sie.sie_dfmp2_destroy(plan)
        del ws1, gam
        torch.cuda.empty_cache()

    # ---- arm 2: end to end through the C ABI with host buffers (H2D of every input + D2H of E, G inside the timed region)
    e2e = None
    if not args.no_e2e:
        step, results, timing, _, _ = make_step(host, PROF | sie.SIE_FLAG_HOST_IO)
        e_warm, e_steps = min(args.warmup, 1), max(1, min(args.steps, 3))
        ms_e2e, _, _ = timed(step, timing, e_warm, e_steps, phys_index)
        E_host = results()
        e2e_stage = timing()
        del step, results, timing
        torch.cuda.empty_cache()

    # ---- roofline of the dominant kernel (pair_kernel): algorithmic flops per launch / mean launch duration
    f_tot = sum(alg_flops(s)["total"] for s in specs)
    _, f_job = reduce_over_ranks(0.0, f_tot, world, dev)        # units all ranks processed
    _, n_job = reduce_over_ranks(0.0, float(len(specs)), world, dev)
    f_pair = sum(alg_flops(s)["pair_kernel"] for s in specs)
    n_pair = max(1, stage["launch_groups"]["pair"])
    pair_ms = stage["ms"]["pair"] / n_pair
    achieved = f_pair / (pair_ms * 1e-3) * 1e-12 if pair_ms > 0 else 0.0
    peak_probe = max(probes["dmma_reg"], probes["dfma_reg"])
    peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
    peak_rule, rule_src = None, None
    if os.path.exists(peaks_file):
        with open(peaks_file) as fh:
            mp = json.load(fh)
        # rule of the task: another dtype's measured peak x the guide's nominal ratio (FP64 tensor 45 : bf16 2250 TFLOP/s)
        peak_rule = float(mp.get("bf16_tflops_sustained", mp.get("bf16_tflops", 0.0))) * 45.0 / 2250.0
        rule_src = "MEASURED_PEAKS.json bf16_tflops_sustained x 45/2250 (guide's nominal FP64:bf16 tensor ratio)"
    sm_mhz = clocks.get("sm_mhz") or 0.0
    roofline = {
        "kernel": "pair_kernel", "bound": "tensor", "achieved": achieved, "peak": peak_probe, "unit": "TFLOP/s",
        "frac": achieved / peak_probe if peak_probe else None,
        "peak_source": "live sie_dfmp2_probe_fp64: register-resident mma.sync.m8n8k4.f64 / DFMA issue-rate loop on all SMs "
                       "(MEASURED_PEAKS.json has no FP64 entry); the larger of the two",
        "probes_tflops": probes,
        "peak_rule": peak_rule, "peak_rule_source": rule_src,
        "peak_nominal_at_clock": 148 * 128 * sm_mhz * 1e6 * 1e-12 if sm_mhz else None,  # 64 DFMA/clk/SM x 2 flop
        "launches": n_pair, "ms_per_launch": pair_ms,
        "algorithmic_flops_per_launch": f_pair,
        "traffic": NCU_PAIR_TRAFFIC_BYTES.get(args.workload),
    }
    if single:
        fx = exec_pair_flops(specs[0], info)
        roofline["executed"] = fx / (pair_ms * 1e-3) * 1e-12 if pair_ms > 0 else None
        roofline["executed_frac"] = roofline["executed"] / peak_probe if peak_probe and roofline["executed"] else None
    # transform stage (A1+A2, incl. unpack): both fractions, SURVEY.md §8(d)
    tr_ms = (stage["ms"]["unpack"] + stage["ms"]["A1_gemm"] + stage["ms"]["A2_gemm"] + stage["ms"]["coeff_transpose"]) / max(1, args.steps)
    f_tr = sum(alg_flops(s)["A1"] + alg_flops(s)["A2"] for s in specs)
    b_tr = sum(8.0 * s.naux * s.npair + 8.0 * s.nocc * s.nvir * s.naux for s in specs)
    hbm_peak = None
    if os.path.exists(peaks_file):
        hbm_peak = float(mp.get("hbm_gbs", 0.0)) or None
    transform = {
        "ms_per_step": tr_ms, "tflops": f_tr / (tr_ms * 1e-3) * 1e-12 if tr_ms > 0 else None,
        "algorithmic_gbs": b_tr / (tr_ms * 1e-3) * 1e-9 if tr_ms > 0 else None, "hbm_peak_gbs": hbm_peak,
        "frac_hbm": (b_tr / (tr_ms * 1e-3) * 1e-9 / hbm_peak) if (tr_ms > 0 and hbm_peak) else None,
        "frac_fp64": (f_tr / (tr_ms * 1e-3) * 1e-12 / peak_probe) if (tr_ms > 0 and peak_probe) else None,
    }

    # ---- CPU oracle beside it (rank 0, N = 1 only): bounded sample, extrapolated
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        secs, spent, desc, cores = oracle_workload_seconds(specs)
        cpu = {"value": f_tot / secs * 1e-12, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
               "extrapolated_s_per_step": secs, "measured_s": spent}

    if rank == 0:
        value = f_job / (ms_step * 1e-3) * 1e-12
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(args.workload, specs, "inputs larger than L2 (no flush needed)" if in_bytes > (126 << 20) else "inputs smaller than L2; L2 not flushed"),
            "clusters_per_s": n_job / (ms_step * 1e-3),
            "E_frag": E_dev if len(E_dev) <= 4 else E_dev[:4],
            "stage_ms_per_step": {k: v / max(1, args.steps) for k, v in stage["ms"].items()},
            "roofline": roofline, "transform": transform, "cpu_baseline": cpu, "clocks": clocks, "gpu_launches": launches,
            "workspace_bytes": ws_bytes, "input_gen_s": t_gen,
        }
        if next1 is not None:
            next1["frac_of_fp64_peak"] = next1["tflops"] / peak_probe if peak_probe else None
            line["next1_rdm_occ"] = next1
        if e2e is None and not args.no_e2e:
            e2e = {"value": f_job / (ms_e2e * 1e-3) * 1e-12, "unit": UNIT, "ms_per_step": ms_e2e,
                   "h2d_bytes_per_step": in_bytes, "d2h_bytes_per_step": out_bytes, "steps": e_steps,
                   "h2d_gbs": in_bytes / (ms_e2e * 1e-3) * 1e-9,
                   "same_result_as_device_arm": bool(all(abs(a - b) <= 1e-12 * abs(a) for a, b in zip(E_dev, E_host)))}
        line["e2e"] = e2e
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------ streamed sweep point
def run_streamed(args) -> None:
    """One cluster whose packed (P|mu nu) does not fit in HBM beside B (config 4, v = 2048: 150.8 GB): the aux blocks
    are generated on the host, uploaded and fed to sie_dfmp2_transform one after the other, then
    sie_dfmp2_energy runs on the resident B.  Not a bench line: the reported time is the SUM of the library's
    event-bracketed device times (inputs are never resident all at once), one pass, no e2e arm."""
    import torch

    import paper_2412_18553_b200 as sie

    torch.cuda.set_device(0)
    spec = workload_specs(args.workload, 0)[0]
    x = make_cluster(spec)
    blk = max(8, min(spec.naux, int(args.stream_gb * 1e9) // (8 * spec.npair)) // 8 * 8)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731
    plan, nbytes = sie.sie_dfmp2_plan(spec.nao, spec.nocc, spec.nvir, spec.naux, 0, sie.SIE_FLAG_PROFILE)
    info = sie.sie_dfmp2_plan_info(plan)
    ws = sie.alloc_workspace(nbytes, "cuda")
    C_occ, C_vir = cu(x.C_occ), cu(x.C_vir)
    pinned = torch.empty((blk, spec.npair), dtype=torch.float64, pin_memory=True)
    Ld = torch.empty((blk, spec.npair), dtype=torch.float64, device="cuda")
    ncpu = max(1, min(32, os.cpu_count() or 8))
    l0 = sie.launch_count()
    with ClockSampler(0) as cs:
        for p0 in range(0, spec.naux, blk):
            p1 = min(spec.naux, p0 + blk)
            x.L_block(p0, p1, out=pinned.numpy()[: p1 - p0], threads=ncpu)
            torch.cuda.synchronize()  # the previous transform is done with Ld
            Ld[: p1 - p0].copy_(pinned[: p1 - p0], non_blocking=True)
            torch.cuda.synchronize()  # ... and the copy with the pinned buffer before the next block is generated into it
            sie.sie_dfmp2_transform(plan, ws, C_occ, C_vir, Ld[: p1 - p0], p0, p1)
        E = torch.zeros(1, dtype=torch.float64, device="cuda")
        G = torch.zeros(spec.nocc, spec.nocc, dtype=torch.float64, device="cuda")
        sie.sie_dfmp2_energy(plan, ws, cu(x.e_occ), cu(x.e_vir), None if spec.rank <= 0 else cu(x.P_frag), E, G)
        torch.cuda.synchronize()
    stage = sie.sie_dfmp2_plan_timing(plan)
    sie.sie_dfmp2_destroy(plan)
    launches = sie.launch_count() - l0
    peak = max(max(sie.sie_dfmp2_probe_fp64(k, 40000, 2)[0] for _ in range(3)) for k in (0, 1))
    f = alg_flops(spec)
    ms = sum(stage["ms"].values())
    pair_ms = stage["ms"]["pair"]
    tr_ms = ms - pair_ms - stage["ms"]["reduce"]
    line = {
        "metric": METRIC, "value": f["total"] / (ms * 1e-3) * 1e-12, "unit": UNIT, "n_gpus": 1, "steps": 1, "warmup": 0,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": dict(workload_config(args.workload, [spec], "inputs larger than L2"), inputs_resident=False,
                       aux_block_rows=blk, note="sum of event-bracketed device times; aux blocks streamed from the host"),
        "clusters_per_s": 1.0 / (ms * 1e-3), "E_frag": [float(E.cpu()[0])],
        "stage_ms_per_step": stage["ms"],
        "roofline": {"kernel": "pair_kernel", "bound": "tensor", "achieved": f["pair_kernel"] / (pair_ms * 1e-3) * 1e-12, "peak": peak,
                     "unit": "TFLOP/s", "frac": f["pair_kernel"] / (pair_ms * 1e-3) * 1e-12 / peak, "traffic": None,
                     "executed": exec_pair_flops(spec, info) / (pair_ms * 1e-3) * 1e-12},
        "transform": {"ms_per_step": tr_ms, "tflops": (f["A1"] + f["A2"]) / (tr_ms * 1e-3) * 1e-12,
                      "frac_fp64": (f["A1"] + f["A2"]) / (tr_ms * 1e-3) * 1e-12 / peak},
        "cpu_baseline": None, "clocks": cs.summary(), "gpu_launches": launches, "workspace_bytes": nbytes, "e2e": None,
    }
    print(json.dumps(line))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="config3")
    ap.add_argument("--impl", default="sie", choices=["sie", "reference"])
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end arm")
    ap.add_argument("--no-cpu", action="store_true", help="skip the CPU oracle leg")
    ap.add_argument("--rdm", action="store_true", help="also time sie_dfmp2_rdm_occ (NEXT-1: occupied MP2 1-RDM block) on the same B")
    ap.add_argument("--streamed", action="store_true", help="feed the packed integrals in aux blocks generated on the fly "
                                                             "(sweep points that do not fit in HBM; not a bench line)")
    ap.add_argument("--stream-gb", type=float, default=8.0, help="size of one streamed aux block in GB")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.streamed:
        run_streamed(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
