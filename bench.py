#!/usr/bin/env python
"""bench.py — one JSON line for the fragment-projected DF-MP2 hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config3] [--impl reference]

A "step" is one pass of the whole hot path (A1-A7: AO->MO transform of every aux row, fused pair kernel,
projector/trace reduction) over one synthetic workload of BASELINE.json:
    config3 (default, the headline)  one cluster o=120 v=1080 nao=1200 naux=4800, packed (P|mu nu) 27.7 GB
    config1                          one cluster o=30 v=270 nao=300 naux=1200
    config2                          96 clusters through sie_dfmp2_batch (clusters/s)
    config4:<k>                      sweep point k in 0..3 (o=64, v=256/512/1024/2048)
    custom:o,v,naux[,rank]           one cluster of that shape (nao=o+v): short slices for ncu captures
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
# dram__bytes_read.sum + dram__bytes_write.sum of ONE pair_kernel launch are read from this table of the committed
# ncu --set full captures (one row per workload: workload,dram_read_bytes,dram_write_bytes,capture file).
NCU_TRAFFIC_TABLE = os.path.join(ROOT, "profiles", "pair_kernel_dram_traffic.csv")


def ncu_pair_traffic(workload: str):
    """-> (bytes per launch or None, name of the profiles/ capture it comes from or None)."""
    try:
        with open(NCU_TRAFFIC_TABLE) as fh:
            rows = [ln.strip().split(",") for ln in fh if ln.strip() and not ln.startswith("#")]
    except OSError:
        return None, None
    hit = None
    for r in rows:
        if len(r) >= 4 and r[0] == workload:
            hit = r  # the last row of a workload is the newest capture
    if hit is None:
        return None, None
    return float(hit[1]) + float(hit[2]), hit[3]


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
        f = [int(x) for x in name.split(":")[1].split(",")]
        o, v, naux = f[:3]
        specs = [ClusterSpec(9, 0, o + v, o, v, naux, f[3] if len(f) > 3 else max(1, o // 2))]  # optional 4th field: projector rank
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


def oracle_workload_seconds(specs):
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
class GpuBench:
    """Everything run_gpu needs to time workloads in ONE process: device, ranks, event timing, clock sampling."""

    def __init__(self):
        import torch
        import torch.distributed as dist

        import paper_2412_18553_b200 as sie  # raises if libsie_dfmp2.so is missing: there is no fallback

        self.torch, self.dist, self.sie = torch, dist, sie
        self.rank, self.world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
        local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU path. Use --impl reference for the CPU oracle.")
        torch.cuda.set_device(local)
        self.dev = torch.device("cuda", local)
        if self.world > 1:
            dist.init_process_group("nccl", device_id=self.dev)
        self.phys_index = local
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            try:
                self.phys_index = int(vis.split(",")[local])
            except (ValueError, IndexError):
                pass
        self.ncpu = max(1, min(32, (os.cpu_count() or 8) // max(1, self.world)))
        self.peak = None
        self.probes = {}
        self.no_pipeline = False

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def probe_peak(self):
        """Live FP64 roofline denominators: register-resident DMMA / DFMA issue loops, smem-fed DMMA (best of 3)."""
        for kind, name in ((0, "dmma_reg"), (1, "dfma_reg"), (2, "dmma_smem")):
            best = 0.0
            for _ in range(3):
                tf, _ms = self.sie.sie_dfmp2_probe_fp64(kind, 40000 if kind != 2 else 10000, 2 if kind != 2 else 1)
                best = max(best, tf)
            self.probes[name] = best
        self.peak = max(self.probes["dmma_reg"], self.probes["dfma_reg"])

    # ---- inputs: generated once on the host (pinned when the e2e arm will read them), then uploaded
    def make_inputs(self, specs, pinned: bool):
        torch = self.torch
        t0 = time.perf_counter()
        host, devc = [], []
        for s in specs:
            x = make_cluster(s)
            L = torch.empty((s.naux, s.npair), dtype=torch.float64, pin_memory=pinned)
            x.L_block(0, s.naux, out=L.numpy(), threads=self.ncpu)
            wrap = (lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()) if pinned else (lambda a: torch.from_numpy(np.ascontiguousarray(a)))
            h = dict(nao=s.nao, nocc=s.nocc, nvir=s.nvir, naux=s.naux, C_occ=wrap(x.C_occ), C_vir=wrap(x.C_vir), L_packed=L,
                     e_occ=wrap(x.e_occ), e_vir=wrap(x.e_vir), P_frag=None if s.rank <= 0 else wrap(x.P_frag))
            devc.append({k: (t.to(self.dev, non_blocking=pinned) if isinstance(t, torch.Tensor) else t) for k, t in h.items()})
            host.append(h if pinned else None)
            if not pinned:
                del L, h
        torch.cuda.synchronize()
        return host, devc, time.perf_counter() - t0

    def make_step(self, specs, data, flags):
        """-> (step(), results(), timing(), plan info, workspace bytes) for the device-resident or the host-I/O arm.
        One plan (host-side object) serves every step: sie_dfmp2_plan_reset between passes."""
        sie, torch, dev = self.sie, self.torch, self.dev
        hostio = bool(flags & sie.SIE_FLAG_HOST_IO)
        mk = (lambda *sh: torch.zeros(*sh, dtype=torch.float64).pin_memory()) if hostio else (lambda *sh: torch.zeros(*sh, dtype=torch.float64, device=dev))
        outs = [(mk(1), mk(s.nocc, s.nocc)) for s in specs]
        acc = {"ms": {k: 0.0 for k in sie.binding.STAGES}, "launch_groups": {k: 0 for k in sie.binding.STAGES}}

        def add(t):
            for k in acc["ms"]:
                acc["ms"][k] += t["ms"][k]
                acc["launch_groups"][k] += t["launch_groups"][k]

        if len(specs) == 1:
            s, d = specs[0], data[0]
            plan, nbytes = sie.sie_dfmp2_plan(s.nao, s.nocc, s.nvir, s.naux, 0, flags)
            info = sie.sie_dfmp2_plan_info(plan)
            ws = sie.alloc_workspace(nbytes, dev)

            def step():
                sie.sie_dfmp2_plan_reset(plan)
                sie.sie_dfmp2_transform(plan, ws, d["C_occ"], d["C_vir"], d["L_packed"], 0, s.naux, host=hostio)
                sie.sie_dfmp2_energy(plan, ws, d["e_occ"], d["e_vir"], d["P_frag"], outs[0][0], outs[0][1], host=hostio)

            def timing():
                add(sie.sie_dfmp2_plan_timing(plan))
                return acc

            def close():
                sie.sie_dfmp2_destroy(plan)
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

            def close():
                pass

        def results():
            torch.cuda.synchronize()
            return [float(e[0]) for e, _ in outs]

        return step, results, timing, close, info, nbytes

    def timed(self, step, timing, warmup, steps, flush=None, side_streams=()):
        """flush(): finishes work a software-pipelined step() still has in flight, inside the timed region;
        side_streams: streams the steps run on (the closing event waits for them)."""
        sie, torch = self.sie, self.torch
        for _ in range(warmup):
            step()
        if flush is not None and warmup > 0:
            flush()  # the timed region starts with an empty pipeline: K transforms and K energies fall inside it
        self.barrier()
        acc = timing()  # drop the warm-up spans
        for k in acc["ms"]:
            acc["ms"][k] = 0.0
            acc["launch_groups"][k] = 0
        l0 = sie.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with ClockSampler(self.phys_index) as cs:
            ev0.record()
            for _ in range(steps):
                step()
            if flush is not None:
                flush()
            for ss in side_streams:
                torch.cuda.current_stream().wait_stream(ss)
            ev1.record()
            self.barrier()
        ms, _ = reduce_over_ranks(ev0.elapsed_time(ev1), 0.0, self.world, self.dev)
        return ms / steps, sie.launch_count() - l0, cs.summary()

    def measure(self, name, steps, warmup, want_e2e, want_rdm=False):
        """Time one workload: device-resident arm (event-timed, stage profile), optional host-I/O e2e arm with the SAME
        steps/warm-up, optional NEXT-1 call.  Returns a dict of raw measurements (this rank's; times are max over ranks)."""
        sie, torch, dev = self.sie, self.torch, self.dev
        specs = workload_specs(name, self.rank)
        host, devc, t_gen = self.make_inputs(specs, pinned=want_e2e)
        in_bytes = sum(sum(t.numel() * 8 for t in d.values() if isinstance(t, torch.Tensor)) for d in devc)
        out_bytes = sum(8 + s.nocc * s.nocc * 8 for s in specs)
        m = {"name": name, "specs": specs, "in_bytes": in_bytes, "out_bytes": out_bytes, "t_gen": t_gen, "steps": steps, "warmup": warmup}

        step, results, timing, close, info, ws_bytes = self.make_step(specs, devc, sie.SIE_FLAG_PROFILE)
        m["ms_step"], m["launches"], m["clocks"] = self.timed(step, timing, warmup, steps)
        m["stage"] = timing()
        m["E"] = results()
        m["info"], m["ws_bytes"] = info, ws_bytes
        close()
        del step, results, timing, close
        torch.cuda.empty_cache()

        m["next1"] = None
        if want_rdm and len(specs) == 1:
            # NEXT-1: both blocks of the MP2 1-RDM on the same transformed B: gamma_occ (fused kernel in amplitude mode, or
            # the general route for nocc > 128) and gamma_vir (general route), each timed as a whole call
            s0, d0 = specs[0], devc[0]
            plan, nb = sie.sie_dfmp2_plan(s0.nao, s0.nocc, s0.nvir, s0.naux, 0, sie.SIE_FLAG_RDM_VIR)
            route = sie.sie_dfmp2_plan_info(plan)["route"]
            ws1 = sie.alloc_workspace(nb, dev)
            sie.sie_dfmp2_transform(plan, ws1, d0["C_occ"], d0["C_vir"], d0["L_packed"], 0, s0.naux)
            o_, v_, x_ = s0.nocc, s0.nvir, s0.naux
            m["next1"] = {"pair_route": ("fused", "reference", "general")[route]}
            for name_, fn, n_, f_alg in (
                    ("rdm_occ", sie.sie_dfmp2_rdm_occ, o_, alg_flops(s0)["pair_kernel"]),
                    ("rdm_vir", sie.sie_dfmp2_rdm_vir, v_, 1.0 * o_ * o_ * v_ * (v_ + 1) * x_ + 2.0 * o_ * o_ * v_ ** 3)):
                gam = torch.zeros(n_, n_, dtype=torch.float64, device=dev)
                tr = torch.zeros(1, dtype=torch.float64, device=dev)
                for _ in range(max(1, min(warmup, 2))):
                    fn(plan, ws1, d0["e_occ"], d0["e_vir"], gam, tr)
                torch.cuda.synchronize()
                ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                reps = max(1, min(steps, 3))
                ev0.record()
                for _ in range(reps):
                    fn(plan, ws1, d0["e_occ"], d0["e_vir"], gam, tr)
                ev1.record()
                torch.cuda.synchronize()
                ms_ = ev0.elapsed_time(ev1) / reps
                # algorithmic flops: SYRK minimum of the pair integrals + the second-level contraction (2 o^3 v^2 for the
                # occupied block, 2 o^2 v^3 for the virtual block)
                m["next1"][name_] = {"ms": ms_, "tflops": f_alg / (ms_ * 1e-3) * 1e-12, "trace": float(tr.cpu()[0]), "algorithmic_flops": f_alg}
                del gam
            # NEXT-3: energy only, projector in factored form Q Q^T (project-first epilogue for rank <= 32), against the
            # G-path energy with P = Q Q^T on the same B
            if route == 0 and s0.rank > 0:
                Qd = torch.from_numpy(np.ascontiguousarray(make_cluster(s0).Q_frag)).to(dev)
                Pd = (Qd @ Qd.T).contiguous()
                E1 = torch.zeros(1, dtype=torch.float64, device=dev)
                G1 = torch.zeros(o_, o_, dtype=torch.float64, device=dev)
                res = {}
                for name_, call in (("energy_lowrank", lambda: sie.sie_dfmp2_energy_lowrank(plan, ws1, d0["e_occ"], d0["e_vir"], Qd, E1)),
                                    ("energy_G_path", lambda: sie.sie_dfmp2_energy(plan, ws1, d0["e_occ"], d0["e_vir"], Pd, E1, G1))):
                    for _ in range(2):
                        call()
                    torch.cuda.synchronize()
                    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    reps = max(1, min(steps, 3))
                    ev0.record()
                    for _ in range(reps):
                        call()
                    ev1.record()
                    torch.cuda.synchronize()
                    res[name_] = {"ms": ev0.elapsed_time(ev1) / reps, "E_frag": float(E1.cpu()[0])}
                m["next1"]["next3_lowrank"] = dict(res, rank=s0.rank)
            sie.sie_dfmp2_destroy(plan)
            del ws1
            torch.cuda.empty_cache()

        m["e2e"] = None
        if want_e2e:
            free_b, _ = torch.cuda.mem_get_info()
            need_b = 2 * (m["ws_bytes"] + in_bytes) + (4 << 30)  # two plans, each with whole-tensor staging
            if len(specs) == 1 and free_b + in_bytes > need_b and not self.no_pipeline:
                # Software-pipelined over steps: two plans (SIE_FLAG_STAGE_FULL) on two streams; the transform of step n+1
                # (its 27.7 GB upload at config 3) is enqueued BEFORE the energy of step n, so the integrals of the next
                # cluster travel while the pair stage of the current one runs.  Every step still uploads all its inputs from
                # pinned host memory and reads E, G back inside the timed region.
                del devc
                devc = None
                torch.cuda.empty_cache()
                s0, h0 = specs[0], host[0]
                fl = sie.SIE_FLAG_PROFILE | sie.SIE_FLAG_HOST_IO | sie.SIE_FLAG_STAGE_FULL
                plans, wss, streams, outs = [], [], [], []
                for _ in range(2):
                    pl, nb = sie.sie_dfmp2_plan(s0.nao, s0.nocc, s0.nvir, s0.naux, 0, fl)
                    plans.append(pl)
                    wss.append(sie.alloc_workspace(nb, dev))
                    streams.append(torch.cuda.Stream(device=dev))
                    outs.append((torch.zeros(1, dtype=torch.float64).pin_memory(), torch.zeros(s0.nocc, s0.nocc, dtype=torch.float64).pin_memory()))
                state = {"k": 0}
                acc = {"ms": {k: 0.0 for k in sie.binding.STAGES}, "launch_groups": {k: 0 for k in sie.binding.STAGES}}

                def energy_of(j):
                    sie.sie_dfmp2_energy(plans[j], wss[j], h0["e_occ"], h0["e_vir"], h0["P_frag"], outs[j][0], outs[j][1], host=True, stream=streams[j])

                def step():
                    k = state["k"]
                    j = k % 2
                    sie.sie_dfmp2_plan_reset(plans[j])
                    sie.sie_dfmp2_transform(plans[j], wss[j], h0["C_occ"], h0["C_vir"], h0["L_packed"], 0, s0.naux, host=True, stream=streams[j])
                    if k > 0:
                        energy_of(1 - j)  # synchronises its own stream only
                    state["k"] = k + 1

                def flush():
                    energy_of((state["k"] - 1) % 2)
                    state["k"] = 0

                def timing():
                    return acc

                ms_e2e, _, _ = self.timed(step, timing, warmup, steps, flush=flush, side_streams=streams)
                torch.cuda.synchronize()
                E_host = [float(outs[0][0][0])]
                ok2 = float(outs[1][0][0]) == float(outs[0][0][0]) if steps + warmup > 1 else True
                for pl in plans:
                    sie.sie_dfmp2_destroy(pl)
                del wss
                m["e2e"] = {"ms": ms_e2e, "E": E_host, "pipelined": True, "both_plans_agree": bool(ok2)}
            else:
                step, results, timing, close, _, _ = self.make_step(specs, host, sie.SIE_FLAG_PROFILE | sie.SIE_FLAG_HOST_IO)
                ms_e2e, _, _ = self.timed(step, timing, warmup, steps)
                E_host = results()
                close()
                del step, results, timing, close
                m["e2e"] = {"ms": ms_e2e, "E": E_host, "pipelined": False}
        del host, devc
        torch.cuda.empty_cache()
        return m

    def summarize(self, m):
        """Derived figures of one measured workload: whole-step rate, pair-kernel roofline, transform fractions."""
        specs, stage, steps = m["specs"], m["stage"], m["steps"]
        f_tot = sum(alg_flops(s)["total"] for s in specs)
        _, f_job = reduce_over_ranks(0.0, f_tot, self.world, self.dev)  # units all ranks processed
        _, n_job = reduce_over_ranks(0.0, float(len(specs)), self.world, self.dev)
        f_pair = sum(alg_flops(s)["pair_kernel"] for s in specs)
        n_pair = max(1, stage["launch_groups"]["pair"])
        pair_ms = stage["ms"]["pair"] / n_pair
        achieved = f_pair / (pair_ms * 1e-3) * 1e-12 if pair_ms > 0 else 0.0
        peak = self.peak
        traffic, traffic_src = ncu_pair_traffic(m["name"])
        roofline = {
            "kernel": "pair_kernel", "bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
            "frac": achieved / peak if peak else None, "launches": n_pair, "ms_per_launch": pair_ms,
            "algorithmic_flops_per_launch": f_pair, "traffic": traffic, "traffic_source": traffic_src,
        }
        if len(specs) == 1:
            fx = exec_pair_flops(specs[0], m["info"])
            roofline["executed"] = fx / (pair_ms * 1e-3) * 1e-12 if pair_ms > 0 else None
            roofline["executed_frac"] = roofline["executed"] / peak if peak and roofline["executed"] else None
        # transform stage (A1 + A2 incl. coefficient copies and, where it still exists, the unpack): both fractions.
        # In a batch the per-cluster transforms overlap on side streams, so the stage SUM is an upper bound of their wall time.
        tr_ms = (stage["ms"]["unpack"] + stage["ms"]["A1_gemm"] + stage["ms"]["A2_gemm"] + stage["ms"]["coeff_transpose"]) / max(1, steps)
        f_tr = sum(alg_flops(s)["A1"] + alg_flops(s)["A2"] for s in specs)
        b_tr = sum(8.0 * s.naux * s.npair + 8.0 * s.nocc * s.nvir * s.naux for s in specs)
        hbm_peak = measured_peaks().get("hbm_gbs")
        transform = {
            "ms_per_step": tr_ms, "tflops": f_tr / (tr_ms * 1e-3) * 1e-12 if tr_ms > 0 else None,
            "algorithmic_gbs": b_tr / (tr_ms * 1e-3) * 1e-9 if tr_ms > 0 else None, "hbm_peak_gbs": hbm_peak,
            "frac_hbm": (b_tr / (tr_ms * 1e-3) * 1e-9 / hbm_peak) if (tr_ms > 0 and hbm_peak) else None,
            "frac_fp64": (f_tr / (tr_ms * 1e-3) * 1e-12 / peak) if (tr_ms > 0 and peak) else None,
        }
        return {"f_tot": f_tot, "f_job": f_job, "n_job": n_job, "value": f_job / (m["ms_step"] * 1e-3) * 1e-12,
                "clusters_per_s": n_job / (m["ms_step"] * 1e-3), "roofline": roofline, "transform": transform}

    def sub_object(self, name, steps, warmup):
        """A time-boxed secondary workload measured in the same process with the same event timing (no e2e arm)."""
        m = self.measure(name, steps, warmup, want_e2e=False)
        z = self.summarize(m)
        s0 = m["specs"][0]
        out = {"workload": name, "clusters": len(m["specs"]), "steps": steps, "warmup": warmup, "ms_per_step": m["ms_step"],
               "tflops": z["value"], "clusters_per_s": z["clusters_per_s"], "pair_ms": z["roofline"]["ms_per_launch"],
               "pair_tflops": z["roofline"]["achieved"], "pair_frac": z["roofline"]["frac"],
               "transform_ms": z["transform"]["ms_per_step"], "transform_tflops": z["transform"]["tflops"],
               "transform_frac": z["transform"]["frac_fp64"], "gpu_launches": m["launches"],
               "sm_mhz": m["clocks"].get("sm_mhz"), "reasons": m["clocks"].get("reasons"),
               "E_frag": m["E"][:2], "stage_ms_per_step": {k: v / max(1, steps) for k, v in m["stage"]["ms"].items()}}
        if len(m["specs"]) == 1:
            out.update({"nocc": s0.nocc, "nvir": s0.nvir, "nao": s0.nao, "naux": s0.naux})
        return out


def measured_peaks() -> dict:
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except (OSError, ValueError):
        return {}


def run_gpu(args) -> None:
    gb = GpuBench()
    gb.no_pipeline = args.no_pipeline
    m = gb.measure(args.workload, args.steps, args.warmup, want_e2e=not args.no_e2e, want_rdm=args.rdm)
    gb.probe_peak()
    z = gb.summarize(m)
    specs, stage, clocks = m["specs"], m["stage"], m["clocks"]
    roofline = z["roofline"]
    mp = measured_peaks()
    sm_mhz = clocks.get("sm_mhz") or 0.0
    roofline.update({
        "peak_source": "live sie_dfmp2_probe_fp64: register-resident mma.sync.m8n8k4.f64 / DFMA issue-rate loop on all SMs "
                       "(MEASURED_PEAKS.json has no FP64 entry); the larger of the two",
        "probes_tflops": gb.probes,
        # rule of the task: another dtype's measured peak x the guide's nominal ratio (FP64 tensor 45 : bf16 2250 TFLOP/s)
        "peak_rule": float(mp.get("bf16_tflops_sustained", mp.get("bf16_tflops", 0.0))) * 45.0 / 2250.0 if mp else None,
        "peak_rule_source": "MEASURED_PEAKS.json bf16_tflops_sustained x 45/2250 (guide's nominal FP64:bf16 tensor ratio)" if mp else None,
        "peak_nominal_at_clock": 148 * 128 * sm_mhz * 1e6 * 1e-12 if sm_mhz else None,  # 64 DFMA/clk/SM x 2 flop
    })

    # ---- the other halves of the metric, time-boxed, same process / same timing: clusters/s of the 96-cluster batch
    #      (config 2) and the roofline fraction at each resident point of the size sweep (config 4)
    batch, sweep, next_rows = None, None, None
    if args.extras and gb.world == 1 and args.workload == "config3":
        k, w = max(1, min(args.steps, 3)), 3
        batch = gb.sub_object("config2", k, w)
        sweep = [gb.sub_object(f"config4:{i}", k, w) for i in range(3)]  # v = 256, 512, 1024 (v = 2048: --streamed)
        # the rows next to the hot path, small time-boxed cases: both 1-RDM blocks and the rank-r energy on
        # config 1; the general route (nocc > 128) on the environment-occupied x impurity-virtual shape; the canonical
        # out-of-core energy with its B store in pinned host memory
        next_rows = {}
        for nm, wl in (("config1", "config1"), ("general_454x64", "custom:454,64,2072,32")):
            mm = gb.measure(wl, 2, 2, want_e2e=False, want_rdm=True)
            zz = gb.summarize(mm)
            ent = dict(mm["next1"] or {}, workload=wl, energy_ms=zz["roofline"]["ms_per_launch"], energy_pair_frac=zz["roofline"]["frac"])
            for kk in ("rdm_occ", "rdm_vir"):
                if kk in ent:
                    ent[kk]["frac_of_fp64_peak"] = ent[kk]["tflops"] / gb.peak if gb.peak else None
            next_rows[nm] = ent
        cm = canonical_measure("128,512,2560,32,host", 4.0)
        next_rows["canonical_out_of_core"] = {kk: cm[kk] for kk in ("nocc", "nvir", "naux", "store", "info", "E_MP2", "transform_ms", "energy_ms",
                                                                "energy_tflops", "energy_frac_of_fp64_peak", "panel_gbs")}

    # ---- CPU oracle beside it (rank 0, N = 1 only): bounded sample, extrapolated
    cpu = None
    if gb.rank == 0 and gb.world == 1 and not args.no_cpu:
        secs, spent, desc, cores = oracle_workload_seconds(specs)
        cpu = {"value": z["f_tot"] / secs * 1e-12, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
               "extrapolated_s_per_step": secs, "measured_s": spent}
        # context: the same oracle's FULL run of this workload, timed once while tests/golden/make_goldens.py wrote the golden
        # (another machine: the build container's 8 cores, shared with compiles) — not this box, not part of `value`
        gj = os.path.join(ROOT, "tests", "golden", f"dense_{args.workload}.json")
        if os.path.exists(gj):
            with open(gj) as fh:
                gm = json.load(fh)
            if "oracle_wall_s_this_run" in gm:
                cpu["full_run_on_build_container"] = {"seconds": gm["oracle_wall_s_this_run"], "threads": gm.get("oracle_threads"),
                                                      "tflops": z["f_tot"] / gm["oracle_wall_s_this_run"] * 1e-12,
                                                      "source": f"tests/golden/dense_{args.workload}.json"}

    if gb.rank == 0:
        l2 = "inputs larger than L2 (no flush needed)" if m["in_bytes"] > (126 << 20) else "inputs smaller than L2; L2 not flushed"
        line = {
            "metric": METRIC, "value": z["value"], "unit": UNIT, "n_gpus": gb.world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": m["ms_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(args.workload, specs, l2),
            "clusters_per_s": z["clusters_per_s"],
            "E_frag": m["E"] if len(m["E"]) <= 4 else m["E"][:4],
            "stage_ms_per_step": {k: v / max(1, args.steps) for k, v in stage["ms"].items()},
            "roofline": roofline, "transform": z["transform"], "cpu_baseline": cpu, "clocks": clocks, "gpu_launches": m["launches"],
            "workspace_bytes": m["ws_bytes"], "input_gen_s": m["t_gen"],
        }
        if m["next1"] is not None:
            for k_ in ("rdm_occ", "rdm_vir"):
                m["next1"][k_]["frac_of_fp64_peak"] = m["next1"][k_]["tflops"] / gb.peak if gb.peak else None
            line["next1_rdm"] = m["next1"]
        if batch is not None:
            line["batch"] = batch
            line["sweep"] = sweep
            line["next_rows"] = next_rows
        e2e = None
        if m["e2e"] is not None:
            ms_e2e = m["e2e"]["ms"]
            e2e = {"value": z["f_job"] / (ms_e2e * 1e-3) * 1e-12, "unit": UNIT, "ms_per_step": ms_e2e,
                   "h2d_bytes_per_step": m["in_bytes"], "d2h_bytes_per_step": m["out_bytes"], "steps": args.steps, "warmup": args.warmup,
                   "h2d_gbs": m["in_bytes"] / (ms_e2e * 1e-3) * 1e-9,
                   "same_result_as_device_arm": bool(all(abs(a - b) <= 1e-12 * abs(a) for a, b in zip(m["E"], m["e2e"]["E"]))),
                   "pipelined_over_steps": m["e2e"].get("pipelined", False),
                   "how": ("two plans (SIE_FLAG_HOST_IO | SIE_FLAG_STAGE_FULL) on two streams: transform of step n+1 enqueued before the "
                           "energy of step n; every step uploads all inputs from pinned host memory and reads E, G back"
                           if m["e2e"].get("pipelined") else "one plan, SIE_FLAG_HOST_IO, steps back to back")}
        line["e2e"] = e2e
        print(json.dumps(line))
    if gb.world > 1:
        gb.dist.destroy_process_group()


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


def run_canonical(args) -> None:
    print(json.dumps(canonical_measure(args.canonical, args.stream_gb)))


def canonical_measure(desc: str, stream_gb: float = 8.0) -> dict:
    """NEXT-2 (not a bench line): whole-system canonical DF-MP2 energy, B store in pinned host memory (out of core) or on the
    device.  desc = o,v,naux[,occ_block[,host|device]]; nao = o + v; the packed integrals are generated and fed in aux
    blocks (never resident at once).  Reports the device time of the two phases (CUDA events) and the panel traffic."""
    import torch

    import paper_2412_18553_b200 as sie

    torch.cuda.set_device(0)
    f = desc.split(",")
    o, v, naux = int(f[0]), int(f[1]), int(f[2])
    occ_block = int(f[3]) if len(f) > 3 else 0
    store = f[4] if len(f) > 4 else "host"
    spec = ClusterSpec(10, 0, o + v, o, v, naux, 0)
    x = make_cluster(spec)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731
    s = sie.CanonicalSolver(spec.nao, o, v, naux, occ_block=occ_block, store=store)
    info = s.info()
    blk = max(8, min(naux, int(stream_gb * 1e9) // (8 * spec.npair)) // 8 * 8)
    pinned = torch.empty((blk, spec.npair), dtype=torch.float64, pin_memory=True)
    Ld = torch.empty((blk, spec.npair), dtype=torch.float64, device="cuda")
    C_occ, C_vir, e_occ, e_vir = cu(x.C_occ), cu(x.C_vir), cu(x.e_occ), cu(x.e_vir)
    ncpu = max(1, min(32, os.cpu_count() or 8))
    l0 = sie.launch_count()
    t_tr = 0.0
    with ClockSampler(0) as cs:
        for p0 in range(0, naux, blk):
            p1 = min(naux, p0 + blk)
            x.L_block(p0, p1, out=pinned.numpy()[: p1 - p0], threads=ncpu)
            Ld[: p1 - p0].copy_(pinned[: p1 - p0])
            torch.cuda.synchronize()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record()
            s.transform(C_occ, C_vir, Ld[: p1 - p0], p0, p1)
            ev1.record()
            torch.cuda.synchronize()
            t_tr += ev0.elapsed_time(ev1)
        E = s.energy(e_occ, e_vir)  # warm-up pass (same work)
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        E = s.energy(e_occ, e_vir)
        ev1.record()
        torch.cuda.synchronize()
        t_en = ev0.elapsed_time(ev1)
    peak = max(max(sie.sie_dfmp2_probe_fp64(k, 40000, 2)[0] for _ in range(3)) for k in (0, 1))
    fl = alg_flops(spec)
    f_pair = 1.0 * o * (o + 1) * v * v * naux  # unordered occupied pairs, full v x v block each: the minimum
    nb = info["n_occ_blocks"]
    panel_bytes = (nb + nb * (nb - 1) // 2) * 8.0 * info["occ_block"] * v * ((naux + 7) // 8 * 8)
    line = {"mode": "canonical (NEXT-2)", "nocc": o, "nvir": v, "nao": o + v, "naux": naux, "store": store, "info": info,
            "E_MP2": float(E.cpu()[0]), "transform_ms": t_tr, "transform_tflops": (fl["A1"] + fl["A2"]) / (t_tr * 1e-3) * 1e-12,
            "energy_ms": t_en, "energy_tflops": f_pair / (t_en * 1e-3) * 1e-12, "energy_frac_of_fp64_peak": f_pair / (t_en * 1e-3) * 1e-12 / peak,
            "fp64_peak_probe": peak, "panel_bytes_to_device_per_energy": panel_bytes,
            "panel_gbs": panel_bytes / (t_en * 1e-3) * 1e-9, "b_store_bytes": s.bstore_bytes, "workspace_bytes": s.workspace_bytes,
            "gpu_launches": sie.launch_count() - l0, "clocks": cs.summary(),
            "note": "device time of each phase (CUDA events); packed integrals generated and fed in aux blocks; data synthetic"}
    s.close()
    return line


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="config3")
    ap.add_argument("--impl", default="sie", choices=["sie", "reference"])
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end arm")
    ap.add_argument("--no-cpu", action="store_true", help="skip the CPU oracle leg")
    ap.add_argument("--no-pipeline", action="store_true", help="e2e arm: one plan, steps back to back (no overlap of the next upload)")
    ap.add_argument("--no-extras", dest="extras", action="store_false",
                    help="skip the time-boxed config-2 batch and config-4 sweep sub-objects of the default config-3 line")
    ap.add_argument("--rdm", action="store_true", help="also time sie_dfmp2_rdm_occ and sie_dfmp2_rdm_vir (NEXT-1: both MP2 1-RDM blocks) on the same B")
    ap.add_argument("--streamed", action="store_true", help="feed the packed integrals in aux blocks generated on the fly "
                                                             "(sweep points that do not fit in HBM; not a bench line)")
    ap.add_argument("--stream-gb", type=float, default=8.0, help="size of one streamed aux block in GB")
    ap.add_argument("--canonical", default="", help="o,v,naux[,occ_block[,host|device]]: whole-system canonical DF-MP2 energy "
                                                     "(NEXT-2, out of core; not a bench line)")
    args = ap.parse_args()
    if args.canonical:
        run_canonical(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.streamed:
        run_streamed(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
