"""Writes the dense full-size goldens under tests/golden/ by calling ONLY ``oracle/`` on the seeded inputs of
``workloads/`` (no CUDA, no torch, nothing from paper_2412_18553_b200/).  SURVEY.md §8(d): "full-run goldens
(E, G) are produced once offline and checked in as small files".

    python tests/golden/make_goldens.py --cases config2,config4_0,config4_1,config3_v256,config4_2,config3,config4_3 \
        --cache /some/scratch/dir [--threads 8]

Cases (BASELINE.json configs; generator recipe in workloads/gen.py):
  config2        all 96 clusters of the batch config: G and E_frag (rank nocc/4 projector) of each
  config3        the dense headline cluster (o=120, v=1080, nao=1200, naux=4800): G, E_frag (rank 60), E(P=I)
  config3_v256   config 3 with C_vir zeroed outside workloads.virtual_subset(spec, 256): the oracle runs the
                 compressed problem (same bytes for the 256 kept columns), G, E, and gamma_occ (Eq. S18)
  config4_k      sweep point k (o=64, v=256/512/1024/2048): G, E_frag (rank 32), E(P=I); gamma_occ for k <= 1
  config4_3_v256 the v=2048 point (nao=2112, naux=8448, packed integrals 150.8 GB) with C_vir zeroed outside 256 seeded
                 columns: the compressed problem for the oracle, the full-size streamed launch for the GPU; G, E, gamma_occ
  config4_3_o8   the same v=2048 point with all 2048 virtuals and all 8448 aux rows dense and C_occ zeroed outside
                 workloads.occupied_subset(spec, 8): the 8 x 8 block of G and gamma_occ on the kept occupieds, E_frag with
                 the matching block of P_frag, E(P=I)

What is computed is exactly oracle.transform_block (O1-O3), oracle.pair_G (O4-O6) and oracle.trace (O7) as they
stand.  The only thing this script adds is bookkeeping: the aux index is fed in blocks (the oracle's own p0/p1
arguments) and the j sum of O6 is fed in chunks of ``--jchunk`` (the oracle's own j0/j1 arguments: "slices add");
chunk results are summed in j order in long double.  Chunks and B are checkpointed under --cache so an
interrupted run resumes; nothing under --cache is read by any test.

Outputs per case: ``dense_<case>.npz`` (arrays) and ``dense_<case>.json`` (energies as repr and hex, sizes,
max|G|, oracle wall time and thread count).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from workloads import config_specs, make_cluster, occupied_subset, virtual_subset  # noqa: E402


def _log(msg):
    print(time.strftime("%H:%M:%S"), msg, flush=True)


def _B(case, x, C_occ, C_vir, cache, threads, pblk=96):
    """O1-O3 in aux blocks; B [nocc'][nvir'][naux]."""
    spec = x.spec
    path = os.path.join(cache, f"B_{case}.npy")
    if os.path.exists(path):
        return np.load(path)
    B = np.zeros((C_occ.shape[1], C_vir.shape[1], spec.naux))
    buf = np.empty((pblk, spec.npair))
    for p0 in range(0, spec.naux, pblk):
        p1 = min(spec.naux, p0 + pblk)
        Lb = x.L_block(p0, p1, out=buf[: p1 - p0], threads=threads)
        oracle.transform_block(C_occ, C_vir, Lb, p0, p1, B)
        if (p0 // pblk) % 10 == 0:
            _log(f"  {case}: transform rows {p1}/{spec.naux}")
    if B.nbytes > (64 << 20):
        np.save(path + ".tmp.npy", B)
        os.replace(path + ".tmp.npy", path)
    return B


def _G(case, B, e_occ, e_vir, cache, jchunk):
    """O4-O6 in j chunks, summed in j order in long double."""
    nocc = B.shape[0]
    acc = np.zeros((nocc, nocc), dtype=np.longdouble)
    for j0 in range(0, nocc, jchunk):
        j1 = min(nocc, j0 + jchunk)
        path = os.path.join(cache, f"G_{case}_j{j0:04d}_{j1:04d}.npy")
        if os.path.exists(path):
            g = np.load(path)
        else:
            t = time.time()
            g = oracle.pair_G(B, e_occ, e_vir, j0, j1)
            np.save(path + ".tmp.npy", g)
            os.replace(path + ".tmp.npy", path)
            _log(f"  {case}: j [{j0},{j1}) of {nocc}  {time.time() - t:.1f} s")
        acc += g.astype(np.longdouble)
    return np.asarray(acc, dtype=np.float64)


def _energies(P_frag, G):
    return {"E_frag": oracle.trace(P_frag, G), "E_identity": oracle.trace(None, G)}


def _write(case, arrays, meta):
    np.savez(os.path.join(HERE, f"dense_{case}.npz"), **arrays)
    for k in list(meta):
        if isinstance(meta[k], float):
            meta[k + "_hex"] = float(meta[k]).hex()
    with open(os.path.join(HERE, f"dense_{case}.json"), "w") as f:
        json.dump(meta, f, indent=1, sort_keys=True)
        f.write("\n")
    _log(f"wrote dense_{case}.npz / .json")


def _spec_meta(spec):
    return {"config_id": spec.config_id, "cluster_id": spec.cluster_id, "nao": spec.nao, "nocc": spec.nocc,
            "nvir": spec.nvir, "naux": spec.naux, "rank": spec.rank, "scale": spec.scale}


def single(case, spec, cache, threads, jchunk, subset=0, want_gamma=False, occ_subset=0):
    t0 = time.time()
    x = make_cluster(spec)
    if subset:
        virt = virtual_subset(spec, subset)
        C_vir, e_vir = np.ascontiguousarray(x.C_vir[:, virt]), np.ascontiguousarray(x.e_vir[virt])
    else:
        virt, C_vir, e_vir = None, x.C_vir, x.e_vir
    C_occ, e_occ, P_frag, occ = x.C_occ, x.e_occ, x.P_frag, None
    if occ_subset:  # zero columns of C_occ give zero rows of B: their pairs contribute nothing to any sum (numerators are 0)
        occ = occupied_subset(spec, occ_subset)
        C_occ, e_occ = np.ascontiguousarray(x.C_occ[:, occ]), np.ascontiguousarray(x.e_occ[occ])
        P_frag = np.ascontiguousarray(x.P_frag[np.ix_(occ, occ)])
    parent = os.path.join(cache, f"B_{case.rsplit('_v', 1)[0]}.npy") if subset else ""
    if subset and os.path.exists(parent):
        # B[i][a][P] of the kept columns is a slice of the parent case's oracle B (every (i,a,P) entry is its own sum over
        # mu, nu in O2-O3: identical operations, identical bits) — saves repeating O1-O2 on all aux rows
        B = np.ascontiguousarray(np.load(parent, mmap_mode="r")[:, virt, :])
        _log(f"  {case}: B sliced from {os.path.basename(parent)}")
    else:
        B = _B(case, x, C_occ, C_vir, cache, threads)
    G = _G(case, B, e_occ, e_vir, cache, jchunk)
    arrays = {"G": G}
    meta = {"case": case, "spec": _spec_meta(spec), "max_abs_G": float(np.max(np.abs(G))), **_energies(P_frag, G)}
    if occ_subset:
        arrays["occupied_subset"] = occ
        meta["occupied_subset"] = int(occ_subset)
    if subset:
        arrays["virtual_subset"] = virt
        meta["virtual_subset"] = int(subset)
    if want_gamma:
        g = oracle.rdm_occ(B, e_occ, e_vir)
        arrays["gamma_occ"] = g
        meta["trace_gamma_occ"] = float(np.trace(g))
    meta["oracle_threads"] = oracle.threads()
    meta["oracle_wall_s_this_run"] = round(time.time() - t0, 1)  # includes checkpoint hits: a lower bound if resumed
    meta["written_by"] = "tests/golden/make_goldens.py (oracle/ only)"
    _write(case, arrays, meta)


def config2(cache, threads):
    t0 = time.time()
    arrays, E, sizes = {}, [], []
    for spec in config_specs(2):
        path = os.path.join(cache, f"G_config2_{spec.cluster_id:03d}.npy")
        x = make_cluster(spec)
        if os.path.exists(path):
            G = np.load(path)
        else:
            G = oracle.pair_G(oracle.transform(x.C_occ, x.C_vir, x.L_packed(threads=threads)), x.e_occ, x.e_vir)
            np.save(path + ".tmp.npy", G)
            os.replace(path + ".tmp.npy", path)
            _log(f"  config2: cluster {spec.cluster_id} (o={spec.nocc}) done")
        arrays[f"G_{spec.cluster_id:03d}"] = G
        E.append(oracle.trace(x.P_frag, G))
        sizes.append(spec.nocc)
    meta = {"case": "config2", "nocc": sizes, "E_frag": E, "E_frag_hex": [float(e).hex() for e in E],
            "oracle_threads": oracle.threads(), "oracle_wall_s_this_run": round(time.time() - t0, 1),
            "written_by": "tests/golden/make_goldens.py (oracle/ only)"}
    np.savez(os.path.join(HERE, "dense_config2.npz"), **arrays)
    with open(os.path.join(HERE, "dense_config2.json"), "w") as f:
        json.dump(meta, f, indent=1, sort_keys=True)
        f.write("\n")
    _log("wrote dense_config2.npz / .json")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cases", required=True)
    ap.add_argument("--cache", required=True)
    ap.add_argument("--threads", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--jchunk", type=int, default=4)
    a = ap.parse_args()
    os.makedirs(a.cache, exist_ok=True)
    oracle.set_threads(a.threads)
    for case in a.cases.split(","):
        _log(f"case {case}")
        if case == "config2":
            config2(a.cache, a.threads)
        elif case == "config3":
            single(case, config_specs(3)[0], a.cache, a.threads, a.jchunk)
        elif case == "config3_v256":
            single(case, config_specs(3)[0], a.cache, a.threads, a.jchunk, subset=256, want_gamma=True)
        elif case == "config4_3_v256":
            single(case, config_specs(4)[6], a.cache, a.threads, a.jchunk, subset=256, want_gamma=True)
        elif case == "config4_3_o8":
            single(case, config_specs(4)[6], a.cache, a.threads, a.jchunk, want_gamma=True, occ_subset=8)
        elif case.startswith("config4_"):
            k = int(case.split("_")[1])
            single(case, config_specs(4)[2 * k], a.cache, a.threads, a.jchunk, want_gamma=(k <= 1))
        else:
            raise SystemExit(f"unknown case {case}")


if __name__ == "__main__":
    main()
