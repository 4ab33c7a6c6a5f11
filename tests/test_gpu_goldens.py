"""Dense full-size parity on BASELINE.json configs 2, 3 and 4 against checked-in oracle results.

The expected values under tests/golden/dense_*.{json,npz} were written by tests/golden/make_goldens.py, which calls ONLY
oracle/ (plain loops, O1-O7 as they stand) on the seeded inputs of workloads/ — hours of CPU time for config 3 and the
large sweep points, which is why they are stored instead of recomputed.  Here the CUDA path regenerates the same seeded
inputs and runs them in the launch configuration bench.py times (one transform call over [0, naux), 148 persistent
CTAs; one sie_dfmp2_batch call for config 2; aux blocks streamed from the host for the sweep point that does not fit
in HBM), and every energy and every G element is compared:

    |E_gpu - E_or| <= 1e-10 |E_or|        max|G_gpu - G_or| <= 1e-11 * max(1, max|G_or|)   (inputs ~ N(0, variance 1/nao), A-9)

A case whose golden file has not been generated yet is skipped with that reason (never silently passed).
"""
import json
import os

import numpy as np
import pytest
import torch

import paper_2412_18553_b200 as sie
from workloads import config_specs, make_cluster, occupied_subset, virtual_subset

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))
E_RTOL = 1e-10
G_ATOL = 1e-11


def _golden(case):
    pj, pz = os.path.join(HERE, "golden", f"dense_{case}.json"), os.path.join(HERE, "golden", f"dense_{case}.npz")
    if not (os.path.exists(pj) and os.path.exists(pz)):
        pytest.skip(f"tests/golden/dense_{case}.* not generated yet (tests/golden/make_goldens.py --cases {case})")
    with open(pj) as f:
        meta = json.load(f)
    return meta, np.load(pz)


def _need_gb(gb):
    free, _ = torch.cuda.mem_get_info()
    if free < gb * 2**30:
        pytest.skip(f"needs {gb} GiB of free device memory")


def _cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _assert_E(E, Eor):
    assert Eor < 0
    assert abs(E - Eor) <= E_RTOL * abs(Eor), (E, Eor, abs(E - Eor) / abs(Eor))


def _assert_G(G, Gor):
    err, mag = float(np.max(np.abs(G - Gor))), float(np.max(np.abs(Gor)))
    assert err <= G_ATOL * max(1.0, mag), (err, mag, err / mag)


def _upload_L(x, spec, threads=16, rows_per_chunk=256):
    """Packed (P|mu nu) of the whole cluster on the device, generated chunk by chunk through one pinned buffer."""
    L = torch.empty((spec.naux, spec.npair), dtype=torch.float64, device="cuda")
    pin = torch.empty((rows_per_chunk, spec.npair), dtype=torch.float64).pin_memory()
    for p0 in range(0, spec.naux, rows_per_chunk):
        p1 = min(spec.naux, p0 + rows_per_chunk)
        x.L_block(p0, p1, out=pin.numpy()[: p1 - p0], threads=threads)
        L[p0:p1].copy_(pin[: p1 - p0])
        torch.cuda.synchronize()
    return L


# ---------------------------------------------------------------------------------------------- config 2: all 96 clusters
def test_config2_all_96_clusters_match_goldens():
    meta, arr = _golden("config2")
    specs = config_specs(2)
    assert len(specs) == 96 and meta["nocc"] == [s.nocc for s in specs]
    _need_gb(70)
    cl = []
    for s in specs:
        x = make_cluster(s)
        cl.append(dict(nao=s.nao, nocc=s.nocc, nvir=s.nvir, naux=s.naux, C_occ=_cu(x.C_occ), C_vir=_cu(x.C_vir),
                       L_packed=_cu(x.L_packed(threads=16)), e_occ=_cu(x.e_occ), e_vir=_cu(x.e_vir), P_frag=_cu(x.P_frag),
                       E_out=torch.zeros(1, dtype=torch.float64, device="cuda"),
                       G_out=torch.zeros(s.nocc, s.nocc, dtype=torch.float64, device="cuda")))
    ws = sie.alloc_workspace(sie.sie_dfmp2_batch_query(cl))
    sie.sie_dfmp2_batch(cl, ws)  # ONE scheduled submission, as bench.py --workload config2 times it
    torch.cuda.synchronize()
    for k, (s, c) in enumerate(zip(specs, cl)):
        _assert_E(float(c["E_out"].cpu()[0]), meta["E_frag"][k])
        _assert_G(c["G_out"].cpu().numpy(), arr[f"G_{k:03d}"])


# ---------------------------------------------------------------------------------------------- config 3: the headline cluster
@pytest.fixture(scope="module")
def config3_inputs():
    spec = config_specs(3)[0]
    free, _ = torch.cuda.mem_get_info()
    if free < 45 * 2**30:
        pytest.skip("needs 45 GiB of free device memory")
    x = make_cluster(spec)
    L = _upload_L(x, spec)
    yield spec, x, L
    del L
    torch.cuda.empty_cache()


def test_config3_dense_full_size_matches_golden(config3_inputs):
    """The dense headline problem, exactly what bench.py times (its printed E_frag is this number)."""
    meta, arr = _golden("config3")
    spec, x, L = config3_inputs
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux)
    info = s.info()
    assert info["TM"] == 120 and info["ncta"] == 148 and info["ntiles"] == 1080 * 1081 // 2
    s.transform(_cu(x.C_occ), _cu(x.C_vir), L, 0, spec.naux)
    e_occ, e_vir = _cu(x.e_occ), _cu(x.e_vir)
    E, G = s.energy(e_occ, e_vir, _cu(x.P_frag))
    E_I, G_I = s.energy(e_occ, e_vir, None)
    torch.cuda.synchronize()
    assert torch.equal(G, G_I)  # A-15: G does not depend on the projector
    _assert_E(float(E.cpu()[0]), meta["E_frag"])
    _assert_E(float(E_I.cpu()[0]), meta["E_identity"])
    _assert_G(G.cpu().numpy(), arr["G"])
    s.close()


def test_config3_dense_aux_256_dense_virtuals_matches_golden(config3_inputs):
    """All 4800 aux rows and all occupied orbitals dense, C_vir zero outside 256 seeded columns: every tile still runs all
    600 K-blocks with non-zero data; the oracle ran the compressed problem (same bytes).  Also the occupied 1-RDM block."""
    meta, arr = _golden("config3_v256")
    spec, x, L = config3_inputs
    virt = virtual_subset(spec, 256)
    assert np.array_equal(virt, arr["virtual_subset"])
    C_vir = np.zeros_like(x.C_vir)
    C_vir[:, virt] = x.C_vir[:, virt]
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux)
    s.transform(_cu(x.C_occ), _cu(C_vir), L, 0, spec.naux)
    e_occ, e_vir = _cu(x.e_occ), _cu(x.e_vir)
    E, G = s.energy(e_occ, e_vir, _cu(x.P_frag))
    gam, tr = s.rdm_occ(e_occ, e_vir)
    torch.cuda.synchronize()
    _assert_E(float(E.cpu()[0]), meta["E_frag"])
    _assert_G(G.cpu().numpy(), arr["G"])
    _assert_G(gam.cpu().numpy(), arr["gamma_occ"])
    assert abs(float(tr.cpu()[0]) - meta["trace_gamma_occ"]) <= E_RTOL * abs(meta["trace_gamma_occ"])
    s.close()


# ---------------------------------------------------------------------------------------------- config 4: the size sweep
@pytest.mark.parametrize("k", [0, 1, 2, 3, "3_v256", "3_o8"])
def test_config4_sweep_point_matches_golden(k):
    """k = "3_v256": the v = 2048 point with C_vir zeroed outside 256 seeded columns (dense aux, dense occupied): the GPU
    streams all 150.8 GB of packed integrals and runs the full-size launch, the oracle ran the compressed problem.
    k = "3_o8": the same point with all 2048 virtuals and all 8448 aux rows dense and C_occ zeroed outside 8 seeded columns:
    every virtual-pair tile of the full-size launch carries non-zeros; the 8 x 8 block of G on the kept occupieds is the
    oracle's compressed problem, the rest of G is exactly zero (zero rows of B give zero integrals and amplitudes)."""
    meta, arr = _golden(f"config4_{k}")
    sub = k if isinstance(k, str) else ""
    k = 3 if sub else k
    spec = config_specs(4)[2 * k]  # rank-32 projector; the P = I run shares G (A-15)
    x = make_cluster(spec)
    occ = None
    if sub == "3_v256":
        virt = virtual_subset(spec, 256)
        assert np.array_equal(virt, arr["virtual_subset"])
        Cz = np.zeros_like(x.C_vir)
        Cz[:, virt] = x.C_vir[:, virt]
        x.C_vir = Cz
    elif sub == "3_o8":
        occ = occupied_subset(spec, 8)
        assert np.array_equal(occ, arr["occupied_subset"])
        Cz = np.zeros_like(x.C_occ)
        Cz[:, occ] = x.C_occ[:, occ]
        x.C_occ = Cz
    _need_gb(8 * spec.naux * spec.npair / 2**30 + 16 if k < 3 else 40)
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux)
    C_occ, C_vir = _cu(x.C_occ), _cu(x.C_vir)
    if k < 3:  # resident, one transform call (bench.py --workload config4:k)
        L = _upload_L(x, spec)
        s.transform(C_occ, C_vir, L, 0, spec.naux)
    else:      # v = 2048: packed integrals 150.8 GB, streamed in aux blocks (bench.py --workload config4:3 --streamed)
        blk = 448
        pin = torch.empty((blk, spec.npair), dtype=torch.float64).pin_memory()
        Ld = torch.empty((blk, spec.npair), dtype=torch.float64, device="cuda")
        for p0 in range(0, spec.naux, blk):
            p1 = min(spec.naux, p0 + blk)
            x.L_block(p0, p1, out=pin.numpy()[: p1 - p0], threads=16)
            torch.cuda.synchronize()
            Ld[: p1 - p0].copy_(pin[: p1 - p0])
            s.transform(C_occ, C_vir, Ld[: p1 - p0], p0, p1)
        L = Ld
    e_occ, e_vir = _cu(x.e_occ), _cu(x.e_vir)
    E, G = s.energy(e_occ, e_vir, _cu(x.P_frag))
    E_I, _ = s.energy(e_occ, e_vir, None, want_G=False)
    torch.cuda.synchronize()
    _assert_E(float(E.cpu()[0]), meta["E_frag"])
    _assert_E(float(E_I.cpu()[0]), meta["E_identity"])
    Gh = G.cpu().numpy()
    if occ is not None:  # everything outside the kept block is exactly zero; the block is the oracle's compressed problem
        mask = np.ones_like(Gh, dtype=bool)
        mask[np.ix_(occ, occ)] = False
        assert not np.any(Gh[mask])
        Gh = Gh[np.ix_(occ, occ)]
    _assert_G(Gh, arr["G"])
    if "gamma_occ" in arr.files:
        gam, _ = s.rdm_occ(e_occ, e_vir)
        gh = gam.cpu().numpy()
        if occ is not None:  # untouched occupieds keep occupation 2 exactly (Eq. S18 with zero amplitudes)
            rest = gh.copy()
            rest[np.ix_(occ, occ)] = 0.0
            expect = 2.0 * np.eye(spec.nocc)
            expect[np.ix_(occ, occ)] = 0.0
            assert np.array_equal(rest, expect)
            gh = gh[np.ix_(occ, occ)]
        _assert_G(gh, arr["gamma_occ"])
    s.close()
    del L
    torch.cuda.empty_cache()
