"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded inputs.

Tolerances (BASELINE.json north_star; DESIGN.md §4 reading A-9):
  * E_frag: |E_gpu - E_or| <= 1e-10 |E_or|
  * G:      literal |dG| <= 1e-11 for the scale="std" inputs (|G| ~ 0.1..1);
            for the literal variance-1/nao inputs (|G| up to 1e4..1e5, ulp ~ 1e-11) the bar is 1e-11 * max(1, max|G_or|).
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_18553_b200 as sie
from paper_2412_18553_b200 import binding
from workloads import ClusterSpec, config_specs, make_cluster

pytestmark = pytest.mark.gpu

E_RTOL = 1e-10
G_ATOL = 1e-11

_ORACLE_CACHE = {}


def oracle_G(spec: ClusterSpec):
    key = (spec.config_id, spec.cluster_id, spec.nao, spec.nocc, spec.nvir, spec.naux, spec.scale)
    if key not in _ORACLE_CACHE:
        x = make_cluster(spec)
        B = oracle.transform(x.C_occ, x.C_vir, x.L_packed(threads=4))
        _ORACLE_CACHE[key] = oracle.pair_G(B, x.e_occ, x.e_vir)
    return _ORACLE_CACHE[key]


def gpu_run(spec: ClusterSpec, flags=0, blocks=None, aux_block=0, want_G=True):
    x = make_cluster(spec)
    host = bool(flags & binding.SIE_FLAG_HOST_IO)
    to = (lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()) if host else (lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda())
    solver = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux, aux_block=aux_block, flags=flags)
    C_occ, C_vir = to(x.C_occ), to(x.C_vir)
    if blocks is None:
        blocks = [(0, spec.naux)]
    keep = []
    for p0, p1 in blocks:
        Lb = to(x.L_block(p0, p1, threads=4))
        keep.append(Lb)
        solver.transform(C_occ, C_vir, Lb, p0, p1)
    P = None if spec.rank <= 0 else to(x.P_frag)
    E, G = solver.energy(to(x.e_occ), to(x.e_vir), P, want_G=want_G)
    torch.cuda.synchronize()
    out = float(E.cpu()[0]), (G.cpu().numpy() if G is not None else None)
    solver.close()
    return out


def check(spec, E, G, Gor=None):
    x = make_cluster(spec)
    Gor = oracle_G(spec) if Gor is None else Gor
    Eor = oracle.trace(None if spec.rank <= 0 else x.P_frag, Gor)
    assert abs(E - Eor) <= E_RTOL * abs(Eor), (E, Eor)
    if G is not None:
        bar = G_ATOL if spec.scale == "std" else G_ATOL * max(1.0, float(np.max(np.abs(Gor))))
        err = float(np.max(np.abs(G - Gor)))
        assert err <= bar, (err, bar, float(np.max(np.abs(Gor))))


# ---------------------------------------------------------------------------------------------- configs 0, 1
@pytest.mark.parametrize("scale", ["var", "std"])
@pytest.mark.parametrize("flags", [0, binding.SIE_FLAG_REFERENCE], ids=["dmma", "reference"])
def test_config0(scale, flags):
    spec = config_specs(0, scale)[0]
    E, G = gpu_run(spec, flags)
    check(spec, E, G)


@pytest.mark.parametrize("scale", ["var", "std"])
def test_config1_projector_and_identity(scale):
    s_rank, s_id = config_specs(1, scale)
    E, G = gpu_run(s_rank, blocks=[(0, 500), (500, 1200)])
    check(s_rank, E, G)
    E2, G2 = gpu_run(s_id)
    check(s_id, E2, G2)
    assert abs(E2 - np.trace(oracle_G(s_id))) <= E_RTOL * abs(E2)  # P = I is the canonical MP2 total
    assert np.array_equal(G, G2)  # G does not depend on P_frag, and the run is bit-reproducible


def test_config1_reference_kernels_agree():
    spec = config_specs(1)[0]
    E, G = gpu_run(spec, binding.SIE_FLAG_REFERENCE)
    check(spec, E, G)


# ---------------------------------------------------------------------------------------------- ragged shapes
RAGGED = [
    # (nocc, nvir, extra_ao, naux): several tiles, ragged tails in every dimension
    (1, 1, 0, 1),
    (1, 3, 2, 5),
    (5, 13, 5, 37),
    (8, 129, 0, 64),
    (17, 50, 3, 100),
    (24, 77, 0, 130),
    (33, 70, 1, 129),
    (48, 100, 0, 96),
    (64, 96, 0, 200),
    (72, 75, 0, 90),
    (81, 40, 1, 70),   # 11 strips: small-strip epilogue, o not a multiple of 8
    (96, 50, 0, 64),   # 12 strips: the largest block on the small-strip epilogue
    (97, 30, 0, 40),   # 13 strips, 104-row tiles: polling-producer kernel, small strip
    (110, 20, 0, 40),  # 14 strips, 112-row tiles
    (121, 12, 0, 24),  # 16 strips, 128-row tiles: warp-0 producer, generic strip
    (120, 140, 0, 200),
    (128, 130, 4, 72),
    # many virtual blocks per tile (ta = 64, 42, 18, 4 with a ragged last block), one block of 127 rows
    (2, 70, 0, 24),
    (3, 200, 1, 9),
    (7, 300, 0, 40),
    (30, 41, 0, 88),
    (127, 3, 0, 16),
]


@pytest.mark.parametrize("nocc,nvir,extra,naux", RAGGED)
def test_ragged_shapes(nocc, nvir, extra, naux):
    spec = ClusterSpec(50, nocc * 1000 + nvir, nocc + nvir + extra, nocc, nvir, naux, max(1, nocc // 3), "std")
    # uneven, out-of-order aux blocks exercise the coverage logic and odd p0 offsets
    cuts = sorted({0, naux, naux // 3, (2 * naux) // 3 + 1 if naux > 3 else naux})
    blocks = [(cuts[i], cuts[i + 1]) for i in range(len(cuts) - 1)][::-1]
    E, G = gpu_run(spec, blocks=blocks, aux_block=7 if naux > 20 else 0)
    check(spec, E, G)


def test_nocc_above_128_uses_general_route():
    spec = ClusterSpec(51, 0, 130 + 20, 130, 20, 24, 10, "std")
    E, G = gpu_run(spec)
    check(spec, E, G)


def test_identity_projector_null_pointer_and_no_G():
    spec = ClusterSpec(52, 0, 40, 6, 34, 50, 0, "std")
    E, G = gpu_run(spec, want_G=False)
    assert G is None
    check(spec, E, None)


# ---------------------------------------------------------------------------------------------- host I/O path
def test_host_io_matches_device_io():
    spec = config_specs(0, "std")[0]
    E, G = gpu_run(spec, binding.SIE_FLAG_HOST_IO, blocks=[(0, 64), (64, 160)], aux_block=16)
    check(spec, E, G)
    Ed, Gd = gpu_run(spec, 0, aux_block=16)
    assert E == Ed and np.array_equal(G, Gd)


# ---------------------------------------------------------------------------------------------- batch
def _batch_run(specs, flags=0):
    host = bool(flags & binding.SIE_FLAG_HOST_IO)
    to = (lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()) if host else (lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda())
    mk = (lambda *s: torch.zeros(*s, dtype=torch.float64).pin_memory()) if host else (lambda *s: torch.zeros(*s, dtype=torch.float64, device="cuda"))
    cl = []
    for s in specs:
        x = make_cluster(s)
        cl.append(dict(nao=s.nao, nocc=s.nocc, nvir=s.nvir, naux=s.naux, C_occ=to(x.C_occ), C_vir=to(x.C_vir),
                       L_packed=to(x.L_packed(threads=4)), e_occ=to(x.e_occ), e_vir=to(x.e_vir),
                       P_frag=None if s.rank <= 0 else to(x.P_frag), E_out=mk(1), G_out=mk(s.nocc, s.nocc)))
    need = sie.sie_dfmp2_batch_query(cl, flags)
    ws = sie.alloc_workspace(need)
    sie.sie_dfmp2_batch(cl, ws, flags)
    torch.cuda.synchronize()
    return [(float(c["E_out"].cpu()[0]), c["G_out"].cpu().numpy()) for c in cl]


@pytest.mark.parametrize("flags", [0, binding.SIE_FLAG_HOST_IO], ids=["device", "host_io"])
def test_batch_of_variable_clusters(flags):
    shapes = [(16, 128, 576), (9, 30, 50), (40, 90, 130), (31, 64, 257), (48, 100, 96), (120, 130, 64), (3, 7, 9)]
    specs = [ClusterSpec(60, k, o + v, o, v, naux, 0 if k == 2 else max(1, o // 4), "std") for k, (o, v, naux) in enumerate(shapes)]
    res = _batch_run(specs, flags)
    for s, (E, G) in zip(specs, res):
        check(s, E, G)
    # a batch gives the same bits as the single-cluster calls only up to the schedule; check it is reproducible
    res2 = _batch_run(specs, flags)
    for (E, G), (E2, G2) in zip(res, res2):
        assert E == E2 and np.array_equal(G, G2)


def test_config2_first_clusters():
    specs = config_specs(2)[:5]
    res = _batch_run(specs)
    for s, (E, G) in zip(specs, res):
        check(s, E, G)


def test_batch_empty_and_reference_flag():
    sie.sie_dfmp2_batch([], sie.alloc_workspace(256))
    specs = [ClusterSpec(61, k, o + v, o, v, naux, 2, "std") for k, (o, v, naux) in enumerate([(6, 20, 30), (10, 12, 17)])]
    for s, (E, G) in zip(specs, _batch_run(specs, binding.SIE_FLAG_REFERENCE)):
        check(s, E, G)


# ---------------------------------------------------------------------------------------------- API behaviour
def test_call_order_and_validation_errors():
    spec = ClusterSpec(53, 0, 30, 4, 26, 20, 2, "std")
    x = make_cluster(spec)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux, flags=binding.SIE_FLAG_VALIDATE)
    C_occ, C_vir, L = cu(x.C_occ), cu(x.C_vir), cu(x.L_packed())
    with pytest.raises(sie.SieError) as ei:
        s.energy(cu(x.e_occ), cu(x.e_vir))
    assert ei.value.status == binding.SIE_ESTATE
    s.transform(C_occ, C_vir, L[:12], 0, 12)
    with pytest.raises(sie.SieError) as ei:
        s.transform(C_occ, C_vir, L[8:], 8, 20)  # overlaps [0,12)
    assert ei.value.status == binding.SIE_EINVAL
    with pytest.raises(sie.SieError) as ei:
        s.energy(cu(x.e_occ), cu(x.e_vir))  # [12,20) still missing
    assert ei.value.status == binding.SIE_ESTATE
    s.transform(C_occ, C_vir, L[12:], 12, 20)
    bad = x.e_vir.copy()
    bad[3] = -1.0  # below max(e_occ): the gap requirement of Eq. S16 is violated
    with pytest.raises(sie.SieError) as ei:
        s.energy(cu(x.e_occ), cu(bad))
    assert ei.value.status == binding.SIE_EGAP
    E, G = s.energy(cu(x.e_occ), cu(x.e_vir), cu(x.P_frag))
    check(spec, float(E.cpu()[0]), G.cpu().numpy())
    with pytest.raises(TypeError):
        s.transform(C_occ.cpu(), C_vir, L, 0, 20)  # host tensor without SIE_FLAG_HOST_IO
    s.close()


def test_energy_can_be_recomputed_with_other_energies_and_projector():
    spec = ClusterSpec(54, 0, 40, 6, 34, 33, 3, "std")
    x = make_cluster(spec)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux)
    s.transform(cu(x.C_occ), cu(x.C_vir), cu(x.L_packed()), 0, spec.naux)
    B = oracle.transform(x.C_occ, x.C_vir, x.L_packed())
    for shift, P in ((0.0, x.P_frag), (0.0, None), (-0.4, x.P_frag.T.copy())):
        eo = x.e_occ + shift
        E, G = s.energy(cu(eo), cu(x.e_vir), None if P is None else cu(P))
        Gor = oracle.pair_G(B, eo, x.e_vir)
        assert np.max(np.abs(G.cpu().numpy() - Gor)) <= G_ATOL
        Eor = oracle.trace(P, Gor)
        assert abs(float(E.cpu()[0]) - Eor) <= E_RTOL * abs(Eor)
    s.close()


def test_launch_counter_counts_our_kernels():
    before = sie.launch_count()
    spec = config_specs(0, "std")[0]
    gpu_run(spec)
    assert sie.launch_count() - before >= 5  # coefficient transposes, A1, A2, pair, reduce


def test_host_io_whole_tensor_staging_and_two_plans_on_two_streams():
    """SIE_FLAG_STAGE_FULL: the packed tensor is staged whole; two plans on two streams, the transform of the second
    enqueued before the energy of the first (the software pipeline of bench.py's e2e arm) give the device-path results."""
    specs = [ClusterSpec(60, k, 70, 10, 60, 90, 3, "std") for k in range(2)]
    xs = [make_cluster(s) for s in specs]
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()  # noqa: E731
    fl = binding.SIE_FLAG_HOST_IO | binding.SIE_FLAG_STAGE_FULL
    solvers = [sie.ClusterSolver(s.nao, s.nocc, s.nvir, s.naux, aux_block=32, flags=fl) for s in specs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    hs = [dict(C_occ=pin(x.C_occ), C_vir=pin(x.C_vir), L=pin(x.L_packed()), e_occ=pin(x.e_occ), e_vir=pin(x.e_vir), P=pin(x.P_frag)) for x in xs]
    solvers[0].transform(hs[0]["C_occ"], hs[0]["C_vir"], hs[0]["L"], 0, specs[0].naux, stream=streams[0])
    solvers[1].transform(hs[1]["C_occ"], hs[1]["C_vir"], hs[1]["L"], 0, specs[1].naux, stream=streams[1])
    out = [solvers[k].energy(hs[k]["e_occ"], hs[k]["e_vir"], hs[k]["P"], stream=streams[k]) for k in range(2)]
    torch.cuda.synchronize()
    for k in range(2):
        check(specs[k], float(out[k][0][0]), out[k][1].numpy())
        solvers[k].close()
    with pytest.raises(sie.SieError):  # the flag needs SIE_FLAG_HOST_IO
        sie.sie_dfmp2_plan(70, 10, 60, 90, 0, binding.SIE_FLAG_STAGE_FULL)
