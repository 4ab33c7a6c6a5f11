"""sie_dfmp2_energy_noalloc: the pair stage + trace with the library's static device scratch (no workspace, no device
allocation) against the existing workspace path, on two calls in a row, and against the CPU oracle.

The two paths launch the same kernels on the same B in the same tile order with the same fixed-order reduction, so the
results must agree bit for bit; the assertion is the tolerance every parity test here uses (E 1e-10 relative, G
1e-11 * max(1, max|G|)), and bit-equality is checked on top.  The static array keeps the previous call's contents:
the second call runs another cluster shape in between and must still reproduce the first result.

Collected last on purpose (the run uses pytest -x); passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_18553_b200 as sie
from paper_2412_18553_b200 import binding
from workloads import ClusterSpec, make_cluster

pytestmark = pytest.mark.gpu

E_RTOL = 1e-10
G_ATOL = 1e-11


def _cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _existing_path(spec, x):
    """sie_dfmp2_plan / _transform / _energy with a caller-provided workspace; returns (E, G, B view of the workspace, solver)."""
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux)
    s.transform(_cu(x.C_occ), _cu(x.C_vir), _cu(x.L_packed(threads=4)), 0, spec.naux)
    E, G = s.energy(_cu(x.e_occ), _cu(x.e_vir), _cu(x.P_frag))
    torch.cuda.synchronize()
    naux_ld = (spec.naux + 7) // 8 * 8
    B = s.workspace[: spec.nvir * spec.nocc * naux_ld * 8]  # B[a][i][P] is the first region of the workspace
    return E, G, B, s


def _noalloc(spec, x, B, P=True):
    E = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    G = torch.full((spec.nocc, spec.nocc), float("nan"), dtype=torch.float64, device="cuda")
    sie.sie_dfmp2_energy_noalloc(spec.nocc, spec.nvir, spec.naux, B, _cu(x.e_occ), _cu(x.e_vir), _cu(x.P_frag) if P else None, E, G)
    torch.cuda.synchronize()
    return E, G


def _assert_close(E, G, Eref, Gref):
    Eref_f = float(Eref.cpu()[0])
    assert abs(float(E.cpu()[0]) - Eref_f) <= E_RTOL * abs(Eref_f)
    Gh, Gr = G.cpu().numpy(), Gref.cpu().numpy()
    assert np.max(np.abs(Gh - Gr)) <= G_ATOL * max(1.0, float(np.max(np.abs(Gr))))


@pytest.mark.parametrize("o,v,naux", [(24, 150, 203), (120, 140, 200), (8, 40, 160)])
def test_noalloc_matches_the_workspace_path_on_two_calls_in_a_row(o, v, naux):
    spec = ClusterSpec(90, o, o + v, o, v, naux, max(1, o // 3), "std")
    x = make_cluster(spec)
    Eref, Gref, B, solver = _existing_path(spec, x)
    E1, G1 = _noalloc(spec, x, B)
    _assert_close(E1, G1, Eref, Gref)
    assert torch.equal(E1, Eref) and torch.equal(G1, Gref)  # same kernels, same order: identical bits
    # another shape through the same static array in between, then the first cluster again: stale contents must not leak
    other = ClusterSpec(90, 1000 + o, 17 + 60, 17, 60, 45, 5, "std")
    xo = make_cluster(other)
    Eo_ref, Go_ref, Bo, so = _existing_path(other, xo)
    Eo, Go = _noalloc(other, xo, Bo)
    _assert_close(Eo, Go, Eo_ref, Go_ref)
    so.close()
    E2, G2 = _noalloc(spec, x, B)
    _assert_close(E2, G2, Eref, Gref)
    assert torch.equal(E2, E1) and torch.equal(G2, G1)
    del E1, G1, E2, G2, Eo, Go
    # and the oracle, element by element
    Gor = oracle.pair_G(oracle.transform(x.C_occ, x.C_vir, x.L_packed(threads=4)), x.e_occ, x.e_vir)
    Eor = oracle.trace(x.P_frag, Gor)
    assert abs(float(Eref.cpu()[0]) - Eor) <= E_RTOL * abs(Eor)
    assert np.max(np.abs(Gref.cpu().numpy() - Gor)) <= G_ATOL * max(1.0, float(np.max(np.abs(Gor))))
    # identity projector through a NULL pointer
    EI, GI = _noalloc(spec, x, B, P=False)
    EI_ref, _ = solver.energy(_cu(x.e_occ), _cu(x.e_vir), None)
    torch.cuda.synchronize()
    assert torch.equal(EI, EI_ref) and torch.equal(GI, Gref)
    solver.close()


def test_noalloc_limits_are_reported_not_overrun():
    cap = sie.sie_dfmp2_noalloc_capacity()
    assert cap == 24 << 20
    assert 0 < sie.sie_dfmp2_noalloc_bytes(120, 1080) <= cap  # BASELINE config 3 fits
    assert sie.sie_dfmp2_noalloc_bytes(128, 2000) > cap and sie.sie_dfmp2_noalloc_bytes(130, 20) == 0
    dummy = torch.zeros(1024, dtype=torch.float64, device="cuda")
    E = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(sie.SieError) as ei:  # too large for the static scratch: refused before anything is enqueued
        sie.sie_dfmp2_energy_noalloc(128, 2000, 64, dummy, dummy, dummy, None, E, None)
    assert ei.value.status == binding.SIE_ETOOBIG and "static scratch" in str(ei.value)
    with pytest.raises(sie.SieError) as ei:  # nocc > 128: not the fused route
        sie.sie_dfmp2_energy_noalloc(130, 20, 64, dummy, dummy, dummy, None, E, None)
    assert ei.value.status == binding.SIE_EUNSUPPORTED
    torch.cuda.synchronize()
    assert float(E.cpu()[0]) == 7.0  # outputs untouched on error
