"""GPU parity of sie_dfmp2_rdm_occ (NEXT-1: occupied block of the MP2 1-RDM, PAPER.md Eq. S18) against oracle.rdm_occ,
element by element on the same seeded inputs.  Tolerance: |d gamma| <= 1e-11 * max(1, max|gamma|) (gamma = 2 - 2 Gamma;
under the literal variance-1/nao inputs |Gamma| reaches 1e3..1e5, under std-1/nao it is ~1e-2 and the bar is literal)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_18553_b200 as sie
from paper_2412_18553_b200 import binding
from workloads import ClusterSpec, config_specs, make_cluster

pytestmark = pytest.mark.gpu
ATOL = 1e-11


def _run(spec, flags=0, energy_too=False):
    x = make_cluster(spec)
    host = bool(flags & binding.SIE_FLAG_HOST_IO)
    to = (lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()) if host else (lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda())
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux, flags=flags)
    s.transform(to(x.C_occ), to(x.C_vir), to(x.L_packed(threads=4)), 0, spec.naux)
    e_occ, e_vir = to(x.e_occ), to(x.e_vir)
    out = {}
    if energy_too:
        E0, G0 = s.energy(e_occ, e_vir, None)
    g, tr = s.rdm_occ(e_occ, e_vir)
    if energy_too:  # the two entry points share the workspace and must not disturb each other
        E1, G1 = s.energy(e_occ, e_vir, None)
        torch.cuda.synchronize()
        assert torch.equal(G0, G1) and torch.equal(E0, E1)
    torch.cuda.synchronize()
    out = g.cpu().numpy(), float(tr.cpu()[0])
    s.close()
    return x, out


def _check(spec, flags=0, energy_too=False):
    x, (g, tr) = _run(spec, flags, energy_too)
    gor = oracle.rdm_occ(oracle.transform(x.C_occ, x.C_vir, x.L_packed(threads=4)), x.e_occ, x.e_vir)
    scale = max(1.0, float(np.max(np.abs(gor))))
    assert np.max(np.abs(g - gor)) <= ATOL * scale, (float(np.max(np.abs(g - gor))), scale)
    assert abs(tr - np.trace(gor)) <= 1e-10 * max(1.0, abs(np.trace(gor)))
    assert np.max(np.abs(g - g.T)) <= 1e-11 * scale
    return g


@pytest.mark.parametrize("scale", ["var", "std"])
@pytest.mark.parametrize("flags", [0, binding.SIE_FLAG_REFERENCE], ids=["dmma", "reference"])
def test_config0(scale, flags):
    _check(config_specs(0, scale)[0], flags)


@pytest.mark.parametrize("scale", ["var", "std"])
def test_config1(scale):
    g = _check(config_specs(1, scale)[0], energy_too=True)
    if scale == "std":  # physically sized amplitudes: occupations stay within [0, 2]
        w = np.linalg.eigvalsh((g + g.T) / 2)
        assert w.min() > 0.0 and w.max() <= 2.0 + 1e-12


@pytest.mark.parametrize("nocc,nvir,extra,naux", [(1, 1, 0, 1), (5, 13, 5, 37), (17, 50, 3, 100), (30, 41, 0, 88), (33, 70, 1, 129),
                                                  (64, 96, 0, 200), (72, 75, 0, 90), (120, 140, 0, 200), (128, 130, 4, 72), (2, 70, 0, 24)])
def test_ragged_shapes(nocc, nvir, extra, naux):
    _check(ClusterSpec(55, nocc * 1000 + nvir, nocc + nvir + extra, nocc, nvir, naux, 1, "std"))


def test_host_io_and_nocc_above_128():
    _check(ClusterSpec(56, 0, 24 + 60, 24, 60, 50, 1, "std"), binding.SIE_FLAG_HOST_IO)
    _check(ClusterSpec(56, 1, 130 + 20, 130, 20, 24, 1, "std"))  # general route (nocc > 128)


def test_closed_form_o1_v1_on_gpu():
    spec = ClusterSpec(57, 0, 2, 1, 1, 9, 1, "std")
    x, (g, tr) = _run(spec)
    B = oracle.transform(x.C_occ, x.C_vir, x.L_packed())
    t = float(np.sum(B * B)) / (2 * x.e_occ[0] - 2 * x.e_vir[0])
    assert g[0, 0] == pytest.approx(2.0 - 2.0 * t * t, rel=1e-13) and tr == pytest.approx(g[0, 0], rel=1e-15)


@pytest.mark.parametrize("flags", [0, binding.SIE_FLAG_HOST_IO, binding.SIE_FLAG_REFERENCE], ids=["device", "host_io", "reference"])
def test_batch_with_rdm_flag(flags):
    """sie_dfmp2_batch(..., SIE_FLAG_RDM_OCC): gamma of every cluster in G_out, Tr gamma in E_out."""
    specs = [ClusterSpec(58, k, o + v, o, v, naux, 1, "std") for k, (o, v, naux) in enumerate([(16, 128, 100), (7, 30, 41), (33, 64, 72), (24, 50, 90)])]
    host = bool(flags & binding.SIE_FLAG_HOST_IO)
    to = (lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()) if host else (lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda())
    mk = (lambda *sh: torch.zeros(*sh, dtype=torch.float64).pin_memory()) if host else (lambda *sh: torch.zeros(*sh, dtype=torch.float64, device="cuda"))
    xs, cl = [], []
    for sp in specs:
        x = make_cluster(sp)
        xs.append(x)
        cl.append(dict(nao=sp.nao, nocc=sp.nocc, nvir=sp.nvir, naux=sp.naux, C_occ=to(x.C_occ), C_vir=to(x.C_vir), L_packed=to(x.L_packed()),
                       e_occ=to(x.e_occ), e_vir=to(x.e_vir), P_frag=to(x.P_frag), E_out=mk(1), G_out=mk(sp.nocc, sp.nocc)))
    fl = flags | binding.SIE_FLAG_RDM_OCC
    ws = sie.alloc_workspace(sie.sie_dfmp2_batch_query(cl, fl))
    sie.sie_dfmp2_batch(cl, ws, fl)
    torch.cuda.synchronize()
    for x, c in zip(xs, cl):
        gor = oracle.rdm_occ(oracle.transform(x.C_occ, x.C_vir, x.L_packed()), x.e_occ, x.e_vir)
        g = c["G_out"].cpu().numpy()
        assert np.max(np.abs(g - gor)) <= ATOL * max(1.0, float(np.max(np.abs(gor))))
        assert abs(float(c["E_out"].cpu()[0]) - np.trace(gor)) <= 1e-10 * max(1.0, abs(np.trace(gor)))
