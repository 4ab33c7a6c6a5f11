"""GPU parity of the any-size pair-stage route (csrc/general.cu) against the CPU oracle, element by element:

  * nocc > 128 — the environment-occupied x impurity-virtual sub-space shape of PAPER.md Eq. S13 (L338): energy, G and
    gamma_occ (Eq. S18) through the slab GEMM / amplitude pass / split-K Gram GEMM route (plan_info route == 2);
  * gamma_vir (Eq. S17) at every size (small-occ x large-vir of Eq. S14 and the mirrored shape), plans created
    with SIE_FLAG_RDM_VIR;
  * Tr gamma_occ + Tr gamma_vir = 2 nocc on the GPU, call-order / flag errors, a batch that mixes routes.

Tolerances as everywhere: E 1e-10 relative; matrices 1e-11 * max(1, max|oracle|) (inputs scale="std" unless stated).
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_18553_b200 as sie
from paper_2412_18553_b200 import binding
from workloads import ClusterSpec, config_specs, make_cluster

pytestmark = pytest.mark.gpu
ATOL = 1e-11


def _cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _solve(spec, flags=0, blocks=None, want=("E", "occ", "vir")):
    x = make_cluster(spec)
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux, flags=flags)
    info = s.info()
    C_occ, C_vir = _cu(x.C_occ), _cu(x.C_vir)
    for p0, p1 in (blocks or [(0, spec.naux)]):
        s.transform(C_occ, C_vir, _cu(x.L_block(p0, p1, threads=4)), p0, p1)
    e_occ, e_vir = _cu(x.e_occ), _cu(x.e_vir)
    out = {}
    if "E" in want:
        E, G = s.energy(e_occ, e_vir, None if spec.rank <= 0 else _cu(x.P_frag))
        out["E"], out["G"] = E, G
    if "occ" in want:
        out["occ"], out["tr_occ"] = s.rdm_occ(e_occ, e_vir)
    if "vir" in want:
        out["vir"], out["tr_vir"] = s.rdm_vir(e_occ, e_vir)
    torch.cuda.synchronize()
    out = {k: (v.cpu().numpy() if v.numel() > 1 else float(v.cpu()[0])) for k, v in out.items()}
    s.close()
    return x, info, out


def _close(got, ref):
    scale = max(1.0, float(np.max(np.abs(ref))))
    err = float(np.max(np.abs(got - ref)))
    assert err <= ATOL * scale, (err, scale)


def _oracle_B(x):
    return oracle.transform(x.C_occ, x.C_vir, x.L_packed(threads=4))


@pytest.mark.parametrize("o,v,extra,naux,rank", [(130, 20, 0, 24, 10), (200, 24, 0, 64, 0), (144, 40, 5, 91, 30), (257, 9, 0, 40, 7),
                                                  (136, 64, 0, 33, 17)])
def test_general_route_energy_G_and_both_rdm_blocks(o, v, extra, naux, rank):
    spec = ClusterSpec(80, o, o + v + extra, o, v, naux, rank, "std")
    cuts = sorted({0, naux // 2, naux})
    blocks = [(cuts[i], cuts[i + 1]) for i in range(len(cuts) - 1)][::-1]
    x, info, out = _solve(spec, flags=binding.SIE_FLAG_RDM_VIR, blocks=blocks)
    assert info["general"] == 1 and info["reference"] == 0
    B = _oracle_B(x)
    Gor = oracle.pair_G(B, x.e_occ, x.e_vir)
    Eor = oracle.trace(None if rank <= 0 else x.P_frag, Gor)
    assert abs(out["E"] - Eor) <= 1e-10 * abs(Eor), (out["E"], Eor)
    _close(out["G"], Gor)
    gocc, gvir = oracle.rdm_occ(B, x.e_occ, x.e_vir), oracle.rdm_vir(B, x.e_occ, x.e_vir)
    _close(out["occ"], gocc)
    _close(out["vir"], gvir)
    assert abs(out["tr_occ"] - np.trace(gocc)) <= 1e-10 * abs(np.trace(gocc))
    assert abs(out["tr_vir"] - np.trace(gvir)) <= 1e-10 * max(1.0, abs(np.trace(gvir)))
    assert abs(out["tr_occ"] + out["tr_vir"] - 2.0 * o) <= 1e-10 * 2.0 * o  # electron count conserved (pin of O9, on the GPU)


@pytest.mark.parametrize("scale", ["var", "std"])
def test_rdm_vir_config0(scale):
    spec = config_specs(0, scale)[0]
    x, info, out = _solve(spec, flags=binding.SIE_FLAG_RDM_VIR)
    assert info["general"] == 0  # fused route for the energy, general route only for gamma_vir
    B = _oracle_B(x)
    _close(out["vir"], oracle.rdm_vir(B, x.e_occ, x.e_vir))
    _close(out["occ"], oracle.rdm_occ(B, x.e_occ, x.e_vir))
    Gor = oracle.pair_G(B, x.e_occ, x.e_vir)
    assert abs(out["E"] - oracle.trace(x.P_frag, Gor)) <= 1e-10 * abs(oracle.trace(x.P_frag, Gor))


@pytest.mark.parametrize("o,v,extra,naux", [(4, 150, 0, 60), (30, 100, 0, 200), (17, 129, 3, 75), (1, 40, 0, 16), (64, 65, 0, 50), (9, 8, 0, 5)])
def test_rdm_vir_small_occ_large_vir_shapes(o, v, extra, naux):
    """The impurity-occupied x environment-virtual shape of Eq. S14 and ragged sizes (v not a multiple of 8 or 128,
    occupied blocks with a ragged tail, nocc + nvir < nao)."""
    spec = ClusterSpec(81, o, o + v + extra, o, v, naux, 0, "std")
    x, info, out = _solve(spec, flags=binding.SIE_FLAG_RDM_VIR, want=("vir", "occ"))
    B = _oracle_B(x)
    gvir = oracle.rdm_vir(B, x.e_occ, x.e_vir)
    _close(out["vir"], gvir)
    assert np.max(np.abs(out["vir"] - out["vir"].T)) <= ATOL * max(1.0, float(np.max(np.abs(gvir))))
    assert abs(out["tr_occ"] + out["tr_vir"] - 2.0 * o) <= 1e-10 * 2.0 * o


def test_rdm_vir_needs_the_plan_flag_and_host_io_works():
    spec = ClusterSpec(82, 0, 50, 6, 44, 30, 0, "std")
    x = make_cluster(spec)
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux)  # no SIE_FLAG_RDM_VIR
    s.transform(_cu(x.C_occ), _cu(x.C_vir), _cu(x.L_packed()), 0, spec.naux)
    with pytest.raises(sie.SieError) as ei:
        s.rdm_vir(_cu(x.e_occ), _cu(x.e_vir))
    assert ei.value.status == binding.SIE_ESTATE
    s.close()
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()  # noqa: E731
    h = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux, flags=binding.SIE_FLAG_HOST_IO | binding.SIE_FLAG_RDM_VIR)
    h.transform(pin(x.C_occ), pin(x.C_vir), pin(x.L_packed()), 0, spec.naux)
    g, tr = h.rdm_vir(pin(x.e_occ), pin(x.e_vir))
    gor = oracle.rdm_vir(_oracle_B(x), x.e_occ, x.e_vir)
    _close(g.numpy(), gor)
    assert abs(float(tr[0]) - np.trace(gor)) <= 1e-10 * max(1.0, abs(np.trace(gor)))
    h.close()


def test_batch_mixes_fused_and_general_clusters():
    shapes = [(16, 40, 50), (150, 12, 40), (33, 64, 72), (129, 20, 24)]
    specs = [ClusterSpec(83, k, o + v, o, v, naux, max(1, o // 4), "std") for k, (o, v, naux) in enumerate(shapes)]
    cl, xs = [], []
    for sp in specs:
        x = make_cluster(sp)
        xs.append(x)
        cl.append(dict(nao=sp.nao, nocc=sp.nocc, nvir=sp.nvir, naux=sp.naux, C_occ=_cu(x.C_occ), C_vir=_cu(x.C_vir), L_packed=_cu(x.L_packed()),
                       e_occ=_cu(x.e_occ), e_vir=_cu(x.e_vir), P_frag=_cu(x.P_frag), E_out=torch.zeros(1, dtype=torch.float64, device="cuda"),
                       G_out=torch.zeros(sp.nocc, sp.nocc, dtype=torch.float64, device="cuda")))
    ws = sie.alloc_workspace(sie.sie_dfmp2_batch_query(cl))
    sie.sie_dfmp2_batch(cl, ws)
    torch.cuda.synchronize()
    for sp, x, c in zip(specs, xs, cl):
        Gor = oracle.pair_G(_oracle_B(x), x.e_occ, x.e_vir)
        Eor = oracle.trace(x.P_frag, Gor)
        assert abs(float(c["E_out"].cpu()[0]) - Eor) <= 1e-10 * abs(Eor), sp
        _close(c["G_out"].cpu().numpy(), Gor)


def test_batch_clusters_sharing_one_integral_tensor():
    """Clusters of one system: different orbital sets C over the SAME (P|mu nu).  Passing one L_packed
    tensor for several batch members makes the library transform them together (one A1 GEMM over the stacked occupied
    columns); results must equal the oracle run on each cluster separately."""
    nao, naux = 96, 70
    shapes = [(12, 60), (30, 66), (7, 40), (20, 70)]
    base = make_cluster(ClusterSpec(84, 99, nao, 8, 8, naux, 0, "std"))
    Lh = base.L_packed()
    L = _cu(Lh)
    cl, xs = [], []
    for k, (o, v) in enumerate(shapes):
        sp = ClusterSpec(84, k, nao, o, v, naux, max(1, o // 3), "std")
        x = make_cluster(sp)
        xs.append(x)
        cl.append(dict(nao=nao, nocc=o, nvir=v, naux=naux, C_occ=_cu(x.C_occ), C_vir=_cu(x.C_vir), L_packed=L, e_occ=_cu(x.e_occ),
                       e_vir=_cu(x.e_vir), P_frag=_cu(x.P_frag), E_out=torch.zeros(1, dtype=torch.float64, device="cuda"),
                       G_out=torch.zeros(o, o, dtype=torch.float64, device="cuda")))
    # one extra member with its own integrals in the same batch
    own = make_cluster(ClusterSpec(84, 50, 40, 6, 30, 33, 2, "std"))
    cl.append(dict(nao=40, nocc=6, nvir=30, naux=33, C_occ=_cu(own.C_occ), C_vir=_cu(own.C_vir), L_packed=_cu(own.L_packed()),
                   e_occ=_cu(own.e_occ), e_vir=_cu(own.e_vir), P_frag=_cu(own.P_frag), E_out=torch.zeros(1, dtype=torch.float64, device="cuda"),
                   G_out=torch.zeros(6, 6, dtype=torch.float64, device="cuda")))
    ws = sie.alloc_workspace(sie.sie_dfmp2_batch_query(cl))  # the query sees the shared tensor: same layout as the call
    l0 = sie.launch_count()
    sie.sie_dfmp2_batch(cl, ws)
    torch.cuda.synchronize()
    assert sie.launch_count() - l0 == 5  # transposes, A1, A2, pair, reduce: the whole batch
    for x, c, Lx in list(zip(xs, cl, [Lh] * 4)) + [(own, cl[-1], own.L_packed())]:
        Gor = oracle.pair_G(oracle.transform(x.C_occ, x.C_vir, Lx), x.e_occ, x.e_vir)
        Eor = oracle.trace(x.P_frag, Gor)
        assert abs(float(c["E_out"].cpu()[0]) - Eor) <= 1e-10 * abs(Eor)
        _close(c["G_out"].cpu().numpy(), Gor)


@pytest.mark.parametrize("o,v,naux,r", [(8, 40, 160, 4), (30, 100, 120, 15), (17, 60, 75, 4), (120, 130, 64, 8), (120, 125, 40, 32),
                                         (120, 125, 40, 33), (33, 70, 50, 1), (64, 96, 100, 32), (5, 9, 7, 5), (128, 130, 24, 17)])
def test_energy_lowrank_matches_oracle_trace(o, v, naux, r):
    """NEXT-3: E_frag = Tr(Q Q^T G) through the project-first epilogue (r <= 32) and its fallback (r > 32)."""
    spec = ClusterSpec(85, o * 1000 + r, o + v, o, v, naux, r, "std")
    x = make_cluster(spec)
    s = sie.ClusterSolver(spec.nao, o, v, naux)
    s.transform(_cu(x.C_occ), _cu(x.C_vir), _cu(x.L_packed(threads=4)), 0, naux)
    e_occ, e_vir = _cu(x.e_occ), _cu(x.e_vir)
    E_lr = s.energy_lowrank(e_occ, e_vir, _cu(x.Q_frag))
    E_full, _ = s.energy(e_occ, e_vir, _cu(x.P_frag))  # the two entry points share the workspace
    E_lr2 = s.energy_lowrank(e_occ, e_vir, _cu(x.Q_frag))
    torch.cuda.synchronize()
    assert torch.equal(E_lr, E_lr2)  # fixed-order reduction of the per-warp partials
    Gor = oracle.pair_G(_oracle_B(x), x.e_occ, x.e_vir)
    Eor = oracle.trace(x.Q_frag @ x.Q_frag.T, Gor)
    assert abs(float(E_lr.cpu()[0]) - Eor) <= 1e-10 * abs(Eor), (float(E_lr.cpu()[0]), Eor)
    assert abs(float(E_full.cpu()[0]) - Eor) <= 1e-10 * abs(Eor)
    s.close()


def test_energy_lowrank_host_io_and_unsupported_route():
    spec = ClusterSpec(85, 7, 60, 10, 50, 40, 3, "std")
    x = make_cluster(spec)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()  # noqa: E731
    h = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux, flags=binding.SIE_FLAG_HOST_IO)
    h.transform(pin(x.C_occ), pin(x.C_vir), pin(x.L_packed()), 0, spec.naux)
    E = h.energy_lowrank(pin(x.e_occ), pin(x.e_vir), pin(x.Q_frag))
    Eor = oracle.trace(x.P_frag, oracle.pair_G(_oracle_B(x), x.e_occ, x.e_vir))
    assert abs(float(E[0]) - Eor) <= 1e-10 * abs(Eor)
    h.close()
    big = ClusterSpec(85, 8, 150, 130, 20, 16, 2, "std")  # general route: not supported, loudly
    xb = make_cluster(big)
    g = sie.ClusterSolver(big.nao, big.nocc, big.nvir, big.naux)
    g.transform(_cu(xb.C_occ), _cu(xb.C_vir), _cu(xb.L_packed()), 0, big.naux)
    with pytest.raises(sie.SieError) as ei:
        g.energy_lowrank(_cu(xb.e_occ), _cu(xb.e_vir), _cu(xb.Q_frag))
    assert ei.value.status == binding.SIE_EUNSUPPORTED
    g.close()


@pytest.mark.parametrize("o,v,extra,naux,occ_block,store", [(8, 40, 0, 160, 0, "device"), (8, 40, 0, 160, 3, "host"), (37, 50, 4, 61, 8, "host"),
                                                          (150, 24, 0, 40, 64, "host"), (130, 9, 0, 33, 7, "device"), (5, 130, 0, 20, 2, "host")])
def test_canonical_out_of_core_energy_matches_oracle(o, v, extra, naux, occ_block, store):
    """NEXT-2: E_MP2 = sum_ij e_ij (P = I) through the occupied-block-pair route with the B store in pinned host memory
    (panels streamed back, ragged last block, nocc > 128) or in device memory; the oracle is its pinned P = I case (pin P-2)."""
    spec = ClusterSpec(86, o * 100 + occ_block, o + v + extra, o, v, naux, 0, "std")
    x = make_cluster(spec)
    s = sie.CanonicalSolver(spec.nao, o, v, naux, occ_block=occ_block, store=store)
    info = s.info()
    if occ_block:
        assert info["occ_block"] == min(occ_block, o) and info["n_occ_blocks"] == -(-o // min(occ_block, o))
    C_occ, C_vir = _cu(x.C_occ), _cu(x.C_vir)
    cuts = sorted({0, naux // 3, naux})
    for p0, p1 in [(cuts[i], cuts[i + 1]) for i in range(len(cuts) - 1)][::-1]:  # aux blocks, out of order
        s.transform(C_occ, C_vir, _cu(x.L_block(p0, p1)), p0, p1)
    E1 = s.energy(_cu(x.e_occ), _cu(x.e_vir))
    E2 = s.energy(_cu(x.e_occ), _cu(x.e_vir))
    torch.cuda.synchronize()
    assert torch.equal(E1, E2)  # fixed-order slot sums
    B = _oracle_B(x)
    Eor = oracle.trace(None, oracle.pair_G(B, x.e_occ, x.e_vir))
    assert abs(float(E1.cpu()[0]) - Eor) <= 1e-10 * abs(Eor), (float(E1.cpu()[0]), Eor)
    # the store itself, element by element: B[i][a][P]
    naux_ld = (naux + 7) // 8 * 8
    Bs = s.B_store.cpu().numpy().reshape(o, v, naux_ld)[:, :, :naux]
    assert np.max(np.abs(Bs - B)) <= 1e-13 * max(1.0, float(np.max(np.abs(B))))
    s.close()


def test_canonical_call_order():
    s = sie.CanonicalSolver(20, 4, 16, 12, store="device")
    with pytest.raises(sie.SieError) as ei:
        s.energy(torch.zeros(4, dtype=torch.float64, device="cuda"), torch.ones(16, dtype=torch.float64, device="cuda"))
    assert ei.value.status == binding.SIE_ESTATE
    s.close()


def test_general_route_block_slab_mode_large_integral_matrix():
    """(o, v) = (129, 260): the integral matrix (o v)^2 doubles is 9 GB, above the whole-matrix SYRK limit, so the general
    route runs its block-slab mode (power-of-two occupied blocks, 3-D tensor map for the column operand, ragged last
    block).  E, G and gamma_occ against the oracle (its O6 loop is ~1e11 long-double operations: the slow test of this file)."""
    o, v, naux = 129, 260, 16
    spec = ClusterSpec(87, 0, o + v, o, v, naux, 40, "std")
    x, info, out = _solve(spec, want=("E", "occ"))
    assert info["general"] == 1
    B = _oracle_B(x)
    Gor = oracle.pair_G(B, x.e_occ, x.e_vir)
    Eor = oracle.trace(x.P_frag, Gor)
    assert abs(out["E"] - Eor) <= 1e-10 * abs(Eor)
    _close(out["G"], Gor)
    _close(out["occ"], oracle.rdm_occ(B, x.e_occ, x.e_vir))


def test_degenerate_sizes_of_the_next_rows():
    """o = v = 1 closed forms through every route that has one (PAPER.md Eq. S15-S18 with a single amplitude t):
    E = (ia|ia)^2 / (2 (e_i - e_a)), gamma_occ = 2 - 2 t^2, gamma_vir = 2 t^2; naux = 1; a one-row, one-column projector."""
    rng = np.random.default_rng(11)
    for naux in (1, 5):
        spec = ClusterSpec(88, naux, 2, 1, 1, naux, 0, "std")
        x = make_cluster(spec)
        Lp = x.L_packed()
        Bv = oracle.transform(x.C_occ, x.C_vir, Lp)[0, 0]
        iaia = float(np.sum(Bv * Bv))
        ei, ea = float(x.e_occ[0]), float(x.e_vir[0])
        t = iaia / (2 * ei - 2 * ea)
        s = sie.ClusterSolver(2, 1, 1, naux, flags=binding.SIE_FLAG_RDM_VIR)
        s.transform(_cu(x.C_occ), _cu(x.C_vir), _cu(Lp), 0, naux)
        e_occ, e_vir = _cu(x.e_occ), _cu(x.e_vir)
        E, G = s.energy(e_occ, e_vir, None)
        El = s.energy_lowrank(e_occ, e_vir, _cu(np.ones((1, 1))))
        go, _ = s.rdm_occ(e_occ, e_vir)
        gv, _ = s.rdm_vir(e_occ, e_vir)
        torch.cuda.synchronize()
        Ecf = iaia * iaia / (2 * (ei - ea))
        for got in (float(E.cpu()[0]), float(El.cpu()[0]), float(G.cpu()[0, 0])):
            assert abs(got - Ecf) <= 1e-12 * abs(Ecf)
        assert abs(float(go.cpu()[0, 0]) - (2 - 2 * t * t)) <= 1e-13 and abs(float(gv.cpu()[0, 0]) - 2 * t * t) <= 1e-13 * max(1.0, 2 * t * t)
        s.close()
        c = sie.CanonicalSolver(2, 1, 1, naux, store="device")
        c.transform(_cu(x.C_occ), _cu(x.C_vir), _cu(Lp), 0, naux)
        Ec = float(c.energy(e_occ, e_vir).cpu()[0])
        assert abs(Ec - Ecf) <= 1e-12 * abs(Ecf)
        c.close()
