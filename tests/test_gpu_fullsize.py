"""Full-size parity (BASELINE.json configs[3], the launch configuration bench.py times: one transform call over
[0, naux), 148 persistent CTAs, 120-row tiles) and the config-4 tile shape.

The oracle needs ~0.5 h for the dense config-3 problem, so these tests use special cases that cut the ORACLE's work
but not the GPU's:

  * sparse-aux x sparse-virtual: (P|mu nu) is non-zero on a handful of aux rows only (first/last row, both sides
    of a K-block boundary, the middle) and C_vir is non-zero on a handful of virtual columns only (first/last, both
    sides of tile boundaries).  The GPU streams all 4800 rows through A1/A2 and runs all 583 740 pair tiles over all
    600 K-blocks and every epilogue; zero rows/columns add exact zeros (x + 0*y == x, 0/D == 0 in IEEE arithmetic),
    so G and E must equal the oracle run on the compressed problem (naux = len(rows), nvir = len(virt)) to the
    usual tolerances.  (The oracle's O6 loop alone is o^3 v^2 long-double operations: hours at v = 1080.)
  * sampled B rows of a dense transform against oracle.transform_block on the same aux rows (B is the first
    region of the workspace, [nvir][nocc][naux_ld]).
  * properties that hold at any size on the dense problem: E <= 0 for P = I, G_ii <= 0 (pin P-5), partition sum of
    projectors (pin P-3), and bit-reproducibility.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2412_18553_b200 as sie
from workloads import config_specs, make_cluster

pytestmark = pytest.mark.gpu

E_RTOL = 1e-10
G_ATOL = 1e-11


def _need_gb(gb):
    free, _ = torch.cuda.mem_get_info()
    if free < gb * 2**30:
        pytest.skip(f"needs {gb} GiB of free device memory")


def _sparse_case(spec, rows, virt):
    x = make_cluster(spec)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731
    Lsub = np.stack([x.L_block(p, p + 1, threads=4)[0] for p in rows])  # [len(rows)][npair]
    L = torch.zeros((spec.naux, spec.npair), dtype=torch.float64, device="cuda")
    L[torch.tensor(rows, device="cuda")] = cu(Lsub)
    C_vir = np.zeros_like(x.C_vir)
    C_vir[:, virt] = x.C_vir[:, virt]
    s = sie.ClusterSolver(spec.nao, spec.nocc, spec.nvir, spec.naux)
    info = s.info()
    s.transform(cu(x.C_occ), cu(C_vir), L, 0, spec.naux)  # one call over [0, naux), as bench.py does
    E, G = s.energy(cu(x.e_occ), cu(x.e_vir), cu(x.P_frag))
    gam, _ = s.rdm_occ(cu(x.e_occ), cu(x.e_vir))  # NEXT-1 on the same B, same special case (0 / D == 0 exactly)
    torch.cuda.synchronize()
    E, G, gam = float(E.cpu()[0]), G.cpu().numpy(), gam.cpu().numpy()
    s.close()
    del L
    torch.cuda.empty_cache()
    # oracle on the compressed problem (same bytes for the non-zero rows / columns)
    Bor = oracle.transform(x.C_occ, np.ascontiguousarray(x.C_vir[:, virt]), Lsub)
    Gor = oracle.pair_G(Bor, x.e_occ, np.ascontiguousarray(x.e_vir[virt]))
    Eor = oracle.trace(x.P_frag, Gor)
    gam_or = oracle.rdm_occ(Bor, x.e_occ, np.ascontiguousarray(x.e_vir[virt]))
    assert np.max(np.abs(gam - gam_or)) <= G_ATOL * max(1.0, float(np.max(np.abs(gam_or))))
    assert np.max(np.abs(gam_or - 2.0 * np.eye(spec.nocc))) > 1e-6  # the special case is not trivially the identity
    return info, E, G, Eor, Gor


def _assert_parity(E, G, Eor, Gor):
    assert Eor < 0
    assert abs(E - Eor) <= E_RTOL * abs(Eor), (E, Eor)
    err = float(np.max(np.abs(G - Gor)))
    assert err <= G_ATOL * max(1.0, float(np.max(np.abs(Gor)))), (err, float(np.max(np.abs(Gor))))


def test_config3_full_size_sparse_matches_oracle():
    spec = config_specs(3)[0]
    _need_gb(40)
    rows = [0, 7, 8, 2399, 3001, 3002, 4792, 4799]
    virt = [0, 1, 2, 17, 500, 539, 540, 541, 777, 1000, 1077, 1078, 1079]
    info, E, G, Eor, Gor = _sparse_case(spec, rows, virt)
    assert info["TM"] == 120 and info["ncta"] == 148 and info["ntiles"] == 1080 * 1081 // 2  # what bench.py launches
    _assert_parity(E, G, Eor, Gor)


def test_config4_shape_sparse_matches_oracle():
    # o = 64: two virtual blocks per 128-row tile, v = 512, naux = 2304 (config 4, k = 1)
    spec = config_specs(4)[2]
    _need_gb(8)
    rows = [0, 15, 16, 1000, 2303]
    virt = [0, 1, 2, 3, 254, 255, 256, 257, 300, 301, 510, 511]  # both blocks of a tile, both sides of tile edges
    info, E, G, Eor, Gor = _sparse_case(spec, rows, virt)
    assert info["TM"] == 128 and info["ta"] == 2
    _assert_parity(E, G, Eor, Gor)


def test_config3_dense_B_rows_and_size_independent_properties():
    """Dense config-3 inputs on a 1/4-aux slice of the transform for B (sampled rows vs the oracle), then the dense
    pair stage on that B: sign, partition and reproducibility properties."""
    spec = config_specs(3)[0].with_(naux=1200)  # same nao/nocc/nvir; 6.9 GB of packed integrals instead of 27.7
    _need_gb(16)
    x = make_cluster(spec)
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()  # noqa: E731
    o, v, naux = spec.nocc, spec.nvir, spec.naux
    s = sie.ClusterSolver(spec.nao, o, v, naux)
    C_occ, C_vir = cu(x.C_occ), cu(x.C_vir)
    for p0 in (800, 0, 400):  # three aux blocks, fed out of order
        Lb = cu(x.L_block(p0, p0 + 400, threads=8))
        s.transform(C_occ, C_vir, Lb, p0, p0 + 400)
        torch.cuda.synchronize()
        del Lb
    naux_ld = (naux + 7) // 8 * 8
    Bdev = s.workspace[: v * o * naux_ld * 8].view(torch.float64).view(v, o, naux_ld)
    sample = [0, 399, 400, 1199]
    for p in sample:
        Bor = np.zeros((o, v, 1))
        oracle.transform_block(x.C_occ, x.C_vir, x.L_block(p, p + 1), 0, 1, Bor)
        got = Bdev[:, :, p].cpu().numpy().T  # [o][v]
        assert np.max(np.abs(got - Bor[:, :, 0])) <= 1e-13 * max(1.0, np.max(np.abs(Bor))), p
    e_occ, e_vir = cu(x.e_occ), cu(x.e_vir)
    E_I, G = s.energy(e_occ, e_vir, None)
    E_I2, G2 = s.energy(e_occ, e_vir, None)
    torch.cuda.synchronize()
    assert torch.equal(G, G2) and torch.equal(E_I, E_I2)  # fixed-order reduction: identical bits
    Gh = G.cpu().numpy()
    assert float(E_I.cpu()[0]) < 0 and np.all(np.diag(Gh) < 0)  # pin P-5
    assert abs(float(E_I.cpu()[0]) - np.trace(Gh)) <= 1e-12 * abs(np.trace(Gh))
    # pin P-3: projectors of an orthogonal partition of the occupied space sum to the total
    rng = np.random.default_rng(5)
    U, _ = np.linalg.qr(rng.standard_normal((o, o)))
    parts, tot = [U[:, :37], U[:, 37:90], U[:, 90:]], 0.0
    for Q in parts:
        E_k, _ = s.energy(e_occ, e_vir, cu(Q @ Q.T), want_G=False)
        tot += float(E_k.cpu()[0])
    assert abs(tot - float(E_I.cpu()[0])) <= 1e-10 * abs(float(E_I.cpu()[0]))
    s.close()
