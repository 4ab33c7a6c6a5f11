"""Pins of the CPU oracle (oracle/) to things other than itself.  All run without a GPU.

Each test names the oracle step it pins (O1..O7, oracle/dfmp2_oracle.c header) and what fixes the
expected value: a hand-worked number (tests/golden/handworked.txt), a closed form, the textbook
closed-shell MP2 expression evaluated from brute-force four-index integrals (a route that never
forms H or B), or an invariant of the mathematics.
"""
import os

import numpy as np
import pytest

import oracle
from workloads import ClusterSpec, make_cluster

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    out = {}
    with open(os.path.join(HERE, "golden", "handworked.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split()
            out[k] = float(v)
    return out


GOLD = _golden()


def _small(seed=0, nocc=3, nvir=5, naux=7, rank=2, extra_ao=0, scale="var"):
    spec = ClusterSpec(900 + seed, 0, nocc + nvir + extra_ao, nocc, nvir, naux, rank, scale)
    x = make_cluster(spec)
    return x, x.L_packed()


def _full_from_packed(Lp, nao):
    """Library route for the packed layout: numpy's tril_indices enumerate the row-major lower triangle."""
    r, c = np.tril_indices(nao)
    F = np.zeros((Lp.shape[0], nao, nao))
    F[:, r, c] = Lp
    F[:, c, r] = Lp
    return F


def _bruteforce_ovov(x, Lp):
    """(ia|jb) through the explicit four-index AO tensor and four quarter transforms (Eq. S49)."""
    nao = x.spec.nao
    F = _full_from_packed(Lp, nao)
    eri = np.einsum("Pmn,Pls->mnls", F, F)  # (mu nu|lam sig) = sum_P L L
    t1 = np.einsum("mnls,mi->inls", eri, x.C_occ)
    t2 = np.einsum("inls,na->ials", t1, x.C_vir)
    t3 = np.einsum("ials,lj->iajs", t2, x.C_occ)
    return np.einsum("iajs,sb->iajb", t3, x.C_vir)


def _textbook_G(ovov, e_occ, e_vir):
    """G[i'][i] = sum_jab [(i'a|jb)/D_{i'jab}] [2(ia|jb) - (ib|ja)] written with numpy broadcasting."""
    D = e_occ[:, None, None, None] + e_occ[None, None, :, None] - e_vir[None, :, None, None] - e_vir[None, None, None, :]
    t = ovov / D  # t[i',a,j,b]
    W = 2.0 * ovov - ovov.transpose(0, 3, 2, 1)  # W[i,a,j,b] = 2(ia|jb) - (ib|ja)
    return np.einsum("pajb,iajb->pi", t, W)


# ----------------------------------------------------------------------------- hand-worked cases (O4-O7)
def test_handworked_case_A_orientation_of_G_and_trace():
    B = np.array([[[1.0]], [[2.0]]])  # [i][a][P]
    G = oracle.pair_G(B, np.array([-1.0, -2.0]), np.array([1.0]))
    for k, (ip, i) in {"A.G00": (0, 0), "A.G01": (0, 1), "A.G10": (1, 0), "A.G11": (1, 1)}.items():
        assert G[ip, i] == pytest.approx(GOLD[k], rel=1e-15, abs=0)
    P01 = np.array([[0.0, 1.0], [0.0, 0.0]])  # P[i=0][i'=1]
    assert oracle.trace(P01, G) == pytest.approx(GOLD["A.E_P01"], rel=1e-15)
    assert oracle.trace(None, G) == pytest.approx(GOLD["A.E_I"], rel=1e-15)
    assert oracle.trace(np.eye(2), G) == pytest.approx(GOLD["A.E_I"], rel=1e-15)


def test_handworked_case_B_single_occupied():
    B = np.array([[[1.0, 0.0], [1.0, 1.0]]])
    G = oracle.pair_G(B, np.array([-1.0]), np.array([1.0, 2.0]))
    assert G[0, 0] == pytest.approx(GOLD["B.G00"], rel=1e-15)


@pytest.mark.parametrize(
    "case,B",
    [
        ("C", [[[1.0, 0.0], [0.0, 1.0]], [[1.0, 1.0], [1.0, -1.0]]]),
        ("D", [[[1.0, 0.0], [0.0, 1.0]], [[0.0, 1.0], [2.0, 0.0]]]),
    ],
)
def test_handworked_cases_C_D_exchange_term(case, B):
    G = oracle.pair_G(np.array(B), np.array([-1.0, -1.0]), np.array([1.0, 1.0]))
    for ip in range(2):
        for i in range(2):
            assert G[ip, i] == pytest.approx(GOLD[f"{case}.G{ip}{i}"], rel=1e-15, abs=1e-15)


def test_handworked_transform_2x2():
    """O1-O3: nao=2, one aux index, packed row (L00, L10, L11) = (5, 7, 11).
    C = identity columns  -> B = L01 = 7 (packed index mu(mu+1)/2+nu = 1).
    C rotated by 45 deg: C_occ=(c,s), C_vir=(-s,c) -> B = cs(L11-L00) + (c^2-s^2) L01 = 0.5*6 = 3."""
    Lp = np.array([[5.0, 7.0, 11.0]])
    B = oracle.transform(np.array([[1.0], [0.0]]), np.array([[0.0], [1.0]]), Lp)
    assert B.shape == (1, 1, 1) and B[0, 0, 0] == 7.0
    c = s = np.sqrt(0.5)
    B = oracle.transform(np.array([[c], [s]]), np.array([[-s], [c]]), Lp)
    assert B[0, 0, 0] == pytest.approx(3.0, rel=1e-15)
    F = oracle.unpack(Lp[0], 2)
    assert np.array_equal(F, np.array([[5.0, 7.0], [7.0, 11.0]]))


# ----------------------------------------------------------------------------- closed form (north_star a)
def test_closed_form_o1_v1():
    """o=v=1: E = G_11 = (ia|ia)^2 / (2 (e_i - e_a)), (ia|ia) = sum_P (B^P)^2."""
    rng = np.random.default_rng(11)
    Bv = rng.standard_normal(9)
    ei, ea = -0.7, 1.3
    G = oracle.pair_G(Bv.reshape(1, 1, 9), np.array([ei]), np.array([ea]))
    iaia = float(np.sum(Bv * Bv))
    expect = iaia * iaia / (2.0 * (ei - ea))
    assert G[0, 0] == pytest.approx(expect, rel=1e-14)
    assert oracle.trace(None, G) == pytest.approx(expect, rel=1e-14)


# ----------------------------------------------------------------------------- brute force (north_star d, b)
@pytest.mark.parametrize("seed,nocc,nvir,naux,extra", [(0, 3, 5, 7, 0), (1, 4, 6, 10, 0), (2, 2, 7, 5, 3)])
def test_bruteforce_four_index_route(seed, nocc, nvir, naux, extra):
    """O1-O4: oracle's DF route (unpack, two half transforms, aux dot) == explicit (mu nu|lam sig) route."""
    x, Lp = _small(seed, nocc, nvir, naux, extra_ao=extra)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    ovov_oracle = np.einsum("iaP,jbP->iajb", B, B)
    ovov_bf = _bruteforce_ovov(x, Lp)
    assert np.max(np.abs(ovov_oracle - ovov_bf)) <= 1e-13 * max(1.0, np.max(np.abs(ovov_bf)))
    # O5-O6 against the textbook expression evaluated on the brute-force integrals
    G = oracle.pair_G(B, x.e_occ, x.e_vir)
    G_bf = _textbook_G(ovov_bf, x.e_occ, x.e_vir)
    assert np.max(np.abs(G - G_bf)) <= 1e-13 * max(1.0, np.max(np.abs(G_bf)))


def test_identity_projector_is_canonical_mp2():
    """P_frag = I  =>  E = sum_ij e_ij, e_ij = sum_ab (ia|jb)[2(ia|jb)-(ib|ja)]/D  (textbook closed-shell MP2)."""
    x, Lp = _small(3, 4, 6, 9)
    ovov = _bruteforce_ovov(x, Lp)
    D = x.e_occ[:, None, None, None] + x.e_occ[None, None, :, None] - x.e_vir[None, :, None, None] - x.e_vir[None, None, None, :]
    e_ij = np.einsum("iajb,iajb->ij", ovov / D, 2.0 * ovov - ovov.transpose(0, 3, 2, 1))
    E, G = oracle.dfmp2(x.C_occ, x.C_vir, Lp, x.e_occ, x.e_vir, None)
    assert E == pytest.approx(float(e_ij.sum()), rel=1e-13)
    assert np.all(e_ij < 0.0)  # P-5: every pair energy is negative
    assert np.all(np.diag(G) < 0.0)


def test_config0_full_vs_bruteforce():
    """The real config 0 (nao=48, o=8, v=40, naux=160): whole oracle chain vs the four-index route."""
    from workloads import config_specs

    x = make_cluster(config_specs(0)[0])
    Lp = x.L_packed()
    E, G = oracle.dfmp2(x.C_occ, x.C_vir, Lp, x.e_occ, x.e_vir, x.P_frag)
    G_bf = _textbook_G(_bruteforce_ovov(x, Lp), x.e_occ, x.e_vir)
    assert np.max(np.abs(G - G_bf)) <= 1e-12 * np.max(np.abs(G_bf))
    assert E == pytest.approx(float(np.sum(x.P_frag * G_bf.T)), rel=1e-12)


# ----------------------------------------------------------------------------- projector properties (north_star c)
def test_fragment_additivity_over_a_partition():
    """Projectors Q_k Q_k^T built from an orthogonal U=[Q_1|Q_2|Q_3] sum to I => fragment energies sum to Tr G."""
    x, Lp = _small(4, 6, 7, 8)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    G = oracle.pair_G(B, x.e_occ, x.e_vir)
    U, _ = np.linalg.qr(np.random.default_rng(5).standard_normal((6, 6)))
    parts = [U[:, :2], U[:, 2:3], U[:, 3:]]
    Es = [oracle.trace(q @ q.T, G) for q in parts]
    assert sum(Es) == pytest.approx(oracle.trace(None, G), rel=1e-13)
    assert oracle.trace(None, G) == pytest.approx(float(np.trace(G)), rel=1e-14)


def test_trace_is_linear_and_uses_P_i_iprime_times_G_iprime_i():
    rng = np.random.default_rng(6)
    G = rng.standard_normal((5, 5))
    P = rng.standard_normal((5, 5))  # deliberately non-symmetric
    assert oracle.trace(P, G) == pytest.approx(float(np.trace(P @ G)), rel=1e-13)
    assert oracle.trace(P, G) != pytest.approx(float(np.trace(P.T @ G)), rel=1e-6)


def test_j_slices_add_up():
    x, Lp = _small(7, 5, 6, 9)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    G = oracle.pair_G(B, x.e_occ, x.e_vir)
    Gs = oracle.pair_G(B, x.e_occ, x.e_vir, 0, 2) + oracle.pair_G(B, x.e_occ, x.e_vir, 2, 5)
    assert np.max(np.abs(G - Gs)) <= 1e-14 * np.max(np.abs(G))


# ----------------------------------------------------------------------------- invariances and scalings (P-6..P-8)
def test_G_is_not_symmetric_unless_occupied_energies_are_equal():
    x, Lp = _small(8, 4, 6, 9)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    G = oracle.pair_G(B, x.e_occ, x.e_vir)
    assert np.max(np.abs(G - G.T)) > 1e-6 * np.max(np.abs(G))
    Geq = oracle.pair_G(B, np.full(4, -0.9), x.e_vir)
    assert np.max(np.abs(Geq - Geq.T)) <= 1e-13 * np.max(np.abs(Geq))


def test_invariances():
    x, Lp = _small(9, 4, 6, 9)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    G = oracle.pair_G(B, x.e_occ, x.e_vir)
    tol = 2e-13 * np.max(np.abs(G))
    # constant shift of all orbital energies leaves every denominator unchanged
    assert np.max(np.abs(oracle.pair_G(B, x.e_occ + 0.25, x.e_vir + 0.25) - G)) <= tol
    # orthogonal rotation of the aux index
    R, _ = np.linalg.qr(np.random.default_rng(1).standard_normal((9, 9)))
    assert np.max(np.abs(oracle.pair_G(np.ascontiguousarray(B @ R), x.e_occ, x.e_vir) - G)) <= tol
    # permuting virtuals (columns of C_vir together with e_vir)
    pv = np.random.default_rng(2).permutation(6)
    Bv = oracle.transform(x.C_occ, np.ascontiguousarray(x.C_vir[:, pv]), Lp)
    assert np.max(np.abs(oracle.pair_G(Bv, x.e_occ, x.e_vir[pv]) - G)) <= tol
    # permuting occupieds permutes rows and columns of G
    po = np.array([2, 0, 3, 1])
    Bo = oracle.transform(np.ascontiguousarray(x.C_occ[:, po]), x.C_vir, Lp)
    Go = oracle.pair_G(Bo, x.e_occ[po], x.e_vir)
    assert np.max(np.abs(Go - G[np.ix_(po, po)])) <= tol
    # a sign flip of one occupied column maps G_{i'i} -> s_i' s_i G_{i'i}
    s = np.array([1.0, -1.0, 1.0, 1.0])
    Gs = oracle.pair_G(oracle.transform(x.C_occ * s[None, :], x.C_vir, Lp), x.e_occ, x.e_vir)
    assert np.max(np.abs(Gs - G * np.outer(s, s))) <= tol


def test_power_of_two_scalings_are_exact():
    x, Lp = _small(10, 3, 5, 8)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    G = oracle.pair_G(B, x.e_occ, x.e_vir)
    assert np.array_equal(oracle.pair_G(B * 2.0, x.e_occ, x.e_vir), G * 16.0)  # L -> sL  =>  G -> s^4 G
    assert np.array_equal(oracle.pair_G(B, x.e_occ * 4.0, x.e_vir * 4.0), G / 4.0)  # e -> se  =>  G -> G/s
    B2 = oracle.transform(x.C_occ, x.C_vir, Lp * 2.0)
    assert np.array_equal(B2, B * 2.0)


def test_transform_blocks_cover_like_one_call():
    x, Lp = _small(12, 3, 5, 11)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    Bb = np.zeros_like(B)
    for p0, p1 in ((4, 9), (0, 4), (9, 11)):
        oracle.transform_block(x.C_occ, x.C_vir, Lp[p0:p1], p0, p1, Bb)
    assert np.array_equal(B, Bb)


def test_nmo_smaller_than_nao():
    """nocc + nvir < nao (reading A-8): unused AO directions must not leak in."""
    x, Lp = _small(13, 3, 4, 6, extra_ao=5)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    F = _full_from_packed(Lp, x.spec.nao)
    B_np = np.einsum("mi,Pmn,na->iaP", x.C_occ, F, x.C_vir)
    assert np.max(np.abs(B - B_np)) <= 1e-14 * max(1.0, np.max(np.abs(B_np)))


def test_P9_blas_route_agrees_with_the_loop_oracle_at_config1_scale():
    """Pin P-9: a second CPU route — unpack with np.tril_indices, BLAS matmuls for both half transforms and
    the pair integrals, vectorised G in plain doubles (different summation order everywhere) — agrees with the loop oracle
    on the dense config-1 problem (o=30, v=270, nao=300, naux=1200) to ~1e-13 relative: the loop oracle's indexing holds
    at a size with many aux blocks, ragged 8-wide dot tails and 72 900 virtual pairs per occupied pair."""
    from workloads import config_specs, make_cluster

    spec = config_specs(1)[0]
    x = make_cluster(spec)
    Lp = x.L_packed(threads=4)
    o, v, nao, naux = spec.nocc, spec.nvir, spec.nao, spec.naux
    iu = np.tril_indices(nao)
    H = np.empty((naux, o, nao))
    F = np.zeros((nao, nao))
    for P in range(naux):  # H^P = C_occ^T L^P with L^P rebuilt from its packed row
        F[iu] = Lp[P]
        F.T[iu] = Lp[P]
        H[P] = x.C_occ.T @ F
    Bnp = np.ascontiguousarray(np.einsum("Pin,na->iaP", H, x.C_vir, optimize=True))  # [o][v][naux]
    Bor = oracle.transform(x.C_occ, x.C_vir, Lp)
    assert np.max(np.abs(Bnp - Bor)) <= 1e-13 * np.max(np.abs(Bor))
    ovov = (Bnp.reshape(o * v, naux) @ Bnp.reshape(o * v, naux).T).reshape(o, v, o, v)  # (ia|jb)
    D = x.e_occ[:, None, None, None] + x.e_occ[None, None, :, None] - x.e_vir[None, :, None, None] - x.e_vir[None, None, None, :]
    t = ovov / D
    W = 2.0 * ovov - ovov.transpose(0, 3, 2, 1)
    Gnp = np.einsum("pajb,iajb->pi", t, W, optimize=True)
    Gor = oracle.pair_G(Bor, x.e_occ, x.e_vir)
    assert np.max(np.abs(Gnp - Gor)) <= 1e-12 * np.max(np.abs(Gor))
    assert abs(np.einsum("ip,pi->", x.P_frag, Gnp) - oracle.trace(x.P_frag, Gor)) <= 1e-12 * abs(oracle.trace(x.P_frag, Gor))
