"""Pins of oracle.rdm_occ and oracle.rdm_vir (NEXT-1): occupied block of the MP2 1-RDM, PAPER.md Eq. S18 (L357),
    gamma_ij = 2 delta_ij - 2 sum_k sum_ab t_ik^ab (2 t_jk^ab - t_jk^ba),  t = (ia|kb) / (e_i + e_k - e_a - e_b).
Pinned to things other than itself: the closed form for o = v = 1, a hand-worked 2-occupied case, the explicit
four-index brute-force route (a path that never forms B), the derivative of the already pinned energy
(gamma_ii = 2 + dE/de_i), and structural facts (symmetry, 2 - gamma positive semi-definite, scalings)."""
import numpy as np
import pytest

import oracle
from test_oracle_pins import _bruteforce_ovov, _small


def test_closed_form_o1_v1():
    rng = np.random.default_rng(3)
    Bv = rng.standard_normal(6)
    ei, ea = -0.9, 0.4
    t = float(np.sum(Bv * Bv)) / (2 * ei - 2 * ea)
    g = oracle.rdm_occ(Bv.reshape(1, 1, 6), np.array([ei]), np.array([ea]))
    assert g[0, 0] == pytest.approx(2.0 - 2.0 * t * t, rel=1e-14)


def test_handworked_two_occupied_one_virtual():
    """o = 2, v = 1, naux = 1, B = [b0, b1]: (ia|ka) = b_i b_k, t_ik = b_i b_k / (e_i + e_k - 2 e_a); with one virtual
    2 t - t~ = t, so gamma_ij = 2 delta_ij - 2 sum_k t_ik t_jk.  Numbers worked by hand:
    b = (1, 2), e_occ = (-1, -2), e_a = 1  ->  D_00 = -4, D_01 = -5, D_11 = -6; t_00 = -1/4, t_01 = -2/5, t_11 = -2/3;
    Gamma_00 = 1/16 + 4/25 = 0.2225, Gamma_01 = (1/4)(2/5) + (2/5)(2/3) = 11/30, Gamma_11 = 4/25 + 4/9 = 136/225."""
    B = np.array([1.0, 2.0]).reshape(2, 1, 1)
    g = oracle.rdm_occ(B, np.array([-1.0, -2.0]), np.array([1.0]))
    expect = np.array([[2 - 2 * 0.2225, -2 * 11 / 30], [-2 * 11 / 30, 2 - 2 * 136 / 225]])
    assert np.max(np.abs(g - expect)) < 1e-14


@pytest.mark.parametrize("seed,nocc,nvir,naux,extra", [(0, 3, 5, 7, 0), (1, 4, 6, 10, 0), (2, 2, 7, 5, 3)])
def test_bruteforce_from_explicit_four_index_amplitudes(seed, nocc, nvir, naux, extra):
    x, Lp = _small(seed, nocc, nvir, naux, extra_ao=extra)
    ovov = _bruteforce_ovov(x, Lp)  # (ia|kb) without ever forming H or B
    e_o, e_v = x.e_occ, x.e_vir
    D = e_o[:, None, None, None] + e_o[None, None, :, None] - e_v[None, :, None, None] - e_v[None, None, None, :]
    t = ovov / D  # t[i,a,k,b]
    Gam = np.einsum("iakb,jakb->ij", t, 2.0 * t - t.transpose(0, 3, 2, 1))
    expect = 2.0 * np.eye(nocc) - 2.0 * Gam
    g = oracle.rdm_occ(oracle.transform(x.C_occ, x.C_vir, Lp), e_o, e_v)
    assert np.max(np.abs(g - expect)) <= 1e-13 * max(1.0, np.max(np.abs(expect)))


def test_diagonal_is_two_plus_energy_derivative():
    """E = sum V(2V - V~)/D  =>  dE/de_k = -2 sum_{j,ab} t_kj^ab (2 t_kj^ab - t_kj^ba), i.e. gamma_kk = 2 + dE/de_k.
    Central differences of the PINNED energy (oracle.pair_G + trace) with h = 1e-4: truncation ~ h^2 E'''."""
    x, Lp = _small(5, 4, 6, 9)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    g = oracle.rdm_occ(B, x.e_occ, x.e_vir)
    E = lambda eo: oracle.trace(None, oracle.pair_G(B, eo, x.e_vir))  # noqa: E731
    h = 1e-4
    for k in range(4):
        d = np.zeros(4)
        d[k] = h
        dE = (E(x.e_occ + d) - E(x.e_occ - d)) / (2 * h)
        assert g[k, k] == pytest.approx(2.0 + dE, abs=2e-6 * max(1.0, abs(dE)))


def test_structure_symmetry_psd_and_scalings():
    x, Lp = _small(7, 5, 8, 11)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    g = oracle.rdm_occ(B, x.e_occ, x.e_vir)
    assert np.max(np.abs(g - g.T)) <= 1e-14 * max(1.0, np.max(np.abs(g)))
    Gam = (2.0 * np.eye(5) - g) / 2.0
    assert np.min(np.linalg.eigvalsh((Gam + Gam.T) / 2)) >= -1e-12 * np.max(np.abs(Gam))  # sum_k,ab [t t + (t - t~)^2 / 2]-type Gram matrix
    assert np.all(np.diag(g) <= 2.0)
    # L -> 2 L  =>  t -> 4 t, Gamma -> 16 Gamma;  e -> 2 e  =>  Gamma -> Gamma / 4  (gamma itself is rounded at ~2: ulp 4e-16)
    g2 = oracle.rdm_occ(2.0 * B, x.e_occ, x.e_vir)
    scale = max(1.0, float(np.max(np.abs(g))))
    assert np.max(np.abs((2.0 * np.eye(5) - g2) - 16.0 * (2.0 * np.eye(5) - g))) <= 1e-13 * scale
    g3 = oracle.rdm_occ(B, 2.0 * x.e_occ, 2.0 * x.e_vir)
    assert np.max(np.abs((2.0 * np.eye(5) - g3) - (2.0 * np.eye(5) - g) / 4.0)) <= 1e-14 * scale
    # an orthogonal rotation of the aux index leaves (ia|kb), hence gamma, unchanged
    Q, _ = np.linalg.qr(np.random.default_rng(1).standard_normal((11, 11)))
    g4 = oracle.rdm_occ(np.ascontiguousarray(B @ Q), x.e_occ, x.e_vir)
    assert np.max(np.abs(g4 - g)) <= 1e-12 * scale


# ---------------------------------------------------------------------------------------------- O9: gamma_ab, Eq. S17 (L355)
def test_vir_closed_form_o1_v1():
    """o = v = 1: gamma_aa = 2 t (2 t - t) = 2 t^2."""
    rng = np.random.default_rng(4)
    Bv = rng.standard_normal(5)
    ei, ea = -0.7, 0.6
    t = float(np.sum(Bv * Bv)) / (2 * ei - 2 * ea)
    g = oracle.rdm_vir(Bv.reshape(1, 1, 5), np.array([ei]), np.array([ea]))
    assert g[0, 0] == pytest.approx(2.0 * t * t, rel=1e-14)


def test_vir_handworked_one_occupied_two_virtuals():
    """o = 1, v = 2, naux = 1, B = [b0, b1]: (ia|ic) = b_a b_c, t^{ac} = b_a b_c / (2 e_i - e_a - e_c) is symmetric, so
    2 t^{bc} - t^{cb} = t^{bc} and gamma_ab = 2 sum_c t^{ac} t^{bc}.  By hand: b = (1, 2), e_i = -1, e_vir = (1, 2):
    D = -4, -5, -6;  t^{00} = -1/4, t^{01} = -2/5, t^{11} = -2/3;
    gamma_00 = 2 (1/16 + 4/25) = 0.445, gamma_01 = 2 (1/10 + 4/15) = 11/15, gamma_11 = 2 (4/25 + 4/9) = 272/225."""
    B = np.array([1.0, 2.0]).reshape(1, 2, 1)
    g = oracle.rdm_vir(B, np.array([-1.0]), np.array([1.0, 2.0]))
    expect = np.array([[0.445, 11 / 15], [11 / 15, 272 / 225]])
    assert np.max(np.abs(g - expect)) < 1e-14


@pytest.mark.parametrize("seed,nocc,nvir,naux,extra", [(0, 3, 5, 7, 0), (1, 4, 6, 10, 0), (2, 2, 7, 5, 3)])
def test_vir_bruteforce_from_explicit_four_index_amplitudes(seed, nocc, nvir, naux, extra):
    """The exchange term: t_ij^cb swaps the two VIRTUAL indices at fixed (i, j); a wrong sign or a swap of the occupied
    pair instead fails here (t[i,a,j,c] from explicit (mu nu|lam sig), a route that never forms B)."""
    x, Lp = _small(seed, nocc, nvir, naux, extra_ao=extra)
    ovov = _bruteforce_ovov(x, Lp)
    e_o, e_v = x.e_occ, x.e_vir
    D = e_o[:, None, None, None] + e_o[None, None, :, None] - e_v[None, :, None, None] - e_v[None, None, None, :]
    t = ovov / D  # t[i,a,j,c]
    expect = 2.0 * np.einsum("iajc,ibjc->ab", t, 2.0 * t - t.transpose(0, 3, 2, 1))
    g = oracle.rdm_vir(oracle.transform(x.C_occ, x.C_vir, Lp), e_o, e_v)
    assert np.max(np.abs(g - expect)) <= 1e-13 * max(1.0, np.max(np.abs(expect)))


def test_vir_trace_conserves_the_electron_count_and_diagonal_is_energy_derivative():
    """Tr gamma_occ + Tr gamma_vir = 2 nocc (what leaves the occupied block arrives in the virtual block), and
    gamma_aa = + dE/de_a of the PINNED energy (central differences, h = 1e-4)."""
    x, Lp = _small(6, 4, 6, 9)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    go, gv = oracle.rdm_occ(B, x.e_occ, x.e_vir), oracle.rdm_vir(B, x.e_occ, x.e_vir)
    assert np.trace(go) + np.trace(gv) == pytest.approx(2.0 * 4, rel=1e-13)
    E = lambda ev: oracle.trace(None, oracle.pair_G(B, x.e_occ, ev))  # noqa: E731
    h = 1e-4
    for a in range(6):
        d = np.zeros(6)
        d[a] = h
        dE = (E(x.e_vir + d) - E(x.e_vir - d)) / (2 * h)
        assert gv[a, a] == pytest.approx(dE, abs=2e-6 * max(1.0, abs(dE)))


def test_vir_structure_symmetry_psd_and_scalings():
    x, Lp = _small(8, 4, 7, 10)
    B = oracle.transform(x.C_occ, x.C_vir, Lp)
    g = oracle.rdm_vir(B, x.e_occ, x.e_vir)
    scale = max(1.0, float(np.max(np.abs(g))))
    assert np.max(np.abs(g - g.T)) <= 1e-14 * scale
    assert np.min(np.linalg.eigvalsh((g + g.T) / 2)) >= -1e-12 * scale and np.all(np.diag(g) >= 0.0)
    assert np.max(np.abs(oracle.rdm_vir(2.0 * B, x.e_occ, x.e_vir) - 16.0 * g)) <= 1e-13 * scale * 16
    assert np.max(np.abs(oracle.rdm_vir(B, 2.0 * x.e_occ, 2.0 * x.e_vir) - g / 4.0)) <= 1e-14 * scale
    # permuting the virtuals permutes rows and columns of gamma_vir
    perm = np.random.default_rng(2).permutation(7)
    gp = oracle.rdm_vir(np.ascontiguousarray(B[:, perm, :]), x.e_occ, x.e_vir[perm])
    assert np.max(np.abs(gp - g[np.ix_(perm, perm)])) <= 1e-13 * scale
