"""Input generator: shapes, distributions, determinism, block-independence (no GPU)."""
import numpy as np

from workloads import ClusterSpec, config_specs, make_cluster, npair


def test_config_shapes_match_baseline_json():
    s0 = config_specs(0)[0]
    assert (s0.nao, s0.nocc, s0.nvir, s0.naux, s0.rank) == (48, 8, 40, 160, 4)
    s1 = config_specs(1)
    assert [(s.nao, s.nocc, s.nvir, s.naux, s.rank) for s in s1] == [(300, 30, 270, 1200, 15), (300, 30, 270, 1200, 0)]
    s2 = config_specs(2)
    assert len(s2) == 96
    for s in s2:
        assert 16 <= s.nocc <= 48 and s.nvir == 8 * s.nocc and s.nao == 9 * s.nocc and s.naux == 4 * s.nao
        assert s.rank == max(1, s.nocc // 4)
    assert len({s.nocc for s in s2}) > 10  # sizes really vary
    s3 = config_specs(3)[0]
    assert (s3.nao, s3.nocc, s3.nvir, s3.naux, s3.rank) == (1200, 120, 1080, 4800, 60)
    s4 = config_specs(4)
    assert [s.nvir for s in s4] == [256, 256, 512, 512, 1024, 1024, 2048, 2048]
    assert all(s.nocc == 64 and s.naux == 4 * s.nao for s in s4)
    assert [s.rank for s in s4] == [32, 0] * 4


def test_inputs_are_deterministic_and_well_formed():
    spec = config_specs(0)[0]
    a, b = make_cluster(spec), make_cluster(spec)
    assert np.array_equal(a.C_occ, b.C_occ) and np.array_equal(a.e_vir, b.e_vir)
    C = np.concatenate([a.C_occ, a.C_vir], axis=1)
    assert np.max(np.abs(C.T @ C - np.eye(48))) < 1e-13  # orthogonal
    assert a.e_occ.min() >= -1.5 and a.e_occ.max() <= -0.3
    assert a.e_vir.min() >= 0.1 and a.e_vir.max() <= 3.0
    P = a.P_frag
    assert np.max(np.abs(P - P.T)) < 1e-14 and np.max(np.abs(P @ P - P)) < 1e-13
    assert abs(np.trace(P) - 4.0) < 1e-12  # rank-4 projector
    assert np.array_equal(make_cluster(spec.with_(rank=0)).P_frag, np.eye(8))


def test_L_blocks_are_blocking_independent_and_scaled():
    spec = ClusterSpec(7, 3, 20, 4, 16, 12, 2)
    x = make_cluster(spec)
    L = x.L_packed()
    assert L.shape == (12, npair(20))
    assert np.array_equal(L[5:9], x.L_block(5, 9))
    assert np.array_equal(L, x.L_block(0, 12, threads=4))
    big = make_cluster(ClusterSpec(7, 4, 100, 10, 90, 40, 2))
    Lb = big.L_packed()
    assert abs(Lb.std() * np.sqrt(100) - 1.0) < 0.02  # variance 1/nao
    Ls = make_cluster(ClusterSpec(7, 4, 100, 10, 90, 40, 2, "std")).L_packed()
    assert np.allclose(Ls * 10.0, Lb)  # std 1/nao variant is the same draw rescaled


def test_orbital_subsets_are_seeded_sorted_and_keep_both_ends():
    """The column subsets of the 'dense aux x k dense virtuals / occupieds' full-size goldens."""
    from workloads import occupied_subset, virtual_subset

    spec = config_specs(4)[6]
    for pick, n, k in ((virtual_subset, spec.nvir, 256), (occupied_subset, spec.nocc, 8)):
        s = pick(spec, k)
        assert s.dtype == np.int64 and s.shape == (k,) and np.array_equal(s, pick(spec, k))
        assert s[0] == 0 and s[-1] == n - 1 and np.all(np.diff(s) > 0)
    # independent streams: the two choices of one spec are not prefixes of one another, other clusters draw other columns
    assert not np.array_equal(occupied_subset(spec, 8), virtual_subset(spec, 8))
    assert not np.array_equal(occupied_subset(spec, 8), occupied_subset(config_specs(4)[4], 8))
