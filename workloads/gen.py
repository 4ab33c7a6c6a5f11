"""Seeded input generators for the five BASELINE.json configs.

Recipe (DESIGN.md §3 "Input recipe"; readings A-9..A-14 of SURVEY.md §8(c)):

* ``C``      : nao x nao orthogonal matrix = Q of QR(Gaussian), columns sign-normalised so
               diag(R) > 0; first ``nocc`` columns occupied, next ``nvir`` virtual.
* ``(P|mu nu)``: the PACKED lower triangle (mu >= nu, idx = mu(mu+1)/2 + nu, aux index slowest)
               is drawn directly, every stored element i.i.d. N(0, variance 1/nao)
               (``scale="var"``, the default) or N(0, std 1/nao) (``scale="std"``).
               One child RNG stream per aux index P, so any aux blocking yields the same tensor
               and the 28 GB tensor of config 3 never has to exist at once.
* ``e_occ``  : uniform in [-1.5, -0.3];  ``e_vir``: uniform in [0.1, 3.0]  (unsorted).
* ``P_frag`` : Q Q^T with Q = sign-normalised QR(Gaussian nocc x rank); rank 0 means identity.

No arithmetic of the method lives here: this file only draws numbers.
"""
from __future__ import annotations

import dataclasses
from concurrent.futures import ThreadPoolExecutor
from typing import List, Optional

import numpy as np

# stream ids inside SeedSequence([config_id, cluster_id, stream_id])
_S_C, _S_EOCC, _S_EVIR, _S_Q, _S_NOCC, _S_SUBSET, _S_OSUBSET = 1, 2, 3, 4, 5, 6, 7
_S_L0 = 100  # aux index P uses stream 100 + P


def npair(nao: int) -> int:
    """Number of stored elements of one packed symmetric nao x nao matrix."""
    return nao * (nao + 1) // 2


@dataclasses.dataclass(frozen=True)
class ClusterSpec:
    config_id: int
    cluster_id: int
    nao: int
    nocc: int
    nvir: int
    naux: int
    rank: int  # 0 => P_frag = identity
    scale: str = "var"  # "var": N(0, variance 1/nao); "std": N(0, std 1/nao)

    @property
    def npair(self) -> int:
        return npair(self.nao)

    def with_(self, **kw) -> "ClusterSpec":
        return dataclasses.replace(self, **kw)


def _rng(spec: ClusterSpec, stream: int) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([spec.config_id, spec.cluster_id, stream]))


def _orthonormal(rng: np.random.Generator, n: int, k: int) -> np.ndarray:
    """Q (n x k) of QR(Gaussian n x k), column signs fixed so that diag(R) > 0 (reading A-11)."""
    a = rng.standard_normal((n, k))
    q, r = np.linalg.qr(a)
    s = np.sign(np.diag(r))
    s[s == 0] = 1.0
    return np.ascontiguousarray(q * s[None, :])


class ClusterInputs:
    """Host-side inputs of one cluster. ``L`` is produced lazily, block by block."""

    def __init__(self, spec: ClusterSpec):
        self.spec = spec
        nao, nocc, nvir = spec.nao, spec.nocc, spec.nvir
        assert nocc >= 1 and nvir >= 1 and nocc + nvir <= nao and spec.naux >= 1
        C = _orthonormal(_rng(spec, _S_C), nao, nao)
        self.C_occ = np.ascontiguousarray(C[:, :nocc])  # [nao][nocc]
        self.C_vir = np.ascontiguousarray(C[:, nocc:nocc + nvir])  # [nao][nvir]
        self.e_occ = _rng(spec, _S_EOCC).uniform(-1.5, -0.3, size=nocc)
        self.e_vir = _rng(spec, _S_EVIR).uniform(0.1, 3.0, size=nvir)
        if spec.rank <= 0:
            self.Q_frag = np.eye(nocc)  # [nocc][rank]: the fragment orbitals in the cluster's occupied basis
            self.P_frag = np.eye(nocc)
        else:
            q = _orthonormal(_rng(spec, _S_Q), nocc, min(spec.rank, nocc))
            self.Q_frag = q
            self.P_frag = np.ascontiguousarray(q @ q.T)

    @property
    def sigma(self) -> float:
        nao = self.spec.nao
        return nao ** -0.5 if self.spec.scale == "var" else 1.0 / nao

    def _fill_row(self, out: np.ndarray, p: int) -> None:
        g = _rng(self.spec, _S_L0 + p)
        g.standard_normal(out=out)
        out *= self.sigma

    def L_block(self, p0: int, p1: int, out: Optional[np.ndarray] = None, threads: int = 1) -> np.ndarray:
        """Packed (P|mu nu) rows [p0, p1): array [(p1-p0)][npair], C-contiguous float64."""
        assert 0 <= p0 <= p1 <= self.spec.naux
        n = self.spec.npair
        if out is None:
            out = np.empty((p1 - p0, n), dtype=np.float64)
        assert out.shape == (p1 - p0, n) and out.dtype == np.float64 and out.flags.c_contiguous
        if threads <= 1 or p1 - p0 < 2:
            for p in range(p0, p1):
                self._fill_row(out[p - p0], p)
        else:
            with ThreadPoolExecutor(max_workers=threads) as ex:
                list(ex.map(lambda p: self._fill_row(out[p - p0], p), range(p0, p1)))
        return out

    def L_packed(self, threads: int = 1) -> np.ndarray:
        return self.L_block(0, self.spec.naux, threads=threads)


def virtual_subset(spec: ClusterSpec, k: int) -> np.ndarray:
    """Sorted, seeded choice of ``k`` of the ``nvir`` virtual columns, always containing the first and the last one.

    Used by the "dense aux x k dense virtuals" full-size parity case: C_vir is zeroed outside these
    columns, so the CPU side only needs the compressed problem while the GPU runs the full-size launch."""
    assert 2 <= k <= spec.nvir
    r = _rng(spec, _S_SUBSET)
    inner = r.choice(np.arange(1, spec.nvir - 1), size=k - 2, replace=False)
    return np.sort(np.concatenate([[0, spec.nvir - 1], inner])).astype(np.int64)


def occupied_subset(spec: ClusterSpec, k: int) -> np.ndarray:
    """Sorted, seeded choice of ``k`` of the ``nocc`` occupied columns, always containing the first and the last one
    (the "dense aux x dense virtuals x k dense occupieds" full-size parity case: C_occ is zeroed outside these columns)."""
    assert 2 <= k <= spec.nocc
    r = _rng(spec, _S_OSUBSET)
    inner = r.choice(np.arange(1, spec.nocc - 1), size=k - 2, replace=False)
    return np.sort(np.concatenate([[0, spec.nocc - 1], inner])).astype(np.int64)


def make_cluster(spec: ClusterSpec) -> ClusterInputs:
    return ClusterInputs(spec)


def _sized(config_id, cluster_id, nocc, nvir, naux, rank, scale) -> ClusterSpec:
    return ClusterSpec(config_id, cluster_id, nocc + nvir, nocc, nvir, naux, rank, scale)


def config_specs(config_id: int, scale: str = "var") -> List[ClusterSpec]:
    """Cluster list of BASELINE.json ``configs[config_id]``.

    Config 1 and 4 are run with the random projector and with P_frag = I: G does not depend on
    P_frag (reading A-15), so those variants share all other inputs (same cluster_id) and differ
    only in ``rank`` (0 = identity).
    """
    if config_id == 0:  # tiny: nao=48 (8+40), naux=160, rank 4
        return [_sized(0, 0, 8, 40, 160, 4, scale)]
    if config_id == 1:  # medium: nao=300 (30+270), naux=1200, rank nocc/2; plus P=I
        return [_sized(1, 0, 30, 270, 1200, 15, scale), _sized(1, 0, 30, 270, 1200, 0, scale)]
    if config_id == 2:  # batch of 96: nocc~U{16..48}, nvir=8 nocc, naux=4 nao, rank nocc/4
        out = []
        for c in range(96):
            r = np.random.default_rng(np.random.SeedSequence([2, c, _S_NOCC]))
            nocc = int(r.integers(16, 48, endpoint=True))
            out.append(_sized(2, c, nocc, 8 * nocc, 4 * 9 * nocc, max(1, nocc // 4), scale))
        return out
    if config_id == 3:  # large: nao=1200 (120+1080), naux=4800, rank 60
        return [_sized(3, 0, 120, 1080, 4800, 60, scale)]
    if config_id == 4:  # sweep: nocc=64, nvir in {256..2048}, naux=4 nao, P=I and rank 32
        out = []
        for k, nvir in enumerate((256, 512, 1024, 2048)):
            out.append(_sized(4, k, 64, nvir, 4 * (64 + nvir), 32, scale))
            out.append(_sized(4, k, 64, nvir, 4 * (64 + nvir), 0, scale))
        return out
    raise ValueError(f"unknown config {config_id}")
