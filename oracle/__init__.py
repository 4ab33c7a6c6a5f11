"""CPU oracle for the fragment-projected DF-MP2 path — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It is a ctypes veneer over oracle/dfmp2_oracle.c (explicit FP64 loops; see
that file's header for the step list O1-O7 and the paper citations).  It shares nothing with
paper_2412_18553_b200/ and imports nothing from it.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Tuple

import numpy as np

from . import build as _build

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        L.sie_oracle_threads.restype = ctypes.c_int
        L.sie_oracle_set_threads.argtypes = [ctypes.c_int]
        L.sie_oracle_unpack.argtypes = [ctypes.c_int, dp, dp]
        L.sie_oracle_transform.argtypes = [ctypes.c_int] * 6 + [dp, dp, dp, dp]
        L.sie_oracle_transform.restype = ctypes.c_int
        L.sie_oracle_pair_G.argtypes = [ctypes.c_int] * 3 + [dp, dp, dp, ctypes.c_int, ctypes.c_int, dp]
        L.sie_oracle_pair_G.restype = ctypes.c_int
        L.sie_oracle_rdm_occ.argtypes = [ctypes.c_int] * 3 + [dp, dp, dp, dp]
        L.sie_oracle_rdm_occ.restype = ctypes.c_int
        L.sie_oracle_rdm_vir.argtypes = [ctypes.c_int] * 3 + [dp, dp, dp, dp]
        L.sie_oracle_rdm_vir.restype = ctypes.c_int
        L.sie_oracle_trace.argtypes = [ctypes.c_int, dp, dp]
        L.sie_oracle_trace.restype = ctypes.c_double
        _lib = L
    return _lib


def _p(a: Optional[np.ndarray]):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def threads() -> int:
    return int(lib().sie_oracle_threads())


def set_threads(n: int) -> None:
    lib().sie_oracle_set_threads(int(n))


def unpack(Lp_row: np.ndarray, nao: int) -> np.ndarray:
    """O1 for one aux index: packed [npair] -> full [nao][nao]."""
    Lp_row = _c(Lp_row)
    assert Lp_row.shape == (nao * (nao + 1) // 2,)
    out = np.empty((nao, nao))
    lib().sie_oracle_unpack(nao, _p(Lp_row), _p(out))
    return out


def transform_block(C_occ, C_vir, Lp_block, p0: int, p1: int, B: np.ndarray) -> None:
    """O1-O3 for aux rows [p0,p1): fills B[i][a][p0:p1] (B is [nocc][nvir][naux])."""
    C_occ, C_vir, Lp_block = _c(C_occ), _c(C_vir), _c(Lp_block)
    nao, nocc = C_occ.shape
    nvir = C_vir.shape[1]
    naux = B.shape[2]
    assert C_vir.shape[0] == nao and B.shape == (nocc, nvir, naux)
    assert Lp_block.shape == (p1 - p0, nao * (nao + 1) // 2) and 0 <= p0 <= p1 <= naux
    rc = lib().sie_oracle_transform(nao, nocc, nvir, naux, p0, p1, _p(C_occ), _p(C_vir), _p(Lp_block), _p(B))
    if rc != 0:
        raise MemoryError("sie_oracle_transform")


def transform(C_occ, C_vir, L_packed) -> np.ndarray:
    """O1-O3: B[i][a][P] from the whole packed tensor [naux][npair]."""
    L_packed = _c(L_packed)
    B = np.zeros((C_occ.shape[1], C_vir.shape[1], L_packed.shape[0]))
    transform_block(C_occ, C_vir, L_packed, 0, L_packed.shape[0], B)
    return B


def pair_G(B, e_occ, e_vir, j0: int = 0, j1: Optional[int] = None) -> np.ndarray:
    """O4-O6: G[i'][i] summed over j in [j0,j1) (default: all j)."""
    B, e_occ, e_vir = _c(B), _c(e_occ), _c(e_vir)
    nocc, nvir, naux = B.shape
    assert e_occ.shape == (nocc,) and e_vir.shape == (nvir,)
    if j1 is None:
        j1 = nocc
    assert 0 <= j0 <= j1 <= nocc
    G = np.empty((nocc, nocc))
    rc = lib().sie_oracle_pair_G(nocc, nvir, naux, _p(B), _p(e_occ), _p(e_vir), j0, j1, _p(G))
    if rc != 0:
        raise MemoryError("sie_oracle_pair_G")
    return G


def rdm_occ(B, e_occ, e_vir) -> np.ndarray:
    """Occupied block of the MP2 1-RDM, gamma_ij of PAPER.md Eq. S18 (L357): [nocc][nocc]."""
    B, e_occ, e_vir = _c(B), _c(e_occ), _c(e_vir)
    nocc, nvir, naux = B.shape
    assert e_occ.shape == (nocc,) and e_vir.shape == (nvir,)
    g = np.empty((nocc, nocc))
    rc = lib().sie_oracle_rdm_occ(nocc, nvir, naux, _p(B), _p(e_occ), _p(e_vir), _p(g))
    if rc != 0:
        raise MemoryError("sie_oracle_rdm_occ")
    return g


def rdm_vir(B, e_occ, e_vir) -> np.ndarray:
    """Virtual block of the MP2 1-RDM, gamma_ab of PAPER.md Eq. S17 (L355): [nvir][nvir]."""
    B, e_occ, e_vir = _c(B), _c(e_occ), _c(e_vir)
    nocc, nvir, naux = B.shape
    assert e_occ.shape == (nocc,) and e_vir.shape == (nvir,)
    g = np.empty((nvir, nvir))
    rc = lib().sie_oracle_rdm_vir(nocc, nvir, naux, _p(B), _p(e_occ), _p(e_vir), _p(g))
    if rc != 0:
        raise MemoryError("sie_oracle_rdm_vir")
    return g


def trace(P_frag, G) -> float:
    """O7: E_frag = sum_{i,i'} P[i][i'] G[i'][i]; P_frag=None means identity."""
    G = _c(G)
    P = None if P_frag is None else _c(P_frag)
    return float(lib().sie_oracle_trace(G.shape[0], _p(P), _p(G)))


def dfmp2(C_occ, C_vir, L_packed, e_occ, e_vir, P_frag) -> Tuple[float, np.ndarray]:
    """Whole path O1-O7 for one cluster: returns (E_frag, G)."""
    B = transform(C_occ, C_vir, L_packed)
    G = pair_G(B, e_occ, e_vir)
    return trace(P_frag, G), G
