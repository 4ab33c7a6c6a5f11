"""Thin Python binding of libsie_dfmp2.so (include/sie_dfmp2.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device memory
(the workspace and the operand tensors) and streams.  There is no CPU fallback: a missing library or a
missing GPU raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import List, Optional, Sequence, Tuple

import torch

SIE_OK, SIE_EINVAL, SIE_ENOMEM, SIE_ECUDA, SIE_ESTATE, SIE_EGAP, SIE_EUNSUPPORTED, SIE_ETOOBIG = range(8)
SIE_FLAG_VALIDATE, SIE_FLAG_REFERENCE, SIE_FLAG_HOST_IO, SIE_FLAG_PROFILE, SIE_FLAG_RDM_OCC, SIE_FLAG_RDM_VIR, SIE_FLAG_STAGE_FULL = 1, 2, 4, 8, 16, 32, 64

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsie_dfmp2.so")

EXPORTS = (
    "sie_dfmp2_plan",
    "sie_dfmp2_transform",
    "sie_dfmp2_energy",
    "sie_dfmp2_energy_lowrank",
    "sie_dfmp2_energy_noalloc",
    "sie_dfmp2_noalloc_bytes",
    "sie_dfmp2_noalloc_capacity",
    "sie_dfmp2_rdm_occ",
    "sie_dfmp2_rdm_vir",
    "sie_dfmp2_batch",
    "sie_dfmp2_plan_reset",
    "sie_dfmp2_canonical_plan",
    "sie_dfmp2_canonical_transform",
    "sie_dfmp2_canonical_energy",
    "sie_dfmp2_canonical_info",
    "sie_dfmp2_canonical_destroy",
    "sie_dfmp2_destroy",
    "sie_dfmp2_strerror",
    "sie_dfmp2_last_cuda_error",
    "sie_dfmp2_launch_count",
    "sie_dfmp2_plan_info",
    "sie_dfmp2_plan_timing",
    "sie_dfmp2_batch_timing",
    "sie_dfmp2_probe_fp64",
)


class SieError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = _lib().sie_dfmp2_strerror(status).decode()
        if status == SIE_ECUDA:
            msg += " — " + _lib().sie_dfmp2_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} (status {status})")


class sie_dfmp2_cluster_t(ctypes.Structure):
    _fields_ = [
        ("nao", ctypes.c_int),
        ("nocc", ctypes.c_int),
        ("nvir", ctypes.c_int),
        ("naux", ctypes.c_int),
        ("C_occ", ctypes.c_void_p),
        ("C_vir", ctypes.c_void_p),
        ("L_packed", ctypes.c_void_p),
        ("e_occ", ctypes.c_void_p),
        ("e_vir", ctypes.c_void_p),
        ("P_frag", ctypes.c_void_p),
        ("E_out", ctypes.c_void_p),
        ("G_out", ctypes.c_void_p),
    ]


_LIB = None


def _lib() -> ctypes.CDLL:
    """Load the CUDA library; raise loudly if it has not been built (no fallback exists)."""
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2412_18553_b200.build` "
                "(nvcc, sm_100a). There is no CPU fallback."
            )
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cu = ctypes.c_void_p, ctypes.c_int, ctypes.c_uint
        L.sie_dfmp2_plan.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, cu, ctypes.POINTER(ctypes.c_size_t)]
        L.sie_dfmp2_plan.restype = ci
        L.sie_dfmp2_transform.argtypes = [vp, vp, vp, vp, vp, ci, ci, vp]
        L.sie_dfmp2_transform.restype = ci
        L.sie_dfmp2_energy.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
        L.sie_dfmp2_energy.restype = ci
        L.sie_dfmp2_rdm_occ.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.sie_dfmp2_rdm_occ.restype = ci
        L.sie_dfmp2_energy_lowrank.argtypes = [vp, vp, vp, vp, vp, ci, vp, vp]
        L.sie_dfmp2_energy_lowrank.restype = ci
        L.sie_dfmp2_energy_noalloc.argtypes = [ci, ci, ci, vp, vp, vp, vp, vp, vp, vp]
        L.sie_dfmp2_energy_noalloc.restype = ci
        L.sie_dfmp2_noalloc_bytes.argtypes = [ci, ci]
        L.sie_dfmp2_noalloc_bytes.restype = ctypes.c_size_t
        L.sie_dfmp2_noalloc_capacity.argtypes = []
        L.sie_dfmp2_noalloc_capacity.restype = ctypes.c_size_t
        L.sie_dfmp2_rdm_vir.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.sie_dfmp2_rdm_vir.restype = ci
        L.sie_dfmp2_batch.argtypes = [ci, ctypes.POINTER(sie_dfmp2_cluster_t), vp, ctypes.c_size_t, ctypes.POINTER(ctypes.c_size_t), cu, vp]
        L.sie_dfmp2_batch.restype = ci
        L.sie_dfmp2_canonical_plan.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, ctypes.POINTER(ctypes.c_size_t), ctypes.POINTER(ctypes.c_size_t)]
        L.sie_dfmp2_canonical_plan.restype = ci
        L.sie_dfmp2_canonical_transform.argtypes = [vp, vp, vp, vp, vp, ci, ci, vp, vp]
        L.sie_dfmp2_canonical_transform.restype = ci
        L.sie_dfmp2_canonical_energy.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.sie_dfmp2_canonical_energy.restype = ci
        L.sie_dfmp2_canonical_info.argtypes = [vp, ctypes.POINTER(ctypes.c_longlong), ci]
        L.sie_dfmp2_canonical_info.restype = ci
        L.sie_dfmp2_canonical_destroy.argtypes = [vp]
        L.sie_dfmp2_canonical_destroy.restype = ci
        L.sie_dfmp2_plan_reset.argtypes = [vp]
        L.sie_dfmp2_plan_reset.restype = ci
        L.sie_dfmp2_destroy.argtypes = [vp]
        L.sie_dfmp2_destroy.restype = ci
        L.sie_dfmp2_strerror.argtypes = [ci]
        L.sie_dfmp2_strerror.restype = ctypes.c_char_p
        L.sie_dfmp2_last_cuda_error.argtypes = []
        L.sie_dfmp2_last_cuda_error.restype = ctypes.c_char_p
        L.sie_dfmp2_launch_count.argtypes = []
        L.sie_dfmp2_launch_count.restype = ctypes.c_ulonglong
        L.sie_dfmp2_plan_info.argtypes = [vp, ctypes.POINTER(ctypes.c_longlong), ci]
        L.sie_dfmp2_plan_info.restype = ci
        dp = ctypes.POINTER(ctypes.c_double)
        L.sie_dfmp2_plan_timing.argtypes = [vp, dp, ci]
        L.sie_dfmp2_plan_timing.restype = ci
        L.sie_dfmp2_batch_timing.argtypes = [dp, ci]
        L.sie_dfmp2_batch_timing.restype = ci
        L.sie_dfmp2_probe_fp64.argtypes = [ci, ci, ci, vp, dp, dp, vp]
        L.sie_dfmp2_probe_fp64.restype = ci
        _LIB = L
    return _LIB


def _check(status: int, where: str) -> None:
    if status != SIE_OK:
        raise SieError(status, where)


def _ptr(t: Optional[torch.Tensor], host: bool, name: str) -> Optional[int]:
    if t is None:
        return None
    if t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name}: need a contiguous float64 tensor")
    if host and t.is_cuda:
        raise TypeError(f"{name}: SIE_FLAG_HOST_IO needs host tensors")
    if not host and not t.is_cuda:
        raise TypeError(f"{name}: need a CUDA tensor (or plan with SIE_FLAG_HOST_IO)")
    return t.data_ptr()


def _stream_ptr(stream: Optional[torch.cuda.Stream]) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


def launch_count() -> int:
    return int(_lib().sie_dfmp2_launch_count())


# ------------------------------------------------------------------------------------------------ C-ABI names
def sie_dfmp2_plan(nao: int, nocc: int, nvir: int, naux: int, aux_block: int = 0, flags: int = 0) -> Tuple[int, int]:
    """-> (plan handle, workspace bytes)."""
    h = ctypes.c_void_p()
    ws = ctypes.c_size_t()
    _check(_lib().sie_dfmp2_plan(ctypes.byref(h), nao, nocc, nvir, naux, aux_block, flags, ctypes.byref(ws)), "sie_dfmp2_plan")
    return h.value, ws.value


def sie_dfmp2_transform(plan: int, workspace: torch.Tensor, C_occ, C_vir, L_packed_block, p0: int, p1: int, *, host=False, stream=None) -> None:
    _check(
        _lib().sie_dfmp2_transform(
            plan, workspace.data_ptr(), _ptr(C_occ, host, "C_occ"), _ptr(C_vir, host, "C_vir"),
            _ptr(L_packed_block, host, "L_packed_block"), p0, p1, _stream_ptr(stream)),
        "sie_dfmp2_transform",
    )


def sie_dfmp2_rdm_occ(plan: int, workspace: torch.Tensor, e_occ, e_vir, gamma_out, trace_out=None, *, host=False, stream=None) -> None:
    """Occupied block of the MP2 1-RDM (PAPER.md Eq. S18) on the transformed workspace; marshalling only."""
    _check(
        _lib().sie_dfmp2_rdm_occ(
            plan, workspace.data_ptr(), _ptr(e_occ, host, "e_occ"), _ptr(e_vir, host, "e_vir"), _ptr(gamma_out, host, "gamma_out"),
            _ptr(trace_out, host, "trace_out"), _stream_ptr(stream)),
        "sie_dfmp2_rdm_occ",
    )


def sie_dfmp2_energy_lowrank(plan: int, workspace: torch.Tensor, e_occ, e_vir, Q, E_out, *, host=False, stream=None) -> None:
    """E_frag = Tr(Q Q^T G) for a factored projector Q [nocc][r] (PAPER.md Eq. S33/S45); marshalling only."""
    if Q.dim() != 2:
        raise TypeError("Q: need a [nocc][r] matrix")
    _check(
        _lib().sie_dfmp2_energy_lowrank(
            plan, workspace.data_ptr(), _ptr(e_occ, host, "e_occ"), _ptr(e_vir, host, "e_vir"), _ptr(Q, host, "Q"), int(Q.shape[1]),
            _ptr(E_out, host, "E_out"), _stream_ptr(stream)),
        "sie_dfmp2_energy_lowrank",
    )


def sie_dfmp2_energy_noalloc(nocc: int, nvir: int, naux: int, B, e_occ, e_vir, P_frag, E_out, G_out, *, stream=None) -> None:
    """Pair stage + trace with the library's static device scratch (no workspace, no device allocation); marshalling only.
    B: device tensor holding [nvir][nocc][ceil8(naux)] doubles (any shape/view, 16-byte aligned)."""
    if B.dtype not in (torch.float64, torch.uint8) or not B.is_cuda or not B.is_contiguous():
        raise TypeError("B: need a contiguous CUDA tensor")
    _check(
        _lib().sie_dfmp2_energy_noalloc(nocc, nvir, naux, B.data_ptr(), _ptr(e_occ, False, "e_occ"), _ptr(e_vir, False, "e_vir"),
                                        _ptr(P_frag, False, "P_frag"), _ptr(E_out, False, "E_out"), _ptr(G_out, False, "G_out"),
                                        _stream_ptr(stream)),
        "sie_dfmp2_energy_noalloc",
    )


def sie_dfmp2_noalloc_bytes(nocc: int, nvir: int) -> int:
    return int(_lib().sie_dfmp2_noalloc_bytes(nocc, nvir))


def sie_dfmp2_noalloc_capacity() -> int:
    return int(_lib().sie_dfmp2_noalloc_capacity())


def sie_dfmp2_rdm_vir(plan: int, workspace: torch.Tensor, e_occ, e_vir, gamma_out, trace_out=None, *, host=False, stream=None) -> None:
    """Virtual block of the MP2 1-RDM (PAPER.md Eq. S17); the plan needs SIE_FLAG_RDM_VIR; marshalling only."""
    _check(
        _lib().sie_dfmp2_rdm_vir(
            plan, workspace.data_ptr(), _ptr(e_occ, host, "e_occ"), _ptr(e_vir, host, "e_vir"), _ptr(gamma_out, host, "gamma_out"),
            _ptr(trace_out, host, "trace_out"), _stream_ptr(stream)),
        "sie_dfmp2_rdm_vir",
    )


def sie_dfmp2_energy(plan: int, workspace: torch.Tensor, e_occ, e_vir, P_frag, E_out, G_out, *, host=False, stream=None) -> None:
    _check(
        _lib().sie_dfmp2_energy(
            plan, workspace.data_ptr(), _ptr(e_occ, host, "e_occ"), _ptr(e_vir, host, "e_vir"), _ptr(P_frag, host, "P_frag"),
            _ptr(E_out, host, "E_out"), _ptr(G_out, host, "G_out"), _stream_ptr(stream)),
        "sie_dfmp2_energy",
    )


def sie_dfmp2_plan_reset(plan: int) -> None:
    _check(_lib().sie_dfmp2_plan_reset(plan), "sie_dfmp2_plan_reset")


def sie_dfmp2_destroy(plan: Optional[int]) -> None:
    if plan:
        _lib().sie_dfmp2_destroy(plan)


def sie_dfmp2_plan_info(plan: int) -> dict:
    buf = (ctypes.c_longlong * 8)()
    n = _lib().sie_dfmp2_plan_info(plan, buf, 8)
    keys = ("TM", "TN", "ta", "o8", "ntiles", "ncta", "aux_subblock", "route")
    d = {k: int(buf[i]) for i, k in enumerate(keys[:n])}
    d["reference"], d["general"] = int(d.get("route") == 1), int(d.get("route") == 2)  # pair-stage route: 0 fused, 1 reference, 2 general
    return d


STAGES = ("coeff_transpose", "unpack", "A1_gemm", "A2_gemm", "pair", "reduce", "reference")


def _timing_dict(buf) -> dict:
    n = len(STAGES)
    return {"ms": {k: float(buf[i]) for i, k in enumerate(STAGES)}, "launch_groups": {k: int(buf[n + i]) for i, k in enumerate(STAGES)}}


def sie_dfmp2_plan_timing(plan: int) -> dict:
    """Per-stage device milliseconds since the last query (plan created with SIE_FLAG_PROFILE)."""
    buf = (ctypes.c_double * (2 * len(STAGES)))()
    _check(_lib().sie_dfmp2_plan_timing(plan, buf, len(buf)), "sie_dfmp2_plan_timing")
    return _timing_dict(buf)


def sie_dfmp2_batch_timing() -> dict:
    buf = (ctypes.c_double * (2 * len(STAGES)))()
    _check(_lib().sie_dfmp2_batch_timing(buf, len(buf)), "sie_dfmp2_batch_timing")
    return _timing_dict(buf)


def sie_dfmp2_probe_fp64(kind: int, iters: int = 20000, ctas_per_sm: int = 2, *, stream=None) -> Tuple[float, float]:
    """-> (TFLOP/s, ms) of the FP64 issue-rate microkernel `kind` (0 DMMA, 1 DFMA, 2 smem-fed DMMA)."""
    scratch = torch.zeros(8, dtype=torch.float64, device="cuda")
    tf, ms = ctypes.c_double(), ctypes.c_double()
    _check(_lib().sie_dfmp2_probe_fp64(kind, iters, ctas_per_sm, scratch.data_ptr(), ctypes.byref(tf), ctypes.byref(ms), _stream_ptr(stream)),
           "sie_dfmp2_probe_fp64")
    return tf.value, ms.value


def _descs(clusters: Sequence[dict], host: bool) -> ctypes.Array:
    arr = (sie_dfmp2_cluster_t * max(1, len(clusters)))()
    for k, c in enumerate(clusters):
        d = arr[k]
        d.nao, d.nocc, d.nvir, d.naux = c["nao"], c["nocc"], c["nvir"], c["naux"]
        for f in ("C_occ", "C_vir", "L_packed", "e_occ", "e_vir", "P_frag", "E_out", "G_out"):
            setattr(d, f, _ptr(c.get(f), host, f))
    return arr


def sie_dfmp2_batch_query(clusters: Sequence[dict], flags: int = 0) -> int:
    """Workspace bytes needed for this batch.  Sizes are enough; when the L_packed tensors are given too, clusters that
    share one tensor are laid out as a shared-integral group (never larger than the private layout)."""
    arr = (sie_dfmp2_cluster_t * max(1, len(clusters)))()
    host = bool(flags & SIE_FLAG_HOST_IO)
    for k, c in enumerate(clusters):
        arr[k].nao, arr[k].nocc, arr[k].nvir, arr[k].naux = c["nao"], c["nocc"], c["nvir"], c["naux"]
        if c.get("L_packed") is not None:
            arr[k].L_packed = _ptr(c["L_packed"], host, "L_packed")
    need = ctypes.c_size_t()
    _check(_lib().sie_dfmp2_batch(len(clusters), arr, None, 0, ctypes.byref(need), flags, None), "sie_dfmp2_batch(query)")
    return need.value


def sie_dfmp2_batch(clusters: Sequence[dict], workspace: torch.Tensor, flags: int = 0, *, stream=None) -> None:
    """clusters: dicts with nao,nocc,nvir,naux and tensors C_occ,C_vir,L_packed,e_occ,e_vir,P_frag|None,E_out,G_out|None."""
    host = bool(flags & SIE_FLAG_HOST_IO)
    arr = _descs(clusters, host)
    need = ctypes.c_size_t()
    _check(
        _lib().sie_dfmp2_batch(len(clusters), arr, workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                               ctypes.byref(need), flags, _stream_ptr(stream)),
        "sie_dfmp2_batch",
    )


# ------------------------------------------------------------------------------------------------ NEXT-2: canonical, out of core
class CanonicalSolver:
    """Whole-system canonical DF-MP2 energy (sie_dfmp2_canonical_*).  The B store is a pinned host tensor
    (``store="host"``, the out-of-core case) or a device tensor (``store="device"``).  Marshalling only."""

    def __init__(self, nao: int, nocc: int, nvir: int, naux: int, occ_block: int = 0, store: str = "host", device="cuda"):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2412_18553_b200 needs a CUDA device (B200, sm_100a); there is no CPU path")
        h, ws, bs = ctypes.c_void_p(), ctypes.c_size_t(), ctypes.c_size_t()
        _check(_lib().sie_dfmp2_canonical_plan(ctypes.byref(h), nao, nocc, nvir, naux, occ_block, ctypes.byref(ws), ctypes.byref(bs)),
               "sie_dfmp2_canonical_plan")
        self.plan, self.workspace_bytes, self.bstore_bytes = h.value, ws.value, bs.value
        self.workspace = alloc_workspace(self.workspace_bytes, device)
        n = self.bstore_bytes // 8
        self.B_store = torch.empty(n, dtype=torch.float64, device=device) if store == "device" else torch.empty(n, dtype=torch.float64).pin_memory()
        self.device = device

    def info(self) -> dict:
        buf = (ctypes.c_longlong * 4)()
        _lib().sie_dfmp2_canonical_info(self.plan, buf, 4)
        return dict(zip(("occ_block", "aux_subblock", "n_occ_blocks", "panel_bytes"), (int(x) for x in buf)))

    def transform(self, C_occ, C_vir, L_block, p0: int, p1: int, stream=None) -> None:
        _check(_lib().sie_dfmp2_canonical_transform(self.plan, self.workspace.data_ptr(), _ptr(C_occ, False, "C_occ"), _ptr(C_vir, False, "C_vir"),
                                                    _ptr(L_block, False, "L_packed_block"), p0, p1, self.B_store.data_ptr(), _stream_ptr(stream)),
               "sie_dfmp2_canonical_transform")

    def energy(self, e_occ, e_vir, stream=None) -> torch.Tensor:
        E = torch.empty(1, dtype=torch.float64, device=self.device)
        _check(_lib().sie_dfmp2_canonical_energy(self.plan, self.workspace.data_ptr(), _ptr(e_occ, False, "e_occ"), _ptr(e_vir, False, "e_vir"),
                                                 self.B_store.data_ptr(), E.data_ptr(), _stream_ptr(stream)),
               "sie_dfmp2_canonical_energy")
        return E

    def close(self) -> None:
        if self.plan:
            _lib().sie_dfmp2_canonical_destroy(self.plan)
        self.plan = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ------------------------------------------------------------------------------------------------ convenience
def alloc_workspace(nbytes: int, device="cuda") -> torch.Tensor:
    """A 256-byte aligned uint8 device tensor (torch's caching allocator returns 512-byte aligned blocks)."""
    t = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
    assert t.data_ptr() % 256 == 0
    return t


class ClusterSolver:
    """One cluster: plan + workspace, transform fed by aux blocks, then energy.  Marshalling only."""

    def __init__(self, nao: int, nocc: int, nvir: int, naux: int, aux_block: int = 0, flags: int = 0, device="cuda"):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2412_18553_b200 needs a CUDA device (B200, sm_100a); there is no CPU path")
        self.nao, self.nocc, self.nvir, self.naux, self.flags = nao, nocc, nvir, naux, flags
        self.host = bool(flags & SIE_FLAG_HOST_IO)
        self.plan, self.workspace_bytes = sie_dfmp2_plan(nao, nocc, nvir, naux, aux_block, flags)
        self.workspace = alloc_workspace(self.workspace_bytes, device)
        self.device = device

    def info(self) -> dict:
        return sie_dfmp2_plan_info(self.plan)

    def transform(self, C_occ, C_vir, L_block, p0: int, p1: int, stream=None) -> None:
        sie_dfmp2_transform(self.plan, self.workspace, C_occ, C_vir, L_block, p0, p1, host=self.host, stream=stream)

    def energy(self, e_occ, e_vir, P_frag=None, want_G: bool = True, stream=None):
        dev = "cpu" if self.host else self.device
        E = torch.empty(1, dtype=torch.float64, device=dev)
        G = torch.empty(self.nocc, self.nocc, dtype=torch.float64, device=dev) if want_G else None
        if self.host:
            E, G = E.pin_memory(), (G.pin_memory() if G is not None else None)
        sie_dfmp2_energy(self.plan, self.workspace, e_occ, e_vir, P_frag, E, G, host=self.host, stream=stream)
        return E, G

    def energy_lowrank(self, e_occ, e_vir, Q, stream=None):
        """-> E_frag = Tr(Q Q^T G) for a factored projector Q [nocc][r]"""
        E = torch.empty(1, dtype=torch.float64, device="cpu" if self.host else self.device)
        if self.host:
            E = E.pin_memory()
        sie_dfmp2_energy_lowrank(self.plan, self.workspace, e_occ, e_vir, Q, E, host=self.host, stream=stream)
        return E

    def rdm_occ(self, e_occ, e_vir, stream=None):
        """-> (gamma [nocc][nocc], Tr gamma)"""
        dev = "cpu" if self.host else self.device
        g = torch.empty(self.nocc, self.nocc, dtype=torch.float64, device=dev)
        tr = torch.empty(1, dtype=torch.float64, device=dev)
        if self.host:
            g, tr = g.pin_memory(), tr.pin_memory()
        sie_dfmp2_rdm_occ(self.plan, self.workspace, e_occ, e_vir, g, tr, host=self.host, stream=stream)
        return g, tr

    def rdm_vir(self, e_occ, e_vir, stream=None):
        """-> (gamma_vir [nvir][nvir], Tr gamma_vir); the solver must have been created with SIE_FLAG_RDM_VIR"""
        dev = "cpu" if self.host else self.device
        g = torch.empty(self.nvir, self.nvir, dtype=torch.float64, device=dev)
        tr = torch.empty(1, dtype=torch.float64, device=dev)
        if self.host:
            g, tr = g.pin_memory(), tr.pin_memory()
        sie_dfmp2_rdm_vir(self.plan, self.workspace, e_occ, e_vir, g, tr, host=self.host, stream=stream)
        return g, tr

    def timing(self) -> dict:
        return sie_dfmp2_plan_timing(self.plan)

    def reset(self) -> None:
        """Forget the transformed rows: the plan and workspace can take the next cluster of the same shape."""
        sie_dfmp2_plan_reset(self.plan)

    def close(self) -> None:
        sie_dfmp2_destroy(self.plan)
        self.plan = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
