"""C-ABI library: loads on a CPU-only host, exports every symbol include/sie_dfmp2.h declares,
host-side planning/validation logic.  No compute calls (those are the -m gpu tests)."""
import ctypes
import os
import re

import pytest

import paper_2412_18553_b200 as sie
from paper_2412_18553_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2412_18553_b200 import build

    build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sie_dfmp2.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sie_dfmp2_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = ctypes.CDLL(binding.LIB_PATH)
    declared = _declared_symbols()
    assert {"sie_dfmp2_plan", "sie_dfmp2_transform", "sie_dfmp2_energy", "sie_dfmp2_batch"} <= set(declared)
    for name in declared:
        assert hasattr(lib, name), name
    assert set(binding.EXPORTS) == set(declared)


def test_library_does_not_link_libcuda():
    """It must load where no driver exists (this container): only the static runtime is linked."""
    import subprocess

    out = subprocess.run(["ldd", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "libcuda.so" not in out


def test_plan_is_host_only_and_reports_workspace():
    plan, ws = sie.sie_dfmp2_plan(48, 8, 40, 160)
    info = sie.sie_dfmp2_plan_info(plan)
    assert info["TM"] == 128 and info["TN"] == 128 and info["o8"] == 8 and info["ta"] == 16  # 16 blocks of o=8 rows
    nblk = (40 + 15) // 16
    assert info["ntiles"] == nblk * (nblk + 1) // 2 and info["reference"] == 0
    assert ws >= 40 * 8 * 160 * 8  # at least B
    sie.sie_dfmp2_destroy(plan)
    # config 3: B alone is ~5 GB; 1080 virtual blocks -> 584k tiles
    plan, ws = sie.sie_dfmp2_plan(1200, 120, 1080, 4800)
    info = sie.sie_dfmp2_plan_info(plan)
    assert info["TM"] == 120 and info["ta"] == 1 and info["o8"] == 120 and info["ntiles"] == 1080 * 1081 // 2 and info["ncta"] == 148
    assert 4.9e9 < ws < 9e9  # B 4.98 GB + an H sub-block of at most 2 GB + partial-G slots
    sie.sie_dfmp2_destroy(plan)
    # o is never padded inside a tile: o=30 -> 4 blocks = 120 rows exactly; o=17 -> 7 blocks = 119 rows -> 120
    for o, ta, t8 in ((30, 4, 120), (17, 7, 120), (33, 3, 104), (65, 1, 72), (128, 1, 128)):
        plan, _ = sie.sie_dfmp2_plan(10 * o, o, 8 * o, 100)
        info = sie.sie_dfmp2_plan_info(plan)
        assert (info["ta"], info["TM"], info["TN"]) == (ta, t8, t8), (o, info)
        sie.sie_dfmp2_destroy(plan)
    # nocc > 128 -> the general (slab / Gram) route; SIE_FLAG_REFERENCE -> the simple kernels; the route is reported, never silent
    plan, ws0 = sie.sie_dfmp2_plan(400, 130, 200, 300)
    info = sie.sie_dfmp2_plan_info(plan)
    assert info["general"] == 1 and info["reference"] == 0 and info["route"] == 2
    sie.sie_dfmp2_destroy(plan)
    plan, _ = sie.sie_dfmp2_plan(400, 130, 200, 300, 0, binding.SIE_FLAG_REFERENCE)
    assert sie.sie_dfmp2_plan_info(plan)["reference"] == 1
    sie.sie_dfmp2_destroy(plan)
    # SIE_FLAG_RDM_VIR reserves the three amplitude slabs of sie_dfmp2_rdm_vir
    plan, ws1 = sie.sie_dfmp2_plan(300, 30, 270, 1200)
    sie.sie_dfmp2_destroy(plan)
    plan, ws2 = sie.sie_dfmp2_plan(300, 30, 270, 1200, 0, binding.SIE_FLAG_RDM_VIR)
    sie.sie_dfmp2_destroy(plan)
    assert ws2 >= ws1 + 3 * 30 * 270 * 270 * 8
    # an amplitude slab beyond 4 GB is refused at plan time (sizes of the out-of-core NEXT-2 row)
    with pytest.raises(sie.SieError) as ei:
        sie.sie_dfmp2_plan(7000, 454, 5903, 19000)
    assert ei.value.status == binding.SIE_EINVAL


@pytest.mark.parametrize("args", [(0, 1, 1, 1), (10, 0, 5, 5), (10, 5, 0, 5), (10, 5, 5, 0), (9, 5, 5, 5), (10, 5, 5, 5, -1), (10, 5, 5, 5, 0, 128)])
def test_plan_rejects_bad_sizes(args):
    with pytest.raises(sie.SieError) as ei:
        sie.sie_dfmp2_plan(*args)
    assert ei.value.status == binding.SIE_EINVAL


def test_batch_query_needs_no_gpu():
    cl = [dict(nao=48, nocc=8, nvir=40, naux=160), dict(nao=144, nocc=16, nvir=128, naux=576)]
    n1 = sie.sie_dfmp2_batch_query(cl[:1])
    n2 = sie.sie_dfmp2_batch_query(cl)
    assert 0 < n1 < n2
    # host I/O adds staging + I/O mirrors but runs the transforms on one lane (device I/O: up to 4 lanes of scratch)
    nh1, nh2 = sie.sie_dfmp2_batch_query(cl[:1], binding.SIE_FLAG_HOST_IO), sie.sie_dfmp2_batch_query(cl, binding.SIE_FLAG_HOST_IO)
    assert n1 < nh1 < nh2
    assert sie.sie_dfmp2_batch_query([]) >= 0


def test_strerror_and_launch_counter():
    lib = binding._lib()
    assert lib.sie_dfmp2_strerror(0) == b"success"
    assert b"gap" in lib.sie_dfmp2_strerror(binding.SIE_EGAP)
    assert sie.launch_count() >= 0


def test_product_does_not_import_oracle():
    """The CUDA path and the oracle share no code: no file of the package mentions the oracle module."""
    pkg = os.path.join(ROOT, "paper_2412_18553_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "dfmp2_oracle" not in src, f
