"""The C-ABI shared library builds for sm_100a, loads without a GPU and exports every symbol that
include/bm.h declares; host-side argument checking works without touching the device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "bm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bm_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_2607_04164_b200 as bm
    L = bm.lib()
    names = _declared_symbols()
    assert {"bm_route", "bm_moe_forward", "bm_workspace_bytes", "bm_status_string"} <= set(names)
    for n in names:
        assert hasattr(L, n), f"libbm.so does not export {n}"
    from paper_2607_04164_b200.binding import EXPORTS
    assert sorted(EXPORTS) == names


def test_library_is_sm100a_tcgen05_tma():
    """SASS evidence that the GEMM kernels are Blackwell-native (B200_PROFILING.md table)."""
    import shutil
    import subprocess
    import paper_2607_04164_b200 as bm
    bm.lib()
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    so = os.path.join(ROOT, "paper_2607_04164_b200", "libbm.so")
    sass = subprocess.run(["cuobjdump", "-sass", so], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    for mnemonic in ("UTCHMMA", "LDTM", "UTMALDG"):
        assert mnemonic in sass, mnemonic


def test_workspace_bytes_and_status_strings():
    import paper_2607_04164_b200 as bm
    small = bm.workspace_bytes(64, 256, 512, 8, 2, 4, 0)
    big = bm.workspace_bytes(8192, 4096, 14336, 8, 2, 4, 0)
    assert 0 < small < big
    # H [T*K, F] + xs [T*K, D] bf16 + out_acc [T, D] f32 dominate
    assert big >= 8192 * 2 * (14336 + 4096) * 2 + 8192 * 4096 * 4
    assert bm.workspace_bytes(-1, 256, 512, 8, 2, 4, 0) == 0
    assert bm.status_string(0) == "BM_OK"
    for code in range(-6, 0):
        assert bm.status_string(code).startswith("BM_ERR_")


def test_argument_errors_are_reported_before_any_device_work():
    """Shape/NULL checks run on the host; without a GPU the remaining calls must fail loudly (BM_ERR_CUDA)."""
    import paper_2607_04164_b200 as bm
    from paper_2607_04164_b200.binding import BmRouting
    L = bm.lib()
    r = BmRouting()
    # K > E
    assert L.bm_route(None, 4, 64, None, None, 2, 3, None, 2, ctypes.byref(r), None, 0, None) == -2
    # D not a multiple of 8
    assert L.bm_route(None, 4, 60, None, None, 8, 2, None, 2, ctypes.byref(r), None, 0, None) == -2
    # NULL routing struct
    assert L.bm_route(None, 4, 64, None, None, 8, 2, None, 2, None, None, 0, None) == -1
    # good shapes, NULL pointers
    assert L.bm_route(None, 4, 64, None, None, 8, 2, None, 2, ctypes.byref(r), None, 0, None) == -1
    import torch
    if not torch.cuda.is_available():
        buf = (ctypes.c_uint8 * 8192)()
        addr = (ctypes.addressof(buf) + 15) & ~15
        p = ctypes.c_void_p(addr)
        r2 = BmRouting(0, 0, 2, 2, *([addr] * 9))
        rc = L.bm_route(p, 4, 64, p, None, 8, 2, p, 2, ctypes.byref(r2), p, 1 << 20, None)
        assert rc == -5, "without a CUDA device the product path must fail loudly, not fall back"


def test_options_round_trip_and_unknown_name():
    import paper_2607_04164_b200 as bm
    old = bm.get_option("PF_PAIR")
    with bm.options(PF_PAIR=1, FUSED_COMBINE=0):
        assert bm.get_option("PF_PAIR") == 1 and bm.get_option("FUSED_COMBINE") == 0
    assert bm.get_option("PF_PAIR") == old and bm.get_option("FUSED_COMBINE") == -1
    with pytest.raises(bm.BmError) as ei:
        bm.set_option("NO_SUCH_OPTION", 1)
    assert ei.value.code == -2
    # every option documented in bm.h exists in the library, and the other way round the table has no undocumented name
    src = open(os.path.join(ROOT, "include", "bm.h")).read()
    doc = src[src.index(" * Options:"):src.index("int bm_set_option")]
    names = []
    for line in doc.splitlines():
        m = re.match(r" \*   ([A-Z][A-Z0-9_]+(?: \([-0-9]+\))?(?:, [A-Z][A-Z0-9_]+(?: \([-0-9]+\))?)*)", line)
        if m:
            names += re.findall(r"[A-Z][A-Z0-9_]+", m.group(1))
    assert len(names) >= 25
    for name in names:
        bm.get_option(name)


def test_forward_info_is_a_host_call():
    """bm_forward_info answers from the host-side sizes alone (no device needed): path and determinism (include/bm.h)."""
    import paper_2607_04164_b200 as bm
    assert bm.bm_forward_info(1, 4, 60, 0, 2048, 1408) == (bm.BM_PATH_GEMV, True)
    assert bm.bm_forward_info(8192, 2, 4, 0, 4096, 14336) == (bm.BM_PATH_PREFILL, True)      # fused, two sources
    assert bm.bm_forward_info(4096, 6, 16, 2, 2048, 1408) == (bm.BM_PATH_PREFILL, True)      # F < 4096: two-pass, slot order
    path, det = bm.bm_forward_info(4096, 4, 60, 0, 2048, 4096)
    assert path == bm.BM_PATH_PREFILL and not det                                             # fused, four sources
    path, det = bm.bm_forward_info(64, 2, 4, 0, 4096, 14336)
    assert path == bm.BM_PATH_DECODE and not det                                              # K splits: order varies
    with pytest.raises(bm.BmError):
        bm.bm_forward_info(4, 99, 4, 0, 64, 64)


def test_host_chunk_plan_is_a_host_call():
    """bm_host_chunks (include/bm.h, bm_moe_layer_host): chunks cover the batch exactly, at most 16, whole 128-row tiles
    except the last; about 2816 tokens where compute outweighs the copies, 2048 elsewhere."""
    import paper_2607_04164_b200 as bm
    assert bm.bm_host_chunks(8192, 14336, 2, 0) == [2816, 2816, 2560]
    assert bm.bm_host_chunks(5631, 14336, 2, 0) == [5631]                                      # below two chunks: one piece
    assert bm.bm_host_chunks(16384, 14336, 2, 0) == [2816] * 5 + [2304]
    assert bm.bm_host_chunks(64, 14336, 2, 0) == [64]
    assert bm.bm_host_chunks(8192, 1408, 4, 0) == [2048] * 4                                   # copies ~ compute: smaller chunks
    assert bm.bm_host_chunks(4095, 1408, 4, 4) == [4095]
    for F, K, S in ((14336, 2, 0), (1408, 4, 4), (4096, 8, 1)):
        for T in (0, 1, 2047, 4096, 4097, 5632, 8192, 8193, 12345, 16384, 65536, 300000):
            c = bm.bm_host_chunks(T, F, K, S)
            assert sum(c) == T and 1 <= len(c) <= 16
            assert all(v > 0 for v in c) or T == 0
            assert all(v % 128 == 0 for v in c[:-1]) and len(set(c[:-1])) <= 1 and c[-1] <= c[0]
    with bm.options(HOST_CHUNK_T=0):
        assert bm.bm_host_chunks(8192, 14336, 2, 0) == [8192]
    with bm.options(HOST_CHUNK_T=512):
        assert bm.bm_host_chunks(3000, 320, 3, 1) == [512] * 5 + [440]
    with pytest.raises(bm.BmError):
        bm.bm_host_chunks(-1, 64, 1, 0)


def test_workspace_layout_invariants():
    """bm_workspace_bytes: monotone in T (a workspace for T_max serves every smaller batch), zero for arguments no call
    accepts, and large enough for the dense decode rows (one H row per active set and token up to 64 tokens)."""
    import paper_2607_04164_b200 as bm
    prev = 0
    for T in (0, 1, 2, 16, 63, 64, 65, 128, 511, 512, 4096, 8192):
        n = bm.workspace_bytes(T, 2048, 1408, 60, 4, 60, 0)
        assert n >= prev
        prev = n
    assert bm.workspace_bytes(64, 2048, 1408, 60, 4, 60, 0) >= 60 * 64 * 1408 * 2            # dense H rows
    assert bm.workspace_bytes(64, 256, 512, 8, 2, 4, 17) == 0                                  # S > BM_MAX_S
    assert bm.BM_MAX_S == 16
