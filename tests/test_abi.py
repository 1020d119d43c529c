"""The C-ABI library loads on a box without a GPU and exports every symbol include/emc.h declares;
argument validation is synchronous and needs no device.  No compute calls here."""
import ctypes
import pathlib
import re

import pytest

import paper_1409_4256_b200 as emc
from paper_1409_4256_b200 import binding

ROOT = pathlib.Path(__file__).resolve().parents[1]


def test_header_symbols_all_exported():
    header = (ROOT / "include" / "emc.h").read_text()
    declared = set(re.findall(r"EMC_API[^;(]*?\b(emc_\w+)\s*\(", header))
    assert declared == set(binding.SYMBOLS)
    lib = emc.load()
    for name in declared:
        assert hasattr(lib, name), name


def test_header_constants_match_binding():
    header = (ROOT / "include" / "emc.h").read_text()
    for name in ("EMC_COMPRESS_WEIGHTED", "EMC_ACCUMULATE", "EMC_UPDATE_RAW", "EMC_MAX_SPANS", "EMC_DEBUG_SIMT", "EMC_GEMM_1CTA",
                 "EMC_PATTERNS_ON_HOST", "EMC_PROFILE_STAGES", "EMC_MAX_COUNT"):
        m = re.search(rf"#define {name}\s+(0x[0-9a-fA-F]+|\d+)u?", header)
        assert m, name
        assert int(m.group(1), 0) == getattr(binding, name)
    for name in ("EMC_ERR_ARG", "EMC_ERR_UNSUPPORTED", "EMC_ERR_WORKSPACE", "EMC_ERR_CUDA", "EMC_ERR_COUNT_RANGE"):
        m = re.search(rf"{name} = (-\d+)", header)
        assert int(m.group(1)) == getattr(binding, name)


def test_version_and_strerror():
    lib = emc.load()
    assert b"sm_100a" in lib.emc_version()
    header = (ROOT / "include" / "emc.h").read_text()
    tiny = float(re.search(r"#define EMC_P_MIN\s+([0-9.e+-]+)f", header).group(1))
    assert tiny == 2.0 ** -126                      # float32's smallest normal number (G20)
    assert lib.emc_strerror(0) == b"ok"
    assert b"workspace" in lib.emc_strerror(emc.EMC_ERR_WORKSPACE)


def test_workspace_bytes_monotone_and_rejects_bad_sizes():
    a = emc.emc_workspace_bytes(32, 1024, 480, 1000)
    b = emc.emc_workspace_bytes(32, 1024, 960, 1000)
    c = emc.emc_workspace_bytes(32, 1024, 480, 1000, emc.EMC_PATTERNS_ON_HOST)
    assert 0 < a < b and c > a
    assert emc.emc_workspace_bytes(1, 1024, 480, 1000) == 0
    assert emc.emc_workspace_bytes(32, 0, 480, 1000) == 0
    assert emc.emc_workspace_bytes(2048, 16, 4, 4) == 0


def test_null_arguments_are_rejected_synchronously():
    lib = emc.load()
    assert lib.emc_expand(None, None, None, None, None, None, 0, None) == emc.EMC_ERR_ARG
    assert lib.emc_check(None, None) == emc.EMC_ERR_ARG
    det = binding._Detector(16, 8, None, 0)
    pat = binding._Patterns(4, 8, emc.binding.EMC_U16)
    # misaligned / missing workspace
    assert lib.emc_loglik(8, None, det, pat, 4, 16, 64, 0, None, 0, None) == emc.EMC_ERR_WORKSPACE
    assert lib.emc_loglik(8, None, det, pat, 4, 16, 3, 0, 256, 1 << 30, None) == emc.EMC_ERR_ARG   # ld_n < N
    m = binding._Model(16, 8)
    rot = binding._Rotations(4, 8, None)
    # model_out aliasing the model is an argument error
    assert lib.emc_iterate(m, det, rot, pat, 1, 0, 8, None, 64, 8, 0, 256, 1 << 30, None, None) == emc.EMC_ERR_ARG
    # host-resident patterns and per-stage timing need the caller's context
    for flag in (emc.EMC_PATTERNS_ON_HOST, emc.EMC_PROFILE_STAGES):
        assert lib.emc_iterate(m, det, rot, pat, 1, 0, 16, None, 64, 8, flag, 256, 1 << 30, None, None) == emc.EMC_ERR_ARG
    assert lib.emc_context_create(None) == emc.EMC_ERR_ARG
    assert lib.emc_context_destroy(None) == emc.EMC_OK
    assert lib.emc_profile_read(None, None, None) == emc.EMC_ERR_ARG
    assert lib.emc_profile_dropped(None) == 0
    # flags a call does not implement are refused, not ignored (rotation chunks run the dense, device-resident path)
    for flag in (emc.EMC_SPARSE_PHOTONS, emc.EMC_PATTERNS_ON_HOST):
        assert lib.emc_iterate_rot_chunked(m, det, rot, pat, 1, 2, 16, 8, flag, 256, 1 << 30, None, None) == emc.EMC_ERR_UNSUPPORTED
    # photon lists index a chunk with 32 bits: chunk x pixels must stay below 2^31
    assert emc.emc_workspace_bytes(32, 65536, 100, 32768, emc.EMC_SPARSE_PHOTONS) == 0
    assert emc.emc_workspace_bytes(32, 65536, 100, 32767, emc.EMC_SPARSE_PHOTONS) > 0
    big = binding._Patterns(40000, 8, emc.binding.EMC_U16)
    det_big = binding._Detector(65536, 8, None, 0)
    assert lib.emc_iterate(m, det_big, rot, big, 1, 0, 16, None, 64, 8, emc.EMC_SPARSE_PHOTONS, 256, 1 << 40, None, None) == emc.EMC_ERR_UNSUPPORTED
    # emc_workspace_view: host-side pointer arithmetic
    ptr, ld = ctypes.c_void_p(), ctypes.c_int()
    assert lib.emc_workspace_view(4096, 16, 16, 4, 4, 0, emc.EMC_VIEW_LOGLIK, ctypes.byref(ptr), ctypes.byref(ld)) == emc.EMC_OK
    assert ptr.value > 4096 and ld.value == 64
    assert lib.emc_workspace_view(4096, 16, 16, 4, 4, emc.EMC_SPARSE_PHOTONS, emc.EMC_VIEW_LOGLIK, ctypes.byref(ptr), ctypes.byref(ld)) == emc.EMC_ERR_UNSUPPORTED
    assert lib.emc_workspace_view(4096, 16, 16, 4, 4, 0, 99, ctypes.byref(ptr), ctypes.byref(ld)) == emc.EMC_ERR_ARG


def test_binding_refuses_cpu_tensors():
    import torch

    with pytest.raises(TypeError):
        emc.emc_expand(torch.zeros(4, 4, 4), torch.zeros(3, 3), torch.zeros(2, 4))
