"""CPU-side checks of the C-ABI boundary: the library builds/loads here (no GPU), exports every symbol
include/rfoe.h declares, and fails loudly -- never falls back -- when no CUDA device is present."""
import ctypes
import os
import re

import pytest

import paper_2301_04642_b200 as rfoe

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "rfoe.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(rfoe_[a-z0-9_]+)\s*\(", txt)))


def test_header_symbols_are_exported():
    L = rfoe.load_library()
    declared = _declared_symbols()
    assert set(declared) == set(rfoe.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name
    assert L.rfoe_version() == 201
    assert L.rfoe_strerror(0) == b"ok" and b"symmetric" in L.rfoe_strerror(5)


def test_stats_struct_matches_header():
    # sizeof(rfoe_stats_t) computed from the header's field list
    n = rfoe.MAX_STEPS
    expect = 12 * 4 + 3 * 8 + 11 * 8 + (n + 1) * 8 * 2 + n * 8 * 2 + (n + 8)
    expect = (expect + 7) // 8 * 8
    assert ctypes.sizeof(rfoe._Stats) == expect


def test_header_is_plain_c_and_struct_size_matches_the_binding(tmp_path):
    """include/rfoe.h compiles as strict C99 (no C++, no torch types) inside a C client that links librfoe.so; the
    compiler's sizeof(rfoe_stats_t) is the binding's."""
    import subprocess

    from tests import abi_client_build

    exe = abi_client_build.build(tmp_path)
    out = subprocess.run([exe, "sizeof"], check=True, capture_output=True, text=True).stdout
    kv = dict(p.split("=") for p in out.split())
    assert int(kv["sizeof_stats"]) == ctypes.sizeof(rfoe._Stats)
    assert int(kv["version"]) == 201 and int(kv["max_steps"]) == rfoe.MAX_STEPS


def test_bounds_static_argument_errors_without_gpu():
    """rfoe_bounds_static settles its arguments before it touches CUDA: null pointers, k < 1, and the size limit of its fixed
    scratch array (RFOE_STATIC_MAX_K, with a message that names it) -- and on a box without a device the first CUDA call fails
    loudly (RFOE_ERR_CUDA with the cudaError_t handed back), it does not fall back to anything."""
    L = rfoe.load_library()
    err = ctypes.c_int(-1)
    fake = ctypes.c_void_p(4096)          # never dereferenced on these paths
    assert L.rfoe_bounds_static(None, 16, fake, None, ctypes.byref(err)) == rfoe.ERR_INVALID_ARG and err.value == 0
    assert L.rfoe_bounds_static(fake, 16, None, None, None) == rfoe.ERR_INVALID_ARG
    assert L.rfoe_bounds_static(fake, 0, fake, None, None) == rfoe.ERR_INVALID_ARG
    assert L.rfoe_bounds_static(fake, rfoe.STATIC_MAX_K + 1, fake, None, ctypes.byref(err)) == rfoe.ERR_STATIC_LIMIT and err.value == 0
    assert b"RFOE_STATIC_MAX_K" in L.rfoe_strerror(rfoe.ERR_STATIC_LIMIT)
    hdr = open(os.path.join(ROOT, "include", "rfoe.h")).read()
    assert re.search(r"#define\s+RFOE_STATIC_MAX_K\s+(\d+)", hdr).group(1) == str(rfoe.STATIC_MAX_K)
    import torch

    if not torch.cuda.is_available():
        rc = L.rfoe_bounds_static(fake, 16, fake, None, ctypes.byref(err))
        assert rc in (rfoe.ERR_CUDA, rfoe.ERR_UNSUPPORTED) and (rc != rfoe.ERR_CUDA or err.value != 0)


def test_argument_errors_without_gpu():
    L = rfoe.load_library()
    h = ctypes.c_void_p()
    assert L.rfoe_create(None, 0, 16) == rfoe.ERR_INVALID_ARG
    assert L.rfoe_create(ctypes.byref(h), 0, 0) == rfoe.ERR_INVALID_ARG
    assert L.rfoe_destroy(None) == rfoe.OK
    assert L.rfoe_set_option(None, 0, 0.0) == rfoe.ERR_INVALID_ARG
    assert L.rfoe_expand_many(None, None, 1, 0, None, None, None, 0, None, None, None, None) == rfoe.ERR_INVALID_ARG
    hs, ss = (ctypes.c_void_p * 1)(None), (ctypes.c_void_p * 1)(None)
    assert L.rfoe_expand_many(hs, ss, 1, 0, None, None, None, 0, None, None, None, None) == rfoe.ERR_INVALID_ARG   # null handle
    assert L.rfoe_expand_many(hs, ss, 0, 0, None, None, None, 0, None, None, None, None) == rfoe.ERR_INVALID_ARG


def test_no_cpu_fallback():
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(rfoe.RfoeError) as ei:
        rfoe.Rfoe(64)
    assert ei.value.status == rfoe.ERR_CUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2301_04642_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2301_04642_b200" not in src and "csrc/" not in src.replace("paper_2301_04642_b200/csrc/", "")
