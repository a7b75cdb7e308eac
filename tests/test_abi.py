"""Boundary checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
``include/mstar_attn.h`` declares; host-side argument validation rejects bad calls before any CUDA work."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_12688_b200 import build, binding
    build.build_library()
    return binding.load_library()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "mstar_attn.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mstar_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = declared_functions()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), "header declares %s but the library does not export it" % n
    from paper_2606_12688_b200 import EXPORTS
    assert sorted(EXPORTS) == names


def test_status_strings_and_version(lib):
    import paper_2606_12688_b200 as m
    assert m.status_string(0) == "MSTAR_OK"
    assert m.status_string(-1) == "MSTAR_ERR_INVALID_ARG"
    assert m.status_string(-2) == "MSTAR_ERR_UNSUPPORTED"
    assert m.status_string(-3) == "MSTAR_ERR_WORKSPACE_TOO_SMALL"
    assert m.status_string(-4) == "MSTAR_ERR_CUDA"
    assert re.match(r"\d+\.\d+\.\d+$", m.version())


def test_workspace_and_partition_queries(lib):
    import paper_2606_12688_b200 as m
    # config 5: 16 seqs x 32 heads x 16 partitions x (128 + 2) floats, plus headers
    assert m.decode_workspace_bytes(16, 32, 128, 16) >= 16 * 32 * 16 * 130 * 4
    assert m.decode_workspace_bytes(16, 32, 128, 1) <= 4096
    assert 1 <= m.decode_auto_partitions(64, 4, 4096) <= 128
    assert m.decode_auto_partitions(1, 1, 1) == 1


def test_host_validation_without_gpu(lib):
    """NULL pool / unsupported geometry / unknown flags are refused on the host, nothing is enqueued."""
    from paper_2606_12688_b200.binding import _KvPoolStruct
    assert lib.mstar_kv_append(None, None, None, None, 4, None) == -1
    bad = _KvPoolStruct(0x1000, 0x2000, 8, 24, 2, 128, 2 * 24 * 128, 24 * 128, 128)   # page_size 24
    assert lib.mstar_kv_append(ctypes.byref(bad), 0x100, 0x100, 0x100, 4, None) == -2
    bad = _KvPoolStruct(0x1000, 0x2000, 8, 16, 2, 96, 2 * 16 * 96, 16 * 96, 96)       # head_dim 96
    assert lib.mstar_kv_append(ctypes.byref(bad), 0x100, 0x100, 0x100, 4, None) == -2
    bad = _KvPoolStruct(0x1010, 0x2000, 8, 16, 2, 128, 2 * 16 * 128, 16 * 128, 128)   # misaligned K base
    assert lib.mstar_kv_append(ctypes.byref(bad), 0x100, 0x100, 0x100, 4, None) == -1
    ok = _KvPoolStruct(0x1000, 0x2000, 8, 16, 2, 128, 2 * 16 * 128, 16 * 128, 128)
    assert lib.mstar_paged_attn_decode(0x100, None, 0x100, ctypes.byref(ok), 0x100, 4, 0x100, 2, 4, 64, 0.1, 1,
                                       0x80, None, 0, None) == -1                     # unknown flag bit
    assert lib.mstar_paged_attn_decode(0x100, None, 0x100, ctypes.byref(ok), 0x100, 4, 0x100, 2, 3, 64, 0.1, 1,
                                       0, None, 0, None) == -1                        # Hq % Hkv != 0
    assert lib.mstar_paged_attn_decode(0x100, None, 0x100, ctypes.byref(ok), 0x100, 4, 0x100, 20000, 4, 64, 0.1, 1,
                                       0, None, 0, None) == -2                        # num_seqs > 16384
    assert lib.mstar_paged_attn_decode_cascade(0x100, None, 0x100, ctypes.byref(ok), 0x100, 4, 0x100, 0x100, 4, 2,
                                               68, 64, 0.1, 0, 0x100, 1 << 20, None) == -2   # cascade, G = 34 > 16
    assert lib.mstar_paged_attn_decode(0x100, None, 0x100, ctypes.byref(ok), 0x100, 4, 0x100, 2, 4, 4096, 0.1, 8,
                                       0, None, 0, None) == -1                        # partitions but no workspace


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_2606_12688_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(binding.MstarError, match="no CPU fallback"):
        binding.load_library()


def test_header_compiles_as_plain_c(tmp_path):
    """include/mstar_attn.h is a C header (extern "C" guards, no C++ types): gcc -std=c99 -pedantic takes it."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        import pytest
        pytest.skip("no gcc")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = tmp_path / "h.c"
    src.write_text('#include "mstar_attn.h"\nint main(void) { return (int)(MSTAR_DECODE_STATIC_WORKSPACE_BYTES >> 30); }\n')
    r = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(root, "include"),
                        "-c", str(src), "-o", str(tmp_path / "h.o")], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
