"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/cx_bwt.h declares; argument errors come back as codes; workspace sizing is monotone."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "cx_bwt.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cx_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_1401_7457_b200 as cx
    L = cx.lib()
    names = _declared()
    assert {"cx_bwt_plan", "cx_bwt_build", "cx_bwt_free", "cx_pack_reads", "cx_bwt_workspace_bytes", "cx_strerror"} <= set(names)
    for n in names:
        assert getattr(L, n) is not None


def test_workspace_bytes_and_argument_errors():
    import paper_1401_7457_b200 as cx
    a = cx.cx_bwt_workspace_bytes(10_000, 1_000_000, max_read_len=100)
    b = cx.cx_bwt_workspace_bytes(1_000_000, 100_000_000, max_read_len=100)
    assert 0 < a < b
    # 4-byte ids: 2*8 (keys) + 2*4 (ids) + 4 (the global path's second position array) bytes per suffix plus flags and tile
    # state (until the global path gave up its own buffers it was 2*8 + 3*4 + 4)
    assert 28 * 101_000_000 < b < 33 * 101_000_000
    # 8-byte ids (read length unknown) with pinned-host output: 2*8 + 2*8 + 2 staging bytes, no position array
    c = cx.cx_bwt_workspace_bytes(1_000_000, 100_000_000, max_read_len=0, out_is_host_pinned=1)
    assert 34 * 101_000_000 < c < 38 * 101_000_000
    c = cx.cx_bwt_workspace_bytes(1_000_000, 100_000_000, max_read_len=100, max_batch_suffixes=10_000_000)
    assert c < b / 5
    d = cx.cx_bwt_workspace_bytes(40_000_000, 6_000_000_000, max_read_len=250)     # 8-byte ids
    assert d > 0
    with pytest.raises(cx.CxError) as e:
        cx.cx_bwt_workspace_bytes(10, 1000, prefix_len=9)
    assert e.value.code == -1
    with pytest.raises(cx.CxError):
        cx.cx_bwt_workspace_bytes(10, 1000, key_bases=30)
    with pytest.raises(cx.CxError):
        cx.cx_bwt_workspace_bytes(10, 1000, shard_index=2, shard_count=2)       # NEXT-2: index must be below the count
    # a sharded plan always needs the multi-batch count table, so it asks for a little more than the unsharded one
    assert cx.cx_bwt_workspace_bytes(10_000, 1_000_000, max_read_len=100, shard_index=1, shard_count=2) > a
    L = cx.lib()
    assert L.cx_bwt_plan(None, 1, 1, None, None, 0) == -1
    assert L.cx_bwt_build(None, None, None, 1, None, None) == -1
    assert L.cx_bwt_free(None) == 0
    assert b"ACGT" in L.cx_strerror(-2)


def test_no_cpu_fallback_in_product():
    """The product never imports the oracle, and the oracle never imports the product."""
    pkg = os.path.join(ROOT, "paper_1401_7457_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(dirpath, f)).read().lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1401_7457_b200" not in src and "from paper_1401_7457_b200" not in src


# ---- a C-language consumer of the header (the boundary is a C ABI, not a Python one) --------------------------------
_C_SRC = os.path.join(ROOT, "tests", "c_consumer", "figure1.c")
_CUDA_INC = os.environ.get("CUDA_HOME", "/usr/local/cuda") + "/include"
_CUDA_LIB = os.environ.get("CUDA_HOME", "/usr/local/cuda") + "/lib64"


def _compile_c_consumer(tmp_path):
    import subprocess
    import paper_1401_7457_b200 as cx
    cx.lib()                                             # builds libcxbwt.so if stale
    pkg = os.path.join(ROOT, "paper_1401_7457_b200")
    exe = str(tmp_path / "figure1")
    # strict C99: the header must not rely on C++ (extern "C" is guarded, cx_stream_t is an incomplete struct pointer)
    subprocess.check_call(["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-I" + os.path.join(ROOT, "include"), "-isystem", _CUDA_INC,
                           _C_SRC, "-o", exe, "-L" + pkg, "-lcxbwt", "-L" + _CUDA_LIB, "-lcudart", "-Wl,-rpath," + pkg, "-Wl,-rpath," + _CUDA_LIB])
    return exe


def test_header_compiles_as_c_and_links(tmp_path):
    assert os.path.exists(_compile_c_consumer(tmp_path))


@pytest.mark.gpu
def test_c_consumer_runs_figure1(tmp_path):
    import subprocess
    r = subprocess.run([_compile_c_consumer(tmp_path)], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.split() == ["TTAAG$TAG$CAGG$", "15"]          # PAPER.md:59, Figure 1
