"""CPU checks of the boundary: libfstc.so builds/loads, exports every symbol include/fstc.h declares,
and the ctypes mirrors of the structs have the layout the C compiler gives them.  No compute calls."""
from __future__ import annotations

import ctypes
import os
import re
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "fstc.h")


@pytest.fixture(scope="module")
def libpath():
    from paper_1805_06383_b200 import build, fstc
    if not os.path.exists(fstc.LIB_PATH):
        if shutil.which("nvcc") is None and not os.path.exists("/usr/local/cuda/bin/nvcc"):
            pytest.skip("libfstc.so not built and no nvcc here")
        build.build()
    return fstc.LIB_PATH


def _declared():
    text = open(HEADER).read()
    return sorted(set(re.findall(r"FSTC_API\s+[\w\s\*]+?\b(fstc_\w+)\s*\(", text)))


def test_header_declares_the_documented_entry_points():
    names = _declared()
    for must in ("fstc_compose", "fstc_pack", "fstc_compose_packed", "fstc_result_free", "fstc_packed_free"):
        assert must in names


def test_library_exports_every_declared_symbol(libpath):
    from paper_1805_06383_b200 import fstc
    L = ctypes.CDLL(libpath)
    names = _declared()
    assert set(names) == set(fstc.EXPORTS)
    for n in names:
        assert hasattr(L, n), n
    L.fstc_version.restype = ctypes.c_int
    assert L.fstc_version() == 3
    L.fstc_strerror.restype = ctypes.c_char_p
    assert L.fstc_strerror(-4) == b"internal capacity limit exceeded"


def test_library_has_sm100a_code(libpath):
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("no cuobjdump")
    out = subprocess.run([cuobjdump, "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_ctypes_struct_layout_matches_the_c_compiler(tmp_path):
    from paper_1805_06383_b200 import fstc
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "fstc.h"\nint main(void){\n'
                   'printf("%zu %zu %zu %zu %zu\\n", sizeof(fstc_fst_t), sizeof(fstc_opts_t), sizeof(fstc_stats_t),'
                   ' sizeof(fstc_result_t), sizeof(fstc_host_result_t));\n'
                   'printf("%zu %zu %zu %zu %zu %zu\\n", offsetof(fstc_fst_t, mem), offsetof(fstc_opts_t, profile),'
                   ' offsetof(fstc_stats_t, ms_total), offsetof(fstc_result_t, expanded), offsetof(fstc_opts_t, alloc_ctx),'
                   ' offsetof(fstc_stats_t, small_path));\nreturn 0;}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    a, b = subprocess.check_output([str(exe)], text=True).strip().split("\n")
    sizes = [int(x) for x in a.split()]
    offs = [int(x) for x in b.split()]
    assert sizes == [ctypes.sizeof(fstc._Fst), ctypes.sizeof(fstc._Opts), ctypes.sizeof(fstc._Stats),
                     ctypes.sizeof(fstc._Result), ctypes.sizeof(fstc._HostResult)]
    assert offs == [fstc._Fst.mem.offset, fstc._Opts.profile.offset, fstc._Stats.ms_total.offset,
                    fstc._Result.expanded.offset, fstc._Opts.alloc_ctx.offset, fstc._Stats.small_path.offset]


def test_static_entry_point_structs_match_the_c_compiler(tmp_path):
    from paper_1805_06383_b200 import fstc
    src = tmp_path / "st.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "fstc.h"\nint main(void){\n'
                   'printf("%zu %zu %zu %zu %d %u\\n", sizeof(fstc_static_header_t), sizeof(fstc_static_out_t),'
                   ' offsetof(fstc_static_header_t, status), offsetof(fstc_static_out_t, header),'
                   ' FSTC_STATIC_MAX_STATES, FSTC_STATIC_SCRATCH_BYTES);\nreturn 0;}\n')
    exe = tmp_path / "st"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(x) for x in subprocess.check_output([str(exe)], text=True).split()]
    assert got == [ctypes.sizeof(fstc._StaticHeader), ctypes.sizeof(fstc._StaticOut), fstc._StaticHeader.status.offset,
                   fstc._StaticOut.header.offset, fstc.STATIC_MAX_STATES, fstc.STATIC_SCRATCH_BYTES]
    assert got[0] == 80


def test_no_product_path_touches_the_oracle():
    """The oracle is test infrastructure: the package must not import or mention it."""
    pkg = os.path.join(ROOT, "paper_1805_06383_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in dirpath.split(os.sep)[-1:]:
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f), errors="ignore").read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "fst_compose_oracle" not in text and "libfst_oracle" not in text, f
